// sfd_warp1024.cuh — the N = 1024 fast path: one warp per line, 32 complex values per thread.
//
// The padded 2N-point transforms of PAPER.md steps (ii)-(ix) (L86-93) have a zero upper half on
// the way in and a discarded upper half on the way out.  Splitting the 2N-point DFT by the parity
// of the frequency index uses both facts exactly (w = exp(-2 pi i / 2N)):
//
//     forward:  X[2k]   = FFT_N(x)[k],            X[2k+1] = FFT_N(x[n] w^n)[k]
//     inverse:  y[n]    = IFFT_N(Y[2k])[n] + w^-n IFFT_N(Y[2k+1])[n]          (n < N)
//
// so a line is two independent "branches" b = 0 (even bins), 1 (odd bins):
//
//     out[n] = sum_b post_b[n] * IFFT_N( H_b[k] * FFT_N( in[n] pre_b[n] ) )[n]
//     pre_1 = pre w^n,  post_1 = post w^-n,  H_0[k] = H[2k],  H_1[k] = H[2k+1]     (plan-time tables)
//
// With N = 1024 = 32 x 32 an N-point FFT is two radix-32 register butterflies around ONE 32 x 32
// transpose, and a warp (32 lanes x 32 values) owns the whole line: the transpose goes through a
// private shared-memory tile guarded by __syncwarp only; no CTA barrier exists on the FFT path.
// Per line this moves 4 x 16 KiB through shared memory instead of 8 x 32 KiB (generic path) and the
// inter-stage twiddles w1024^(lane * k1) are per-thread constants kept in registers for the whole
// (persistent) kernel.
#pragma once
#include "sfd_fft_core.cuh"

namespace sfdw {

using sfd::cadd;
using sfd::cmul;
using sfd::csub;

constexpr int N = 1024;     // line length handled by this path
constexpr int XS = 34;      // row stride (complex) of the transpose tile: 16-byte aligned rows,
                            // conflict-free for both the 8-byte column writes and 16-byte row reads
constexpr int XB = 32 * XS;  // complex elements of one warp's transpose tile

// a * exp(DIR * 2 pi i * K / 32)
template <int DIR, int K> __device__ __forceinline__ float2 mul_w32(float2 a) {
    if constexpr (K % 2 == 0) {
        return sfd::mul_w16<DIR, K / 2>(a);
    } else {
        constexpr float C[8] = {0.98078528040323044913f, 0.83146961230254523708f,
                                0.55557023301960222474f, 0.19509032201612826785f,
                                -0.19509032201612826785f, -0.55557023301960222474f,
                                -0.83146961230254523708f, -0.98078528040323044913f};
        constexpr float S[8] = {0.19509032201612826785f, 0.55557023301960222474f,
                                0.83146961230254523708f, 0.98078528040323044913f,
                                0.98078528040323044913f, 0.83146961230254523708f,
                                0.55557023301960222474f, 0.19509032201612826785f};
        constexpr float c = C[K / 2], s = DIR * S[K / 2];
        return make_float2(a.x * c - a.y * s, a.x * s + a.y * c);
    }
}

// 32-point DFT in registers, natural order in and out, W = exp(DIR * 2 pi i / 32):
// X[k] = E[k] + W^k O[k], X[k+16] = E[k] - W^k O[k] with E/O the 16-point DFTs of the even/odd
// inputs.
template <int DIR> __device__ __forceinline__ void dft32(float2 (&a)[32]) {
    float2 e[16], o[16];
#pragma unroll
    for (int s = 0; s < 16; ++s) {
        e[s] = a[2 * s];
        o[s] = a[2 * s + 1];
    }
    sfd::dft16<DIR, false>(e);
    sfd::dft16<DIR, false>(o);
#define SFDW_BF(K)                                   \
    {                                                \
        const float2 t = mul_w32<DIR, K>(o[K]);      \
        a[K] = cadd(e[K], t);                        \
        a[K + 16] = csub(e[K], t);                   \
    }
    SFDW_BF(0) SFDW_BF(1) SFDW_BF(2) SFDW_BF(3) SFDW_BF(4) SFDW_BF(5) SFDW_BF(6) SFDW_BF(7)
    SFDW_BF(8) SFDW_BF(9) SFDW_BF(10) SFDW_BF(11) SFDW_BF(12) SFDW_BF(13) SFDW_BF(14) SFDW_BF(15)
#undef SFDW_BF
}

// 1024-point FFT of one warp.  In: v[r] = x[lane + 32 r].  Out: v[r] = X[lane + 32 r].
// tw[k] = exp(-2 pi i lane k / 1024) (this thread's inter-stage twiddles), xb = the warp's tile.
template <int DIR>
__device__ __forceinline__ void fft1024(float2 (&v)[32], int lane, float2 *xb,
                                        const float2 (&tw)[32]) {
    dft32<DIR>(v);  // over n1 for n2 = lane: v[k1]
#pragma unroll
    for (int k = 1; k < 32; ++k) {
        const float2 w = DIR < 0 ? tw[k] : make_float2(tw[k].x, -tw[k].y);
        v[k] = cmul(v[k], w);
    }
#pragma unroll
    for (int k = 0; k < 32; ++k) xb[k * XS + lane] = v[k];  // (k1 = k, n2 = lane)
    __syncwarp();
    const float4 *row = reinterpret_cast<const float4 *>(xb + lane * XS);  // k1 = lane, all n2
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const float4 t = row[q];
        v[2 * q] = make_float2(t.x, t.y);
        v[2 * q + 1] = make_float2(t.z, t.w);
    }
    __syncwarp();
    dft32<DIR>(v);  // over n2 for k1 = lane: v[k2] = X[lane + 32 k2]
}

// One branch of a line, in place: v *= pre is done by the caller; here FFT, x H_b, inverse FFT.
__device__ __forceinline__ void branch(float2 (&v)[32], int lane, float2 *xb,
                                       const float2 (&tw)[32], const float2 *__restrict__ Hb) {
    fft1024<-1>(v, lane, xb, tw);
#pragma unroll
    for (int k = 0; k < 32; ++k) v[k] = cmul(v[k], __ldg(Hb + lane + 32 * k));
    fft1024<+1>(v, lane, xb, tw);
}

__device__ __forceinline__ void load_twiddles(float2 (&tw)[32], int lane,
                                              const float2 *__restrict__ twl) {
#pragma unroll
    for (int k = 0; k < 32; ++k) tw[k] = __ldg(twl + k * 32 + lane);
}

// ---- pass y: 4 adjacent hologram columns per CTA (one per warp) -----------------------------------
constexpr int YC = 4;           // columns per CTA
constexpr int CS = N + 4;       // stride (complex) between the CTA's column buffers: puts columns
                                // c and c+2 sixteen banks apart for the transposed read-out
struct SmemY {
    float2 xb[YC][XB];
    float2 col[YC][CS];
    unsigned int tile[N];       // uint8 input: row n0 -> the 4 bytes of columns col0..col0+3
};

template <typename TIn>
__device__ __forceinline__ void pass_y_cta(SmemY &sm, const TIn *__restrict__ holo,
                                           const float2 *__restrict__ tab,  // view's [pre2|post2|..]
                                           const float2 *__restrict__ H2, const float2 (&tw)[32],
                                           float2 *__restrict__ Bv, int col0) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if constexpr (sizeof(TIn) == 1) {
        __syncthreads();  // previous item's readers of tile / col are done
#pragma unroll
        for (int i = 0; i < N / 128; ++i) {
            const int row = threadIdx.x + 128 * i;
            sm.tile[row] = __ldg(reinterpret_cast<const unsigned int *>(holo + (size_t)row * N + col0));
        }
        __syncthreads();
    } else {
        __syncthreads();
    }
    float2 *xb = sm.xb[warp];
    float2 *col = sm.col[warp];
#pragma unroll 1
    for (int b = 0; b < 2; ++b) {
        const float2 *pre = tab + b * N;             // pre_y branch b (carries 1/255 for uint8)
        const float2 *post = tab + 2 * N + b * N;    // c0 post_y branch b
        float2 v[32];
#pragma unroll
        for (int r = 0; r < 32; ++r) {
            const int n0 = lane + 32 * r;
            float a;
            if constexpr (sizeof(TIn) == 1)
                a = (float)((sm.tile[n0] >> (8 * warp)) & 0xffu);
            else
                a = __ldg(holo + (size_t)n0 * N + col0 + warp);
            const float2 p = __ldg(pre + n0);
            v[r] = make_float2(a * p.x, a * p.y);
        }
        branch(v, lane, xb, tw, H2 + b * N);
        if (b == 0) {
#pragma unroll
            for (int r = 0; r < 32; ++r) col[lane + 32 * r] = cmul(v[r], __ldg(post + lane + 32 * r));
        } else {
#pragma unroll
            for (int r = 0; r < 32; ++r) {
                const float2 p = __ldg(post + lane + 32 * r), e = col[lane + 32 * r];
                col[lane + 32 * r] = make_float2(fmaf(v[r].x, p.x, fmaf(-v[r].y, p.y, e.x)),
                                                 fmaf(v[r].x, p.y, fmaf(v[r].y, p.x, e.y)));
            }
        }
    }
    __syncthreads();
    // transposed read-out: 32-byte row chunks B[n1][col0..col0+3], two lanes per row
#pragma unroll
    for (int i = 0; i < 2 * N / 128; ++i) {
        const int idx = threadIdx.x + 128 * i, n1 = idx >> 1, h = idx & 1;
        const float2 a = sm.col[2 * h][n1], c = sm.col[2 * h + 1][n1];
        *reinterpret_cast<float4 *>(Bv + (size_t)n1 * N + col0 + 2 * h) = make_float4(a.x, a.y, c.x, c.y);
    }
}

// ---- pass x: one row of B per warp ---------------------------------------------------------------
struct SmemXWarp {
    float2 xb[XB];
    float2 keep[N];  // branch-0 result while branch 1 runs
};

// Returns the largest intensity of the row on lane-local terms (reduce across the warp outside).
__device__ __forceinline__ float pass_x_warp(SmemXWarp &sm, const float2 *__restrict__ in,
                                             const float2 *__restrict__ tab,
                                             const float2 *__restrict__ H2, const float2 (&tw)[32],
                                             float2 *__restrict__ field, float *__restrict__ inten) {
    const int lane = threadIdx.x & 31;
    float mx = 0.f;
#pragma unroll 1
    for (int b = 0; b < 2; ++b) {
        const float2 *pre = tab + b * N;
        const float2 *post = tab + 2 * N + b * N;
        float2 v[32];
#pragma unroll
        for (int r = 0; r < 32; ++r) v[r] = cmul(in[lane + 32 * r], __ldg(pre + lane + 32 * r));
        branch(v, lane, sm.xb, tw, H2 + b * N);
        if (b == 0) {
#pragma unroll
            for (int r = 0; r < 32; ++r)
                sm.keep[lane + 32 * r] = cmul(v[r], __ldg(post + lane + 32 * r));
        } else {
#pragma unroll
            for (int r = 0; r < 32; ++r) {
                const int m1 = lane + 32 * r;
                const float2 p = __ldg(post + m1), e = sm.keep[m1];
                const float2 u = make_float2(fmaf(v[r].x, p.x, fmaf(-v[r].y, p.y, e.x)),
                                             fmaf(v[r].x, p.y, fmaf(v[r].y, p.x, e.y)));
                if (field) field[m1] = u;
                const float I = u.x * u.x + u.y * u.y;
                if (inten) inten[m1] = I;
                mx = fmaxf(mx, I);
            }
        }
    }
    return mx;
}

}  // namespace sfdw
