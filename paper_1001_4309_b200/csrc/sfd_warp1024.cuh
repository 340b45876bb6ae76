// sfd_warp1024.cuh — the N = 1024 fast path: one warp pair per line, 32 complex values per thread.
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
// transpose, and a warp (32 lanes x 32 values) owns a whole branch: the transpose goes through a
// private shared-memory tile guarded by __syncwarp only; no CTA barrier exists on the FFT path.
// Per line this moves 4 x 16 KiB through shared memory instead of 8 x 32 KiB (generic path) and the
// inter-stage twiddles w1024^(lane * k1) are per-thread constants kept in registers for the whole
// (persistent) kernel.
//
// A line is worked on by a PAIR of warps, one per branch, which meet once per line at a named
// barrier to add their partial results (each warp finishes and stores one half of the line).  With
// 8 warps per SM that is 4 lines in flight per SM: the 4096 lines of a 4-view pass take
// 4096 / (148 x 4) = 6.92 -> 7 rounds, 98.8 % of them filled (one warp per line and 12 warps per SM
// would take 2.3 -> 3 rounds, 77 % filled).  Every table
// stream (pre, H, post) is fetched into a 32-value register vector P one phase ahead of its use,
// and pass x gets its input rows by bulk async copy (TMA) into a double-buffered tile.
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

// Packed fp32 pairs (sm_100 FADD2): one instruction adds/subtracts both components of a complex
// number.  The lane-op rate of the FMA pipe is unchanged, but a complex add costs one issue slot
// instead of two — butterflies are mostly complex adds, so the radix-32 DFT shrinks from 440 to
// about 310 instructions.
__device__ __forceinline__ float2 padd(float2 a, float2 b) {
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;"
        : "=l"(r)
        : "l"(*reinterpret_cast<unsigned long long *>(&a)),
          "l"(*reinterpret_cast<unsigned long long *>(&b)));
    return *reinterpret_cast<float2 *>(&r);
}
__device__ __forceinline__ float2 psub(float2 a, float2 b) {
    unsigned long long r;
    asm("sub.rn.f32x2 %0, %1, %2;"
        : "=l"(r)
        : "l"(*reinterpret_cast<unsigned long long *>(&a)),
          "l"(*reinterpret_cast<unsigned long long *>(&b)));
    return *reinterpret_cast<float2 *>(&r);
}
// a + DIR*i*b and a - DIR*i*b (component swap: scalar adds)
template <int DIR> __device__ __forceinline__ float2 add_ib(float2 a, float2 b) {
    return DIR > 0 ? make_float2(a.x - b.y, a.y + b.x) : make_float2(a.x + b.y, a.y - b.x);
}
template <int DIR> __device__ __forceinline__ void pdft4(float2 &a0, float2 &a1, float2 &a2, float2 &a3) {
    const float2 s0 = padd(a0, a2), d0 = psub(a0, a2), s1 = padd(a1, a3), t = psub(a1, a3);
    a0 = padd(s0, s1);
    a2 = psub(s0, s1);
    a1 = add_ib<DIR>(d0, t);
    a3 = add_ib<-DIR>(d0, t);
}
// 16-point DFT, natural order in and out (same factorisation as sfd::dft16)
template <int DIR> __device__ __forceinline__ void pdft16(float2 (&a)[16]) {
    using sfd::mul_w16;
    pdft4<DIR>(a[0], a[4], a[8], a[12]);
    pdft4<DIR>(a[1], a[5], a[9], a[13]);
    pdft4<DIR>(a[2], a[6], a[10], a[14]);
    pdft4<DIR>(a[3], a[7], a[11], a[15]);
    a[5] = mul_w16<DIR, 1>(a[5]);   a[6] = mul_w16<DIR, 2>(a[6]);   a[7] = mul_w16<DIR, 3>(a[7]);
    a[9] = mul_w16<DIR, 2>(a[9]);   a[10] = mul_w16<DIR, 4>(a[10]); a[11] = mul_w16<DIR, 6>(a[11]);
    a[13] = mul_w16<DIR, 3>(a[13]); a[14] = mul_w16<DIR, 6>(a[14]); a[15] = mul_w16<DIR, 9>(a[15]);
    pdft4<DIR>(a[0], a[1], a[2], a[3]);
    pdft4<DIR>(a[4], a[5], a[6], a[7]);
    pdft4<DIR>(a[8], a[9], a[10], a[11]);
    pdft4<DIR>(a[12], a[13], a[14], a[15]);
    float2 t;
    t = a[1];  a[1] = a[4];   a[4] = t;
    t = a[2];  a[2] = a[8];   a[8] = t;
    t = a[3];  a[3] = a[12];  a[12] = t;
    t = a[6];  a[6] = a[9];   a[9] = t;
    t = a[7];  a[7] = a[13];  a[13] = t;
    t = a[11]; a[11] = a[14]; a[14] = t;
}

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
    pdft16<DIR>(e);
    pdft16<DIR>(o);
#define SFDW_BF(K)                                   \
    {                                                \
        const float2 t = mul_w32<DIR, K>(o[K]);      \
        a[K] = padd(e[K], t);                        \
        a[K + 16] = psub(e[K], t);                   \
    }
    SFDW_BF(0) SFDW_BF(1) SFDW_BF(2) SFDW_BF(3) SFDW_BF(4) SFDW_BF(5) SFDW_BF(6) SFDW_BF(7)
    SFDW_BF(8) SFDW_BF(9) SFDW_BF(10) SFDW_BF(11) SFDW_BF(12) SFDW_BF(13) SFDW_BF(14) SFDW_BF(15)
#undef SFDW_BF
}

// 1024-point forward FFT of one warp.  In: v[r] = x[lane + 32 r].  Out: v[r] = X[lane + 32 r].
// tw[k] = exp(-2 pi i lane k / 1024) (this thread's inter-stage twiddles), xb = the warp's tile.
// The two radix-32 stages share one copy of the butterfly code (rolled loop): the whole line
// transform then fits the instruction cache, which an unrolled version (~140 KB of SASS) does not.
__device__ __forceinline__ void fft1024(float2 (&v)[32], int lane, float2 *xb,
                                        const float2 (&tw)[32]) {
#pragma unroll 1
    for (int stage = 0; stage < 2; ++stage) {
        dft32<-1>(v);  // stage 0: over n1 for n2 = lane -> v[k1]; stage 1: over n2 for k1 = lane
        if (stage == 0) {
#pragma unroll
            for (int k = 1; k < 32; ++k) v[k] = cmul(v[k], tw[k]);
#pragma unroll
            for (int k = 0; k < 32; ++k) xb[k * XS + lane] = v[k];  // (k1 = k, n2 = lane)
            __syncwarp();
            const float4 *row = reinterpret_cast<const float4 *>(xb + lane * XS);  // k1 = lane
#pragma unroll
            for (int q = 0; q < 16; ++q) {
                const float4 t = row[q];
                v[2 * q] = make_float2(t.x, t.y);
                v[2 * q + 1] = make_float2(t.z, t.w);
            }
            __syncwarp();
        }
    }
}

// ---- small PTX helpers ---------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void *p) {
    return (unsigned)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void pair_sync(int pair) {  // named barrier of the two warps of a pair
    asm volatile("bar.sync %0, 64;" ::"r"(pair + 1) : "memory");
}
__device__ __forceinline__ void mbar_init(unsigned long long *bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
// arm `bar` for `bytes` and start a 1-D bulk copy global -> shared that completes on it
__device__ __forceinline__ void bulk_load(void *dst, const void *src, unsigned bytes,
                                          unsigned long long *bar) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
                 "r"(bytes)
                 : "memory");
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
            "r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "W_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra D_%=;\n"
        "bra W_%=;\n"
        "D_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}

__device__ __forceinline__ void load_twiddles(float2 (&tw)[32], int lane,
                                              const float2 *__restrict__ twl) {
#pragma unroll
    for (int k = 0; k < 32; ++k) tw[k] = __ldg(twl + k * 32 + lane);
}
// P <- 32 table values of this thread (element lane + 32 r)
__device__ __forceinline__ void fetch(float2 (&P)[32], const float2 *__restrict__ tab, int lane) {
#pragma unroll
    for (int r = 0; r < 32; ++r) P[r] = __ldg(tab + lane + 32 * r);
}

// One branch of a line, in place (the caller has applied pre): forward FFT, x H_b, inverse FFT.
// The inverse is run as conj(FFT(conj(.))) so that both transforms execute the same code; the
// conjugations are sign flips inside the H multiply and inside the post multiply.
// On entry P holds H_b; on return P holds post_b and v = post_b * (branch result) — this warp's
// partial sums for all 1024 outputs of the line.
__device__ __forceinline__ void branch(float2 (&v)[32], float2 (&P)[32], int lane, float2 *xb,
                                       const float2 (&tw)[32], const float2 *__restrict__ post) {
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {
        fft1024(v, lane, xb, tw);
        if (pass == 0) {
#pragma unroll
            for (int k = 0; k < 32; ++k) {  // v = conj(v * H)
                const float2 h = P[k], a = v[k];
                v[k] = make_float2(a.x * h.x - a.y * h.y, -(a.x * h.y) - a.y * h.x);
            }
            fetch(P, post, lane);  // lands during the second FFT
        }
    }
#pragma unroll
    for (int k = 0; k < 32; ++k) {  // v = post * conj(v)
        const float2 p = P[k], w = v[k];
        v[k] = make_float2(p.x * w.x + p.y * w.y, p.y * w.x - p.x * w.y);
    }
}

// The two warps of a pair hold partial sums v (branch B) for all 32 x 32 outputs of a line.  Warp B
// finishes outputs r in [16 B, 16 B + 16) (element lane + 32 r): it hands the other 16 to its
// partner through xch[1 - B], meets it at the pair's named barrier and adds what it was handed.
// Afterwards v[16 B + q], q < 16, are final.
template <int B>
__device__ __forceinline__ void add_halves(float2 (&v)[32], float2 (*xch)[512], int lane, int pair) {
#pragma unroll
    for (int q = 0; q < 16; ++q) xch[1 - B][q * 32 + lane] = v[16 * (1 - B) + q];
    pair_sync(pair);
#pragma unroll
    for (int q = 0; q < 16; ++q) v[16 * B + q] = padd(v[16 * B + q], xch[B][q * 32 + lane]);
}

// ---- pass y: 4 adjacent hologram columns per CTA, one warp pair per column -----------------------
constexpr int YC = 4;      // columns per CTA
constexpr int CS = N + 4;  // stride (complex) between the CTA's column buffers: puts columns c and
                           // c+2 sixteen banks apart for the transposed read-out
template <typename TIn> struct SmemY {
    float2 xb[2 * YC][XB];
    float2 xch[YC][2][512];
    float2 col[YC][CS];
    // uint8: tile[buf][n0] = the 4 bytes of columns col0..col0+3 of row n0;
    // float: tile[buf][c * N + n0]
    unsigned int tile[2][sizeof(TIn) == 1 ? N : YC * N];
};

template <typename TIn> struct TileRegs {
    unsigned int w[4];   // uint8: 4 rows x 4 packed columns
    float4 f[4];         // float: 4 rows x 4 columns
};

template <typename TIn>
__device__ __forceinline__ void tile_load(TileRegs<TIn> &t, const TIn *__restrict__ holo, int col0) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const size_t row = threadIdx.x + 256 * i;
        if constexpr (sizeof(TIn) == 1)
            t.w[i] = __ldg(reinterpret_cast<const unsigned int *>(holo + row * N + col0));
        else
            t.f[i] = __ldg(reinterpret_cast<const float4 *>(holo + row * N + col0));
    }
}
template <typename TIn>
__device__ __forceinline__ void tile_store(const TileRegs<TIn> &t, unsigned int *tile) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int row = threadIdx.x + 256 * i;
        if constexpr (sizeof(TIn) == 1) {
            tile[row] = t.w[i];
        } else {
            float *f = reinterpret_cast<float *>(tile);
            f[row] = t.f[i].x;
            f[N + row] = t.f[i].y;
            f[2 * N + row] = t.f[i].z;
            f[3 * N + row] = t.f[i].w;
        }
    }
}

// Persistent CTA of 256 threads: work item = (view, group of 4 columns).
// tabY: [V][4][N] = pre b0 | pre b1 | c0 post b0 | c0 post b1;  H2: [V][2][N];  Bout: [V][N][N].
template <typename TIn, int B>
__device__ __forceinline__ void pass_y_loop(SmemY<TIn> &sm, const TIn *__restrict__ holo,
                                            const float2 *__restrict__ tabY,
                                            const float2 *__restrict__ H2,
                                            const float2 (&tw)[32], float2 *__restrict__ Bout, int V) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, c = warp >> 1;
    constexpr int groups = N / YC;
    const int items = V * groups;
    int item = blockIdx.x;
    if (item >= items) return;
    float2 *xb = sm.xb[warp];
    float2 P[32];
    {
        TileRegs<TIn> t;
        tile_load<TIn>(t, holo, (item % groups) * YC);
        fetch(P, tabY + (size_t)(item / groups) * 4 * N + B * N, lane);
        tile_store<TIn>(t, sm.tile[0]);
    }
    __syncthreads();
    int tb = 0;
    for (; item < items; item += gridDim.x) {
        const int view = item / groups, col0 = (item % groups) * YC;
        const int next = item + gridDim.x;
        const bool has_next = next < items;
        TileRegs<TIn> t;
        if (has_next) tile_load<TIn>(t, holo, (next % groups) * YC);
        float2 v[32];
#pragma unroll
        for (int r = 0; r < 32; ++r) {
            const int n0 = lane + 32 * r;
            float a;
            if constexpr (sizeof(TIn) == 1)
                a = (float)((sm.tile[tb][n0] >> (8 * c)) & 0xffu);
            else
                a = reinterpret_cast<const float *>(sm.tile[tb])[c * N + n0];
            v[r] = make_float2(a * P[r].x, a * P[r].y);
        }
        fetch(P, H2 + (size_t)view * 2 * N + B * N, lane);
        branch(v, P, lane, xb, tw, tabY + (size_t)view * 4 * N + 2 * N + B * N);
        if (has_next) fetch(P, tabY + (size_t)(next / groups) * 4 * N + B * N, lane);
        add_halves<B>(v, sm.xch[c], lane, c);
#pragma unroll
        for (int q = 0; q < 16; ++q) sm.col[c][lane + 32 * (16 * B + q)] = v[16 * B + q];
        if (has_next) tile_store<TIn>(t, sm.tile[tb ^ 1]);
        __syncthreads();
        // transposed read-out: 32-byte row chunks B[n1][col0..col0+3], two lanes per row
        float2 *Bv = Bout + (size_t)view * N * N;
#pragma unroll
        for (int i = 0; i < 2 * N / 256; ++i) {
            const int idx = threadIdx.x + 256 * i, n1 = idx >> 1, h = idx & 1;
            const float2 a = sm.col[2 * h][n1], d = sm.col[2 * h + 1][n1];
            *reinterpret_cast<float4 *>(Bv + (size_t)n1 * N + col0 + 2 * h) =
                make_float4(a.x, a.y, d.x, d.y);
        }
        __syncthreads();  // col / xch reusable, next tile visible
        tb ^= 1;
    }
}

// ---- pass x: one row of B per warp pair -----------------------------------------------------------
constexpr int XP = 4;  // pairs per CTA
struct SmemX {
    float2 xb[2 * XP][XB];
    float2 xch[XP][2][2][512];   // [pair][line parity][destination warp][16 x 32]
    float2 inb[XP][2][N];        // [pair][line parity] input row (bulk async copy destination)
    unsigned long long bar[XP][2];
};

// tabX: [V][4][N] = pre b0 | pre b1 | post b0 | post b1;  H2: [V][2][N].
template <int B>
__device__ __forceinline__ void pass_x_loop(SmemX &sm, const float2 *__restrict__ Bin,
                                            const float2 *__restrict__ tabX,
                                            const float2 *__restrict__ H2, const float2 (&tw)[32],
                                            float2 *__restrict__ field, float *__restrict__ inten,
                                            unsigned int *vmax, int V) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, pair = warp >> 1;
    const int lines = V * N, G = gridDim.x * XP;
    int line = blockIdx.x * XP + pair;
    if (line >= lines) return;
    float2 *xb = sm.xb[warp];
    const bool issuer = B == 0 && lane == 0;
    if (issuer) bulk_load(sm.inb[pair][0], Bin + (size_t)line * N, N * sizeof(float2), &sm.bar[pair][0]);
    float2 P[32];
    fetch(P, tabX + (size_t)(line / N) * 4 * N + B * N, lane);
    for (int it = 0; line < lines; line += G, ++it) {
        const int buf = it & 1, view = line / N, next = line + G;
        const bool has_next = next < lines;
        if (has_next && issuer)
            bulk_load(sm.inb[pair][buf ^ 1], Bin + (size_t)next * N, N * sizeof(float2),
                      &sm.bar[pair][buf ^ 1]);
        mbar_wait(&sm.bar[pair][buf], (it >> 1) & 1);
        float2 v[32];
#pragma unroll
        for (int r = 0; r < 32; ++r) v[r] = cmul(sm.inb[pair][buf][lane + 32 * r], P[r]);
        fetch(P, H2 + (size_t)view * 2 * N + B * N, lane);
        branch(v, P, lane, xb, tw, tabX + (size_t)view * 4 * N + 2 * N + B * N);
        if (has_next) fetch(P, tabX + (size_t)(next / N) * 4 * N + B * N, lane);
        add_halves<B>(v, sm.xch[pair][buf], lane, pair);
        float mx = 0.f;
        const size_t off = (size_t)line * N;
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const int m1 = lane + 32 * (16 * B + q);
            const float2 u = v[16 * B + q];
            if (field) field[off + m1] = u;
            const float I = u.x * u.x + u.y * u.y;
            if (inten) inten[off + m1] = I;
            mx = fmaxf(mx, I);
        }
        if (vmax != nullptr) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
            // intensities are >= 0, so their float bit patterns order like unsigned integers
            if (lane == 0) atomicMax(vmax + view, __float_as_uint(mx));
        }
    }
}

}  // namespace sfdw
