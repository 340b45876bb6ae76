// sfd_fft_core.cuh — per-thread building blocks of the fused chirp-z (Bluestein) line transform.
//
// One "line" is one 1-D scaled DFT of PAPER.md Eq.(1) L50-54 along x or along y:
//
//     out[j] = post[j] * sum_{m<N} in[m] pre[m] h[j-m],   j in [0,N),   h[d] = exp(i pi S d^2) (Eq. 4)
//
// computed as the paper computes it (steps (ii)-(ix), L86-93): zero-pad to M = 2N, forward FFT,
// multiply by the cached spectrum H = FFT_M(h)/M, inverse FFT, keep the first N samples.
//
// A line is worked on by T = M/16 threads; thread j keeps 16 complex values in registers, register
// slot s always standing for element j + s*T of the current array ("slot invariant").  The FFT is a
// Stockham autosort FFT of 2 or 3 passes (radix 16 / 8 / 4 register butterflies); between passes
// the line is exchanged through shared memory (scatter in Stockham order, gather by the slot
// invariant).  The last pass of the forward FFT leaves natural order in exactly the slots the first
// pass of the inverse FFT reads, so the spectrum multiply and the turn-around need no exchange.
// The zero half of the padded input (slots 8..15 of the first pass) and the discarded half of the
// output (slots 8..15 of the last pass) are never loaded / stored, and their arithmetic is pruned.
//
// Everything here is __host__ __device__ so the same code can be stepped on a CPU for debugging;
// the product only ever runs it on the GPU.
#pragma once
#include <cuda_runtime.h>

#if defined(__CUDACC__)
#define SFD_HD __host__ __device__ __forceinline__
#define SFD_CE __host__ __device__ static constexpr
#else
#define SFD_HD inline
#define SFD_CE static constexpr
#endif

#if defined(__CUDA_ARCH__)
#define SFD_LDG(p) __ldg(p)
#else
#define SFD_LDG(p) (*(p))
#endif

namespace sfd {

// Plan constants (FFT twiddles, pre / H / post tables) of the Fresnel line code: for padded lengths up to
// M = 1024 the generic kernels hand in shared-memory copies (sfd_kernels.cu, Staged), read with plain
// loads; otherwise they are global pointers read through the non-coherent path.
SFD_CE bool tables_staged(int log2m) { return log2m <= 10; }
template <bool SM> SFD_HD float2 tab_ld(const float2 *p) {
    if constexpr (SM)
        return *p;
    else
        return SFD_LDG(p);
}

SFD_HD float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
SFD_HD float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
SFD_HD float2 cmul(float2 a, float2 b) {
    return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
// a * (DIR * i)
template <int DIR> SFD_HD float2 mul_di(float2 a) {
    return DIR > 0 ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
}
// a * exp(DIR * 2 pi i * E / 16), E a compile-time exponent
template <int DIR, int E> SFD_HD float2 mul_w16(float2 a) {
    constexpr int e = ((E % 16) + 16) % 16;
    constexpr float C1 = 0.92387953251128675613f;  // cos(pi/8)
    constexpr float S1 = 0.38268343236508977173f;  // sin(pi/8)
    constexpr float H = 0.70710678118654752440f;   // cos(pi/4)
    if (e == 0) return a;
    if (e == 4) return mul_di<DIR>(a);
    if (e == 8) return make_float2(-a.x, -a.y);
    if (e == 12) return mul_di<-DIR>(a);
    if (e == 2) return make_float2(H * (a.x - DIR * a.y), H * (a.y + DIR * a.x));
    if (e == 6) return make_float2(H * (-a.x - DIR * a.y), H * (DIR * a.x - a.y));
    if (e == 10) return make_float2(H * (DIR * a.y - a.x), H * (-a.y - DIR * a.x));
    if (e == 14) return make_float2(H * (a.x + DIR * a.y), H * (a.y - DIR * a.x));
    // odd exponents: generic constant multiply, w = (c, DIR*s)
    constexpr float c = (e == 1 || e == 15) ? C1 : (e == 3 || e == 13) ? S1
                       : (e == 5 || e == 11) ? -S1 : -C1;  // 7, 9
    constexpr float s0 = (e == 1 || e == 7) ? S1 : (e == 3 || e == 5) ? C1
                        : (e == 9 || e == 15) ? -S1 : -C1;  // 11, 13
    constexpr float s = DIR * s0;
    return make_float2(a.x * c - a.y * s, a.x * s + a.y * c);
}

// ---- in-register DFTs, natural order in and out, W = exp(DIR * 2 pi i / r) -------------------
SFD_HD void dft2(float2 &a0, float2 &a1) {
    float2 t = a0;
    a0 = cadd(t, a1);
    a1 = csub(t, a1);
}
template <int DIR> SFD_HD void dft4(float2 &a0, float2 &a1, float2 &a2, float2 &a3) {
    float2 s0 = cadd(a0, a2), d0 = csub(a0, a2);
    float2 s1 = cadd(a1, a3), d1 = mul_di<DIR>(csub(a1, a3));
    a0 = cadd(s0, s1);
    a2 = csub(s0, s1);
    a1 = cadd(d0, d1);
    a3 = csub(d0, d1);
}
// DFT4 whose inputs 2 and 3 are zero
template <int DIR> SFD_HD void dft4_half(float2 &a0, float2 &a1, float2 &a2, float2 &a3) {
    float2 x0 = a0, x1 = a1, ix1 = mul_di<DIR>(a1);
    a0 = cadd(x0, x1);
    a1 = cadd(x0, ix1);
    a2 = csub(x0, x1);
    a3 = csub(x0, ix1);
}
template <int DIR> SFD_HD void dft8(float2 (&a)[8]) {
    // n = p + 2b: two DFT4 over b, twiddle W8^(p*kb), DFT2 over p; output k = kb + 4 kp
    dft4<DIR>(a[0], a[2], a[4], a[6]);
    dft4<DIR>(a[1], a[3], a[5], a[7]);
    float2 y0 = a[1], y1 = mul_w16<DIR, 2>(a[3]), y2 = mul_w16<DIR, 4>(a[5]),
           y3 = mul_w16<DIR, 6>(a[7]);
    float2 e0 = a[0], e1 = a[2], e2 = a[4], e3 = a[6];
    a[0] = cadd(e0, y0); a[4] = csub(e0, y0);
    a[1] = cadd(e1, y1); a[5] = csub(e1, y1);
    a[2] = cadd(e2, y2); a[6] = csub(e2, y2);
    a[3] = cadd(e3, y3); a[7] = csub(e3, y3);
}
// HALF: inputs 8..15 are zero (the zero-padded half of the line in the first forward pass)
template <int DIR, bool HALF> SFD_HD void dft16(float2 (&a)[16]) {
    // n = p + 4b: four DFT4 over b (Y_p[kb]), twiddle W16^(p*kb), four DFT4 over p; k = kb + 4 kp
    if (HALF) {
        dft4_half<DIR>(a[0], a[4], a[8], a[12]);
        dft4_half<DIR>(a[1], a[5], a[9], a[13]);
        dft4_half<DIR>(a[2], a[6], a[10], a[14]);
        dft4_half<DIR>(a[3], a[7], a[11], a[15]);
    } else {
        dft4<DIR>(a[0], a[4], a[8], a[12]);
        dft4<DIR>(a[1], a[5], a[9], a[13]);
        dft4<DIR>(a[2], a[6], a[10], a[14]);
        dft4<DIR>(a[3], a[7], a[11], a[15]);
    }
    // now a[p + 4 kb] = Y_p[kb]
    a[5] = mul_w16<DIR, 1>(a[5]);   a[6] = mul_w16<DIR, 2>(a[6]);   a[7] = mul_w16<DIR, 3>(a[7]);
    a[9] = mul_w16<DIR, 2>(a[9]);   a[10] = mul_w16<DIR, 4>(a[10]); a[11] = mul_w16<DIR, 6>(a[11]);
    a[13] = mul_w16<DIR, 3>(a[13]); a[14] = mul_w16<DIR, 6>(a[14]); a[15] = mul_w16<DIR, 9>(a[15]);
    // DFT4 over p for each kb; results X[kb + 4 kp] land in a[4 kb + kp] -> transpose afterwards
    dft4<DIR>(a[0], a[1], a[2], a[3]);
    dft4<DIR>(a[4], a[5], a[6], a[7]);
    dft4<DIR>(a[8], a[9], a[10], a[11]);
    dft4<DIR>(a[12], a[13], a[14], a[15]);
    float2 t;
    t = a[1];  a[1] = a[4];   a[4] = t;
    t = a[2];  a[2] = a[8];   a[8] = t;
    t = a[3];  a[3] = a[12];  a[12] = t;
    t = a[6];  a[6] = a[9];   a[9] = t;
    t = a[7];  a[7] = a[13];  a[13] = t;
    t = a[11]; a[11] = a[14]; a[14] = t;
}

// ---- pass schedule ---------------------------------------------------------------------------
template <int LOG2M> struct Sched {
    static_assert(LOG2M >= 7 && LOG2M <= 12, "padded length must be 128..4096");
    static constexpr int M = 1 << LOG2M;
    static constexpr int N = M / 2;   // un-padded line length
    static constexpr int T = M / 16;  // threads per line
    static constexpr int NP = LOG2M <= 8 ? 2 : 3;
    SFD_CE int radix(int p) {
        return LOG2M == 7    ? (p == 0 ? 16 : 8)
               : LOG2M == 8  ? 16
               : LOG2M == 9  ? (p == 0 ? 16 : p == 1 ? 8 : 4)
               : LOG2M == 10 ? (p < 2 ? 16 : 4)
               : LOG2M == 11 ? (p < 2 ? 16 : 8)
                             : 16;
    }
    SFD_CE int ns(int p) { return p == 0 ? 1 : ns(p - 1) * radix(p - 1); }
    static constexpr int PADDED = M + M / 16;  // shared-memory elements per line (1 pad per 16)
};

// CTA shapes of the generic kernels: columns per CTA in a column pass / rows per CTA in a row pass,
// by transform length M = 2^LOG2M
template <int LOG2M> struct Tile {
    static constexpr int T = Sched<LOG2M>::T;
    static constexpr int C = LOG2M <= 7 ? 16 : LOG2M <= 9 ? 8 : LOG2M <= 11 ? 4 : 2;
    static constexpr int RPC = T >= 128 ? 1 : 128 / T;
    static constexpr int THREADS_Y = C * T;
    static constexpr int THREADS_X = RPC * T;
    static constexpr size_t SMEM_Y = sizeof(float2) * Sched<LOG2M>::PADDED * C;
    static constexpr size_t SMEM_X = sizeof(float2) * Sched<LOG2M>::PADDED * RPC;
};

// Shared-memory view of one line: element pos of the line lives at base[(pos + pos/16) * ISTR].
template <int ISTR> struct LineSmem {
    float2 *base;
    SFD_HD float2 &at(int pos) const { return base[(pos + (pos >> 4)) * ISTR]; }
};

// Twiddle (pass P >= 1) and butterfly of pass P on the register slots.  tw[x] = exp(-2 pi i x/M).
template <int LOG2M, int P, int DIR, bool HALF_IN, bool SMTW = false>
SFD_HD void pass_compute(float2 (&v)[16], int j, const float2 *__restrict__ tw) {
    using S = Sched<LOG2M>;
    constexpr int R = S::radix(P), Q = 16 / R, NS = S::ns(P), STEP = S::M / (NS * R);
#pragma unroll
    for (int q = 0; q < Q; ++q) {
        float2 a[R];
        const int k = (j + q * S::T) & (NS - 1);
#pragma unroll
        for (int t = 0; t < R; ++t) a[t] = v[q + t * Q];
        if (P > 0) {
#pragma unroll
            for (int t = 1; t < R; ++t) {
                float2 w = tab_ld<SMTW>(tw + k * t * STEP);
                if (DIR > 0) w.y = -w.y;
                a[t] = cmul(a[t], w);
            }
        }
        if constexpr (R == 16) dft16<DIR, HALF_IN>(a);
        else if constexpr (R == 8) dft8<DIR>(a);
        else if constexpr (R == 4) dft4<DIR>(a[0], a[1], a[2], a[3]);
        else dft2(a[0], a[1]);
#pragma unroll
        for (int t = 0; t < R; ++t) v[q + t * Q] = a[t];
    }
}

// Stockham scatter of the outputs of pass P (P < NP-1) into shared memory.
template <int LOG2M, int P, int ISTR>
SFD_HD void scatter(const float2 (&v)[16], int j, LineSmem<ISTR> sm) {
    using S = Sched<LOG2M>;
    constexpr int R = S::radix(P), Q = 16 / R, NS = S::ns(P);
#pragma unroll
    for (int q = 0; q < Q; ++q) {
        const int jq = j + q * S::T, k = jq & (NS - 1);
        const int j0 = (jq - k) * R + k;
#pragma unroll
        for (int t = 0; t < R; ++t) sm.at(j0 + t * NS) = v[q + t * Q];
    }
}
template <int LOG2M, int ISTR> SFD_HD void gather(float2 (&v)[16], int j, LineSmem<ISTR> sm) {
#pragma unroll
    for (int s = 0; s < 16; ++s) v[s] = sm.at(j + s * Sched<LOG2M>::T);
}

// One whole FFT of direction DIR on the slots (all passes; SYNC() is a barrier over every thread
// that shares this shared-memory buffer).
template <int LOG2M, int DIR, bool HALF_IN, int ISTR, class SyncF, bool SMTW = false>
SFD_HD void fft_line(float2 (&v)[16], int j, LineSmem<ISTR> sm, const float2 *__restrict__ tw,
                     SyncF sync) {
    using S = Sched<LOG2M>;
    pass_compute<LOG2M, 0, DIR, HALF_IN, SMTW>(v, j, tw);
    scatter<LOG2M, 0, ISTR>(v, j, sm);
    sync();
    gather<LOG2M, ISTR>(v, j, sm);
    sync();
    pass_compute<LOG2M, 1, DIR, false, SMTW>(v, j, tw);
    if constexpr (S::NP == 3) {
        scatter<LOG2M, 1, ISTR>(v, j, sm);
        sync();
        gather<LOG2M, ISTR>(v, j, sm);
        sync();
        pass_compute<LOG2M, 2, DIR, false, SMTW>(v, j, tw);
    }
}

// The fused line transform on values already pre-multiplied: forward FFT (zero half pruned),
// multiply by H (which carries the 1/M of the inverse), inverse FFT.  On return slots 0..7 hold
// samples j + s*T (< N) of the linear convolution; slots 8..15 are the discarded half.
template <int LOG2M, int ISTR, class SyncF>
SFD_HD void chirpz_line(float2 (&v)[16], int j, LineSmem<ISTR> sm, const float2 *__restrict__ tw,
                        const float2 *__restrict__ H, SyncF sync) {
    using S = Sched<LOG2M>;
#pragma unroll
    for (int s = 8; s < 16; ++s) v[s] = make_float2(0.f, 0.f);
    constexpr bool SM = tables_staged(LOG2M);
    fft_line<LOG2M, -1, true, ISTR, SyncF, SM>(v, j, sm, tw, sync);
#pragma unroll
    for (int s = 0; s < 16; ++s) v[s] = cmul(v[s], tab_ld<SM>(H + j + s * S::T));
    fft_line<LOG2M, +1, false, ISTR, SyncF, SM>(v, j, sm, tw, sync);
}

// ---- the two passes of a reconstruction --------------------------------------------------------
// The grid is Ny rows by Nx columns; tables and B are already offset to the CTA's view.
// Pass y (steps (ii)-(ix) along y): a CTA takes C adjacent hologram columns of one view; thread
// (l, j), l fastest, works on column col0 + l; the line length is Ny = Sched<LOG2M>::N.
// in = hologram sample (real) * pre_y[n0] (Eq. 3, the 1/255 of uint8 input folded into the table),
// out * post_y[n1] (Eq. 2 y-part, times c0) is written to the row-major intermediate B[n1][m0]
// (nx columns) in 8C-byte chunks.  hstride = elements between hologram rows.
// The hologram and B are produced by whatever ran before in the stream (a copy, pass y): they are
// read with plain loads, not through the non-coherent path.
template <int LOG2M, int C, typename TIn, class SyncF>
SFD_HD void pass_y_body(int tid, int tile, float2 *smem, const TIn *holo, long long hstride, int nx,
                        const float2 *__restrict__ pre_y, const float2 *__restrict__ Hy,
                        const float2 *__restrict__ post_y, const float2 *__restrict__ tw,
                        float2 *B, SyncF sync) {
    using S = Sched<LOG2M>;
    constexpr int T = S::T;
    const int l = tid % C, j = tid / C;
    const int col = tile * C + l;
    float2 v[16];
#pragma unroll
    for (int s = 0; s < 8; ++s) {
        const int n0 = j + s * T;
        const float a = (float)holo[(size_t)n0 * hstride + col];
        const float2 p = tab_ld<tables_staged(LOG2M)>(pre_y + n0);
        v[s] = make_float2(a * p.x, a * p.y);
    }
    LineSmem<C> sm{smem + l};
    chirpz_line<LOG2M, C>(v, j, sm, tw, Hy, sync);
#pragma unroll
    for (int s = 0; s < 8; ++s) {
        const int n1 = j + s * T;
        B[(size_t)n1 * nx + col] = cmul(v[s], tab_ld<tables_staged(LOG2M)>(post_y + n1));
    }
}

// Pass x (steps (ii)-(x) along x): a CTA takes RPC adjacent rows of one view; thread (l, j), j
// fastest, works on row tile * RPC + l of the view; the line length is Nx = Sched<LOG2M>::N.
// in = B[n1][m0] * pre_x[m0], out * post_x[m1] is the field u1[n1][m1]; intensity = |u1|^2 (Eq. 5).
// B, field, inten are offset to the view.  Returns the largest intensity this thread produced.
template <int LOG2M, int RPC, bool MOM, class SyncF>
SFD_HD float pass_x_body(int tid, int tile, float2 *smem, const float2 *B,
                         const float2 *__restrict__ pre_x, const float2 *__restrict__ Hx,
                         const float2 *__restrict__ post_x, const float2 *__restrict__ tw,
                         float2 *__restrict__ field, float *__restrict__ inten, SyncF sync,
                         float &s1, float &s2) {
    using S = Sched<LOG2M>;
    constexpr int N = S::N, T = S::T;
    const int l = tid / T, j = tid % T;
    const size_t row = (size_t)tile * RPC + l;
    const float2 *in = B + row * N;
    float2 v[16];
#pragma unroll
    for (int s = 0; s < 8; ++s) {
        const int m0 = j + s * T;
        v[s] = cmul(in[m0], tab_ld<tables_staged(LOG2M)>(pre_x + m0));
    }
    LineSmem<1> sm{smem + l * S::PADDED};
    chirpz_line<LOG2M, 1>(v, j, sm, tw, Hx, sync);
    float mx = 0.f;
#pragma unroll
    for (int s = 0; s < 8; ++s) {
        const int m1 = j + s * T;
        const float2 u = cmul(v[s], tab_ld<tables_staged(LOG2M)>(post_x + m1));
        if (field) field[row * N + m1] = u;
        const float I = u.x * u.x + u.y * u.y;
        if (inten) inten[row * N + m1] = I;
        mx = I > mx ? I : mx;
        if (MOM) {      // this thread's share of sum I and sum I^2 (focus moments, row f2)
            s1 += I;
            s2 += I * I;
        }
    }
    return mx;
}

}  // namespace sfd
