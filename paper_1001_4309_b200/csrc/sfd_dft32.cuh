// sfd_dft32.cuh — the 32-point register butterflies of the warp-per-branch kernels, FMA-formulated.
//
// A 1024-point FFT of a warp (sfd_warp1024.cuh) is two radix-32 stages around one 32 x 32
// transpose.  Both stages are written here as radix-2 decimation-in-time butterflies
//
//     x' = a + w b,     y' = a - w b = 2 a - x'
//
// which cost 6 multiply-add operations per butterfly with a general w (2 + 2 for the two components
// of x', 1 + 1 for y') instead of the 4 multiply/FMA + 4 adds of "multiply, then add and subtract";
// the butterflies with w = 1 and w = -i stay 4 plain adds.  The fp32 pipe of a sub-partition takes
// one warp instruction per cycle whether it is an add or an FMA, and a packed f32x2 instruction
// (sm_100 FADD2 / FFMA2) occupies it for two cycles but costs ONE issue slot - and the issue slot
// is what the partner warp of the sub-partition needs for its shared-memory phase.  So both counts
// matter (measured: a scalar-only version of these butterflies, fewer pipe cycles but more
// instructions than the packed radix-4 butterflies of round 1, was 5 % SLOWER):
//
//                                                          instructions   pipe cycles
//     round 1: dft32 (radix 4 x 4 x 2, packed adds)            310           464
//              + 31 inter-stage twiddle multiplies              124           172
//     dft32      (stage A, constant twiddles)                   292           388
//     dft32_tw   (stage B: the inter-stage twiddles folded      400           480
//                 into the butterfly twiddles)
//
// Sign tracking.  y' = 2a - x' needs a negated operand, which fma.rn.f32x2 does not have; the
// butterflies therefore store Y = x' - 2a = -y' (one FFMA2 with the constant pair (-2, -2)).  Both
// halves of a DIT block carry the same sign pattern (all blocks of a level are processed alike), so
// the operands a and b of every butterfly have EQUAL signs and the formulas hold unchanged on the
// stored values; only the outputs come out as
//
//     stored[k] = s(k) true[k],   s(k) = (-1)^popcount(k)          (k = output index 0..31)
//
// which the consumers absorb at no cost: after stage A the sign depends on k1, which the transpose
// turns into the lane index, so it is folded into the plan-time tables that multiply the result of
// stage B (sfd_plan.cpp, `lane_sign`); after stage B it depends on the register index, a compile-time
// constant that picks the signs of the table multiply (sfdb::out_sign).
//
// Folding of the twiddles: with g = exp(-2 pi i lane / 1024) stage B needs
// Y[k] = sum_r x[r] g^r W32^(r k).  Writing F_n(x; G)[k] = sum_{j<n} x[j] G^j Wn^(j k) the even/odd
// split gives
//     F_n(x; G)[k]       = F_{n/2}(x_even; G^2)[k] + G Wn^k F_{n/2}(x_odd; G^2)[k]
//     F_n(x; G)[k + n/2] = F_{n/2}(x_even; G^2)[k] - G Wn^k F_{n/2}(x_odd; G^2)[k]
// so every butterfly of the size-n level uses T_n[k] = g^(32/n) Wn^k = exp(-2 pi i (lane + 32 k)/(32 n)),
// k < n/2: 16 + 8 + 4 + 2 + 1 = 31 per-lane constants (the same 62 registers the separate twiddle
// multiply needed), built at plan time in extended precision (sfd_plan.cpp).
//
// y' = 2a - x' reuses the rounded x': its error is that of x' plus one rounding, i.e. the same order
// as computing a - w b afresh.
//
// Everything is __host__ __device__ so that the CPU suite can step the butterflies without a GPU
// (sfd_host_dft32 in sfd.h); the product only ever runs them on the GPU.
#pragma once
#include "sfd_fft_core.cuh"

namespace sfdb {

// sign of stored output k of dft32 / dft32_tw relative to the true DFT value
SFD_CE int out_sign(int k) {
    return ((k ^ (k >> 1) ^ (k >> 2) ^ (k >> 3) ^ (k >> 4)) & 1) ? -1 : 1;
}

// packed pairs: (a.x + b.x, a.y + b.y), (a.x - b.x, a.y - b.y), (a.x c.x + d.x, a.y c.y + d.y)
SFD_HD float2 add2(float2 a, float2 b) {
#if defined(__CUDA_ARCH__)
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;"
        : "=l"(r)
        : "l"(*reinterpret_cast<unsigned long long *>(&a)),
          "l"(*reinterpret_cast<unsigned long long *>(&b)));
    return *reinterpret_cast<float2 *>(&r);
#else
    return make_float2(a.x + b.x, a.y + b.y);
#endif
}
SFD_HD float2 sub2(float2 a, float2 b) {
#if defined(__CUDA_ARCH__)
    unsigned long long r;
    asm("sub.rn.f32x2 %0, %1, %2;"
        : "=l"(r)
        : "l"(*reinterpret_cast<unsigned long long *>(&a)),
          "l"(*reinterpret_cast<unsigned long long *>(&b)));
    return *reinterpret_cast<float2 *>(&r);
#else
    return make_float2(a.x - b.x, a.y - b.y);
#endif
}
SFD_HD float2 fma2(float2 a, float2 c, float2 d) {
#if defined(__CUDA_ARCH__)
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;"
        : "=l"(r)
        : "l"(*reinterpret_cast<unsigned long long *>(&a)),
          "l"(*reinterpret_cast<unsigned long long *>(&c)),
          "l"(*reinterpret_cast<unsigned long long *>(&d)));
    return *reinterpret_cast<float2 *>(&r);
#else
    return make_float2(fmaf(a.x, c.x, d.x), fmaf(a.y, c.y, d.y));
#endif
}

// Butterflies on stored values: X = a + w b, Y = X - 2a (= -(a - w b)).
SFD_HD void bf(float2 &a, float2 &b, float c, float s) {  // w = (c, s)
    const float2 x = make_float2(fmaf(c, b.x, fmaf(-s, b.y, a.x)), fmaf(c, b.y, fmaf(s, b.x, a.y)));
    b = fma2(a, make_float2(-2.f, -2.f), x);
    a = x;
}
SFD_HD void bf_one(float2 &a, float2 &b) {  // w = 1
    const float2 x = add2(a, b);
    b = sub2(b, a);
    a = x;
}
SFD_HD void bf_minus_i(float2 &a, float2 &b) {  // w = -i: w b = (b.y, -b.x)
    const float2 x = make_float2(a.x + b.y, a.y - b.x);
    b = make_float2(b.y - a.x, -a.y - b.x);
    a = x;
}

// cos / sin of 2 pi k / 32, 0 <= k < 16
SFD_CE float cos32(int k) {
    constexpr float C[9] = {1.f, 0.98078528040323044913f, 0.92387953251128675613f,
                            0.83146961230254523708f, 0.70710678118654752440f,
                            0.55557023301960222474f, 0.38268343236508977173f,
                            0.19509032201612826785f, 0.f};
    return k <= 8 ? C[k] : -C[16 - k];
}
SFD_CE float sin32(int k) { return k <= 8 ? cos32(8 - k) : cos32(k - 8); }

// In-place radix-2 DIT on registers a[0..31].  The data are kept in bit-reversed *positions*: the
// size-n sub-transform number q (of 32/n) lives in a[q n .. q n + n), its input j being element
// brev(j) of that block after the initial (compile-time, free) renaming done by the callers below.
// level<n>: combine the two size-n/2 halves of every size-n block.
// Twiddle of butterfly k of a size-n block: W32^(k 32/n) = exp(-2 pi i k / n).
template <int n> SFD_HD void level_const(float2 (&a)[32]) {
#pragma unroll
    for (int q = 0; q < 32; q += n)
#pragma unroll
        for (int k = 0; k < n / 2; ++k) {
            const int e = k * (32 / n);  // exponent of W32
            float2 &x = a[q + k], &y = a[q + k + n / 2];
            if (e == 0)
                bf_one(x, y);
            else if (e == 8)
                bf_minus_i(x, y);
            else
                bf(x, y, cos32(e), -sin32(e));
        }
}

// the register renaming that puts natural-order input into DIT (bit-reversed) order
SFD_CE int brev5(int i) {
    return ((i & 1) << 4) | ((i & 2) << 2) | (i & 4) | ((i & 8) >> 2) | ((i & 16) >> 4);
}
SFD_HD void bit_reverse(float2 (&a)[32]) {
#pragma unroll
    for (int i = 0; i < 32; ++i) {
        const int j = brev5(i);
        if (i < j) {
            const float2 t = a[i];
            a[i] = a[j];
            a[j] = t;
        }
    }
}

// 32-point forward DFT (W = exp(-2 pi i / 32)), natural order in and out; stored output k =
// out_sign(k) x the DFT value (sign tracking, see the top of the file).
SFD_HD void dft32(float2 (&a)[32]) {
    bit_reverse(a);
    level_const<2>(a);
    level_const<4>(a);
    level_const<8>(a);
    level_const<16>(a);
    level_const<32>(a);
}

// Twiddles of dft32_tw for one lane: t[n/2 - 1 + k] = T_n[k] = exp(-2 pi i (lane + 32 k) / (32 n)),
// n = 2, 4, 8, 16, 32, k < n/2  (t[0] = T_2[0], t[1..2] = T_4, t[3..6] = T_8, t[7..14] = T_16,
// t[15..30] = T_32).
constexpr int NTW = 31;
template <int n> SFD_HD void level_tw(float2 (&a)[32], const float2 (&t)[NTW]) {
#pragma unroll
    for (int q = 0; q < 32; q += n)
#pragma unroll
        for (int k = 0; k < n / 2; ++k) {
            const float2 w = t[n / 2 - 1 + k];
            bf(a[q + k], a[q + k + n / 2], w.x, w.y);
        }
}
// Y[k] = sum_r a[r] g^r W32^(r k), g = exp(-2 pi i lane / 1024): stage B of the four-step FFT with
// its inter-stage twiddles folded in.  Natural order in and out, stored output k = out_sign(k) Y[k].
SFD_HD void dft32_tw(float2 (&a)[32], const float2 (&t)[NTW]) {
    bit_reverse(a);
    level_tw<2>(a, t);
    level_tw<4>(a, t);
    level_tw<8>(a, t);
    level_tw<16>(a, t);
    level_tw<32>(a, t);
}

}  // namespace sfdb
