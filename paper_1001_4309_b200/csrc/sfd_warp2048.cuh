// sfd_warp2048.cuh — the N = 2048 kernels: the warp-per-branch scheme of sfd_warp1024.cuh with four
// branches per line.
//
// The padded transform of a 2048-point line has length L = 4096.  Splitting its DFT by the
// frequency index modulo 4 (one radix-4 step with the zero half skipped on the way in and the
// discarded half skipped on the way out, w = exp(-2 pi i / L)) gives four independent branches
// b = 0..3 of 1024-point transforms (n' < 1024):
//
//     forward:  X[4k+b] = FFT_1024(y_b)[k],   y_b[n'] = x[n'] w^(b n') + x[n'+1024] w^(b (n'+1024))
//     inverse:  y[n]    = sum_b w^(-b n) g_b[n mod 1024],   g_b = IFFT_1024(H[4k+b] X[4k+b]) 1024
//
// so with the plan-time tables (x = in pre, out = post y)
//     preA_b = pre[n'] w^(b n'),  preB_b = pre[n'+1024] w^(b (n'+1024)),  H_b[k] = H[4k+b],
//     postA_b = post[n'] w^(-b n'),  postB_b = post[n'+1024] w^(-b (n'+1024))
// a line is   out[n'] = sum_b postA_b g_b,  out[n'+1024] = sum_b postB_b g_b,
//             g_b = IFFT(H_b FFT(in[n'] preA_b + in[n'+1024] preB_b)).
// A warp owns a branch exactly as in the N = 1024 kernels (same `branch()`, same transpose tile,
// same twiddles); four warps (a quad) work on a line, a CTA of 8 warps on two lines.  Warp b of a
// quad finishes output quarter b (n in [512 b, 512 b + 512)): the other three quarters of its
// partial sums go to the exchange area, one quad barrier later it adds what the others left for it.
// The five tables of a branch sit in the tensor-memory quarter of its sub-partition (320 columns,
// one view: a CTA works inside one view, the launcher gives every view floor(SMs / V) CTAs).
#pragma once
#include "sfd_warp1024.cuh"

namespace sfdq {

using namespace sfdw;  // N = 1024 is the branch length here

constexpr int NL = 2048;            // line length
constexpr int NBR = 4;              // branches per line
constexpr int QTABS = NBR * 5 * N;  // complex elements of one view's tables of one pass: [4][5][N]
// tensor-memory columns of the five tables of a branch
constexpr int TQ_PREA = 0, TQ_PREB = 64, TQ_H = 128, TQ_POSTA = 192, TQ_POSTB = 256, TQ_TW = 320;
// work units per view: pass x 2 rows (ny / 2 units), pass y 4 columns, 2 per quad (nx / 4 units)

__device__ __forceinline__ void quad_sync(int quad) {  // named barrier of the four warps of a quad
    asm volatile("bar.sync %0, 128;" ::"r"(quad + 1) : "memory");
}
__device__ __forceinline__ void cta_sync() { asm volatile("bar.sync 0;" ::: "memory"); }

// The two warps of a sub-partition copy the 20 chunks (5 tables x 4 chunks of 8 values) of
// `view`, branch warp & 3, into their quarter: warp w chunks 0..9, warp w + 4 chunks 10..19, five
// chunks (40 loads per thread) in flight at a time.  tab: the [4][5][N] block of view 0 in global
// memory, vstride complex values between views.
__device__ __forceinline__ void tmq_fill(unsigned quarter, const float2 *__restrict__ tab,
                                         long long vstride, int view, int warp, int lane) {
    const float2 *src = tab + (size_t)view * vstride + (size_t)(warp & 3) * 5 * N + lane;
#pragma unroll 1
    for (int h = 0; h < 2; ++h) {
        const int ch0 = 10 * (warp >> 2) + 5 * h;
        TChunk c[5];
#pragma unroll
        for (int j = 0; j < 5; ++j)
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const float2 x = __ldg(src + 32 * (8 * (ch0 + j) + i));
                c[j].w[2 * i] = __float_as_uint(x.x);
                c[j].w[2 * i + 1] = __float_as_uint(x.y);
            }
#pragma unroll
        for (int j = 0; j < 5; ++j) tm_st(c[j], quarter + 16 * (ch0 + j));
    }
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ unsigned tmq_setup(unsigned *slot, const float2 *__restrict__ tab,
                                              long long vstride, int view, const float2 *__restrict__ twl) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (warp == 0) tm_alloc(slot);
    tm_sync_cta();
    const unsigned base = *reinterpret_cast<volatile unsigned *>(slot);
    tmq_fill(tm_quarter(base, warp), tab, vstride, view, warp, lane);
    if (warp < 4) tm_fill_twiddles(tm_quarter(base, warp) + TQ_TW, twl, lane);
    tm_sync_cta();
    return base;
}

// A CTA takes a contiguous range [a0, a1) of the V * units work units of a launch.  The five tables
// of a branch fill 320 of the 512 tensor-memory columns, so only one view's tables are resident: a
// range that crosses into the next view (at most once: the grid has at least V CTAs) is walked as
// two segments with the tables reloaded in between (segment() is CTA-uniform).
struct Range { int view, u0, u1; };
struct Span {
    int a0, a1, units;
    __device__ int first_view() const { return a0 < a1 ? a0 / units : 0; }
    __device__ Range segment(int s) const {  // s = 0, 1; empty if u0 >= u1
        const int view = first_view() + s, lo = view * units, hi = lo + units;
        return Range{view, (a0 > lo ? a0 : lo) - lo, (a1 < hi ? a1 : hi) - lo};
    }
};
__device__ __forceinline__ Span cta_span(int V, int units) {
    const long long total = (long long)V * units;
    return Span{(int)(total * blockIdx.x / gridDim.x), (int)(total * (blockIdx.x + 1) / gridDim.x), units};
}
// all warps have finished with the resident tables: load those of `view`
__device__ __forceinline__ void tmq_refill(unsigned base, const float2 *__restrict__ tab,
                                           long long vstride, int view) {
    tm_sync_cta();
    tmq_fill(tm_quarter(base, threadIdx.x >> 5), tab, vstride, view, threadIdx.x >> 5, threadIdx.x & 31);
    tm_sync_cta();
}

// Exchange area of a warp: three quarters of 16 x 32 values for the other three warps of the quad
// (slot = target quarter with the source's own skipped).  Slots 0 and 1 live in the warp's transpose
// tile, which is idle between two branch() calls, slot 2 in ex.v[warp].
struct Exch { float2 v[8][16 * 32]; };
__device__ __forceinline__ float2 *exch_slot(float2 (*xb)[XB], Exch &ex, int warp, int slot) {
    return slot < 2 ? xb[warp] + slot * (16 * 32) : ex.v[warp];
}

// g = this warp's branch result for n' = lane + 32 r.  Multiplies it by postA_b / postB_b, keeps
// output quarter b in `mine` (final after quad_collect) and leaves the other three quarters in
// the exchange area.  Output quarter oq covers n = lane + 32 (16 oq + i): oq < 2 uses postA and
// g[16 oq + i], oq >= 2 uses postB and g[16 (oq - 2) + i].
__device__ __forceinline__ void quad_scatter(const float2 (&g)[32], float2 (&mine)[16], unsigned tq,
                                             int b, int lane, float2 (*xb)[XB], Exch &ex, int warp) {
    TChunk c0, c1;
    tm_ld(c0, tq + TQ_POSTA);
#pragma unroll
    for (int oq = 0; oq < 4; ++oq) {
        const unsigned tab = tq + (oq < 2 ? TQ_POSTA : TQ_POSTB) + 32 * (oq & 1);
        float2 *dst = exch_slot(xb, ex, warp, oq < b ? oq : oq > 0 ? oq - 1 : 0) + lane;
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            TChunk &c = j ? c1 : c0;
            tm_wait(c);
            if (j == 0)
                tm_ld(c1, tab + 16);
            else if (oq < 3)
                tm_ld(c0, tq + (oq + 1 < 2 ? TQ_POSTA : TQ_POSTB) + 32 * ((oq + 1) & 1));
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const float2 w = cmul(g[16 * (oq & 1) + 8 * j + i], tm_val(c, i));
                if (oq == b)
                    mine[8 * j + i] = w;
                else
                    dst[(8 * j + i) * 32] = w;
            }
        }
    }
}
// after the quad barrier: add what the other three warps of the quad left for quarter b
__device__ __forceinline__ void quad_collect(float2 (&mine)[16], int b, int lane, float2 (*xb)[XB],
                                             Exch &ex, int warp) {
#pragma unroll
    for (int d = 1; d < 4; ++d) {
        const int bo = (b + d) & 3;  // the other branch
        const float2 *src = exch_slot(xb, ex, (warp & 4) | bo, b < bo ? b : b - 1) + lane;
#pragma unroll
        for (int i = 0; i < 16; ++i) mine[i] = padd(mine[i], src[i * 32]);
    }
}

// ---- pass x: two rows of B per CTA ------------------------------------------------------------------
struct SmemXQ {
    float2 xb[8][XB];
    Exch ex;
    float2 inb[2][NL];  // input row of each quad (bulk async copy destination)
    unsigned long long ibar[2];
    unsigned tmem;
};

__device__ __forceinline__ void pass_x_quad(SmemXQ &sm, const float2 *Bin, int ny, unsigned tq,
                                            unsigned tt, float2 *__restrict__ field,
                                            float *__restrict__ inten, unsigned int *vmax,
                                            double *mom, Range rg, unsigned &iphase) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, quad = warp >> 2, b = warp & 3;
    float2 *xb = sm.xb[warp];
    const float2 *in = sm.inb[quad] + lane;
    const bool issuer = b == 0 && lane == 0;
    bool pending = false;  // (iphase: parity of the quad's input barrier, carried across segments)
    const Turns turns = turns_make(warp, 8, 5, true);  // named barriers 5..12
    turns_open(turns, warp, 8);
    for (int u = rg.u0; u < rg.u1; ++u) {
        const size_t row = (size_t)rg.view * ny + 2 * u + quad;
        if (!pending && issuer)
            bulk_load(sm.inb[quad], Bin + row * NL, NL * sizeof(float2), &sm.ibar[quad]);
        const bool has_next = u + 1 < rg.u1;
        mbar_wait(&sm.ibar[quad], iphase);
        iphase ^= 1;
        float2 v[32];
        {   // v = in[n'] preA_b + in[n' + 1024] preB_b
            TChunk ca, cb;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                tm_ld(ca, tq + TQ_PREA + 16 * j);
                tm_ld(cb, tq + TQ_PREB + 16 * j);
                tm_wait(ca);
                tm_wait(cb);
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const int r = 8 * j + i;
                    v[r] = padd(cmul(in[32 * r], tm_val(ca, i)), cmul(in[32 * r + N], tm_val(cb, i)));
                }
            }
        }
        // all four warps have consumed the row and read the previous line's exchange area
        quad_sync(quad);
        if (has_next && issuer) {
            fence_async_smem();
            bulk_load(sm.inb[quad], Bin + (row + 2) * NL, NL * sizeof(float2), &sm.ibar[quad]);
        }
        pending = has_next;
        branch<false>(v, lane, xb, tt, tq + TQ_H, turns);
        float2 mine[16];
        quad_scatter(v, mine, tq, b, lane, sm.xb, sm.ex, warp);
        quad_sync(quad);
        quad_collect(mine, b, lane, sm.xb, sm.ex, warp);
        float mx = 0.f, s1 = 0.f, s2 = 0.f;
        const size_t off = row * NL;
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const int m1 = lane + 32 * (16 * b + i);
            const float2 w = mine[i];
            if (field) field[off + m1] = w;
            const float I = w.x * w.x + w.y * w.y;
            if (inten) inten[off + m1] = I;
            mx = fmaxf(mx, I);
            if (mom != nullptr) {
                s1 += I;
                s2 = fmaf(I, I, s2);
            }
        }
        if (mom != nullptr) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                s1 += __shfl_xor_sync(0xffffffffu, s1, o);
                s2 += __shfl_xor_sync(0xffffffffu, s2, o);
            }
            if (lane == 0) {
                atomicAdd(mom + 2 * rg.view, (double)s1);
                atomicAdd(mom + 2 * rg.view + 1, (double)s2);
            }
        }
        if (vmax != nullptr) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
            if (lane == 0) atomicMax(vmax + rg.view, __float_as_uint(mx));
        }
    }
    turns_close(turns, warp);
}

// ---- pass y: four adjacent hologram columns per CTA, two per quad -------------------------------------
// Work unit u of a view = columns 4 u .. 4 u + 3; quad q transforms columns 4 u + 2 q and
// 4 u + 2 q + 1 one after the other.  The final sums of all four columns meet in one staging tile
// [n1][4] that one thread hands to the TMA unit: 32 bytes = one full sector per row of B.  (With
// 16-byte rows B, which at this size does not fit L2, cost 1.2 GB of DRAM traffic per launch for
// 0.5 GB of payload: half-written sectors are read back and merged.)
// Hologram samples reach shared memory as slabs, kept as [quad][k][n'][h] column pairs with rows n' and
// n' + 1024 side by side (one read gives both samples a thread folds together):
//   float  each quad fetches its own 2 columns of one unit, 8 bytes per row (sub_load / sub_store);
//   uint8  the CTA fetches the 16 columns of FOUR units, 16 bytes per row, once (slab16_*): a row of
//          the hologram is one shared-memory wavefront per load instruction however few of its bytes
//          are wanted, and the two quads want the same rows - per-quad slabs of 8 columns cost four
//          times the wavefronts per unit (measured: the slab tail was 15 % of a line's period).
//          The tile is handed over with two mbarriers (empty: all 8 warps have read their last
//          column of the slab; full: all 8 warps have stored their rows of the next one).
template <typename TIn> struct SubSlab {  // uint8
    using elem = uint2;
    static constexpr int IPS = 4;
    static constexpr bool CTA_WIDE = true;
    __device__ static int col(int u, int q) { return 16 * (u / 4); }
};
template <> struct SubSlab<float> {
    using elem = float2;
    static constexpr int IPS = 1;
    static constexpr bool CTA_WIDE = false;
    __device__ static int col(int u, int q) { return 4 * u + 2 * q; }
};
constexpr int YBOXW = 8;  // floats per row of a TMA store box of pass y (4 complex columns)
template <typename TIn> struct SmemYQ {
    float2 xb[8][XB];
    Exch ex;
    alignas(128) float2 stage[NL][4];  // [n1][column of the unit]: final sums, TMA store source
    typename TileElem<TIn>::type tile[2][SubSlab<TIn>::IPS][N][2];  // [quad][k][n'][h]
    unsigned long long full, empty;  // hand-over of the CTA-wide slab (uint8), 8 arrivals each
    unsigned tmem;
};
template <typename TIn> struct SubRegs { typename SubSlab<TIn>::elem e[16]; };

// the 128 threads of a quad fetch rows qt, qt + 128, .. of the slab that starts at column col
template <typename TIn>
__device__ __forceinline__ void sub_load(SubRegs<TIn> &t, const TIn *holo, long long hstride,
                                         int col, int qt) {
#pragma unroll
    for (int i = 0; i < 16; ++i)
        t.e[i] = *reinterpret_cast<const typename SubSlab<TIn>::elem *>(
            holo + (size_t)(qt + 128 * i) * hstride + col);
}
template <typename TIn>
__device__ __forceinline__ void sub_prefetch(const TIn *holo, long long hstride, int col, int qt) {
#pragma unroll
    for (int i = 0; i < 16; ++i)
        asm volatile("prefetch.global.L2 [%0];" ::"l"(holo + (size_t)(qt + 128 * i) * hstride + col));
}
__device__ __forceinline__ void sub_store(const SubRegs<unsigned char> &t,
                                          unsigned short (*tile)[N][2], int qt, int quad) {
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int n0 = qt + 128 * i, n = n0 & (N - 1), h = n0 >> 10;
        tile[0][n][h] = (unsigned short)(t.e[i].x >> (16 * quad));
        tile[1][n][h] = (unsigned short)(t.e[i].y >> (16 * quad));
    }
}
__device__ __forceinline__ void sub_store(const SubRegs<float> &t, float2 (*tile)[N][2], int qt,
                                          int quad) {
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const int n0 = qt + 128 * i;
        tile[0][n0 & (N - 1)][n0 >> 10] = t.e[i];
    }
}
// uint8, CTA-wide: the 256 threads fetch rows tid, tid + 256, .. (16 bytes each) of the slab that starts
// at column col and split them into the two quads' tiles: byte 4 k + 2 q + c = unit k, quad q, column c
struct Slab16 { uint4 e[8]; };
__device__ __forceinline__ void slab16_load(Slab16 &t, const unsigned char *holo, long long hstride,
                                            int col, int tid) {
#pragma unroll
    for (int i = 0; i < 8; ++i)
        t.e[i] = *reinterpret_cast<const uint4 *>(holo + (size_t)(tid + 256 * i) * hstride + col);
}
__device__ __forceinline__ void slab16_store(const Slab16 &t, unsigned short (*tile)[4][N][2], int tid) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int n0 = tid + 256 * i, n = n0 & (N - 1), h = n0 >> 10;
        const unsigned w[4] = {t.e[i].x, t.e[i].y, t.e[i].z, t.e[i].w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            tile[0][k][n][h] = (unsigned short)(w[k] & 0xffffu);
            tile[1][k][n][h] = (unsigned short)(w[k] >> 16);
        }
    }
}
__device__ __forceinline__ void slab16_load(Slab16 &, const float *, long long, int, int) {}
__device__ __forceinline__ void slab16_store(const Slab16 &, float2 (*)[1][N][2], int) {}
// both samples (rows n' and n' + 1024) of column c of the pair
__device__ __forceinline__ float2 fold_values(const unsigned short (&e)[2], int c) {
    const unsigned w = *reinterpret_cast<const unsigned *>(e);  // [n'] low half, [n' + 1024] high half
    return make_float2(
        __uint_as_float(__byte_perm(w, 0x4B000000u, c ? 0x7651u : 0x7650u)) - 8388608.f,
        __uint_as_float(__byte_perm(w, 0x4B000000u, c ? 0x7653u : 0x7652u)) - 8388608.f);
}
__device__ __forceinline__ float2 fold_values(const float2 (&e)[2], int c) {
    const float4 w = *reinterpret_cast<const float4 *>(e);
    return c ? make_float2(w.y, w.w) : make_float2(w.x, w.z);
}

// tmB: tensor map of B seen as float [V * NL][2 nx] with box YBOXW x YBOX; hstride = elements
// between hologram rows.
template <typename TIn>
__device__ __forceinline__ void pass_y_quad(SmemYQ<TIn> &sm, const TIn *holo, long long hstride,
                                            unsigned tq, unsigned tt, const void *tmB,
                                            Range rg, unsigned &ph_full, unsigned &ph_empty) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, quad = warp >> 2, b = warp & 3;
    const int qt = threadIdx.x & 127;
    constexpr int IPS = SubSlab<TIn>::IPS;
    if (rg.u0 >= rg.u1) return;  // CTA-uniform
    float2 *xb = sm.xb[warp];
    float2 *stg = &sm.stage[0][0];
    const bool leader = threadIdx.x == 0;  // issues and retires the bulk stores
    constexpr bool CTA_WIDE = SubSlab<TIn>::CTA_WIDE;
    auto warp_arrive = [&](unsigned long long *bar) {
        __syncwarp();
        if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
    };
    if (CTA_WIDE) {
        Slab16 t;
        slab16_load(t, holo, hstride, SubSlab<TIn>::col(rg.u0, quad), threadIdx.x);
        slab16_store(t, sm.tile, threadIdx.x);
        warp_arrive(&sm.full);
    } else {
        SubRegs<TIn> t;
        sub_load<TIn>(t, holo, hstride, SubSlab<TIn>::col(rg.u0, quad), qt);
        sub_store(t, sm.tile[quad], qt, quad);
        quad_sync(quad);
    }
    bool fresh = CTA_WIDE;  // a slab this warp has not yet waited for is on its way into the tile
    const Turns turns = turns_make(warp, 8, 5, true);  // named barriers 5..12
    turns_open(turns, warp, 8);
    for (int u = rg.u0; u < rg.u1; ++u) {
        const int k = u % IPS;
        const bool next_slab = u + 1 < rg.u1 && k == IPS - 1;
#pragma unroll 1
        for (int cc = 0; cc < 2; ++cc) {  // the quad's two columns, one after the other
            float2 v[32];
            if (CTA_WIDE && fresh) {  // all 8 warps have stored their rows of this slab
                mbar_wait(&sm.full, ph_full);
                ph_full ^= 1;
                fresh = false;
            }
            {   // v = a[n'] preA_b + a[n' + 1024] preB_b (a real)
                TChunk ca, cb;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    tm_ld(ca, tq + TQ_PREA + 16 * j);
                    tm_ld(cb, tq + TQ_PREB + 16 * j);
                    tm_wait(ca);
                    tm_wait(cb);
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const int r = 8 * j + i;
                        const float2 a = fold_values(sm.tile[quad][k][lane + 32 * r], cc);
                        const float2 pa = tm_val(ca, i), pb = tm_val(cb, i);
                        v[r] = make_float2(fmaf(a.y, pb.x, a.x * pa.x), fmaf(a.y, pb.y, a.x * pa.y));
                    }
                }
            }
            // the next sub-slab is pulled towards L2 now and loaded after the branch: 32 registers of
            // slab held across the butterflies spilled (measured: 0.91 ms per launch of config 4 with
            // the loads here, 0.72 ms with the prefetch)
            if (cc == 1 && next_slab) {
                if (CTA_WIDE)
                    warp_arrive(&sm.empty);  // this warp's last read of the slab
                else
                    sub_prefetch<TIn>(holo, hstride, SubSlab<TIn>::col(u + 1, quad), qt);
            }
            quad_sync(quad);  // the previous column's exchange area has been read by all four warps
            branch<false>(v, lane, xb, tt, tq + TQ_H, turns);
            // The two quads share the staging tile (32-byte rows of B need all four columns of the
            // unit) but must not share a CTA-wide barrier: that lines up the two warps of every
            // sub-partition (w and w + 4 sit in different quads), which then run their butterflies at
            // the same time and their shared-memory phases at the same time.  Instead warp 0, which
            // issues the bulk stores, tells quad 1 when the tile is free (named barrier 13: it arrives,
            // quad 1 waits - it has arrived long before) and is told when the tile is complete (named
            // barrier 14: everybody else arrives, warp 0 waits).
            if (cc == 0 && warp == 0) {
                // the previous unit's bulk stores must have left the staging tile before it is rewritten
                if (leader) bulk_wait_read();
                __syncwarp();
                asm volatile("bar.arrive 13, 160;" ::: "memory");
            }
            float2 mine[16];
            quad_scatter(v, mine, tq, b, lane, sm.xb, sm.ex, warp);
            quad_sync(quad);
            if (cc == 0 && quad == 1) asm volatile("bar.sync 13, 160;" ::: "memory");
            quad_collect(mine, b, lane, sm.xb, sm.ex, warp);
#pragma unroll
            for (int i = 0; i < 16; ++i) stg[(lane + 32 * (16 * b + i)) * 4 + 2 * quad + cc] = mine[i];
            if (cc == 1) {
                if (next_slab && CTA_WIDE) {
                    Slab16 t;
                    slab16_load(t, holo, hstride, SubSlab<TIn>::col(u + 1, quad), threadIdx.x);
                    mbar_wait(&sm.empty, ph_empty);  // both quads have read their last column of the slab
                    ph_empty ^= 1;
                    slab16_store(t, sm.tile, threadIdx.x);
                    warp_arrive(&sm.full);
                    fresh = true;
                } else if (next_slab) {  // the tile was last read before this column's first barrier
                    SubRegs<TIn> t;
                    sub_load<TIn>(t, holo, hstride, SubSlab<TIn>::col(u + 1, quad), qt);
                    sub_store(t, sm.tile[quad], qt, quad);
                }
                fence_async_smem();  // staging writes -> async proxy
                quad_sync(quad);     // this quad's columns are in the staging tile, its next slab visible
                if (warp == 0)
                    asm volatile("bar.sync 14, 256;" ::: "memory");  // staging tile complete (both quads)
                else
                    asm volatile("bar.arrive 14, 256;" ::: "memory");
                if (leader) {
#pragma unroll
                    for (int j = 0; j < NL / YBOX; ++j)
                        tma_store_2d(tmB, stg + j * YBOX * 4, 8 * u, rg.view * NL + j * YBOX);
                    bulk_commit();
                }
            }
        }
    }
    if (leader) bulk_wait_read();  // shared memory must outlive the last store's reads
    turns_close(turns, warp);
}

}  // namespace sfdq
