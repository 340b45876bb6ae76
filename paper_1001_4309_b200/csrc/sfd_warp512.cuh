// sfd_warp512.cuh — lines of length 512: one warp per line, no branch split.
//
// A 512-point line pads to exactly M = 1024 points, the size of the warp FFT of sfd_warp1024.cuh
// (32 lanes x 32 complex values in registers, two radix-32 stages around one 32 x 32 transpose):
//
//     out[n] = post[n] IFFT_1024( H[k] FFT_1024( in[n] pre[n] padded with zeros ) )[n],   n < 512
//
// is ONE call of sfdw::branch() with the upper half of the input registers zero and the upper half of
// the output registers dropped.  No split by the parity of the frequency index, hence no partner
// warp, no exchange of partial sums and no barrier on the transform path: a warp loads a line,
// transforms it and stores it.  What is left of the inter-warp traffic of the N = 1024 kernels:
//   pass y  the 8 warps of a CTA share the 8-byte input slab of a round (8 adjacent columns; the two
//           slab buffers are handed over with mbarriers, not with a CTA-wide barrier, which would line
//           up the two warps of every sub-partition: see pass_y_loop), and the two warps of a pair share a
//           staging tile [n1][2 columns] so that the TMA store writes 16-byte rows of B (one pair
//           barrier per line, staging double-buffered);
//   pass x  nothing (rows arrive by per-warp bulk copies, outputs leave as coalesced stores);
// plus the turn-taking of the two warps of a sub-partition (sfdw::Turns).
// Tables of a view in tensor memory, the same in all four lane quarters (every warp runs the same
// transform): pre (16 values per lane) | H (32) | conj(post) (16) = 128 columns per view set, three
// sets (a CTA's contiguous range of lines touches at most two views when the grid has >= V CTAs;
// the third set is spare), the stage-B twiddles behind them.
#pragma once
#include "sfd_warp1024.cuh"

namespace sfdh {

using namespace sfdw;  // N = 1024 is the padded length here

constexpr int NH = 512;                          // line length
constexpr int TH_SET = 128, TH_H = 32, TH_TW = 384;  // columns: set stride, H inside a set, twiddles
constexpr int HTABS = NH + N + NH;               // complex elements of one view's tables of one pass

// the R = 2 warps of a sub-partition copy the 8 chunks of `view` into set `set` of their quarter
__device__ __forceinline__ void tmh_fill(unsigned quarter, int set, const float2 *__restrict__ tab,
                                         long long vstride, int view, int warp, int lane) {
    const float2 *src = tab + (size_t)view * vstride + lane;
    const int ch0 = 4 * (warp >> 2);
    TChunk c[4];
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const float2 x = __ldg(src + 32 * (8 * (ch0 + j) + i));
            c[j].w[2 * i] = __float_as_uint(x.x);
            c[j].w[2 * i + 1] = __float_as_uint(x.y);
        }
#pragma unroll
    for (int j = 0; j < 4; ++j) tm_st(c[j], quarter + set * TH_SET + 16 * (ch0 + j));
}
__device__ __forceinline__ unsigned tmh_setup(unsigned *slot, const float2 *__restrict__ tab,
                                              long long vstride, int total, int per_view,
                                              const float2 *__restrict__ twl) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int a0 = (int)((long long)total * blockIdx.x / gridDim.x);
    const int a1 = (int)((long long)total * (blockIdx.x + 1) / gridDim.x);
    if (warp == 0) tm_alloc(slot);
    tm_sync_cta();
    const unsigned base = *reinterpret_cast<volatile unsigned *>(slot);
    if (a0 < a1) {
        const unsigned q = tm_quarter(base, warp);
        const int view0 = a0 / per_view;
        tmh_fill(q, 0, tab, vstride, view0, warp, lane);
        if ((a1 - 1) / per_view != view0) tmh_fill(q, 1, tab, vstride, view0 + 1, warp, lane);
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    }
    if (warp < 4) tm_fill_twiddles(tm_quarter(base, warp) + TH_TW, twl, lane);
    tm_sync_cta();
    return base;
}

// ---- pass x: one row of B per warp ------------------------------------------------------------------
struct SmemXH {
    float2 xb[8][XB];
    float2 inb[8][NH];  // input row of each warp (bulk async copy destination)
    unsigned long long ibar[8];
    unsigned tmem;
};

// A CTA takes a contiguous range of the V ny rows and walks it in rounds of 8, warp w taking row
// l0 + 8 r + w.  ny (a power of two) is a run-time value; tabX: pre | H | conj(post) per view.
__device__ __forceinline__ void pass_x_half(SmemXH &sm, const float2 *Bin, int ny, unsigned tq,
                                            float2 *__restrict__ field, float *__restrict__ inten,
                                            unsigned int *vmax, double *mom, int V) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int lgn = 31 - __clz(ny);
    const int lines = V * ny;
    const int l0 = (int)((long long)lines * blockIdx.x / gridDim.x);
    const int l1 = (int)((long long)lines * (blockIdx.x + 1) / gridDim.x);
    if (l0 >= l1) return;  // CTA-uniform
    float2 *xb = sm.xb[warp];
    const float2 *in = sm.inb[warp] + lane;
    const int view0 = l0 >> lgn;
    unsigned iphase = 0;
    const Turns turns = turns_make(warp, 8, 5, true);
    turns_open(turns, warp, 8);
    if (lane == 0 && l0 + warp < l1)
        bulk_load(sm.inb[warp], Bin + (size_t)(l0 + warp) * NH, NH * sizeof(float2), &sm.ibar[warp]);
    for (int L = l0 + warp; L - warp < l1; L += 8) {
        if (L >= l1) {  // warp-uniform: no row left for this warp in the last round
            turns_skip(turns);
            continue;
        }
        const int view = L >> lgn;
        const unsigned tpre = tq + (view - view0) * TH_SET;  // pre | H | conj(post)
        mbar_wait(&sm.ibar[warp], iphase);
        iphase ^= 1;
        float2 v[32];
        {
            TChunk c0, c1;
            tm_ld(c0, tpre);
            tm_ld(c1, tpre + 16);
            tm_wait(c0);
            tm_wait(c1);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                v[i] = cmul(in[32 * i], tm_val(c0, i));
                v[8 + i] = cmul(in[32 * (8 + i)], tm_val(c1, i));
            }
#pragma unroll
            for (int r = 16; r < 32; ++r) v[r] = make_float2(0.f, 0.f);
        }
        __syncwarp();  // every lane has consumed the row
        if (lane == 0 && L + 8 < l1) {
            fence_async_smem();
            bulk_load(sm.inb[warp], Bin + (size_t)(L + 8) * NH, NH * sizeof(float2), &sm.ibar[warp]);
        }
        branch<true, 2>(v, lane, xb, tq + TH_TW, tpre + TH_H, turns);
        float mx = 0.f, s1 = 0.f, s2 = 0.f;
        const size_t off = (size_t)L * NH;
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const int m1 = lane + 32 * q;
            const float2 w = v[q];
            if (field) field[off + m1] = w;
            const float I = w.x * w.x + w.y * w.y;
            if (inten) inten[off + m1] = I;
            mx = fmaxf(mx, I);
            s1 += I;
            s2 = fmaf(I, I, s2);
        }
        if (mom != nullptr) {  // focus moments (row f2): sum I, sum I^2 of the view
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                s1 += __shfl_xor_sync(0xffffffffu, s1, o);
                s2 += __shfl_xor_sync(0xffffffffu, s2, o);
            }
            if (lane == 0) {
                atomicAdd(mom + 2 * view, (double)s1);
                atomicAdd(mom + 2 * view + 1, (double)s2);
            }
        }
        if (vmax != nullptr) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
            if (lane == 0) atomicMax(vmax + view, __float_as_uint(mx));
        }
    }
    turns_close(turns, warp);
}

// ---- pass y: one hologram column per warp, 8 adjacent columns per CTA and round ---------------------
// Input slab of a round: 8 columns of every hologram row (uint8: 8 bytes, float: 32 bytes), kept in
// shared memory as [pair][n0] column pairs (the layout of the N = 1024 kernels' tile), two buffers.
template <typename TIn> struct SlabH;
template <> struct SlabH<unsigned char> {
    struct Regs { uint2 e[2]; };
    __device__ static void load(Regs &t, const unsigned char *holo, long long hstride, int col, int tid) {
#pragma unroll
        for (int i = 0; i < 2; ++i)
            t.e[i] = *reinterpret_cast<const uint2 *>(holo + (size_t)(tid + 256 * i) * hstride + col);
    }
    __device__ static void store(const Regs &t, unsigned short (*tile)[NH], int tid) {
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            tile[0][tid + 256 * i] = (unsigned short)(t.e[i].x & 0xffffu);
            tile[1][tid + 256 * i] = (unsigned short)(t.e[i].x >> 16);
            tile[2][tid + 256 * i] = (unsigned short)(t.e[i].y & 0xffffu);
            tile[3][tid + 256 * i] = (unsigned short)(t.e[i].y >> 16);
        }
    }
};
template <> struct SlabH<float> {
    struct Regs { float4 e[2][2]; };
    __device__ static void load(Regs &t, const float *holo, long long hstride, int col, int tid) {
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const float4 *p = reinterpret_cast<const float4 *>(holo + (size_t)(tid + 256 * i) * hstride + col);
            t.e[i][0] = p[0];
            t.e[i][1] = p[1];
        }
    }
    __device__ static void store(const Regs &t, float2 (*tile)[NH], int tid) {
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            tile[0][tid + 256 * i] = make_float2(t.e[i][0].x, t.e[i][0].y);
            tile[1][tid + 256 * i] = make_float2(t.e[i][0].z, t.e[i][0].w);
            tile[2][tid + 256 * i] = make_float2(t.e[i][1].x, t.e[i][1].y);
            tile[3][tid + 256 * i] = make_float2(t.e[i][1].z, t.e[i][1].w);
        }
    }
};
template <typename TIn> struct SmemYH {
    float2 xb[8][XB];
    alignas(128) float2 stage[4][2][NH][2];  // [pair][buffer][n1][column of the pair]: TMA store source
    typename TileElem<TIn>::type tile[2][4][NH];  // [buffer][pair][n0]: the CTA's slab
    unsigned long long full[2], empty[2];  // slab buffers: stored by all 8 warps / read by all 8 warps
    unsigned tmem;
};

// Work item = (view, 8 adjacent columns); a CTA takes a contiguous range of items.  nx (a multiple
// of 16) and the hologram's row stride are run-time values.  tmB: tensor map of B seen as float
// [V * NH][2 nx] with box 4 x YBOX.
template <typename TIn>
__device__ __forceinline__ void pass_y_half(SmemYH<TIn> &sm, const TIn *holo, long long hstride,
                                            int nx, unsigned tq, const void *tmB, int V) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, pair = warp >> 1, c = warp & 1;
    const int ipv = nx >> 3, lgi = 31 - __clz(ipv);
    const int items = V * ipv;
    const int i0 = (int)((long long)items * blockIdx.x / gridDim.x);
    const int i1 = (int)((long long)items * (blockIdx.x + 1) / gridDim.x);
    if (i0 >= i1) return;  // CTA-uniform
    float2 *xb = sm.xb[warp];
    const bool leader = c == 0 && lane == 0;  // issues and retires the pair's bulk stores
    const int view0 = i0 >> lgi;
    auto warp_arrive = [&](unsigned long long *bar) {  // this warp's rows are stored / read
        __syncwarp();
        if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
    };
    typename SlabH<TIn>::Regs t;
    SlabH<TIn>::load(t, holo, hstride, 8 * (i0 & (ipv - 1)), threadIdx.x);
    SlabH<TIn>::store(t, sm.tile[0], threadIdx.x);
    warp_arrive(&sm.full[0]);
    unsigned ph_full = 0, ph_empty = 0;  // bit b: parity of the next completion of full[b] / empty[b]
    const Turns turns = turns_make(warp, 8, 5, true);
    turns_open(turns, warp, 8);
    for (int item = i0; item < i1; ++item) {
        const int view = item >> lgi, g = item & (ipv - 1), buf = (item - i0) & 1;
        const unsigned tpre = tq + (view - view0) * TH_SET;
        const bool has_next = item + 1 < i1;
        // the slab of this round is complete (all 8 warps stored their rows during the round before)
        mbar_wait(&sm.full[buf], (ph_full >> buf) & 1u);
        ph_full ^= 1u << buf;
        float2 v[32];
        {
            TChunk c0, c1;
            tm_ld(c0, tpre);
            tm_ld(c1, tpre + 16);
            tm_wait(c0);
            tm_wait(c1);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const float a0 = tile_value(sm.tile[buf][pair][lane + 32 * i], c);
                const float a1 = tile_value(sm.tile[buf][pair][lane + 32 * (8 + i)], c);
                const float2 p0 = tm_val(c0, i), p1 = tm_val(c1, i);
                v[i] = make_float2(a0 * p0.x, a0 * p0.y);
                v[8 + i] = make_float2(a1 * p1.x, a1 * p1.y);
            }
#pragma unroll
            for (int r = 16; r < 32; ++r) v[r] = make_float2(0.f, 0.f);
        }
        if (has_next) SlabH<TIn>::load(t, holo, hstride, 8 * ((g + 1) & (ipv - 1)), threadIdx.x);
        warp_arrive(&sm.empty[buf]);  // this warp has read its column of the slab
        branch<true, 2>(v, lane, xb, tq + TH_TW, tpre + TH_H, turns);
        if (has_next) {
            if (item > i0) {  // all 8 warps have read the slab of the round before out of that buffer
                mbar_wait(&sm.empty[buf ^ 1], (ph_empty >> (buf ^ 1)) & 1u);
                ph_empty ^= 1u << (buf ^ 1);
            }
            SlabH<TIn>::store(t, sm.tile[buf ^ 1], threadIdx.x);
            warp_arrive(&sm.full[buf ^ 1]);
        }
        // staging buffer `buf` of the pair: its last bulk store (two lines ago) has read it - the leader
        // made sure of that before the pair barrier of the line before, which orders it before these writes
        float2 *stg = &sm.stage[pair][buf][0][0];
#pragma unroll
        for (int q = 0; q < 16; ++q) stg[(lane + 32 * q) * 2 + c] = v[q];
        fence_async_smem();  // staging writes -> async proxy
        if (leader) bulk_wait_read();  // the store of the line before (other buffer) has read its tile
        pair_sync(pair);               // both columns of the pair are in the staging tile
        if (leader) {
            if (item == i0) pdl_wait();  // B belongs to the kernel before this one until it has completed
#pragma unroll
            for (int j = 0; j < NH / YBOX; ++j)
                tma_store_2d(tmB, stg + j * YBOX * 2, 2 * (8 * g + 2 * pair), view * NH + j * YBOX);
            bulk_commit();
        }
    }
    if (leader) bulk_wait_read();  // shared memory must outlive the last store's reads
    turns_close(turns, warp);
}

}  // namespace sfdh
