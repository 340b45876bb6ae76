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
//
// A line is worked on by a PAIR of warps, one per branch, which meet at a named barrier to add
// their partial results (each warp finishes and stores one half of the line); the half a warp
// hands over travels through its own transpose tile, which is idle by then.
//
// What bounds these kernels (measured): a single warp saturates its
// sub-partition's fp32 pipe during a radix-32 butterfly (FMA-formulated, sfd_dft32.cuh: 388 and 480
// operations for the two stages of an FFT, about 2060 per warp and line), and the chain of
// shared-memory phases of a line (two transposes, exchange, input, stores: 430 wavefronts per warp
// and line, latency-bound in the in-order LSU pipe) is as long again.  So everything that can leave the LSU pipe has left it: the three table vectors of a branch
// (pre_b, H_b, conj(post_b)) live in tensor memory and are read with tcgen05.ld, pass x receives
// its rows by bulk async copy issued a line ahead, pass y hands its output tile to the TMA unit,
// and a CTA walks a CONTIGUOUS range of lines so that it touches at most two views.  Both kernels
// are launched with programmatic stream serialization: their prologue (mbarriers, twiddles,
// tensor-memory tables) overlaps the tail of the kernel before them.
#pragma once
#include "sfd_dft32.cuh"
#include "sfd_fft_core.cuh"

namespace sfdw {

using sfd::cadd;
using sfd::cmul;
using sfd::csub;

constexpr int N = 1024;     // line length handled by this path
constexpr int XS = 34;      // row stride (complex) of the transpose tile: 16-byte aligned rows,
                            // conflict-free for both the 8-byte column writes and 16-byte row reads
constexpr int XB = 32 * XS;  // complex elements of one warp's transpose tile

// Packed fp32 pairs (sm_100 FADD2): one instruction adds both components of a complex number (one
// issue slot instead of two; the pipe is occupied for two cycles all the same).  Used where partial
// sums of two warps are added.
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
constexpr int TWN = sfdb::NTW;  // per-lane twiddles of stage B (sfd_dft32.cuh), held in registers

// ---- small PTX helpers ---------------------------------------------------------------------------
// programmatic dependent launch: let the next kernel of the stream start early / wait until the
// kernels before this one have completed and their writes are visible
__device__ __forceinline__ void pdl_launch_dependents() {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
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
// orders this thread's earlier generic-proxy shared-memory accesses before later async-proxy ones
__device__ __forceinline__ void fence_async_smem() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
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

// twl: [31][32] at [j][lane], T_n[k] of sfd_dft32.cuh at j = n/2 - 1 + k (plan constant)
__device__ __forceinline__ void load_twiddles(float2 (&tw)[TWN], int lane,
                                              const float2 *__restrict__ twl) {
#pragma unroll
    for (int j = 0; j < TWN; ++j) tw[j] = __ldg(twl + j * 32 + lane);
}

// Tables of one view and one pass as they sit in global memory ([V][2][3][N], plan time) and in
// shared memory: for branch b the vectors pre_b, H_b, conj(post_b).
constexpr int TABS = 2 * 3 * N;  // complex elements

// ---- tables in tensor memory --------------------------------------------------------------------
// The three table vectors of a branch are read once per line and thread (96 complex values): from
// shared memory that is a third of all shared-memory wavefronts of a line, on the pipe that also
// carries the transposes.  Tensor memory (256 KB per SM, 128 lanes x 512 columns of 32 bits, unused
// here otherwise: there is no MMA on this path) has its own read path into the register file
// (tcgen05.ld, 148 B/clk per sub-partition measured - sfd_measure_memory_pipes -, no contention between
// sub-partitions), and its shape fits: a warp may touch only the 32 lanes of its sub-partition, lane l
// of warp w holds what thread l needs.  Both warps of a sub-partition (w, w + 4) run the same branch b = w & 1, so each
// lane quarter holds, per view set s (a CTA's lines lie in at most two views), 192 columns:
//     column 192 s + 64 t + 2 r + {0, 1} = re, im of table t (pre_b, H_b, conj(post_b)) at lane + 32 r
// A chunk is 16 columns = 8 complex values; tcgen05.wait::ld waits for every load in flight, so
// the loops below wait for chunk j, start chunk j + 1 and then use chunk j.
constexpr int TM_COLS = 512;      // allocated columns (all of it: one CTA per SM)
constexpr int TM_SET = 192;       // columns of one view set
constexpr int TM_TAB = 64;        // columns of one table
constexpr int TM_TW = 2 * TM_SET;  // 64 columns of stage-B twiddles (31 per-lane values + pad)
struct TChunk { unsigned w[16]; };
#define SFDW_O16(c) "=r"(c.w[0]), "=r"(c.w[1]), "=r"(c.w[2]), "=r"(c.w[3]), "=r"(c.w[4]), "=r"(c.w[5]), \
    "=r"(c.w[6]), "=r"(c.w[7]), "=r"(c.w[8]), "=r"(c.w[9]), "=r"(c.w[10]), "=r"(c.w[11]), "=r"(c.w[12]), \
    "=r"(c.w[13]), "=r"(c.w[14]), "=r"(c.w[15])
#define SFDW_IO16(c) "+r"(c.w[0]), "+r"(c.w[1]), "+r"(c.w[2]), "+r"(c.w[3]), "+r"(c.w[4]), "+r"(c.w[5]), \
    "+r"(c.w[6]), "+r"(c.w[7]), "+r"(c.w[8]), "+r"(c.w[9]), "+r"(c.w[10]), "+r"(c.w[11]), "+r"(c.w[12]), \
    "+r"(c.w[13]), "+r"(c.w[14]), "+r"(c.w[15])
#define SFDW_I16(c) "r"(c.w[0]), "r"(c.w[1]), "r"(c.w[2]), "r"(c.w[3]), "r"(c.w[4]), "r"(c.w[5]), \
    "r"(c.w[6]), "r"(c.w[7]), "r"(c.w[8]), "r"(c.w[9]), "r"(c.w[10]), "r"(c.w[11]), "r"(c.w[12]), \
    "r"(c.w[13]), "r"(c.w[14]), "r"(c.w[15])
// same, tied to `dep` so that the load is issued before anything that consumes dep afterwards
__device__ __forceinline__ void tm_ld_before(TChunk &c, unsigned taddr, float &dep) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%17];"
        : SFDW_O16(c), "+f"(dep)
        : "r"(taddr));
}
__device__ __forceinline__ void tm_ld(TChunk &c, unsigned taddr) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : SFDW_O16(c)
        : "r"(taddr));
}
// the registers of `c` are valid afterwards (they are operands so that no use moves above the wait)
__device__ __forceinline__ void tm_wait(TChunk &c) {
    asm volatile("tcgen05.wait::ld.sync.aligned;" : SFDW_IO16(c));
}
__device__ __forceinline__ void tm_st(const TChunk &c, unsigned taddr) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%16], "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15};" ::SFDW_I16(c),
        "r"(taddr)
        : "memory");
}
__device__ __forceinline__ float2 tm_val(const TChunk &c, int i) {
    return make_float2(__uint_as_float(c.w[2 * i]), __uint_as_float(c.w[2 * i + 1]));
}
// warp 0 allocates all columns and publishes the base address in *slot
__device__ __forceinline__ void tm_alloc(unsigned *slot) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(
                     smem_u32(slot)),
                 "n"(TM_COLS)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tm_free(unsigned base) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(base), "n"(TM_COLS)
                 : "memory");
}
__device__ __forceinline__ void tm_sync_cta() {  // makes tcgen05.st of other warps visible
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
}
// this warp's lane quarter
__device__ __forceinline__ unsigned tm_quarter(unsigned base, int warp) {
    return base + ((unsigned)(32 * (warp & 3)) << 16);
}
// The R = NW / 4 warps of a sub-partition copy the tables of `view`, branch warp & 1, into set `set`
// of their quarter: warp w + 4 r the chunks 12 r / R .. (12 of them: pre_b, H_b, conj(post_b), four
// chunks of 8 values each).  All loads of a thread are issued before the first store (and before
// the allocation): one trip to L2 per set.
// tab: the [2][3][N] block of view 0 in global memory, vstride complex values between views
template <int NW> struct TFill { TChunk c[12 / (NW / 4)]; };
template <int NW>
__device__ __forceinline__ void tm_fill_load(TFill<NW> &f, const float2 *__restrict__ tab,
                                             long long vstride, int view, int warp, int lane) {
    constexpr int CH = 12 / (NW / 4);
    const float2 *src = tab + (size_t)view * vstride + (size_t)(warp & 1) * 3 * N + lane;
    const int ch0 = CH * (warp >> 2);  // first chunk of this warp; chunk = 8 values, 4 chunks per table
#pragma unroll
    for (int j = 0; j < CH; ++j)
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const float2 x = __ldg(src + 32 * (8 * (ch0 + j) + i));  // table t = chunk / 4 starts at t * N
            f.c[j].w[2 * i] = __float_as_uint(x.x);
            f.c[j].w[2 * i + 1] = __float_as_uint(x.y);
        }
}
template <int NW>
__device__ __forceinline__ void tm_fill_store(const TFill<NW> &f, unsigned quarter, int set, int warp) {
    constexpr int CH = 12 / (NW / 4);
    const int ch0 = CH * (warp >> 2);
#pragma unroll
    for (int j = 0; j < CH; ++j) tm_st(f.c[j], quarter + set * TM_SET + 16 * (ch0 + j));
}
// twl: [31][32] at [j][lane] (plan constant) -> 4 chunks of 8 values in this lane quarter; all 31
// loads of a thread in flight together (tw_load before the allocation, tw_store after it)
struct TwFill { TChunk c[4]; };
__device__ __forceinline__ void tw_load(TwFill &f, const float2 *__restrict__ twl, int lane) {
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const float2 x = (8 * j + i < 31) ? __ldg(twl + (8 * j + i) * 32 + lane) : make_float2(0.f, 0.f);
            f.c[j].w[2 * i] = __float_as_uint(x.x);
            f.c[j].w[2 * i + 1] = __float_as_uint(x.y);
        }
}
__device__ __forceinline__ void tw_store(const TwFill &f, unsigned taddr) {
#pragma unroll
    for (int j = 0; j < 4; ++j) tm_st(f.c[j], taddr + 16 * j);
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tm_fill_twiddles(unsigned taddr, const float2 *__restrict__ twl, int lane) {
    TwFill f;
    tw_load(f, twl, lane);
    tw_store(f, taddr);
}
// Kernel prologue (all NW warps): allocate, fill the one or two view sets this CTA's contiguous
// range [total b / g, total (b + 1) / g) of work units touches (per_view units per view) and the
// twiddle columns, make them visible.  Returns the base address; tm_finish releases it at the end of
// the kernel.
template <int NW>
__device__ __forceinline__ unsigned tm_setup(unsigned *slot, const float2 *__restrict__ tab,
                                             long long vstride, int total, int per_view,
                                             const float2 *__restrict__ twl) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int a0 = (int)((long long)total * blockIdx.x / gridDim.x);
    const int a1 = (int)((long long)total * (blockIdx.x + 1) / gridDim.x);
    const int view0 = a0 < a1 ? a0 / per_view : 0;
    TFill<NW> f;
    TwFill ft;
    if (a0 < a1) tm_fill_load<NW>(f, tab, vstride, view0, warp, lane);  // on their way during the allocation
    if (warp < 4) tw_load(ft, twl, lane);
    if (warp == 0) tm_alloc(slot);
    tm_sync_cta();
    const unsigned base = *reinterpret_cast<volatile unsigned *>(slot);
    if (a0 < a1) {
        const unsigned q = tm_quarter(base, warp);
        tm_fill_store<NW>(f, q, 0, warp);
        if ((a1 - 1) / per_view != view0) {
            tm_fill_load<NW>(f, tab, vstride, view0 + 1, warp, lane);
            tm_fill_store<NW>(f, q, 1, warp);
        }
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    }
    if (warp < 4) tw_store(ft, tm_quarter(base, warp) + TM_TW);
    tm_sync_cta();
    return base;
}
__device__ __forceinline__ void tm_finish(unsigned base) {
    tm_sync_cta();
    if ((threadIdx.x >> 5) == 0) tm_free(base);
}
// Coupling of the warps that share an SM sub-partition (warps w, w + 4, w + 8, .. of a CTA).
// The butterfly phases of a line load the sub-partition's fp32 pipe, the phases between them
// (transposes, table and input reads, exchange, stores) the SM-wide shared-memory pipe; left alone
// the warps of an SM drift into the same phase and the shared-memory pipe sees bursts.  The warps of
// a sub-partition pass a turn round a ring (w -> w + 4 -> .. -> w) around the two transposes of a
// branch: bar.sync on one's own named barrier before the stores into the tile, bar.arrive on the
// successor's after the loads from it (thread count 64).  This does not exclude anything; it bounds
// how far the warps drift apart.  Measured with two warps per sub-partition in round 1 (DESIGN.md
// 5.4: no coupling, strict mbarrier tokens, rendezvous, the same hand-off around the butterfly
// phases): the fastest by 1 to 11 %.
// A CTA has 15 named barriers; a kernel with more warps than that leaves for turns (pass x: 12 warps,
// 6 pair barriers) keeps the ring on mbarriers instead (count 1: the predecessor's lane 0 arrives after
// its __syncwarp, the warp polls the parity of its own): `mb` set, mine / next shared-memory addresses.
// At most one arrival is ever pending on a barrier (a warp's next turn needs the whole ring to go round),
// so a phase cannot be overrun.
struct Turns {
    unsigned mine, next;  // named barriers first .. first + NW - 1 (or mbarrier addresses)
    bool on;
    bool mb = false;
    mutable unsigned ph = 0;  // mbarrier mode: parity of this warp's next turn
};
__device__ __forceinline__ void turn_begin(const Turns &t) {
    if (!t.on) return;
    if (t.mb) {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "W_%=:\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
            "@p bra D_%=;\n"
            "bra W_%=;\n"
            "D_%=:\n"
            "}\n" ::"r"(t.mine),
            "r"(t.ph)
            : "memory");
        t.ph ^= 1;
    } else {
        asm volatile("bar.sync %0, 64;" ::"r"(t.mine) : "memory");
    }
}
__device__ __forceinline__ void turn_end(const Turns &t) {  // (the callers put a __syncwarp in front)
    if (!t.on) return;
    if (t.mb) {
        if ((threadIdx.x & 31) == 0)
            asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(t.next) : "memory");
    } else {
        asm volatile("bar.arrive %0, 64;" ::"r"(t.next) : "memory");
    }
}
// Warps 0..3 own the first turn: the last warps of the ring pass on a turn at the start and warps
// 0..3 take one more after their last line, so that every barrier sees as many arrivals as waits.
// Every warp of a sub-partition must take the same number of turns (a warp without work in a round
// takes empty ones: turns_skip).
__device__ __forceinline__ Turns turns_make(int warp, int nwarps, unsigned first, bool on) {
    const int succ = warp + 4 < nwarps ? warp + 4 : (warp & 3);
    return Turns{first + warp, first + succ, on};
}
// the same ring on the mbarriers bars[0 .. nwarps) (initialised with count 1)
__device__ __forceinline__ Turns turns_make_mb(int warp, int nwarps, unsigned long long *bars, bool on) {
    const int succ = warp + 4 < nwarps ? warp + 4 : (warp & 3);
    Turns t{smem_u32(bars + warp), smem_u32(bars + succ), on};
    t.mb = true;
    return t;
}
__device__ __forceinline__ void turns_open(const Turns &t, int warp, int nwarps) {
    if (warp + 4 >= nwarps) turn_end(t);
}
__device__ __forceinline__ void turns_close(const Turns &t, int warp) {
    if (warp < 4) turn_begin(t);
}
__device__ __forceinline__ void turns_skip(const Turns &t) {  // the two turns of a line, empty
    turn_begin(t);
    turn_end(t);
    turn_begin(t);
    turn_end(t);
}

// stage B with its 31 twiddles streamed from tensor memory (tt: first twiddle column of this
// quarter) through the two chunk buffers: chunk j = t[8j .. 8j+7] of sfdb::dft32_tw
__device__ __forceinline__ void tw_bf(float2 &a, float2 &b, const TChunk &c, int i) {
    const float2 w = tm_val(c, i);
    sfdb::bf(a, b, w.x, w.y);
}
__device__ __forceinline__ void dft32_tw_tm(float2 (&a)[32], unsigned tt, TChunk &c0, TChunk &c1) {
    tm_ld(c0, tt);
    tm_ld(c1, tt + 16);
    sfdb::bit_reverse(a);
    tm_wait(c0);
    tm_wait(c1);
#pragma unroll
    for (int q = 0; q < 32; q += 2) tw_bf(a[q], a[q + 1], c0, 0);                     // level 2: t[0]
#pragma unroll
    for (int q = 0; q < 32; q += 4)
#pragma unroll
        for (int k = 0; k < 2; ++k) tw_bf(a[q + k], a[q + k + 2], c0, 1 + k);        // level 4: t[1..2]
#pragma unroll
    for (int q = 0; q < 32; q += 8)
#pragma unroll
        for (int k = 0; k < 4; ++k) tw_bf(a[q + k], a[q + k + 4], c0, 3 + k);        // level 8: t[3..6]
    tw_bf(a[0], a[8], c0, 7);                                                        // level 16, k = 0: t[7]
    tw_bf(a[16], a[24], c0, 7);
    tm_ld_before(c0, tt + 32, a[0].x);                                               // t[16..23] on their way
#pragma unroll
    for (int q = 0; q < 32; q += 16)
#pragma unroll
        for (int k = 1; k < 8; ++k) tw_bf(a[q + k], a[q + k + 8], c1, k - 1);        // k = 1..7: t[8..14]
    tw_bf(a[0], a[16], c1, 7);                                                       // level 32, k = 0: t[15]
    tm_wait(c0);
    tm_ld_before(c1, tt + 48, a[0].x);                                               // t[24..30]
#pragma unroll
    for (int k = 1; k < 9; ++k) tw_bf(a[k], a[k + 16], c0, k - 1);                   // k = 1..8: t[16..23]
    tm_wait(c1);
#pragma unroll
    for (int k = 9; k < 16; ++k) tw_bf(a[k], a[k + 16], c1, k - 9);                  // k = 9..15: t[24..30]
}

// NOUT: chunks of 8 registers of the result that the caller keeps (the N = 512 kernels need the first
// two: the post multiply skips the rest).
template <bool POST = true, int NOUT = 4>
__device__ __forceinline__ void branch(float2 (&v)[32], int lane, float2 *xb,
                                       unsigned tt, unsigned t, const Turns &turns) {
#pragma unroll 1
    for (int f = 0; f < 2; ++f) {
        sfdb::dft32(v);
        turn_begin(turns);
#pragma unroll
        for (int k = 0; k < 32; ++k) xb[k * XS + lane] = v[k];  // (k1 = k, n2 = lane)
        __syncwarp();
        const float4 *row = reinterpret_cast<const float4 *>(xb + lane * XS);  // k1 = lane
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const float4 w = row[q];
            v[2 * q] = make_float2(w.x, w.y);
            v[2 * q + 1] = make_float2(w.z, w.w);
        }
        __syncwarp();
        turn_end(turns);
        TChunk c0, c1;
        const unsigned ta = t + f * TM_TAB;
        const bool mul = POST || f == 0;
        dft32_tw_tm(v, tt, c0, c1);
        if (mul) tm_ld(c0, ta);
        // v[k] now holds out_sign(k) x the FFT value (sign tracking of sfd_dft32.cuh; the sign stage A
        // left behind depends on the lane and sits in the tables): the compile-time sign is applied
        // together with the conjugation / the table multiply
        if (!mul) {
#pragma unroll
            for (int k = 0; k < 32; ++k) {
                if (sfdb::out_sign(k) > 0)
                    v[k].y = -v[k].y;
                else
                    v[k].x = -v[k].x;
            }
        } else {
#pragma unroll
            for (int j = 0; j < 4; ++j) {  // v = conj(sign v * table)
                if (NOUT < 4 && f == 1 && j >= NOUT) break;
                TChunk &c = (j & 1) ? c1 : c0;
                tm_wait(c);
                if (j < 3 && !(NOUT < 4 && f == 1 && j + 1 >= NOUT)) tm_ld((j & 1) ? c0 : c1, ta + 16 * (j + 1));
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const float sg = (float)sfdb::out_sign(8 * j + i);
                    const float2 h = tm_val(c, i);
                    const float ax = sg * v[8 * j + i].x, ay = sg * v[8 * j + i].y;
                    v[8 * j + i] = make_float2(ax * h.x - ay * h.y, -(ax * h.y) - ay * h.x);
                }
            }
        }
    }
}

// The two warps of a pair hold partial sums v (branch B) for all 32 x 32 outputs of a line.  Warp B
// finishes outputs r in [16 B, 16 B + 16) (element lane + 32 r): it leaves the other 16 in its own
// transpose tile `mine` (idle by now), meets its partner at the pair's named barrier and adds what
// the partner left in `theirs`.  Afterwards v[16 B + q], q < 16, are final.  The caller must put a
// pair barrier (or a CTA barrier) between this and the next write to the tile.
template <int B>
__device__ __forceinline__ void add_halves(float2 (&v)[32], float2 *mine, const float2 *theirs,
                                           int lane, int pair) {
#pragma unroll
    for (int q = 0; q < 16; ++q) mine[q * 32 + lane] = v[16 * (1 - B) + q];
    pair_sync(pair);
#pragma unroll
    for (int q = 0; q < 16; ++q) v[16 * B + q] = padd(v[16 * B + q], theirs[q * 32 + lane]);
}

// ---- pass y: hologram columns, 8 warps per CTA ------------------------------------------------------
// A CTA works inside one view (the launcher gives every view cpv = SMs / V CTAs) and its tensor-memory
// quarters hold the tables of BOTH branches of that view (2 x 192 columns + the twiddles).  Its
// columns come in two kinds of rounds:
//
//   solo rounds   8 adjacent columns, one per warp.  A warp runs branch 0 of its column, parks the
//                 partial sums in registers, runs branch 1 and adds: no partner, no exchange through
//                 shared memory, no barrier between warps on the transform path.  The two warps of a
//                 pair (columns 2p, 2p + 1) meet only at their staging tile [n1][2 columns], from
//                 which one thread hands 16-byte rows of B to the TMA unit.
//   split rounds  4 adjacent columns, a group of four warps per 2 columns, one warp per (column,
//                 branch): the two warps of a column exchange halves of their partial sums through
//                 their transpose tiles (idle by then) and each finishes half of the outputs; the
//                 group's four warps meet at a staging tile.  This is how every column ran in round 1.
//
// Why both: a warp runs a line in two branch-runs when it runs it alone, so solo work comes in units
// of two runs, and V N / (8 x 148) = 3.46 columns per warp would round up to 4 columns = 8 runs.  The
// CTA's whole blocks of 8 columns run solo (3 rounds = 6 runs at config 2), the columns left over in a
// view (136 of 1024) are dealt out in half blocks and run split (1 run): 7 runs, as before, six of
// them without exchange.  Measured on the way: a round of the split kernels 4.31 us, a round of the
// exchange-free N = 512 kernels 3.59 us.
//
// Write-out.  B is [n1][m0] and a column's outputs are one element per row: written by the LSU that
// is one 128-byte wavefront per row and store instruction.  Instead the warps put their final sums
// into a dense staging tile [n1][2 columns] (16 bytes per row) and one thread hands the tile to the
// TMA unit (cp.async.bulk.tensor, shared -> global, four boxes of 256 rows x 16 bytes): the scatter
// costs the LSU pipe nothing and runs beside the next butterflies.
// Read-in.  The CTA reads the 8 hologram columns of a round as one slab (uint8: 8 bytes of every row,
// float: 32) and keeps it in shared memory as four planes [pair of columns][n0] (a 2-byte load per
// row and column costs the LSU one wavefront per row just the same as the 8-byte one); the slab of
// the next round is fetched into registers behind the tile reads of this round and stored into the
// second buffer after the first branch.  The two buffers are handed over with mbarriers (full: all 8
// warps have stored their rows; empty: all 8 warps have read theirs), NOT with a CTA-wide barrier: a
// __syncthreads per round lines up the two warps of every sub-partition, which then run their
// butterflies at the same time and their shared-memory phases at the same time - measured 4.9 us per
// run against 4.3 us for the split rounds it was meant to beat.  With the mbarriers a warp may be up
// to a run ahead of the slowest, and the stagger the turn-taking builds up survives.
constexpr int YBOX = 256;   // rows of one TMA store box (the tensor map is built with this box)
template <typename TIn> struct TileElem {            // uint8
    using type = unsigned short;                     // 2 uint8 columns of a row
};
template <> struct TileElem<float> {
    using type = float2;                             // 2 float columns of a row
};
template <typename TIn> struct SmemY {
    float2 xb[8][XB];
    alignas(128) float2 stage[4][N][2];  // [pair][n1][column of the pair]: final sums, TMA store source
    typename TileElem<TIn>::type tile[2][4][N];  // [buffer][pair of columns][n0]: the slab of a round
    unsigned long long full[2], empty[2];  // slab buffers: stored by all 8 warps / read by all 8 warps
    unsigned tmem;  // base address of the tensor-memory allocation
};

// the 256 threads of the CTA fetch rows tid, tid + 256, .. of the 8 columns that start at column col
// (plain loads: the hologram was written by whatever ran before this kernel in the stream)
template <typename TIn> struct SlabRegs;
template <> struct SlabRegs<unsigned char> { uint2 e[4]; };
template <> struct SlabRegs<float> { float4 e[4][2]; };
__device__ __forceinline__ void slab_load(SlabRegs<unsigned char> &t, const unsigned char *holo,
                                          long long hstride, int col, int tid) {
#pragma unroll
    for (int i = 0; i < 4; ++i)
        t.e[i] = *reinterpret_cast<const uint2 *>(holo + (size_t)(tid + 256 * i) * hstride + col);
}
__device__ __forceinline__ void slab_load(SlabRegs<float> &t, const float *holo, long long hstride,
                                          int col, int tid) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float4 *p = reinterpret_cast<const float4 *>(holo + (size_t)(tid + 256 * i) * hstride + col);
        t.e[i][0] = p[0];
        t.e[i][1] = p[1];
    }
}
__device__ __forceinline__ void slab_store(const SlabRegs<unsigned char> &t, unsigned short (*tile)[N],
                                           int tid) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        tile[0][tid + 256 * i] = (unsigned short)(t.e[i].x & 0xffffu);
        tile[1][tid + 256 * i] = (unsigned short)(t.e[i].x >> 16);
        tile[2][tid + 256 * i] = (unsigned short)(t.e[i].y & 0xffffu);
        tile[3][tid + 256 * i] = (unsigned short)(t.e[i].y >> 16);
    }
}
__device__ __forceinline__ void slab_store(const SlabRegs<float> &t, float2 (*tile)[N], int tid) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        tile[0][tid + 256 * i] = make_float2(t.e[i][0].x, t.e[i][0].y);
        tile[1][tid + 256 * i] = make_float2(t.e[i][0].z, t.e[i][0].w);
        tile[2][tid + 256 * i] = make_float2(t.e[i][1].x, t.e[i][1].y);
        tile[3][tid + 256 * i] = make_float2(t.e[i][1].z, t.e[i][1].w);
    }
}
// uint8 -> float without the conversion unit (I2F shares the MIO queue with shared memory and is
// quarter rate): one byte permute drops the sample into the mantissa of 2^23, one add removes 2^23
__device__ __forceinline__ float tile_value(unsigned short e, int c) {
    return __uint_as_float(__byte_perm((unsigned)e, 0x4B000000u, c ? 0x7651u : 0x7650u)) - 8388608.f;
}
__device__ __forceinline__ float tile_value(float2 e, int c) { return c ? e.y : e.x; }

__device__ __forceinline__ void group_sync(int group) {  // named barrier of the four warps of a group
    asm volatile("bar.sync %0, 128;" ::"r"(group + 1) : "memory");
}
__device__ __forceinline__ void ypair_sync(int pair) {  // pass y: the two warps of a pair (solo rounds)
    asm volatile("bar.sync %0, 64;" ::"r"(pair + 11) : "memory");
}
// 2-D tiled bulk store shared -> global through tensor map `tm` (box fixed by the map); c0 = float
// index within the row of B, c1 = row of B (view * N + n1)
__device__ __forceinline__ void tma_store_2d(const void *tm, const void *src, int c0, int c1) {
    asm volatile(
        "cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%2, %3}], [%1];" ::"l"(tm),
        "r"(smem_u32(src)), "r"(c0), "r"(c1)
        : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
// all earlier bulk stores of this thread have finished READING shared memory
__device__ __forceinline__ void bulk_wait_read() {
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}

// Columns of a view for CTA j of cpv: whole blocks of 8 columns (solo rounds), then half blocks of 4
// out of what cpv does not divide (split rounds).
struct YPlan {
    int solo, split, blk0, half0, cpv;  // rounds of each kind, first block, first leftover column
    __device__ static YPlan make(int nx, int j, int cpv) {
        const int nblk = nx >> 3, solo = nblk / cpv, left = nblk - solo * cpv, halves = 2 * left;
        return YPlan{solo, halves > j ? (halves - j + cpv - 1) / cpv : 0, j * solo, 8 * solo * cpv + 4 * j, cpv};
    }
    __device__ int rounds() const { return solo + split; }
    // first of the 4 (split) or 8 (solo) columns of round r
    __device__ int col(int r) const { return r < solo ? 8 * (blk0 + r) : half0 + 4 * cpv * (r - solo); }
};

// Both branches' tables of `view` into every lane quarter: branch b at column b * TM_SET.  The two
// warps of a sub-partition copy 12 chunks each, six at a time.  tab: the [2][3][N] block of view 0.
__device__ __forceinline__ unsigned tm_setup_both(unsigned *slot, const float2 *__restrict__ tab,
                                                  long long vstride, int view,
                                                  const float2 *__restrict__ twl) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const float2 *src = tab + (size_t)view * vstride + lane;
    const int ch0 = 12 * (warp >> 2);
    TFill<8> f;
    TwFill ft;
    auto load = [&](int first) {
#pragma unroll
        for (int j = 0; j < 6; ++j)
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const float2 x = __ldg(src + 32 * (8 * (first + j) + i));
                f.c[j].w[2 * i] = __float_as_uint(x.x);
                f.c[j].w[2 * i + 1] = __float_as_uint(x.y);
            }
    };
    load(ch0);
    if (warp < 4) tw_load(ft, twl, lane);
    if (warp == 0) tm_alloc(slot);
    tm_sync_cta();
    const unsigned base = *reinterpret_cast<volatile unsigned *>(slot);
    const unsigned q = tm_quarter(base, warp);
#pragma unroll
    for (int j = 0; j < 6; ++j) tm_st(f.c[j], q + 16 * (ch0 + j));
    load(ch0 + 6);
#pragma unroll
    for (int j = 0; j < 6; ++j) tm_st(f.c[j], q + 16 * (ch0 + 6 + j));
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    if (warp < 4) tw_store(ft, q + TM_TW);
    tm_sync_cta();
    return base;
}

template <int B>
__device__ __forceinline__ void y_hand_over(const float2 (&v)[32], float2 *xb, int lane) {
#pragma unroll
    for (int q = 0; q < 16; ++q) xb[q * 32 + lane] = v[16 * (1 - B) + q];
}
template <int B>
__device__ __forceinline__ void y_finish(const float2 (&v)[32], const float2 *xbp, float2 *stg,
                                         int lane, int c) {
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const float2 w = padd(v[16 * B + q], xbp[q * 32 + lane]);
        stg[(lane + 32 * (16 * B + q)) * 2 + c] = w;
    }
}

// tabY: [2][3][N] per view (post carries c0, pre the 1/255 of uint8 input) in tensor memory, branch b
// at tq + b * TM_SET; tmB: tensor map of B seen as float [V * N][2 nx] with box 4 x YBOX.  The line
// length is N = 1024 = the number of hologram rows Ny; the number of columns nx (a multiple of 16) and
// the hologram's row stride are run-time values.  The loop runs over branch-runs so that the line
// transform (branch()) exists once in the code: a solo round is two runs, a split round one.
template <typename TIn>
__device__ __forceinline__ void pass_y_loop(SmemY<TIn> &sm, const TIn *holo, long long hstride,
                                            int nx, unsigned tq, unsigned tt, const void *tmB,
                                            int view, const YPlan yp) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, tid = threadIdx.x;
    const int pair = warp >> 1, b = warp & 1, group = warp >> 2, c = pair & 1;
    const int runs = 2 * yp.solo + yp.split;
    if (runs == 0) return;  // CTA-uniform
    float2 *xb = sm.xb[warp];
    const float2 *xbp = sm.xb[warp ^ 1];
    const bool pair_leader = b == 0 && lane == 0;       // solo rounds: the pair's bulk stores
    const bool group_leader = (tid & 127) == 0;         // split rounds: the group's (the leader of pair 2 group)
    bool waited = false;  // this thread has waited for the kernel before this one (see the first store)
    auto warp_arrive = [&](unsigned long long *bar) {  // this warp's rows are stored / read
        __syncwarp();
        if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
    };
    {
        SlabRegs<TIn> t;
        slab_load(t, holo, hstride, yp.col(0) & ~7, tid);
        slab_store(t, sm.tile[0], tid);
        warp_arrive(&sm.full[0]);
    }
    unsigned ph_full = 0, ph_empty = 0;  // bit b: parity of the next completion of full[b] / empty[b] to wait for
    const Turns turns = turns_make(warp, 8, 3, true);  // named barriers 3..10
    turns_open(turns, warp, 8);
    SlabRegs<TIn> t;
    float2 acc[32];
    int round = -1;
    for (int run = 0; run < runs; ++run) {
        const bool solo = run < 2 * yp.solo, first = !solo || (run & 1) == 0;
        if (first) {
            ++round;
            // the slab of this round is complete (all 8 warps stored their rows during the round before)
            mbar_wait(&sm.full[round & 1], (ph_full >> (round & 1)) & 1u);
            ph_full ^= 1u << (round & 1);
        }
        const int col0 = yp.col(round), buf = round & 1;
        const bool has_next = first && round + 1 < yp.rounds();
        // this warp's column of the round, its place in the slab, its branch
        const int br = solo ? (run & 1) : b;
        const int plane = solo ? pair : ((col0 & 7) >> 1) + group;
        const int byte = solo ? b : c;
        const unsigned tpre = tq + br * TM_SET;  // pre_b | H_b | conj(post_b)
        float2 v[32];
        {
            TChunk c0, c1;
            tm_ld(c0, tpre);
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                TChunk &ch = (j & 1) ? c1 : c0;
                tm_wait(ch);
                if (j < 3) tm_ld((j & 1) ? c0 : c1, tpre + 16 * (j + 1));
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const float a = tile_value(sm.tile[buf][plane][lane + 32 * (8 * j + i)], byte);
                    const float2 p = tm_val(ch, i);
                    v[8 * j + i] = make_float2(a * p.x, a * p.y);
                }
            }
        }
        // the next slab is fetched behind the tile reads: its loads touch one row per lane (32
        // wavefronts each) and would hold up everything queued after them
        if (has_next) slab_load(t, holo, hstride, yp.col(round + 1) & ~7, tid);
        if (!solo || br == 1) warp_arrive(&sm.empty[buf]);  // this warp's last read of the round's slab
        branch(v, lane, xb, tt, tpre + TM_TAB, turns);
        if (has_next) {
            if (round >= 1) {  // all 8 warps have read the slab of the round before out of that buffer
                mbar_wait(&sm.empty[buf ^ 1], (ph_empty >> (buf ^ 1)) & 1u);
                ph_empty ^= 1u << (buf ^ 1);
            }
            slab_store(t, sm.tile[buf ^ 1], tid);
            warp_arrive(&sm.full[buf ^ 1]);
        }
        if (solo && br == 0) {  // park branch 0
#pragma unroll
            for (int r = 0; r < 32; ++r) acc[r] = v[r];
            continue;
        }
        // Programmatic dependent launch: the only thing pass y does to memory that the kernel before
        // it may still be using is to overwrite B (pass x of the frame before reads it), and the only
        // threads that do so are the store leaders.  They wait in front of their first store instead
        // of at the top of the kernel: a CTA that got its SM early (the CTAs of the kernel before do
        // not all finish together) works on its first columns meanwhile.  The hologram is never written
        // by a kernel of this library; whatever else produced it was complete before this kernel could
        // start (only our own kernels release their dependents early).
        if (solo) {
            float2 *stg = &sm.stage[pair][0][0];
            // the pair's previous bulk store has left the staging tile before it is rewritten
            if (pair_leader) bulk_wait_read();
            ypair_sync(pair);
#pragma unroll
            for (int r = 0; r < 32; ++r) stg[(lane + 32 * r) * 2 + b] = padd(v[r], acc[r]);
            fence_async_smem();  // staging writes -> async proxy
            ypair_sync(pair);    // both columns of the pair are in the staging tile
            if (pair_leader) {
                if (!waited) pdl_wait();
                waited = true;
#pragma unroll
                for (int j = 0; j < N / YBOX; ++j)
                    tma_store_2d(tmB, stg + j * YBOX * 2, 2 * (col0 + 2 * pair), view * N + j * YBOX);
                bulk_commit();
            }
        } else {
            float2 *stg = &sm.stage[2 * group][0][0];
            if (group_leader) bulk_wait_read();
            if (b == 0)
                y_hand_over<0>(v, xb, lane);
            else
                y_hand_over<1>(v, xb, lane);
            group_sync(group);  // partner's hand-over visible; staging tile free
            if (b == 0)
                y_finish<0>(v, xbp, stg, lane, c);
            else
                y_finish<1>(v, xbp, stg, lane, c);
            fence_async_smem();  // staging writes -> async proxy
            group_sync(group);   // staging tile complete, hand-over tiles free
            if (group_leader) {
                if (!waited) pdl_wait();
                waited = true;
#pragma unroll
                for (int j = 0; j < N / YBOX; ++j)
                    tma_store_2d(tmB, stg + j * YBOX * 2, 2 * (col0 + 2 * group), view * N + j * YBOX);
                bulk_commit();
            }
        }
    }
    if (lane == 0) bulk_wait_read();  // shared memory must outlive the last stores' reads
    turns_close(turns, warp);
}

// ---- pass x: one row of B per warp pair -----------------------------------------------------------
// Warps per CTA of pass x: 12, three per sub-partition (147 registers per thread with the twiddles in
// tensor memory).  The loop below is written for any multiple of four; measured at config 2 with the
// turn-taking ring on mbarriers (6 pair barriers + 12 turn barriers exceed the 15 named barriers of a
// CTA): 8 warps 34.3 us per launch (33.7 with the ring on named barriers), 12 warps 32.4, 14 warps 34.8
// (128 registers, spills, uneven sub-partitions), 16 warps 32.6 with a slower step.  V N / 148 = 27.7
// lines per CTA are 5 rounds of 6 lines (92 % full) against 7 rounds of 4 (99 %): without the ring the
// third warp only made up for that (33.9 us); with it, it is 4 % ahead.
constexpr int NWX = 12;
template <int NW> struct SmemX {
    float2 xb[NW][XB];
    float2 inb[NW / 2][N];  // input row of each pair (bulk async copy destination)
    unsigned long long ibar[NW / 2];
    unsigned long long tbar[NW];  // turn-taking ring (mbarriers, count 1)
    unsigned tmem;  // base address of the tensor-memory allocation
};

// exchange of the halves, stores, reductions of one line for branch B (see y_hand_over)
template <int B>
__device__ __forceinline__ void x_finish(float2 (&v)[32], float2 *xb, const float2 *xbp, int lane,
                                         int pair, float2 *__restrict__ field,
                                         float *__restrict__ inten, size_t off, double *mom,
                                         unsigned int *vmax, int view) {
    add_halves<B>(v, xb, xbp, lane, pair);
    float mx = 0.f, s1 = 0.f, s2 = 0.f;
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const int m1 = lane + 32 * (16 * B + q);
        const float2 w = v[16 * B + q];
        if (field) field[off + m1] = w;
        const float I = w.x * w.x + w.y * w.y;
        if (inten) inten[off + m1] = I;
        mx = fmaxf(mx, I);
    }
    if (mom != nullptr) {  // focus moments (row f2): sum I, sum I^2 of the view
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const float2 w = v[16 * B + q];
            const float I = w.x * w.x + w.y * w.y;
            s1 += I;
            s2 = fmaf(I, I, s2);
        }
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
        // intensities are >= 0, so their float bit patterns order like unsigned integers
        if (lane == 0) atomicMax(vmax + view, __float_as_uint(mx));
    }
}

// A CTA takes a contiguous range of the V ny rows (at most two views: the launcher sizes the grid
// accordingly) and walks it in rounds of XP = NW / 2 rows, pair p taking row l0 + XP r + p of round
// r; in the last round the pairs beyond the end of the range idle.  The line length is N = 1024 =
// the number of columns Nx; the number of rows per view ny (a power of two) is a run-time value.
// tabX: [2][3][N] per view.
template <int NW, bool TURNS>
__device__ __forceinline__ void pass_x_loop(SmemX<NW> &sm, const float2 *Bin, int ny, unsigned tq,
                                            unsigned tt, float2 *__restrict__ field,
                                            float *__restrict__ inten, unsigned int *vmax,
                                            double *mom, int V) {
    constexpr int XP = NW / 2;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, pair = warp >> 1;
    const int lgn = 31 - __clz(ny);
    const int lines = V * ny;
    const int l0 = (int)((long long)lines * blockIdx.x / gridDim.x);
    const int l1 = (int)((long long)lines * (blockIdx.x + 1) / gridDim.x);
    if (l0 >= l1) return;  // CTA-uniform
    float2 *xb = sm.xb[warp];
    const float2 *xbp = sm.xb[warp ^ 1];
    const float2 *in = sm.inb[pair] + lane;
    const int b = warp & 1;
    const bool issuer = b == 0 && lane == 0;
    const int view0 = l0 >> lgn;
    unsigned iphase = 0;
    // turn-taking of the warps w, w + 4, .. of a sub-partition (named barriers 1 .. XP are the pairs')
    const Turns turns = turns_make_mb(warp, NW, sm.tbar, TURNS);
    turns_open(turns, warp, NW);
    if (issuer && l0 + pair < l1)
        bulk_load(sm.inb[pair], Bin + (size_t)(l0 + pair) * N, N * sizeof(float2), &sm.ibar[pair]);
    for (int L = l0 + pair; L - pair < l1; L += XP) {
        if (L >= l1) {  // pair-uniform: no row left for this pair in the last round
            turns_skip(turns);
            continue;
        }
        const int view = L >> lgn;
        const unsigned tpre = tq + (view - view0) * TM_SET;  // pre_b | H_b | conj(post_b)
        const bool has_next = L + XP < l1;
        mbar_wait(&sm.ibar[pair], iphase);
        iphase ^= 1;
        float2 v[32];
        {
            TChunk c0, c1;
            tm_ld(c0, tpre);
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                TChunk &ch = (j & 1) ? c1 : c0;
                tm_wait(ch);
                if (j < 3) tm_ld((j & 1) ? c0 : c1, tpre + 16 * (j + 1));
#pragma unroll
                for (int i = 0; i < 8; ++i)
                    v[8 * j + i] = cmul(in[32 * (8 * j + i)], tm_val(ch, i));
            }
        }
        // both warps have consumed the input row and finished with each other's transpose tile
        pair_sync(pair);
        if (has_next && issuer) {
            fence_async_smem();
            bulk_load(sm.inb[pair], Bin + (size_t)(L + XP) * N, N * sizeof(float2), &sm.ibar[pair]);
        }
        branch(v, lane, xb, tt, tpre + TM_TAB, turns);
        if (b == 0)
            x_finish<0>(v, xb, xbp, lane, pair, field, inten, (size_t)L * N, mom, vmax, view);
        else
            x_finish<1>(v, xb, xbp, lane, pair, field, inten, (size_t)L * N, mom, vmax, view);
    }
    turns_close(turns, warp);
}

}  // namespace sfdw
