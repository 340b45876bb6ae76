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
// (tcgen05.ld, 64 B/clk per sub-partition measured, no contention between sub-partitions), and its
// shape fits: a warp may touch only the 32 lanes of its sub-partition, lane l of warp w holds what
// thread l needs.  Both warps of a sub-partition (w, w + 4) run the same branch b = w & 1, so each
// lane quarter holds, per view set s (a CTA's lines lie in at most two views), 192 columns:
//     column 192 s + 64 t + 2 r + {0, 1} = re, im of table t (pre_b, H_b, conj(post_b)) at lane + 32 r
// A chunk is 16 columns = 8 complex values; tcgen05.wait::ld waits for every load in flight, so
// the loops below wait for chunk j, start chunk j + 1 and then use chunk j.
constexpr int TM_COLS = 512;      // allocated columns (all of it: one CTA per SM)
constexpr int TM_SET = 192;       // columns of one view set
constexpr int TM_TAB = 64;        // columns of one table
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
// The two warps of a sub-partition copy the tables of `view`, branch warp & 1, into set `set` of
// their quarter: warp w the chunks 0..5 (pre_b and half of H_b), warp w + 4 the chunks 6..11.  All
// 48 loads of a thread are issued before the first store (and before the allocation): one trip
// to L2 per set.
// tab: the [2][3][N] block of view 0 in global memory, vstride complex values between views
struct TFill { TChunk c[6]; };
__device__ __forceinline__ void tm_fill_load(TFill &f, const float2 *__restrict__ tab,
                                             long long vstride, int view, int warp, int lane) {
    const float2 *src = tab + (size_t)view * vstride + (size_t)(warp & 1) * 3 * N + lane;
    const int ch0 = 6 * (warp >> 2);  // first chunk of this warp; chunk = 8 values, 4 chunks per table
#pragma unroll
    for (int j = 0; j < 6; ++j)
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const float2 x = __ldg(src + 32 * (8 * (ch0 + j) + i));  // table t = chunk / 4 starts at t * N
            f.c[j].w[2 * i] = __float_as_uint(x.x);
            f.c[j].w[2 * i + 1] = __float_as_uint(x.y);
        }
}
__device__ __forceinline__ void tm_fill_store(const TFill &f, unsigned quarter, int set, int warp) {
    const int ch0 = 6 * (warp >> 2);
#pragma unroll
    for (int j = 0; j < 6; ++j) tm_st(f.c[j], quarter + set * TM_SET + 16 * (ch0 + j));
}
// Kernel prologue (all threads): allocate, fill the one or two view sets this CTA's contiguous
// range [total b / g, total (b + 1) / g) of work units touches (per_view units per view), make
// them visible.  Returns the base address; tm_finish releases it at the end of the kernel.
__device__ __forceinline__ unsigned tm_setup(unsigned *slot, const float2 *__restrict__ tab,
                                             long long vstride, int total, int per_view) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int a0 = (int)((long long)total * blockIdx.x / gridDim.x);
    const int a1 = (int)((long long)total * (blockIdx.x + 1) / gridDim.x);
    const int view0 = a0 < a1 ? a0 / per_view : 0;
    TFill f;
    if (a0 < a1) tm_fill_load(f, tab, vstride, view0, warp, lane);  // on their way during the allocation
    if (warp == 0) tm_alloc(slot);
    tm_sync_cta();
    const unsigned base = *reinterpret_cast<volatile unsigned *>(slot);
    if (a0 < a1) {
        const unsigned q = tm_quarter(base, warp);
        tm_fill_store(f, q, 0, warp);
        if ((a1 - 1) / per_view != view0) {
            tm_fill_load(f, tab, vstride, view0 + 1, warp, lane);
            tm_fill_store(f, q, 1, warp);
        }
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    }
    tm_sync_cta();
    return base;
}
__device__ __forceinline__ void tm_finish(unsigned base) {
    tm_sync_cta();
    if ((threadIdx.x >> 5) == 0) tm_free(base);
}
// Coupling of the two warps that share an SM sub-partition (warps w and w + 4 of an 8-warp CTA).
// The butterfly phases of a line load the sub-partition's fp32 pipe, the phases between them
// (transposes, table and input reads, exchange, stores) the SM-wide shared-memory pipe; left alone
// the warps of an SM drift into the same phase and the shared-memory pipe sees bursts.  The two
// warps hand a turn to each other around the two transposes of a branch: bar.sync on one's own
// named barrier before the stores into the tile, bar.arrive on the partner's after the loads from it
// (thread count 64).  This does not exclude anything; it bounds how far the two warps drift apart.
// Measured against the alternatives in round 1 (no coupling, strict mbarrier tokens,
// rendezvous, the same hand-off around the butterfly phases): the fastest by 1 to 11 %.
struct Turns {
    unsigned mine, theirs;  // named barriers 5..12
    bool on;
};
__device__ __forceinline__ void turn_begin(const Turns &t) {
    if (t.on) asm volatile("bar.sync %0, 64;" ::"r"(t.mine) : "memory");
}
__device__ __forceinline__ void turn_end(const Turns &t) {
    if (t.on) asm volatile("bar.arrive %0, 64;" ::"r"(t.theirs) : "memory");
}
// Warps 0..3 own the first turn; warps 4..7 pass on their first one and warps 0..3 add one after
// their last line, so that both warps of a sub-partition take the same number of turns.
__device__ __forceinline__ Turns turns_make(int warp, bool on) {
    const unsigned sp = warp & 3, up = warp >> 2;
    return Turns{5u + 2 * sp + up, 5u + 2 * sp + 1 - up, on};
}
__device__ __forceinline__ void turns_open(const Turns &t, int warp) {
    if ((warp >> 2) == 1) turn_end(t);
}
__device__ __forceinline__ void turns_close(const Turns &t, int warp) {
    if ((warp >> 2) == 0) turn_begin(t);
}

// One branch of a line, in place (the caller has applied pre): forward FFT, x H_b, inverse FFT,
// x post_b.  The inverse is run as conj(FFT(conj(.))) so that both transforms execute the same code:
//     v <- conj(FFT(v) H_b);  v <- conj(FFT(v) conj(post_b)) = post_b IFFT(H_b FFT(v)) N
// (the 1/N sits in H).  t = tensor-memory address of H_b in this warp's quarter; conj(post_b) follows it.
// Both tables carry the lane sign of sfd_dft32.cuh: entry lane + 32 r is multiplied by out_sign(lane).
// A 1024-point FFT of a warp (four-step, in v[r] = x[lane + 32 r], out v[r] = X[lane + 32 r]):
//     stage A   32-point DFT over n1 (element lane + 32 n1) in registers            sfdb::dft32
//     transpose 32 x 32 through the warp's tile xb: lane becomes k1, register n2
//     stage B   32-point DFT over n2 with the inter-stage twiddles exp(-2 pi i k1 n2 / 1024)
//               folded into its butterflies (tw: 31 per-lane constants)             sfdb::dft32_tw
// The two FFTs of the branch share one copy of the code (rolled loop): the line transform then fits
// the instruction cache.  On return v = this warp's partial sums for all 1024 outputs.
// POST = false (N = 2048 kernels, sfd_warp2048.cuh): the last multiply is left to the caller, on
// return v = IFFT(H_b FFT(v)) N.
template <bool POST = true>
__device__ __forceinline__ void branch(float2 (&v)[32], int lane, float2 *xb,
                                       const float2 (&tw)[TWN], unsigned t, const Turns &turns) {
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
        if (mul) tm_ld_before(c0, ta, v[0].x);  // in flight during the butterflies
        sfdb::dft32_tw(v, tw);
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
                TChunk &c = (j & 1) ? c1 : c0;
                tm_wait(c);
                if (j < 3) tm_ld((j & 1) ? c0 : c1, ta + 16 * (j + 1));
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

// ---- pass y: 4 adjacent hologram columns per CTA ---------------------------------------------------
// The CTA is two independent halves of four warps (half h = warps 4h .. 4h+3 = two warp pairs);
// half h transforms columns col0 + 2h and col0 + 2h + 1 of the CTA's current item.  Nothing
// synchronises the two halves with each other except the turn-taking of the warps that share a
// sub-partition (warps w and w + 4).
//
// Write-out.  B is [n1][m0] and a column's outputs are one element per row: written by the LSU
// that is one 128-byte wavefront per row and store instruction (the v5 profile: 28 % of the
// data-pipe time of this kernel).  Instead the warps of a half put their final sums into a dense
// staging tile [n1][2 columns] (16 bytes per row) and one thread hands the tile to the TMA unit
// (cp.async.bulk.tensor, shared -> global, four boxes of 256 rows x 16 bytes): the scatter costs the
// LSU pipe nothing and runs beside the next item's butterflies.
constexpr int WY = 8;  // warps per CTA
constexpr int YC = 4;  // columns per item
constexpr int YBOX = 256;  // rows of one TMA store box (the tensor map is built with this box)
// Input slab of a half: SLAB_BYTES = 8 bytes of every hologram row = 2 columns x IPS items.  Half h
// of item (slab s, k) transforms columns YC IPS s + 2 IPS h + 2 k + {0, 1}: the half reads its slab
// once per IPS items with one 8-byte load per row (a 2-byte load per row and item costs the LSU one
// wavefront per row just the same) and keeps it in shared memory as [k][n0] column pairs.
template <typename TIn> struct TileElem {            // uint8: 4 items per slab
    using type = unsigned short;                     // 2 uint8 columns of a row
    using slab = uint2;
    static constexpr int IPS = 4;
};
template <> struct TileElem<float> {                 // float: 1 item per slab
    using type = float2;                             // 2 float columns of a row
    using slab = float2;
    static constexpr int IPS = 1;
};
template <typename TIn> struct SmemY {
    float2 xb[WY][XB];
    alignas(128) float2 stage[2][N][2];  // [half][n1][column of the half]: final sums, TMA store source
    typename TileElem<TIn>::type tile[2][TileElem<TIn>::IPS][N];  // [half][k][n0]: the half's slab
    unsigned tmem;  // base address of the tensor-memory allocation
};

template <typename TIn> struct TileRegs { typename TileElem<TIn>::slab e[8]; };

// the 128 threads of a half fetch rows ht, ht + 128, .. of the slab that starts at column col
// (plain loads: the hologram was written by whatever ran before this kernel in the stream)
template <typename TIn>
__device__ __forceinline__ void tile_load(TileRegs<TIn> &t, const TIn *holo, long long hstride,
                                          int col, int ht) {
#pragma unroll
    for (int i = 0; i < 8; ++i)
        t.e[i] = *reinterpret_cast<const typename TileElem<TIn>::slab *>(
            holo + (size_t)(ht + 128 * i) * hstride + col);
}
__device__ __forceinline__ void tile_store(const TileRegs<unsigned char> &t,
                                           unsigned short (*tile)[N], int ht) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        tile[0][ht + 128 * i] = (unsigned short)(t.e[i].x & 0xffffu);
        tile[1][ht + 128 * i] = (unsigned short)(t.e[i].x >> 16);
        tile[2][ht + 128 * i] = (unsigned short)(t.e[i].y & 0xffffu);
        tile[3][ht + 128 * i] = (unsigned short)(t.e[i].y >> 16);
    }
}
__device__ __forceinline__ void tile_store(const TileRegs<float> &t, float2 (*tile)[N], int ht) {
#pragma unroll
    for (int i = 0; i < 8; ++i) tile[0][ht + 128 * i] = t.e[i];
}
// uint8 -> float without the conversion unit (I2F shares the MIO queue with shared memory and is
// quarter rate): one byte permute drops the sample into the mantissa of 2^23, one add removes 2^23
__device__ __forceinline__ float tile_value(unsigned short e, int c) {
    return __uint_as_float(__byte_perm((unsigned)e, 0x4B000000u, c ? 0x7651u : 0x7650u)) - 8388608.f;
}
__device__ __forceinline__ float tile_value(float2 e, int c) { return c ? e.y : e.x; }

__device__ __forceinline__ void half_sync(int half) {  // named barrier of the four warps of a half
    asm volatile("bar.sync %0, 128;" ::"r"(half + 1) : "memory");
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

// Persistent CTA of 256 threads: work item = (view, group of 4 columns); a CTA takes a contiguous
// range of items (at most two views: the launcher sizes the grid accordingly).  The line length is
// N = 1024 = the number of hologram rows Ny; the number of columns nx (a multiple of 16) and the
// hologram's row stride are run-time values (rectangular grids, windows inside a wider frame).
// tabY: [2][3][N] per view (post carries c0, pre the 1/255 of uint8 input); tmB: tensor map of B seen
// as float [V * N][2 nx] with box 4 x YBOX.
// Per item a warp (column c of its half, branch B) transforms its column, hands the half of the
// outputs it does not finish to its partner through its own transpose tile (idle by then), adds
// what the partner left for it and writes 16 final values per thread into the staging tile.
// The two places of a line that depend on the branch index at compile time (which half of the
// register vector stays) are small functions instantiated for B = 0, 1 and entered through a
// warp-uniform branch; everything else is ONE copy of code for all eight warps (half the
// instruction-cache footprint of two template copies of the whole loop: measured, the
// no_instruction stalls of the N = 2048 kernels, written this way, are a third of those of two copies).
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

template <typename TIn>
__device__ __forceinline__ void pass_y_loop(SmemY<TIn> &sm, const TIn *holo, long long hstride,
                                            int nx, unsigned tq, const float2 (&tw)[TWN],
                                            const void *tmB, int V) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int half = warp >> 2, c = (warp >> 1) & 1, ht = threadIdx.x & 127, b = warp & 1;
    const int groups = nx / YC, lgg = 31 - __clz(groups);  // nx is a power of two: shifts, not divisions
    const int items = V * groups;
    const int i0 = (int)((long long)items * blockIdx.x / gridDim.x);
    const int i1 = (int)((long long)items * (blockIdx.x + 1) / gridDim.x);
    if (i0 >= i1) return;  // CTA-uniform
    float2 *xb = sm.xb[warp];
    const float2 *xbp = sm.xb[warp ^ 1];
    float2 *stg = &sm.stage[half][0][0];
    const bool leader = ht == 0;  // issues and retires the half's bulk stores
    const int view0 = i0 >> lgg;
    constexpr int IPS = TileElem<TIn>::IPS;
    // groups % IPS == 0 (nx is a multiple of 16): a slab never straddles two views
    {
        TileRegs<TIn> t;
        tile_load<TIn>(t, holo, hstride, (i0 & (groups - 1)) / IPS * (YC * IPS) + 2 * IPS * half, ht);
        tile_store(t, sm.tile[half], ht);
    }
    half_sync(half);
    const Turns turns = turns_make(warp, true);
    turns_open(turns, warp);
    for (int item = i0; item < i1; ++item) {
        const int view = item >> lgg, g = item & (groups - 1), k = g % IPS;
        const int colh = g / IPS * (YC * IPS) + 2 * IPS * half + 2 * k;
        const unsigned tpre = tq + (view - view0) * TM_SET;  // pre_b | H_b | conj(post_b)
        const bool has_next = item + 1 < i1 && k == IPS - 1;  // the next item opens a new slab
        TileRegs<TIn> t;
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
                    const float a = tile_value(sm.tile[half][k][lane + 32 * (8 * j + i)], c);
                    const float2 p = tm_val(ch, i);
                    v[8 * j + i] = make_float2(a * p.x, a * p.y);
                }
            }
        }
        // the next slab is fetched behind the tile reads: its loads touch one row per lane (32
        // wavefronts each) and would hold up everything queued after them
        if (has_next)
            tile_load<TIn>(t, holo, hstride, ((item + 1) & (groups - 1)) / IPS * (YC * IPS) + 2 * IPS * half, ht);
        branch(v, lane, xb, tw, tpre + TM_TAB, turns);
        // the previous item's bulk stores must have left the staging tile before it is rewritten
        if (leader) bulk_wait_read();
        if (b == 0)
            y_hand_over<0>(v, xb, lane);
        else
            y_hand_over<1>(v, xb, lane);
        half_sync(half);  // partner's hand-over visible; staging tile and input tile free
        if (b == 0)
            y_finish<0>(v, xbp, stg, lane, c);
        else
            y_finish<1>(v, xbp, stg, lane, c);
        if (has_next) tile_store(t, sm.tile[half], ht);
        fence_async_smem();  // staging writes -> async proxy
        half_sync(half);     // staging tile complete, next input tile visible, hand-over tiles free
        if (leader) {
#pragma unroll
            for (int j = 0; j < N / YBOX; ++j)
                tma_store_2d(tmB, stg + j * YBOX * 2, 2 * colh, view * N + j * YBOX);
            bulk_commit();
        }
    }
    if (leader) bulk_wait_read();  // shared memory must outlive the last store's reads
    turns_close(turns, warp);
}

// ---- pass x: one row of B per warp pair -----------------------------------------------------------
constexpr int WX = 8;        // warps per CTA
constexpr int XP = WX / 2;   // pairs per CTA = rows in flight per CTA
struct SmemX {
    float2 xb[WX][XB];
    float2 inb[XP][N];  // input row of each pair (bulk async copy destination)
    unsigned long long ibar[XP];
    unsigned tmem;  // base address of the tensor-memory allocation
};

// Work unit = (view, group of XP adjacent rows); a CTA takes a contiguous range of units, so all
// its pairs are always in the same view.  The line length is N = 1024 = the number of columns Nx;
// the number of rows per view ny (a multiple of XP) is a run-time value.  tabX: [2][3][N] per view.
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

__device__ __forceinline__ void pass_x_loop(SmemX &sm, const float2 *Bin, int ny, unsigned tq,
                                            const float2 (&tw)[TWN], float2 *__restrict__ field,
                                            float *__restrict__ inten, unsigned int *vmax,
                                            double *mom, int V) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, pair = warp >> 1;
    const int gpv = ny / XP, lgv = 31 - __clz(gpv);  // units per view; ny is a power of two
    const int units = V * gpv;
    const int u0 = (int)((long long)units * blockIdx.x / gridDim.x);
    const int u1 = (int)((long long)units * (blockIdx.x + 1) / gridDim.x);
    if (u0 >= u1) return;  // CTA-uniform
    float2 *xb = sm.xb[warp];
    const float2 *xbp = sm.xb[warp ^ 1];
    const float2 *in = sm.inb[pair] + lane;
    const int b = warp & 1;
    const bool issuer = b == 0 && lane == 0;
    const int view0 = u0 >> lgv;
    unsigned iphase = 0;
    bool pending = false;  // the pair's input row is already on its way
    // turn-taking of warps w and w + 4 (needs every warp of the CTA to run the same number of
    // lines: XP divides ny)
    static_assert(WX == 8, "turn-taking pairs warps w and w + 4");
    const Turns turns = turns_make(warp, true);
    turns_open(turns, warp);
    for (int u = u0; u < u1; ++u) {
        const int view = u >> lgv, line = (u & (gpv - 1)) * XP + pair;
        const unsigned tpre = tq + (view - view0) * TM_SET;  // pre_b | H_b | conj(post_b)
        const size_t row = (size_t)view * ny + line;
        if (!pending && issuer)
            bulk_load(sm.inb[pair], Bin + row * N, N * sizeof(float2), &sm.ibar[pair]);
        const int nu = u + 1, nline = (nu & (gpv - 1)) * XP + pair;
        const bool has_next = nu < u1;
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
            bulk_load(sm.inb[pair], Bin + ((size_t)(nu >> lgv) * ny + nline) * N, N * sizeof(float2),
                      &sm.ibar[pair]);
        }
        pending = has_next;
        branch(v, lane, xb, tw, tpre + TM_TAB, turns);
        if (b == 0)
            x_finish<0>(v, xb, xbp, lane, pair, field, inten, row * N, mom, vmax, view);
        else
            x_finish<1>(v, xb, xbp, lane, pair, field, inten, row * N, mom, vmax, view);
    }
    turns_close(turns, warp);
}

}  // namespace sfdw
