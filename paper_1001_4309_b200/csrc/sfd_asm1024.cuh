// sfd_asm1024.cuh — angular-spectrum propagation on a 1024 x 1024 grid with the warp FFT of the
// Shifted-Fresnel fast path (the generic line-FFT kernels of sfd_asm.cu serve
// every other size).
//
//     u(z_p) = IFFT2[ FFT2[u0] * H_p ]                                   (sfd_asm.cu, include/sfd.h)
//
// A 1024-point line is one warp: 32 lanes x 32 complex registers, two radix-32 register butterflies
// (sfd_dft32.cuh) around one 32 x 32 transpose through a private shared-memory tile.  Element
// i = lane + 32 r of a line sits in register r of lane `lane` on the way in, and frequency
// k = lane + 32 r in the same place on the way out, so transforms chain without any reordering.
//
// Sign tracking.  The butterflies leave stored[k] = sigma(k) X[k], sigma(k) = (-1)^popcount(k) (sign
// tracking of sfd_dft32.cuh: popcount of the lane bits after stage A, of the register bits after stage
// B).  No kernel here undoes it on its own output; the signs travel with the data and cancel where a
// table or the final store touches every element anyway:
//
//   k_asm1024_rows_fwd  per row n:      A~[n][kx]  = sigma(kx) FFT_x(u0[n][:])[kx]
//   k_asm1024_cols      per column kx:  a = fft(A~[:][kx])       = sigma(ky) sigma(kx) FFT2(u0)[ky][kx]
//                       per plane p:    w = conj(a * T_p[kx][ky]),  T_p = sigma(ky) sigma(kx) H_p[ky][kx] / N^2
//                                       W~[p][n][kx] = fft(w)[n] = sigma(n) conj(c_p[n][kx]),
//                                       c_p = IFFT_y(FFT2(u0) H_p)  (inverse as conj(FFT(conj(.))))
//   k_asm1024_rows_inv  per row n:      t = fft(W~[p][n][:]) = sigma(m) sigma(n) conj(u_p[n][m])
//                                       u_p[n][m] = sigma(m) sigma(n) conj(t[m])  -> field, |u|^2, arg u
//
// The table T_p is the plan's transfer function stored TRANSPOSED ([p][kx][ky], a column of H is a
// contiguous line) with the signs and the 1/N^2 of the two inverse transforms folded in at plan time.
// The column kernel transforms a column forward ONCE and keeps the spectrum in registers for all
// planes of the plan (1 + P transforms per column instead of 2 P).
//
// Memory paths.  Rows are read and written by plain coalesced 8-byte accesses (a warp instruction
// covers 256 contiguous bytes).  A column is one element per row: the 8 transform warps of a CTA take 8
// adjacent columns and a ninth warp has the TMA unit move their [1024 rows][8 columns] tile between
// global and shared memory in both directions (see `cols` below).  The tile the CTA received its
// input in is its staging tile on the way out: the store of plane p runs beside the transform of plane
// p + 1 and has long left the tile when that one's results arrive.  Whatever a warp reads next from
// global memory - its next row, its next line of T - is on its way into shared memory as a bulk async
// copy while it transforms.  No CTA-wide barrier exists in the loops.
#pragma once
#include "sfd_warp1024.cuh"

namespace sfda {

using namespace sfdw;

constexpr int NWA = 8;  // warps per CTA of all three kernels

// sigma of the lane part of an index (the register part is sfdb::out_sign, a compile-time constant)
__device__ __forceinline__ float lane_sigma(int lane) { return (__popc(lane) & 1) ? -1.f : 1.f; }

// forward 1024-point FFT of a warp: v[r] = x[lane + 32 r] -> v[k] = sigma(lane + 32 k) X[lane + 32 k]
__device__ __forceinline__ void fft1024(float2 (&v)[32], int lane, float2 *xb, const float2 (&tw)[TWN]) {
    sfdb::dft32(v);
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
    sfdb::dft32_tw(v, tw);
}

// 2-D tiled bulk load global -> shared through tensor map `tm` (box fixed by the map), completing on
// `bar` (the caller has armed it with the byte count)
__device__ __forceinline__ void tma_load_2d(const void *tm, void *dst, int c0, int c1,
                                            unsigned long long *bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::
            "r"(smem_u32(dst)), "l"(tm), "r"(c0), "r"(c1), "r"(smem_u32(bar))
        : "memory");
}
__device__ __forceinline__ void mbar_expect(unsigned long long *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}

__device__ __forceinline__ float2 sample(const float *p, size_t i) { return make_float2(p[i], 0.f); }
__device__ __forceinline__ float2 sample(const float2 *p, size_t i) { return p[i]; }

struct SmemR {
    float2 xb[NWA][XB];
};

// rows of u0 -> A~ (row spectra, signs left in)
template <typename TIn>
__device__ __forceinline__ void rows_fwd(SmemR &sm, const TIn *u0, const float2 *__restrict__ twl,
                                         float2 *A, int rows) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float2 tw[TWN];
    load_twiddles(tw, lane, twl);  // plan constant
    pdl_wait();  // u0 and A belong to the kernels before this one
    for (int row = blockIdx.x * NWA + warp; row < rows; row += gridDim.x * NWA) {
        float2 v[32];
#pragma unroll
        for (int r = 0; r < 32; ++r) v[r] = sample(u0, (size_t)row * N + lane + 32 * r);
        fft1024(v, lane, sm.xb[warp], tw);
#pragma unroll
        for (int k = 0; k < 32; ++k) A[(size_t)row * N + lane + 32 * k] = v[k];
    }
}

struct SmemI {
    float2 xb[NWA][XB];
    alignas(128) float2 inb[NWA][N];  // a warp's next row (bulk async copy destination)
    unsigned long long ibar[NWA];
};

// rows of W~ -> field, intensity, phase.  rows = P * 1024; row L belongs to plane L / 1024.  A warp's
// next row is on its way into shared memory (bulk async copy) while it transforms the current one.
template <bool PHASE>
__device__ __forceinline__ void rows_inv(SmemI &sm, const float2 *W, const float2 *__restrict__ twl,
                                         float2 *__restrict__ field, float *__restrict__ inten,
                                         float *__restrict__ phase, int rows) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int step = gridDim.x * NWA;
    float2 tw[TWN];
    load_twiddles(tw, lane, twl);
    pdl_wait();
    int row = blockIdx.x * NWA + warp;
    if (lane == 0 && row < rows)
        bulk_load(sm.inb[warp], W + (size_t)row * N, N * sizeof(float2), &sm.ibar[warp]);
    unsigned ph = 0;
    for (; row < rows; row += step) {
        mbar_wait(&sm.ibar[warp], ph);
        ph ^= 1;
        float2 v[32];
#pragma unroll
        for (int r = 0; r < 32; ++r) v[r] = sm.inb[warp][lane + 32 * r];
        __syncwarp();
        if (lane == 0 && row + step < rows) {
            fence_async_smem();
            bulk_load(sm.inb[warp], W + (size_t)(row + step) * N, N * sizeof(float2), &sm.ibar[warp]);
        }
        fft1024(v, lane, sm.xb[warp], tw);
        // u = sigma(m) sigma(n) conj(t): sigma(n) of the row and sigma of the lane part of m at run
        // time, the register part of m at compile time
        const float sg = lane_sigma(lane) * ((__popc(row & (N - 1)) & 1) ? -1.f : 1.f);
        const size_t o = (size_t)row * N + lane;
#pragma unroll
        for (int k = 0; k < 32; ++k) {
            const float s = sfdb::out_sign(k) > 0 ? sg : -sg;
            const float2 u = make_float2(s * v[k].x, -s * v[k].y);
            if (field) field[o + 32 * k] = u;
            if (inten) inten[o + 32 * k] = u.x * u.x + u.y * u.y;
            if (PHASE) phase[o + 32 * k] = atan2f(u.y, u.x);
        }
    }
}

// ---- columns ---------------------------------------------------------------------------------------
// A CTA works on blocks of 8 adjacent columns, one per transform warp, and moves them as ONE tile
// [1024 rows][8 columns] (64 bytes per row, four TMA boxes of 256 rows): the TMA unit spends about a
// cycle per box row whatever its width (measured: 2.4 us to load or store the same block as four
// tiles of 16-byte rows, which made the unit - not the butterflies - the bound of this kernel), so
// rows are made as wide as the CTA has columns.  A ninth warp owns the tile traffic; the transform
// warps never wait for one another, only for the tile:
//
//   TMA warp (one thread)                               transform warp w (column 8 blk + w)
//   load the block's tile                  -> in_full -> read column w of the tile, arrive in_read
//   wait in_read (8 arrivals), arrive empty             forward transform, keep the spectrum
//   per plane: wait staged (8 arrivals),                per plane: multiply by T_p, transform,
//              store the tile, wait until it has        wait empty, write column w into the tile,
//              been read, arrive empty                  arrive staged
//
// The tile is SWIZZLE_64B on both tensor maps: the 16-byte chunk c of row n sits at chunk
// c ^ ((n >> 1) & 3), which spreads a column (one 8-byte element per row) over 8 of the 16 bank pairs
// instead of 2 (4 wavefronts per warp access instead of 16; 2 would be the ideal).
// Registers: a transform warp keeps two lines and the twiddles (about 230 registers), the TMA thread
// needs a handful.  A sub-partition's register file holds 512 per lane, and warps are given theirs in
// fours (one per sub-partition), so the CTA is launched as three groups of four warps at 168 registers
// and the groups then trade (setmaxnreg): the third group - the TMA warp and three warps that exit -
// drops to 24, the two transform groups rise to 240.
constexpr int NTC = 32 * (NWA + 4);  // threads per CTA of the column kernel
struct SmemC {
    alignas(1024) float2 tile[N][NWA];  // input block, then staging of each plane's results (swizzled)
    alignas(128) float2 tb[NWA][N];     // a warp's next table line T_p[kx][:]
    float2 xb[NWA][XB];
    unsigned long long tbar[NWA];       // a warp's table line has landed
    unsigned long long in_full, in_read, staged, empty;
};
__device__ __forceinline__ void mbar_arrive(unsigned long long *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// tmA: tensor map of A~ seen as float [1024][2048], tmW: of W~ seen as float [P * 1024][2048], both
// with box 16 x YBOX and SWIZZLE_64B.  Tt: [P][kx][ky] (see the top of the file); the line a warp
// multiplies by next is fetched into shared memory (bulk async copy) a transform ahead - the first one
// before the kernel waits for the row pass, it is a plan constant.
__device__ __forceinline__ void cols(SmemC &sm, const void *tmA, const void *tmW,
                                     const float2 *__restrict__ Tt, const float2 *__restrict__ twl,
                                     int P) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nblk = N / NWA;
    if (warp >= NWA) {  // the TMA warp
        asm volatile("setmaxnreg.dec.sync.aligned.u32 24;");
        if (warp != NWA || lane != 0) return;
        unsigned ph_read = 0, ph_staged = 0;
        pdl_wait();  // A~ comes from the row kernel; W~ is read by the row kernel of the call before
        for (int blk = blockIdx.x; blk < nblk; blk += gridDim.x) {
            mbar_expect(&sm.in_full, N * NWA * sizeof(float2));
#pragma unroll
            for (int j = 0; j < N / YBOX; ++j)
                tma_load_2d(tmA, &sm.tile[j * YBOX][0], 2 * NWA * blk, j * YBOX, &sm.in_full);
            mbar_wait(&sm.in_read, ph_read);
            ph_read ^= 1;
            mbar_arrive(&sm.empty);
            for (int p = 0; p < P; ++p) {
                mbar_wait(&sm.staged, ph_staged);
                ph_staged ^= 1;
#pragma unroll
                for (int j = 0; j < N / YBOX; ++j)
                    tma_store_2d(tmW, &sm.tile[j * YBOX][0], 2 * NWA * blk, p * N + j * YBOX);
                bulk_commit();
                bulk_wait_read();  // the tile has been read: free for the next plane / the next block
                if (p + 1 < P) mbar_arrive(&sm.empty);
            }
        }
        return;
    }
    asm volatile("setmaxnreg.inc.sync.aligned.u32 240;");
    float2 tw[TWN];
    load_twiddles(tw, lane, twl);
    if (lane == 0 && (int)blockIdx.x < nblk)
        bulk_load(sm.tb[warp], Tt + (size_t)(NWA * blockIdx.x + warp) * N, N * sizeof(float2), &sm.tbar[warp]);
    unsigned ph_full = 0, ph_empty = 0, tphase = 0;
    // this warp's column inside the swizzled tile: element (row lane + 32 r, column warp)
    float2 *mine = &sm.tile[lane][0] + 2 * ((warp >> 1) ^ ((lane >> 1) & 3)) + (warp & 1);
    for (int blk = blockIdx.x; blk < nblk; blk += gridDim.x) {
        const int col = NWA * blk + warp;
        // transform 0 is the forward one of the column (tile -> spectrum a, kept for all planes),
        // transform 1 + p the inverse one of plane p; one loop so that the code of a transform exists
        // once (two copies do not fit the instruction cache)
        float2 v[32], a[32];
#pragma unroll 1
        for (int t = 0; t <= P; ++t) {
            const int p = t - 1;
            if (t == 0) {
                mbar_wait(&sm.in_full, ph_full);
                ph_full ^= 1;
#pragma unroll
                for (int r = 0; r < 32; ++r) v[r] = mine[32 * NWA * r];
                __syncwarp();
                if (lane == 0) mbar_arrive(&sm.in_read);
            } else {
                mbar_wait(&sm.tbar[warp], tphase);
                tphase ^= 1;
#pragma unroll
                for (int k = 0; k < 32; ++k) v[k] = sm.tb[warp][lane + 32 * k];
                __syncwarp();
                if (lane == 0) {  // the next table line of this warp: next plane, or plane 0 of the next block
                    const bool more = p + 1 < P;
                    if (more || blk + (int)gridDim.x < nblk) {
                        const size_t line = more ? (size_t)(p + 1) * N + col
                                                 : (size_t)(NWA * (blk + gridDim.x) + warp);
                        fence_async_smem();
                        bulk_load(sm.tb[warp], Tt + line * N, N * sizeof(float2), &sm.tbar[warp]);
                    }
                }
#pragma unroll
                for (int k = 0; k < 32; ++k)  // conj(a T)
                    v[k] = make_float2(a[k].x * v[k].x - a[k].y * v[k].y,
                                       -(a[k].x * v[k].y) - a[k].y * v[k].x);
            }
            fft1024(v, lane, sm.xb[warp], tw);
            if (t == 0) {
#pragma unroll
                for (int k = 0; k < 32; ++k) a[k] = v[k];
                continue;
            }
            mbar_wait(&sm.empty, ph_empty);  // everybody has read the input / the store before has left
            ph_empty ^= 1;
#pragma unroll
            for (int k = 0; k < 32; ++k) mine[32 * NWA * k] = v[k];
            fence_async_smem();  // staging writes -> async proxy
            __syncwarp();
            if (lane == 0) mbar_arrive(&sm.staged);
        }
    }
}

}  // namespace sfda
