// sfd_asm2048.cuh — angular-spectrum propagation on a 2048 x 2048 grid (the 2N grid of the hologram
// generator of SURVEY.md §8(d) for N = 1024): the three kernels of sfd_asm1024.cuh with a PAIR of
// warps per line.
//
// A 2048-point transform is one radix-2 step around two 1024-point warp transforms (sfd_asm1024.cuh,
// fft1024), w = exp(-2 pi i / 2048), k, j < 1024:
//
//   decimation in time       warp h transforms x_h[j] = x[2 j + h]:  E = FFT(x_0), O = FFT(x_1)
//   (strided in, halves out) X[k] = E[k] + w^k O[k] (warp 0),  X[k + 1024] = E[k] - w^k O[k] (warp 1)
//   decimation in frequency  warp h holds y_h[k] = y[k + 1024 h]:  e = y_0 + y_1,  o = (y_0 - y_1) w^k
//   (halves in, strided out) Z[2 j] = FFT(e)[j] (warp 0),  Z[2 j + 1] = FFT(o)[j] (warp 1)
//
// Either way each warp needs the other's 32 values per lane once: they cross through the transpose
// tiles, which are idle outside fft1024, between two pair barriers.  w^k for k = lane + 32 r is
// w^lane (one register) times exp(-2 pi i r / 64) (compile-time constants folded into the add).
//
// Rows use the first form (a warp reads every second element of the row and writes one contiguous
// half of the result).  A column uses the second form forward - its halves are rows n and n + 1024 of
// the tile - which leaves the spectrum interleaved, Z[2 j + h] in warp h: exactly what the first form
// wants as input for the inverse transform, whose halves go back to rows n and n + 1024.  The table
// T_p[kx] is stored per warp in that order: [p][kx][h][j] = sigma(j) sigma(kx mod 1024) H_p[2 j + h][kx] / N^2.
//
// Sign tracking as in sfd_asm1024.cuh: both halves of a pair carry sigma(k) of the 1024-point index,
// so the radix-2 steps work on the stored values unchanged and a 2048-point result carries
// sigma(index mod 1024).
#pragma once
#include "sfd_asm1024.cuh"

namespace sfda2 {

using namespace sfda;

constexpr int NL = 2048;       // line length
constexpr int NPAIR = NWA / 2;  // lines a CTA works on at a time

// w^(lane + 32 r) = w^lane * exp(-2 pi i r / 64): one per-lane register (from the plan's table of
// exp(-2 pi i k / 2048)) and compile-time constants, so the radix-2 step reads no table
SFD_CE float cos64(int r) {  // cos(2 pi r / 64), r < 32
    constexpr float C[17] = {1.f, 0.99518472667219688624f, 0.98078528040323044913f, 0.95694033573220886494f,
                             0.92387953251128675613f, 0.88192126434835502971f, 0.83146961230254523708f,
                             0.77301045336273696081f, 0.70710678118654752440f, 0.63439328416364549822f,
                             0.55557023301960222474f, 0.47139673682599764856f, 0.38268343236508977173f,
                             0.29028467725446236764f, 0.19509032201612826785f, 0.09801714032956060199f, 0.f};
    return r <= 16 ? C[r] : -C[32 - r];
}
SFD_CE float sin64(int r) { return r <= 16 ? cos64(16 - r) : cos64(r - 16); }

// e + exp(-2 pi i r / 64) (wd o); wd = w^lane for warp 0, -w^lane for warp 1 (which subtracts): the
// constant factor is folded into the add
__device__ __forceinline__ float2 dit_one(float2 e, float2 o, float2 wd, int r) {
    const float2 t = make_float2(wd.x * o.x - wd.y * o.y, wd.x * o.y + wd.y * o.x);
    return make_float2(fmaf(cos64(r), t.x, fmaf(sin64(r), t.y, e.x)),
                       fmaf(cos64(r), t.y, fmaf(-sin64(r), t.x, e.y)));
}
// v = this warp's 1024-point transform (E for h = 0, O for h = 1), theirs = the partner's, already in
// its tile -> this warp's half of the 2048-point transform (wl = w^lane)
__device__ __forceinline__ void dit_finish(float2 (&v)[32], int h, int lane, const float2 *theirs, float2 wl) {
    if (h == 0) {
#pragma unroll
        for (int r = 0; r < 32; ++r) v[r] = dit_one(v[r], theirs[r * 32 + lane], wl, r);
    } else {
        const float2 wd = make_float2(-wl.x, -wl.y);
#pragma unroll
        for (int r = 0; r < 32; ++r) v[r] = dit_one(theirs[r * 32 + lane], v[r], wd, r);
    }
}
__device__ __forceinline__ void dit_combine(float2 (&v)[32], int h, int lane, int pair, float2 *mine,
                                            const float2 *theirs, float2 wl) {
#pragma unroll
    for (int r = 0; r < 32; ++r) mine[r * 32 + lane] = v[r];
    pair_sync(pair);
    dit_finish(v, h, lane, theirs, wl);
    pair_sync(pair);  // the partner has read this warp's tile before the next transpose writes it
}
// v = this warp's half y_h -> the input of its 1024-point transform (e for h = 0, o for h = 1)
__device__ __forceinline__ void dif_split(float2 (&v)[32], int h, int lane, int pair, float2 *mine,
                                          const float2 *theirs, float2 wl) {
#pragma unroll
    for (int r = 0; r < 32; ++r) mine[r * 32 + lane] = v[r];
    pair_sync(pair);
#pragma unroll
    for (int r = 0; r < 32; ++r) {
        const float2 p = theirs[r * 32 + lane];
        if (h == 0) {
            v[r] = make_float2(v[r].x + p.x, v[r].y + p.y);
        } else {
            const float2 d = make_float2(p.x - v[r].x, p.y - v[r].y);
            const float2 t = make_float2(wl.x * d.x - wl.y * d.y, wl.x * d.y + wl.y * d.x);
            v[r] = make_float2(cos64(r) * t.x + sin64(r) * t.y, cos64(r) * t.y - sin64(r) * t.x);
        }
    }
    pair_sync(pair);
}

struct SmemI2 {
    float2 xb[NWA][XB];
    alignas(128) float2 inb[NPAIR][NL];  // a pair's next row (bulk async copy destination)
    unsigned long long ibar[NPAIR];
};

// rows of u0 -> A~[n][kx] = sigma(kx mod 1024) FFT_x(u0[n][:])[kx]; a pair per row, the pair's next row
// on its way into shared memory while it transforms the current one
template <typename TIn>
__device__ __forceinline__ void rows_fwd(SmemI2 &sm, const TIn *u0, const float2 *__restrict__ twl,
                                         const float2 *__restrict__ w2048, float2 *A, int rows) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, pair = warp >> 1, h = warp & 1;
    const int step = gridDim.x * NPAIR;
    const bool issuer = h == 0 && lane == 0;
    float2 tw[TWN];
    load_twiddles(tw, lane, twl);
    const float2 wl = __ldg(w2048 + lane);
    pdl_wait();  // u0 and A belong to the kernels before this one
    int row = blockIdx.x * NPAIR + pair;
    if (issuer && row < rows)
        bulk_load(sm.inb[pair], u0 + (size_t)row * NL, NL * sizeof(TIn), &sm.ibar[pair]);
    unsigned ph = 0;
    const TIn *in = reinterpret_cast<const TIn *>(sm.inb[pair]);
    for (; row < rows; row += step) {
        mbar_wait(&sm.ibar[pair], ph);
        ph ^= 1;
        float2 v[32];
#pragma unroll
        for (int r = 0; r < 32; ++r) v[r] = sample(in, 2 * (lane + 32 * r) + h);
        fft1024(v, lane, sm.xb[warp], tw);
        float2 *mine = sm.xb[warp];
#pragma unroll
        for (int r = 0; r < 32; ++r) mine[r * 32 + lane] = v[r];
        pair_sync(pair);  // both warps have read the row long ago: the next one may land
        if (issuer && row + step < rows) {
            fence_async_smem();
            bulk_load(sm.inb[pair], u0 + (size_t)(row + step) * NL, NL * sizeof(TIn), &sm.ibar[pair]);
        }
        dit_finish(v, h, lane, sm.xb[warp ^ 1], wl);
        pair_sync(pair);
#pragma unroll
        for (int k = 0; k < 32; ++k) A[(size_t)row * NL + N * h + lane + 32 * k] = v[k];
    }
}

// rows of W~ -> field, intensity, phase; rows = P * 2048.  A pair's next row is on its way into
// shared memory while it transforms the current one.
template <bool PHASE>
__device__ __forceinline__ void rows_inv(SmemI2 &sm, const float2 *W, const float2 *__restrict__ twl,
                                         const float2 *__restrict__ w2048, float2 *__restrict__ field,
                                         float *__restrict__ inten, float *__restrict__ phase, int rows) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, pair = warp >> 1, h = warp & 1;
    const int step = gridDim.x * NPAIR;
    const bool issuer = h == 0 && lane == 0;
    float2 tw[TWN];
    load_twiddles(tw, lane, twl);
    const float2 wl = __ldg(w2048 + lane);
    pdl_wait();
    int row = blockIdx.x * NPAIR + pair;
    if (issuer && row < rows)
        bulk_load(sm.inb[pair], W + (size_t)row * NL, NL * sizeof(float2), &sm.ibar[pair]);
    unsigned ph = 0;
    for (; row < rows; row += step) {
        mbar_wait(&sm.ibar[pair], ph);
        ph ^= 1;
        float2 v[32];
#pragma unroll
        for (int r = 0; r < 32; ++r) v[r] = sm.inb[pair][2 * (lane + 32 * r) + h];
        fft1024(v, lane, sm.xb[warp], tw);
        {   // dit_combine with the next row's copy started behind its first barrier (both warps have
            // read the row by then)
            float2 *mine = sm.xb[warp];
            const float2 *theirs = sm.xb[warp ^ 1];
#pragma unroll
            for (int r = 0; r < 32; ++r) mine[r * 32 + lane] = v[r];
            pair_sync(pair);
            if (issuer && row + step < rows) {
                fence_async_smem();
                bulk_load(sm.inb[pair], W + (size_t)(row + step) * NL, NL * sizeof(float2), &sm.ibar[pair]);
            }
            dit_finish(v, h, lane, theirs, wl);
            pair_sync(pair);
        }
        // u = sigma(m) sigma(n) conj(t), both sigmas of the index modulo 1024
        const float sg = lane_sigma(lane) * ((__popc(row & (N - 1)) & 1) ? -1.f : 1.f);
        const size_t o = (size_t)row * NL + N * h + lane;
#pragma unroll
        for (int k = 0; k < 32; ++k) {
            const float s = sfdb::out_sign(k) > 0 ? sg : -sg;
            const float2 u = make_float2(s * v[k].x, -s * v[k].y);
            if (field) field[o + 32 * k] = u;
            if (inten) inten[o + 32 * k] = u.x * u.x + u.y * u.y;
            if (PHASE) sm.xb[warp][k * 32 + lane] = u;
        }
        // arg u in a ROLLED loop over values parked in the (idle) transpose tile: 32 inlined atan2f are as
        // long as the transform itself and do not fit the instruction cache beside it
        if (PHASE) {
            const float2 *pu = sm.xb[warp] + lane;
#pragma unroll 2
            for (int k = 0; k < 32; ++k) {
                const float2 u = pu[k * 32];
                phase[o + 32 * k] = atan2f(u.y, u.x);
            }
            __syncwarp();  // all lanes have read the tile before the next transpose writes it
        }
    }
}

// ---- columns: 4 adjacent columns per CTA, a pair per column ------------------------------------------
// The tile [2048 rows][4 columns] (32 bytes per row, eight TMA boxes of 256 rows) is moved by a ninth
// warp exactly as in sfd_asm1024.cuh (in_full / in_read / staged / empty, register trade by
// setmaxnreg).  SWIZZLE_32B on both tensor maps: the 16-byte chunk c of row n sits at chunk
// c ^ ((n >> 2) & 1), a column access is 4 shared-memory wavefronts instead of 8.
struct SmemC2 {
    alignas(1024) float2 tile[NL][NPAIR];  // input block, then staging of each plane's results (swizzled)
    alignas(128) float2 tb[NWA][N];        // a warp's next table line T_p[kx][h][:]
    float2 xb[NWA][XB];
    unsigned long long tbar[NWA];
    unsigned long long in_full, in_read, staged, empty;
};

// tmA: tensor map of A~ seen as float [2048][4096], tmW: of W~ seen as float [P * 2048][4096], both
// with box 8 x YBOX and SWIZZLE_32B.  Tt: [P][kx][h][j] (see the top of the file).
__device__ __forceinline__ void cols(SmemC2 &sm, const void *tmA, const void *tmW,
                                     const float2 *__restrict__ Tt, const float2 *__restrict__ twl,
                                     const float2 *__restrict__ w2048, int P) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nblk = NL / NPAIR;
    if (warp >= NWA) {  // the TMA warp
        asm volatile("setmaxnreg.dec.sync.aligned.u32 24;");
        if (warp != NWA || lane != 0) return;
        unsigned ph_read = 0, ph_staged = 0;
        pdl_wait();  // A~ comes from the row kernel; W~ is read by the row kernel of the call before
        for (int blk = blockIdx.x; blk < nblk; blk += gridDim.x) {
            mbar_expect(&sm.in_full, NL * NPAIR * sizeof(float2));
#pragma unroll
            for (int j = 0; j < NL / YBOX; ++j)
                tma_load_2d(tmA, &sm.tile[j * YBOX][0], 2 * NPAIR * blk, j * YBOX, &sm.in_full);
            mbar_wait(&sm.in_read, ph_read);
            ph_read ^= 1;
            mbar_arrive(&sm.empty);
            for (int p = 0; p < P; ++p) {
                mbar_wait(&sm.staged, ph_staged);
                ph_staged ^= 1;
#pragma unroll
                for (int j = 0; j < NL / YBOX; ++j)
                    tma_store_2d(tmW, &sm.tile[j * YBOX][0], 2 * NPAIR * blk, p * NL + j * YBOX);
                bulk_commit();
                bulk_wait_read();  // the tile has been read: free for the next plane / the next block
                if (p + 1 < P) mbar_arrive(&sm.empty);
            }
        }
        return;
    }
    asm volatile("setmaxnreg.inc.sync.aligned.u32 240;");
    const int pair = warp >> 1, h = warp & 1;
    float2 tw[TWN];
    load_twiddles(tw, lane, twl);
    const float2 wl = __ldg(w2048 + lane);
    if (lane == 0 && (int)blockIdx.x < nblk)
        bulk_load(sm.tb[warp], Tt + ((size_t)(NPAIR * blockIdx.x + pair) * 2 + h) * N, N * sizeof(float2),
                  &sm.tbar[warp]);
    unsigned ph_full = 0, ph_empty = 0, tphase = 0;
    // this warp's half column inside the swizzled tile: element (row lane + 32 r + 1024 h, column pair)
    float2 *mine = &sm.tile[lane + N * h][0] + 2 * ((pair >> 1) ^ ((lane >> 2) & 1)) + (pair & 1);
    float2 *xb = sm.xb[warp];
    const float2 *xbp = sm.xb[warp ^ 1];
    for (int blk = blockIdx.x; blk < nblk; blk += gridDim.x) {
        const int col = NPAIR * blk + pair;
        // transform 0: the column forward (decimation in frequency: halves in, Z[2 j + h] out, kept);
        // transform 1 + p: the inverse one of plane p (decimation in time: Z[2 j + h] in, halves out)
        float2 v[32], a[32];
#pragma unroll 1
        for (int t = 0; t <= P; ++t) {
            const int p = t - 1;
            if (t == 0) {
                mbar_wait(&sm.in_full, ph_full);
                ph_full ^= 1;
#pragma unroll
                for (int r = 0; r < 32; ++r) v[r] = mine[32 * NPAIR * r];
                __syncwarp();
                if (lane == 0) mbar_arrive(&sm.in_read);
                dif_split(v, h, lane, pair, xb, xbp, wl);
            } else {
                mbar_wait(&sm.tbar[warp], tphase);
                tphase ^= 1;
#pragma unroll
                for (int k = 0; k < 32; ++k) v[k] = sm.tb[warp][lane + 32 * k];
                __syncwarp();
                if (lane == 0) {  // the next table line of this warp: next plane, or plane 0 of the next block
                    const bool more = p + 1 < P;
                    if (more || blk + (int)gridDim.x < nblk) {
                        const size_t line = more ? ((size_t)(p + 1) * NL + col) * 2 + h
                                                 : (size_t)(NPAIR * (blk + gridDim.x) + pair) * 2 + h;
                        fence_async_smem();
                        bulk_load(sm.tb[warp], Tt + line * N, N * sizeof(float2), &sm.tbar[warp]);
                    }
                }
#pragma unroll
                for (int k = 0; k < 32; ++k)  // conj(a T)
                    v[k] = make_float2(a[k].x * v[k].x - a[k].y * v[k].y,
                                       -(a[k].x * v[k].y) - a[k].y * v[k].x);
            }
            fft1024(v, lane, xb, tw);
            if (t == 0) {
#pragma unroll
                for (int k = 0; k < 32; ++k) a[k] = v[k];
                continue;
            }
            dit_combine(v, h, lane, pair, xb, xbp, wl);
            mbar_wait(&sm.empty, ph_empty);  // everybody has read the input / the store before has left
            ph_empty ^= 1;
#pragma unroll
            for (int k = 0; k < 32; ++k) mine[32 * NPAIR * k] = v[k];
            fence_async_smem();  // staging writes -> async proxy
            __syncwarp();
            if (lane == 0) mbar_arrive(&sm.staged);
        }
    }
}

}  // namespace sfda2
