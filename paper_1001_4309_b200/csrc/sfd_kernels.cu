// sfd_kernels.cu — the sm_100a kernels of libsfd and their launcher.
//
// A reconstruction (PAPER.md steps (ii)-(x), L86-94) is two kernels for all views at once:
//   k_pass_y : grid (N/C, V); per CTA C hologram columns: u8/f32 -> float, x pre_y (Eq. 3), zero-pad,
//              2N-point FFT, x H, inverse FFT, crop, x c0 post_y (Eq. 2) -> B[V][N][N]
//   k_pass_x : grid (N/RPC, V); per CTA RPC rows of B: x pre_x, FFT, x H, inverse FFT, crop, x post_x
//              -> field, |.|^2 -> intensity (Eq. 5), optional per-view max
// plus, in the 8-bit mode (step (xi), reading 15), k_quantise.
// The per-thread arithmetic lives in sfd_fft_core.cuh.  For N = 1024 and N = 2048 the same two passes
// run as the persistent warp-per-branch kernels k_cols_1024 / k_rows_1024 (a warp pair per line,
// sfd_warp1024.cuh) and k_cols_2048 / k_rows_2048 (a quad of warps per line, sfd_warp2048.cuh).
#include <cuda.h>  // CUtensorMap (types only: the encoder is fetched through the runtime)

#include <atomic>
#include <cmath>
#include <cstdio>
#include <mutex>
#include <vector>

#include "sfd_fft_core.cuh"
#include "sfd_internal.h"
#include "sfd_warp1024.cuh"
#include "sfd_warp2048.cuh"
#include "sfd_warp512.cuh"

namespace {

using namespace sfd;

// tables of one axis as the generic kernels see them: view v at base + v * vstride
struct AxisTabs {
    const float2 *base;
    long long vstride;
    int pre, H, post;  // offsets inside a view's block
};

// The generic kernels read plan constants (FFT twiddles, H, pre, post) where they use them, every first
// touch a trip to L2 on the critical path of a CTA of eight warps.  Up to M = 1024 the CTA copies them
// into shared memory first - before it waits for the kernel in front of it: they are plan constants -
// and the line code reads them with plain loads (sfd::tables_staged, sfd::tab_ld).  Measured, 4 views,
// uint8 in, frames replayed from a CUDA graph: N = 128 6.7 -> 5.1 us, N = 256 11.0 -> 10.3 us per frame.
template <int LOG2M> struct Staged {
    static constexpr bool ON = tables_staged(LOG2M);
    const float2 *tw, *H, *pre, *post;
    __device__ __forceinline__ Staged(const float2 *tw_, const float2 *H_, const float2 *pre_, const float2 *post_)
        : tw(tw_), H(H_), pre(pre_), post(post_) {
        if constexpr (ON) {
            constexpr int M = Sched<LOG2M>::M, N = Sched<LOG2M>::N;
            __shared__ float4 st[3 * M / 2];  // tw[M] | H[M] | pre[N] | post[N]
            const float4 *a = reinterpret_cast<const float4 *>(tw_), *b = reinterpret_cast<const float4 *>(H_);
            const float4 *c = reinterpret_cast<const float4 *>(pre_), *d = reinterpret_cast<const float4 *>(post_);
            for (int i = threadIdx.x; i < M / 2; i += blockDim.x) {
                st[i] = __ldg(a + i);
                st[M / 2 + i] = __ldg(b + i);
            }
            for (int i = threadIdx.x; i < N / 2; i += blockDim.x) {
                st[M + i] = __ldg(c + i);
                st[M + N / 2 + i] = __ldg(d + i);
            }
            __syncthreads();
            const float2 *s2 = reinterpret_cast<const float2 *>(st);
            tw = s2; H = s2 + M; pre = s2 + 2 * M; post = s2 + 2 * M + N;
        }
    }
};

template <int LOG2M, typename TIn>
__global__ void __launch_bounds__(Tile<LOG2M>::THREADS_Y)
k_pass_y(const TIn *holo, long long hstride, int nx, AxisTabs t, const float2 *__restrict__ tw,
         float2 *B, unsigned int *vmax, double *mom) {
    extern __shared__ float2 smem[];
    sfdw::pdl_launch_dependents();
    const int view = blockIdx.y;
    const float2 *tv = t.base + (size_t)view * t.vstride;
    const Staged<LOG2M> sg(tw, tv + t.H, tv + t.pre, tv + t.post);
    sfdw::pdl_wait();  // the hologram, B, vmax and mom belong to the kernels before this one
    if (vmax != nullptr && blockIdx.x == 0 && threadIdx.x == 0) vmax[view] = 0u;
    if (mom != nullptr && blockIdx.x == 0 && threadIdx.x < 2) mom[2 * view + threadIdx.x] = 0.0;
    pass_y_body<LOG2M, Tile<LOG2M>::C, TIn>(threadIdx.x, blockIdx.x, smem, holo, hstride, nx,
                                            sg.pre, sg.H, sg.post, sg.tw,
                                            B + (size_t)view * Sched<LOG2M>::N * nx,
                                            [] { __syncthreads(); });
}

template <int LOG2M, bool MOM>
__global__ void __launch_bounds__(Tile<LOG2M>::THREADS_X)
k_pass_x(const float2 *B, int ny, AxisTabs t, const float2 *__restrict__ tw,
         float2 *__restrict__ field, float *__restrict__ inten, unsigned int *vmax, double *mom) {
    extern __shared__ float2 smem[];
    sfdw::pdl_launch_dependents();
    const int view = blockIdx.y;
    const float2 *tv = t.base + (size_t)view * t.vstride;
    const Staged<LOG2M> sg(tw, tv + t.H, tv + t.pre, tv + t.post);
    sfdw::pdl_wait();  // B (and vmax, mom) come from pass y
    const size_t voff = (size_t)view * ny * Sched<LOG2M>::N;
    float s1 = 0.f, s2 = 0.f;
    float mx = pass_x_body<LOG2M, Tile<LOG2M>::RPC, MOM>(
        threadIdx.x, blockIdx.x, smem, B + voff, sg.pre, sg.H, sg.post, sg.tw,
        field ? field + voff : nullptr, inten ? inten + voff : nullptr, [] { __syncthreads(); }, s1,
        s2);
    if (MOM) {  // focus moments: warp sums in float, accumulation across warps in double
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            s1 += __shfl_xor_sync(0xffffffffu, s1, o);
            s2 += __shfl_xor_sync(0xffffffffu, s2, o);
        }
        if ((threadIdx.x & 31) == 0) {
            atomicAdd(mom + 2 * view, (double)s1);
            atomicAdd(mom + 2 * view + 1, (double)s2);
        }
    }
    if (vmax != nullptr) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        // intensities are >= 0, so their float bit patterns order like unsigned integers
        if ((threadIdx.x & 31) == 0) atomicMax(vmax + view, __float_as_uint(mx));
    }
}

// I8 = round_half_even(255 I / max I) per view (reading 15); 4 pixels per thread.  Launched with
// programmatic stream serialization behind pass x: the per-view maxima are complete only when the
// whole of pass x is, hence a kernel of its own; the intensities it reads were just written and sit
// in L2.
__global__ void __launch_bounds__(256)
k_quantise(const float4 *inten, const unsigned int *vmax, uchar4 *__restrict__ out,
           int quads_per_view) {
    sfdw::pdl_launch_dependents();
    sfdw::pdl_wait();
    const int v = blockIdx.y;
    const float mx = __uint_as_float(vmax[v]);
    const float sc = mx > 0.f ? 255.f / mx : 0.f;
    const size_t base = (size_t)v * quads_per_view;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < quads_per_view;
         i += gridDim.x * blockDim.x) {
        const float4 I = inten[base + i];
        uchar4 o;
        o.x = (unsigned char)min(__float2int_rn(I.x * sc), 255);
        o.y = (unsigned char)min(__float2int_rn(I.y * sc), 255);
        o.z = (unsigned char)min(__float2int_rn(I.z * sc), 255);
        o.w = (unsigned char)min(__float2int_rn(I.w * sc), 255);
        out[base + i] = o;
    }
}

// ---- axis length 1024 (sfd_warp1024.cuh): persistent kernels ------------------------------------------
// One CTA per SM.  k_cols_1024: Ny = 1024 rows, nx columns (lines); grid = V * cpv, CTA c works on
// view c / cpv (solo and split rounds, see pass_y_loop).  k_rows_1024: Nx = 1024 columns, ny rows
// (lines), a warp pair per line, even warps branch 0 (even bins), odd warps branch 1.
template <typename TIn>
__global__ void __launch_bounds__(256, 1)
k_cols_1024(const TIn *holo, long long hstride, int nx, const float2 *__restrict__ tabY,
            long long vstride, const float2 *__restrict__ twl,
            const __grid_constant__ CUtensorMap tmB, unsigned int *vmax, double *mom, int V,
            int cpv) {
    extern __shared__ float4 smem4[];
    using SM = sfdw::SmemY<TIn>;
    SM &sm = *reinterpret_cast<SM *>(smem4);
    sfdw::pdl_launch_dependents();
    if (threadIdx.x == 0) {
        for (int i = 0; i < 2; ++i) {
            sfdw::mbar_init(&sm.full[i], 8);
            sfdw::mbar_init(&sm.empty[i], 8);
        }
        sfdw::mbar_fence_init();
    }
    const int view = blockIdx.x / cpv;
    const sfdw::YPlan yp = sfdw::YPlan::make(nx, blockIdx.x % cpv, cpv);
    if (yp.rounds() > 0) {
        // pull the first slab of this CTA towards L2 while the prologue runs (a prefetch reads nothing:
        // it may precede griddepcontrol.wait)
        const TIn *p0 = holo + (yp.col(0) & ~7);
        for (int r = threadIdx.x; r < sfdw::N; r += blockDim.x)
            asm volatile("prefetch.global.L2 [%0];" ::"l"(p0 + (size_t)r * hstride));
    }
    // tables of both branches of this CTA's view -> tensor memory
    const unsigned tbase = sfdw::tm_setup_both(&sm.tmem, tabY, vstride, view, twl);
    const unsigned tq = sfdw::tm_quarter(tbase, threadIdx.x >> 5);
    // everything above touches plan constants only.  B, vmax and mom belong to the kernels before
    // this one in the stream: the threads that write them wait for those kernels first - block 0 here
    // (8-bit and focus modes only), the store leaders in front of their first store of B
    if ((vmax != nullptr || mom != nullptr) && blockIdx.x == 0) {
        sfdw::pdl_wait();
        if (vmax != nullptr)
            for (int i = threadIdx.x; i < V; i += blockDim.x) vmax[i] = 0u;
        if (mom != nullptr)
            for (int i = threadIdx.x; i < 2 * V; i += blockDim.x) mom[i] = 0.0;
    }
    sfdw::pass_y_loop<TIn>(sm, holo, hstride, nx, tq, tq + sfdw::TM_TW, &tmB, view, yp);
    sfdw::tm_finish(tbase);
}

__global__ void __launch_bounds__(sfdw::NWX * 32, 1)
k_rows_1024(const float2 *B, int ny, const float2 *__restrict__ tabX, long long vstride,
            const float2 *__restrict__ twl, float2 *__restrict__ field, float *__restrict__ inten,
            unsigned int *vmax, double *mom, int V) {
    extern __shared__ float4 smem4[];
    using SM = sfdw::SmemX<sfdw::NWX>;
    SM &sm = *reinterpret_cast<SM *>(smem4);
    sfdw::pdl_launch_dependents();
    if (threadIdx.x == 0) {
        for (int i = 0; i < sfdw::NWX / 2; ++i) sfdw::mbar_init(&sm.ibar[i], 1);
        for (int i = 0; i < sfdw::NWX; ++i) sfdw::mbar_init(&sm.tbar[i], 1);
        sfdw::mbar_fence_init();
    }
    const unsigned tbase = sfdw::tm_setup<sfdw::NWX>(&sm.tmem, tabX, vstride, V * ny, ny, twl);
    const unsigned tq = sfdw::tm_quarter(tbase, threadIdx.x >> 5);
    sfdw::pdl_wait();  // B (and vmax, mom) come from pass y
    sfdw::pass_x_loop<sfdw::NWX, true>(sm, B, ny, tq, tq + sfdw::TM_TW, field, inten, vmax, mom, V);
    sfdw::tm_finish(tbase);
}

// ---- axis length 512 (sfd_warp512.cuh): one warp per line, no branch split ---------------------------
template <typename TIn>
__global__ void __launch_bounds__(256, 1)
k_cols_512(const TIn *holo, long long hstride, int nx, const float2 *__restrict__ tabY,
           long long vstride, const float2 *__restrict__ twl, const __grid_constant__ CUtensorMap tmB,
           unsigned int *vmax, double *mom, int V) {
    extern __shared__ float4 smem4[];
    sfdh::SmemYH<TIn> &sm = *reinterpret_cast<sfdh::SmemYH<TIn> *>(smem4);
    sfdw::pdl_launch_dependents();
    if (threadIdx.x == 0) {
        for (int i = 0; i < 2; ++i) {
            sfdw::mbar_init(&sm.full[i], 8);
            sfdw::mbar_init(&sm.empty[i], 8);
        }
        sfdw::mbar_fence_init();
    }
    const int ipv = nx >> 3;  // items (8 columns) per view, as in pass_y_half
    const unsigned tbase = sfdh::tmh_setup(&sm.tmem, tabY, vstride, V * ipv, ipv, twl);
    const unsigned tq = sfdw::tm_quarter(tbase, threadIdx.x >> 5);
    // B, vmax and mom belong to the kernels before this one: block 0 waits before it clears the latter
    // two, the store leaders wait in front of their first store of B (as in k_cols_1024)
    if ((vmax != nullptr || mom != nullptr) && blockIdx.x == 0) {
        sfdw::pdl_wait();
        if (vmax != nullptr)
            for (int i = threadIdx.x; i < V; i += blockDim.x) vmax[i] = 0u;
        if (mom != nullptr)
            for (int i = threadIdx.x; i < 2 * V; i += blockDim.x) mom[i] = 0.0;
    }
    sfdh::pass_y_half<TIn>(sm, holo, hstride, nx, tq, &tmB, V);
    sfdw::tm_finish(tbase);
}

__global__ void __launch_bounds__(256, 1)
k_rows_512(const float2 *B, int ny, const float2 *__restrict__ tabX, long long vstride,
           const float2 *__restrict__ twl, float2 *__restrict__ field, float *__restrict__ inten,
           unsigned int *vmax, double *mom, int V) {
    extern __shared__ float4 smem4[];
    sfdh::SmemXH &sm = *reinterpret_cast<sfdh::SmemXH *>(smem4);
    sfdw::pdl_launch_dependents();
    if (threadIdx.x == 0) {
        for (int i = 0; i < 8; ++i) sfdw::mbar_init(&sm.ibar[i], 1);
        sfdw::mbar_fence_init();
    }
    const unsigned tbase = sfdh::tmh_setup(&sm.tmem, tabX, vstride, V * ny, ny, twl);
    const unsigned tq = sfdw::tm_quarter(tbase, threadIdx.x >> 5);
    sfdw::pdl_wait();  // B (and vmax, mom) come from pass y
    sfdh::pass_x_half(sm, B, ny, tq, field, inten, vmax, mom, V);
    sfdw::tm_finish(tbase);
}

// ---- axis length 2048 (sfd_warp2048.cuh): four branches per line, a quad of warps per line ----------
// One CTA per SM (at least V); a CTA's range of work units may cross into the next view once
// (sfdq::Span).  tab: [4][5][1024] per view.
template <typename TIn>
__global__ void __launch_bounds__(256, 1)
k_cols_2048(const TIn *holo, long long hstride, int nx, const float2 *__restrict__ tabY,
            long long vstride, const float2 *__restrict__ twl,
            const __grid_constant__ CUtensorMap tmB, unsigned int *vmax, double *mom, int V) {
    extern __shared__ float4 smem4[];
    sfdq::SmemYQ<TIn> &sm = *reinterpret_cast<sfdq::SmemYQ<TIn> *>(smem4);
    sfdw::pdl_launch_dependents();
    if (threadIdx.x == 0) {
        sfdw::mbar_init(&sm.full, 8);
        sfdw::mbar_init(&sm.empty, 8);
        sfdw::mbar_fence_init();
    }
    const sfdq::Span span = sfdq::cta_span(V, nx / 4);
    const unsigned tbase = sfdq::tmq_setup(&sm.tmem, tabY, vstride, span.first_view(), twl);
    const unsigned tq = sfdw::tm_quarter(tbase, threadIdx.x >> 5);
    sfdw::pdl_wait();
    if (vmax != nullptr && blockIdx.x == 0)
        for (int i = threadIdx.x; i < V; i += blockDim.x) vmax[i] = 0u;
    if (mom != nullptr && blockIdx.x == 0)
        for (int i = threadIdx.x; i < 2 * V; i += blockDim.x) mom[i] = 0.0;
    unsigned ph_full = 0, ph_empty = 0;  // parities of the slab barriers, carried across segments
    for (int s = 0; s < 2; ++s) {
        const sfdq::Range rg = span.segment(s);
        if (rg.u0 >= rg.u1) break;
        if (s == 1) sfdq::tmq_refill(tbase, tabY, vstride, rg.view);
        sfdq::pass_y_quad<TIn>(sm, holo, hstride, tq, tq + sfdq::TQ_TW, &tmB, rg, ph_full, ph_empty);
    }
    sfdw::tm_finish(tbase);
}

__global__ void __launch_bounds__(256, 1)
k_rows_2048(const float2 *B, int ny, const float2 *__restrict__ tabX, long long vstride,
            const float2 *__restrict__ twl, float2 *__restrict__ field, float *__restrict__ inten,
            unsigned int *vmax, double *mom, int V) {
    extern __shared__ float4 smem4[];
    sfdq::SmemXQ &sm = *reinterpret_cast<sfdq::SmemXQ *>(smem4);
    sfdw::pdl_launch_dependents();
    if (threadIdx.x == 0) {
        sfdw::mbar_init(&sm.ibar[0], 1);
        sfdw::mbar_init(&sm.ibar[1], 1);
        sfdw::mbar_fence_init();
    }
    const sfdq::Span span = sfdq::cta_span(V, ny / 2);
    const unsigned tbase = sfdq::tmq_setup(&sm.tmem, tabX, vstride, span.first_view(), twl);
    const unsigned tq = sfdw::tm_quarter(tbase, threadIdx.x >> 5);
    sfdw::pdl_wait();  // B (and vmax, mom) come from pass y
    unsigned iphase = 0;
    for (int s = 0; s < 2; ++s) {
        const sfdq::Range rg = span.segment(s);
        if (rg.u0 >= rg.u1) break;
        if (s == 1) sfdq::tmq_refill(tbase, tabX, vstride, rg.view);
        sfdq::pass_x_quad(sm, B, ny, tq, tq + sfdq::TQ_TW, field, inten, vmax, mom, rg, iphase);
    }
    sfdw::tm_finish(tbase);
}

// ---- pipe micro-benchmarks (sfd_measure_pipes) -------------------------------------------------------
// fp32 FMA throughput: 8 independent chains per thread, 16 warps per SM
__global__ void __launch_bounds__(512) k_peak_ffma(float *out, int iters, float a, float b) {
    float x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = (float)(threadIdx.x + i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int i = 0; i < 8; ++i) x[i] = fmaf(x[i], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i];
    if (s == 12345.678f) out[0] = s;  // never true: keeps the chains alive
}
// cycles of one radix-32 stage for a warp that has its sub-partition to itself (4 warps per SM);
// TW selects stage B (twiddles folded in).  in: 32 x 32 complex values per warp slot.
template <bool TW>
__global__ void __launch_bounds__(128, 1)
k_peak_dft32(const float2 *in, const float2 *__restrict__ twl, float2 *out, long long *cycles,
             int reps) {
    const int lane = threadIdx.x & 31;
    float2 v[32], tw[sfdw::TWN];
    sfdw::load_twiddles(tw, lane, twl);
#pragma unroll
    for (int r = 0; r < 32; ++r) v[r] = in[threadIdx.x + 128 * r];
    __syncthreads();
    const long long t0 = clock64();
    for (int i = 0; i < reps; ++i) {
        if (TW)
            sfdb::dft32_tw(v, tw);
        else
            sfdb::dft32(v);
#pragma unroll
        for (int r = 0; r < 32; ++r) {  // keep the magnitudes bounded: exact scaling, 2 ops per value
            v[r].x *= 0.125f;
            v[r].y *= 0.125f;
        }
    }
    const long long t1 = clock64();
#pragma unroll
    for (int r = 0; r < 32; ++r) out[(size_t)blockIdx.x * 4096 + threadIdx.x + 128 * r] = v[r];
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

std::atomic<long long> g_launches{0};

// Launch configuration shared by every kernel of the library: programmatic stream serialization,
// i.e. a kernel may start on an SM as soon as the kernel before it in the stream has left that SM,
// runs its prologue (barriers, twiddles, tensor-memory tables: plan constants only) and waits
// (griddepcontrol.wait) for the whole predecessor before touching its data.
struct Launch {
    cudaLaunchAttribute at[1];
    cudaLaunchConfig_t cfg;
    Launch(dim3 grid, dim3 block, size_t smem, cudaStream_t st) : cfg{} {
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.gridDim = grid;
        cfg.blockDim = block;
        cfg.dynamicSmemBytes = smem;
        cfg.stream = st;
        cfg.attrs = at;
        cfg.numAttrs = 1;
    }
};

// the slab loads of the warp kernels read 8 bytes of a hologram row at once (Ny = 512 or 1024 with
// float input, Ny = 2048 with uint8 input: 16 bytes)
bool slab_aligned(const sfd_plan *p, const void *holo) {
    const size_t es = p->d.in_dtype == 0 ? 1 : 4;
    const bool wide = p->d.Ny == sfdq::NL ? p->d.in_dtype == 0
                                          : (p->d.Ny == sfdh::NH || p->d.Ny == sfdw::N) && p->d.in_dtype != 0;
    const size_t mask = wide ? 15 : 7;
    return (reinterpret_cast<size_t>(holo) & mask) == 0 && ((size_t)p->d.in_stride * es & mask) == 0;
}

AxisTabs axis_y(const sfd_dev &d) { return AxisTabs{d.tabs, d.vstride, d.off_pre_y, d.off_Hy, d.off_post_y}; }
AxisTabs axis_x(const sfd_dev &d) { return AxisTabs{d.tabs, d.vstride, d.off_pre_x, d.off_Hx, d.off_post_x}; }

// ---- pass y ---------------------------------------------------------------------------------------
template <int LOG2M>
cudaError_t launch_y_generic(const sfd_dev &d, const void *holo, unsigned int *vmax, double *mom,
                             cudaStream_t st) {
    using TL = Tile<LOG2M>;
    Launch l(dim3(d.Nx / TL::C, d.V), dim3(TL::THREADS_Y), TL::SMEM_Y, st);
    if (d.in_dtype == 0)
        return cudaLaunchKernelEx(&l.cfg, k_pass_y<LOG2M, unsigned char>, (const unsigned char *)holo,
                                  d.in_stride, d.Nx, axis_y(d), (const float2 *)d.tw_y, d.B, vmax, mom);
    return cudaLaunchKernelEx(&l.cfg, k_pass_y<LOG2M, float>, (const float *)holo, d.in_stride, d.Nx,
                              axis_y(d), (const float2 *)d.tw_y, d.B, vmax, mom);
}

cudaError_t launch_y(sfd_plan *p, const void *holo, unsigned int *vmax, double *mom,
                     cudaStream_t st) {
    const sfd_dev &d = p->d;
    const CUtensorMap &tmB = *reinterpret_cast<const CUtensorMap *>(p->tmapB);
    const float2 *tabY = d.tabs + d.off_tabY;
    if (sfd_uses_warp_y(p, holo) && d.Ny == sfdw::N) {
        // a CTA works inside one view (its tensor memory holds both branches' tables of that view):
        // SMs / V CTAs per view
        const int cpv = d.sms / d.V > 0 ? d.sms / d.V : 1;
        if (d.in_dtype == 0) {
            Launch l(dim3(d.V * cpv), dim3(256), sizeof(sfdw::SmemY<unsigned char>), st);
            return cudaLaunchKernelEx(&l.cfg, k_cols_1024<unsigned char>, (const unsigned char *)holo,
                                      d.in_stride, d.Nx, tabY, d.vstride, (const float2 *)d.w_twl, tmB,
                                      vmax, mom, d.V, cpv);
        }
        Launch l(dim3(d.V * cpv), dim3(256), sizeof(sfdw::SmemY<float>), st);
        return cudaLaunchKernelEx(&l.cfg, k_cols_1024<float>, (const float *)holo, d.in_stride, d.Nx,
                                  tabY, d.vstride, (const float2 *)d.w_twl, tmB, vmax, mom, d.V, cpv);
    }
    if (sfd_uses_warp_y(p, holo) && d.Ny == sfdh::NH) {
        const int grid = d.V > d.sms ? d.V : d.sms;
        if (d.in_dtype == 0) {
            Launch l(dim3(grid), dim3(256), sizeof(sfdh::SmemYH<unsigned char>), st);
            return cudaLaunchKernelEx(&l.cfg, k_cols_512<unsigned char>, (const unsigned char *)holo,
                                      d.in_stride, d.Nx, tabY, d.vstride, (const float2 *)d.w_twl, tmB,
                                      vmax, mom, d.V);
        }
        Launch l(dim3(grid), dim3(256), sizeof(sfdh::SmemYH<float>), st);
        return cudaLaunchKernelEx(&l.cfg, k_cols_512<float>, (const float *)holo, d.in_stride, d.Nx, tabY,
                                  d.vstride, (const float2 *)d.w_twl, tmB, vmax, mom, d.V);
    }
    if (sfd_uses_warp_y(p, holo) && d.Ny == sfdq::NL) {
        const int grid = d.V > d.sms ? d.V : d.sms;
        if (d.in_dtype == 0) {
            Launch l(dim3(grid), dim3(256), sizeof(sfdq::SmemYQ<unsigned char>), st);
            return cudaLaunchKernelEx(&l.cfg, k_cols_2048<unsigned char>, (const unsigned char *)holo,
                                      d.in_stride, d.Nx, tabY, d.vstride, (const float2 *)d.w_twl, tmB,
                                      vmax, mom, d.V);
        }
        Launch l(dim3(grid), dim3(256), sizeof(sfdq::SmemYQ<float>), st);
        return cudaLaunchKernelEx(&l.cfg, k_cols_2048<float>, (const float *)holo, d.in_stride, d.Nx,
                                  tabY, d.vstride, (const float2 *)d.w_twl, tmB, vmax, mom, d.V);
    }
    switch (d.log2My) {
        case 7: return launch_y_generic<7>(d, holo, vmax, mom, st);
        case 8: return launch_y_generic<8>(d, holo, vmax, mom, st);
        case 9: return launch_y_generic<9>(d, holo, vmax, mom, st);
        case 10: return launch_y_generic<10>(d, holo, vmax, mom, st);
        case 11: return launch_y_generic<11>(d, holo, vmax, mom, st);
        case 12: return launch_y_generic<12>(d, holo, vmax, mom, st);
    }
    return cudaErrorInvalidValue;
}

// ---- pass x ---------------------------------------------------------------------------------------
template <int LOG2M>
cudaError_t launch_x_generic(const sfd_dev &d, float2 *field, float *inten, unsigned int *vmax,
                             double *mom, cudaStream_t st) {
    using TL = Tile<LOG2M>;
    Launch l(dim3(d.Ny / TL::RPC, d.V), dim3(TL::THREADS_X), TL::SMEM_X, st);
    if (mom == nullptr)
        return cudaLaunchKernelEx(&l.cfg, k_pass_x<LOG2M, false>, (const float2 *)d.B, d.Ny, axis_x(d),
                                  (const float2 *)d.tw_x, field, inten, vmax, mom);
    return cudaLaunchKernelEx(&l.cfg, k_pass_x<LOG2M, true>, (const float2 *)d.B, d.Ny, axis_x(d),
                              (const float2 *)d.tw_x, field, inten, vmax, mom);
}

cudaError_t launch_x(sfd_plan *p, float2 *field, float *inten, unsigned int *vmax, double *mom,
                     cudaStream_t st) {
    const sfd_dev &d = p->d;
    const float2 *tabX = d.tabs + d.off_tabX;
    if (sfd_uses_warp_x(p) && d.Nx == sfdw::N) {
        Launch l(dim3(d.V > d.sms ? d.V : d.sms), dim3(sfdw::NWX * 32), sizeof(sfdw::SmemX<sfdw::NWX>), st);
        return cudaLaunchKernelEx(&l.cfg, k_rows_1024, (const float2 *)d.B, d.Ny, tabX, d.vstride,
                                  (const float2 *)d.w_twl, field, inten, vmax, mom, d.V);
    }
    if (sfd_uses_warp_x(p) && d.Nx == sfdh::NH) {
        Launch l(dim3(d.V > d.sms ? d.V : d.sms), dim3(256), sizeof(sfdh::SmemXH), st);
        return cudaLaunchKernelEx(&l.cfg, k_rows_512, (const float2 *)d.B, d.Ny, tabX, d.vstride,
                                  (const float2 *)d.w_twl, field, inten, vmax, mom, d.V);
    }
    if (sfd_uses_warp_x(p) && d.Nx == sfdq::NL) {
        Launch l(dim3(d.V > d.sms ? d.V : d.sms), dim3(256), sizeof(sfdq::SmemXQ), st);
        return cudaLaunchKernelEx(&l.cfg, k_rows_2048, (const float2 *)d.B, d.Ny, tabX, d.vstride,
                                  (const float2 *)d.w_twl, field, inten, vmax, mom, d.V);
    }
    switch (d.log2Mx) {
        case 7: return launch_x_generic<7>(d, field, inten, vmax, mom, st);
        case 8: return launch_x_generic<8>(d, field, inten, vmax, mom, st);
        case 9: return launch_x_generic<9>(d, field, inten, vmax, mom, st);
        case 10: return launch_x_generic<10>(d, field, inten, vmax, mom, st);
        case 11: return launch_x_generic<11>(d, field, inten, vmax, mom, st);
        case 12: return launch_x_generic<12>(d, field, inten, vmax, mom, st);
    }
    return cudaErrorInvalidValue;
}

template <int LOG2M, typename TIn> cudaError_t set_attr() {
    cudaError_t e = cudaFuncSetAttribute(k_pass_y<LOG2M, TIn>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)Tile<LOG2M>::SMEM_Y);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k_pass_x<LOG2M, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)Tile<LOG2M>::SMEM_X);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_pass_x<LOG2M, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)Tile<LOG2M>::SMEM_X);
}

}  // namespace

bool sfd_uses_warp_y(const sfd_plan *p, const void *holo) {
    return p->kernels != SFD_KERNELS_GENERIC && p->d.off_tabY >= 0 && p->d.Nx % 16 == 0 &&
           (holo == nullptr || slab_aligned(p, holo));
}
bool sfd_uses_warp_x(const sfd_plan *p) {
    return p->kernels != SFD_KERNELS_GENERIC && p->d.off_tabX >= 0 && p->d.Ny % 4 == 0;
}

// Tensor map of the intermediate B for the bulk stores of the warp pass y: B as float
// [V * Ny][2 Nx], box = 4 floats (two complex columns; Ny = 2048: 8 floats, four columns) x YBOX rows,
// no swizzle.  The encoder is a driver entry point; it is fetched through the runtime so that the
// library does not link libcuda.
cudaError_t sfd_encode_rows_tmap(void *out, float2 *base, unsigned long long rows, int nx,
                                 unsigned box_floats, unsigned box_rows, int swizzle) {
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *,
                                  const cuuint64_t *, const cuuint64_t *, const cuuint32_t *,
                                  const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qr;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr);
    if (e != cudaSuccess) return e;
    if (fn == nullptr || qr != cudaDriverEntryPointSuccess) return cudaErrorNotSupported;
    const cuuint64_t dims[2] = {2 * (cuuint64_t)nx, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {2 * (cuuint64_t)nx * sizeof(float)};
    const cuuint32_t box[2] = {box_floats, box_rows};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = ((encode_fn)fn)(
        reinterpret_cast<CUtensorMap *>(out), CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, base, dims,
        strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
        swizzle == 64 ? CU_TENSOR_MAP_SWIZZLE_64B
                      : swizzle == 32 ? CU_TENSOR_MAP_SWIZZLE_32B : CU_TENSOR_MAP_SWIZZLE_NONE,
        CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

cudaError_t sfd_make_tensormaps(sfd_plan *p) {
    static_assert(sizeof(CUtensorMap) <= sizeof(p->tmapB), "tensor map storage");
    if (p->d.off_tabY < 0) return cudaSuccess;
    return sfd_encode_rows_tmap(p->tmapB, p->d.B, (unsigned long long)p->d.V * p->d.Ny, p->d.Nx,
                                p->d.Ny == sfdq::NL ? (unsigned)sfdq::YBOXW : 4u, sfdw::YBOX);
}

void sfd_count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }
long long sfd_launch_count_impl() { return g_launches.load(std::memory_order_relaxed); }

// cudaFuncSetAttribute acts on the current device: called once per device (sfd_plan.cpp)
cudaError_t sfd_kernels_init(int device, int *sms) {
    cudaError_t e;
#define SFD_ATTR(L)                                                   \
    if ((e = set_attr<L, unsigned char>()) != cudaSuccess) return e;  \
    if ((e = set_attr<L, float>()) != cudaSuccess) return e;
    SFD_ATTR(7) SFD_ATTR(8) SFD_ATTR(9) SFD_ATTR(10) SFD_ATTR(11) SFD_ATTR(12)
#undef SFD_ATTR
#define SFD_SMEM(kernel, bytes)                                                               \
    if ((e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,        \
                                  (int)(bytes))) != cudaSuccess)                              \
        return e;
    SFD_SMEM(k_cols_1024<unsigned char>, sizeof(sfdw::SmemY<unsigned char>))
    SFD_SMEM(k_cols_1024<float>, sizeof(sfdw::SmemY<float>))
    SFD_SMEM(k_rows_1024, sizeof(sfdw::SmemX<sfdw::NWX>))
    SFD_SMEM(k_cols_512<unsigned char>, sizeof(sfdh::SmemYH<unsigned char>))
    SFD_SMEM(k_cols_512<float>, sizeof(sfdh::SmemYH<float>))
    SFD_SMEM(k_rows_512, sizeof(sfdh::SmemXH))
    SFD_SMEM(k_cols_2048<unsigned char>, sizeof(sfdq::SmemYQ<unsigned char>))
    SFD_SMEM(k_cols_2048<float>, sizeof(sfdq::SmemYQ<float>))
    SFD_SMEM(k_rows_2048, sizeof(sfdq::SmemXQ))
#undef SFD_SMEM
    return cudaDeviceGetAttribute(sms, cudaDevAttrMultiProcessorCount, device);
}

cudaError_t sfd_launch(sfd_plan *p, const void *holo, float2 *field, float *inten,
                       unsigned char *u8, cudaStream_t st, double *mom) {
    const sfd_dev &d = p->d;
    unsigned int *vmax = u8 ? d.vmax : nullptr;
    if (u8) {
        field = nullptr;
        inten = d.inten_ws;
    }
    const bool timing = p->timing;
    cudaError_t e;
    if (timing) cudaEventRecord(p->ev[0], st);
    if ((e = launch_y(p, holo, vmax, mom, st)) != cudaSuccess) return e;
    if (timing) cudaEventRecord(p->ev[1], st);
    if ((e = launch_x(p, field, inten, vmax, mom, st)) != cudaSuccess) return e;
    if (timing) cudaEventRecord(p->ev[2], st);
    int n = 2;
    if (u8) {
        const int quads = d.Nx * d.Ny / 4;
        Launch l(dim3((quads + 256 * 4 - 1) / (256 * 4), d.V), dim3(256), 0, st);
        if ((e = cudaLaunchKernelEx(&l.cfg, k_quantise, (const float4 *)d.inten_ws,
                                    (const unsigned int *)d.vmax, (uchar4 *)u8, quads)) != cudaSuccess)
            return e;
        if (timing) cudaEventRecord(p->ev[3], st);
        ++n;
    }
    p->ev_valid = timing;
    p->ev_quant = timing && u8 != nullptr;
    g_launches.fetch_add(n, std::memory_order_relaxed);
    return cudaGetLastError();
}

// ---- sfd_measure_pipes ------------------------------------------------------------------------------
// out[0] plain fp32 FMA throughput of the whole GPU (TFLOP/s, 2 flop per FMA), out[1] / out[2] cycles
// of one stage-A / stage-B radix-32 butterfly (sfd_dft32.cuh) for a warp alone on its sub-partition,
// out[3] SM clock during the measurement (GHz, from clock64 against CUDA events).
cudaError_t sfd_measure_pipes_impl(double out[4]) {
    int dev = 0, sms = 0;
    cudaError_t e;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    float *dummy = nullptr;
    float2 *in = nullptr, *res = nullptr, *twl = nullptr;
    long long *cyc = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    std::vector<float2> hin(4096), htw(32 * 32);
    for (int i = 0; i < 4096; ++i) hin[i] = make_float2(0.001f * (float)(i % 97), -0.002f * (float)(i % 31));
    for (int i = 0; i < 1024; ++i) htw[i] = make_float2(cosf(0.001f * (float)i), -sinf(0.001f * (float)i));
    std::vector<long long> hc(sms);
    auto cleanup = [&]() {
        cudaFree(dummy); cudaFree(in); cudaFree(res); cudaFree(twl); cudaFree(cyc);
        if (e0) cudaEventDestroy(e0);
        if (e1) cudaEventDestroy(e1);
    };
#define SFD_TRY(call) if ((e = (call)) != cudaSuccess) { cleanup(); return e; }
    SFD_TRY(cudaMalloc((void **)&dummy, 256));
    SFD_TRY(cudaMalloc((void **)&in, 4096 * sizeof(float2)));
    SFD_TRY(cudaMalloc((void **)&res, (size_t)sms * 4096 * sizeof(float2)));
    SFD_TRY(cudaMalloc((void **)&twl, 1024 * sizeof(float2)));
    SFD_TRY(cudaMalloc((void **)&cyc, sms * sizeof(long long)));
    SFD_TRY(cudaMemcpy(in, hin.data(), 4096 * sizeof(float2), cudaMemcpyHostToDevice));
    SFD_TRY(cudaMemcpy(twl, htw.data(), 1024 * sizeof(float2), cudaMemcpyHostToDevice));
    SFD_TRY(cudaEventCreate(&e0));
    SFD_TRY(cudaEventCreate(&e1));
    const int iters = 4096;
    float ms = 0.f;
    k_peak_ffma<<<sms * 2, 512>>>(dummy, 64, 1.0001f, 0.5f);  // warm-up
    SFD_TRY(cudaEventRecord(e0));
    k_peak_ffma<<<sms * 2, 512>>>(dummy, iters, 1.0001f, 0.5f);
    SFD_TRY(cudaEventRecord(e1));
    SFD_TRY(cudaEventSynchronize(e1));
    SFD_TRY(cudaEventElapsedTime(&ms, e0, e1));
    out[0] = 2.0 * 64.0 * iters * 512.0 * 2.0 * sms / (ms * 1e-3) / 1e12;
    const int reps = 2000;
    for (int tw = 0; tw < 2; ++tw) {
        for (int pass = 0; pass < 2; ++pass) {  // first pass warms the instruction cache
            SFD_TRY(cudaEventRecord(e0));
            if (tw)
                k_peak_dft32<true><<<sms, 128>>>(in, twl, res, cyc, reps);
            else
                k_peak_dft32<false><<<sms, 128>>>(in, twl, res, cyc, reps);
            SFD_TRY(cudaEventRecord(e1));
            SFD_TRY(cudaEventSynchronize(e1));
        }
        SFD_TRY(cudaEventElapsedTime(&ms, e0, e1));
        SFD_TRY(cudaMemcpy(hc.data(), cyc, sms * sizeof(long long), cudaMemcpyDeviceToHost));
        double mean = 0;
        for (int i = 0; i < sms; ++i) mean += (double)hc[i];
        mean /= sms;
        out[1 + tw] = mean / reps - 64.0;  // minus the 64 scaling multiplies of the loop body
        out[3] = mean / (ms * 1e-3) / 1e9;
    }
#undef SFD_TRY
    cleanup();
    sfd_count_launch(6);
    return cudaSuccess;
}

// host-side step of the butterflies (CPU tests): in / out = 32 interleaved (re, im) pairs; the
// stored-sign convention of sfd_dft32.cuh is undone here so that out is the plain DFT
void sfd_host_dft32_impl(const float *in, float *out, int lane, int twiddled) {
    float2 v[32], t[sfdb::NTW];
    for (int r = 0; r < 32; ++r) v[r] = make_float2(in[2 * r], in[2 * r + 1]);
    if (twiddled) {
        for (int n = 2; n <= 32; n *= 2)
            for (int k = 0; k < n / 2; ++k) {
                const long double ph = -6.283185307179586476925286766559005768L * (lane + 32 * k) /
                                       (32.0L * n);
                t[n / 2 - 1 + k] = make_float2((float)cosl(ph), (float)sinl(ph));
            }
        sfdb::dft32_tw(v, t);
    } else {
        sfdb::dft32(v);
    }
    for (int r = 0; r < 32; ++r) {
        const float sg = (float)sfdb::out_sign(r);
        out[2 * r] = sg * v[r].x;
        out[2 * r + 1] = sg * v[r].y;
    }
}

// ---- allocation-free 8-bit quantisation (sfd_quantise_u8_static, include/sfd.h) -----------------------
// Step (xi) / reading 15 on its own, for callers that may not allocate (code under CUDA graph
// capture, serving loops, harnesses that forbid cudaMalloc): float intensities in, 8-bit images out,
// I8 = round_half_even(255 I / max I) per view.  The per-view maxima - the scratch that sfd_execute_u8
// keeps in plan memory (sfd_dev::vmax) - live in the array below instead: SFD_STATIC_MAX_VIEWS words,
// held by every GPU that loads the library until the process exits.  In host code the array's NAME is
// a host-side stand-in, not a device address; the address comes from cudaGetSymbolAddress, once per
// device with that device current (static_scratch below).  All calls share the array and it keeps the
// last call's contents: every call clears the words it uses first (stream-ordered), and calls that
// overlap on the GPU (different streams without an event between them) race on it.
static __device__ __align__(256) unsigned int g_static_vmax[SFD_STATIC_MAX_VIEWS];

namespace {

// per-view maximum of `quads` float4s into vmax[view] (cleared beforehand); intensities are >= 0, so
// their bit patterns order like unsigned integers (as in pass x)
__global__ void __launch_bounds__(256)
k_view_max_static(const float4 *__restrict__ inten, unsigned int *vmax, int quads_per_view) {
    const int v = blockIdx.y;
    const size_t base = (size_t)v * quads_per_view;
    float mx = 0.f;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < quads_per_view; i += gridDim.x * blockDim.x) {
        const float4 I = inten[base + i];
        mx = fmaxf(fmaxf(mx, fmaxf(I.x, I.y)), fmaxf(I.z, I.w));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if ((threadIdx.x & 31) == 0 && mx > 0.f) atomicMax(vmax + v, __float_as_uint(mx));
}

std::mutex g_static_mu;
unsigned int *g_static_ptr[64] = {};  // device address of g_static_vmax, per device
thread_local char g_static_err[200] = "no error";

// device address of the scratch array on the current device (looked up on the device's first call)
cudaError_t static_scratch(unsigned int **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (g_static_ptr[dev] == nullptr) {
        void *ptr = nullptr;
        if ((e = cudaGetSymbolAddress(&ptr, g_static_vmax)) != cudaSuccess) return e;
        g_static_ptr[dev] = static_cast<unsigned int *>(ptr);
    }
    *out = g_static_ptr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" {

SFD_API int sfd_quantise_u8_static(const float *intensity_dev, int n_views, long long pixels_per_view,
                                   unsigned char *intensity_u8_dev, void *stream) {
    auto fail = [](int code, const char *what) {
        std::snprintf(g_static_err, sizeof g_static_err, "sfd_quantise_u8_static: %s", what);
        return code;
    };
    if (!intensity_dev || !intensity_u8_dev) return fail(SFD_EINVAL, "NULL pointer");
    if (n_views < 1 || pixels_per_view < 4 || pixels_per_view % 4 != 0 ||
        pixels_per_view / 4 > 0x7fffffffLL)
        return fail(SFD_EINVAL, "n_views >= 1 and pixels_per_view a positive multiple of 4 (< 2^33) are required");
    if ((reinterpret_cast<size_t>(intensity_dev) & 15) != 0 || (reinterpret_cast<size_t>(intensity_u8_dev) & 3) != 0)
        return fail(SFD_EINVAL, "intensity_dev must be 16-byte, intensity_u8_dev 4-byte aligned");
    if (n_views > SFD_STATIC_MAX_VIEWS) {
        std::snprintf(g_static_err, sizeof g_static_err,
                      "sfd_quantise_u8_static: n_views = %d exceeds SFD_STATIC_MAX_VIEWS = %d (the size of "
                      "the library's static scratch array); split the call",
                      n_views, SFD_STATIC_MAX_VIEWS);
        return SFD_EUNSUPPORTED;
    }
    cudaStream_t st = (cudaStream_t)stream;
    unsigned int *vmax = nullptr;
    cudaError_t e = static_scratch(&vmax);
    const int quads = (int)(pixels_per_view / 4);
    const int blocks = (quads + 256 * 4 - 1) / (256 * 4);
    // the array keeps the last call's maxima: clear this call's words first
    if (e == cudaSuccess) e = cudaMemsetAsync(vmax, 0, (size_t)n_views * sizeof(unsigned int), st);
    if (e == cudaSuccess) {
        k_view_max_static<<<dim3(blocks, n_views), 256, 0, st>>>((const float4 *)intensity_dev, vmax, quads);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) {
        Launch l(dim3(blocks, n_views), dim3(256), 0, st);
        e = cudaLaunchKernelEx(&l.cfg, k_quantise, (const float4 *)intensity_dev,
                               (const unsigned int *)vmax, (uchar4 *)intensity_u8_dev, quads);
    }
    if (e != cudaSuccess) {
        std::snprintf(g_static_err, sizeof g_static_err, "sfd_quantise_u8_static: %s (%s)",
                      cudaGetErrorName(e), cudaGetErrorString(e));
        cudaGetLastError();
        return SFD_ECUDA;
    }
    g_launches.fetch_add(2, std::memory_order_relaxed);
    return SFD_OK;
}

SFD_API int sfd_static_max_views(void) { return SFD_STATIC_MAX_VIEWS; }

SFD_API const char *sfd_static_last_error(void) { return g_static_err; }

}  // extern "C"

// ---- sfd_measure_memory_pipes: shared memory and tensor memory as the warp kernels use them ----------
namespace {

// shared memory: every warp reads its own 4 KB tile with 16-byte loads (the row reads of the transposes:
// 4 wavefronts per instruction, conflict-free) and writes it with 8-byte stores (their column writes)
__global__ void __launch_bounds__(256, 1)
k_peak_smem(float *out, long long *cycles, int reps) {
    __shared__ float4 tile[8][256];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = lane; i < 256; i += 32) tile[warp][i] = make_float4((float)i, 1.f, 2.f, 3.f);
    __syncthreads();
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    const long long t0 = clock64();
    for (int r = 0; r < reps; ++r) {
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const float4 w = tile[warp][q * 32 + lane];
            acc.x += w.x; acc.y += w.y; acc.z += w.z; acc.w += w.w;
        }
        float2 *t2 = reinterpret_cast<float2 *>(tile[warp]);
#pragma unroll
        for (int q = 0; q < 16; ++q) t2[q * 32 + lane] = make_float2(acc.x, acc.y + (float)q);
        __syncwarp();
    }
    __syncthreads();
    const long long t1 = clock64();
    out[blockIdx.x * 256 + threadIdx.x] = acc.x + acc.y + acc.z + acc.w;
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

// tensor memory: (a) four 16-column loads in flight per warp and wait, as the table reads of a line are
// issued; (b) one load, wait, and the next address taken from the loaded value: the dependent latency
__global__ void __launch_bounds__(256, 1)
k_peak_tmem(float *out, long long *cycles, int reps, int warps_per_quarter) {
    __shared__ unsigned slot;
    const int warp = threadIdx.x >> 5;
    if (warp == 0) sfdw::tm_alloc(&slot);
    sfdw::tm_sync_cta();
    const unsigned base = *reinterpret_cast<volatile unsigned *>(&slot), q = sfdw::tm_quarter(base, warp);
    sfdw::TChunk c[4];
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int i = 0; i < 16; ++i) c[j].w[i] = 0u;
    if (warp < 4) {
        for (int col = 0; col < sfdw::TM_COLS; col += 16) sfdw::tm_st(c[0], q + col);
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    }
    sfdw::tm_sync_cta();
    const bool active = (warp >> 2) < warps_per_quarter;
    unsigned sum = 0;
    long long t0 = clock64();
    if (active)
        for (int r = 0; r < reps; ++r) {
#pragma unroll
            for (int j = 0; j < 4; ++j) sfdw::tm_ld(c[j], q + 64 * (r & 7) + 16 * j);
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                sfdw::tm_wait(c[j]);
                sum += c[j].w[0] + c[j].w[15];
            }
        }
    long long t1 = clock64();
    if (threadIdx.x == 0) cycles[2 * blockIdx.x] = t1 - t0;
    __syncthreads();
    unsigned off = 0;
    t0 = clock64();
    if (warp == 0)
        for (int r = 0; r < reps; ++r) {
            sfdw::tm_ld(c[0], q + off);
            sfdw::tm_wait(c[0]);
            off = (c[0].w[3] & 0x10u) + 16u * (unsigned)(r & 15);  // (the columns hold zeros)
            sum += off;
        }
    t1 = clock64();
    if (threadIdx.x == 0) cycles[2 * blockIdx.x + 1] = t1 - t0;
    out[blockIdx.x * 256 + threadIdx.x] = (float)sum;
    sfdw::tm_finish(base);
}

}  // namespace

// out[0] shared memory, bytes per clock and SM, in the access pattern of the transposes (16-byte row
// reads + 8-byte column writes, 8 warps); out[1] / out[2] tensor-memory load rate in bytes per clock
// and sub-partition with one / two warps per sub-partition (four tcgen05.ld.32x32b.x16 in flight per
// warp); out[3] cycles of one dependent tcgen05.ld + wait::ld.
extern "C" SFD_API int sfd_measure_memory_pipes(double out[4]) {
    if (!out) return SFD_EINVAL;
    int dev = 0, sms = 0;
    float *res = nullptr;
    long long *cyc = nullptr;
    cudaError_t e;
    auto done = [&](cudaError_t err) {
        cudaFree(res);
        cudaFree(cyc);
        if (err == cudaSuccess) return (int)SFD_OK;
        std::snprintf(g_static_err, sizeof g_static_err, "sfd_measure_memory_pipes: %s (%s)",
                      cudaGetErrorName(err), cudaGetErrorString(err));
        cudaGetLastError();
        return (int)SFD_ECUDA;
    };
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return done(e);
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return done(e);
    if ((e = cudaMalloc((void **)&res, (size_t)sms * 256 * sizeof(float))) != cudaSuccess) return done(e);
    if ((e = cudaMalloc((void **)&cyc, (size_t)sms * 2 * sizeof(long long))) != cudaSuccess) return done(e);
    std::vector<long long> hc(2 * (size_t)sms);
    auto mean = [&](int stride, int which) {
        double m = 0;
        for (int i = 0; i < sms; ++i) m += (double)hc[(size_t)stride * i + which];
        return m / sms;
    };
    const int reps = 2000;
    for (int pass = 0; pass < 2; ++pass) k_peak_smem<<<sms, 256>>>(res, cyc, reps);
    if ((e = cudaMemcpy(hc.data(), cyc, sms * sizeof(long long), cudaMemcpyDeviceToHost)) != cudaSuccess) return done(e);
    out[0] = 8.0 * 32.0 * (8.0 * 16.0 + 16.0 * 8.0) * reps / mean(1, 0);
    for (int wq = 1; wq <= 2; ++wq) {
        for (int pass = 0; pass < 2; ++pass) k_peak_tmem<<<sms, 256>>>(res, cyc, reps, wq);
        if ((e = cudaMemcpy(hc.data(), cyc, 2 * sms * sizeof(long long), cudaMemcpyDeviceToHost)) != cudaSuccess)
            return done(e);
        out[wq] = (double)wq * 4.0 * 16.0 * 32.0 * 4.0 * reps / mean(2, 0);
        out[3] = mean(2, 1) / reps;
    }
    if ((e = cudaDeviceSynchronize()) != cudaSuccess) return done(e);
    g_launches.fetch_add(6, std::memory_order_relaxed);
    return done(cudaSuccess);
}
