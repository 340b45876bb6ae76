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

#include "sfd_fft_core.cuh"
#include "sfd_internal.h"
#include "sfd_warp1024.cuh"
#include "sfd_warp2048.cuh"

namespace {

using namespace sfd;

// columns per CTA in pass y / rows per CTA in pass x, by padded length
template <int LOG2M> struct Tile {
    static constexpr int T = Sched<LOG2M>::T;
    static constexpr int C = LOG2M <= 7 ? 16 : LOG2M <= 9 ? 8 : LOG2M <= 11 ? 4 : 2;
    static constexpr int RPC = T >= 128 ? 1 : 128 / T;
    static constexpr int THREADS_Y = C * T;
    static constexpr int THREADS_X = RPC * T;
    static constexpr size_t SMEM_Y = sizeof(float2) * Sched<LOG2M>::PADDED * C;
    static constexpr size_t SMEM_X = sizeof(float2) * Sched<LOG2M>::PADDED * RPC;
};

template <int LOG2M, typename TIn>
__global__ void __launch_bounds__(Tile<LOG2M>::THREADS_Y)
k_pass_y(const TIn *__restrict__ holo, const float2 *__restrict__ pre_y,
         const float2 *__restrict__ H, const float2 *__restrict__ post_y,
         const float2 *__restrict__ tw, float2 *__restrict__ B, unsigned int *vmax, double *mom) {
    extern __shared__ float2 smem[];
    sfdw::pdl_launch_dependents();
    sfdw::pdl_wait();  // the hologram, B, vmax and mom belong to the kernels before this one
    if (vmax != nullptr && blockIdx.x == 0 && threadIdx.x == 0) vmax[blockIdx.y] = 0u;
    if (mom != nullptr && blockIdx.x == 0 && threadIdx.x < 2) mom[2 * blockIdx.y + threadIdx.x] = 0.0;
    pass_y_body<LOG2M, Tile<LOG2M>::C, TIn>(threadIdx.x, blockIdx.x, blockIdx.y, smem, holo, pre_y,
                                            H, post_y, tw, B, [] { __syncthreads(); });
}

template <int LOG2M, bool MOM>
__global__ void __launch_bounds__(Tile<LOG2M>::THREADS_X)
k_pass_x(const float2 *__restrict__ B, const float2 *__restrict__ pre_x,
         const float2 *__restrict__ H, const float2 *__restrict__ post_x,
         const float2 *__restrict__ tw, float2 *__restrict__ field, float *__restrict__ inten,
         unsigned int *vmax, double *mom) {
    extern __shared__ float2 smem[];
    sfdw::pdl_launch_dependents();
    sfdw::pdl_wait();  // B (and vmax, mom) come from pass y
    float s1 = 0.f, s2 = 0.f;
    float mx = pass_x_body<LOG2M, Tile<LOG2M>::RPC, MOM>(threadIdx.x, blockIdx.x, blockIdx.y, smem, B,
                                                    pre_x, H, post_x, tw, field, inten,
                                                    [] { __syncthreads(); }, s1, s2);
    if (MOM) {  // focus moments: warp sums in float, accumulation across warps in double
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            s1 += __shfl_xor_sync(0xffffffffu, s1, o);
            s2 += __shfl_xor_sync(0xffffffffu, s2, o);
        }
        if ((threadIdx.x & 31) == 0) {
            atomicAdd(mom + 2 * blockIdx.y, (double)s1);
            atomicAdd(mom + 2 * blockIdx.y + 1, (double)s2);
        }
    }
    if (vmax != nullptr) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        // intensities are >= 0, so their float bit patterns order like unsigned integers
        if ((threadIdx.x & 31) == 0) atomicMax(vmax + blockIdx.y, __float_as_uint(mx));
    }
}

// I8 = round_half_even(255 I / max I) per view (reading 15); 4 pixels per thread.
__global__ void __launch_bounds__(256)
k_quantise(const float4 *__restrict__ inten, const unsigned int *__restrict__ vmax,
           uchar4 *__restrict__ out, int quads_per_view) {
    const int v = blockIdx.y;
    const float mx = __uint_as_float(vmax[v]);
    const float sc = mx > 0.f ? 255.f / mx : 0.f;
    const size_t base = (size_t)v * quads_per_view;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < quads_per_view;
         i += gridDim.x * blockDim.x) {
        const float4 I = __ldg(inten + base + i);
        uchar4 o;
        o.x = (unsigned char)min(__float2int_rn(I.x * sc), 255);
        o.y = (unsigned char)min(__float2int_rn(I.y * sc), 255);
        o.z = (unsigned char)min(__float2int_rn(I.z * sc), 255);
        o.w = (unsigned char)min(__float2int_rn(I.w * sc), 255);
        out[base + i] = o;
    }
}

// ---- N = 1024 fast path (sfd_warp1024.cuh): persistent kernels, one warp pair per line --------------
// One CTA per SM.  Even warps run branch 0 (even bins), odd warps branch 1.
template <typename TIn>
__global__ void __launch_bounds__(sfdw::WY * 32, 1)
k_cols_1024(const TIn *__restrict__ holo, const float2 *__restrict__ tabY,
            const float2 *__restrict__ twl, const __grid_constant__ CUtensorMap tmB,
            unsigned int *vmax, double *mom, int V) {
    extern __shared__ float4 smem4[];
    sfdw::SmemY<TIn> &sm = *reinterpret_cast<sfdw::SmemY<TIn> *>(smem4);
    sfdw::pdl_launch_dependents();
    float2 tw[sfdw::TWN];
    sfdw::load_twiddles(tw, threadIdx.x & 31, twl);
    {   // pull the first slab of this CTA towards L2 while the prologue runs (a prefetch reads nothing:
        // it may precede griddepcontrol.wait)
        constexpr int groups = sfdw::N / sfdw::YC, IPS = sfdw::TileElem<TIn>::IPS;
        const int i0 = (int)((long long)V * groups * blockIdx.x / gridDim.x);
        const TIn *p0 = holo + (i0 % groups) / IPS * (sfdw::YC * IPS);
#pragma unroll
        for (int i = 0; i < 4; ++i)
            asm volatile("prefetch.global.L2 [%0];" ::"l"(p0 + (size_t)(threadIdx.x + 256 * i) * sfdw::N));
    }
    // tables of this CTA's view(s) -> tensor memory (the barriers inside also publish the mbarriers)
    const unsigned tbase = sfdw::tm_setup(&sm.tmem, tabY, V * (sfdw::N / sfdw::YC), sfdw::N / sfdw::YC);
    const unsigned tq = sfdw::tm_quarter(tbase, threadIdx.x >> 5);
    // everything above touches plan constants only; the hologram, B, vmax and mom belong to the
    // kernels before this one in the stream
    sfdw::pdl_wait();
    if (vmax != nullptr && blockIdx.x == 0)
        for (int i = threadIdx.x; i < V; i += blockDim.x) vmax[i] = 0u;
    if (mom != nullptr && blockIdx.x == 0)
        for (int i = threadIdx.x; i < 2 * V; i += blockDim.x) mom[i] = 0.0;
    sfdw::pass_y_loop<TIn>(sm, holo, tq, tw, &tmB, V);
    sfdw::tm_finish(tbase);
}

__global__ void __launch_bounds__(sfdw::WX * 32, 1)
k_rows_1024(const float2 *__restrict__ B, const float2 *__restrict__ tabX,
            const float2 *__restrict__ twl, float2 *__restrict__ field, float *__restrict__ inten,
            unsigned int *vmax, double *mom, int V) {
    extern __shared__ float4 smem4[];
    sfdw::SmemX &sm = *reinterpret_cast<sfdw::SmemX *>(smem4);
    sfdw::pdl_launch_dependents();
    if (threadIdx.x == 0) {
        for (int i = 0; i < sfdw::XP; ++i) sfdw::mbar_init(&sm.ibar[i], 1);
        sfdw::mbar_fence_init();
    }
    float2 tw[sfdw::TWN];
    sfdw::load_twiddles(tw, threadIdx.x & 31, twl);
    constexpr int gpv = (sfdw::N + sfdw::XP - 1) / sfdw::XP;  // units per view, as in pass_x_loop
    const unsigned tbase = sfdw::tm_setup(&sm.tmem, tabX, V * gpv, gpv);
    const unsigned tq = sfdw::tm_quarter(tbase, threadIdx.x >> 5);
    sfdw::pdl_wait();  // B (and vmax, mom) come from pass y
    sfdw::pass_x_loop(sm, B, tq, tw, field, inten, vmax, mom, V);
    sfdw::tm_finish(tbase);
}

// ---- N = 2048 (sfd_warp2048.cuh): four branches per line, a quad of warps per line ------------------
// grid = V * cpv CTAs: CTA c works on view c / cpv.  tab: [V][4][5][1024].
template <typename TIn>
__global__ void __launch_bounds__(256, 1)
k_cols_2048(const TIn *__restrict__ holo, const float2 *__restrict__ tabY,
            const float2 *__restrict__ twl, const __grid_constant__ CUtensorMap tmB,
            unsigned int *vmax, double *mom, int V, int cpv) {
    extern __shared__ float4 smem4[];
    sfdq::SmemYQ<TIn> &sm = *reinterpret_cast<sfdq::SmemYQ<TIn> *>(smem4);
    sfdw::pdl_launch_dependents();
    float2 tw[sfdw::TWN];
    sfdw::load_twiddles(tw, threadIdx.x & 31, twl);
    const sfdq::Range rg = sfdq::cta_range(cpv, sfdq::QUY);
    const unsigned tbase = sfdq::tmq_setup(&sm.tmem, tabY, rg.view);
    const unsigned tq = sfdw::tm_quarter(tbase, threadIdx.x >> 5);
    sfdw::pdl_wait();
    if (vmax != nullptr && blockIdx.x == 0)
        for (int i = threadIdx.x; i < V; i += blockDim.x) vmax[i] = 0u;
    if (mom != nullptr && blockIdx.x == 0)
        for (int i = threadIdx.x; i < 2 * V; i += blockDim.x) mom[i] = 0.0;
    sfdq::pass_y_quad<TIn>(sm, holo, tq, tw, &tmB, rg);
    sfdw::tm_finish(tbase);
}

__global__ void __launch_bounds__(256, 1)
k_rows_2048(const float2 *__restrict__ B, const float2 *__restrict__ tabX,
            const float2 *__restrict__ twl, float2 *__restrict__ field, float *__restrict__ inten,
            unsigned int *vmax, double *mom, int cpv) {
    extern __shared__ float4 smem4[];
    sfdq::SmemXQ &sm = *reinterpret_cast<sfdq::SmemXQ *>(smem4);
    sfdw::pdl_launch_dependents();
    if (threadIdx.x == 0) {
        sfdw::mbar_init(&sm.ibar[0], 1);
        sfdw::mbar_init(&sm.ibar[1], 1);
        sfdw::mbar_fence_init();
    }
    float2 tw[sfdw::TWN];
    sfdw::load_twiddles(tw, threadIdx.x & 31, twl);
    const sfdq::Range rg = sfdq::cta_range(cpv, sfdq::QUX);
    const unsigned tbase = sfdq::tmq_setup(&sm.tmem, tabX, rg.view);
    const unsigned tq = sfdw::tm_quarter(tbase, threadIdx.x >> 5);
    sfdw::pdl_wait();  // B (and vmax, mom) come from pass y
    sfdq::pass_x_quad(sm, B, tq, tw, field, inten, vmax, mom, rg);
    sfdw::tm_finish(tbase);
}

std::atomic<long long> g_launches{0};
int g_sms = 0;

cudaError_t launch_warp1024(sfd_plan *p, const void *holo, float2 *field, float *inten,
                            unsigned char *u8, double *mom, cudaStream_t st) {
    const sfd_dev &d = p->d;
    const int V = d.V;
    unsigned int *vmax = u8 ? d.vmax : nullptr;
    if (u8) {
        field = nullptr;
        inten = d.inten_ws;
    }
    const bool timing = p->timing;
    if (timing) cudaEventRecord(p->ev[0], st);
    // one CTA per SM, but at least V CTAs: a CTA's contiguous range of items (rows) then touches at
    // most two views (the kernels hold two table sets)
    const int gy = V > g_sms ? V : g_sms;
    const CUtensorMap &tmB = *reinterpret_cast<const CUtensorMap *>(p->tmapB);
    // Programmatic dependent launch: a kernel may start on an SM as soon as the kernel before it in
    // the stream has left that SM, runs its prologue (barriers, twiddles, tensor-memory tables) and
    // waits (griddepcontrol.wait) for the whole predecessor before touching its data.
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(gy);
    cfg.blockDim = dim3(sfdw::WY * 32);
    cfg.stream = st;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    cudaError_t le;
    if (d.in_dtype == 0) {
        cfg.dynamicSmemBytes = sizeof(sfdw::SmemY<unsigned char>);
        le = cudaLaunchKernelEx(&cfg, k_cols_1024<unsigned char>, (const unsigned char *)holo,
                                (const float2 *)d.w_tabY, (const float2 *)d.w_twl, tmB, vmax, mom, V);
    } else {
        cfg.dynamicSmemBytes = sizeof(sfdw::SmemY<float>);
        le = cudaLaunchKernelEx(&cfg, k_cols_1024<float>, (const float *)holo,
                                (const float2 *)d.w_tabY, (const float2 *)d.w_twl, tmB, vmax, mom, V);
    }
    if (le != cudaSuccess) return le;
    if (timing) cudaEventRecord(p->ev[1], st);
    cfg.blockDim = dim3(sfdw::WX * 32);
    cfg.dynamicSmemBytes = sizeof(sfdw::SmemX);
    le = cudaLaunchKernelEx(&cfg, k_rows_1024, (const float2 *)d.B, (const float2 *)d.w_tabX,
                            (const float2 *)d.w_twl, field, inten, vmax, mom, V);
    if (le != cudaSuccess) return le;
    if (timing) cudaEventRecord(p->ev[2], st);
    int n = 2;
    if (u8) {
        const int quads = sfdw::N * sfdw::N / 4;
        dim3 gq((quads + 256 * 4 - 1) / (256 * 4), V);
        k_quantise<<<gq, 256, 0, st>>>((const float4 *)d.inten_ws, d.vmax, (uchar4 *)u8, quads);
        if (timing) cudaEventRecord(p->ev[3], st);
        ++n;
    }
    p->ev_valid = timing;
    p->ev_quant = timing && u8 != nullptr;
    g_launches.fetch_add(n, std::memory_order_relaxed);
    return cudaGetLastError();
}

cudaError_t launch_warp2048(sfd_plan *p, const void *holo, float2 *field, float *inten,
                            unsigned char *u8, double *mom, cudaStream_t st) {
    const sfd_dev &d = p->d;
    const int V = d.V;
    unsigned int *vmax = u8 ? d.vmax : nullptr;
    if (u8) {
        field = nullptr;
        inten = d.inten_ws;
    }
    const bool timing = p->timing;
    if (timing) cudaEventRecord(p->ev[0], st);
    const int cpv = g_sms / V > 0 ? g_sms / V : 1;  // CTAs per view: a CTA works inside one view
    const CUtensorMap &tmB = *reinterpret_cast<const CUtensorMap *>(p->tmapB);
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(V * cpv);
    cfg.blockDim = dim3(256);
    cfg.stream = st;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    cudaError_t le;
    if (d.in_dtype == 0) {
        cfg.dynamicSmemBytes = sizeof(sfdq::SmemYQ<unsigned char>);
        le = cudaLaunchKernelEx(&cfg, k_cols_2048<unsigned char>, (const unsigned char *)holo,
                                (const float2 *)d.w_tabY, (const float2 *)d.w_twl, tmB, vmax, mom, V,
                                cpv);
    } else {
        cfg.dynamicSmemBytes = sizeof(sfdq::SmemYQ<float>);
        le = cudaLaunchKernelEx(&cfg, k_cols_2048<float>, (const float *)holo,
                                (const float2 *)d.w_tabY, (const float2 *)d.w_twl, tmB, vmax, mom, V,
                                cpv);
    }
    if (le != cudaSuccess) return le;
    if (timing) cudaEventRecord(p->ev[1], st);
    cfg.dynamicSmemBytes = sizeof(sfdq::SmemXQ);
    le = cudaLaunchKernelEx(&cfg, k_rows_2048, (const float2 *)d.B, (const float2 *)d.w_tabX,
                            (const float2 *)d.w_twl, field, inten, vmax, mom, cpv);
    if (le != cudaSuccess) return le;
    if (timing) cudaEventRecord(p->ev[2], st);
    int n = 2;
    if (u8) {
        const int quads = sfdq::NL * sfdq::NL / 4;
        dim3 gq((quads + 256 * 4 - 1) / (256 * 4), V);
        k_quantise<<<gq, 256, 0, st>>>((const float4 *)d.inten_ws, d.vmax, (uchar4 *)u8, quads);
        if (timing) cudaEventRecord(p->ev[3], st);
        ++n;
    }
    p->ev_valid = timing;
    p->ev_quant = timing && u8 != nullptr;
    g_launches.fetch_add(n, std::memory_order_relaxed);
    return cudaGetLastError();
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

template <int LOG2M>
cudaError_t launch_t(sfd_plan *p, const void *holo, float2 *field, float *inten,
                     unsigned char *u8, double *mom, cudaStream_t st) {
    using TL = Tile<LOG2M>;
    const sfd_dev &d = p->d;
    const int N = d.N, V = d.V;
    unsigned int *vmax = u8 ? d.vmax : nullptr;
    if (u8) {
        field = nullptr;
        inten = d.inten_ws;
    }
    const bool timing = p->timing;
    if (timing) cudaEventRecord(p->ev[0], st);
    // programmatic dependent launch (as for the warp kernels): the launch latency of a kernel
    // overlaps the tail of the kernel before it; the small sizes are launch-bound
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(N / TL::C, V);
    cfg.blockDim = dim3(TL::THREADS_Y);
    cfg.dynamicSmemBytes = TL::SMEM_Y;
    cfg.stream = st;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    cudaError_t le;
    if (d.in_dtype == 0)
        le = cudaLaunchKernelEx(&cfg, k_pass_y<LOG2M, unsigned char>, (const unsigned char *)holo,
                                (const float2 *)d.pre_y, (const float2 *)d.H, (const float2 *)d.post_y,
                                (const float2 *)d.tw, d.B, vmax, mom);
    else
        le = cudaLaunchKernelEx(&cfg, k_pass_y<LOG2M, float>, (const float *)holo,
                                (const float2 *)d.pre_y, (const float2 *)d.H, (const float2 *)d.post_y,
                                (const float2 *)d.tw, d.B, vmax, mom);
    if (le != cudaSuccess) return le;
    if (timing) cudaEventRecord(p->ev[1], st);
    cfg.gridDim = dim3(N / TL::RPC, V);
    cfg.blockDim = dim3(TL::THREADS_X);
    cfg.dynamicSmemBytes = TL::SMEM_X;
    if (mom == nullptr)
        le = cudaLaunchKernelEx(&cfg, k_pass_x<LOG2M, false>, (const float2 *)d.B, (const float2 *)d.pre_x,
                                (const float2 *)d.Hx, (const float2 *)d.post_x, (const float2 *)d.tw, field,
                                inten, vmax, mom);
    else
        le = cudaLaunchKernelEx(&cfg, k_pass_x<LOG2M, true>, (const float2 *)d.B, (const float2 *)d.pre_x,
                                (const float2 *)d.Hx, (const float2 *)d.post_x, (const float2 *)d.tw, field,
                                inten, vmax, mom);
    if (le != cudaSuccess) return le;
    if (timing) cudaEventRecord(p->ev[2], st);
    int n = 2;
    if (u8) {
        const int quads = N * N / 4;
        dim3 gq((quads + 256 * 4 - 1) / (256 * 4), V);
        k_quantise<<<gq, 256, 0, st>>>((const float4 *)d.inten_ws, d.vmax, (uchar4 *)u8, quads);
        if (timing) cudaEventRecord(p->ev[3], st);
        ++n;
    }
    p->ev_valid = timing;
    p->ev_quant = timing && u8 != nullptr;
    g_launches.fetch_add(n, std::memory_order_relaxed);
    return cudaGetLastError();
}

}  // namespace

// Tensor map of the intermediate B for the bulk stores of k_cols_1024: B as float [V * N][2 N],
// box = 4 floats (two complex columns; N = 2048: 8 floats, four columns) x YBOX rows, no swizzle.  The encoder is a driver entry
// point; it is fetched through the runtime so that the library does not link libcuda.
cudaError_t sfd_make_tensormaps(sfd_plan *p) {
    static_assert(sizeof(CUtensorMap) <= sizeof(p->tmapB), "tensor map storage");
    if ((p->d.N != sfdw::N && p->d.N != sfdq::NL) || p->d.w_twl == nullptr) return cudaSuccess;
    const cuuint64_t n = (cuuint64_t)p->d.N;
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *,
                                  const cuuint64_t *, const cuuint64_t *, const cuuint32_t *,
                                  const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qr;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr);
    if (e != cudaSuccess) return e;
    if (fn == nullptr || qr != cudaDriverEntryPointSuccess) return cudaErrorNotSupported;
    const cuuint64_t dims[2] = {2 * n, (cuuint64_t)p->d.V * n};
    const cuuint64_t strides[1] = {2 * n * sizeof(float)};
    const cuuint32_t box[2] = {p->d.N == sfdq::NL ? (cuuint32_t)sfdq::YBOXW : 4u, sfdw::YBOX};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = ((encode_fn)fn)(
        reinterpret_cast<CUtensorMap *>(p->tmapB), CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, p->d.B, dims,
        strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
        CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

void sfd_count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }
long long sfd_launch_count_impl() { return g_launches.load(std::memory_order_relaxed); }

cudaError_t sfd_kernels_init() {
    cudaError_t e;
#define SFD_ATTR(L)                                                   \
    if ((e = set_attr<L, unsigned char>()) != cudaSuccess) return e;  \
    if ((e = set_attr<L, float>()) != cudaSuccess) return e;
    SFD_ATTR(7) SFD_ATTR(8) SFD_ATTR(9) SFD_ATTR(10) SFD_ATTR(11) SFD_ATTR(12)
#undef SFD_ATTR
    if ((e = cudaFuncSetAttribute(k_cols_1024<unsigned char>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)sizeof(sfdw::SmemY<unsigned char>))) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_cols_1024<float>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)sizeof(sfdw::SmemY<float>))) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_rows_1024, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)sizeof(sfdw::SmemX))) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_cols_2048<unsigned char>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)sizeof(sfdq::SmemYQ<unsigned char>))) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_cols_2048<float>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)sizeof(sfdq::SmemYQ<float>))) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_rows_2048, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)sizeof(sfdq::SmemXQ))) != cudaSuccess) return e;
    int dev = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&g_sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    return cudaSuccess;
}

cudaError_t sfd_launch(sfd_plan *p, const void *holo, float2 *field, float *inten,
                       unsigned char *u8, cudaStream_t st, double *mom) {
    // N = 1024: warp-pair-per-line kernels (their slab loads read 8 bytes of a hologram row at once:
    // the hologram must be aligned accordingly)
    if (p->d.N == sfdw::N && p->kernels != SFD_KERNELS_GENERIC && p->d.w_twl != nullptr &&
        (reinterpret_cast<size_t>(holo) & (p->d.in_dtype == 0 ? 7 : 15)) == 0)
        return launch_warp1024(p, holo, field, inten, u8, mom, st);
    if (p->d.N == sfdq::NL && p->kernels != SFD_KERNELS_GENERIC && p->d.w_twl != nullptr &&
        (reinterpret_cast<size_t>(holo) & (p->d.in_dtype == 0 ? 7 : 15)) == 0)
        return launch_warp2048(p, holo, field, inten, u8, mom, st);
    switch (p->d.log2M) {
        case 7: return launch_t<7>(p, holo, field, inten, u8, mom, st);
        case 8: return launch_t<8>(p, holo, field, inten, u8, mom, st);
        case 9: return launch_t<9>(p, holo, field, inten, u8, mom, st);
        case 10: return launch_t<10>(p, holo, field, inten, u8, mom, st);
        case 11: return launch_t<11>(p, holo, field, inten, u8, mom, st);
        case 12: return launch_t<12>(p, holo, field, inten, u8, mom, st);
    }
    return cudaErrorInvalidValue;
}
