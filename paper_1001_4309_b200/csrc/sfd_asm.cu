// sfd_asm.cu — angular-spectrum propagation on the line-FFT code of libsfd.
//
//     u(z) = IFFT2[ FFT2[u0] * H ],   H(fx, fy) = exp(i 2 pi z sqrt(1/lambda^2 - fx^2 - fy^2))
//
// on the periodic Ny x Nx grid (no padding), evanescent components cut, optionally band-limited
// (include/sfd.h, sfd_asm_plan_create).  The transfer function does not factorise into an x- and a
// y-part, so the two-pass trick of the Shifted-Fresnel path (reading 20) does not apply;
// the 2-D transforms are row and column line FFTs with the multiply fused between the forward and the
// inverse column transform:
//
//   k_asm_rows_fwd  per row:     u0 (real f32 or complex64) -> FFT_Nx                    -> A[ny][kx]
//   k_asm_cols      per column:  A -> FFT_Ny -> x H[plane][ky][kx] -> IFFT_Ny             -> W[plane][ny][kx]
//   k_asm_rows_inv  per row:     W -> IFFT_Nx -> field, |u|^2, arg u
//
// The row transform is shared by all planes (depths) of a plan.  H is cached per plan like the
// chirp-kernel spectra of the Fresnel path, built once on the device in float64 (the phase
// z sqrt(.) is about 1e5 cycles: float32 cannot hold it) with the 1/(Nx Ny) of the inverse folded in.
// Line FFTs: the Stockham register/shared-memory code of sfd_fft_core.cuh (fft_line), 128..4096
// points.  All three kernels are chained by programmatic dependent launch.  A 1024 x 1024 grid runs
// the same three steps as warp-FFT kernels (k_asm1024_*, sfd_asm1024.cuh) on a transposed,
// sign-folded copy of H.
#include <cuda.h>  // CUtensorMap (types only: the encoder is fetched through the runtime)
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <new>
#include <vector>

#include "sfd.h"
#include "sfd_asm1024.cuh"
#include "sfd_asm2048.cuh"
#include "sfd_fft_core.cuh"
#include "sfd_internal.h"

namespace {

using namespace sfd;

__device__ __forceinline__ void pdl_launch_dependents() {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

__device__ __forceinline__ float2 load_sample(const float *p, size_t i) { return make_float2(p[i], 0.f); }
__device__ __forceinline__ float2 load_sample(const float2 *p, size_t i) { return p[i]; }

// H[p][ky][kx] in float64, stored as complex64 with the 1/(Nx Ny) of the inverse transforms
// (warp_layout: transposed and sign-folded for the 1024 x 1024 kernels)
__global__ void __launch_bounds__(256)
k_asm_transfer(float2 *H, int Nx, int Ny, double lambda, double px, double py, const double *z,
               int band_limit, int warp_layout) {
    const int kx = blockIdx.x * blockDim.x + threadIdx.x, ky = blockIdx.y, p = blockIdx.z;
    if (kx >= Nx) return;
    const double fx = (double)(2 * kx < Nx ? kx : kx - Nx) / ((double)Nx * px);
    const double fy = (double)(2 * ky < Ny ? ky : ky - Ny) / ((double)Ny * py);
    const double w2 = 1.0 / (lambda * lambda) - fx * fx - fy * fy;
    bool keep = w2 > 0.0;
    if (band_limit) {
        const double dfx = 1.0 / ((double)Nx * px), dfy = 1.0 / ((double)Ny * py);
        const double flx = 1.0 / (lambda * sqrt((2.0 * dfx * z[p]) * (2.0 * dfx * z[p]) + 1.0));
        const double fly = 1.0 / (lambda * sqrt((2.0 * dfy * z[p]) * (2.0 * dfy * z[p]) + 1.0));
        keep = keep && fabs(fx) <= flx && fabs(fy) <= fly;
    }
    float2 h = make_float2(0.f, 0.f);
    if (keep) {
        double c = z[p] * sqrt(w2);
        c -= rint(c);
        double sn, cs;
        sincospi(2.0 * c, &sn, &cs);
        const double sc = 1.0 / ((double)Nx * (double)Ny);
        h = make_float2((float)(cs * sc), (float)(sn * sc));
    }
    if (!warp_layout) {
        H[((size_t)p * Ny + ky) * Nx + kx] = h;
    } else if (warp_layout == 1) {  // T_p[kx][ky] = sigma(ky) sigma(kx) H_p[ky][kx] / (Nx Ny), sfd_asm1024.cuh
        if ((__popc(kx) + __popc(ky)) & 1) h = make_float2(-h.x, -h.y);
        H[((size_t)p * Nx + kx) * Ny + ky] = h;
    } else {  // T_p[kx][ky & 1][ky >> 1] = sigma(ky >> 1) sigma(kx mod 1024) H_p[ky][kx] / (Nx Ny), sfd_asm2048.cuh
        if ((__popc(kx & 1023) + __popc(ky >> 1)) & 1) h = make_float2(-h.x, -h.y);
        H[(((size_t)p * Nx + kx) * 2 + (ky & 1)) * 1024 + (ky >> 1)] = h;
    }
}

// ---- 1024 x 1024: warp-FFT kernels (sfd_asm1024.cuh), 8 warps per CTA, one CTA per SM ---------------
template <typename TIn>
__global__ void __launch_bounds__(256, 1)
k_asm1024_rows_fwd(const TIn *u0, const float2 *__restrict__ twl, float2 *A, int rows) {
    extern __shared__ float4 smem4[];
    pdl_launch_dependents();
    sfda::rows_fwd<TIn>(*reinterpret_cast<sfda::SmemR *>(smem4), u0, twl, A, rows);
}

__global__ void __launch_bounds__(sfda::NTC, 1)
k_asm1024_cols(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmW,
               const float2 *__restrict__ Tt, const float2 *__restrict__ twl, int P) {
    extern __shared__ float4 smem4[];
    // the swizzle pattern of the tile is a function of the shared-memory address: 1024-byte alignment
    sfda::SmemC &sm = *reinterpret_cast<sfda::SmemC *>(
        (reinterpret_cast<uintptr_t>(smem4) + 1023) & ~(uintptr_t)1023);
    pdl_launch_dependents();
    if (threadIdx.x == 0) {
        for (int i = 0; i < sfda::NWA; ++i) sfdw::mbar_init(&sm.tbar[i], 1);
        sfdw::mbar_init(&sm.in_full, 1);
        sfdw::mbar_init(&sm.in_read, sfda::NWA);
        sfdw::mbar_init(&sm.staged, sfda::NWA);
        sfdw::mbar_init(&sm.empty, 1);
        sfdw::mbar_fence_init();
    }
    __syncthreads();
    sfda::cols(sm, &tmA, &tmW, Tt, twl, P);
}

// ---- 2048 x 2048: a pair of warps per line (sfd_asm2048.cuh) -----------------------------------------
template <typename TIn>
__global__ void __launch_bounds__(256, 1)
k_asm2048_rows_fwd(const TIn *u0, const float2 *__restrict__ twl, const float2 *__restrict__ w2048,
                   float2 *A, int rows) {
    extern __shared__ float4 smem4[];
    sfda2::SmemI2 &sm = *reinterpret_cast<sfda2::SmemI2 *>(smem4);
    pdl_launch_dependents();
    if (threadIdx.x == 0) {
        for (int i = 0; i < sfda2::NPAIR; ++i) sfdw::mbar_init(&sm.ibar[i], 1);
        sfdw::mbar_fence_init();
    }
    __syncthreads();
    sfda2::rows_fwd<TIn>(sm, u0, twl, w2048, A, rows);
}

__global__ void __launch_bounds__(sfda::NTC, 1)
k_asm2048_cols(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmW,
               const float2 *__restrict__ Tt, const float2 *__restrict__ twl,
               const float2 *__restrict__ w2048, int P) {
    extern __shared__ float4 smem4[];
    sfda2::SmemC2 &sm = *reinterpret_cast<sfda2::SmemC2 *>(
        (reinterpret_cast<uintptr_t>(smem4) + 1023) & ~(uintptr_t)1023);
    pdl_launch_dependents();
    if (threadIdx.x == 0) {
        for (int i = 0; i < sfda::NWA; ++i) sfdw::mbar_init(&sm.tbar[i], 1);
        sfdw::mbar_init(&sm.in_full, 1);
        sfdw::mbar_init(&sm.in_read, sfda::NWA);
        sfdw::mbar_init(&sm.staged, sfda::NWA);
        sfdw::mbar_init(&sm.empty, 1);
        sfdw::mbar_fence_init();
    }
    __syncthreads();
    sfda2::cols(sm, &tmA, &tmW, Tt, twl, w2048, P);
}

template <bool PHASE>
__global__ void __launch_bounds__(256, 1)
k_asm2048_rows_inv(const float2 *W, const float2 *__restrict__ twl, const float2 *__restrict__ w2048,
                   float2 *__restrict__ field, float *__restrict__ inten, float *__restrict__ phase,
                   int rows) {
    extern __shared__ float4 smem4[];
    sfda2::SmemI2 &sm = *reinterpret_cast<sfda2::SmemI2 *>(smem4);
    pdl_launch_dependents();
    if (threadIdx.x == 0) {
        for (int i = 0; i < sfda2::NPAIR; ++i) sfdw::mbar_init(&sm.ibar[i], 1);
        sfdw::mbar_fence_init();
    }
    __syncthreads();
    sfda2::rows_inv<PHASE>(sm, W, twl, w2048, field, inten, phase, rows);
}

template <bool PHASE>
__global__ void __launch_bounds__(256, 1)
k_asm1024_rows_inv(const float2 *W, const float2 *__restrict__ twl, float2 *__restrict__ field,
                   float *__restrict__ inten, float *__restrict__ phase, int rows) {
    extern __shared__ float4 smem4[];
    sfda::SmemI &sm = *reinterpret_cast<sfda::SmemI *>(smem4);
    pdl_launch_dependents();
    if (threadIdx.x == 0) {
        for (int i = 0; i < sfda::NWA; ++i) sfdw::mbar_init(&sm.ibar[i], 1);
        sfdw::mbar_fence_init();
    }
    __syncthreads();
    sfda::rows_inv<PHASE>(sm, W, twl, field, inten, phase, rows);
}

template <int LOG2N, typename TIn>
__global__ void __launch_bounds__(Tile<LOG2N>::THREADS_X)
k_asm_rows_fwd(const TIn *in, const float2 *__restrict__ tw, float2 *A) {
    extern __shared__ float2 smem[];
    using S = Sched<LOG2N>;
    constexpr int T = S::T, RPC = Tile<LOG2N>::RPC, Nx = S::M;
    pdl_launch_dependents();
    pdl_wait();
    const int l = threadIdx.x / T, j = threadIdx.x % T;
    const size_t row = (size_t)blockIdx.x * RPC + l;
    float2 v[16];
#pragma unroll
    for (int s = 0; s < 16; ++s) v[s] = load_sample(in, row * Nx + j + s * T);
    fft_line<LOG2N, -1, false, 1>(v, j, LineSmem<1>{smem + l * S::PADDED}, tw, [] { __syncthreads(); });
#pragma unroll
    for (int s = 0; s < 16; ++s) A[row * Nx + j + s * T] = v[s];
}

template <int LOG2N>
__global__ void __launch_bounds__(Tile<LOG2N>::THREADS_Y)
k_asm_cols(const float2 *A, const float2 *__restrict__ H, const float2 *__restrict__ tw, float2 *W,
           int nx) {
    extern __shared__ float2 smem[];
    using S = Sched<LOG2N>;
    constexpr int T = S::T, C = Tile<LOG2N>::C, Ny = S::M;
    pdl_launch_dependents();
    const int l = threadIdx.x % C, j = threadIdx.x / C;
    const int col = blockIdx.x * C + l;
    const size_t plane = (size_t)blockIdx.y * Ny * nx;
    float2 h[16];
#pragma unroll
    for (int s = 0; s < 16; ++s) h[s] = __ldg(H + plane + (size_t)(j + s * T) * nx + col);  // plan constant
    pdl_wait();  // A comes from the row pass
    float2 v[16];
#pragma unroll
    for (int s = 0; s < 16; ++s) v[s] = A[(size_t)(j + s * T) * nx + col];
    LineSmem<C> sm{smem + l};
    auto sync = [] { __syncthreads(); };
    fft_line<LOG2N, -1, false, C>(v, j, sm, tw, sync);
#pragma unroll
    for (int s = 0; s < 16; ++s) v[s] = cmul(v[s], h[s]);
    fft_line<LOG2N, +1, false, C>(v, j, sm, tw, sync);
#pragma unroll
    for (int s = 0; s < 16; ++s) W[plane + (size_t)(j + s * T) * nx + col] = v[s];
}

template <int LOG2N>
__global__ void __launch_bounds__(Tile<LOG2N>::THREADS_X)
k_asm_rows_inv(const float2 *W, const float2 *__restrict__ tw, float2 *__restrict__ field,
               float *__restrict__ inten, float *__restrict__ phase, int ny) {
    extern __shared__ float2 smem[];
    using S = Sched<LOG2N>;
    constexpr int T = S::T, RPC = Tile<LOG2N>::RPC, Nx = S::M;
    pdl_launch_dependents();
    pdl_wait();
    const int l = threadIdx.x / T, j = threadIdx.x % T;
    const size_t row = (size_t)blockIdx.y * ny + (size_t)blockIdx.x * RPC + l;
    float2 v[16];
#pragma unroll
    for (int s = 0; s < 16; ++s) v[s] = W[row * Nx + j + s * T];
    fft_line<LOG2N, +1, false, 1>(v, j, LineSmem<1>{smem + l * S::PADDED}, tw, [] { __syncthreads(); });
#pragma unroll
    for (int s = 0; s < 16; ++s) {
        const size_t o = row * Nx + j + s * T;
        const float2 u = v[s];
        if (field) field[o] = u;
        if (inten) inten[o] = u.x * u.x + u.y * u.y;
        if (phase) phase[o] = atan2f(u.y, u.x);
    }
}

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

}  // namespace

struct sfd_asm_plan {
    int Nx = 0, Ny = 0, lx = 0, ly = 0, P = 0, in_dtype = 0, band_limit = 0, device = 0;
    double lambda = 0, px = 0, py = 0;
    float2 *H = nullptr;     // [P][Ny][Nx]
    float2 *A = nullptr;     // [Ny][Nx]      row spectra of the input
    float2 *W = nullptr;     // [P][Ny][Nx]   after the column pass
    float2 *tw_x = nullptr;  // [Nx] exp(-2 pi i k / Nx)
    float2 *tw_y = nullptr;  // [Ny]
    // 1 = 1024 x 1024, 2 = 2048 x 2048: warp-FFT kernels; H holds T then (sfd_asm1024.cuh / sfd_asm2048.cuh)
    int warp = 0;
    int sms = 0;
    float2 *twl = nullptr;  // [31][32] stage-B twiddles of the warp FFT (sfd_dft32.cuh)
    alignas(64) unsigned char tmapA[128] = {};
    alignas(64) unsigned char tmapW[128] = {};
    long long device_bytes = 0;
};

namespace {

thread_local char g_asm_err[256] = "no CUDA error";
int asm_fail(cudaError_t e, const char *where) {
    std::snprintf(g_asm_err, sizeof g_asm_err, "%s: %s (%s)", where, cudaGetErrorName(e),
                  cudaGetErrorString(e));
    cudaGetLastError();
    return SFD_ECUDA;
}
#define ASM_CUDA(call)                                      \
    do {                                                    \
        cudaError_t e_ = (call);                            \
        if (e_ != cudaSuccess) return asm_fail(e_, #call);  \
    } while (0)

int log2_exact(int n) {
    if (n < 1) return -1;
    int l = 0;
    while ((1 << l) < n) ++l;
    return (1 << l) == n ? l : -1;
}

template <int L> cudaError_t asm_attrs() {
    cudaError_t e;
#define ASM_SMEM(kernel, bytes)                                                            \
    if ((e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,     \
                                  (int)(bytes))) != cudaSuccess)                           \
        return e;
    ASM_SMEM((k_asm_rows_fwd<L, float>), Tile<L>::SMEM_X)
    ASM_SMEM((k_asm_rows_fwd<L, float2>), Tile<L>::SMEM_X)
    ASM_SMEM((k_asm_cols<L>), Tile<L>::SMEM_Y)
    ASM_SMEM((k_asm_rows_inv<L>), Tile<L>::SMEM_X)
#undef ASM_SMEM
    return cudaSuccess;
}

template <int L>
cudaError_t rows_fwd(const sfd_asm_plan *p, const void *in, cudaStream_t st) {
    Launch l(dim3(p->Ny / Tile<L>::RPC), dim3(Tile<L>::THREADS_X), Tile<L>::SMEM_X, st);
    if (p->in_dtype == SFD_F32)
        return cudaLaunchKernelEx(&l.cfg, k_asm_rows_fwd<L, float>, (const float *)in,
                                  (const float2 *)p->tw_x, p->A);
    return cudaLaunchKernelEx(&l.cfg, k_asm_rows_fwd<L, float2>, (const float2 *)in,
                              (const float2 *)p->tw_x, p->A);
}
template <int L> cudaError_t cols(const sfd_asm_plan *p, cudaStream_t st) {
    Launch l(dim3(p->Nx / Tile<L>::C, p->P), dim3(Tile<L>::THREADS_Y), Tile<L>::SMEM_Y, st);
    return cudaLaunchKernelEx(&l.cfg, k_asm_cols<L>, (const float2 *)p->A, (const float2 *)p->H,
                              (const float2 *)p->tw_y, p->W, p->Nx);
}
template <int L>
cudaError_t rows_inv(const sfd_asm_plan *p, float2 *field, float *inten, float *phase,
                     cudaStream_t st) {
    Launch l(dim3(p->Ny / Tile<L>::RPC, p->P), dim3(Tile<L>::THREADS_X), Tile<L>::SMEM_X, st);
    return cudaLaunchKernelEx(&l.cfg, k_asm_rows_inv<L>, (const float2 *)p->W, (const float2 *)p->tw_x,
                              field, inten, phase, p->Ny);
}

#define ASM_DISPATCH(log2n, call)                 \
    switch (log2n) {                              \
        case 7: return call<7>;                   \
        case 8: return call<8>;                   \
        case 9: return call<9>;                   \
        case 10: return call<10>;                 \
        case 11: return call<11>;                 \
        case 12: return call<12>;                 \
    }                                             \
    return nullptr;

typedef cudaError_t (*fwd_fn)(const sfd_asm_plan *, const void *, cudaStream_t);
typedef cudaError_t (*cols_fn)(const sfd_asm_plan *, cudaStream_t);
typedef cudaError_t (*inv_fn)(const sfd_asm_plan *, float2 *, float *, float *, cudaStream_t);
fwd_fn pick_fwd(int l) { ASM_DISPATCH(l, rows_fwd) }
cols_fn pick_cols(int l) { ASM_DISPATCH(l, cols) }
inv_fn pick_inv(int l) { ASM_DISPATCH(l, rows_inv) }

cudaError_t asm_attrs_1024() {
    cudaError_t e;
#define ASM_SMEM(kernel, bytes)                                                            \
    if ((e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,     \
                                  (int)(bytes))) != cudaSuccess)                           \
        return e;
    ASM_SMEM(k_asm1024_rows_fwd<float>, sizeof(sfda::SmemR))
    ASM_SMEM(k_asm1024_rows_fwd<float2>, sizeof(sfda::SmemR))
    ASM_SMEM(k_asm1024_cols, sizeof(sfda::SmemC) + 1024)
    ASM_SMEM(k_asm1024_rows_inv<false>, sizeof(sfda::SmemI))
    ASM_SMEM(k_asm1024_rows_inv<true>, sizeof(sfda::SmemI))
    ASM_SMEM(k_asm2048_rows_fwd<float>, sizeof(sfda2::SmemI2))
    ASM_SMEM(k_asm2048_rows_fwd<float2>, sizeof(sfda2::SmemI2))
    ASM_SMEM(k_asm2048_cols, sizeof(sfda2::SmemC2) + 1024)
    ASM_SMEM(k_asm2048_rows_inv<false>, sizeof(sfda2::SmemI2))
    ASM_SMEM(k_asm2048_rows_inv<true>, sizeof(sfda2::SmemI2))
#undef ASM_SMEM
    return cudaSuccess;
}

// the three kernels of the 1024 x 1024 path
cudaError_t launch_1024(const sfd_asm_plan *p, const void *in, float2 *field, float *inten,
                        float *phase, cudaStream_t st) {
    constexpr int NW = sfda::NWA, N = sfdw::N;
    cudaError_t e;
    {
        Launch l(dim3(N / NW), dim3(32 * NW), sizeof(sfda::SmemR), st);
        if (p->in_dtype == SFD_F32)
            e = cudaLaunchKernelEx(&l.cfg, k_asm1024_rows_fwd<float>, (const float *)in,
                                   (const float2 *)p->twl, p->A, N);
        else
            e = cudaLaunchKernelEx(&l.cfg, k_asm1024_rows_fwd<float2>, (const float2 *)in,
                                   (const float2 *)p->twl, p->A, N);
        if (e != cudaSuccess) return e;
    }
    {
        Launch l(dim3(N / NW), dim3(sfda::NTC), sizeof(sfda::SmemC) + 1024, st);
        e = cudaLaunchKernelEx(&l.cfg, k_asm1024_cols, *reinterpret_cast<const CUtensorMap *>(p->tmapA),
                               *reinterpret_cast<const CUtensorMap *>(p->tmapW), (const float2 *)p->H,
                               (const float2 *)p->twl, p->P);
        if (e != cudaSuccess) return e;
    }
    const int rows = p->P * N, ctas = rows / NW < p->sms ? rows / NW : p->sms;
    Launch l(dim3(ctas), dim3(32 * NW), sizeof(sfda::SmemI), st);
    if (phase)
        return cudaLaunchKernelEx(&l.cfg, k_asm1024_rows_inv<true>, (const float2 *)p->W,
                                  (const float2 *)p->twl, field, inten, phase, rows);
    return cudaLaunchKernelEx(&l.cfg, k_asm1024_rows_inv<false>, (const float2 *)p->W,
                              (const float2 *)p->twl, field, inten, phase, rows);
}

// the three kernels of the 2048 x 2048 path
cudaError_t launch_2048(const sfd_asm_plan *p, const void *in, float2 *field, float *inten,
                        float *phase, cudaStream_t st) {
    constexpr int NW = sfda::NWA, NP = sfda2::NPAIR, NL = sfda2::NL;
    const float2 *w = p->tw_x;  // exp(-2 pi i k / 2048): its first 1024 entries are the radix-2 twiddles
    cudaError_t e;
    {
        Launch l(dim3(NL / NP < p->sms ? NL / NP : p->sms), dim3(32 * NW), sizeof(sfda2::SmemI2), st);
        if (p->in_dtype == SFD_F32)
            e = cudaLaunchKernelEx(&l.cfg, k_asm2048_rows_fwd<float>, (const float *)in,
                                   (const float2 *)p->twl, w, p->A, NL);
        else
            e = cudaLaunchKernelEx(&l.cfg, k_asm2048_rows_fwd<float2>, (const float2 *)in,
                                   (const float2 *)p->twl, w, p->A, NL);
        if (e != cudaSuccess) return e;
    }
    {
        Launch l(dim3(NL / NP < p->sms ? NL / NP : p->sms), dim3(sfda::NTC), sizeof(sfda2::SmemC2) + 1024, st);
        e = cudaLaunchKernelEx(&l.cfg, k_asm2048_cols, *reinterpret_cast<const CUtensorMap *>(p->tmapA),
                               *reinterpret_cast<const CUtensorMap *>(p->tmapW), (const float2 *)p->H,
                               (const float2 *)p->twl, w, p->P);
        if (e != cudaSuccess) return e;
    }
    const int rows = p->P * NL, ctas = rows / NP < p->sms ? rows / NP : p->sms;
    Launch l(dim3(ctas), dim3(32 * NW), sizeof(sfda2::SmemI2), st);
    if (phase)
        return cudaLaunchKernelEx(&l.cfg, k_asm2048_rows_inv<true>, (const float2 *)p->W,
                                  (const float2 *)p->twl, w, field, inten, phase, rows);
    return cudaLaunchKernelEx(&l.cfg, k_asm2048_rows_inv<false>, (const float2 *)p->W,
                              (const float2 *)p->twl, w, field, inten, phase, rows);
}

bool g_attr_done[64] = {};

}  // namespace

extern "C" {

int sfd_asm_plan_create(sfd_asm_plan **out, int Nx, int Ny, int n_planes, double lambda, double px,
                        double py, const double *z, int in_dtype, int band_limit) {
    if (!out) return SFD_EINVAL;
    *out = nullptr;
    if (!z || Nx < 1 || Ny < 1 || n_planes < 1) return SFD_EINVAL;
    if (!(lambda > 0.0) || !(px > 0.0) || !(py > 0.0) || !std::isfinite(lambda) ||
        !std::isfinite(px) || !std::isfinite(py))
        return SFD_EINVAL;
    for (int i = 0; i < n_planes; ++i)
        if (!std::isfinite(z[i])) return SFD_EINVAL;
    if (in_dtype != SFD_F32 && in_dtype != SFD_C64) return SFD_EINVAL;
    const int lx = log2_exact(Nx), ly = log2_exact(Ny);
    if (lx < 7 || lx > 12 || ly < 7 || ly > 12) return SFD_EUNSUPPORTED;
    int device = 0;
    ASM_CUDA(cudaGetDevice(&device));
    if (device < 0 || device >= 64) return SFD_EUNSUPPORTED;
    if (!g_attr_done[device]) {  // dynamic shared-memory opt-in, once per device
        ASM_CUDA(asm_attrs<7>());
        ASM_CUDA(asm_attrs<8>());
        ASM_CUDA(asm_attrs<9>());
        ASM_CUDA(asm_attrs<10>());
        ASM_CUDA(asm_attrs<11>());
        ASM_CUDA(asm_attrs<12>());
        ASM_CUDA(asm_attrs_1024());
        g_attr_done[device] = true;
    }
    sfd_asm_plan *p = new (std::nothrow) sfd_asm_plan;
    if (!p) return SFD_ENOMEM;
    p->Nx = Nx; p->Ny = Ny; p->lx = lx; p->ly = ly; p->P = n_planes;
    p->in_dtype = in_dtype; p->band_limit = band_limit != 0; p->device = device;
    p->lambda = lambda; p->px = px; p->py = py;
    p->warp = Nx == sfdw::N && Ny == sfdw::N ? 1 : Nx == sfda2::NL && Ny == sfda2::NL ? 2 : 0;
    ASM_CUDA(cudaDeviceGetAttribute(&p->sms, cudaDevAttrMultiProcessorCount, device));
    const size_t nn = (size_t)Nx * Ny, P = n_planes;
    auto fail = [&](int code) {
        sfd_asm_plan_destroy(p);
        return code;
    };
    cudaError_t e;
    if ((e = cudaMalloc((void **)&p->H, P * nn * sizeof(float2))) != cudaSuccess ||
        (e = cudaMalloc((void **)&p->W, P * nn * sizeof(float2))) != cudaSuccess ||
        (e = cudaMalloc((void **)&p->A, nn * sizeof(float2))) != cudaSuccess ||
        (e = cudaMalloc((void **)&p->tw_x, (size_t)(Nx + Ny + 32 * 32) * sizeof(float2))) != cudaSuccess)
        return fail(e == cudaErrorMemoryAllocation ? SFD_ENOMEM : asm_fail(e, "cudaMalloc"));
    p->tw_y = p->tw_x + Nx;
    p->twl = p->tw_y + Ny;
    p->device_bytes =
        (long long)((2 * P + 1) * nn * sizeof(float2) + (size_t)(Nx + Ny + 32 * 32) * sizeof(float2));
    {
        std::vector<float2> tw((size_t)Nx + Ny + 32 * 32, make_float2(0.f, 0.f));
        const long double two_pi = 6.283185307179586476925286766559005768L;
        // stage-B twiddles of the warp FFT: [j][lane], j = n/2 - 1 + k, exp(-2 pi i (lane + 32 k)/(32 n))
        for (int n = 2; n <= 32; n *= 2)
            for (int k = 0; k < n / 2; ++k)
                for (int lane = 0; lane < 32; ++lane) {
                    const long double a = two_pi * (lane + 32 * k) / (32 * n);
                    tw[(size_t)Nx + Ny + (n / 2 - 1 + k) * 32 + lane] =
                        make_float2((float)cosl(a), (float)-sinl(a));
                }
        for (int k = 0; k < Nx; ++k)
            tw[k] = make_float2((float)cosl(two_pi * k / Nx), (float)-sinl(two_pi * k / Nx));
        for (int k = 0; k < Ny; ++k)
            tw[(size_t)Nx + k] = make_float2((float)cosl(two_pi * k / Ny), (float)-sinl(two_pi * k / Ny));
        if ((e = cudaMemcpy(p->tw_x, tw.data(), tw.size() * sizeof(float2), cudaMemcpyHostToDevice)) !=
            cudaSuccess)
            return fail(asm_fail(e, "cudaMemcpy twiddles"));
    }
    double *zd = nullptr;
    if ((e = cudaMalloc((void **)&zd, P * sizeof(double))) != cudaSuccess)
        return fail(asm_fail(e, "cudaMalloc z"));
    e = cudaMemcpy(zd, z, P * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        k_asm_transfer<<<dim3((Nx + 255) / 256, Ny, n_planes), 256>>>(p->H, Nx, Ny, lambda, px, py, zd,
                                                                     p->band_limit, p->warp);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    cudaFree(zd);
    if (e != cudaSuccess) return fail(asm_fail(e, "k_asm_transfer"));
    if (p->warp) {
        static_assert(sizeof(CUtensorMap) <= sizeof(p->tmapA), "tensor map storage");
        // column tiles: 8 columns (64-byte rows) at 1024, 4 columns (32-byte rows) at 2048
        const unsigned bw = p->warp == 1 ? 2 * sfda::NWA : 2 * sfda2::NPAIR;
        const int swz = p->warp == 1 ? 64 : 32;
        if ((e = sfd_encode_rows_tmap(p->tmapA, p->A, (unsigned long long)Ny, Nx, bw, sfdw::YBOX, swz)) !=
                cudaSuccess ||
            (e = sfd_encode_rows_tmap(p->tmapW, p->W, P * (unsigned long long)Ny, Nx, bw, sfdw::YBOX, swz)) !=
                cudaSuccess)
            return fail(asm_fail(e, "cuTensorMapEncodeTiled"));
    }
    sfd_count_launch(1);
    *out = p;
    return SFD_OK;
}

int sfd_asm_execute(sfd_asm_plan *p, const void *u0_dev, void *field_dev, float *intensity_dev,
                    float *phase_dev, void *stream) {
    if (!p || !u0_dev || (!field_dev && !intensity_dev && !phase_dev)) return SFD_EINVAL;
    // the 2048 x 2048 kernels fetch input rows as bulk copies
    if (p->warp == 2 && (reinterpret_cast<uintptr_t>(u0_dev) & 15) != 0) return SFD_EINVAL;
    int prev = -1;
    ASM_CUDA(cudaGetDevice(&prev));
    if (prev != p->device) ASM_CUDA(cudaSetDevice(p->device));
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e;
    if (p->warp == 1) {
        e = launch_1024(p, u0_dev, (float2 *)field_dev, intensity_dev, phase_dev, st);
    } else if (p->warp == 2) {
        e = launch_2048(p, u0_dev, (float2 *)field_dev, intensity_dev, phase_dev, st);
    } else {
        e = pick_fwd(p->lx)(p, u0_dev, st);
        if (e == cudaSuccess) e = pick_cols(p->ly)(p, st);
        if (e == cudaSuccess) e = pick_inv(p->lx)(p, (float2 *)field_dev, intensity_dev, phase_dev, st);
    }
    if (prev != p->device) cudaSetDevice(prev);
    if (e != cudaSuccess) return asm_fail(e, "sfd_asm_execute");
    sfd_count_launch(3);
    return SFD_OK;
}

int sfd_asm_plan_destroy(sfd_asm_plan *p) {
    if (!p) return SFD_OK;
    int prev = -1;
    if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
    if (prev != p->device) cudaSetDevice(p->device);
    if (p->H) cudaFree(p->H);
    if (p->W) cudaFree(p->W);
    if (p->A) cudaFree(p->A);
    if (p->tw_x) cudaFree(p->tw_x);
    if (prev >= 0 && prev != p->device) cudaSetDevice(prev);
    delete p;
    return SFD_OK;
}

long long sfd_asm_plan_device_bytes(const sfd_asm_plan *p) { return p ? p->device_bytes : SFD_EINVAL; }

const char *sfd_asm_last_cuda_error(void) { return g_asm_err; }

}  // extern "C"
