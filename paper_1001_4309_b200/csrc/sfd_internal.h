// sfd_internal.h — what sfd_plan.cpp (host logic) and sfd_kernels.cu (device code) share.
#pragma once
#include <cuda_runtime.h>

#include "sfd.h"

#include <complex>
#include <vector>

struct sfd_stream_state;  // pinned double-buffer pipeline (sfd_plan.cpp)
struct sfd_update_ring;   // pinned staging slots of sfd_plan_update_view*_async (sfd_plan.cpp)

// Device-side description of a plan.  The grid is Ny rows (y, index n) by Nx columns (x, index m);
// pass y runs Nx lines of length Ny, pass x runs Ny lines of length Nx (padded to My = 2 Ny,
// Mx = 2 Nx inside the kernels).
//
// All tables of one view are contiguous (one H2D copy updates a view): view v starts at
// tabs + v * vstride and holds, at the offsets below (complex64 elements),
//   pre_y[Ny]   Eq.(3) y-part (x 1/255 for uint8 input)      post_y[Ny]  Eq.(2) y-part x c0
//   pre_x[Nx]   Eq.(3) x-part                                post_x[Nx]  Eq.(2) x-part
//   Hy[My]      FFT_My(h)/My, h of Eq.(4) wrapped, S = S_y   Hx[Mx]      the same with S = S_x
//   tabY, tabX  branch tables of the warp kernels for an axis of length 1024 ([2][3][1024]:
//               pre_b | H_b | conj(post_b), sfd_warp1024.cuh) or 2048 ([4][5][1024]:
//               preA_b | preB_b | H_b | postA_b | postB_b, sfd_warp2048.cuh); absent otherwise
struct sfd_dev {
    int Nx = 0, Ny = 0, Mx = 0, My = 0, log2Mx = 0, log2My = 0, V = 0, in_dtype = 0;
    float2 *tabs = nullptr;
    long long vstride = 0;
    int off_pre_y = 0, off_post_y = 0, off_pre_x = 0, off_post_x = 0, off_Hy = 0, off_Hx = 0;
    int off_tabY = -1, off_tabX = -1;  // -1: that axis runs the generic kernels
    float2 *tw_y = nullptr;   // [My] exp(-2 pi i x / My)   (generic kernels)
    float2 *tw_x = nullptr;   // [Mx]
    float2 *w_twl = nullptr;  // [31][32] stage-B twiddles of the warp FFT (sfd_dft32.cuh)
    // workspace
    float2 *B = nullptr;           // [V][Ny][Nx] intermediate between pass y and pass x
    float *inten_ws = nullptr;     // [V][Ny][Nx] intensity scratch of the 8-bit mode
    unsigned int *vmax = nullptr;  // [V] per-view max intensity (float bits)
    // hologram window inside the caller's frame (sfd_plan_set_input_window)
    long long in_stride = 0;  // elements between rows of the frame
    long long in_offset = 0;  // elements from the frame pointer to sample [0][0] of the window
    int sms = 0;              // multiprocessors of the plan's device
};

struct sfd_plan {
    sfd_dev d;
    int device = 0;
    double lambda = 0;
    // per view; p1, p2, Ox, Oy are the x-axis values (and the y-axis ones in the square API)
    std::vector<double> p1, p2, z, Ox, Oy, p1y, p2y, O0x, O0y;
    // host FFT twiddles of the table builder, exp(-2 pi i k / M) for k < M/2, per axis (cached:
    // they depend on the size only and dominate the cost of rebuilding a view)
    std::vector<std::complex<double>> wy, wx;
    void *table_alloc = nullptr;
    int kernels = SFD_KERNELS_AUTO;
    long long device_bytes = 0;
    bool timing = false;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    bool ev_valid = false, ev_quant = false;
    sfd_stream_state *ss = nullptr;
    sfd_update_ring *ur = nullptr;
    double last_update_host_ms = 0.0;
    // CUtensorMap of B (bulk stores of the warp pass y), built by sfd_make_tensormaps
    alignas(64) unsigned char tmapB[128] = {};
};

// Enqueue the kernels of one reconstruction on `st` (sfd_kernels.cu).  `holo` already points at
// sample [0][0] of the hologram window.  `u8` non-NULL selects the 8-bit mode (intensity into the
// plan's scratch, per-view max, quantise).  `mom` non-NULL: [V][2] doubles on the device receive
// sum I and sum I^2 of every view (focus moments); field and inten may then both be NULL.
cudaError_t sfd_launch(sfd_plan *p, const void *holo, float2 *field, float *inten,
                       unsigned char *u8, cudaStream_t st, double *mom = nullptr);
// true if pass y / pass x of this plan run the warp-per-branch kernels for a hologram at `holo`
bool sfd_uses_warp_y(const sfd_plan *p, const void *holo);
bool sfd_uses_warp_x(const sfd_plan *p);
// Per-device kernel attribute set-up (dynamic shared memory opt-in); call with the device current.
cudaError_t sfd_kernels_init(int device, int *sms);
void sfd_count_launch(int n);
// Builds the plan's tensor maps (after B is allocated; no-op when pass y runs the generic kernels).
cudaError_t sfd_make_tensormaps(sfd_plan *p);
// Tensor map (128 bytes at `out`, 64-byte aligned) of a complex64 matrix [rows][nx] seen as float
// [rows][2 nx], tiled in boxes of box_floats x box_rows (the column tiles of the warp kernels);
// swizzle = 32 / 64: the 16-byte chunks of a 32- / 64-byte box row are permuted in shared memory
// (SWIZZLE_32B / SWIZZLE_64B), 0: none
cudaError_t sfd_encode_rows_tmap(void *out, float2 *base, unsigned long long rows, int nx,
                                 unsigned box_floats, unsigned box_rows, int swizzle = 0);
// fp32 pipe micro-benchmarks (sfd_kernels.cu), see sfd_measure_pipes in sfd.h
cudaError_t sfd_measure_pipes_impl(double out[4]);
// host-side step of the register butterflies (sfd_kernels.cu, compiled for the host as well)
void sfd_host_dft32_impl(const float *in, float *out, int lane, int twiddled);
