// sfd_internal.h — what sfd_plan.cpp (host logic) and sfd_kernels.cu (device code) share.
#pragma once
#include <cuda_runtime.h>

#include "sfd.h"

#include <vector>

struct sfd_stream_state;  // pinned double-buffer pipeline (sfd_plan.cpp)

// Device-side description of a plan, passed by value to the launcher.
struct sfd_dev {
    int N = 0, M = 0, log2M = 0, V = 0, in_dtype = 0;
    // complex64 tables, one device allocation; per view contiguous
    float2 *pre_y = nullptr;   // [V][N]  Eq.(3) y-part (x 1/255 for uint8 input)
    float2 *post_y = nullptr;  // [V][N]  Eq.(2) y-part x c0
    float2 *pre_x = nullptr;   // [V][N]  Eq.(3) x-part
    float2 *post_x = nullptr;  // [V][N]  Eq.(2) x-part
    float2 *H = nullptr;       // [V][M]  y axis: FFT_M(h)/M, h of Eq.(4) wrapped, S = S_y
    float2 *Hx = nullptr;      // [V][M]  x axis: the same with S = S_x
    float2 *tw = nullptr;      // [M]     exp(-2 pi i x / M)
    // workspace
    float2 *B = nullptr;           // [V][N][N] intermediate between pass y and pass x
    float *inten_ws = nullptr;     // [V][N][N] intensity scratch of the 8-bit mode
    unsigned int *vmax = nullptr;  // [V] per-view max intensity (float bits)
    // N = 1024 fast path (sfd_warp1024.cuh); branch b = 0 even bins, 1 odd bins of the 2N-point DFT
    // per view and branch b: pre_b | H_b | conj(post_b), H_0[k] = H[2k], H_1[k] = H[2k+1]
    // (N = 2048, sfd_warp2048.cuh: four branches, [V][4][5][1024]: preA_b | preB_b | H_b | postA_b | postB_b)
    float2 *w_tabY = nullptr;  // [V][2][3][N]  pre carries 1/255 (uint8 input), post carries c0
    float2 *w_tabX = nullptr;  // [V][2][3][N]
    float2 *w_twl = nullptr;   // [32][32]   exp(-2 pi i lane k / 1024) at [k][lane]
};


struct sfd_plan {
    sfd_dev d;
    int device = 0;
    double lambda = 0;
    // per view; p1, p2, Ox, Oy are the x-axis values (and the y-axis ones in the square API)
    std::vector<double> p1, p2, z, Ox, Oy, p1y, p2y, O0x, O0y;
    void *table_alloc = nullptr;
    void *fast_alloc = nullptr;
    int kernels = SFD_KERNELS_AUTO;
    long long device_bytes = 0;
    bool timing = false;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    bool ev_valid = false, ev_quant = false;
    sfd_stream_state *ss = nullptr;
    // CUtensorMap of B (bulk stores of the N = 1024 pass y), built by sfd_make_tensormaps
    alignas(64) unsigned char tmapB[128] = {};
};

// Enqueue the kernels of one reconstruction on `st` (sfd_kernels.cu).  `u8` non-NULL selects the
// 8-bit mode (intensity into the plan's scratch, per-view max, quantise).  Returns a cudaError_t.
// `mom` non-NULL: [V][2] doubles on the device receive sum I and sum I^2 of every view (focus
// moments); field and inten may then both be NULL.
cudaError_t sfd_launch(sfd_plan *p, const void *holo, float2 *field, float *inten,
                       unsigned char *u8, cudaStream_t st, double *mom = nullptr);
// One-time per-process kernel attribute set-up (dynamic shared memory opt-in).
cudaError_t sfd_kernels_init();
void sfd_count_launch(int n);
// Builds the plan's tensor maps (after B is allocated; no-op when the fast path is not in use).
cudaError_t sfd_make_tensormaps(sfd_plan *p);
