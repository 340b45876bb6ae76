// sfd_plan.cpp — host side of libsfd: argument checking, the float64 table builder, plan life
// cycle, execute entry points, live view updates and the pinned double-buffered real-time stream.
//
// Tables (Eq.(2)-(4), L58-65, with the readings of DESIGN.md §3): every phase is formed in
// cycles in extended precision, reduced modulo 1, summed and only then turned into a complex
// number, so the float32 values that reach the GPU carry one rounding each.
#include <cuda_runtime.h>

#include <chrono>
#include <cmath>
#include <complex>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "sfd.h"
#include "sfd_internal.h"

long long sfd_launch_count_impl();

namespace {

typedef long double ld;
typedef std::complex<double> cd;

thread_local char g_cuda_err[256] = "no CUDA error";

int cuda_fail(cudaError_t e, const char *where) {
    std::snprintf(g_cuda_err, sizeof g_cuda_err, "%s: %s (%s)", where, cudaGetErrorName(e),
                  cudaGetErrorString(e));
    cudaGetLastError();  // clear the sticky-less error state
    return SFD_ECUDA;
}
#define SFD_CUDA(call)                                          \
    do {                                                        \
        cudaError_t e_ = (call);                                \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call);     \
    } while (0)

// Makes the plan's device current for the duration of a call and restores the caller's device.
class DeviceGuard {
public:
    explicit DeviceGuard(int want) {
        if (cudaGetDevice(&prev_) != cudaSuccess) {
            prev_ = -1;
            cudaGetLastError();
        }
        if (prev_ != want) {
            err_ = cudaSetDevice(want);
            switched_ = err_ == cudaSuccess;
        }
    }
    ~DeviceGuard() {
        if (switched_ && prev_ >= 0) cudaSetDevice(prev_);
    }
    cudaError_t error() const { return err_; }

private:
    int prev_ = -1;
    bool switched_ = false;
    cudaError_t err_ = cudaSuccess;
};
#define SFD_ON_DEVICE(p)                                                         \
    DeviceGuard guard_((p)->device);                                             \
    if (guard_.error() != cudaSuccess) return cuda_fail(guard_.error(), "cudaSetDevice")

const ld TWO_PI = 6.283185307179586476925286766559005768L;

inline ld frac1(ld c) { return c - rintl(c); }  // cycles -> (-1/2, 1/2]
// exp(2 pi i c): the phase is summed and reduced modulo 1 in extended precision (it reaches 1e5
// cycles); the reduced phase |c| <= 1/2 then goes through the double-precision sincos (error 1e-16,
// nine orders below the float32 rounding that follows, and five times faster than cosl/sinl: the
// table builder is what a live view update costs on the host)
inline cd cis_cycles(ld c) {
    const double r = (double)(TWO_PI * frac1(c));
    double sn, cs;
    sincos(r, &sn, &cs);
    return cd(cs, sn);
}

// exp(-2 pi i k / n), k < n/2, evaluated directly (no recurrence)
std::vector<cd> fft_twiddles(size_t n) {
    std::vector<cd> w(n / 2);
    for (size_t k = 0; k < n / 2; ++k) w[k] = cis_cycles(-(ld)k / (ld)n);
    return w;
}

// In-place radix-2 FFT, double, forward sign; w = fft_twiddles(a.size()).
void fft_host(std::vector<cd> &a, const std::vector<cd> &w) {
    const size_t n = a.size();
    for (size_t i = 1, j = 0; i < n; ++i) {
        size_t bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) std::swap(a[i], a[j]);
    }
    for (size_t len = 2; len <= n; len <<= 1) {
        const size_t step = n / len;
        for (size_t i = 0; i < n; i += len)
            for (size_t k = 0; k < len / 2; ++k) {
                cd u = a[i + k], t = a[i + k + len / 2] * w[k * step];
                a[i + k] = u + t;
                a[i + k + len / 2] = u - t;
            }
    }
}

// One axis of one view.  `off` is the shift of the reconstruction window along this axis, `off0`
// the shift of the hologram window (O_x0 / O_y0 of Eq.(2)-(3), L58-62; 0 in the square API).
//   pre[m]  = exp(i pi x0^2/(lambda z)) exp(-i 2 pi m p1 a1/(lambda z)) exp(-i pi S m^2)   Eq.(3)
//   post[m] = exp(i pi x1^2/(lambda z)) exp(-i 2 pi a0 x1/(lambda z)) exp(-i pi S m^2)     Eq.(2)
// with x0 = a0 + m p1, a0 = -N/2 p1 + off0, x1 = a1 + m p2, a1 = -N/2 p2 + off,
// S = p1 p2/(lambda z).
void axis_tables(int N, double lambda, double p1, double p2, double z, double off, cd *pre,
                 cd *post, double off0 = 0.0) {
    const ld lz = (ld)lambda * (ld)z;
    const ld S = (ld)p1 * (ld)p2 / lz;
    const ld a0 = -(ld)N / 2 * (ld)p1 + (ld)off0;
    const ld a1 = -(ld)N / 2 * (ld)p2 + (ld)off;
    for (int m = 0; m < N; ++m) {
        const ld x0 = a0 + (ld)m * p1, x1 = a1 + (ld)m * p2;
        const ld chirp = frac1(-S * (ld)m * (ld)m / 2);
        pre[m] = cis_cycles(frac1(x0 * x0 / (2 * lz)) + frac1(-(ld)m * p1 * a1 / lz) + chirp);
        post[m] = cis_cycles(frac1(x1 * x1 / (2 * lz)) + frac1(-a0 * x1 / lz) + chirp);
    }
}

// Spectrum of the wrapped 1-D chirp kernel of Eq.(4): h[j] = exp(i pi S d^2), d = j (j <= N),
// d = j - M (j > N), M = 2N; returns FFT_M(h)/M (the 1/M of the inverse FFT folded in, reading 8).
// w = fft_twiddles(M).
void kernel_spectrum(int N, double lambda, double p1, double p2, double z, cd *H,
                     const std::vector<cd> &w) {
    const int M = 2 * N;
    const ld S = (ld)p1 * (ld)p2 / ((ld)lambda * (ld)z);
    std::vector<cd> h(M);
    for (int j = 0; j < M; ++j) {
        const ld d = j <= N ? (ld)j : (ld)(j - M);
        h[j] = cis_cycles(S * d * d / 2);
    }
    fft_host(h, w);
    for (int k = 0; k < M; ++k) H[k] = h[k] / (double)M;
}

// c0 = p1x p1y exp(i 2 pi z/lambda) / (i lambda z)   (constant of Eq.(2) times the area element)
cd c0_factor(double lambda, double p1x, double p1y, double z) {
    const cd e = cis_cycles((ld)z / (ld)lambda);
    return (p1x * p1y) * e / (cd(0, 1) * (lambda * z));
}

bool finite_pos(double v) { return std::isfinite(v) && v > 0.0; }

int check_view(double lambda, double p1, double p2, double z, double Ox, double Oy) {
    if (!finite_pos(lambda) || !finite_pos(p1) || !finite_pos(p2)) return SFD_EINVAL;
    if (!std::isfinite(z) || z == 0.0) return SFD_EINVAL;
    if (!std::isfinite(Ox) || !std::isfinite(Oy)) return SFD_EINVAL;
    return SFD_OK;
}

int log2_exact(int n) {
    if (n < 1) return -1;
    int l = 0;
    while ((1 << l) < n) ++l;
    return (1 << l) == n ? l : -1;
}

void to_f32(const cd *src, float2 *dst, size_t n, cd scale = cd(1, 0)) {
    for (size_t i = 0; i < n; ++i) {
        const cd v = src[i] * scale;
        dst[i] = make_float2((float)v.real(), (float)v.imag());
    }
}

// The butterflies of the warp FFT leave stage-A output k1 multiplied by (-1)^popcount(k1) (sign
// tracking, sfd_dft32.cuh); k1 is the lane that multiplies table entry lane + 32 r after stage B, so
// the sign goes into every table that follows an FFT (H_b and the post tables).
double lane_sign(int n) {
    const int l = n & 31;
    return ((l ^ (l >> 1) ^ (l >> 2) ^ (l >> 3) ^ (l >> 4)) & 1) ? -1.0 : 1.0;
}

// Branch tables of an axis of length 1024 (sfd_warp1024.cuh): the 2N-point DFT split by the parity
// of the frequency index, w = exp(-2 pi i / 2N); layout [2][3][N]: for branch b the vectors
//   pre_b = pre w^(b n),  H_b[k] = H[2k + b],  conj(post_b) = conj(post w^(-b n))
// (each times its scale; H = the float32 M-point kernel spectrum), formed in float64.
// tw = fft_twiddles(2N): tw[n] = exp(-2 pi i n / 2N) = w^n.
void branch_tables(int N, const cd *pre, const cd *post, cd pre_scale, cd post_scale,
                   const float2 *H, float2 *out, const std::vector<cd> &tw) {
    for (int n = 0; n < N; ++n) {
        const cd w = tw[n];
        const float sg = (float)lane_sign(n);
        const cd t[4] = {pre[n] * pre_scale, pre[n] * pre_scale * w,
                         (double)sg * std::conj(post[n] * post_scale),
                         (double)sg * std::conj(post[n] * post_scale * std::conj(w))};
        for (int b = 0; b < 2; ++b) {
            float2 *o = out + (size_t)b * 3 * N;
            o[n] = make_float2((float)t[b].real(), (float)t[b].imag());
            o[N + n] = make_float2(sg * H[2 * n + b].x, sg * H[2 * n + b].y);
            o[2 * N + n] = make_float2((float)t[2 + b].real(), (float)t[2 + b].imag());
        }
    }
}

// Tables of an axis of length 2048 (sfd_warp2048.cuh): the 4096-point DFT split by the frequency
// index modulo 4, w = exp(-2 pi i / 4096); layout [4][5][1024]: for branch b the vectors
//   preA_b = pre[n] w^(b n), preB_b = pre[n+1024] w^(b (n+1024)), H_b[k] = H[4k+b],
//   postA_b = post[n] w^(-b n), postB_b = post[n+1024] w^(-b (n+1024))            (n, k < 1024)
// tw = fft_twiddles(4096): w^e = tw[e] for e < 2048, -tw[e - 2048] above.
void branch_tables4(const cd *pre, const cd *post, cd pre_scale, cd post_scale, const float2 *H,
                    float2 *out, const std::vector<cd> &tw) {
    const int Nb = 1024;
    for (int b = 0; b < 4; ++b)
        for (int n = 0; n < Nb; ++n) {
            float2 *o = out + (size_t)b * 5 * Nb + n;
            for (int half = 0; half < 2; ++half) {
                const int m = n + half * Nb;
                const int e = (b * m) & 4095;
                const cd w = e < 2048 ? tw[e] : -tw[e - 2048];
                const cd a = pre[m] * pre_scale * w,
                         c = lane_sign(n) * post[m] * post_scale * std::conj(w);
                o[(size_t)half * Nb] = make_float2((float)a.real(), (float)a.imag());
                o[(size_t)(3 + half) * Nb] = make_float2((float)c.real(), (float)c.imag());
            }
            o[(size_t)2 * Nb] = make_float2((float)lane_sign(n) * H[4 * n + b].x,
                                            (float)lane_sign(n) * H[4 * n + b].y);
        }
}

// Tables of an axis of length 512 (sfd_warp512.cuh): the padded transform is the 1024-point warp FFT
// itself, no branch split; layout pre[512] | H[1024] | conj(post)[512], the two tables that follow an
// FFT with the lane sign.
void tables512(const cd *pre, const cd *post, cd pre_scale, cd post_scale, const float2 *H,
               float2 *out) {
    for (int n = 0; n < 512; ++n) {
        const cd a = pre[n] * pre_scale, c = lane_sign(n) * std::conj(post[n] * post_scale);
        out[n] = make_float2((float)a.real(), (float)a.imag());
        out[512 + 1024 + n] = make_float2((float)c.real(), (float)c.imag());
    }
    for (int k = 0; k < 1024; ++k) {
        const float sg = (float)lane_sign(k);
        out[512 + k] = make_float2(sg * H[k].x, sg * H[k].y);
    }
}

size_t fast_elems(int n) {
    return n == 512 ? (size_t)2048 : n == 1024 ? 6 * (size_t)1024 : n == 2048 ? 20 * (size_t)1024 : 0;
}

// All float32 tables of view v in the device layout of sfd_dev (one contiguous block of
// d.vstride complex values).  The y axis uses (p1y, p2y, O0y, Oy), the x axis (p1, p2, O0x, Ox):
// S_x and S_y may differ (Eq.(2)-(4), L58-67).
void build_view_f32(const sfd_plan *p, int v, float2 *out) {
    const sfd_dev &d = p->d;
    const int nmax = d.Nx > d.Ny ? d.Nx : d.Ny;
    std::vector<cd> a(nmax), b(nmax), h(2 * (size_t)nmax);
    const double in_scale = d.in_dtype == SFD_U8 ? 1.0 / 255.0 : 1.0;
    const cd c0 = c0_factor(p->lambda, p->p1[v], p->p1y[v], p->z[v]);
    float2 *Hy = out + d.off_Hy, *Hx = out + d.off_Hx;
    // y axis
    kernel_spectrum(d.Ny, p->lambda, p->p1y[v], p->p2y[v], p->z[v], h.data(), p->wy);
    to_f32(h.data(), Hy, d.My);
    axis_tables(d.Ny, p->lambda, p->p1y[v], p->p2y[v], p->z[v], p->Oy[v], a.data(), b.data(),
                p->O0y[v]);
    to_f32(a.data(), out + d.off_pre_y, d.Ny, cd(in_scale, 0));
    to_f32(b.data(), out + d.off_post_y, d.Ny, c0);
    if (d.off_tabY >= 0 && d.Ny == 512)
        tables512(a.data(), b.data(), cd(in_scale, 0), c0, Hy, out + d.off_tabY);
    if (d.off_tabY >= 0 && d.Ny == 1024)
        branch_tables(d.Ny, a.data(), b.data(), cd(in_scale, 0), c0, Hy, out + d.off_tabY, p->wy);
    if (d.off_tabY >= 0 && d.Ny == 2048)
        branch_tables4(a.data(), b.data(), cd(in_scale, 0), c0, Hy, out + d.off_tabY, p->wy);
    // x axis
    kernel_spectrum(d.Nx, p->lambda, p->p1[v], p->p2[v], p->z[v], h.data(), p->wx);
    to_f32(h.data(), Hx, d.Mx);
    axis_tables(d.Nx, p->lambda, p->p1[v], p->p2[v], p->z[v], p->Ox[v], a.data(), b.data(),
                p->O0x[v]);
    to_f32(a.data(), out + d.off_pre_x, d.Nx);
    to_f32(b.data(), out + d.off_post_x, d.Nx);
    if (d.off_tabX >= 0 && d.Nx == 512)
        tables512(a.data(), b.data(), cd(1, 0), cd(1, 0), Hx, out + d.off_tabX);
    if (d.off_tabX >= 0 && d.Nx == 1024)
        branch_tables(d.Nx, a.data(), b.data(), cd(1, 0), cd(1, 0), Hx, out + d.off_tabX, p->wx);
    if (d.off_tabX >= 0 && d.Nx == 2048)
        branch_tables4(a.data(), b.data(), cd(1, 0), cd(1, 0), Hx, out + d.off_tabX, p->wx);
}

// Per-device one-time set-up: cudaFuncSetAttribute applies to the device that is current, so a
// process that makes plans on several GPUs needs it once on each.
std::mutex g_init_mutex;
int g_sms[64] = {};

int device_init(int device, int *sms) {
    std::lock_guard<std::mutex> lock(g_init_mutex);
    if (device < 0 || device >= 64) return SFD_EUNSUPPORTED;
    if (g_sms[device] == 0) {
        int n = 0;
        SFD_CUDA(sfd_kernels_init(device, &n));
        g_sms[device] = n;
    }
    *sms = g_sms[device];
    return SFD_OK;
}

}  // namespace

// ---- real-time stream state --------------------------------------------------------------------
struct sfd_stream_state {
    cudaStream_t s_in = nullptr, s_comp = nullptr, s_out = nullptr;
    void *d_holo[2] = {nullptr, nullptr};
    unsigned char *d_out[2] = {nullptr, nullptr};
    cudaEvent_t e_in[2] = {nullptr, nullptr}, e_comp[2] = {nullptr, nullptr},
                e_out[2] = {nullptr, nullptr}, e_t0 = nullptr, e_t1 = nullptr;
};

// ---- staging of live view updates ---------------------------------------------------------------
// sfd_plan_update_view*_async builds a view's tables into one of SLOTS page-locked staging blocks
// and enqueues ONE host-to-device copy on the caller's stream; the event recorded behind the copy
// says when the block may be rewritten.
struct sfd_update_ring {
    static constexpr int SLOTS = 4;
    float2 *slot[SLOTS] = {nullptr, nullptr, nullptr, nullptr};
    cudaEvent_t done[SLOTS] = {nullptr, nullptr, nullptr, nullptr};
    bool used[SLOTS] = {false, false, false, false};
    int next = 0;
};

namespace {

void stream_state_free(sfd_stream_state *s) {
    if (!s) return;
    for (int b = 0; b < 2; ++b) {
        if (s->d_holo[b]) cudaFree(s->d_holo[b]);
        if (s->d_out[b]) cudaFree(s->d_out[b]);
        if (s->e_in[b]) cudaEventDestroy(s->e_in[b]);
        if (s->e_comp[b]) cudaEventDestroy(s->e_comp[b]);
        if (s->e_out[b]) cudaEventDestroy(s->e_out[b]);
    }
    if (s->e_t0) cudaEventDestroy(s->e_t0);
    if (s->e_t1) cudaEventDestroy(s->e_t1);
    if (s->s_in) cudaStreamDestroy(s->s_in);
    if (s->s_comp) cudaStreamDestroy(s->s_comp);
    if (s->s_out) cudaStreamDestroy(s->s_out);
    delete s;
}

size_t window_elems(const sfd_plan *p) { return (size_t)p->d.Nx * p->d.Ny; }

// the plan's device is current (SFD_ON_DEVICE in the caller)
int stream_state_make(sfd_plan *p) {
    if (p->ss) return SFD_OK;
    sfd_stream_state *s = new (std::nothrow) sfd_stream_state;
    if (!s) return SFD_ENOMEM;
    p->ss = s;  // freed by sfd_plan_destroy even when half built
    const size_t nn = window_elems(p);
    const size_t in_bytes = nn * (p->d.in_dtype == SFD_U8 ? 1 : 4);
    SFD_CUDA(cudaStreamCreateWithFlags(&s->s_in, cudaStreamNonBlocking));
    SFD_CUDA(cudaStreamCreateWithFlags(&s->s_comp, cudaStreamNonBlocking));
    SFD_CUDA(cudaStreamCreateWithFlags(&s->s_out, cudaStreamNonBlocking));
    for (int b = 0; b < 2; ++b) {
        SFD_CUDA(cudaMalloc(&s->d_holo[b], in_bytes));
        SFD_CUDA(cudaMalloc((void **)&s->d_out[b], nn * p->d.V));
        SFD_CUDA(cudaEventCreateWithFlags(&s->e_in[b], cudaEventDisableTiming));
        SFD_CUDA(cudaEventCreateWithFlags(&s->e_comp[b], cudaEventDisableTiming));
        SFD_CUDA(cudaEventCreateWithFlags(&s->e_out[b], cudaEventDisableTiming));
        p->device_bytes += (long long)(in_bytes + nn * p->d.V);
    }
    SFD_CUDA(cudaEventCreate(&s->e_t0));
    SFD_CUDA(cudaEventCreate(&s->e_t1));
    return SFD_OK;
}

void update_ring_free(sfd_update_ring *r) {
    if (!r) return;
    for (int i = 0; i < sfd_update_ring::SLOTS; ++i) {
        if (r->slot[i]) cudaFreeHost(r->slot[i]);
        if (r->done[i]) cudaEventDestroy(r->done[i]);
    }
    delete r;
}

int update_ring_make(sfd_plan *p) {
    if (p->ur) return SFD_OK;
    sfd_update_ring *r = new (std::nothrow) sfd_update_ring;
    if (!r) return SFD_ENOMEM;
    p->ur = r;
    for (int i = 0; i < sfd_update_ring::SLOTS; ++i) {
        SFD_CUDA(cudaMallocHost((void **)&r->slot[i], (size_t)p->d.vstride * sizeof(float2)));
        SFD_CUDA(cudaEventCreateWithFlags(&r->done[i], cudaEventDisableTiming));
    }
    return SFD_OK;
}

// Rebuild the tables of view v from the plan's current parameters and copy them to the device:
// one cudaMemcpyAsync from a pinned staging slot on `st`, ordered like any other work of that stream
// (after the executes enqueued before it, before those enqueued after it).  wait = true blocks
// until the copy has landed.
int upload_view(sfd_plan *p, int v, cudaStream_t st, bool wait) {
    int rc = update_ring_make(p);
    if (rc != SFD_OK) return rc;
    sfd_update_ring *r = p->ur;
    const int i = r->next;
    r->next = (i + 1) % sfd_update_ring::SLOTS;
    if (r->used[i]) SFD_CUDA(cudaEventSynchronize(r->done[i]));  // the slot's last copy has read it
    const auto t0 = std::chrono::steady_clock::now();
    build_view_f32(p, v, r->slot[i]);
    p->last_update_host_ms =
        std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
    SFD_CUDA(cudaMemcpyAsync(p->d.tabs + (size_t)v * p->d.vstride, r->slot[i],
                             (size_t)p->d.vstride * sizeof(float2), cudaMemcpyHostToDevice, st));
    SFD_CUDA(cudaEventRecord(r->done[i], st));
    r->used[i] = true;
    if (wait) SFD_CUDA(cudaEventSynchronize(r->done[i]));
    return SFD_OK;
}

int set_view(sfd_plan *p, int view, double p1x, double p1y, double p2x, double p2y, double z,
             double O0x, double O0y, double O1x, double O1y) {
    if (!p || view < 0 || view >= p->d.V) return SFD_EINVAL;
    if (check_view(p->lambda, p1x, p2x, z, O1x, O0x) != SFD_OK) return SFD_EINVAL;
    if (check_view(p->lambda, p1y, p2y, z, O1y, O0y) != SFD_OK) return SFD_EINVAL;
    p->p1[view] = p1x;
    p->p1y[view] = p1y;
    p->p2[view] = p2x;
    p->p2y[view] = p2y;
    p->z[view] = z;
    p->Ox[view] = O1x;
    p->Oy[view] = O1y;
    p->O0x[view] = O0x;
    p->O0y[view] = O0y;
    return SFD_OK;
}

const void *window_ptr(const sfd_plan *p, const void *frame) {
    return (const char *)frame + p->d.in_offset * (p->d.in_dtype == SFD_U8 ? 1 : 4);
}

// the frame loop of sfd_stream_run; any failure is reported through the single exit of the caller
int stream_frames(sfd_plan *p, sfd_stream_state *s, const void *holograms_pinned, int n_frames,
                  unsigned char *out_pinned) {
    const size_t nn = window_elems(p);
    const size_t in_bytes = nn * (p->d.in_dtype == SFD_U8 ? 1 : 4);
    const size_t out_bytes = nn * p->d.V;
    // the device copy of a frame is the dense window: the window set on the plan applies to
    // sfd_execute*, the stream reads dense [Ny][Nx] frames from the host
    struct Dense {
        sfd_plan *p;
        long long stride, offset;
        explicit Dense(sfd_plan *q) : p(q), stride(q->d.in_stride), offset(q->d.in_offset) {
            p->d.in_stride = p->d.Nx;
            p->d.in_offset = 0;
        }
        ~Dense() {
            p->d.in_stride = stride;
            p->d.in_offset = offset;
        }
    } dense(p);
    SFD_CUDA(cudaEventRecord(s->e_t0, s->s_in));
    for (int f = 0; f < n_frames; ++f) {
        const int b = f & 1;
        // (i) H2D of frame f into input buffer b, once the compute of frame f-2 has read it
        if (f >= 2) SFD_CUDA(cudaStreamWaitEvent(s->s_in, s->e_comp[b], 0));
        SFD_CUDA(cudaMemcpyAsync(s->d_holo[b], (const char *)holograms_pinned + (size_t)f * in_bytes,
                                 in_bytes, cudaMemcpyHostToDevice, s->s_in));
        SFD_CUDA(cudaEventRecord(s->e_in[b], s->s_in));
        // (ii)-(x) + quantise, once the D2H of frame f-2 has drained output buffer b
        SFD_CUDA(cudaStreamWaitEvent(s->s_comp, s->e_in[b], 0));
        if (f >= 2) SFD_CUDA(cudaStreamWaitEvent(s->s_comp, s->e_out[b], 0));
        SFD_CUDA(sfd_launch(p, s->d_holo[b], nullptr, nullptr, s->d_out[b], s->s_comp));
        SFD_CUDA(cudaEventRecord(s->e_comp[b], s->s_comp));
        // (xi) D2H of the 8-bit views
        SFD_CUDA(cudaStreamWaitEvent(s->s_out, s->e_comp[b], 0));
        SFD_CUDA(cudaMemcpyAsync(out_pinned + (size_t)f * out_bytes, s->d_out[b], out_bytes,
                                 cudaMemcpyDeviceToHost, s->s_out));
        SFD_CUDA(cudaEventRecord(s->e_out[b], s->s_out));
    }
    SFD_CUDA(cudaEventRecord(s->e_t1, s->s_out));
    return SFD_OK;
}

}  // namespace

// ---- C ABI -------------------------------------------------------------------------------------
extern "C" {

int sfd_host_tables(int N, double lambda, double p1, double p2, double z, double off, double *pre,
                    double *post, double *H) {
    return sfd_host_tables_general(N, lambda, p1, p2, z, 0.0, off, pre, post, H);
}

int sfd_host_tables_general(int N, double lambda, double p1, double p2, double z, double off0,
                            double off, double *pre, double *post, double *H) {
    if (!pre || !post || !H || log2_exact(N) < 0 || N < 2) return SFD_EINVAL;
    if (check_view(lambda, p1, p2, z, off, off0) != SFD_OK) return SFD_EINVAL;
    std::vector<cd> a(N), b(N), h(2 * (size_t)N);
    axis_tables(N, lambda, p1, p2, z, off, a.data(), b.data(), off0);
    kernel_spectrum(N, lambda, p1, p2, z, h.data(), fft_twiddles(2 * (size_t)N));
    std::memcpy(pre, a.data(), sizeof(cd) * N);
    std::memcpy(post, b.data(), sizeof(cd) * N);
    std::memcpy(H, h.data(), sizeof(cd) * 2 * N);
    return SFD_OK;
}

int sfd_host_dft32(const float *in, float *out, int lane, int twiddled) {
    if (!in || !out || lane < 0 || lane > 31) return SFD_EINVAL;
    sfd_host_dft32_impl(in, out, lane, twiddled);
    return SFD_OK;
}

int sfd_plan_create(sfd_plan **out, int N, int n_views, double lambda, const double *p1,
                    const double *p2, const double *z, const double *Ox, const double *Oy,
                    int in_dtype) {
    if (!out) return SFD_EINVAL;
    *out = nullptr;
    if (!p1 || !p2 || !z || !Ox || !Oy || n_views < 1) return SFD_EINVAL;
    const std::vector<double> zero(n_views, 0.0);
    return sfd_plan_create_rect(out, N, N, n_views, lambda, p1, p1, p2, p2, z, zero.data(),
                                zero.data(), Ox, Oy, in_dtype);
}

int sfd_plan_create_general(sfd_plan **out, int N, int n_views, double lambda, const double *p1x,
                            const double *p1y, const double *p2x, const double *p2y,
                            const double *z, const double *O0x, const double *O0y,
                            const double *O1x, const double *O1y, int in_dtype) {
    return sfd_plan_create_rect(out, N, N, n_views, lambda, p1x, p1y, p2x, p2y, z, O0x, O0y, O1x,
                                O1y, in_dtype);
}

int sfd_plan_create_rect(sfd_plan **out, int Nx, int Ny, int n_views, double lambda,
                         const double *p1x, const double *p1y, const double *p2x,
                         const double *p2y, const double *z, const double *O0x,
                         const double *O0y, const double *O1x, const double *O1y, int in_dtype) {
    if (!out) return SFD_EINVAL;
    *out = nullptr;
    if (!p1x || !p1y || !p2x || !p2y || !z || !O0x || !O0y || !O1x || !O1y) return SFD_EINVAL;
    if (Nx < 1 || Ny < 1 || n_views < 1) return SFD_EINVAL;
    if (in_dtype != SFD_U8 && in_dtype != SFD_F32) return SFD_EINVAL;
    for (int v = 0; v < n_views; ++v) {
        if (check_view(lambda, p1x[v], p2x[v], z[v], O1x[v], O0x[v]) != SFD_OK) return SFD_EINVAL;
        if (check_view(lambda, p1y[v], p2y[v], z[v], O1y[v], O0y[v]) != SFD_OK) return SFD_EINVAL;
    }
    // a size this build has no kernels for is a valid request that is not implemented
    const int lx = log2_exact(Nx), ly = log2_exact(Ny);
    if (lx < 6 || lx > 11 || ly < 6 || ly > 11) return SFD_EUNSUPPORTED;
    int device = 0;
    SFD_CUDA(cudaGetDevice(&device));
    int sms = 0;
    int rc = device_init(device, &sms);
    if (rc != SFD_OK) return rc;

    sfd_plan *p = new (std::nothrow) sfd_plan;
    if (!p) return SFD_ENOMEM;
    sfd_dev &d = p->d;
    p->device = device;
    d.sms = sms;
    d.Nx = Nx;
    d.Ny = Ny;
    d.Mx = 2 * Nx;
    d.My = 2 * Ny;
    d.log2Mx = lx + 1;
    d.log2My = ly + 1;
    d.V = n_views;
    d.in_dtype = in_dtype;
    d.in_stride = Nx;
    d.in_offset = 0;
    p->lambda = lambda;
    p->p1.assign(p1x, p1x + n_views);
    p->p2.assign(p2x, p2x + n_views);
    p->z.assign(z, z + n_views);
    p->Ox.assign(O1x, O1x + n_views);
    p->Oy.assign(O1y, O1y + n_views);
    p->p1y.assign(p1y, p1y + n_views);
    p->p2y.assign(p2y, p2y + n_views);
    p->O0x.assign(O0x, O0x + n_views);
    p->O0y.assign(O0y, O0y + n_views);
    p->wy = fft_twiddles((size_t)d.My);
    p->wx = fft_twiddles((size_t)d.Mx);

    auto fail = [&](int code) {
        sfd_plan_destroy(p);
        return code;
    };
    // table layout of one view (complex64 elements), the stride rounded up to 128 bytes
    int o = 0;
    d.off_pre_y = o;   o += Ny;
    d.off_post_y = o;  o += Ny;
    d.off_pre_x = o;   o += Nx;
    d.off_post_x = o;  o += Nx;
    d.off_Hy = o;      o += d.My;
    d.off_Hx = o;      o += d.Mx;
    if (fast_elems(Ny)) { d.off_tabY = o; o += (int)fast_elems(Ny); }
    if (fast_elems(Nx)) { d.off_tabX = o; o += (int)fast_elems(Nx); }
    d.vstride = (o + 15) & ~15;
    const size_t V = n_views, nn = (size_t)Nx * Ny;
    const size_t n_tab = V * (size_t)d.vstride + d.My + d.Mx + 32 * 32;  // + FFT twiddles + w_twl
    cudaError_t e;
    if ((e = cudaMalloc(&p->table_alloc, n_tab * sizeof(float2))) != cudaSuccess)
        return fail(e == cudaErrorMemoryAllocation ? SFD_ENOMEM : cuda_fail(e, "cudaMalloc tables"));
    d.tabs = (float2 *)p->table_alloc;
    d.tw_y = d.tabs + V * (size_t)d.vstride;
    d.tw_x = d.tw_y + d.My;
    d.w_twl = d.tw_x + d.Mx;
    if ((e = cudaMalloc((void **)&d.B, V * nn * sizeof(float2))) != cudaSuccess)
        return fail(e == cudaErrorMemoryAllocation ? SFD_ENOMEM : cuda_fail(e, "cudaMalloc B"));
    if ((e = cudaMalloc((void **)&d.inten_ws, V * nn * sizeof(float))) != cudaSuccess)
        return fail(e == cudaErrorMemoryAllocation ? SFD_ENOMEM : cuda_fail(e, "cudaMalloc I"));
    if ((e = cudaMalloc((void **)&d.vmax, V * sizeof(unsigned int))) != cudaSuccess)
        return fail(cuda_fail(e, "cudaMalloc vmax"));
    p->device_bytes = (long long)(n_tab * sizeof(float2) + V * nn * 12 + V * 4);

    {   // plan constants: FFT twiddles exp(-2 pi i x / M) of both axes (generic kernels) and the
        // stage-B twiddles of the warp FFT (sfd_dft32.cuh): [j][lane], j = n/2 - 1 + k,
        // T_n[k] = exp(-2 pi i (lane + 32 k) / (32 n)), n = 2, 4, .., 32, k < n/2
        std::vector<float2> c((size_t)d.My + d.Mx + 32 * 32, make_float2(0.f, 0.f));
        for (int x = 0; x < d.My; ++x) {
            const cd w = cis_cycles(-(ld)x / (ld)d.My);
            c[x] = make_float2((float)w.real(), (float)w.imag());
        }
        for (int x = 0; x < d.Mx; ++x) {
            const cd w = cis_cycles(-(ld)x / (ld)d.Mx);
            c[(size_t)d.My + x] = make_float2((float)w.real(), (float)w.imag());
        }
        float2 *twl = c.data() + d.My + d.Mx;
        for (int n = 2; n <= 32; n *= 2)
            for (int k = 0; k < n / 2; ++k)
                for (int lane = 0; lane < 32; ++lane) {
                    const cd w = cis_cycles(-(ld)(lane + 32 * k) / (ld)(32 * n));
                    twl[(n / 2 - 1 + k) * 32 + lane] = make_float2((float)w.real(), (float)w.imag());
                }
        if ((e = cudaMemcpy(d.tw_y, c.data(), c.size() * sizeof(float2), cudaMemcpyHostToDevice)) !=
            cudaSuccess)
            return fail(cuda_fail(e, "cudaMemcpy twiddles"));
    }
    for (int v = 0; v < n_views; ++v)
        if ((rc = upload_view(p, v, cudaStreamLegacy, false)) != SFD_OK) return fail(rc);
    // every table has landed before the plan is handed out: the kernels read them in their prologue,
    // on whatever stream (possibly a non-blocking one) the caller launches
    if ((e = cudaDeviceSynchronize()) != cudaSuccess) return fail(cuda_fail(e, "cudaDeviceSynchronize"));
    if ((e = sfd_make_tensormaps(p)) != cudaSuccess) return fail(cuda_fail(e, "cuTensorMapEncodeTiled"));
    for (int i = 0; i < 4; ++i)
        if ((e = cudaEventCreate(&p->ev[i])) != cudaSuccess) return fail(cuda_fail(e, "cudaEventCreate"));
    *out = p;
    return SFD_OK;
}

int sfd_plan_set_input_window(sfd_plan *p, long long row_stride, int row0, int col0) {
    if (!p || row0 < 0 || col0 < 0 || row_stride < 0) return SFD_EINVAL;
    if (row_stride == 0) row_stride = p->d.Nx;
    if (row_stride < (long long)col0 + p->d.Nx) return SFD_EINVAL;
    p->d.in_stride = row_stride;
    p->d.in_offset = (long long)row0 * row_stride + col0;
    return SFD_OK;
}

int sfd_plan_update_view(sfd_plan *p, int view, double p1, double p2, double z, double Ox,
                         double Oy) {
    const int rc = set_view(p, view, p1, p1, p2, p2, z, 0.0, 0.0, Ox, Oy);
    if (rc != SFD_OK) return rc;
    SFD_ON_DEVICE(p);
    return upload_view(p, view, cudaStreamLegacy, true);
}

int sfd_plan_update_view_general(sfd_plan *p, int view, double p1x, double p1y, double p2x,
                                 double p2y, double z, double O0x, double O0y, double O1x,
                                 double O1y) {
    const int rc = set_view(p, view, p1x, p1y, p2x, p2y, z, O0x, O0y, O1x, O1y);
    if (rc != SFD_OK) return rc;
    SFD_ON_DEVICE(p);
    return upload_view(p, view, cudaStreamLegacy, true);
}

int sfd_plan_update_view_async(sfd_plan *p, int view, double p1, double p2, double z, double Ox,
                               double Oy, void *stream) {
    const int rc = set_view(p, view, p1, p1, p2, p2, z, 0.0, 0.0, Ox, Oy);
    if (rc != SFD_OK) return rc;
    SFD_ON_DEVICE(p);
    return upload_view(p, view, (cudaStream_t)stream, false);
}

int sfd_plan_update_view_general_async(sfd_plan *p, int view, double p1x, double p1y, double p2x,
                                       double p2y, double z, double O0x, double O0y, double O1x,
                                       double O1y, void *stream) {
    const int rc = set_view(p, view, p1x, p1y, p2x, p2y, z, O0x, O0y, O1x, O1y);
    if (rc != SFD_OK) return rc;
    SFD_ON_DEVICE(p);
    return upload_view(p, view, (cudaStream_t)stream, false);
}

double sfd_plan_last_update_host_ms(const sfd_plan *p) { return p ? p->last_update_host_ms : -1.0; }

int sfd_execute(sfd_plan *p, const void *hologram_dev, void *field_dev, float *intensity_dev,
                void *stream) {
    if (!p || !hologram_dev || (!field_dev && !intensity_dev)) return SFD_EINVAL;
    SFD_ON_DEVICE(p);
    SFD_CUDA(sfd_launch(p, window_ptr(p, hologram_dev), (float2 *)field_dev, intensity_dev, nullptr,
                        (cudaStream_t)stream));
    return SFD_OK;
}

int sfd_execute_focus(sfd_plan *p, const void *hologram_dev, double *moments_dev,
                      float *intensity_dev, void *stream) {
    if (!p || !hologram_dev || !moments_dev) return SFD_EINVAL;
    SFD_ON_DEVICE(p);
    SFD_CUDA(sfd_launch(p, window_ptr(p, hologram_dev), nullptr, intensity_dev, nullptr,
                        (cudaStream_t)stream, moments_dev));
    return SFD_OK;
}

int sfd_execute_u8(sfd_plan *p, const void *hologram_dev, unsigned char *intensity_u8_dev,
                   void *stream) {
    if (!p || !hologram_dev || !intensity_u8_dev) return SFD_EINVAL;
    SFD_ON_DEVICE(p);
    SFD_CUDA(sfd_launch(p, window_ptr(p, hologram_dev), nullptr, nullptr, intensity_u8_dev,
                        (cudaStream_t)stream));
    return SFD_OK;
}

int sfd_stream_run(sfd_plan *p, const void *holograms_pinned, int n_frames,
                   unsigned char *out_pinned, double *seconds) {
    if (!p || !holograms_pinned || !out_pinned || n_frames < 0) return SFD_EINVAL;
    if (seconds) *seconds = 0.0;
    if (n_frames == 0) return SFD_OK;
    SFD_ON_DEVICE(p);
    int rc = stream_state_make(p);
    if (rc != SFD_OK) return rc;
    sfd_stream_state *s = p->ss;
    const bool timing = p->timing;
    p->timing = false;  // the per-kernel events belong to sfd_execute*
    rc = stream_frames(p, s, holograms_pinned, n_frames, out_pinned);
    p->timing = timing;
    // single exit: whatever was enqueued has drained before the caller may touch (or free) its
    // pinned buffers, also after a failure half way through the loop
    const cudaError_t e0 = cudaStreamSynchronize(s->s_in), e1 = cudaStreamSynchronize(s->s_comp),
                      e2 = cudaStreamSynchronize(s->s_out);
    if (rc != SFD_OK) return rc;
    SFD_CUDA(e0);
    SFD_CUDA(e1);
    SFD_CUDA(e2);
    float ms = 0.f;
    SFD_CUDA(cudaEventElapsedTime(&ms, s->e_t0, s->e_t1));
    if (seconds) *seconds = (double)ms * 1e-3;
    return SFD_OK;
}

int sfd_plan_destroy(sfd_plan *p) {
    if (!p) return SFD_OK;
    DeviceGuard guard(p->device);
    stream_state_free(p->ss);
    update_ring_free(p->ur);
    if (p->table_alloc) cudaFree(p->table_alloc);
    if (p->d.B) cudaFree(p->d.B);
    if (p->d.inten_ws) cudaFree(p->d.inten_ws);
    if (p->d.vmax) cudaFree(p->d.vmax);
    for (int i = 0; i < 4; ++i)
        if (p->ev[i]) cudaEventDestroy(p->ev[i]);
    delete p;
    return SFD_OK;
}

int sfd_plan_get_n(const sfd_plan *p) { return p ? p->d.Nx : SFD_EINVAL; }
int sfd_plan_get_nx(const sfd_plan *p) { return p ? p->d.Nx : SFD_EINVAL; }
int sfd_plan_get_ny(const sfd_plan *p) { return p ? p->d.Ny : SFD_EINVAL; }
int sfd_plan_get_views(const sfd_plan *p) { return p ? p->d.V : SFD_EINVAL; }
int sfd_plan_get_m(const sfd_plan *p) { return p ? p->d.Mx : SFD_EINVAL; }
int sfd_plan_get_device(const sfd_plan *p) { return p ? p->device : SFD_EINVAL; }
long long sfd_plan_device_bytes(const sfd_plan *p) { return p ? p->device_bytes : SFD_EINVAL; }

int sfd_plan_select_kernels(sfd_plan *p, int which) {
    if (!p || (which != SFD_KERNELS_AUTO && which != SFD_KERNELS_GENERIC)) return SFD_EINVAL;
    p->kernels = which;
    return SFD_OK;
}

int sfd_plan_uses_warp_kernels(const sfd_plan *p) {
    if (!p) return SFD_EINVAL;
    return (sfd_uses_warp_y(p, nullptr) ? 1 : 0) | (sfd_uses_warp_x(p) ? 2 : 0);
}

int sfd_plan_set_timing(sfd_plan *p, int enable) {
    if (!p) return SFD_EINVAL;
    p->timing = enable != 0;
    if (!p->timing) p->ev_valid = p->ev_quant = false;
    return SFD_OK;
}

int sfd_plan_last_kernel_ms(sfd_plan *p, float ms[3]) {
    if (!p || !ms) return SFD_EINVAL;
    ms[0] = ms[1] = ms[2] = 0.f;
    if (!p->ev_valid) return SFD_EINVAL;
    SFD_ON_DEVICE(p);
    SFD_CUDA(cudaEventSynchronize(p->ev[p->ev_quant ? 3 : 2]));
    SFD_CUDA(cudaEventElapsedTime(&ms[0], p->ev[0], p->ev[1]));
    SFD_CUDA(cudaEventElapsedTime(&ms[1], p->ev[1], p->ev[2]));
    if (p->ev_quant) SFD_CUDA(cudaEventElapsedTime(&ms[2], p->ev[2], p->ev[3]));
    return SFD_OK;
}

int sfd_measure_pipes(double out[4]) {
    if (!out) return SFD_EINVAL;
    SFD_CUDA(sfd_measure_pipes_impl(out));
    return SFD_OK;
}

long long sfd_launch_count(void) { return sfd_launch_count_impl(); }

const char *sfd_error_string(int code) {
    switch (code) {
        case SFD_OK: return "success";
        case SFD_EINVAL: return "invalid argument";
        case SFD_ENOMEM: return "out of memory";
        case SFD_ECUDA: return "CUDA runtime error (see sfd_last_cuda_error)";
        case SFD_EUNSUPPORTED: return "unsupported request";
    }
    return "unknown error code";
}

const char *sfd_last_cuda_error(void) { return g_cuda_err; }

const char *sfd_version(void) { return "sfd 0.2 sm_100a"; }

}  // extern "C"
