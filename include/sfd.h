/* sfd.h — C ABI of libsfd: Shifted-Fresnel diffraction on one NVIDIA B200 (sm_100a).
 *
 * What the library computes (arxiv/paper_1001_4309, §2.1, Eq.(1)-(5), L50-71; step list
 * (i)-(xi), L85-95): from one N x N in-line hologram u0 sampled at pitch p1, for each of n_views
 * views with its own depth z, reconstruction pitch p2 and off-axis shift (Ox, Oy), the complex
 * field
 *
 *     u1[n1][m1] = c0 * sum_{n0,m0} u0[n0][m0] * exp(i pi [(x1-x0)^2 + (y1-y0)^2] / (lambda z)),
 *     x0 = (m0 - N/2) p1,  y0 = (n0 - N/2) p1,  x1 = (m1 - N/2) p2 + Ox,  y1 = (n1 - N/2) p2 + Oy,
 *     c0 = p1^2 exp(i 2 pi z / lambda) / (i lambda z),
 *
 * and its intensity I = |u1|^2 (Eq. 5).  This is Eq.(1) with all of C1 (Eq. 2) kept and the area
 * element p1^2 included (readings 1, 2, 9, 10).  It is evaluated as the paper evaluates
 * it — pre-chirp (Eq. 3), zero-padded 2N-point FFT, multiply by the spectrum of the chirp kernel h
 * (Eq. 4), inverse FFT, crop, post-chirp (Eq. 2) — but, h being separable, as two fused passes of
 * 1-D length-2N transforms (first along y, then along x); see DESIGN.md §5.
 *
 * Conventions
 *   - Arrays are row-major [n][m]: n <-> y <-> row, m <-> x <-> fastest index.
 *   - All lengths are SI metres.  All per-view parameter arrays are HOST arrays of n_views doubles
 *     and are copied at plan creation (the caller may free them afterwards).
 *   - Pointers named *_dev are DEVICE pointers on the plan's device (the device current when the
 *     plan was created); *_pinned are page-locked HOST pointers.  The caller owns them.
 *   - The plan owns its device tables, the cached chirp-kernel spectra and its workspace.
 *   - Every call returns an int: 0 = SFD_OK, negative = error.  No exception crosses the ABI.
 *   - One sfd_execute* may be in flight per plan (shared workspace); distinct plans are
 *     independent.  Calls on one plan must be issued from one host thread at a time.
 */
#ifndef SFD_H
#define SFD_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sfd_plan sfd_plan; /* opaque */

#if defined(__GNUC__)
#define SFD_API __attribute__((visibility("default")))
#else
#define SFD_API
#endif

/* error codes */
#define SFD_OK 0
#define SFD_EINVAL (-1)       /* bad argument (NULL, size, non-finite parameter, z == 0, ...) */
#define SFD_ENOMEM (-2)       /* host or device allocation failed */
#define SFD_ECUDA (-3)        /* a CUDA runtime call failed; see sfd_last_cuda_error() */
#define SFD_EUNSUPPORTED (-4) /* valid request that this build does not implement (a grid side that
                                 is not a power of two in 64..2048; more than 64 devices) */

/* hologram sample types (argument in_dtype) */
#define SFD_U8 0  /* unsigned 8-bit CCD samples; the method sees value/255 (reading 12) */
#define SFD_F32 1 /* float32 samples used as they are */
#define SFD_C64 2 /* complex64 samples (re, im interleaved); angular-spectrum plans only */

/* Create a plan for one hologram size and a fixed set of views (S = p1 p2/(lambda z);
 * Eq.(2)-(4)).  Builds, in float64 on the host, the 1-D chirp tables of Eq.(2)-(3) and the spectrum
 * of the 1-D chirp kernel of Eq.(4) for every view (steps (v)-(vi) L89-90, done once here instead
 * of every frame), uploads them as complex64 and allocates the workspace
 * (n_views * N * N complex64 + n_views * N * N float32).
 *   out      receives the plan; *out = NULL on failure.
 *   N        hologram / output side >= 1; this build has kernels for powers of two in 64..2048 and
 *            returns SFD_EUNSUPPORTED for every other size.
 *   n_views  >= 1.
 *   lambda   wavelength > 0.
 *   p1,p2,z,Ox,Oy  host arrays [n_views]: hologram pitch (> 0), reconstruction pitch (> 0), depth
 *            (finite, != 0; negative = conjugate reconstruction), shifts of the output window.
 *   in_dtype SFD_U8 or SFD_F32.
 * Errors: SFD_EINVAL, SFD_EUNSUPPORTED, SFD_ENOMEM, SFD_ECUDA.
 * The device current at the call becomes the plan's device; later calls on the plan may be made with
 * any device current (the library switches to the plan's device and back). */
SFD_API int sfd_plan_create(sfd_plan **out, int N, int n_views, double lambda, const double *p1,
                    const double *p2, const double *z, const double *Ox, const double *Oy,
                    int in_dtype);

/* Reconstruct all views of one hologram (steps (ii)-(x), L86-94).  Asynchronous on `stream`
 * (a cudaStream_t passed as void*; NULL = the legacy default stream); no host synchronisation.
 *   hologram_dev   [N][N] samples of the plan's in_dtype.
 *   field_dev      [n_views][N][N] complex64 (re, im interleaved), or NULL to skip the field.
 *   intensity_dev  [n_views][N][N] float32, or NULL to skip the intensity.
 * At least one output must be non-NULL.  Errors: SFD_EINVAL, SFD_ECUDA.
 * The call only enqueues kernels on `stream` (no allocation, no host synchronisation), so it may be
 * captured in a CUDA graph (with per-kernel timing off); the kernels of one call and of consecutive
 * calls are chained by programmatic dependent launch. */
SFD_API int sfd_execute(sfd_plan *plan, const void *hologram_dev, void *field_dev, float *intensity_dev,
                void *stream);

/* Real-time variant (step (xi) L95, reading 15): intensity returned as 8-bit images, per view
 * I8 = round_half_even(255 * I / max(I)) (an all-zero view gives zeros).
 *   intensity_u8_dev  [n_views][N][N] unsigned char.  Asynchronous on `stream`. */
SFD_API int sfd_execute_u8(sfd_plan *plan, const void *hologram_dev, unsigned char *intensity_u8_dev,
                   void *stream);

/* Allocation-free variant of step (xi) (L95, reading 15) for callers that cannot call cudaMalloc (code
 * under CUDA graph capture, tight serving loops, harnesses that forbid it): no plan, no workspace.
 *   intensity_dev     [n_views][pixels_per_view] float32 on the device, values >= 0 (e.g. the intensity
 *                     output of sfd_execute), 16-byte aligned; pixels_per_view a multiple of 4
 *   intensity_u8_dev  [n_views][pixels_per_view] unsigned char on the device, 4-byte aligned; per view
 *                     I8 = round_half_even(255 * I / max(I)) (an all-zero view gives zeros) - the same
 *                     arithmetic and the same quantisation kernel as sfd_execute_u8
 * The per-view maxima are kept in a static device array inside the library (SFD_STATIC_MAX_VIEWS
 * 32-bit words = 4 KiB, present on every GPU that loads the library until the process exits); the
 * call enqueues a clear of the words it uses and two kernels on `stream` and returns.  It calls no
 * cudaMalloc / cudaFree or any allocating routine (the first call on a device looks up the array's
 * address).  ALL calls share that array: calls on one stream are ordered and safe; calls that may
 * overlap on the GPU (different streams without an event between them) race on it and must be
 * serialised by the caller.
 * Errors: SFD_EINVAL (NULL, sizes, alignment), SFD_EUNSUPPORTED if n_views > SFD_STATIC_MAX_VIEWS
 * (split the call), SFD_ECUDA; sfd_static_last_error() gives the text of this thread's last failure. */
#define SFD_STATIC_MAX_VIEWS 1024
SFD_API int sfd_quantise_u8_static(const float *intensity_dev, int n_views, long long pixels_per_view,
                                   unsigned char *intensity_u8_dev, void *stream);
SFD_API int sfd_static_max_views(void);
SFD_API const char *sfd_static_last_error(void);

/* Depth stacks / focus sweep ("different depths along the depth direction",
 * PAPER.md L33 and Fig. 1): a plan whose views differ only in z is a depth stack of one hologram.
 * This call runs the same two passes and, fused into the last one, reduces every view to its first
 * two intensity moments
 *     moments_dev[2 v] = sum over the N x N window of I,   moments_dev[2 v + 1] = sum of I^2
 * (device array of 2 n_views doubles; per-thread partial sums in float32, accumulation across warps
 * in float64 with atomics: the last bits depend on the order of arrival).  The paper defines no
 * focus measure (reading 21); any variance-type measure follows from the two moments,
 * e.g. the normalised variance N^2 sum I^2 / (sum I)^2 - 1.  intensity_dev ([n_views][N][N] float32)
 * may be NULL: nothing but the moments is then written.  Asynchronous on `stream`. */
SFD_API int sfd_execute_focus(sfd_plan *plan, const void *hologram_dev, double *moments_dev,
                              float *intensity_dev, void *stream);

/* Real-time stream (steps (i)-(xi) repeated, L83-97): reconstruct n_frames holograms that sit in
 * page-locked host memory, double-buffering the H2D copies against compute and the D2H copies of
 * the 8-bit results, on three internal streams.  Blocking: returns when out_pinned is complete.
 *   holograms_pinned  [n_frames][N][N] samples of the plan's in_dtype (pinned host memory).
 *   out_pinned        [n_frames][n_views][N][N] unsigned char (pinned host memory).
 *   seconds           if non-NULL, receives the device-measured time (CUDA events) from the start
 *                     of the first H2D copy to the end of the last D2H copy. */
SFD_API int sfd_stream_run(sfd_plan *plan, const void *holograms_pinned, int n_frames,
                   unsigned char *out_pinned, double *seconds);

/* Replace the parameters of one view (0 <= view < n_views) and rebuild its tables and cached
 * spectrum (the paper's user steers z, p2, Ox, Oy live: L33, L73, L123).  Blocking form: the new
 * tables are on the device when the call returns (ordered on the legacy default stream); do not call
 * it while an execute of this plan is in flight on a non-blocking stream. */
SFD_API int sfd_plan_update_view(sfd_plan *plan, int view, double p1, double p2, double z, double Ox,
                         double Oy);

/* Live steering without a host-device synchronisation: the tables of the view are built on the host
 * (float64, about a millisecond at N = 1024: sfd_plan_last_update_host_ms) into a page-locked staging
 * block and ONE asynchronous copy is enqueued on `stream`.  Stream order does the rest: executes
 * enqueued on that stream before the call still see the old view, executes enqueued after it the new
 * one, and the call is legal while earlier executes are in flight.  Use the stream the executes of
 * this plan run on.  At most 4 updates are in flight per plan (a fifth waits for the first copy). */
SFD_API int sfd_plan_update_view_async(sfd_plan *plan, int view, double p1, double p2, double z,
                                       double Ox, double Oy, void *stream);
SFD_API int sfd_plan_update_view_general_async(sfd_plan *plan, int view, double p1x, double p1y,
                                               double p2x, double p2y, double z, double O0x,
                                               double O0y, double O1x, double O1y, void *stream);
/* Host time, in milliseconds, the table builder took in the most recent update of this plan. */
SFD_API double sfd_plan_last_update_host_ms(const sfd_plan *plan);

/* General geometry (Eq.(2)-(4) L58-65 and the definitions L67 keep
 * separate x and y sampling pitches, hence S_x = p1x p2x/(lambda z) != S_y = p1y p2y/(lambda z), and
 * offsets (O_x0, O_y0) of the hologram window next to (O_x1, O_y1) of the reconstruction window).
 * Physical coordinates (reading 1 of DESIGN.md): x0 = (m0 - N/2) p1x + O0x, y0 = (n0 - N/2) p1y + O0y,
 * x1 = (m1 - N/2) p2x + O1x, y1 = (n1 - N/2) p2y + O1y, all lengths in metres, arrays [n_views] on
 * the host.  sfd_plan_create is this call with p1x = p1y, p2x = p2y, O0 = 0.
 * Each axis gets its own chirp tables and its own cached kernel spectrum.  Same errors. */
SFD_API int sfd_plan_create_general(sfd_plan **out, int N, int n_views, double lambda,
                                    const double *p1x, const double *p1y, const double *p2x,
                                    const double *p2y, const double *z, const double *O0x,
                                    const double *O0y, const double *O1x, const double *O1y,
                                    int in_dtype);
SFD_API int sfd_plan_update_view_general(sfd_plan *plan, int view, double p1x, double p1y,
                                         double p2x, double p2y, double z, double O0x, double O0y,
                                         double O1x, double O1y);

/* Rectangular grids (Eq.(2)-(3), L58-62, carry N_x and N_y separately): the hologram and every
 * output are [Ny][Nx] (Ny rows along y, Nx samples along x); the optical axis sits at index
 * (Ny/2, Nx/2).  Pass y runs Nx lines of length Ny, pass x Ny lines of length Nx; each axis picks its
 * kernels by its own length.  Nx, Ny: powers of two in 64..2048 (else SFD_EUNSUPPORTED).
 * sfd_plan_create_general is this call with Nx = Ny = N. */
SFD_API int sfd_plan_create_rect(sfd_plan **out, int Nx, int Ny, int n_views, double lambda,
                                 const double *p1x, const double *p1y, const double *p2x,
                                 const double *p2y, const double *z, const double *O0x,
                                 const double *O0y, const double *O1x, const double *O1y,
                                 int in_dtype);

/* Hologram window inside a larger frame (the 1 360 x 1 024 CCD frame is cut down to
 * 1 024 x 1 024; reading 13: a crop, which keeps the 4.65 um pitch the paper then uses, L107).
 * After this call the hologram_dev argument of sfd_execute* points at the FRAME: rows of
 * row_stride samples, of which the plan reads the Ny x Nx window whose first sample is
 * frame[row0][col0] - in place, no copy.  row_stride = 0 restores the dense default (row_stride =
 * Nx, row0 = col0 = 0).  A physical shift of the window goes into O0x / O0y of the plan (the centred
 * crop needs none).  The warp-per-branch kernels need the window's first sample and the row stride on
 * 8-byte boundaries (uint8: col0 and row_stride multiples of 8 on an aligned frame); otherwise the
 * generic kernels run.  sfd_stream_run always reads dense frames.
 * Errors: SFD_EINVAL (negative values, row_stride < col0 + Nx). */
SFD_API int sfd_plan_set_input_window(sfd_plan *plan, long long row_stride, int row0, int col0);

/* Destroy a plan and free everything it owns.  NULL is accepted. */
SFD_API int sfd_plan_destroy(sfd_plan *plan);

/* Plan queries (host): Nx (also as "n"), Ny, n_views, padded FFT length Mx = 2 Nx, the plan's device,
 * bytes of device memory owned. */
SFD_API int sfd_plan_get_n(const sfd_plan *plan);
SFD_API int sfd_plan_get_nx(const sfd_plan *plan);
SFD_API int sfd_plan_get_ny(const sfd_plan *plan);
SFD_API int sfd_plan_get_device(const sfd_plan *plan);
SFD_API int sfd_plan_get_views(const sfd_plan *plan);
SFD_API int sfd_plan_get_m(const sfd_plan *plan);
SFD_API long long sfd_plan_device_bytes(const sfd_plan *plan);

/* Kernel selection.  SFD_KERNELS_AUTO (default): an axis of length 1024 or 2048 runs the
 * warp-per-branch kernels, every other length the generic shared-memory Stockham
 * kernels.
 * SFD_KERNELS_GENERIC forces the generic kernels at every size (tests, A/B timing).  Both compute
 * the same transform; results differ by fp32 rounding only.  Errors: SFD_EINVAL. */
#define SFD_KERNELS_AUTO 0
#define SFD_KERNELS_GENERIC 1
SFD_API int sfd_plan_select_kernels(sfd_plan *plan, int which);

/* Which passes of sfd_execute* on this plan currently run the warp-per-branch kernels: bit 0 = pass
 * y (k_cols_1024 / k_cols_2048; for an aligned hologram), bit 1 = pass x (k_rows_1024 /
 * k_rows_2048); 0 = both run the generic kernels (k_pass_y, k_pass_x); SFD_EINVAL for NULL. */
SFD_API int sfd_plan_uses_warp_kernels(const sfd_plan *plan);

/* Timing aid for benchmarks: CUDA-event time, in milliseconds, of each of the two hot kernels
 * (pass y, pass x) of the most recent execute call on this plan, recorded on the stream they
 * were launched on.  Synchronises on those events.  ms[0] = pass y, ms[1] = pass x,
 * ms[2] = quantise (0 when not run).  Requires sfd_plan_set_timing(plan, 1) beforehand. */
SFD_API int sfd_plan_set_timing(sfd_plan *plan, int enable);
SFD_API int sfd_plan_last_kernel_ms(sfd_plan *plan, float ms[3]);

/* Number of kernel launches issued by all sfd_execute* / sfd_stream_run calls of this process. */
SFD_API long long sfd_launch_count(void);

/* Host-only diagnostic (no GPU needed): the float64 tables the plan builds for ONE axis of one view,
 * before rounding to complex64: pre[N] (Eq. 3), post[N] (Eq. 2 without c0) and the cached kernel
 * spectrum H[2N] = FFT_2N(h)/(2N) (Eq. 4), each as interleaved (re, im) doubles in caller-owned host
 * arrays of 2N, 2N and 4N doubles.  `off` is the window shift along that axis.  N: power of two. */
SFD_API int sfd_host_tables(int N, double lambda, double p1, double p2, double z, double off, double *pre,
                    double *post, double *H);

/* Host-only diagnostic (no GPU needed): one radix-32 stage of the warp FFT as the kernels compute it
 * (sfd_dft32.cuh, fp32, FMA-formulated radix-2 butterflies), stepped on the CPU.  in / out: 32 complex
 * values as interleaved (re, im) floats.  twiddled = 0: out[k] = sum_r in[r] exp(-2 pi i r k / 32)
 * (stage A); twiddled = 1: out[k] = sum_r in[r] exp(-2 pi i (r lane / 1024 + r k / 32)) (stage B of
 * lane `lane`, 0..31, inter-stage twiddles folded in). */
SFD_API int sfd_host_dft32(const float *in, float *out, int lane, int twiddled);

/* Measured pipe rates of the current device, the denominators bench.py reports against:
 * out[0] plain fp32 FMA throughput of the whole GPU in TFLOP/s (2 flop per FMA), out[1] / out[2]
 * cycles of one stage-A / stage-B radix-32 butterfly for a warp that has its sub-partition to
 * itself, out[3] the SM clock during the measurement in GHz.  Runs a few milliseconds of kernels on
 * the legacy default stream and synchronises.  Errors: SFD_EINVAL, SFD_ECUDA. */
SFD_API int sfd_measure_pipes(double out[4]);

/* Measured rates of the two on-chip memories as the warp kernels use them, current device:
 * out[0] shared memory in bytes per clock and SM for the access pattern of the 32 x 32 transposes
 * (16-byte row reads + 8-byte column writes, 8 warps per SM); out[1] / out[2] tensor-memory load rate
 * in bytes per clock and sub-partition with one / two warps per sub-partition (four
 * tcgen05.ld.32x32b.x16 in flight per warp, as the table reads of a line are issued); out[3] cycles of
 * one dependent tcgen05.ld + tcgen05.wait::ld.  Runs a few milliseconds of kernels on the legacy
 * default stream and synchronises.  Errors: SFD_EINVAL, SFD_ECUDA (text: sfd_static_last_error). */
SFD_API int sfd_measure_memory_pipes(double out[4]);

/* The same for a hologram window shifted by off0 along that axis (general geometry). */
SFD_API int sfd_host_tables_general(int N, double lambda, double p1, double p2, double z, double off0,
                                    double off, double *pre, double *post, double *H);

/* ---- angular-spectrum propagation -------------------------------------------
 * Digital holographic microscopy observes "both the amplitude and phase of a specimen".
 * Next to the paper's Shifted-Fresnel transform the library carries the exact (non-paraxial)
 * propagator that SURVEY.md 8(d) uses to define the synthetic holograms:
 *
 *     u(z) = IFFT2[ FFT2[u0] * H ],   H(fx, fy) = exp(i 2 pi z sqrt(1/lambda^2 - fx^2 - fy^2)),
 *
 * on the periodic Ny x Nx grid of pitch (px, py) - a circular convolution, no padding; the caller pads
 * if wrap-around matters.  fx = kx/(Nx px) with bins kx >= Nx/2 negative; components with
 * fx^2 + fy^2 >= 1/lambda^2 (evanescent) are set to zero; band_limit != 0 also zeroes, per axis,
 * |f| > 1/(lambda sqrt((2 z/(N p))^2 + 1)).  One plan holds n_planes depths z[] of one input: the row
 * transform of the input is shared, H is cached per plane (built on the device in float64 at plan
 * creation, 8 bytes per sample and plane).  Three launches per call: the fp32 line-FFT kernels of the
 * generic Fresnel path, and for 1024 x 1024 and 2048 x 2048 grids the warp FFT of the
 * Fresnel fast path, whose column kernel transforms a column forward once for all planes.
 *   Nx, Ny     powers of two in 128..4096 (else SFD_EUNSUPPORTED); z[] finite, any sign, 0 allowed.
 *   in_dtype   SFD_F32 (real input) or SFD_C64.
 * sfd_asm_execute: u0_dev [Ny][Nx] of in_dtype (16-byte aligned for a 2048 x 2048 plan); outputs [n_planes][Ny][Nx]: field_dev complex64,
 * intensity_dev float32 = |u|^2, phase_dev float32 = atan2(im, re) in (-pi, pi]; each may be NULL, not
 * all three.  Asynchronous on `stream`; calls on one plan must be ordered (one stream, or events): the
 * plan owns the intermediates between its three kernels.
 * Errors: SFD_EINVAL, SFD_EUNSUPPORTED, SFD_ENOMEM, SFD_ECUDA (text: sfd_asm_last_cuda_error). */
typedef struct sfd_asm_plan sfd_asm_plan; /* opaque */
SFD_API int sfd_asm_plan_create(sfd_asm_plan **out, int Nx, int Ny, int n_planes, double lambda,
                                double px, double py, const double *z, int in_dtype, int band_limit);
SFD_API int sfd_asm_execute(sfd_asm_plan *plan, const void *u0_dev, void *field_dev,
                            float *intensity_dev, float *phase_dev, void *stream);
SFD_API int sfd_asm_plan_destroy(sfd_asm_plan *plan);
SFD_API long long sfd_asm_plan_device_bytes(const sfd_asm_plan *plan);
SFD_API const char *sfd_asm_last_cuda_error(void);

/* Static description of an error code / of the last CUDA error seen by this thread. */
SFD_API const char *sfd_error_string(int code);
SFD_API const char *sfd_last_cuda_error(void);

/* Library version, e.g. "sfd 0.1 sm_100a". */
SFD_API const char *sfd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SFD_H */
