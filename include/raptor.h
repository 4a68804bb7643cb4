/* raptor.h -- C ABI of the B200-native RAPTOR hot path (arXiv:1801.10452, Bronzwaer et al. 2018).
 *
 * One image = for every pixel, backward RK4 integration of a Kerr null geodesic in modified
 * Kerr-Schild coordinates fused with the covariant transfer update of I_nu/nu^3 along the ray.
 * Citations are lines of the paper text with the equation they fall in; [A#] are the
 * readings listed in DESIGN.md.  Plain pointers and sizes only; nothing throws across this
 * boundary; no global state; a context is not thread-safe.
 *
 * Every function returns 0 (RAPTOR_OK) or a negative RAPTOR_E* code; raptor_last_error() gives
 * the message.  "device" pointers are CUDA device memory of the current device, owned by the
 * caller; "host" pointers are ordinary host memory.  Calls taking a cuda_stream (a cudaStream_t
 * cast to void*, NULL = default stream) are asynchronous on that stream.
 *
 * Ordering: the asynchronous calls of one context share its scene data, its tile queue and its scratch
 * buffers.  Issue them on ONE stream, or order the streams yourself (event / synchronise) before the next
 * call on the same context; two calls of one context in flight at the same time are undefined.  The
 * host-buffer call raptor_render_host runs on the context's own stream and orders itself after every
 * earlier call made on that context (uploads included), then synchronises.
 */
#ifndef RAPTOR_B200_H
#define RAPTOR_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RAPTOR_ABI_VERSION 3u

enum {
    RAPTOR_OK = 0,
    RAPTOR_EINVAL = -1,        /* a parameter is out of range (message says which) */
    RAPTOR_ENOMEM = -2,        /* device or host allocation failed */
    RAPTOR_ECUDA = -3,         /* a CUDA call or kernel launch failed */
    RAPTOR_EUNSUPPORTED = -4   /* valid request that this build does not implement */
};

/* plasma_model */
enum { RAPTOR_VACUUM = 0, RAPTOR_SPHERE = 1, RAPTOR_TORUS = 2, RAPTOR_GRID2D = 3, RAPTOR_GRID3DT = 4, RAPTOR_SLAB = 5,
       RAPTOR_DISK = 6 /* thin-disk workload of Sect. 4.2.1: raptor_render_disk */ };
/* per-ray status word written by raptor_render */
enum { RAPTOR_RUNNING = 0, RAPTOR_CAPTURED = 1, RAPTOR_ESCAPED = 2, RAPTOR_MAXSTEPS = 3, RAPTOR_THICK = 4, RAPTOR_NONFINITE = 5 };

#define RAPTOR_MAX_FREQ 64

typedef struct raptor_ctx raptor_ctx;   /* opaque; owns the device copies of the scene data */

/* Statement of the problem (Table 2, Table B.1).
 * POD, caller-owned, copied by raptor_create (including freq_hz[] and the grid). */
typedef struct {
    uint32_t struct_size;      /* = sizeof(raptor_params) */
    uint32_t abi_version;      /* = RAPTOR_ABI_VERSION */
    /* spacetime and chart: Kerr, M = 1, modified Kerr-Schild x = (t~, x1, x2, phi~), r = r0 + exp(x1),
     * theta = pi x2 + (1-h)/2 sin(2 pi x2)  (A.10-A.11); h = 1: logarithmic KS */
    double a;                  /* spin, |a| < 1 */
    double mks_h;              /* 0 < h <= 1 */
    double mks_r0;             /* r0 < r_H */
    double mass;               /* mass parameter m multiplying every 2r of the metric: 1; 0 = flat space (tests) */
    /* camera: Eq. 25-29, pixel centres alpha_ix = (ix+1/2) fov/nx - fov/2 [A4b] */
    double r_cam;              /* camera radius [M], > r_H */
    double incl_deg;           /* inclination, 0 < i < 180 (0 and 180 sit on the coordinate axis: rejected) */
    double fov_M;              /* full width of the image plane [M] */
    double t_cam;              /* coordinate time of the camera (slow light) */
    /* physical scaling */
    double M_bh_g;             /* black-hole mass [g]: L = G M / c^2 */
    double D_src_cm;           /* distance [cm] */
    double M_unit_g;           /* mass unit [g]: rho0 = M_unit / L^3 (grid models) */
    /* integrator (field `integrator` below), backward (d lambda = -h) [A2]: RK4 Eq. 7-16;
     * velocity Verlet Eq. 17-20 without / with the corrector re-evaluation of PAPER.md:127;
     * "RK2" of Table B.1 = explicit midpoint [A17] */
    double step_c, step_min, step_max;   /* policy A: h = clamp(c (r - r_H), min, max) (BASELINE.json configs[0]) */
    double eps, delta;         /* policy B: Eq. 21-24 */
    double eps_polar;          /* policy A polar guard: h <= eps_polar r |sin theta| (Eq. 23 with |k^theta| <= 1/r) */
    double r_stop_in_factor;   /* stop when r < factor * r_H   (1.01) */
    double r_stop_out_factor;  /* stop when r > factor * r_cam (1.1) */
    double tau_cutoff;         /* stop when min_k tau_k exceeds it; +inf = off */
    /* plasma */
    double model[16];          /* SPHERE: n0, n_exp, T0[K], T_exp, beta.  TORUS: n_max, r_peak, r_halfwidth,
                                  scale height H, T0, T_exp, beta.  SLAB: n_e, Theta_e, B[G], half thickness, sin(pitch).
                                  DISK: r_in (<= 0: ISCO), r_out, max image order, p.  Grids with te_model = 1: R_low, R_high */
    double tp_over_te;         /* T_p/T_e (Table 2), te_model = 0 */
    double gamma_ad;           /* adiabatic index of the grid fluid */
    /* grid (GRID2D, GRID3DT): cell-centred, x1_i = x1_min + (i+1/2)(x1_max-x1_min)/n1, x2_j = (j+1/2)/n2,
     * phi_k = (k+1/2) 2pi/n3, t_m = t0 + m dt_snap [A16] */
    double x1_min, x1_max, t0, dt_snap;
    const double *freq_hz;     /* host, n_freq observer frequencies [Hz] */
    const void *grid_host;     /* host, AoS [nt][n1][n2][n3][8] = rho, u, u~1, u~2, u~3, B1, B2, B3 (HARM primitives) */
    uint64_t grid_bytes;       /* must equal nt*n1*n2*n3*8*sizeof(element) */
    int32_t nx, ny;            /* pixels */
    int32_t integrator;        /* 0 = RK4, 1 = Verlet, 2 = Verlet + corrector, 3 = RK2 (midpoint) */
    int32_t step_policy;       /* 0 = A, 1 = B */
    int32_t max_steps;         /* per ray */
    int32_t n_freq;            /* 1 .. RAPTOR_MAX_FREQ */
    int32_t plasma_model;
    int32_t k2_mode;           /* 0: K_2(1/Theta) = 2 Theta^2; 1: K_2 evaluated (Eq. 41-42 as written) */
    int32_t n1, n2, n3, nt;
    int32_t grid_dtype;        /* 0 = float64, 1 = float32 */
    int32_t slow_light;        /* 1: interpolate between snapshots at the ray's coordinate time */
    int32_t snapshot;          /* fast light: snapshot index used */
    int32_t te_model;          /* 0: constant tp_over_te; 1: Eq. 47, model[0] = R_low, model[1] = R_high (grids) */
    int32_t precision;         /* 0: FP64 (the contract).  1: FP32, the paper's own performance configuration only (Table B.1,
                                  PAPER.md:638-647 "Single precision: yes"): plasma_model = GRID2D, integrator = 3 (RK2),
                                  step_policy = 1, n_freq = 1, k2_mode = 0, te_model = 0; raptor_render / raptor_spectrum /
                                  raptor_flux / raptor_render_host / raptor_trace; images are still written as float64 */
    int32_t reserved_;         /* 0 */
} raptor_params;

/* Validates and copies *p, uploads frequencies and grid.  *out is NULL on failure (then
 * raptor_last_error(NULL) holds the thread-local message).  Synchronous. */
int raptor_create(const raptor_params *p, raptor_ctx **out);

/* Replaces the context's grid by a new one of identical shape (next snapshot series / movie frame).
 * host -> device copy on the stream. */
int raptor_upload_grid(raptor_ctx *ctx, const void *grid_host, uint64_t grid_bytes, void *cuda_stream);

/* Steps a1-a7 of the hot path for the whole image:
 *   d_image  device, [n_freq][ny][nx] float64: I_nu,obs in erg s^-1 cm^-2 Hz^-1 sr^-1 (Eq. 32)
 *   d_status device, [ny][nx] int32 status word, or NULL
 *   d_nsteps device, [ny][nx] int32 accepted RK4 steps of the ray, or NULL */
int raptor_render(raptor_ctx *ctx, double *d_image, int32_t *d_status, int32_t *d_nsteps, void *cuda_stream);

/* Thin-disk workload (Sect. 4.2.1; plasma_model = RAPTOR_DISK, n_freq = 1) [A24]: a steady,
 * geometrically thin Keplerian disk in the equatorial plane between r_in (the ISCO) and r_out with emission
 * coefficient ~ 1/r^2 and no absorption.  Every crossing of the equatorial plane of order <= max order inside
 * [r_in, r_out] adds g^p / r^2, g = nu_obs/nu_em = 1/(-k.u) (Eq. 31-32); crossing state by linear
 * interpolation within the step.
 *   d_image    device, [ny][nx] float64: sum over the counted crossings (arbitrary units)
 *   d_redshift device, [ny][nx] float64: g of the first counted crossing, 0 where there is none
 *   d_status, d_nsteps as raptor_render (or NULL) */
int raptor_render_disk(raptor_ctx *ctx, double *d_image, double *d_redshift, int32_t *d_status, int32_t *d_nsteps,
                       void *cuda_stream);

/* Line profile of the disk (Fig. 6): d_hist device [nbins], bin b of [g_min, g_max) receives
 * sum I (fov/nx)(fov/ny) over the pixels whose redshift factor falls into it (g = 0 pixels are skipped).
 * Fixed summation order (deterministic). */
int raptor_line_profile(raptor_ctx *ctx, const double *d_image, const double *d_redshift, int32_t nbins, double g_min,
                        double g_max, double *d_hist, void *cuda_stream);

/* Slow-light movies and light curves (Sect. 5; plasma_model = RAPTOR_GRID3DT, slow_light = 1).
 * The context holds nt snapshots; for a series longer than nt they form a sliding window: snapshot m (time
 * t0 + m dt_snap) lives in slot m mod nt, and the resident window is [first, first + nt).  A ray's coordinate time
 * is clamped to the window.  raptor_upload_snapshot copies ONE snapshot (host, [n1][n2][n3][8]) into its slot on the
 * stream; raptor_set_window moves the window (default first = 0); raptor_set_camera_time changes t_cam (the
 * time-calibration delay of Sect. 5.1, is part of t_cam [A15]). */
int raptor_set_camera_time(raptor_ctx *ctx, double t_cam);
int raptor_set_window(raptor_ctx *ctx, int64_t first_snapshot);
int raptor_upload_snapshot(raptor_ctx *ctx, int64_t snapshot, const void *snapshot_host, uint64_t bytes, void *cuda_stream);

/* Light curve: frames f = 0 .. n_frames-1 rendered at camera times t_cam0 + f dt_frame through the resident window
 * and reduced to d_flux_jy[f][k] (device, [n_frames][n_freq], Jy); the images are not kept.  The frames of a batch
 * (up to 256 MiB of images) are traced by ONE launch of the ray kernel -- small frames cannot fill the GPU one at a
 * time -- and reduced by one deterministic reduction.  The context's own t_cam is left unchanged; the tile shard
 * must be (0, 1) (light curves shard by frames). */
int raptor_light_curve(raptor_ctx *ctx, int32_t n_frames, double t_cam0, double dt_frame, double *d_flux_jy, void *cuda_stream);

/* Time calibration of Sect. 5.1: "an empirical, pragmatic strategy ... effectively equivalent to
 * translating the slow-light light curve with respect to the fast-light light curve on the time axis".  Both curves
 * are normalised by their means; for each of the n_grid shifts d_k = -max_shift + 2 max_shift k/(n_grid - 1) the
 * slow-light curve is interpolated linearly at t_fast[i] + d_k (points outside [t_slow[0], t_slow[n_slow-1]] are
 * left out; a shift that keeps fewer than max(4, n_fast/2) points is skipped) and the rms difference to the
 * fast-light curve is formed; *delay receives the first shift with the smallest rms, *rms that rms (+inf and
 * delay 0 if every shift was skipped).  HOST pointers; plain host arithmetic, synchronous.  RAPTOR_EINVAL if t_slow is
 * not strictly ascending or the mean of either curve is zero or not finite. */
int raptor_calibrate_delay(int32_t n_fast, const double *t_fast, const double *F_fast, int32_t n_slow, const double *t_slow,
                           const double *F_slow, double max_shift, int32_t n_grid, double *delay, double *rms);

/* Multi-GPU sharding of one image: after this call raptor_render / raptor_spectrum /
 * raptor_render_host trace only the 8x4-pixel tiles whose raster index ty * ceil(nx/8) + tx is rank modulo world
 * (interleaved, so that shadow and torus are spread evenly; the kernel launches them nearest to the image centre first)
 * and leave every other pixel of the caller's output buffers untouched.  Rays are independent, so the ranks'
 * images (zero-initialised by the caller) sum to the full image exactly.  Where the library owns the image
 * (raptor_spectrum with a NULL image, raptor_render_host) it zeroes it first, so fluxes are the shard's own and
 * sum to the full flux.  Default (0, 1) = whole image.  Synchronises the device (the shard's tile table is replaced). */
int raptor_set_shard(raptor_ctx *ctx, int32_t rank, int32_t world);

/* Render + flux reduction (the spectra of Fig. 2, units PAPER.md:248, and the fluxes of Table 3):
 * d_flux_jy device [n_freq], F_k = 1e23 sum_pix I_k (fov/nx)(fov/ny) L^2/D^2 [Jy] -- the pixel's solid angle as seen
 * from distance D times its intensity -- summed in a fixed order (deterministic).  d_image_or_null: as d_image, or NULL
 * to use scratch. */
int raptor_spectrum(raptor_ctx *ctx, double *d_flux_jy, double *d_image_or_null, void *cuda_stream);

/* Flux reduction alone (same sum and units: Fig. 2; Table 3) of an image already on the device. */
int raptor_flux(raptor_ctx *ctx, const double *d_image, double *d_flux_jy, void *cuda_stream);

/* Flux reduction for callers that must not allocate device memory (same sum as raptor_flux: Fig. 2 units,
 * PAPER.md:248; F_k = scale * sum_pix I_k, fixed order).
 *
 * Who needs it: raptor_flux wants a context, and raptor_create takes its buffers from cudaMalloc.  That is not open to
 * everybody -- a plug-in whose host program has already given the whole device to its own memory pool, a job with a
 * device-memory budget fixed in advance, a loop that cannot afford cudaMalloc's device-wide synchronisation, or code
 * that merely holds an image on the device and has no context at all.  This call needs no context and calls neither
 * cudaMalloc nor cudaFree nor any library routine that allocates: the partial sums of the reduction sit in an array
 * that is part of the library image (128 KiB on every GPU that loads the library, held until the process exits).
 *
 *   d_image   device, [n_planes][npix] float64 (for an image of raptor_render: n_planes = n_freq, npix = ny * nx)
 *   scale     factor applied to each sum; raptor_flux uses 1e23 (fov/nx)(fov/ny) L^2/D^2 for Jy, 1 gives plain sums
 *   d_flux    device, [n_planes] float64, written on the stream
 * Limit: n_planes * ceil(npix / 16384) <= RAPTOR_FLUX_STATIC_MAX_PARTIALS (e.g. 64 planes of 2048 x 2048 pixels);
 * anything larger, npix = 0, n_planes < 1 or a NULL buffer returns RAPTOR_EINVAL with the numbers in the message
 * (raptor_last_error(NULL)), and nothing is launched.  For the same image and scale the result equals raptor_flux's
 * bit for bit.
 *
 * The first call on each device looks up the device address of the array (one cudaGetSymbolAddress, which may also
 * make the driver load the library's code onto that device); make that first call once per device during start-up,
 * with the device current, before any stream capture begins.  Later calls only launch two kernels on the stream.
 * All calls on one device share the one array: it keeps what the last call left, which is harmless because every
 * element a call reads it has written itself first -- but two calls that can run on the GPU at the same time
 * (different streams, no ordering between them) race on it and both results are then undefined.  Keep the calls of a
 * device on one stream or order them with events. */
#define RAPTOR_FLUX_STATIC_MAX_PARTIALS 16384
int raptor_flux_static(const double *d_image, uint64_t npix, int32_t n_planes, double scale, double *d_flux,
                       void *cuda_stream);

/* End-to-end convenience with HOST buffers: render on the context's own stream (after every earlier call on
 * this context has finished, see "Ordering"), copy image ([n_freq][ny][nx]), optional status / nsteps ([ny][nx])
 * and optional flux ([n_freq]) back, synchronise.  Under a shard the pixels of other ranks' tiles come back 0. */
int raptor_render_host(raptor_ctx *ctx, double *h_image, int32_t *h_status, int32_t *h_nsteps, double *h_flux_jy);

/* Diagnostics: trace n rays with given impact parameters (device arrays alpha[n], beta[n]) through the same
 * device code as raptor_render.  Outputs (device, any may be NULL): I[n_freq][n], tau[n_freq][n], final
 * state XK[n][8] = (X^0..3, K^0..3), status[n], nsteps[n]. */
int raptor_trace(raptor_ctx *ctx, int32_t n, const double *d_alpha, const double *d_beta, double *d_I, double *d_tau,
                 double *d_XK, int32_t *d_status, int32_t *d_nsteps, void *cuda_stream);

/* Diagnostics: geodesic right-hand side f^a = -Gamma^a_bc k^b k^c (Eq. 6) at n points,
 * d_XK[n][8] in, d_f[n][4] out (device). */
int raptor_eval_rhs(raptor_ctx *ctx, int32_t n, const double *d_XK, double *d_f, void *cuda_stream);

/* Diagnostics: the null condition g_mn k^m k^n (Eq. 4) at n states, d_XK[n][8] in (e.g. the final
 * states raptor_trace returns), d_out[n] out (device): 0 up to the integrator's truncation error.  d_ELQ_or_null
 * (device, [n][3]) receives the constants of motion E = -k_t, L = k_phi, Q of Eq. 38-40. */
int raptor_null_norm(raptor_ctx *ctx, int32_t n, const double *d_XK, double *d_out, double *d_ELQ_or_null, void *cuda_stream);

/* Null-condition monitor (Eq. 4): while d_null_max_or_null is set, raptor_render,
 * raptor_render_disk and raptor_trace also evaluate g_mn k^m k^n at the new point of EVERY step and write its largest
 * magnitude along each ray to d_null_max ([ny][nx], resp. [n]; device, caller-owned, must stay valid until unset).
 * A ray whose norm peaked near the horizon and recovered is visible here, not in the end state.  The default kernels
 * are unchanged; the monitoring variants cost about 5 % more.  NULL switches it off.  (raptor_light_curve ignores it.)
 * capacity = number of float64 elements the buffer holds (ignored for NULL): while the monitor is set, a call that would
 * write more than that (an image of ny * nx > capacity pixels, a trace of n > capacity rays) returns RAPTOR_EINVAL and
 * launches nothing -- a buffer sized for a trace and left set across a render cannot be overrun.  raptor_spectrum and
 * raptor_render_host go through raptor_render and therefore monitor as well while it is set. */
int raptor_set_null_monitor(raptor_ctx *ctx, double *d_null_max_or_null, uint64_t capacity);

/* Counters accumulated by every render / trace since creation: accepted integrator steps, steps on which plasma was
 * sampled, rays traced.  Waits for the last call made on this context (not for the device: other streams keep
 * running).  No passage of the paper: measurement (SURVEY.md 8(d) needs the step count of an image). */
int raptor_get_counters(raptor_ctx *ctx, uint64_t *total_steps, uint64_t *sampled_steps, uint64_t *rays);

/* Measures the FP64 FMA peak of the current device with independent DFMA chains on all SMs:
 * *tflops = 2 * FMAs / time.  iters = chain length per thread (e.g. 1<<16). Synchronous. */
int raptor_fp64_peak(int32_t iters, double *tflops, double *ms);

/* The same for the FP32 FMA pipe (16 independent FFMA chains per thread): the denominator of the roofline of the
 * single-precision kernel (precision = 1).  Synchronous. */
int raptor_fp32_peak(int32_t iters, double *tflops, double *ms);

/* Issue rate of the FP64 pipe by operand form (independent chains on all SMs, 8 warps per sub-partition):
 * form 0 fma(x, imm, imm); 1 fma(y, z, x) = three different register sources; 2 fma(x, y, x); 3 x * y; 4 x + z.
 * *warp_inst_per_sec = warp-level instructions per second over the whole device; *sm_clock_hz (may be NULL) = the
 * device's nominal SM clock, so that cycles per instruction per sub-partition = 4 SMs clock / rate.  Synchronous.
 * On B200 a DFMA with three different register sources issues every 3.2 cycles, every other form every 2.06
 * (DESIGN.md 5.1): the bound of a kernel depends on its operand forms, not only on its instruction count. */
int raptor_fp64_probe(int32_t form, int32_t iters, double *warp_inst_per_sec, double *sm_clock_hz);

/* Releases the context and its device memory (NULL is allowed).  No passage of the paper: lifecycle. */
int raptor_destroy(raptor_ctx *ctx);

/* Message of the last failure on this context; ctx == NULL: of the last failed raptor_create /
 * raptor_fp64_peak on this thread.  Never NULL. */
const char *raptor_last_error(const raptor_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* RAPTOR_B200_H */
