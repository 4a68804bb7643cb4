// raptor_api.cu -- the C ABI of include/raptor.h: validation, scene upload, launches.  Host code only.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <limits>
#include <new>
#include <utility>
#include <vector>

#include "../../include/raptor.h"
#include "raptor_kernels.h"

using namespace raptor;

struct raptor_ctx;
static int ensure_scratch(raptor_ctx* ctx);
static int mark(raptor_ctx* ctx, cudaStream_t s);

struct raptor_ctx {
    raptor_params p;
    KP kp;
    int device = 0, sm_count = 148;
    int shard_rank = 0, shard_world = 1;   // raptor_set_shard
    long long window_lo = 0;               // raptor_set_window
    void* d_grid = nullptr;
    size_t grid_bytes = 0;
    double* d_freq = nullptr;
    double nu0 = 0.0;                      // first frequency (precision = 1 has exactly one)
    unsigned int* d_queue = nullptr;
    unsigned int* d_order = nullptr;       // tiles of one image sorted by the distance of their centre from the image centre
    unsigned int* d_order_shard = nullptr; // the same for this rank's tiles (tile index mod world == rank), raptor_set_shard
    std::vector<unsigned> order_host;
    unsigned long long* d_counters = nullptr;
    double* d_partial = nullptr;      // flux partial sums [n_freq][chunks]
    double* d_profile_partial = nullptr;   // line-profile partial sums [nbins][chunks]
    double* d_lc_partial = nullptr;        // light-curve partial sums [frames * n_freq][chunks]
    size_t lc_planes = 0;
    int profile_bins = 0;
    double* d_scratch_image = nullptr;
    double* d_scratch_flux = nullptr;
    size_t scratch_pixels = 0;
    cudaStream_t own_stream = nullptr;
    KPf kpf;                               // precision = 1
    float* d_grid_f32 = nullptr;           // precision = 1: (float) of d_grid
    double* d_null_max = nullptr;          // raptor_set_null_monitor: caller-owned output of the next render / trace calls
    uint64_t null_max_capacity = 0;        // elements the caller said it holds
    cudaEvent_t ev_last = nullptr;         // recorded after every asynchronous call: raptor_render_host orders itself after it
    char err[512] = {0};
};

static thread_local char g_err[512] = "";

static int fail(raptor_ctx* ctx, int code, const char* fmt, ...) {
    char* dst = ctx ? ctx->err : g_err;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 512, fmt, ap);
    va_end(ap);
    return code;
}
#define CK(ctx, call)                                                                                      \
    do {                                                                                                   \
        cudaError_t e_ = (call);                                                                           \
        if (e_ != cudaSuccess)                                                                             \
            return fail(ctx, e_ == cudaErrorMemoryAllocation ? RAPTOR_ENOMEM : RAPTOR_ECUDA, "%s: %s", #call, \
                        cudaGetErrorString(e_));                                                           \
    } while (0)

// theta(x2) of A.11 and its inverse by Newton-Raphson, A.14-A.16, on the lower half and mirrored
// ([A22]: as printed the iteration cycles for theta near pi when h < 1).  Once per image, on the host.
static double x2_of_theta(double h, double theta) {
    const bool mirror = theta > 0.5 * kPI;
    const double target = mirror ? kPI - theta : theta;
    double x = 0.01;
    for (int it = 0; it < 200; ++it) {
        double f = kPI * x + 0.5 * (1.0 - h) * std::sin(2.0 * kPI * x) - target;      // A.15
        double fp = kPI * (1.0 + (1.0 - h) * std::cos(2.0 * kPI * x));                // A.16
        if (std::fabs(fp) < 1e-12) { x = 0.05; continue; }
        double xn = x - f / fp;                                                       // A.14
        if (xn < 0.0 || xn > 1.0) xn = 0.05;
        bool done = std::fabs(xn - x) < 1e-15;
        x = xn;
        if (done) break;
    }
    return mirror ? 1.0 - x : x;
}

static size_t grid_elem_size(const raptor_params& p) { return p.grid_dtype == 1 ? sizeof(float) : sizeof(double); }
static uint64_t grid_expected_bytes(const raptor_params& p) {
    return (uint64_t)p.nt * p.n1 * p.n2 * p.n3 * 8ull * grid_elem_size(p);
}

static int validate(const raptor_params* p) {
    if (!p) return fail(nullptr, RAPTOR_EINVAL, "params is NULL");
    if (p->struct_size != sizeof(raptor_params)) return fail(nullptr, RAPTOR_EINVAL, "struct_size %u != %zu", p->struct_size, sizeof(raptor_params));
    if (p->abi_version != RAPTOR_ABI_VERSION) return fail(nullptr, RAPTOR_EINVAL, "abi_version %u != %u", p->abi_version, RAPTOR_ABI_VERSION);
    if (!(std::fabs(p->a) < 1.0)) return fail(nullptr, RAPTOR_EINVAL, "spin |a| must be < 1");
    if (!(p->mass >= 0.0)) return fail(nullptr, RAPTOR_EINVAL, "mass parameter must be >= 0");
    if (!(p->mks_h > 0.0 && p->mks_h <= 1.0)) return fail(nullptr, RAPTOR_EINVAL, "mks_h must be in (0,1]");
    if (!(p->incl_deg > 0.0 && p->incl_deg < 180.0)) return fail(nullptr, RAPTOR_EINVAL, "inclination must be in (0,180) deg: 0 and 180 sit on the coordinate axis");
    if (p->nx < 1 || p->ny < 1) return fail(nullptr, RAPTOR_EINVAL, "nx, ny must be >= 1");
    if ((long long)p->nx * p->ny > (1ll << 31) - 64) return fail(nullptr, RAPTOR_EINVAL, "too many pixels");
    if (p->n_freq < 1 || p->n_freq > RAPTOR_MAX_FREQ || !p->freq_hz) return fail(nullptr, RAPTOR_EINVAL, "n_freq must be 1..%d with freq_hz set", RAPTOR_MAX_FREQ);
    for (int k = 0; k < p->n_freq; ++k)
        if (!(p->freq_hz[k] > 0.0) || !std::isfinite(p->freq_hz[k])) return fail(nullptr, RAPTOR_EINVAL, "freq_hz[%d] must be positive", k);
    double disc = p->mass * p->mass - p->a * p->a;
    double rH = disc >= 0.0 ? p->mass + std::sqrt(disc) : 0.0;
    if (!(p->r_cam > rH) || !(p->r_cam > p->mks_r0)) return fail(nullptr, RAPTOR_EINVAL, "r_cam must be outside the horizon");
    if (!(p->mks_r0 < rH || p->mass == 0.0)) return fail(nullptr, RAPTOR_EINVAL, "mks_r0 must be < r_H");
    if (!(p->fov_M > 0.0)) return fail(nullptr, RAPTOR_EINVAL, "fov_M must be > 0");
    if (p->integrator < 0 || p->integrator > 3) return fail(nullptr, RAPTOR_EINVAL, "integrator %d: 0 RK4, 1 Verlet, 2 Verlet + corrector, 3 RK2", p->integrator);
    if (p->step_policy != 0 && p->step_policy != 1) return fail(nullptr, RAPTOR_EINVAL, "step_policy must be 0 or 1");
    if (p->step_policy == 0 && !(p->step_min > 0.0 && p->step_max >= p->step_min && p->step_c >= 0.0 && p->eps_polar > 0.0))
        return fail(nullptr, RAPTOR_EINVAL, "policy A needs 0 < step_min <= step_max, step_c >= 0, eps_polar > 0");
    if (p->step_policy == 1 && !(p->eps > 0.0 && p->delta > 0.0)) return fail(nullptr, RAPTOR_EINVAL, "policy B needs eps > 0, delta > 0");
    if (p->max_steps < 1) return fail(nullptr, RAPTOR_EINVAL, "max_steps must be >= 1");
    if (!(p->r_stop_in_factor > 0.0) || !(p->r_stop_out_factor >= 1.0)) return fail(nullptr, RAPTOR_EINVAL, "bad r_stop factors");
    if (std::isnan(p->tau_cutoff)) return fail(nullptr, RAPTOR_EINVAL, "tau_cutoff is NaN");
    if (p->plasma_model < 0 || p->plasma_model > 6) return fail(nullptr, RAPTOR_EINVAL, "unknown plasma_model %d", p->plasma_model);
    if (p->plasma_model == RAPTOR_DISK) {
        if (p->n_freq != 1) return fail(nullptr, RAPTOR_EINVAL, "DISK: n_freq must be 1 (the line is monochromatic in the emitter frame)");
        if (!(p->model[1] > 0.0) || !(p->model[2] >= 1.0) || !std::isfinite(p->model[3]))
            return fail(nullptr, RAPTOR_EINVAL, "DISK: model = [r_in (<= 0: ISCO), r_out > 0, max_order >= 1, p]");
    }
    if (p->precision != 0 && p->precision != 1) return fail(nullptr, RAPTOR_EINVAL, "precision %d: 0 (FP64) or 1 (FP32)", p->precision);
    if (p->precision == 1 && !(p->plasma_model == RAPTOR_GRID2D && p->integrator == 3 && p->step_policy == 1 && p->n_freq == 1 &&
                               p->k2_mode == 0 && p->te_model == 0))
        return fail(nullptr, RAPTOR_EUNSUPPORTED, "precision 1 (FP32) is built for the paper's performance configuration only: "
                                                  "GRID2D, integrator 3 (RK2), step_policy 1, n_freq 1, k2_mode 0, te_model 0");
    if (p->k2_mode != 0 && p->k2_mode != 1) return fail(nullptr, RAPTOR_EINVAL, "k2_mode %d: 0 (K2 = 2 Theta^2, PAPER.md:303) or 1 (exact K2)", p->k2_mode);
    if (p->te_model != 0 && p->te_model != 1) return fail(nullptr, RAPTOR_EINVAL, "te_model %d: 0 (constant T_p/T_e) or 1 (Eq. 47)", p->te_model);
    if (p->te_model == 1 && !(p->model[0] >= 0.0 && p->model[1] >= 0.0)) return fail(nullptr, RAPTOR_EINVAL, "te_model 1 needs model[0] = R_low >= 0, model[1] = R_high >= 0");
    if (!(p->M_bh_g > 0.0) || !(p->D_src_cm > 0.0)) return fail(nullptr, RAPTOR_EINVAL, "M_bh_g and D_src_cm must be > 0");
    if (p->plasma_model == RAPTOR_GRID2D || p->plasma_model == RAPTOR_GRID3DT) {
        if (p->n1 < 2 || p->n2 < 2 || p->n3 < 1 || p->nt < 1) return fail(nullptr, RAPTOR_EINVAL, "grid dims: n1, n2 >= 2, n3, nt >= 1");
        if (p->plasma_model == RAPTOR_GRID2D && (p->n3 != 1 || p->nt != 1 || p->grid_dtype != 0))
            return fail(nullptr, RAPTOR_EINVAL, "GRID2D is [n1][n2][8] float64 (n3 = nt = 1)");
        if (p->plasma_model == RAPTOR_GRID3DT && p->grid_dtype != 1)
            return fail(nullptr, RAPTOR_EUNSUPPORTED, "GRID3DT is built for float32 cells (grid_dtype = 1)");
        if (!(p->x1_max > p->x1_min)) return fail(nullptr, RAPTOR_EINVAL, "x1_max must be > x1_min");
        if (!p->grid_host) return fail(nullptr, RAPTOR_EINVAL, "grid_host is NULL");
        if (p->grid_bytes != grid_expected_bytes(*p)) return fail(nullptr, RAPTOR_EINVAL, "grid_bytes %llu != nt*n1*n2*n3*8*elem = %llu", (unsigned long long)p->grid_bytes, (unsigned long long)grid_expected_bytes(*p));
        if (p->snapshot < 0 || p->snapshot >= p->nt) return fail(nullptr, RAPTOR_EINVAL, "snapshot out of range");
        if (p->nt > 1 && p->slow_light && !(p->dt_snap > 0.0)) return fail(nullptr, RAPTOR_EINVAL, "dt_snap must be > 0");
        if (!(p->M_unit_g > 0.0)) return fail(nullptr, RAPTOR_EINVAL, "M_unit_g must be > 0 for grid models");
        if (!(p->gamma_ad > 1.0) || !(p->tp_over_te >= 0.0)) return fail(nullptr, RAPTOR_EINVAL, "gamma_ad > 1, tp_over_te >= 0");
    }
    return RAPTOR_OK;
}

// innermost stable circular orbit of the equatorial Kerr geodesics (Bardeen, Press & Teukolsky 1972)
static double r_isco(double a) {
    const double z1 = 1.0 + std::cbrt(1.0 - a * a) * (std::cbrt(1.0 + a) + std::cbrt(1.0 - a));
    const double z2 = std::sqrt(3.0 * a * a + z1 * z1);
    const double sg = a > 0.0 ? 1.0 : (a < 0.0 ? -1.0 : 0.0);
    return 3.0 + z2 - sg * std::sqrt((3.0 - z1) * (3.0 + z1 + 2.0 * z2));
}

static void build_kp(raptor_ctx* c) {
    const raptor_params& p = c->p;
    KP& k = c->kp;
    std::memset(&k, 0, sizeof(k));
    k.a = p.a; k.a2 = p.a * p.a; k.twoa = 2.0 * p.a; k.m = p.mass; k.twom = 2.0 * p.mass; k.omh = 1.0 - p.mks_h; k.r0 = p.mks_r0;
    k.pi_omh = kPI * k.omh; k.half_omh = 0.5 * k.omh; k.d2th_c = (-2.0 * kPI * kPI) * k.omh;
    const double inc = p.incl_deg * (kPI / 180.0);
    k.r_cam = p.r_cam; k.sin_i = std::sin(inc); k.cos_i = std::cos(inc);
    k.sq1mc2 = std::sqrt(1.0 - k.cos_i * k.cos_i);
    k.x1_cam = std::log(p.r_cam - p.mks_r0);
    k.x2_cam = x2_of_theta(p.mks_h, inc);
    k.dth_cam = kPI * (1.0 + (1.0 - p.mks_h) * std::cos(2.0 * kPI * k.x2_cam));
    k.t_cam = p.t_cam;
    k.fov = p.fov_M; k.pix_dx = p.fov_M / p.nx; k.pix_dy = p.fov_M / p.ny;
    k.step_c = p.step_c; k.step_min = p.step_min; k.step_max = p.step_max;
    k.eps = p.eps; k.delta = p.delta; k.eps_polar = p.eps_polar;
    const double disc = p.mass * p.mass - p.a * p.a;
    k.rH = disc >= 0.0 ? p.mass + std::sqrt(disc) : 0.0;
    k.step_c_rH = -p.step_c * k.rH;
    k.r_in = p.r_stop_in_factor * k.rH; k.r_out = p.r_stop_out_factor * p.r_cam;
    k.tau_cutoff = p.tau_cutoff; k.use_tau_cutoff = std::isfinite(p.tau_cutoff) ? 1 : 0;
    k.Lcm = kG * p.M_bh_g / (kC * kC);
    const double rho0 = p.M_unit_g / (k.Lcm * k.Lcm * k.Lcm);
    k.ne_scale = rho0 / (kMP + kME);                                     // Eq. 46
    k.B0 = kC * std::sqrt(4.0 * kPI * rho0);
    k.thetae_scale = (kMP / kME) * (p.gamma_ad - 1.0) / (1.0 + p.tp_over_te);
    k.thetae_num = (kMP / kME) * (p.gamma_ad - 1.0); k.gm1 = p.gamma_ad - 1.0; k.te_model = p.te_model;
    for (int i = 0; i < 16; ++i) k.model[i] = p.model[i];
    k.disk_r_in = p.model[0] > 0.0 ? p.model[0] : r_isco(p.a);
    if (p.n1 > 0) {
        const double d1 = (p.x1_max - p.x1_min) / p.n1;
        k.x1_first = p.x1_min + 0.5 * d1; k.inv_d1 = 1.0 / d1;
    }
    // pre-rejection range of the plasma sampler (KP::samp_r_lo/hi): a superset of where the exact tests can succeed
    k.samp_r_lo = 0.0; k.samp_r_hi = std::numeric_limits<double>::infinity();
    if ((p.plasma_model == M_GRID2D || p.plasma_model == M_GRID3DT) && p.n1 > 0) {
        const double d1 = (p.x1_max - p.x1_min) / p.n1;
        k.samp_r_lo = (p.mks_r0 + std::exp(k.x1_first)) * (1.0 - 1e-9);
        k.samp_r_hi = (p.mks_r0 + std::exp(k.x1_first + (p.n1 - 1) * d1)) * (1.0 + 1e-9);
    } else if (p.plasma_model == M_TORUS) {
        k.samp_r_lo = std::max(0.0, (p.model[1] - std::fabs(p.model[2])) * (1.0 - 1e-9));
        k.samp_r_hi = (p.model[1] + std::fabs(p.model[2])) * (1.0 + 1e-9);
    }
    k.r0_nz = p.mks_r0 != 0.0 ? 1 : 0;
    k.t0 = p.t0; k.inv_dt = p.dt_snap > 0.0 ? 1.0 / p.dt_snap : 0.0;
    k.grid = c->d_grid; k.freq = c->d_freq;
    k.nx = p.nx; k.ny = p.ny; k.integrator = p.integrator; k.step_policy = p.step_policy; k.max_steps = p.max_steps; k.n_freq = p.n_freq;
    k.k2_mode = p.k2_mode; k.n1 = p.n1; k.n2 = p.n2; k.n3 = p.n3; k.nt = p.nt;
    k.slow_light = p.slow_light; k.snapshot = p.snapshot;
}

// float copies of the kernel parameters (precision = 1); every value is computed in double and rounded once
static void build_kpf(raptor_ctx* c) {
    const KP& k = c->kp;
    KPf& f = c->kpf;
    std::memset(&f, 0, sizeof(f));
    f.a = (float)k.a; f.a2 = (float)k.a2; f.twoa = (float)k.twoa; f.m = (float)k.m; f.twom = (float)k.twom; f.omh = (float)k.omh; f.r0 = (float)k.r0;
    f.r_cam = (float)k.r_cam; f.sin_i = (float)k.sin_i; f.cos_i = (float)k.cos_i; f.sq1mc2 = (float)k.sq1mc2;
    f.x1_cam = (float)k.x1_cam; f.x2_cam = (float)k.x2_cam; f.dth_cam = (float)k.dth_cam; f.t_cam = (float)k.t_cam; f.fov = (float)k.fov;
    f.eps = (float)k.eps; f.delta = (float)k.delta; f.r_in = (float)k.r_in; f.r_out = (float)k.r_out; f.tau_cutoff = (float)k.tau_cutoff;
    f.Lcm = (float)k.Lcm; f.ne_scale = (float)k.ne_scale; f.B0 = (float)k.B0; f.thetae_scale = (float)k.thetae_scale;
    f.x1_first = (float)k.x1_first; f.inv_d1 = (float)k.inv_d1; f.nu_obs = (float)c->nu0;
    f.grid = c->d_grid_f32;
    f.nx = k.nx; f.ny = k.ny; f.max_steps = k.max_steps; f.n1 = k.n1; f.n2 = k.n2; f.use_tau_cutoff = k.use_tau_cutoff;
}

extern "C" int raptor_create(const raptor_params* p, raptor_ctx** out) {
    if (!out) return fail(nullptr, RAPTOR_EINVAL, "out is NULL");
    *out = nullptr;
    int rc = validate(p);
    if (rc) return rc;
    raptor_ctx* c = new (std::nothrow) raptor_ctx;
    if (!c) return fail(nullptr, RAPTOR_ENOMEM, "host allocation failed");
    c->p = *p;
#define CKC(call)                                                                            \
    do {                                                                                     \
        cudaError_t e_ = (call);                                                             \
        if (e_ != cudaSuccess) {                                                             \
            int code = fail(nullptr, e_ == cudaErrorMemoryAllocation ? RAPTOR_ENOMEM : RAPTOR_ECUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
            raptor_destroy(c);                                                               \
            return code;                                                                     \
        }                                                                                    \
    } while (0)
    CKC(cudaGetDevice(&c->device));
    CKC(cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, c->device));
    CKC(cudaStreamCreateWithFlags(&c->own_stream, cudaStreamNonBlocking));
    CKC(cudaEventCreateWithFlags(&c->ev_last, cudaEventDisableTiming));
    {
        // per-frequency constants of the transfer update: nu_k, nu_k^(1/6) (Eq. 43), c^2 / (2 h nu_k^3) (Eq. 45)
        double tab[3 * RAPTOR_MAX_FREQ];
        for (int k = 0; k < p->n_freq; ++k) {
            const double nu = p->freq_hz[k];
            if (k == 0) c->nu0 = nu;
            tab[k] = nu;
            tab[p->n_freq + k] = std::cbrt(std::sqrt(nu));
            tab[2 * p->n_freq + k] = (kC * kC) / (2.0 * kHPL * nu * nu * nu);
        }
        CKC(cudaMalloc(&c->d_freq, sizeof(double) * 3 * p->n_freq));
        CKC(cudaMemcpy(c->d_freq, tab, sizeof(double) * 3 * p->n_freq, cudaMemcpyHostToDevice));
    }
    CKC(cudaMalloc(&c->d_queue, sizeof(unsigned int)));
    {
        // launch order of the 8x4-pixel tiles: by the impact parameter of the tile centre, nearest first (ties: by index)
        const int ntx = (p->nx + 7) / 8, nty = (p->ny + 3) / 4;
        std::vector<std::pair<double, unsigned>> key((size_t)ntx * nty);
        for (int ty = 0; ty < nty; ++ty)
            for (int tx = 0; tx < ntx; ++tx) {
                const double al = ((tx * 8 + 4.0) / p->nx - 0.5) * p->fov_M, be = ((ty * 4 + 2.0) / p->ny - 0.5) * p->fov_M;
                key[(size_t)ty * ntx + tx] = {al * al + be * be, (unsigned)(ty * ntx + tx)};
            }
        std::sort(key.begin(), key.end());
        std::vector<unsigned> order(key.size());
        for (size_t i = 0; i < key.size(); ++i) order[i] = key[i].second;
        CKC(cudaMalloc(&c->d_order, sizeof(unsigned) * order.size()));
        CKC(cudaMalloc(&c->d_order_shard, sizeof(unsigned) * order.size()));
        CKC(cudaMemcpy(c->d_order, order.data(), sizeof(unsigned) * order.size(), cudaMemcpyHostToDevice));
        c->order_host.swap(order);
    }
    CKC(cudaMalloc(&c->d_counters, 3 * sizeof(unsigned long long)));
    CKC(cudaMemset(c->d_counters, 0, 3 * sizeof(unsigned long long)));
    const size_t npix = (size_t)p->nx * p->ny;
    CKC(cudaMalloc(&c->d_partial, sizeof(double) * p->n_freq * (size_t)flux_chunks(npix)));
    CKC(cudaMalloc(&c->d_scratch_flux, sizeof(double) * p->n_freq));
    if (p->plasma_model == RAPTOR_GRID2D || p->plasma_model == RAPTOR_GRID3DT) {
        c->grid_bytes = (size_t)p->grid_bytes;
        CKC(cudaMalloc(&c->d_grid, c->grid_bytes));
        CKC(cudaMemcpy(c->d_grid, p->grid_host, c->grid_bytes, cudaMemcpyHostToDevice));
        if (p->precision == 1) {
            const size_t n = c->grid_bytes / sizeof(double);
            CKC(cudaMalloc(&c->d_grid_f32, n * sizeof(float)));
            CKC(launch_grid_to_f32((const double*)c->d_grid, c->d_grid_f32, n, 0));
            CKC(cudaDeviceSynchronize());
        }
    }
#undef CKC
    c->p.freq_hz = nullptr;      // the context owns device copies only
    c->p.grid_host = nullptr;
    build_kp(c);
    if (p->precision == 1) build_kpf(c);
    *out = c;
    return RAPTOR_OK;
}

extern "C" int raptor_upload_grid(raptor_ctx* ctx, const void* grid_host, uint64_t grid_bytes, void* cuda_stream) {
    if (!ctx) return fail(nullptr, RAPTOR_EINVAL, "ctx is NULL");
    if (!ctx->d_grid) return fail(ctx, RAPTOR_EINVAL, "context has no grid");
    if (!grid_host || grid_bytes != ctx->grid_bytes) return fail(ctx, RAPTOR_EINVAL, "grid_bytes %llu != %zu", (unsigned long long)grid_bytes, ctx->grid_bytes);
    CK(ctx, cudaMemcpyAsync(ctx->d_grid, grid_host, ctx->grid_bytes, cudaMemcpyHostToDevice, (cudaStream_t)cuda_stream));
    if (ctx->d_grid_f32)
        CK(ctx, launch_grid_to_f32((const double*)ctx->d_grid, ctx->d_grid_f32, ctx->grid_bytes / sizeof(double), (cudaStream_t)cuda_stream));
    return mark(ctx, (cudaStream_t)cuda_stream);
}

// Ordering rule (include/raptor.h): the asynchronous calls of one context share its scene data, tile queue and
// scratch buffers, so the caller issues them on ONE stream (or orders its streams itself); every such call leaves
// an event behind, and raptor_render_host, which runs on the context's own stream, waits for it.
static int mark(raptor_ctx* ctx, cudaStream_t s) {
    CK(ctx, cudaEventRecord(ctx->ev_last, s));
    return RAPTOR_OK;
}

static int run_rays(raptor_ctx* ctx, RenderOut& O, cudaStream_t s) {
    O.queue = ctx->d_queue;
    O.order = O.alpha ? nullptr : ctx->d_order;
    if (O.order && ctx->shard_world > 1 && O.tile_stride == (unsigned)ctx->shard_world) {
        // a shard owns the tiles whose index is rank mod world; it launches them in the same nearest-first order
        O.order = ctx->d_order_shard; O.tile_offset = 0; O.tile_stride = 1;
    }
    O.counters = ctx->d_counters;
    if (O.frames <= 1) O.null_max = ctx->d_null_max;
    if (O.null_max) {
        // the monitor buffer was sized by the caller for one kind of call: refuse the call that would write past its end
        const uint64_t need = O.alpha ? (uint64_t)O.nrays : (uint64_t)ctx->p.nx * (uint64_t)ctx->p.ny;
        if (need > ctx->null_max_capacity)
            return fail(ctx, RAPTOR_EINVAL, "null monitor buffer holds %llu elements, this call writes %llu: unset it or set a larger one",
                        (unsigned long long)ctx->null_max_capacity, (unsigned long long)need);
    }
    if (O.tile_stride == 0) { O.tile_offset = 0; O.tile_stride = 1; }
    CK(ctx, cudaMemsetAsync(ctx->d_queue, 0, sizeof(unsigned int), s));
    if (ctx->p.precision == 1) {
        if (O.frames > 1 || O.null_max) return fail(ctx, RAPTOR_EUNSUPPORTED, "precision 1 (FP32): no light curves, no null monitor");
        ctx->kpf.t_cam = (float)ctx->kp.t_cam;
        CK(ctx, launch_render_f32(ctx->kpf, O, ctx->sm_count, s));
    } else {
        CK(ctx, launch_render(ctx->kp, ctx->p.plasma_model, O, ctx->sm_count, s));
    }
    return mark(ctx, s);
}

extern "C" int raptor_render(raptor_ctx* ctx, double* d_image, int32_t* d_status, int32_t* d_nsteps, void* cuda_stream) {
    if (!ctx) return fail(nullptr, RAPTOR_EINVAL, "ctx is NULL");
    if (!d_image) return fail(ctx, RAPTOR_EINVAL, "d_image is NULL");
    RenderOut O;
    std::memset(&O, 0, sizeof(O));
    const unsigned all_tiles = (unsigned)(((ctx->p.nx + 7) / 8) * ((ctx->p.ny + 3) / 4));
    // shard: rank r of w takes tiles r, r+w, r+2w, ... (interleaved so that shadow and torus spread evenly)
    O.tile_offset = (unsigned)ctx->shard_rank; O.tile_stride = (unsigned)ctx->shard_world;
    O.ntiles = all_tiles > O.tile_offset ? (all_tiles - O.tile_offset + O.tile_stride - 1) / O.tile_stride : 0;
    O.image = d_image; O.status = d_status; O.nsteps = d_nsteps;
    if (O.ntiles == 0) return RAPTOR_OK;
    return run_rays(ctx, O, (cudaStream_t)cuda_stream);
}

extern "C" int raptor_render_disk(raptor_ctx* ctx, double* d_image, double* d_redshift, int32_t* d_status, int32_t* d_nsteps,
                                  void* cuda_stream) {
    if (!ctx) return fail(nullptr, RAPTOR_EINVAL, "ctx is NULL");
    if (ctx->p.plasma_model != RAPTOR_DISK) return fail(ctx, RAPTOR_EINVAL, "raptor_render_disk needs plasma_model = RAPTOR_DISK");
    if (!d_image || !d_redshift) return fail(ctx, RAPTOR_EINVAL, "NULL buffer");
    RenderOut O;
    std::memset(&O, 0, sizeof(O));
    const unsigned all_tiles = (unsigned)(((ctx->p.nx + 7) / 8) * ((ctx->p.ny + 3) / 4));
    O.tile_offset = (unsigned)ctx->shard_rank; O.tile_stride = (unsigned)ctx->shard_world;
    O.ntiles = all_tiles > O.tile_offset ? (all_tiles - O.tile_offset + O.tile_stride - 1) / O.tile_stride : 0;
    O.image = d_image; O.tau = d_redshift; O.status = d_status; O.nsteps = d_nsteps;
    if (O.ntiles == 0) return RAPTOR_OK;
    return run_rays(ctx, O, (cudaStream_t)cuda_stream);
}

extern "C" int raptor_line_profile(raptor_ctx* ctx, const double* d_image, const double* d_redshift, int32_t nbins, double g_min,
                                   double g_max, double* d_hist, void* cuda_stream) {
    if (!ctx) return fail(nullptr, RAPTOR_EINVAL, "ctx is NULL");
    if (!d_image || !d_redshift || !d_hist) return fail(ctx, RAPTOR_EINVAL, "NULL buffer");
    if (nbins < 1 || nbins > 65535 || !(g_max > g_min)) return fail(ctx, RAPTOR_EINVAL, "need 1 <= nbins <= 65535 and g_max > g_min");
    const size_t npix = (size_t)ctx->p.nx * ctx->p.ny;
    if (ctx->profile_bins < nbins) {
        if (ctx->d_profile_partial) cudaFree(ctx->d_profile_partial);
        ctx->d_profile_partial = nullptr; ctx->profile_bins = 0;
        CK(ctx, cudaMalloc(&ctx->d_profile_partial, sizeof(double) * nbins * (size_t)flux_chunks(npix)));
        ctx->profile_bins = nbins;
    }
    const double area = (ctx->p.fov_M / ctx->p.nx) * (ctx->p.fov_M / ctx->p.ny);
    CK(ctx, launch_profile(d_image, d_redshift, npix, nbins, g_min, g_max, area, ctx->d_profile_partial, d_hist, (cudaStream_t)cuda_stream));
    return mark(ctx, (cudaStream_t)cuda_stream);
}

// ---- slow-light movies and light curves (Sect. 5) -----------------------------------------
extern "C" int raptor_set_camera_time(raptor_ctx* ctx, double t_cam) {
    if (!ctx) return fail(nullptr, RAPTOR_EINVAL, "ctx is NULL");
    if (!std::isfinite(t_cam)) return fail(ctx, RAPTOR_EINVAL, "t_cam must be finite");
    ctx->p.t_cam = t_cam; ctx->kp.t_cam = t_cam;
    return RAPTOR_OK;
}

extern "C" int raptor_set_window(raptor_ctx* ctx, int64_t first_snapshot) {
    if (!ctx) return fail(nullptr, RAPTOR_EINVAL, "ctx is NULL");
    if (ctx->p.plasma_model != RAPTOR_GRID3DT) return fail(ctx, RAPTOR_EINVAL, "raptor_set_window needs plasma_model = RAPTOR_GRID3DT");
    if (first_snapshot < 0 || first_snapshot > (1ll << 40)) return fail(ctx, RAPTOR_EINVAL, "first_snapshot out of range");
    ctx->window_lo = first_snapshot;
    ctx->kp.snap_lo = (double)first_snapshot;
    ctx->kp.snap_lo_mod = (int)(first_snapshot % ctx->p.nt);
    return RAPTOR_OK;
}

extern "C" int raptor_upload_snapshot(raptor_ctx* ctx, int64_t snapshot, const void* host, uint64_t bytes, void* cuda_stream) {
    if (!ctx) return fail(nullptr, RAPTOR_EINVAL, "ctx is NULL");
    if (ctx->p.plasma_model != RAPTOR_GRID3DT || !ctx->d_grid) return fail(ctx, RAPTOR_EINVAL, "raptor_upload_snapshot needs plasma_model = RAPTOR_GRID3DT");
    const size_t one = ctx->grid_bytes / (size_t)ctx->p.nt;
    if (!host || bytes != one) return fail(ctx, RAPTOR_EINVAL, "snapshot bytes %llu != n1*n2*n3*8*elem = %zu", (unsigned long long)bytes, one);
    if (snapshot < 0) return fail(ctx, RAPTOR_EINVAL, "snapshot index < 0");
    const size_t slot = (size_t)(snapshot % ctx->p.nt);
    CK(ctx, cudaMemcpyAsync((char*)ctx->d_grid + slot * one, host, one, cudaMemcpyHostToDevice, (cudaStream_t)cuda_stream));
    return mark(ctx, (cudaStream_t)cuda_stream);
}

// frames of a light curve rendered per launch: the image scratch is frames x n_freq x npix doubles
static const size_t kLightCurveScratchBytes = 256u << 20;

extern "C" int raptor_light_curve(raptor_ctx* ctx, int32_t n_frames, double t_cam0, double dt_frame, double* d_flux_jy, void* cuda_stream) {
    if (!ctx) return fail(nullptr, RAPTOR_EINVAL, "ctx is NULL");
    if (n_frames < 0 || (n_frames > 0 && !d_flux_jy)) return fail(ctx, RAPTOR_EINVAL, "n_frames < 0 or d_flux_jy NULL");
    if (!std::isfinite(t_cam0) || !std::isfinite(dt_frame)) return fail(ctx, RAPTOR_EINVAL, "t_cam0, dt_frame must be finite");
    if (ctx->shard_world != 1) return fail(ctx, RAPTOR_EUNSUPPORTED, "raptor_light_curve shards by frames, not by tiles: reset raptor_set_shard(0, 1)");
    if (n_frames == 0) return RAPTOR_OK;
    const raptor_params& p = ctx->p;
    const size_t npix = (size_t)p.nx * p.ny, per_frame = npix * p.n_freq;
    size_t batch = kLightCurveScratchBytes / (per_frame * sizeof(double));
    if (batch < 1) batch = 1;
    if (batch > (size_t)n_frames) batch = (size_t)n_frames;
    const unsigned tiles = (unsigned)(((p.nx + 7) / 8) * ((p.ny + 3) / 4));
    if ((unsigned long long)tiles * batch > 0x7fffffffull) batch = 0x7fffffffull / tiles;
    if (batch * p.n_freq > 65535) batch = 65535 / p.n_freq;                 // grid.y of the flux reduction
    // scratch for `batch` images and their flux partial sums
    if (ctx->scratch_pixels < batch * per_frame) {
        if (ctx->d_scratch_image) cudaFree(ctx->d_scratch_image);
        ctx->d_scratch_image = nullptr; ctx->scratch_pixels = 0;
        CK(ctx, cudaMalloc(&ctx->d_scratch_image, batch * per_frame * sizeof(double)));
        ctx->scratch_pixels = batch * per_frame;
    }
    const size_t planes = batch * p.n_freq;
    if (ctx->lc_planes < planes) {
        if (ctx->d_lc_partial) cudaFree(ctx->d_lc_partial);
        ctx->d_lc_partial = nullptr; ctx->lc_planes = 0;
        CK(ctx, cudaMalloc(&ctx->d_lc_partial, sizeof(double) * planes * (size_t)flux_chunks(npix)));
        ctx->lc_planes = planes;
    }
    const double L = ctx->kp.Lcm;
    const double scale = 1e23 * (p.fov_M / p.nx) * (p.fov_M / p.ny) * L * L / (p.D_src_cm * p.D_src_cm);
    cudaStream_t s = (cudaStream_t)cuda_stream;
    for (size_t f0 = 0; f0 < (size_t)n_frames; f0 += batch) {
        const size_t nb = std::min(batch, (size_t)n_frames - f0);
        RenderOut O;
        std::memset(&O, 0, sizeof(O));
        O.frames = (unsigned)nb; O.tiles_per_frame = tiles; O.ntiles = tiles * (unsigned)nb;
        O.t_cam0 = t_cam0 + (double)f0 * dt_frame; O.dt_frame = dt_frame;
        O.image = ctx->d_scratch_image;
        if (nb == 1) { O.frames = 1; }       // single frame: the ordinary path with its own camera time
        const double keep = ctx->kp.t_cam;
        double* keep_mon = ctx->d_null_max;          // the monitor buffer is one image: not for a batch of frames
        ctx->d_null_max = nullptr;
        if (nb == 1) ctx->kp.t_cam = O.t_cam0;
        int rc = run_rays(ctx, O, s);
        ctx->kp.t_cam = keep;
        ctx->d_null_max = keep_mon;
        if (rc) return rc;
        // the batch is [nb][n_freq][npix] = nb * n_freq planes: one deterministic reduction for all of them
        CK(ctx, launch_flux(ctx->d_scratch_image, npix, (int)(nb * p.n_freq), scale, ctx->d_lc_partial,
                            d_flux_jy + f0 * p.n_freq, s));
    }
    return mark(ctx, s);
}

extern "C" int raptor_calibrate_delay(int32_t n_fast, const double* t_fast, const double* F_fast, int32_t n_slow, const double* t_slow,
                                      const double* F_slow, double max_shift, int32_t n_grid, double* delay, double* rms) {
    if (n_fast < 1 || n_slow < 2 || !t_fast || !F_fast || !t_slow || !F_slow || !delay || !rms)
        return fail(nullptr, RAPTOR_EINVAL, "raptor_calibrate_delay: need n_fast >= 1, n_slow >= 2 and non-NULL arrays");
    if (!(max_shift >= 0.0) || n_grid < 1) return fail(nullptr, RAPTOR_EINVAL, "raptor_calibrate_delay: max_shift >= 0, n_grid >= 1");
    double mf = 0.0, ms = 0.0;
    for (int i = 0; i < n_fast; ++i) mf += F_fast[i];
    for (int i = 0; i < n_slow; ++i) ms += F_slow[i];
    mf /= n_fast; ms /= n_slow;
    if (!(mf != 0.0) || !(ms != 0.0) || !std::isfinite(mf) || !std::isfinite(ms))
        return fail(nullptr, RAPTOR_EINVAL, "raptor_calibrate_delay: the mean of a light curve is zero or not finite (curves are normalised by their means)");
    for (int i = 1; i < n_slow; ++i)
        if (!(t_slow[i] > t_slow[i - 1])) return fail(nullptr, RAPTOR_EINVAL, "raptor_calibrate_delay: t_slow must be strictly ascending (t_slow[%d] <= t_slow[%d])", i, i - 1);
    const int need = std::max(4, n_fast / 2);
    double best_d = 0.0, best = INFINITY;
    for (int k = 0; k < n_grid; ++k) {
        const double d = n_grid > 1 ? -max_shift + 2.0 * max_shift * k / (n_grid - 1) : 0.0;
        double acc = 0.0;
        int used = 0, j = 0;
        for (int i = 0; i < n_fast; ++i) {
            const double ts = t_fast[i] + d;
            if (ts < t_slow[0] || ts > t_slow[n_slow - 1]) continue;
            while (j + 2 < n_slow && t_slow[j + 1] < ts) ++j;          // t_fast ascending is the common case ...
            while (j > 0 && t_slow[j] > ts) --j;                       // ... but not required
            const double w = (ts - t_slow[j]) / (t_slow[j + 1] - t_slow[j]);
            const double res = (F_slow[j] + w * (F_slow[j + 1] - F_slow[j])) / ms - F_fast[i] / mf;
            acc += res * res;
            ++used;
        }
        if (used < need) continue;
        const double r = std::sqrt(acc / used);
        if (r < best) { best = r; best_d = d; }
    }
    *delay = best_d; *rms = best;
    return RAPTOR_OK;
}

extern "C" int raptor_set_shard(raptor_ctx* ctx, int32_t rank, int32_t world) {
    if (!ctx) return fail(nullptr, RAPTOR_EINVAL, "ctx is NULL");
    if (world < 1 || rank < 0 || rank >= world) return fail(ctx, RAPTOR_EINVAL, "shard: need 0 <= rank < world");
    if (world > 1) {
        std::vector<unsigned> mine;
        for (unsigned t : ctx->order_host)
            if (t % (unsigned)world == (unsigned)rank) mine.push_back(t);
        CK(ctx, cudaDeviceSynchronize());            // a launch in flight may still read the previous table
        if (!mine.empty()) CK(ctx, cudaMemcpy(ctx->d_order_shard, mine.data(), sizeof(unsigned) * mine.size(), cudaMemcpyHostToDevice));
    }
    // only now: a failed upload above leaves the previous (rank, world) together with its own table
    ctx->shard_rank = rank; ctx->shard_world = world;
    return RAPTOR_OK;
}

extern "C" int raptor_set_null_monitor(raptor_ctx* ctx, double* d_null_max_or_null, uint64_t capacity) {
    if (!ctx) return fail(nullptr, RAPTOR_EINVAL, "ctx is NULL");
    if (d_null_max_or_null && capacity == 0) return fail(ctx, RAPTOR_EINVAL, "null monitor: capacity must be >= 1 element");
    ctx->d_null_max = d_null_max_or_null;
    ctx->null_max_capacity = d_null_max_or_null ? capacity : 0;
    return RAPTOR_OK;
}

extern "C" int raptor_flux(raptor_ctx* ctx, const double* d_image, double* d_flux_jy, void* cuda_stream) {
    if (!ctx) return fail(nullptr, RAPTOR_EINVAL, "ctx is NULL");
    if (!d_image || !d_flux_jy) return fail(ctx, RAPTOR_EINVAL, "NULL buffer");
    const raptor_params& p = ctx->p;
    const double L = ctx->kp.Lcm;
    const double scale = 1e23 * (p.fov_M / p.nx) * (p.fov_M / p.ny) * L * L / (p.D_src_cm * p.D_src_cm);
    CK(ctx, launch_flux(d_image, (size_t)p.nx * p.ny, p.n_freq, scale, ctx->d_partial, d_flux_jy, (cudaStream_t)cuda_stream));
    return mark(ctx, (cudaStream_t)cuda_stream);
}

// The reduction of raptor_flux for callers that cannot allocate (include/raptor.h): no context, partial sums in the
// library's own __device__ array (raptor_flux_static.cu).  Nothing here or below it calls cudaMalloc / cudaFree.
static_assert(RAPTOR_FLUX_STATIC_MAX_PARTIALS == kFluxStaticSlots, "header limit and array size must agree");
extern "C" int raptor_flux_static(const double* d_image, uint64_t npix, int32_t n_planes, double scale, double* d_flux,
                                  void* cuda_stream) {
    if (!d_image || !d_flux) return fail(nullptr, RAPTOR_EINVAL, "raptor_flux_static: NULL buffer");
    if (npix == 0 || n_planes < 1) return fail(nullptr, RAPTOR_EINVAL, "raptor_flux_static: need npix >= 1 and n_planes >= 1");
    const uint64_t chunks = (npix + 16383) / 16384;
    if (chunks > (uint64_t)kFluxStaticSlots || chunks * (uint64_t)n_planes > (uint64_t)kFluxStaticSlots)
        return fail(nullptr, RAPTOR_EINVAL,
                    "raptor_flux_static: %d planes x %llu chunks of 16384 pixels = %llu partial sums, the built-in scratch holds %d "
                    "(use raptor_flux, which allocates, for larger images)",
                    n_planes, (unsigned long long)chunks, (unsigned long long)(chunks * (uint64_t)n_planes), kFluxStaticSlots);
    CK(nullptr, launch_flux_static(d_image, (size_t)npix, n_planes, scale, d_flux, (cudaStream_t)cuda_stream));
    return RAPTOR_OK;
}

static int ensure_scratch(raptor_ctx* ctx) {
    const size_t need = (size_t)ctx->p.nx * ctx->p.ny * ctx->p.n_freq;
    if (ctx->scratch_pixels < need) {
        if (ctx->d_scratch_image) cudaFree(ctx->d_scratch_image);
        ctx->d_scratch_image = nullptr; ctx->scratch_pixels = 0;
        CK(ctx, cudaMalloc(&ctx->d_scratch_image, need * sizeof(double)));
        ctx->scratch_pixels = need;
    }
    return RAPTOR_OK;
}

extern "C" int raptor_spectrum(raptor_ctx* ctx, double* d_flux_jy, double* d_image_or_null, void* cuda_stream) {
    if (!ctx) return fail(nullptr, RAPTOR_EINVAL, "ctx is NULL");
    if (!d_flux_jy) return fail(ctx, RAPTOR_EINVAL, "d_flux_jy is NULL");
    double* img = d_image_or_null;
    if (!img) {
        int rc = ensure_scratch(ctx);
        if (rc) return rc;
        img = ctx->d_scratch_image;
        // a shard writes only its own tiles: the rest of the scratch image must read as zero (raptor.h, raptor_set_shard)
        if (ctx->shard_world > 1)
            CK(ctx, cudaMemsetAsync(img, 0, (size_t)ctx->p.nx * ctx->p.ny * ctx->p.n_freq * sizeof(double), (cudaStream_t)cuda_stream));
    }
    int rc = raptor_render(ctx, img, nullptr, nullptr, cuda_stream);
    if (rc) return rc;
    return raptor_flux(ctx, img, d_flux_jy, cuda_stream);
}

extern "C" int raptor_render_host(raptor_ctx* ctx, double* h_image, int32_t* h_status, int32_t* h_nsteps, double* h_flux_jy) {
    if (!ctx) return fail(nullptr, RAPTOR_EINVAL, "ctx is NULL");
    if (!h_image) return fail(ctx, RAPTOR_EINVAL, "h_image is NULL");
    int rc = ensure_scratch(ctx);
    if (rc) return rc;
    const size_t npix = (size_t)ctx->p.nx * ctx->p.ny;
    cudaStream_t s = ctx->own_stream;
    CK(ctx, cudaStreamWaitEvent(s, ctx->ev_last, 0));          // after every earlier call on this context (uploads, renders)
    int32_t *d_status = nullptr, *d_nsteps = nullptr;
    // every CUDA call of the body goes through `step`, so that the two temporaries are released on every way out
    cudaError_t ce = cudaSuccess;
    const char* what = "";
#define STEP(call) do { if (!rc && ce == cudaSuccess) { ce = (call); if (ce != cudaSuccess) what = #call; } } while (0)
    if (h_status) STEP(cudaMallocAsync(&d_status, npix * sizeof(int32_t), s));
    if (h_nsteps) STEP(cudaMallocAsync(&d_nsteps, npix * sizeof(int32_t), s));
    if (ctx->shard_world > 1) {                                // pixels of other ranks' tiles read as zero
        STEP(cudaMemsetAsync(ctx->d_scratch_image, 0, npix * ctx->p.n_freq * sizeof(double), s));
        if (d_status) STEP(cudaMemsetAsync(d_status, 0, npix * sizeof(int32_t), s));
        if (d_nsteps) STEP(cudaMemsetAsync(d_nsteps, 0, npix * sizeof(int32_t), s));
    }
    if (ce == cudaSuccess) rc = raptor_render(ctx, ctx->d_scratch_image, d_status, d_nsteps, s);
    if (ce == cudaSuccess && !rc && h_flux_jy) rc = raptor_flux(ctx, ctx->d_scratch_image, ctx->d_scratch_flux, s);
    STEP(cudaMemcpyAsync(h_image, ctx->d_scratch_image, npix * ctx->p.n_freq * sizeof(double), cudaMemcpyDeviceToHost, s));
    if (h_status) STEP(cudaMemcpyAsync(h_status, d_status, npix * sizeof(int32_t), cudaMemcpyDeviceToHost, s));
    if (h_nsteps) STEP(cudaMemcpyAsync(h_nsteps, d_nsteps, npix * sizeof(int32_t), cudaMemcpyDeviceToHost, s));
    if (h_flux_jy) STEP(cudaMemcpyAsync(h_flux_jy, ctx->d_scratch_flux, ctx->p.n_freq * sizeof(double), cudaMemcpyDeviceToHost, s));
#undef STEP
    if (d_status) cudaFreeAsync(d_status, s);
    if (d_nsteps) cudaFreeAsync(d_nsteps, s);
    const cudaError_t se = cudaStreamSynchronize(s);
    if (ce != cudaSuccess)
        return fail(ctx, ce == cudaErrorMemoryAllocation ? RAPTOR_ENOMEM : RAPTOR_ECUDA, "%s: %s", what, cudaGetErrorString(ce));
    if (rc) return rc;
    CK(ctx, se);
    return RAPTOR_OK;
}

extern "C" int raptor_trace(raptor_ctx* ctx, int32_t n, const double* d_alpha, const double* d_beta, double* d_I, double* d_tau,
                            double* d_XK, int32_t* d_status, int32_t* d_nsteps, void* cuda_stream) {
    if (!ctx) return fail(nullptr, RAPTOR_EINVAL, "ctx is NULL");
    if (n < 0 || (n > 0 && (!d_alpha || !d_beta))) return fail(ctx, RAPTOR_EINVAL, "n < 0 or NULL alpha/beta");
    if (n == 0) return RAPTOR_OK;
    RenderOut O;
    std::memset(&O, 0, sizeof(O));
    O.ntiles = (unsigned)((n + 31) / 32);
    O.alpha = d_alpha; O.beta = d_beta; O.nrays = n;
    O.image = d_I; O.tau = d_tau; O.XK = d_XK; O.status = d_status; O.nsteps = d_nsteps;
    return run_rays(ctx, O, (cudaStream_t)cuda_stream);
}

extern "C" int raptor_eval_rhs(raptor_ctx* ctx, int32_t n, const double* d_XK, double* d_f, void* cuda_stream) {
    if (!ctx) return fail(nullptr, RAPTOR_EINVAL, "ctx is NULL");
    if (n < 0 || (n > 0 && (!d_XK || !d_f))) return fail(ctx, RAPTOR_EINVAL, "n < 0 or NULL buffer");
    if (n == 0) return RAPTOR_OK;
    CK(ctx, launch_eval_rhs(ctx->kp, n, d_XK, d_f, (cudaStream_t)cuda_stream));
    return RAPTOR_OK;
}

extern "C" int raptor_null_norm(raptor_ctx* ctx, int32_t n, const double* d_XK, double* d_out, double* d_ELQ_or_null, void* cuda_stream) {
    if (!ctx) return fail(nullptr, RAPTOR_EINVAL, "ctx is NULL");
    if (n < 0 || (n > 0 && (!d_XK || !d_out))) return fail(ctx, RAPTOR_EINVAL, "n < 0 or NULL buffer");
    if (n == 0) return RAPTOR_OK;
    CK(ctx, launch_null_norm(ctx->kp, n, d_XK, d_out, d_ELQ_or_null, (cudaStream_t)cuda_stream));
    return RAPTOR_OK;
}

extern "C" int raptor_get_counters(raptor_ctx* ctx, uint64_t* total_steps, uint64_t* sampled_steps, uint64_t* rays) {
    if (!ctx) return fail(nullptr, RAPTOR_EINVAL, "ctx is NULL");
    unsigned long long h[3];
    CK(ctx, cudaEventSynchronize(ctx->ev_last));     // the last call made on this context; other streams of the process keep running
    CK(ctx, cudaMemcpyAsync(h, ctx->d_counters, sizeof(h), cudaMemcpyDeviceToHost, ctx->own_stream));
    CK(ctx, cudaStreamSynchronize(ctx->own_stream));
    if (total_steps) *total_steps = h[0];
    if (sampled_steps) *sampled_steps = h[1];
    if (rays) *rays = h[2];
    return RAPTOR_OK;
}

extern "C" int raptor_fp64_peak(int32_t iters, double* tflops, double* ms) {
    if (iters < 1 || !tflops) return fail(nullptr, RAPTOR_EINVAL, "iters < 1 or tflops NULL");
    int dev = 0, sms = 0;
    CK(nullptr, cudaGetDevice(&dev));
    CK(nullptr, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double* d_out = nullptr;
    CK(nullptr, cudaMalloc(&d_out, sizeof(double)));
    cudaEvent_t e0, e1;
    CK(nullptr, cudaEventCreate(&e0));
    CK(nullptr, cudaEventCreate(&e1));
    const int blocks = sms * 8;
    float best = 1e30f;
    cudaError_t err = cudaSuccess;
    for (int rep = 0; rep < 4 && err == cudaSuccess; ++rep) {       // rep 0 warms up
        cudaEventRecord(e0, 0);
        err = launch_fp64_peak(iters, blocks, d_out, 0);
        cudaEventRecord(e1, 0);
        if (err == cudaSuccess) err = cudaEventSynchronize(e1);
        float t = 0.f;
        cudaEventElapsedTime(&t, e0, e1);
        if (rep > 0 && t < best) best = t;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d_out);
    if (err != cudaSuccess) return fail(nullptr, RAPTOR_ECUDA, "fp64 probe: %s", cudaGetErrorString(err));
    const double flops = 2.0 * 8.0 * (double)iters * 256.0 * (double)blocks;
    *tflops = flops / (best * 1e-3) * 1e-12;
    if (ms) *ms = best;
    return RAPTOR_OK;
}

extern "C" int raptor_fp32_peak(int32_t iters, double* tflops, double* ms) {
    if (iters < 1 || !tflops) return fail(nullptr, RAPTOR_EINVAL, "iters < 1 or tflops NULL");
    int dev = 0, sms = 0;
    CK(nullptr, cudaGetDevice(&dev));
    CK(nullptr, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    float* d_out = nullptr;
    CK(nullptr, cudaMalloc(&d_out, sizeof(float)));
    cudaEvent_t e0, e1;
    CK(nullptr, cudaEventCreate(&e0));
    CK(nullptr, cudaEventCreate(&e1));
    const int blocks = sms * 8;
    float best = 1e30f;
    cudaError_t err = cudaSuccess;
    for (int rep = 0; rep < 4 && err == cudaSuccess; ++rep) {       // rep 0 warms up
        cudaEventRecord(e0, 0);
        err = launch_fp32_peak(iters, blocks, d_out, 0);
        cudaEventRecord(e1, 0);
        if (err == cudaSuccess) err = cudaEventSynchronize(e1);
        float t = 0.f;
        cudaEventElapsedTime(&t, e0, e1);
        if (rep > 0 && t < best) best = t;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d_out);
    if (err != cudaSuccess) return fail(nullptr, RAPTOR_ECUDA, "fp32 probe: %s", cudaGetErrorString(err));
    const double flops = 2.0 * 16.0 * (double)iters * 256.0 * (double)blocks;
    *tflops = flops / (best * 1e-3) * 1e-12;
    if (ms) *ms = best;
    return RAPTOR_OK;
}

extern "C" int raptor_fp64_probe(int32_t form, int32_t iters, double* warp_inst_per_sec, double* sm_clock_hz) {
    if (form < 0 || form > 4 || iters < 1 || !warp_inst_per_sec) return fail(nullptr, RAPTOR_EINVAL, "form 0..4, iters >= 1, output not NULL");
    int dev = 0, sms = 0, khz = 0;
    CK(nullptr, cudaGetDevice(&dev));
    CK(nullptr, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    CK(nullptr, cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev));
    double* d_out = nullptr;
    CK(nullptr, cudaMalloc(&d_out, sizeof(double)));
    cudaEvent_t e0, e1;
    CK(nullptr, cudaEventCreate(&e0));
    CK(nullptr, cudaEventCreate(&e1));
    const int blocks = sms * 4;                                     // 4 x 256 threads: 8 warps per sub-partition
    float best = 1e30f;
    cudaError_t err = cudaSuccess;
    for (int rep = 0; rep < 4 && err == cudaSuccess; ++rep) {       // rep 0 warms up
        cudaEventRecord(e0, 0);
        err = launch_fp64_form(form, iters, blocks, d_out, 0);
        cudaEventRecord(e1, 0);
        if (err == cudaSuccess) err = cudaEventSynchronize(e1);
        float t = 0.f;
        cudaEventElapsedTime(&t, e0, e1);
        if (rep > 0 && t < best) best = t;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d_out);
    if (err != cudaSuccess) return fail(nullptr, RAPTOR_ECUDA, "fp64 form probe: %s", cudaGetErrorString(err));
    *warp_inst_per_sec = 8.0 * (double)iters * 8.0 * (double)blocks / (best * 1e-3);     // 8 chains x 8 warps per CTA
    if (sm_clock_hz) *sm_clock_hz = 1e3 * (double)khz;
    return RAPTOR_OK;
}

extern "C" int raptor_destroy(raptor_ctx* ctx) {
    if (!ctx) return RAPTOR_OK;
    cudaFree(ctx->d_grid); cudaFree(ctx->d_grid_f32); cudaFree(ctx->d_freq); cudaFree(ctx->d_queue); cudaFree(ctx->d_order); cudaFree(ctx->d_order_shard); cudaFree(ctx->d_counters);
    cudaFree(ctx->d_partial); cudaFree(ctx->d_profile_partial); cudaFree(ctx->d_lc_partial); cudaFree(ctx->d_scratch_image); cudaFree(ctx->d_scratch_flux);
    if (ctx->own_stream) cudaStreamDestroy(ctx->own_stream);
    if (ctx->ev_last) cudaEventDestroy(ctx->ev_last);
    delete ctx;
    return RAPTOR_OK;
}

extern "C" const char* raptor_last_error(const raptor_ctx* ctx) { return ctx ? ctx->err : g_err; }
