/* raptor_oracle.c -- CPU ORACLE for the RAPTOR hot path.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, real-precision implementation of what the path computes, written from
 * the paper (/root/reference/PAPER.md = Bronzwaer et al., RAPTOR I, arXiv:1801.10452) step by
 * step in the paper's order and notation.  It shares no code, header, table or helper with
 * the CUDA path under paper_1801_10452_b200/csrc/; neither includes nor links the other.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load this file's shared library.
 *
 * The method is an iteration (fixed-order RK4 stepping + a quadrature along the ray), so the
 * oracle is the algorithm itself, with no blocking, fusion or reordering:
 *   - metric of the chart we integrate in (modified Kerr-Schild, A.10-A.13 PAPER.md:599-605),
 *     its analytic first derivatives, and ALL connection coefficients by Eq. 2;
 *   - f^a = -Gamma^a_bc k^b k^c (Eq. 6) by a triple loop;
 *   - RK4 exactly as printed, Eq. 7-16;
 *   - camera, Eq. 25-29 built in Boyer-Lindquist and carried to KS by the
 *     matrix A.5 and to MKS by A.8-A.9;
 *   - backward transfer, Eq. 36-37 with the constant-coefficient step of
 *     Eq. 35, thermal synchrotron Eq. 42-44, Kirchhoff +
 *     Planck Eq. 45, unit scaling Eq. 46.
 * Readings of points the paper leaves open are the [A#] items of SURVEY.md 8(c), repeated in
 * DESIGN.md; each is tagged where it is used.
 *
 * Pins (tests/test_oracle_*.py, all run without a GPU): metric identities, Gamma against
 * finite differences of the metric, conserved E/L/Q, 4th-order convergence, sqrt(27) shadow,
 * Bardeen critical curve incl. Table 1 of the paper, flat-space straight lines, redshift
 * closed forms, uniform-slab closed forms (I = jL, I = S(1-exp(-tau)), I -> B_nu), the
 * emissivity fit against direct quadrature over the Maxwell-Juettner distribution, the
 * cyclotron frequency the paper prints, multilinear-interpolation exactness,
 * both step rules (Eq. 21-24 and the configs[0] clamp with and without the polar guard), the
 * optical-depth cut-off exit, pixel centres and the [k][iy][ix] image layout by hand computation.
 * The fluid-frame block (nu_hat, pitch angle, field seeds, sampling guard) is pinned THROUGH orc_transfer /
 * orc_trace_ray against aberration, Doppler and gravitational-redshift closed forms (tests/test_oracle_fluid_frame.py).
 * Parity unpinned (definitions, not derivable -- see DESIGN.md): the VALUES of the step-rule
 * constants of BASELINE.json configs[0] and of eps_polar, the end-point sampling of the quadrature
 * [A8], the amplitudes of the synthetic plasma models, and Table 3 / Fig. 7-13 of the paper
 * (datasets absent).  Every function of this file has a pin.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (oracle/oracle.py does it).
 */
#include <math.h>
#include <tgmath.h>   /* type-generic sin, exp, ... : the float functions when real = float */
#undef I              /* <complex.h>'s imaginary unit, pulled in by <tgmath.h>: I is the intensity here */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ---- CGS constants [A19]; the oracle's own copy --------------------------------------- */
#define ORC_C      2.99792458e10
#define ORC_G      6.6743e-8
#define ORC_E      4.80320471e-10
#define ORC_ME     9.1093837e-28
#define ORC_MP     1.67262192e-24
#define ORC_KB     1.380649e-16
#define ORC_HPL    6.62607015e-27
#define ORC_PI     3.14159265358979323846

enum { ORC_VACUUM = 0, ORC_SPHERE = 1, ORC_TORUS = 2, ORC_GRID2D = 3, ORC_GRID3DT = 4, ORC_SLAB = 5, ORC_DISK = 6 };
enum { ORC_RUNNING = 0, ORC_CAPTURED = 1, ORC_ESCAPED = 2, ORC_MAXSTEPS = 3, ORC_THICK = 4, ORC_NONFINITE = 5 };

/* Working precision.  Default: double (the contract, BASELINE.json: "FP64").  The same source compiled with
 * -DORC_REAL=float -fsingle-precision-constant is the single-precision oracle of the paper's own performance
 * configuration (Table B.1 "Single precision: yes") -- liboracle_f32.so, 8(f) f1; <tgmath.h> then
 * selects the float math functions.  Nothing else differs between the two builds. */
#ifndef ORC_REAL
#define ORC_REAL double
#endif
typedef ORC_REAL real;

typedef struct {
    real a, mks_h, mks_r0, mass;
    real r_cam, incl_deg, fov_M, t_cam;
    double M_bh_g, D_src_cm, M_unit_g;      /* [g], [cm], [g]: beyond the range of a float, always double */
    real step_c, step_min, step_max, eps, delta, eps_polar;
    real r_stop_in_factor, r_stop_out_factor, tau_cutoff;
    real model[16];
    real tp_over_te, gamma_ad;
    real x1_min, x1_max, t0, dt_snap;
    const real *freq_hz;
    const void *grid;
    int32_t nx, ny, integrator, step_policy, max_steps, n_freq, plasma_model, k2_mode;
    int32_t n1, n2, n3, nt, grid_dtype, slow_light, snapshot, te_model;
} orc_params;

/* ======================================================================================= */
/* Chart: MKS(h, r0).  x^A_KS = (t, r0 + exp x1, theta(x2), phi)          A.10-A.11          */
/* ======================================================================================= */
void orc_mks_theta(real h, real x2, real *th, real *dth, real *d2th)
{
    *th = ORC_PI * x2 + 0.5 * (1.0 - h) * sin(2.0 * ORC_PI * x2);              /* A.11 */
    *dth = ORC_PI * (1.0 + (1.0 - h) * cos(2.0 * ORC_PI * x2));                /* A.13 */
    *d2th = -2.0 * ORC_PI * ORC_PI * (1.0 - h) * sin(2.0 * ORC_PI * x2);
}

/* Newton-Raphson inverse of A.11, Eq. A.14-A.16: small trial value,
 * reset to 0.05 whenever the iterate leaves [0,1] or f' -> 0.  Returns iterations used. */
int orc_x2_of_theta(real h, real theta, real tol, real *x2_out)
{
    /* As printed the iteration cycles (overshoot past 1 -> reset -> overshoot ...) for theta near pi
     * when h < 1, because theta(x2) is steep at x2 = 0 and shallow at x2 = 1/2.  theta(1 - x2) =
     * pi - theta(x2), so the lower half theta <= pi/2, where theta(x2) is concave and Newton from a
     * small trial value converges monotonically, is solved and mirrored [A22 in DESIGN.md]. */
    int mirror = theta > 0.5 * ORC_PI;
    real target = mirror ? ORC_PI - theta : theta;
    real x = 0.01;
    int it;
    for (it = 0; it < 200; ++it) {
        real th, dth, d2;
        orc_mks_theta(h, x, &th, &dth, &d2);
        if (fabs(dth) < 1e-12) { x = 0.05; continue; }
        real xn = x - (th - target) / dth;                                   /* A.14 */
        if (xn < 0.0 || xn > 1.0) xn = 0.05;
        if (fabs(xn - x) < tol) { x = xn; ++it; break; }
        x = xn;
    }
    *x2_out = mirror ? 1.0 - x : x;
    return it;
}

/* Ingoing Kerr-Schild metric in spherical coordinates (t~, r, theta, phi~), the chart reached
 * from Boyer-Lindquist by A.1-A.5 [A1].  m = mass parameter (1; 0 = flat). */
void orc_metric_ks(real a, real m, real r, real th, real g[4][4])
{
    real s = sin(th), c = cos(th), s2 = s * s;
    real Sig = r * r + a * a * c * c;
    real f = 2.0 * m * r / Sig;
    memset(g, 0, 16 * sizeof(real));
    g[0][0] = -(1.0 - f);
    g[0][1] = g[1][0] = f;
    g[0][3] = g[3][0] = -f * a * s2;
    g[1][1] = 1.0 + f;
    g[1][3] = g[3][1] = -a * s2 * (1.0 + f);
    g[2][2] = Sig;
    g[3][3] = s2 * (Sig + a * a * s2 * (1.0 + f));
}

void orc_metric_ks_inv(real a, real m, real r, real th, real gi[4][4])
{
    real s = sin(th), c = cos(th), s2 = s * s;
    real Sig = r * r + a * a * c * c;
    real Del = r * r - 2.0 * m * r + a * a;
    real f = 2.0 * m * r / Sig;
    memset(gi, 0, 16 * sizeof(real));
    gi[0][0] = -(1.0 + f);
    gi[0][1] = gi[1][0] = f;
    gi[1][1] = Del / Sig;
    gi[1][3] = gi[3][1] = a / Sig;
    gi[2][2] = 1.0 / Sig;
    gi[3][3] = 1.0 / (Sig * s2);
}

/* d/dr and d/dtheta of the KS metric (analytic). */
static void metric_ks_deriv(real a, real m, real r, real th, real dr[4][4], real dt[4][4])
{
    real s = sin(th), c = cos(th), s2 = s * s;
    real Sig = r * r + a * a * c * c;
    real f = 2.0 * m * r / Sig;
    real Sig_r = 2.0 * r, Sig_t = -2.0 * a * a * s * c;
    real f_r = 2.0 * m / Sig - 2.0 * m * r * Sig_r / (Sig * Sig);
    real f_t = -2.0 * m * r * Sig_t / (Sig * Sig);
    real s2_t = 2.0 * s * c;
    memset(dr, 0, 16 * sizeof(real));
    memset(dt, 0, 16 * sizeof(real));
    dr[0][0] = f_r;                          dt[0][0] = f_t;
    dr[0][1] = dr[1][0] = f_r;               dt[0][1] = dt[1][0] = f_t;
    dr[0][3] = dr[3][0] = -a * s2 * f_r;     dt[0][3] = dt[3][0] = -a * (f_t * s2 + f * s2_t);
    dr[1][1] = f_r;                          dt[1][1] = f_t;
    dr[1][3] = dr[3][1] = -a * s2 * f_r;     dt[1][3] = dt[3][1] = -a * (s2_t * (1.0 + f) + s2 * f_t);
    dr[2][2] = Sig_r;                        dt[2][2] = Sig_t;
    dr[3][3] = s2 * (Sig_r + a * a * s2 * f_r);
    dt[3][3] = s2_t * (Sig + a * a * s2 * (1.0 + f)) + s2 * (Sig_t + a * a * (s2_t * (1.0 + f) + s2 * f_t));
}

/* Lambda_a = d x^a_KS / d x^a_MKS (diagonal), A.12-A.13; and its derivative along its own axis */
static void mks_jac(const orc_params *P, const real X[4], real *r, real *th, real Lam[4], real dLam[4])
{
    real dth, d2th;
    real ex = exp(X[1]);
    *r = P->mks_r0 + ex;                                                       /* A.10 */
    orc_mks_theta(P->mks_h, X[2], th, &dth, &d2th);
    Lam[0] = 1.0; Lam[1] = ex;  Lam[2] = dth;  Lam[3] = 1.0;
    dLam[0] = 0.0; dLam[1] = ex; dLam[2] = d2th; dLam[3] = 0.0;
}

/* g^MKS_ab = Lam_a Lam_b g^KS_ab (no sum) */
void orc_metric_mks(const orc_params *P, const real X[4], real g[4][4])
{
    real r, th, Lam[4], dLam[4], gk[4][4];
    mks_jac(P, X, &r, &th, Lam, dLam);
    orc_metric_ks(P->a, P->mass, r, th, gk);
    for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) g[a][b] = Lam[a] * Lam[b] * gk[a][b];
}

void orc_metric_mks_inv(const orc_params *P, const real X[4], real gi[4][4])
{
    real r, th, Lam[4], dLam[4], gk[4][4];
    mks_jac(P, X, &r, &th, Lam, dLam);
    orc_metric_ks_inv(P->a, P->mass, r, th, gk);
    for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) gi[a][b] = gk[a][b] / (Lam[a] * Lam[b]);
}

/* dg[c][a][b] = d g^MKS_ab / d x^c  (c = 1, 2 only; the metric does not depend on t, phi) */
void orc_dmetric_mks(const orc_params *P, const real X[4], real dg[4][4][4])
{
    real r, th, Lam[4], dLam[4], gk[4][4], dr[4][4], dt[4][4];
    mks_jac(P, X, &r, &th, Lam, dLam);
    orc_metric_ks(P->a, P->mass, r, th, gk);
    metric_ks_deriv(P->a, P->mass, r, th, dr, dt);
    memset(dg, 0, 64 * sizeof(real));
    for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) {
        /* d/dx1: dr/dx1 = Lam_1; Lam_1 itself depends on x1 */
        real dLL1 = (a == 1 ? dLam[1] : 0.0) * Lam[b] + Lam[a] * (b == 1 ? dLam[1] : 0.0);
        dg[1][a][b] = dLL1 * gk[a][b] + Lam[a] * Lam[b] * dr[a][b] * Lam[1];
        real dLL2 = (a == 2 ? dLam[2] : 0.0) * Lam[b] + Lam[a] * (b == 2 ? dLam[2] : 0.0);
        dg[2][a][b] = dLL2 * gk[a][b] + Lam[a] * Lam[b] * dt[a][b] * Lam[2];
    }
}

/* Eq. 2: Gamma^a_mn = 1/2 g^{ar} [ d_m g_nr + d_n g_mr - d_r g_mn ]            */
void orc_christoffel_mks(const orc_params *P, const real X[4], real Gam[4][4][4])
{
    real gi[4][4], dg[4][4][4];
    orc_metric_mks_inv(P, X, gi);
    orc_dmetric_mks(P, X, dg);
    for (int a = 0; a < 4; ++a)
        for (int m = 0; m < 4; ++m)
            for (int n = 0; n < 4; ++n) {
                real acc = 0.0;
                for (int r = 0; r < 4; ++r)
                    acc += gi[a][r] * (dg[m][n][r] + dg[n][m][r] - dg[r][m][n]);
                Gam[a][m][n] = 0.5 * acc;
            }
}

/* Eq. 6: f^a = -Gamma^a_mn k^m k^n                                              */
void orc_rhs(const orc_params *P, const real X[4], const real K[4], real f[4])
{
    real Gam[4][4][4];
    orc_christoffel_mks(P, X, Gam);
    for (int a = 0; a < 4; ++a) {
        real acc = 0.0;
        for (int m = 0; m < 4; ++m) for (int n = 0; n < 4; ++n) acc += Gam[a][m][n] * K[m] * K[n];
        f[a] = -acc;
    }
}

/* Eq. 4: g_mn k^m k^n */
real orc_null_norm(const orc_params *P, const real X[4], const real K[4])
{
    real g[4][4], acc = 0.0;
    orc_metric_mks(P, X, g);
    for (int m = 0; m < 4; ++m) for (int n = 0; n < 4; ++n) acc += g[m][n] * K[m] * K[n];
    return acc;
}

/* Eq. 38-40, mu = 0: E = -k_t, L = k_phi, Q = k_th^2 + cos^2 th [ -a^2 k_t^2 + k_phi^2/sin^2 th ]
 * k_t, k_phi, k_theta are the same in BL and KS; k_theta = k_{x2} / theta'. */
void orc_conserved(const orc_params *P, const real X[4], const real K[4], real *E, real *L, real *Q)
{
    real g[4][4], kc[4], r, th, Lam[4], dLam[4];
    orc_metric_mks(P, X, g);
    mks_jac(P, X, &r, &th, Lam, dLam);
    for (int m = 0; m < 4; ++m) { kc[m] = 0.0; for (int n = 0; n < 4; ++n) kc[m] += g[m][n] * K[n]; }
    real kth = kc[2] / Lam[2];
    real s = sin(th), c = cos(th);
    *E = -kc[0];
    *L = kc[3];
    *Q = kth * kth + c * c * (-P->a * P->a * kc[0] * kc[0] + kc[3] * kc[3] / (s * s));
}

static real horizon_radius(const orc_params *P)
{
    real d = P->mass * P->mass - P->a * P->a;
    return d >= 0.0 ? P->mass + sqrt(d) : 0.0;
}
real orc_horizon(const orc_params *P) { return horizon_radius(P); }

/* ======================================================================================= */
/* Camera, Eq. 25-29, E = 1 [A3], a^2 in Eq. 26 and Eq. 29 [A4], k^r > 0 [A2] */
/* ======================================================================================= */
void orc_camera_ab(const orc_params *P, real alpha, real beta, real X[4], real K[4])
{
    const real a = P->a, m = P->mass, r = P->r_cam;
    const real inc = P->incl_deg * (ORC_PI / 180.0);
    const real s = sin(inc), c = cos(inc);
    real L = -alpha * sqrt(1.0 - c * c);                                     /* Eq. 25 */
    real Q = beta * beta + c * c * (alpha * alpha - a * a);                  /* Eq. 26 [A4] */
    real sgn = (beta > 0.0) - (beta < 0.0);
    real k_th = sgn * sqrt(fabs(Q - L * L * (c * c) / (s * s) + a * a * c * c));   /* Eq. 29 [A4] */
    /* raise with the Boyer-Lindquist inverse metric (k_t = -1, k_phi = L: Eq. 27-28) */
    real Sig = r * r + a * a * c * c;
    real Del = r * r - 2.0 * m * r + a * a;
    real Pp = (r * r + a * a) - a * L;
    real R = Pp * Pp - Del * ((L - a) * (L - a) + Q);                        /* null condition */
    real kr = sqrt(R) / Sig;                                                 /* k^r > 0 [A2] */
    real kt = ((r * r + a * a) * Pp / Del + a * (L - a * s * s)) / Sig;
    real kph = (a * Pp / Del + L / (s * s) - a) / Sig;
    real kth = k_th / Sig;
    /* BL -> KS, matrix A.5 */
    real kt_ks = kt + (2.0 * m * r / Del) * kr;
    real kph_ks = kph + (a / Del) * kr;
    /* KS -> MKS, A.8-A.9; x2(i) by Newton-Raphson A.14-A.16 */
    real x2, th, dth, d2th;
    orc_x2_of_theta(P->mks_h, inc, 1e-15, &x2);
    orc_mks_theta(P->mks_h, x2, &th, &dth, &d2th);
    X[0] = P->t_cam; X[1] = log(r - P->mks_r0); X[2] = x2; X[3] = 0.0;
    K[0] = kt_ks; K[1] = kr / (r - P->mks_r0); K[2] = kth / dth; K[3] = kph_ks;
}

/* pixel centres [A4b]: alpha_ix = (ix + 1/2) fov/nx - fov/2, beta_iy likewise */
void orc_pixel_ab(const orc_params *P, int ix, int iy, real *alpha, real *beta)
{
    *alpha = (ix + 0.5) * P->fov_M / P->nx - 0.5 * P->fov_M;
    *beta = (iy + 0.5) * P->fov_M / P->ny - 0.5 * P->fov_M;
}

/* ======================================================================================= */
/* Step rule and RK4                                                                         */
/* ======================================================================================= */
real orc_step_size(const orc_params *P, const real X[4], const real K[4])
{
    if (P->step_policy == 0) {
        /* policy A [A6]: h = clamp(c (r - r_H), min, max)  (BASELINE.json configs[0]), with the
         * polar guard h <= eps_polar * r |sin theta| (Eq. 23, with |k^theta|
         * replaced by its E = 1 bound 1/r), floored at step_min.  Without a guard rays that
         * graze the spin axis take steps much longer than their distance to the coordinate
         * singularity and blow up. */
        real r, th, Lam[4], dLam[4];
        mks_jac(P, X, &r, &th, Lam, dLam);
        real h = P->step_c * (r - horizon_radius(P));
        if (h < P->step_min) h = P->step_min;
        if (h > P->step_max) h = P->step_max;
        real hp = P->eps_polar * r * fabs(sin(th));
        if (hp < h) h = hp;
        if (h < P->step_min) h = P->step_min;
        return h;
    } else {
        /* policy B: Eq. 21-24 on the MKS components */
        real x2 = X[2];
        x2 = x2 - 2.0 * floor(0.5 * x2);          /* into [0,2) */
        if (x2 > 1.0) x2 = 2.0 - x2;              /* folded into [0,1] */
        real d1 = P->eps / (fabs(K[1]) + P->delta);                          /* Eq. 22 */
        real d2 = P->eps * fmin(x2, 1.0 - x2) / (fabs(K[2]) + P->delta);     /* Eq. 23 */
        real d3 = P->eps / (fabs(K[3]) + P->delta);                          /* Eq. 24 */
        return 1.0 / (1.0 / fabs(d1) + 1.0 / fabs(d2) + 1.0 / fabs(d3));       /* Eq. 21 */
    }
}

/* Eq. 7-16, exactly as printed */
void orc_rk4_step(const orc_params *P, real X[4], real K[4], real dl)
{
    real C1x[4], C2x[4], C3x[4], C4x[4], C1k[4], C2k[4], C3k[4], C4k[4];
    real f[4], Xs[4], Ks[4];
    int i;
    orc_rhs(P, X, K, f);
    for (i = 0; i < 4; ++i) { C1x[i] = dl * K[i]; C1k[i] = dl * f[i]; }                       /* 7, 11 */
    for (i = 0; i < 4; ++i) { Xs[i] = X[i] + 0.5 * C1x[i]; Ks[i] = K[i] + 0.5 * C1k[i]; }
    orc_rhs(P, Xs, Ks, f);
    for (i = 0; i < 4; ++i) { C2x[i] = dl * (K[i] + 0.5 * C1k[i]); C2k[i] = dl * f[i]; }      /* 8, 12 */
    for (i = 0; i < 4; ++i) { Xs[i] = X[i] + 0.5 * C2x[i]; Ks[i] = K[i] + 0.5 * C2k[i]; }
    orc_rhs(P, Xs, Ks, f);
    for (i = 0; i < 4; ++i) { C3x[i] = dl * (K[i] + 0.5 * C2k[i]); C3k[i] = dl * f[i]; }      /* 9, 13 */
    for (i = 0; i < 4; ++i) { Xs[i] = X[i] + C3x[i]; Ks[i] = K[i] + C3k[i]; }
    orc_rhs(P, Xs, Ks, f);
    for (i = 0; i < 4; ++i) { C4x[i] = dl * (K[i] + C3k[i]); C4k[i] = dl * f[i]; }            /* 10, 14 */
    for (i = 0; i < 4; ++i) {
        X[i] = X[i] + (1.0 / 6.0) * (C1x[i] + 2.0 * C2x[i] + 2.0 * C3x[i] + C4x[i]);          /* 15 */
        K[i] = K[i] + (1.0 / 6.0) * (C1k[i] + 2.0 * C2k[i] + 2.0 * C3k[i] + C4k[i]);          /* 16 */
    }
}
/* Note on Eq. 8-10: the paper prints C_{2,x} = dl (k + C_{1,x}/2); the x-increment of an RK4
 * stage is dl times the STAGE wavevector, i.e. k + C_{1,k}/2 -- with C_{1,x} the printed form
 * would add a length to a wavevector.  Read as the k-coefficient [A21 in DESIGN.md]. */

/* Velocity Verlet, Eq. 17-20.  (dk/dl)_n is evaluated from the current (x_n, k_n) at the
 * start of every step [A23 in DESIGN.md]: the scheme is then a map of (x_n, k_n) alone, and the paper's cost
 * argument (fewer evaluations of the connection) is unaffected because the connection at x_n was
 * already evaluated by the previous step's Eq. 19.  corrector != 0 adds the refinement of PAPER.md:127: Eq. 19
 * re-evaluated with k_{n+1,p} = k_{n+1}, then Eq. 20 again. */
void orc_verlet_step(const orc_params *P, real X[4], real K[4], real dl, int corrector)
{
    real fn[4], fn1[4], Xn[4], Kp[4], Kn[4];
    int i;
    orc_rhs(P, X, K, fn);
    for (i = 0; i < 4; ++i) Xn[i] = X[i] + K[i] * dl + 0.5 * fn[i] * (dl * dl);              /* 17 */
    for (i = 0; i < 4; ++i) Kp[i] = K[i] + fn[i] * dl;                                       /* 18 */
    orc_rhs(P, Xn, Kp, fn1);                                                                 /* 19 */
    for (i = 0; i < 4; ++i) Kn[i] = K[i] + 0.5 * (fn[i] + fn1[i]) * dl;                      /* 20 */
    if (corrector) {
        orc_rhs(P, Xn, Kn, fn1);                                                             /* 19 with k_{n+1} */
        for (i = 0; i < 4; ++i) Kn[i] = K[i] + 0.5 * (fn[i] + fn1[i]) * dl;                  /* 20 again */
    }
    for (i = 0; i < 4; ++i) { X[i] = Xn[i]; K[i] = Kn[i]; }
}

/* "RK2": Table B.1 names it, the paper never defines it.  Read as the explicit midpoint
 * method, the two-stage member of the family Eq. 7-16 belong to [A17]. */
void orc_rk2_step(const orc_params *P, real X[4], real K[4], real dl)
{
    real f[4], Xs[4], Ks[4];
    int i;
    orc_rhs(P, X, K, f);
    for (i = 0; i < 4; ++i) { Xs[i] = X[i] + 0.5 * dl * K[i]; Ks[i] = K[i] + 0.5 * dl * f[i]; }
    orc_rhs(P, Xs, Ks, f);
    for (i = 0; i < 4; ++i) { X[i] = X[i] + dl * Ks[i]; K[i] = K[i] + dl * f[i]; }
}

/* integrator: 0 = RK4 (Eq. 7-16), 1 = Verlet (Eq. 17-20), 2 = Verlet + corrector, 3 = RK2 [A17] */
void orc_step(const orc_params *P, real X[4], real K[4], real dl)
{
    switch (P->integrator) {
        case 1: orc_verlet_step(P, X, K, dl, 0); break;
        case 2: orc_verlet_step(P, X, K, dl, 1); break;
        case 3: orc_rk2_step(P, X, K, dl); break;
        default: orc_rk4_step(P, X, K, dl); break;
    }
}

/* ======================================================================================= */
/* Grid interpolation [A16] / O6                                                             */
/* ======================================================================================= */
static real grid_val(const orc_params *P, long m, long i, long j, long k, int f)
{
    size_t idx = ((((size_t)m * P->n1 + i) * P->n2 + j) * P->n3 + k) * 8 + f;
    if (P->grid_dtype == 1) return (real)((const float *)P->grid)[idx];
    return (real)((const double *)P->grid)[idx];
}

/* returns 1 and the 8 interpolated primitives, or 0 if outside the radial range */
int orc_grid_interp(const orc_params *P, const real X[4], real prim[8])
{
    real d1 = (P->x1_max - P->x1_min) / P->n1;
    real f1 = (X[1] - (P->x1_min + 0.5 * d1)) / d1;
    if (!(f1 >= 0.0) || f1 > (real)(P->n1 - 1)) return 0;
    long i0 = (long)floor(f1);
    if (i0 > P->n1 - 2) i0 = P->n1 - 2;
    if (i0 < 0) i0 = 0;
    real w1 = f1 - (real)i0;
    long i1 = (P->n1 > 1) ? i0 + 1 : i0;

    real x2 = X[2], ph = X[3];
    if (x2 < 0.0) { x2 = -x2; ph += ORC_PI; }
    else if (x2 > 1.0) { x2 = 2.0 - x2; ph += ORC_PI; }
    real f2 = x2 * P->n2 - 0.5;
    if (f2 < 0.0) f2 = 0.0;
    if (f2 > (real)(P->n2 - 1)) f2 = (real)(P->n2 - 1);
    long j0 = (long)floor(f2);
    if (j0 > P->n2 - 2) j0 = P->n2 - 2;
    if (j0 < 0) j0 = 0;
    real w2 = f2 - (real)j0;
    long j1 = (P->n2 > 1) ? j0 + 1 : j0;

    long k0 = 0, k1 = 0; real w3 = 0.0;
    if (P->n3 > 1) {
        real twopi = 2.0 * ORC_PI;
        ph = ph - twopi * floor(ph / twopi);
        real f3 = ph / (twopi / P->n3) - 0.5;
        real fl = floor(f3);
        w3 = f3 - fl;
        k0 = (long)fl;
        k0 = ((k0 % P->n3) + P->n3) % P->n3;
        k1 = (k0 + 1) % P->n3;
    }
    long m0 = P->snapshot, m1 = P->snapshot; real w4 = 0.0;
    if (P->nt > 1 && P->slow_light) {
        real f4 = (X[0] - P->t0) / P->dt_snap;
        if (!(f4 >= 0.0)) f4 = 0.0;
        if (f4 > (real)(P->nt - 1)) f4 = (real)(P->nt - 1);
        m0 = (long)floor(f4);
        if (m0 > P->nt - 2) m0 = P->nt - 2;
        w4 = f4 - (real)m0;
        m1 = m0 + 1;
    }
    for (int f = 0; f < 8; ++f) {
        real acc = 0.0;
        for (int dm = 0; dm < 2; ++dm) for (int di = 0; di < 2; ++di)
            for (int dj = 0; dj < 2; ++dj) for (int dk = 0; dk < 2; ++dk) {
                real w = (dm ? w4 : 1.0 - w4) * (di ? w1 : 1.0 - w1) * (dj ? w2 : 1.0 - w2) * (dk ? w3 : 1.0 - w3);
                if (w == 0.0) continue;
                acc += w * grid_val(P, dm ? m1 : m0, di ? i1 : i0, dj ? j1 : j0, dk ? k1 : k0, f);
            }
        prim[f] = acc;
    }
    return 1;
}

/* ======================================================================================= */
/* Plasma models, O5                                                                         */
/* ======================================================================================= */
static real dot4(real g[4][4], const real A[4], const real B[4])
{
    real acc = 0.0;
    for (int m = 0; m < 4; ++m) for (int n = 0; n < 4; ++n) acc += g[m][n] * A[m] * B[n];
    return acc;
}

/* Returns 1 if plasma is present at X and fills n_e [cm^-3], Theta_e, B [G], u^mu (MKS),
 * p^mu (direction of the field four-vector, orthogonal to u), sin_fixed (<0 unless SLAB). */
int orc_plasma(const orc_params *P, const real X[4], real *ne, real *thetae, real *Bg,
               real u[4], real p[4], real *sin_fixed)
{
    real g[4][4], gi[4][4], r, th, Lam[4], dLam[4];
    const real *M = P->model;
    *sin_fixed = -1.0;
    mks_jac(P, X, &r, &th, Lam, dLam);
    if (P->plasma_model == ORC_VACUUM) return 0;
    orc_metric_mks(P, X, g);

    if (P->plasma_model == ORC_SPHERE || P->plasma_model == ORC_TORUS) {
        real n, Te, beta, seed[4] = {0, 0, 0, 0};
        if (P->plasma_model == ORC_SPHERE) {
            /* model = [n0, n_exp, T0, T_exp, beta]; free fall from rest at infinity [A14] */
            n = M[0] * pow(r, M[1]);
            Te = M[2] * pow(r, M[3]);
            beta = M[4];
            real m = P->mass, a = P->a;
            real ucov[4] = {-1.0, 0.0, 0.0, 0.0};
            real sq = sqrt(2.0 * m * r * (r * r + a * a));
            ucov[1] = (m > 0.0) ? -2.0 * m * r / (2.0 * m * r + sq) : 0.0;     /* u_r in KS */
            ucov[1] *= Lam[1];                                                 /* u_{x1} = Lam_1 u_r */
            orc_metric_mks_inv(P, X, gi);
            for (int a_ = 0; a_ < 4; ++a_) { u[a_] = 0.0; for (int b = 0; b < 4; ++b) u[a_] += gi[a_][b] * ucov[b]; }
            seed[1] = 1.0;                                                     /* radial field */
        } else {
            /* model = [n_max, r_peak, r_halfwidth, H, T0, T_exp, beta]; Keplerian on spheres [A14] */
            real xr = (r - M[1]) / M[2];
            real bump = 1.0 - xr * xr;
            if (!(bump > 0.0)) return 0;
            real c = cos(th);
            n = M[0] * bump * bump * exp(-c * c / (2.0 * M[3] * M[3]));
            Te = M[4] * pow(r, M[5]);
            beta = M[6];
            real Om = 1.0 / (pow(r, 1.5) + P->a);
            real den = -g[0][0] - 2.0 * Om * g[0][3] - Om * Om * g[3][3];
            if (!(den > 0.0)) return 0;
            real ut = 1.0 / sqrt(den);
            u[0] = ut; u[1] = 0.0; u[2] = 0.0; u[3] = ut * Om;
            seed[3] = 1.0;                                                     /* toroidal field */
        }
        if (!(n > 0.0)) return 0;
        *ne = n;
        *thetae = ORC_KB * Te / (ORC_ME * ORC_C * ORC_C);
        *Bg = sqrt(8.0 * ORC_PI * n * ORC_KB * Te / beta);                     /* beta = n k T / (B^2/8pi) */
        real su = dot4(g, seed, u);
        for (int a_ = 0; a_ < 4; ++a_) p[a_] = seed[a_] + su * u[a_];          /* projection orthogonal to u */
        return 1;
    }
    if (P->plasma_model == ORC_SLAB) {
        /* model = [n_e, Theta_e, B, half_thickness, sin(pitch)]; static fluid */
        real z = r * cos(th);
        if (!(fabs(z) < M[3])) return 0;
        *ne = M[0]; *thetae = M[1]; *Bg = M[2]; *sin_fixed = M[4];
        u[0] = 1.0 / sqrt(-g[0][0]); u[1] = u[2] = u[3] = 0.0;
        p[0] = p[1] = p[2] = 0.0; p[3] = 1.0;
        return 1;
    }
    /* GRID2D / GRID3DT: HARM primitives [A16] */
    real prim[8];
    if (!orc_grid_interp(P, X, prim)) return 0;
    real rho = prim[0], uu = prim[1];
    if (!(rho > 0.0)) return 0;
    orc_metric_mks_inv(P, X, gi);
    real alpha_l = 1.0 / sqrt(-gi[0][0]);
    real betai[4] = {0.0, gi[0][1] * alpha_l * alpha_l, gi[0][2] * alpha_l * alpha_l, gi[0][3] * alpha_l * alpha_l};
    real ut3[4] = {0.0, prim[2], prim[3], prim[4]};
    real q = 0.0;
    for (int i = 1; i < 4; ++i) for (int j = 1; j < 4; ++j) q += g[i][j] * ut3[i] * ut3[j];
    real gam = sqrt(1.0 + q);
    u[0] = gam / alpha_l;
    for (int i = 1; i < 4; ++i) u[i] = ut3[i] - gam * betai[i] / alpha_l;
    real B3[4] = {0.0, prim[5], prim[6], prim[7]};
    real bt = 0.0;
    for (int i = 1; i < 4; ++i) for (int m = 0; m < 4; ++m) bt += g[i][m] * B3[i] * u[m];
    p[0] = bt;
    for (int i = 1; i < 4; ++i) p[i] = (B3[i] + bt * u[i]) / u[0];
    real Lcm = ORC_G * P->M_bh_g / (ORC_C * ORC_C);
    real rho0 = P->M_unit_g / (Lcm * Lcm * Lcm);
    real B0 = ORC_C * sqrt(4.0 * ORC_PI * rho0);
    *ne = rho * rho0 / (ORC_MP + ORC_ME);                                      /* Eq. 46 */
    real bsq = dot4(g, p, p);
    *Bg = sqrt(bsq > 0.0 ? bsq : 0.0) * B0;
    /* T_p/T_e: constant (Table 2) or, te_model = 1, Eq. 47:
     * R = R_low/(1+beta_p^2) + R_high beta_p^2/(1+beta_p^2), beta_p = P_gas/P_mag, P_gas = (gamma-1) u,
     * P_mag = b^2/2 (code units); model[0] = R_low, model[1] = R_high.  b^2 = 0 is the limit beta_p -> inf. */
    real R = P->tp_over_te;
    if (P->te_model == 1) {
        if (bsq > 0.0) {
            real beta_p = (P->gamma_ad - 1.0) * uu / (0.5 * bsq);
            real b2 = beta_p * beta_p;
            R = M[0] * (1.0 / (1.0 + b2)) + M[1] * (b2 / (1.0 + b2));
        } else R = M[1];
    }
    *thetae = (ORC_MP / ORC_ME) * (P->gamma_ad - 1.0) * (uu / rho) / (1.0 + R);
    return 1;
}

/* ======================================================================================= */
/* Emission, absorption, transfer update                                                     */
/* ======================================================================================= */
/* Eq. 45 */
real orc_planck(real nu, real thetae)
{
    real x = ORC_HPL * nu / (ORC_ME * ORC_C * ORC_C * thetae);
    return (2.0 * ORC_HPL * nu * nu * nu / (ORC_C * ORC_C)) / expm1(x);
}

/* modified Bessel K2 by quadrature: K_2(x) = int_0^inf exp(-x cosh t) cosh(2t) dt (k2_mode = 1) */
real orc_bessel_k2(real x)
{
    /* trapezoid in t is spectrally accurate for this integrand */
    real tmax = acosh(1.0 + 745.0 / x) + 1.0, acc = 0.0;
    int n = 4000;
    real dt = tmax / n;
    for (int i = 0; i <= n; ++i) {
        real t = i * dt, w = (i == 0 || i == n) ? 0.5 : 1.0;
        acc += w * exp(-x * cosh(t)) * cosh(2.0 * t);
    }
    return acc * dt;
}

/* Eq. 42-44 with the prefactor sqrt(2) pi [A12], K2 -> 2 Theta^2 */
real orc_emissivity(real nu, real ne, real thetae, real Bg, real sin_th, int k2_mode)
{
    real nu_c = ORC_E * Bg / (2.0 * ORC_PI * ORC_ME * ORC_C);
    real nu_s = (2.0 / 9.0) * nu_c * thetae * thetae * sin_th;                /* Eq. 44 */
    if (!(nu_s > 0.0) || !(ne > 0.0)) return 0.0;                              /* [A13] */
    real Xx = nu / nu_s;                                                     /* Eq. 43 */
    real K2 = (k2_mode == 1) ? orc_bessel_k2(1.0 / thetae) : 2.0 * thetae * thetae;
    if (!(K2 > 0.0)) return 0.0;                                               /* K_2 underflow (Theta_e < ~1/745) [A13] */
    real term = sqrt(Xx) + pow(2.0, 11.0 / 12.0) * pow(Xx, 1.0 / 6.0);
    return ne * (sqrt(2.0) * ORC_PI * ORC_E * ORC_E * nu_s / (3.0 * ORC_C * K2)) * term * term * exp(-cbrt(Xx));
}

/* Backward update over one step with constant j, alpha [A9]:
 *   dtau = nu_hat alpha L h                       (Eq. 36)
 *   I   += (j / nu_hat^2) L h exp(-tau) w(dtau),  w = (1 - exp(-dtau))/dtau  (Eq. 35 + 37)
 *   tau += dtau                                                                              */
void orc_transfer_update(real *I, real *tau, real j, real alpha, real nu_hat, real Lcm, real h)
{
    real dtau = nu_hat * alpha * Lcm * h;
    real w = (dtau > 0.0) ? -expm1(-dtau) / dtau : 1.0;
    *I += (j / (nu_hat * nu_hat)) * Lcm * h * exp(-*tau) * w;
    *tau += dtau;
}

/* O7: transfer at the new point for every frequency.  Returns 1 if plasma was sampled. */
int orc_transfer(const orc_params *P, const real X[4], const real K[4], real h, real *I, real *tau)
{
    real ne, thetae, Bg, u[4], p[4], sin_fixed, g[4][4];
    if (!orc_plasma(P, X, &ne, &thetae, &Bg, u, p, &sin_fixed)) return 0;
    orc_metric_mks(P, X, g);
    real nu_hat = -dot4(g, K, u);                                            /* Eq. 31 */
    real sin_th;
    if (sin_fixed >= 0.0) sin_th = sin_fixed;
    else {
        real pp = dot4(g, p, p);
        real cos_th = dot4(g, K, p) / (nu_hat * sqrt(pp));                   /* [A11] */
        real s2 = 1.0 - cos_th * cos_th;
        sin_th = sqrt(s2 > 0.0 ? s2 : 0.0);
        if (!(pp > 0.0)) sin_th = 0.0;
    }
    real Lcm = ORC_G * P->M_bh_g / (ORC_C * ORC_C);
    for (int k = 0; k < P->n_freq; ++k) {
        real nu = nu_hat * P->freq_hz[k];
        real j = orc_emissivity(nu, ne, thetae, Bg, sin_th, P->k2_mode);
        real Bnu = orc_planck(nu, thetae);
        real alpha = (j > 0.0 && Bnu > 0.0) ? j / Bnu : 0.0;                 /* Kirchhoff */
        orc_transfer_update(&I[k], &tau[k], j, alpha, nu_hat, Lcm, h);
    }
    return 1;
}

/* ======================================================================================= */
/* Thin-disk workload, Sect. 4.2.1 (Fig. 5-6) [A24]     */
/* ======================================================================================= */
/* Innermost stable circular orbit of the equatorial Kerr geodesics (Bardeen, Press & Teukolsky 1972, the
 * reference the paper gives at PAPER.md:267); a > 0: prograde disk, a < 0: retrograde. */
real orc_r_isco(real a)
{
    real z1 = 1.0 + cbrt(1.0 - a * a) * (cbrt(1.0 + a) + cbrt(1.0 - a));
    real z2 = sqrt(3.0 * a * a + z1 * z1);
    real sg = (a > 0.0) - (a < 0.0);
    return 3.0 + z2 - sg * sqrt((3.0 - z1) * (3.0 + z1 + 2.0 * z2));
}

/* One step of a ray went from (Xp, Kp) to (X, K).  The equatorial plane is x2 = 1/2 (mod 1) in every MKS(h)
 * chart (A.11: theta(1/2 + n) = pi/2 + n pi).  If the step crossed it, the crossing state is the linear
 * interpolation of the MKS state in the step, the emitter is the circular equatorial geodesic
 * u = u^t (1, 0, 0, Omega), Omega = 1/(r^{3/2} + a), and the redshift factor is g = nu_obs/nu_em = 1/(-k.u)
 * (Eq. 31, E = 1).  model = [r_in (<= 0: ISCO), r_out, max_order, p]: a crossing of order
 * n <= max_order with r_in <= r <= r_out adds g^p r^-2 (emission coefficient ~ 1/r^2, no absorption,
 * PAPER.md:267; p = 3 is Eq. 32).  Returns 1 if the plane was crossed; *counted = 1 if it added. */
int orc_disk_crossing(const orc_params *P, const real Xp[4], const real Kp[4], const real X[4],
                      const real K[4], int order, real *dI, real *g_out, real *r_out_x, int *counted)
{
    real fa = floor(Xp[2] - 0.5), fb = floor(X[2] - 0.5);
    *counted = 0;
    if (fa == fb) return 0;
    real plane = 0.5 + (fa > fb ? fa : fb);
    real w = (plane - Xp[2]) / (X[2] - Xp[2]);
    real Xc[4], Kc[4];
    for (int i = 0; i < 4; ++i) { Xc[i] = Xp[i] + w * (X[i] - Xp[i]); Kc[i] = Kp[i] + w * (K[i] - Kp[i]); }
    Xc[2] = plane;
    real r = P->mks_r0 + exp(Xc[1]);
    real r_in = P->model[0] > 0.0 ? P->model[0] : orc_r_isco(P->a);
    *r_out_x = r;
    if (order > (int)P->model[2] || !(r >= r_in) || !(r <= P->model[1])) return 1;
    real g[4][4], u[4];
    orc_metric_mks(P, Xc, g);
    real Om = 1.0 / (pow(r, 1.5) + P->a);
    real den = -g[0][0] - 2.0 * Om * g[0][3] - Om * Om * g[3][3];
    if (!(den > 0.0)) return 1;
    u[0] = 1.0 / sqrt(den); u[1] = 0.0; u[2] = 0.0; u[3] = u[0] * Om;
    real nu_hat = -dot4(g, Kc, u);
    real gg = 1.0 / nu_hat;
    *dI = pow(gg, P->model[3]) / (r * r);
    *g_out = gg;
    *counted = 1;
    return 1;
}

/* ======================================================================================= */
/* Ray loop O4 and image driver                                                              */
/* ======================================================================================= */
typedef struct {
    int32_t status, nsteps, nsampled, pad_;
    real null_max;      /* max |g k k| seen along the ray */
    real X[4], K[4];    /* final state */
} orc_ray_result;

/* path: optional [max_path][8] buffer receiving (X,K) after every step (NULL to skip);
 * monitor_null != 0 additionally evaluates Eq. 4 after every step (slow; diagnostics only). */
void orc_trace_ray(const orc_params *P, real alpha, real beta, real *I, real *tau,
                   orc_ray_result *res, real *path, int max_path, int monitor_null)
{
    real X[4], K[4];
    const real rH = horizon_radius(P);
    const real r_in = P->r_stop_in_factor * rH, r_out = P->r_stop_out_factor * P->r_cam;
    int n = 0, ns = 0, ncross = 0, status = ORC_RUNNING;
    real nmax = 0.0;
    orc_camera_ab(P, alpha, beta, X, K);
    for (int k = 0; k < P->n_freq; ++k) { I[k] = 0.0; tau[k] = 0.0; }
    for (;;) {
        real r = P->mks_r0 + exp(X[1]);
        if (r < r_in) { status = ORC_CAPTURED; break; }                        /* [A7] */
        if (r > r_out) { status = ORC_ESCAPED; break; }
        if (n >= P->max_steps) { status = ORC_MAXSTEPS; break; }
        if (isfinite(P->tau_cutoff)) {
            real tmin = tau[0];
            for (int k = 1; k < P->n_freq; ++k) if (tau[k] < tmin) tmin = tau[k];
            if (tmin > P->tau_cutoff) { status = ORC_THICK; break; }
        }
        real h = orc_step_size(P, X, K);
        real Xp[4], Kp[4];
        memcpy(Xp, X, 4 * sizeof(real)); memcpy(Kp, K, 4 * sizeof(real));
        orc_step(P, X, K, -h);                                                 /* backward [A2] */
        ++n;
        int fin = 1;
        for (int i = 0; i < 4; ++i) if (!isfinite(X[i]) || !isfinite(K[i])) fin = 0;
        if (!fin) { status = ORC_NONFINITE; break; }
        if (path && n <= max_path) { memcpy(path + 8 * (n - 1), X, 4 * sizeof(real)); memcpy(path + 8 * (n - 1) + 4, K, 4 * sizeof(real)); }
        real rn = P->mks_r0 + exp(X[1]);
        if (P->plasma_model == ORC_DISK) {
            /* thin disk: I[0] = sum of g^p / r^2 over the counted crossings, tau[0] = g of the first counted one */
            real dI, gg, rx; int counted;
            if (orc_disk_crossing(P, Xp, Kp, X, K, ncross + 1, &dI, &gg, &rx, &counted)) {
                ++ncross;
                if (counted) { I[0] += dI; if (ns == 0) tau[0] = gg; ++ns; }
            }
        } else
        if (rn >= r_in && rn <= r_out) ns += orc_transfer(P, X, K, h, I, tau); /* [A8] end-point sample */
        if (monitor_null) { real nn = fabs(orc_null_norm(P, X, K)); if (nn > nmax) nmax = nn; }
    }
    if (res) {
        res->status = status; res->nsteps = n; res->nsampled = ns; res->null_max = nmax;
        memcpy(res->X, X, 4 * sizeof(real)); memcpy(res->K, K, 4 * sizeof(real));
    }
}

/* O8: image[k][iy][ix] = I_nu,obs [erg s^-1 cm^-2 Hz^-1 sr^-1] for rows row0 <= iy < row1 in
 * steps of row_stride (a stride > 1 is used only for bounded timing samples); status / nsteps
 * ([ny][nx]) may be NULL.  Parallel over image rows only.  *steps, *sampled: totals. */
int orc_render_rows2(const orc_params *P, real *image, real *tau_image, int32_t *status, int32_t *nsteps,
                     int row0, int row1, int row_stride, uint64_t *steps, uint64_t *sampled);
int orc_render_rows(const orc_params *P, real *image, int32_t *status, int32_t *nsteps,
                    int row0, int row1, int row_stride, uint64_t *steps, uint64_t *sampled)
{
    return orc_render_rows2(P, image, NULL, status, nsteps, row0, row1, row_stride, steps, sampled);
}

/* as orc_render_rows; tau_image ([n_freq][ny][nx] or NULL) receives tau_k of every ray (thin disk: the
 * redshift factor g of the first counted crossing, 0 if none) */
int orc_render_rows2(const orc_params *P, real *image, real *tau_image, int32_t *status, int32_t *nsteps,
                     int row0, int row1, int row_stride, uint64_t *steps, uint64_t *sampled)
{
    uint64_t tot = 0, tots = 0;
    if (row_stride < 1) row_stride = 1;
    #pragma omp parallel for schedule(dynamic, 1) reduction(+:tot, tots)
    for (int iy = row0; iy < row1; iy += row_stride) {
        real *I = (real *)malloc(sizeof(real) * 2 * (size_t)P->n_freq), *tau = I + P->n_freq;
        for (int ix = 0; ix < P->nx; ++ix) {
            real al, be;
            orc_ray_result res;
            orc_pixel_ab(P, ix, iy, &al, &be);
            orc_trace_ray(P, al, be, I, tau, &res, NULL, 0, 0);
            for (int k = 0; k < P->n_freq; ++k) image[((size_t)k * P->ny + iy) * P->nx + ix] = I[k];
            if (tau_image) for (int k = 0; k < P->n_freq; ++k) tau_image[((size_t)k * P->ny + iy) * P->nx + ix] = tau[k];
            if (status) status[(size_t)iy * P->nx + ix] = res.status;
            if (nsteps) nsteps[(size_t)iy * P->nx + ix] = res.nsteps;
            tot += (uint64_t)res.nsteps; tots += (uint64_t)res.nsampled;
        }
        free(I);
    }
    if (steps) *steps = tot;
    if (sampled) *sampled = tots;
    return 0;
}

int orc_render(const orc_params *P, real *image, int32_t *status, int32_t *nsteps)
{
    return orc_render_rows(P, image, status, nsteps, 0, P->ny, 1, NULL, NULL);
}

/* O8: F_k [Jy] = 1e23 * sum_pix I_k * (fov/nx)(fov/ny) L^2 / D^2, Kahan-compensated, row-major order */
void orc_flux(const orc_params *P, const real *image, real *flux_jy)
{
    /* the sum and the scale factor are double in every build: D^2 ~ 7e44 cm^2 is beyond the range of a float */
    double Lcm = ORC_G * P->M_bh_g / (ORC_C * ORC_C);
    double scale = 1e23 * ((double)P->fov_M / P->nx) * ((double)P->fov_M / P->ny) * Lcm * Lcm / (P->D_src_cm * P->D_src_cm);
    size_t npix = (size_t)P->nx * P->ny;
    for (int k = 0; k < P->n_freq; ++k) {
        double s = 0.0, c = 0.0;
        for (size_t i = 0; i < npix; ++i) {
            double y = (double)image[(size_t)k * npix + i] - c, t = s + y;
            c = (t - s) - y; s = t;
        }
        flux_jy[k] = (real)(s * scale);
    }
}

/* Line profile of the thin disk (Fig. 6): hist[b] = sum over pixels whose redshift factor g falls
 * in bin b of [g_min, g_max) of I * (fov/nx)(fov/ny); pixels with g = 0 (no crossing) are skipped.  Row-major
 * order, plain summation per bin. */
void orc_line_profile(const orc_params *P, const real *image_I, const real *image_g, int nbins,
                      real g_min, real g_max, real *hist)
{
    size_t npix = (size_t)P->nx * P->ny;
    real area = (P->fov_M / P->nx) * (P->fov_M / P->ny);
    for (int b = 0; b < nbins; ++b) hist[b] = 0.0;
    for (size_t i = 0; i < npix; ++i) {
        real g = image_g[i];
        if (!(g > 0.0)) continue;
        real fb = floor((g - g_min) / (g_max - g_min) * nbins);
        if (fb < 0.0 || fb >= (real)nbins) continue;
        hist[(int)fb] += image_I[i] * area;
    }
}

/* Time calibration of Sect. 5.1: "translating the slow-light light curve with respect to the
 * fast-light light curve on the time axis".  Step by step: normalise both curves by their means; for every trial shift
 * d_k = -max_shift + 2 max_shift k/(n_grid-1): interpolate the slow curve linearly at t_fast[i] + d_k (skipping
 * points outside the slow curve's time range; a shift that keeps fewer than max(4, n_fast/2) points is skipped),
 * take the rms difference; keep the first shift with the smallest rms.  Returns that shift, *rms_out the rms
 * (HUGE_VAL if no shift qualified). */
real orc_calibrate_delay(int n_fast, const real *t_fast, const real *F_fast, int n_slow, const real *t_slow,
                         const real *F_slow, real max_shift, int n_grid, real *rms_out)
{
    real mean_f = 0.0, mean_s = 0.0, best_d = 0.0, best = HUGE_VAL;
    for (int i = 0; i < n_fast; ++i) mean_f += F_fast[i] / n_fast;
    for (int i = 0; i < n_slow; ++i) mean_s += F_slow[i] / n_slow;
    int need = n_fast / 2 > 4 ? n_fast / 2 : 4;
    for (int k = 0; k < n_grid; ++k) {
        real d = (n_grid > 1) ? -max_shift + 2.0 * max_shift * k / (n_grid - 1) : 0.0;
        real sum = 0.0;
        int used = 0;
        for (int i = 0; i < n_fast; ++i) {
            real t = t_fast[i] + d;
            if (t < t_slow[0] || t > t_slow[n_slow - 1]) continue;
            int seg = 0;
            while (seg < n_slow - 2 && t_slow[seg + 1] < t) ++seg;            /* t_slow[seg] <= t <= t_slow[seg+1] */
            real Fs = F_slow[seg] + (F_slow[seg + 1] - F_slow[seg]) * (t - t_slow[seg]) / (t_slow[seg + 1] - t_slow[seg]);
            real diff = Fs / mean_s - F_fast[i] / mean_f;
            sum += diff * diff;
            ++used;
        }
        if (used < need) continue;
        real rms = sqrt(sum / used);
        if (rms < best) { best = rms; best_d = d; }
    }
    *rms_out = best;
    return best_d;
}

size_t orc_sizeof_params(void) { return sizeof(orc_params); }
size_t orc_sizeof_ray_result(void) { return sizeof(orc_ray_result); }
