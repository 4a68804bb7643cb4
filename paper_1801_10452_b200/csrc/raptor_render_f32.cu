// raptor_render_f32.cu -- single-precision variant of the ray kernel for the paper's OWN performance configuration
// (Table B.1: "Single precision: yes", integration scheme "RK2", step rule
// Eq. 21-24 with eps = 0.03, radiative transfer on): GRID2D plasma, explicit midpoint [A17], policy B, one frequency,
// optional tau cut-off.  Everything else of the C ABI stays FP64 (the contract of BASELINE.json); this kernel exists to
// put a like-for-like number beside the paper's 104,900 geodesics/s (GTX 1080, FP32).
//
// Same discrete algorithm as the FP64 kernel, every quantity a float.  No incremental geometry:
// expf / sincospif at both points of a step; reciprocals and the divisions of the step rule and the transfer update
// are the hardware approximations (MUFU.RCP, 1 ulp) -- the paper's build used pgcc "fastmath" (Table B.2).  Constants outside the float range (G M/c^2 in cm, distances)
// never enter the kernel: the host passes the in-range combinations (L in cm, n_e scale, B0, ...).
#include <cuda_runtime.h>
#include <stdint.h>

#include "raptor_kernels.h"

namespace raptor {

namespace f32 {

constexpr float kPIf = 3.14159265358979323846f;
// CGS constants [A19], float copies
constexpr float kCf = 2.99792458e10f, kEf = 4.80320471e-10f, kMEf = 9.1093837e-28f, kHPLf = 6.62607015e-27f;

struct Geomf { float ex, r, s, c, dth, d2th; };

__device__ __forceinline__ float rcpf(float x) { return __fdividef(1.0f, x); }       // MUFU.RCP

__device__ __forceinline__ void geom_eval(const KPf& P, float x1, float x2, Geomf& G) {
    G.ex = expf(x1);
    G.r = P.r0 + G.ex;                                              // A.10
    float s2, c2;
    sincospif(2.0f * x2, &s2, &c2);
    // A.11 in units of pi: theta/pi = x2 + (1-h)/(2 pi) sin(2 pi x2), so that sincospif reduces the argument exactly
    const float thp = fmaf((0.5f / kPIf) * P.omh, s2, x2);
    G.dth = kPIf * fmaf(P.omh, c2, 1.0f);                           // A.13
    G.d2th = (-2.0f * kPIf * kPIf) * P.omh * s2;
    sincospif(thp, &G.s, &G.c);
}

// Geodesic right-hand side, Eq. 6 in MKS: the Euler-Lagrange form of raptor_device.cuh, in float
__device__ __forceinline__ void geodesic_rhs(const KPf& P, const Geomf& G, float Kt, float K1, float K2, float Kp,
                                             float& ft, float& f1, float& f2, float& fp) {
    const float a = P.a, a2 = P.a2, r = G.r, s = G.s, c = G.c;
    const float kt = Kt, kr = G.ex * K1, kh = G.dth * K2, kp = Kp;
    const float ss = s * s, sc = s * c;
    const float a2cc = fmaf(-a2, ss, a2);
    const float rsq = r * r;
    const float Sig = rsq + a2cc, rr = rsq + a2;
    const float iS = rcpf(Sig), iss = rcpf(ss), iex = rcpf(G.ex), idth = rcpf(G.dth);
    const float tm = P.twom * iS;
    const float f = r * tm;
    const float mi2 = tm * iS;
    const float f_r = mi2 * (a2cc - rsq);
    const float asc2 = P.twoa * sc;
    const float f_h = (mi2 * r) * (a * asc2);
    const float ass = a * ss;
    const float ell = kt + fmaf(-ass, kp, kr);
    const float fdot = fmaf(f_r, kr, f_h * kh);
    const float hell2 = (0.5f * ell) * ell;
    const float kh2 = kh * kh;
    const float H_r = fmaf(r, fmaf(ss * kp, kp, kh2), f_r * hell2);
    const float D = fmaf(fdot, ell, f * H_r);
    const float W = fmaf(f, ell, kr);
    const float rrkp = rr * kp;
    const float m2rkr = -2.0f * (r * kr);
    const float HhS = fmaf(m2rkr, kh, fmaf(sc, fmaf(a2, kh2, kp * fmaf(-P.twoa, W, rrkp)), f_h * hell2));
    const float U = fmaf(asc2 * kh, kp, H_r - D);
    const float cot2kh = (sc * iss) * (kh + kh);
    const float V = fmaf(m2rkr, kp, fmaf(cot2kh, fmaf(a, W, -rrkp), a * D));
    const float Ah = HhS * iS;
    const float Ar = fmaf(rr, U, ass * V) * iS;
    ft = D;
    fp = fmaf(a, U, V) * iS;
    f1 = fmaf(Ar, iex, -K1 * K1);
    f2 = fmaf(-G.d2th * K2, K2, Ah) * idth;
}

// Camera, Eq. 25-29 + A.5 + A.8-A.9, in float
__device__ __forceinline__ void camera_ray(const KPf& P, float alpha, float beta, float X[4], float K[4]) {
    const float a = P.a, m = P.m, r = P.r_cam, s = P.sin_i, c = P.cos_i;
    const float L = -alpha * P.sq1mc2;
    const float Q = fmaf(beta, beta, c * c * (alpha * alpha - P.a2));
    const float sgn = (beta > 0.0f) ? 1.0f : ((beta < 0.0f) ? -1.0f : 0.0f);
    const float k_th = sgn * sqrtf(fabsf(Q - L * L * (c * c) / (s * s) + P.a2 * c * c));
    const float Sig = r * r + P.a2 * c * c;
    const float Del = r * r - 2.0f * m * r + P.a2;
    const float Pp = (r * r + P.a2) - a * L;
    const float R = Pp * Pp - Del * ((L - a) * (L - a) + Q);
    const float kr = sqrtf(R) / Sig;
    const float kt = ((r * r + P.a2) * Pp / Del + a * (L - a * s * s)) / Sig;
    const float kph = (a * Pp / Del + L / (s * s) - a) / Sig;
    const float kth = k_th / Sig;
    X[0] = P.t_cam; X[1] = P.x1_cam; X[2] = P.x2_cam; X[3] = 0.0f;
    K[0] = kt + (2.0f * m * r / Del) * kr;
    K[1] = kr / (r - P.r0);
    K[2] = kth / P.dth_cam;
    K[3] = kph + (a / Del) * kr;
}

// Step rule B, Eq. 21-24
__device__ __forceinline__ float step_size(const KPf& P, float x2, float K1, float K2, float Kp) {
    float xf = x2 - 2.0f * floorf(0.5f * x2);
    if (xf > 1.0f) xf = 2.0f - xf;
    // 1/dl = sum_i 1/dl_i: the same value from 2 divisions instead of 7
    const float inv = (fabsf(K1) + P.delta) + __fdividef(fabsf(K2) + P.delta, fminf(xf, 1.0f - xf)) + (fabsf(Kp) + P.delta);
    return __fdividef(P.eps, inv);
}

// bilinear sample of the 2-D grid [A16] (float cells, 32 B each)
__device__ __forceinline__ bool grid2d_interp(const KPf& P, float x1, float x2, float q[8]) {
    const float f1 = (x1 - P.x1_first) * P.inv_d1;
    if (!(f1 >= 0.0f) || f1 > (float)(P.n1 - 1)) return false;
    const int i0 = max(min((int)f1, P.n1 - 2), 0);
    const float w1 = f1 - (float)i0;
    if (x2 < 0.0f) x2 = -x2; else if (x2 > 1.0f) x2 = 2.0f - x2;
    float f2 = fmaf(x2, (float)P.n2, -0.5f);
    f2 = fminf(fmaxf(f2, 0.0f), (float)(P.n2 - 1));
    const int j0 = max(min((int)f2, P.n2 - 2), 0);
    const float w2 = f2 - (float)j0;
    const float4* g = reinterpret_cast<const float4*>(P.grid);
    const float w[4] = {(1.0f - w1) * (1.0f - w2), (1.0f - w1) * w2, w1 * (1.0f - w2), w1 * w2};
    const size_t cell[4] = {(size_t)i0 * P.n2 + j0, (size_t)i0 * P.n2 + j0 + 1, (size_t)(i0 + 1) * P.n2 + j0, (size_t)(i0 + 1) * P.n2 + j0 + 1};
#pragma unroll
    for (int i = 0; i < 8; ++i) q[i] = 0.0f;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float4 t0 = __ldg(g + 2 * cell[k]), t1 = __ldg(g + 2 * cell[k] + 1);
        q[0] = fmaf(w[k], t0.x, q[0]); q[1] = fmaf(w[k], t0.y, q[1]); q[2] = fmaf(w[k], t0.z, q[2]); q[3] = fmaf(w[k], t0.w, q[3]);
        q[4] = fmaf(w[k], t1.x, q[4]); q[5] = fmaf(w[k], t1.y, q[5]); q[6] = fmaf(w[k], t1.z, q[6]); q[7] = fmaf(w[k], t1.w, q[7]);
    }
    return true;
}

struct Metf { float Sig, rr, ss, ass, f; };
__device__ __forceinline__ float ks_dot(const Metf& M, float At, float Ar, float Ah, float Ap, float Bt, float Br, float Bh, float Bp) {
    const float lA = At + Ar - M.ass * Ap, lB = Bt + Br - M.ass * Bp;
    const float e = Ar * Br - At * Bt + M.Sig * Ah * Bh + M.rr * M.ss * Ap * Bp - M.ass * (Ar * Bp + Ap * Br);
    return fmaf(M.f * lA, lB, e);
}

// plasma sample + transfer update at the new point (O5-O7 of DESIGN.md), HARM primitives [A16], constant T_p/T_e
__device__ __forceinline__ bool transfer(const KPf& P, const Geomf& G, const float X[4], const float K[4], float h, float& I, float& tau) {
    float q[8];
    if (!grid2d_interp(P, X[1], X[2], q)) return false;
    if (!(q[0] > 1e-30f && q[0] < 1e30f)) return false;      // positive normal density only: MUFU.RCP flushes denormals, maps huge to 0
    Metf M;
    M.ss = G.s * G.s; M.ass = P.a * M.ss; M.Sig = fmaf(G.r, G.r, P.a2 * G.c * G.c); M.rr = fmaf(G.r, G.r, P.a2);
    M.f = 2.0f * P.m * G.r * rcpf(M.Sig);
    const float kt = K[0], kr = G.ex * K[1], kh = G.dth * K[2], kp = K[3];
    const float rho = q[0], uu = q[1];
    const float Ur = G.ex * q[2], Uh = G.dth * q[3], Up = q[4];
    const float Br = G.ex * q[5], Bh = G.dth * q[6], Bp = q[7];
    const float opf = 1.0f + M.f, ialpha = sqrtf(opf);
    const float qq = ks_dot(M, 0.0f, Ur, Uh, Up, 0.0f, Ur, Uh, Up);
    if (!(qq < 1e30f)) return false;                                            // infinite or NaN velocity in the cell: no plasma
    const float gam = sqrtf(1.0f + qq);
    const float ut = gam * ialpha, ur = fmaf(-gam * ialpha, M.f * rcpf(opf), Ur), uh = Uh, up = Up;
    const float bt = ks_dot(M, 0.0f, Br, Bh, Bp, ut, ur, uh, up);
    const float iut = rcpf(ut);
    const float pt = bt, pr = fmaf(bt, ur, Br) * iut, ph = fmaf(bt, uh, Bh) * iut, pp = fmaf(bt, up, Bp) * iut;
    const float ne = rho * P.ne_scale;                                          // Eq. 46
    const float bsq = ks_dot(M, pt, pr, ph, pp, pt, pr, ph, pp);
    const float B = sqrtf(fmaxf(bsq, 0.0f)) * P.B0;
    const float thetae = P.thetae_scale * (uu * rcpf(rho));
    const float nu_hat = -ks_dot(M, kt, kr, kh, kp, ut, ur, uh, up);            // Eq. 31
    const float cos_th = ks_dot(M, kt, kr, kh, kp, pt, pr, ph, pp) * rcpf(nu_hat * sqrtf(bsq));
    const float sin_th = (bsq > 0.0f) ? sqrtf(fmaxf(1.0f - cos_th * cos_th, 0.0f)) : 0.0f;
    // Eq. 42-45 with sqrt(2) pi [A12] and K_2 = 2 Theta^2
    const float nu = nu_hat * P.nu_obs;
    const float nu_c = (kEf / (2.0f * kPIf * kMEf * kCf)) * B;
    const float nu_s = (2.0f / 9.0f) * nu_c * thetae * thetae * sin_th;         // Eq. 44
    float j = 0.0f;
    if (nu_s > 0.0f && ne > 0.0f) {
        const float Xx = nu * rcpf(nu_s);
        const float s6 = cbrtf(sqrtf(Xx));
        const float term = fmaf(s6 * s6, s6, 1.8877486253633870f * s6);
        const float K2 = 2.0f * thetae * thetae;
        j = ne * (1.4142135623730951f * kPIf * kEf * kEf * nu_s / (3.0f * kCf * K2)) * term * term * expf(-s6 * s6);
    }
    const float x = (kHPLf / (kMEf * kCf * kCf)) * nu * rcpf(thetae);                // h nu / (m_e c^2 Theta)
    const float Bnu = (2.0f * kHPLf * nu * nu * nu / (kCf * kCf)) / expm1f(x);  // Eq. 45 (evaluated left to right: in range)
    const float alpha = (j > 0.0f && Bnu > 0.0f) ? j / Bnu : 0.0f;              // Kirchhoff
    const float dtau = nu_hat * alpha * P.Lcm * h;                              // Eq. 36
    const float w = (dtau > 0.0f) ? -expm1f(-dtau) / dtau : 1.0f;               // Eq. 35 [A9]
    I += (j / (nu_hat * nu_hat)) * P.Lcm * h * expf(-tau) * w;                  // Eq. 37 + 32
    tau += dtau;
    return true;
}

__device__ __forceinline__ bool finite_f(float v) { return (__float_as_int(v) & 0x7f800000) != 0x7f800000; }

}  // namespace f32

#ifndef RAPTOR_F32_CTAS_PER_SM
#define RAPTOR_F32_CTAS_PER_SM 4      // 16 warps per SM: 3.5 tiles per warp on a 512^2 image (8 CTAs: 1.7, a long tail)
#endif

__global__ void __launch_bounds__(128) k_render_f32(const __grid_constant__ KPf P, const RenderOut O) {
    using namespace f32;
    const int lane = threadIdx.x & 31;
    const int ntx = (P.nx + 7) >> 3;
    unsigned long long steps = 0, sampled = 0, rays = 0;
    for (;;) {
        unsigned int tile = 0;
        if (lane == 0) tile = atomicAdd(O.queue, 1u);
        tile = __shfl_sync(0xffffffffu, tile, 0);
        if (tile >= O.ntiles) break;
        tile = O.tile_offset + tile * O.tile_stride;
        float alpha, beta;
        long long pix;
        bool active;
        if (O.alpha) {
            pix = (long long)tile * 32 + lane;
            active = pix < O.nrays;
            alpha = active ? (float)O.alpha[pix] : 0.0f;
            beta = active ? (float)O.beta[pix] : 0.0f;
        } else {
            // tile order (O.order, built at raptor_create / raptor_set_shard): by the impact parameter of the tile centre,
            // nearest first: the longest rays (photon ring; under the step rule of Eq. 21-24 everything near the hole)
            // start first and the launch ends on the uniform outer tiles instead of waiting for a late long tile
            const unsigned t = __ldg(O.order + tile);
            const int ty = (int)(t / (unsigned)ntx), tx = (int)(t - (unsigned)ty * (unsigned)ntx);
            const int ix = (tx << 3) + (lane & 7), iy = (ty << 2) + (lane >> 3);
            active = ix < P.nx && iy < P.ny;
            alpha = ((float)ix + 0.5f) * P.fov / (float)P.nx - 0.5f * P.fov;       // pixel centres [A4b]
            beta = ((float)iy + 0.5f) * P.fov / (float)P.ny - 0.5f * P.fov;
            pix = (long long)iy * P.nx + ix;
        }
        if (active) {
            float X[4], K[4], I = 0.0f, tau = 0.0f;
            camera_ray(P, alpha, beta, X, K);
            int n = 0, ns = 0, st = S_RUNNING;
            Geomf G;
            geom_eval(P, X[1], X[2], G);
            for (;;) {
                if (G.r < P.r_in) { st = S_CAPTURED; break; }                     // [A7]
                if (G.r > P.r_out) { st = S_ESCAPED; break; }
                if (n >= P.max_steps) { st = S_MAXSTEPS; break; }
                if (P.use_tau_cutoff && tau > P.tau_cutoff) { st = S_THICK; break; }
                const float h = step_size(P, X[2], K[1], K[2], K[3]);
                const float dl = -h, hl = 0.5f * dl;                               // backward [A2]
                // "RK2" of Table B.1 = explicit midpoint [A17]
                float f0, f1, f2, f3, k0, k1, k2, k3;
                geodesic_rhs(P, G, K[0], K[1], K[2], K[3], f0, f1, f2, f3);
                k0 = fmaf(hl, f0, K[0]); k1 = fmaf(hl, f1, K[1]); k2 = fmaf(hl, f2, K[2]); k3 = fmaf(hl, f3, K[3]);
                Geomf Gm;
                geom_eval(P, fmaf(hl, K[1], X[1]), fmaf(hl, K[2], X[2]), Gm);
                geodesic_rhs(P, Gm, k0, k1, k2, k3, f0, f1, f2, f3);
                X[0] = fmaf(dl, k0, X[0]); X[1] = fmaf(dl, k1, X[1]); X[2] = fmaf(dl, k2, X[2]); X[3] = fmaf(dl, k3, X[3]);
                K[0] = fmaf(dl, f0, K[0]); K[1] = fmaf(dl, f1, K[1]); K[2] = fmaf(dl, f2, K[2]); K[3] = fmaf(dl, f3, K[3]);
                ++n;
                const bool fin = finite_f(X[0]) & finite_f(X[1]) & finite_f(X[2]) & finite_f(X[3]) &
                                 finite_f(K[0]) & finite_f(K[1]) & finite_f(K[2]) & finite_f(K[3]);
                if (!fin) { st = S_NONFINITE; break; }
                geom_eval(P, X[1], X[2], G);
                if (G.r >= P.r_in && G.r <= P.r_out)                               // [A8] end-point sample
                    ns += transfer(P, G, X, K, h, I, tau) ? 1 : 0;
            }
            steps += (unsigned)n; sampled += (unsigned)ns; rays += 1;
            if (O.image) O.image[pix] = (double)I;
            if (O.tau) O.tau[pix] = (double)tau;
            if (O.status) O.status[pix] = st;
            if (O.nsteps) O.nsteps[pix] = n;
            if (O.XK) {
#pragma unroll
                for (int i = 0; i < 4; ++i) { O.XK[pix * 8 + i] = (double)X[i]; O.XK[pix * 8 + 4 + i] = (double)K[i]; }
            }
        }
        __syncwarp();
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        steps += __shfl_down_sync(0xffffffffu, steps, o);
        sampled += __shfl_down_sync(0xffffffffu, sampled, o);
        rays += __shfl_down_sync(0xffffffffu, rays, o);
    }
    if (lane == 0) {
        atomicAdd(O.counters + 0, steps);
        atomicAdd(O.counters + 1, sampled);
        atomicAdd(O.counters + 2, rays);
    }
}

// float -> float conversion of a float64 grid (once per upload): the values the float oracle reads, (float)double
__global__ void k_grid_to_f32(const double* __restrict__ src, float* __restrict__ dst, size_t n) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = (float)src[i];
}

cudaError_t launch_grid_to_f32(const double* d_src, float* d_dst, size_t n, cudaStream_t stream) {
    k_grid_to_f32<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(d_src, d_dst, n);
    return cudaGetLastError();
}

cudaError_t launch_render_f32(const KPf& P, const RenderOut& O, int sm_count, cudaStream_t stream) {
    const int block = 128, warps = block / 32;
    int per_sm = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_render_f32, block, 0);
    if (e != cudaSuccess) return e;
    if (per_sm > RAPTOR_F32_CTAS_PER_SM) per_sm = RAPTOR_F32_CTAS_PER_SM;
    if (per_sm < 1) per_sm = 1;
    long long want = ((long long)O.ntiles + warps - 1) / warps;
    int grid = sm_count * per_sm;
    if (want < grid) grid = (int)(want > 0 ? want : 1);
    k_render_f32<<<grid, block, 0, stream>>>(P, O);
    return cudaGetLastError();
}

}  // namespace raptor
