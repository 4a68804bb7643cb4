// raptor_render.cu -- the fused geodesic + radiative-transfer kernel k_render (sm_100a, FP64).
//
// Design: one ray per thread with the whole state in registers; persistent
// warps pull 8x4-pixel tiles from a global atomic counter (work queue at warp granularity: a warp's
// 32 rays are image neighbours, so they stay in lock-step through vacuum / plasma and end within a
// few steps of each other, while the queue absorbs the 2x spread in ray length between tiles);
// the geometry of a point (exp, sincos) is evaluated once and shared by the transfer update, the
// termination test, the step rule and RK4 stage 1; multi-frequency I/tau live in shared memory.
//
// Compiled once per plasma model (-DRAPTOR_MODEL=0..5, in parallel, see build.py) or, without the
// macro, for all six models in one translation unit.
#include <cuda_runtime.h>
#include <stdint.h>

#include "raptor_device.cuh"
#include "raptor_kernels.h"

namespace raptor {

#ifndef RAPTOR_REFRESH
#define RAPTOR_REFRESH 63      // library exp / sincos at the base point every (RAPTOR_REFRESH + 1)-th step
#endif

// --------------------------------------------------------------------------------------------
// One ray (O4 of DESIGN.md).  I/tau access is abstracted: registers (single frequency) or shared memory.
// FULLX: also integrate X^t and X^phi (needed by the 3-D / slow-light sampler and by the trace output);
// the metric does not depend on them, so for the other models they are dead and are not computed.
//
// RK4, Eq. 7-16, with y = (X, K), y' = (K, f(X, K)), step dl = -h [A2]:
//   stage wavevectors  k_2 = K + dl/2 f_1,  k_3 = K + dl/2 f_2,  k_4 = K + dl f_3
//   stage points       X + dl/2 K,  X + dl/2 k_2,  X + dl k_3
//   X' = X + dl/6 (K + 2 k_2 + 2 k_3 + k_4) = X + dl (K + dl/6 (f_1 + f_2 + f_3))
//   K' = K + dl/6 (f_1 + 2 f_2 + 2 f_3 + f_4)
// Only (x1, x2) enter f.  Their exp / sin / cos come incrementally (raptor_device.cuh): stage 2 and stage 4
// from the base point, stage 3 from stage 2 (offset (dl/2)^2 f_1) and the new base point from stage 4
// (offset dl^2/6 (f_1 - 2 f_2 + f_3)), both of which are second / third order small.
// --------------------------------------------------------------------------------------------
// MON: also evaluate the null condition g_mn k^m k^n (Eq. 4) at the new point of every step and keep
// its largest magnitude along the ray (8(a) a3 "null-condition check"); diagnostics, built with FULLX only.
// R0: the chart has r0 != 0 (A.10); every contract configuration has r0 = 0, for which r = e^x1 costs nothing.
template <int MODEL, bool H1, bool MULTI, bool FULLX, int INTEG, bool MON, bool R0>
__device__ __forceinline__ void trace_ray(const KP& P, double alpha, double beta, double t_cam, double* __restrict__ sI,
                                          double* __restrict__ sTau, int sstride, double& I0, double& tau0,
                                          double X[4], double K[4], int& status, int& nsteps, int& nsampled, double& null_max) {
    camera_ray(P, alpha, beta, X, K);
    X[0] = t_cam;
    double I = 0.0, tau = 0.0;
    if (MULTI) {
        for (int k = 0; k < P.n_freq; ++k) { sI[k * sstride] = 0.0; sTau[k * sstride] = 0.0; }
    }
    int n = 0, ns = 0, ncross = 0, st = S_RUNNING;
    double nmax = 0.0;
    // tau cut-off: the optical depths change on sampled steps only, so the comparison with the cut-off is made there
    // and the loop head tests a flag (same exit, same step count: the head tests run in the oracle's order)
    bool thick = P.use_tau_cutoff && 0.0 > P.tau_cutoff;
    Geom G;
    { Geom T; geom_eval_call<H1>(P.r0, P.omh, X[1], X[2], &T); G = T; }
    bool fin = true;                    // the state after the last step is finite
    for (;;) {
        // the exits of the loop as ONE branch (which of them it was is sorted out after the loop, in the order of [A7]:
        // non-finite state right after the step, then horizon, escape, step cap, optical-depth cap at the head of the
        // next iteration); r = r0 + e^x1 is positive (or +inf): compared on the integer pipe
        if (!fin | pos_lt(G.r, P.r_in) | pos_lt(P.r_out, G.r) | (n >= P.max_steps) | thick) break;
        const double h = step_size(P, G, X[2], K[1], K[2], K[3]);
        const double dl = -h;                                                  // backward [A2]
        double x1p = 0.0, x2p = 0.0, Kp[4] = {0.0, 0.0, 0.0, 0.0};             // thin disk: state before the step
        if (MODEL == M_DISK) { x1p = X[1]; x2p = X[2]; Kp[0] = K[0]; Kp[1] = K[1]; Kp[2] = K[2]; Kp[3] = K[3]; }
        const double hl = 0.5 * dl;
        Geom Gs;                        // geometry of the last stage point: the new base point is reached from it
        double t1, t2;                  // new point minus that stage point: x1 offset, x2 offset as an angle (shift_angle)
        if (INTEG == I_RK4) {
            double f0, f1, f2, f3;          // stage acceleration
            double k0, k1, k2, k3;          // stage wavevector
            double a0, a1, a2, a3;          // t, phi: f_1 + 2 f_2 + 2 f_3 + f_4; x1, x2: f_1 until the end
            double s0 = 0.0, s1, s2, s3 = 0.0;   // f_1 + f_2 + f_3   (components t, phi only with FULLX)
            Geom Gt;
            // stage 1 at (X, K)
            geodesic_rhs(P, G, K[0], K[1], K[2], K[3], f0, f1, f2, f3);
            a0 = f0; a1 = f1; a2 = f2; a3 = f3;
            // stage 2 at X + dl/2 K, K + dl/2 f_1
            k0 = fma(hl, f0, K[0]); k1 = fma(hl, f1, K[1]); k2 = fma(hl, f2, K[2]); k3 = fma(hl, f3, K[3]);
            // x2 offsets as angles (2 pi d2, or pi d2 for h = 1): ahl = c dl/2, al = c dl
            const double al = shift_angle<H1>(dl), ahl = 0.5 * al;
            const double d12 = hl * K[1], g22 = ahl * K[2];                        // stage-2 point minus X
            geom_shift<H1, R0>(P, G, X[1], X[2], d12, g22, Gs);
            // stage-3 point minus stage-2 point: dl/2 (k_2 - K) = (dl/2)^2 f_1
            const double e1 = fma(hl, k1, -d12), e2 = fma(ahl, k2, -g22);
            const double x1s2 = fma(hl, K[1], X[1]), x2s2 = fma(hl, K[2], X[2]);   // stage-2 point (library fallback only)
            geodesic_rhs(P, Gs, k0, k1, k2, k3, f0, f1, f2, f3);
            if (FULLX) { s0 = a0 + f0; s3 = a3 + f3; }
            s1 = a1 + f1; s2 = a2 + f2;
            a0 = fma(2.0, f0, a0); a3 = fma(2.0, f3, a3);
            // stage 3 at X + dl/2 k_2, K + dl/2 f_2
            k0 = fma(hl, f0, K[0]); k1 = fma(hl, f1, K[1]); k2 = fma(hl, f2, K[2]); k3 = fma(hl, f3, K[3]);
            geom_shift<H1, R0, false, true>(P, Gs, x1s2, x2s2, e1, e2, Gt);
            geodesic_rhs(P, Gt, k0, k1, k2, k3, f0, f1, f2, f3);
            if (FULLX) { s0 += f0; s3 += f3; }
            s1 += f1; s2 += f2;
            a0 = fma(2.0, f0, a0); a3 = fma(2.0, f3, a3);
            // stage 4 at X + dl k_3, K + dl f_3
            const double d14 = dl * k1, g24 = al * k2;                             // stage-4 point minus X
            geom_shift<H1, R0>(P, G, X[1], X[2], d14, g24, Gs);
            k0 = fma(dl, f0, K[0]); k1 = fma(dl, f1, K[1]); k2 = fma(dl, f2, K[2]); k3 = fma(dl, f3, K[3]);
            geodesic_rhs(P, Gs, k0, k1, k2, k3, f0, f1, f2, f3);
            // f_1 + 2 f_2 + 2 f_3 + f_4: t, phi accumulated; x1, x2 from the sum the position update needs anyway,
            // 2 (f_1 + f_2 + f_3) + (f_4 - f_1)
            a0 += f0; a3 += f3;
            a1 = fma(2.0, s1, f1 - a1); a2 = fma(2.0, s2, f2 - a2);
            const double d6 = dl * (1.0 / 6.0);
            const double w1 = fma(d6, s1, K[1]), w2 = fma(d6, s2, K[2]);           // Eq. 15: X' = X + dl (K + dl/6 S)
            // new point minus stage-4 point: dl (K + dl/6 S) - dl k_3
            t1 = fma(dl, w1, -d14); t2 = fma(al, w2, -g24);
            if (FULLX) { X[0] = fma(dl, fma(d6, s0, K[0]), X[0]); X[3] = fma(dl, fma(d6, s3, K[3]), X[3]); }
            X[1] = fma(dl, w1, X[1]); X[2] = fma(dl, w2, X[2]);
            K[0] = fma(d6, a0, K[0]); K[1] = fma(d6, a1, K[1]); K[2] = fma(d6, a2, K[2]); K[3] = fma(d6, a3, K[3]);   // Eq. 16
        } else if (INTEG == I_RK2) {
            // "RK2" of Table B.1, read as the explicit midpoint method [A17]
            double f0, f1, f2, f3, k0, k1, k2, k3;
            geodesic_rhs(P, G, K[0], K[1], K[2], K[3], f0, f1, f2, f3);
            k0 = fma(hl, f0, K[0]); k1 = fma(hl, f1, K[1]); k2 = fma(hl, f2, K[2]); k3 = fma(hl, f3, K[3]);
            const double d1 = hl * K[1], d2 = hl * K[2];
            geom_shift<H1, R0>(P, G, X[1], X[2], d1, shift_angle<H1>(d2), Gs);
            geodesic_rhs(P, Gs, k0, k1, k2, k3, f0, f1, f2, f3);
            // new point minus midpoint: dl k_mid - dl/2 K
            t1 = fma(dl, k1, -d1); t2 = shift_angle<H1>(fma(dl, k2, -d2));
            if (FULLX) { X[0] = fma(dl, k0, X[0]); X[3] = fma(dl, k3, X[3]); }
            X[1] = fma(dl, k1, X[1]); X[2] = fma(dl, k2, X[2]);
            K[0] = fma(dl, f0, K[0]); K[1] = fma(dl, f1, K[1]); K[2] = fma(dl, f2, K[2]); K[3] = fma(dl, f3, K[3]);
        } else {
            // velocity Verlet, Eq. 17-20; (dk/dl)_n from the current (x_n, k_n) [A23];
            // I_VERLET_C: Eq. 19 re-evaluated with k_{n+1,p} = k_{n+1}, then Eq. 20 again
            double f0, f1, f2, f3, g0, g1, g2, g3, p0, p1, p2, p3;
            geodesic_rhs(P, G, K[0], K[1], K[2], K[3], f0, f1, f2, f3);
            const double hd2 = 0.5 * (dl * dl);
            t1 = fma(hd2, f1, dl * K[1]); t2 = fma(hd2, f2, dl * K[2]);                        // Eq. 17
            if (FULLX) { X[0] += fma(hd2, f0, dl * K[0]); X[3] += fma(hd2, f3, dl * K[3]); }
            X[1] += t1; X[2] += t2;
            p0 = fma(dl, f0, K[0]); p1 = fma(dl, f1, K[1]); p2 = fma(dl, f2, K[2]); p3 = fma(dl, f3, K[3]);   // Eq. 18
            geom_shift<H1, R0, true>(P, G, X[1], X[2], t1, shift_angle<H1>(t2), Gs);
            geodesic_rhs(P, Gs, p0, p1, p2, p3, g0, g1, g2, g3);                                // Eq. 19
            p0 = fma(hl, f0 + g0, K[0]); p1 = fma(hl, f1 + g1, K[1]);                           // Eq. 20
            p2 = fma(hl, f2 + g2, K[2]); p3 = fma(hl, f3 + g3, K[3]);
            if (INTEG == I_VERLET_C) {
                geodesic_rhs(P, Gs, p0, p1, p2, p3, g0, g1, g2, g3);
                p0 = fma(hl, f0 + g0, K[0]); p1 = fma(hl, f1 + g1, K[1]);
                p2 = fma(hl, f2 + g2, K[2]); p3 = fma(hl, f3 + g3, K[3]);
            }
            K[0] = p0; K[1] = p1; K[2] = p2; K[3] = p3;
            t1 = 0.0; t2 = 0.0;                                                                 // Gs is the new point
        }
        ++n;
        // RK4: a non-finite X' = X + dl (K + dl/6 S) means a non-finite S (K was finite on entry), and then K' = K + dl/6 (2 S + f_4 - f_1)
        // (or its t, phi form) is non-finite too: testing K' alone is the same test
        fin = is_finite_bits(K[0]) & is_finite_bits(K[1]) & is_finite_bits(K[2]) & is_finite_bits(K[3]);
        if (INTEG != I_RK4) {
            fin = fin & is_finite_bits(X[1]) & is_finite_bits(X[2]);
            if (FULLX) fin = fin & is_finite_bits(X[0]) & is_finite_bits(X[3]);
        }
        // a non-finite state leaves the loop at its head; until then it must not be sampled or monitored
        // ---- new point: geometry shared by transfer, termination, step rule and the next stage 1 ----
        // incremental from stage 4; re-evaluated with the library functions every (RAPTOR_REFRESH+1)-th step so
        // that the round-off of the increments cannot accumulate (n is warp-uniform: a tile's lanes start together)
        if ((n & RAPTOR_REFRESH) == 0) { Geom T; geom_eval_call<H1>(P.r0, P.omh, X[1], X[2], &T); G = T; }
        else if (INTEG == I_VERLET || INTEG == I_VERLET_C) G = Gs;
        else geom_shift<H1, R0, true, true>(P, Gs, X[1], X[2], t1, t2, G);                 // t2: an angle
        if (MON && fin) {
            Met M;
            met_eval(P, G, M);
            const double kr = G.ex * K[1], kh = G.dth * K[2];
            nmax = fmax(nmax, fabs(ks_dot(M, K[0], kr, kh, K[3], K[0], kr, kh, K[3])));
        }
        if (MODEL == M_DISK) {
            // I = sum of g^p / r^2 over the counted crossings, tau = g of the first counted one
            double dI, gg;
            bool counted;
            if (fin && disk_crossing(P, x1p, x2p, Kp, X, K, ncross + 1, dI, gg, counted)) {
                ++ncross;
                if (counted) { I += dI; if (ns == 0) tau = gg; ++ns; if (P.use_tau_cutoff) thick = tau > P.tau_cutoff; }
            }
        } else
        if (MODEL != M_VACUUM && fin && !pos_lt(G.r, P.r_in) && !pos_lt(P.r_out, G.r)) {   // [A8] end-point sample
            Plasma pl;
            if (plasma_sample<MODEL>(P, G, X, K[0], G.ex * K[1], G.dth * K[2], K[3], pl)) {
                ++ns;
                EmisConst E;
                emis_prepare(P, pl, h, E);
                if (MULTI) {
                    // two frequencies per iteration: their (branch-free) updates are independent chains
                    const int nf = P.n_freq;
                    const double* __restrict__ fq = P.freq;
                    int k = 0;
                    for (; k + 1 < nf; k += 2) {
                        double Ia = sI[k * sstride], ta = sTau[k * sstride];
                        double Ib = sI[(k + 1) * sstride], tb = sTau[(k + 1) * sstride];
                        transfer_one(pl, E, __ldg(fq + k), __ldg(fq + nf + k), __ldg(fq + 2 * nf + k), Ia, ta);
                        transfer_one(pl, E, __ldg(fq + k + 1), __ldg(fq + nf + k + 1), __ldg(fq + 2 * nf + k + 1), Ib, tb);
                        sI[k * sstride] = Ia; sTau[k * sstride] = ta;
                        sI[(k + 1) * sstride] = Ib; sTau[(k + 1) * sstride] = tb;
                    }
                    if (k < nf) {
                        double Ia = sI[k * sstride], ta = sTau[k * sstride];
                        transfer_one(pl, E, __ldg(fq + k), __ldg(fq + nf + k), __ldg(fq + 2 * nf + k), Ia, ta);
                        sI[k * sstride] = Ia; sTau[k * sstride] = ta;
                    }
                } else {
                    transfer_one(pl, E, __ldg(P.freq), __ldg(P.freq + 1), __ldg(P.freq + 2), I, tau);
                }
                if (P.use_tau_cutoff) {
                    double tmin = tau;
                    if (MULTI) {
                        tmin = sTau[0];
                        for (int k = 1; k < P.n_freq; ++k) tmin = fmin(tmin, sTau[k * sstride]);
                    }
                    thick = tmin > P.tau_cutoff;                               // false for a NaN
                }
            }
        }
    }
    st = !fin ? S_NONFINITE : pos_lt(G.r, P.r_in) ? S_CAPTURED : pos_lt(P.r_out, G.r) ? S_ESCAPED
       : n >= P.max_steps ? S_MAXSTEPS : S_THICK;
    I0 = I; tau0 = tau; null_max = nmax;
    status = st; nsteps = n; nsampled = ns;
}

// --------------------------------------------------------------------------------------------
// Persistent-warp driver: tiles of 8x4 pixels (render) or 32 consecutive rays (trace) from a global queue.
// --------------------------------------------------------------------------------------------
template <int MODEL, bool H1, bool MULTI, bool FULLX, int INTEG, bool MON, bool R0>
__global__ void __launch_bounds__(MULTI ? RAPTOR_BLOCK_MULTI : RAPTOR_BLOCK, MULTI ? (RAPTOR_BLOCK * RAPTOR_MIN_BLOCKS) / RAPTOR_BLOCK_MULTI : RAPTOR_MIN_BLOCKS)
k_render(const __grid_constant__ KP P, const RenderOut O) {
    extern __shared__ double smem[];
    const int lane = threadIdx.x & 31;
    double* sI = MULTI ? smem + threadIdx.x : nullptr;                         // [k][thread]: conflict-free
    double* sTau = MULTI ? smem + (size_t)P.n_freq * blockDim.x + threadIdx.x : nullptr;
    const int sstride = blockDim.x;
    const int ntx = (P.nx + 7) >> 3;
    unsigned long long steps = 0, sampled = 0, rays = 0;
    for (;;) {
        unsigned int tile = 0;
        if (lane == 0) tile = atomicAdd(O.queue, 1u);
        tile = __shfl_sync(0xffffffffu, tile, 0);
        if (tile >= O.ntiles) break;
        // light-curve batch: O.frames images of the same scene at camera times t_cam0 + frame dt_frame in one launch
        unsigned int frame = 0;
        double t_cam = P.t_cam;
        if (O.frames > 1) {
            frame = tile / O.tiles_per_frame;
            tile -= frame * O.tiles_per_frame;
            t_cam = fma((double)frame, O.dt_frame, O.t_cam0);
        }
        tile = O.tile_offset + tile * O.tile_stride;                           // multi-GPU shard: interleaved tiles
        double alpha, beta;
        long long pix;
        bool active;
        if (O.alpha) {                                                         // trace mode: explicit impact parameters
            pix = (long long)tile * 32 + lane;
            active = pix < O.nrays;
            alpha = active ? O.alpha[pix] : 0.0;
            beta = active ? O.beta[pix] : 0.0;
        } else {
            // tile order (O.order, built at raptor_create / raptor_set_shard): by the impact parameter of the tile centre,
            // nearest first: the longest rays (photon ring; under the step rule of Eq. 21-24 everything near the hole)
            // start first and the launch ends on the uniform outer tiles instead of waiting for a late long tile
            const unsigned t = __ldg(O.order + tile);
            const int ty = (int)(t / (unsigned)ntx), tx = (int)(t - (unsigned)ty * (unsigned)ntx);
            const int ix = (tx << 3) + (lane & 7), iy = (ty << 2) + (lane >> 3);
            active = ix < P.nx && iy < P.ny;
            alpha = fma((double)ix + 0.5, P.pix_dx, -0.5 * P.fov);             // pixel centres [A4b]
            beta = fma((double)iy + 0.5, P.pix_dy, -0.5 * P.fov);
            pix = (long long)iy * P.nx + ix;
        }
        if (active) {
            double X[4], K[4], I0, tau0, nmax;
            int status, n, ns;
            trace_ray<MODEL, H1, MULTI, FULLX, INTEG, MON, R0>(P, alpha, beta, t_cam, sI, sTau, sstride, I0, tau0, X, K, status, n, ns, nmax);
            steps += (unsigned)n; sampled += (unsigned)ns; rays += 1;
            const size_t npix = O.alpha ? (size_t)O.nrays : (size_t)P.nx * P.ny;
            if (O.image) {
                double* img = O.image + (size_t)frame * P.n_freq * npix;
                if (MULTI) { for (int k = 0; k < P.n_freq; ++k) img[(size_t)k * npix + pix] = sI[k * sstride]; }
                else img[pix] = I0;
            }
            if (O.tau) {
                if (MULTI) { for (int k = 0; k < P.n_freq; ++k) O.tau[(size_t)k * npix + pix] = sTau[k * sstride]; }
                else O.tau[pix] = tau0;
            }
            if (MON && O.null_max) O.null_max[pix] = nmax;
            if (O.status) O.status[pix] = status;
            if (O.nsteps) O.nsteps[pix] = n;
            if (FULLX && O.XK) {
#pragma unroll
                for (int i = 0; i < 4; ++i) { O.XK[pix * 8 + i] = X[i]; O.XK[pix * 8 + 4 + i] = K[i]; }
            }
        }
        __syncwarp();
    }
    // counters: warp reduce, one atomic per warp
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

template <int MODEL, bool H1, bool MULTI, bool FULLX, int INTEG, bool MON, bool R0>
static cudaError_t launch_one(const KP& P, const RenderOut& O, int grid, int block, cudaStream_t stream) {
    size_t smem = MULTI ? (size_t)2 * P.n_freq * block * sizeof(double) : 0;
    auto kern = k_render<MODEL, H1, MULTI, FULLX, INTEG, MON, R0>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    kern<<<grid, block, smem, stream>>>(P, O);
    return cudaGetLastError();
}

template <int MODEL, bool FULLX, int INTEG, bool MON, bool R0>
static cudaError_t launch_hm(const KP& P, const RenderOut& O, bool h1, bool multi, int grid, int block, cudaStream_t s) {
    if (h1) return multi ? launch_one<MODEL, true, true, FULLX, INTEG, MON, R0>(P, O, grid, block, s) : launch_one<MODEL, true, false, FULLX, INTEG, MON, R0>(P, O, grid, block, s);
    return multi ? launch_one<MODEL, false, true, FULLX, INTEG, MON, R0>(P, O, grid, block, s) : launch_one<MODEL, false, false, FULLX, INTEG, MON, R0>(P, O, grid, block, s);
}

template <int MODEL, int INTEG>
cudaError_t launch_model(const KP& P, const RenderOut& O, bool h1, bool multi, bool fullx, int grid, int block, cudaStream_t s) {
    // The lean kernels (no X^t / X^phi, r0 = 0) serve RK4 on the models that do not read t, phi; everything else is
    // FULLX: the 3-D / slow-light sampler reads X^t, X^phi, the trace output wants them, and the second-order
    // integrators (8(f) f1) are built in that form only.  A chart with r0 != 0 and the per-step null monitor run on the
    // general kernels (FULLX, R0; MON only there).
    if (O.null_max) return launch_hm<MODEL, true, INTEG, true, true>(P, O, h1, multi, grid, block, s);
    if (P.r0_nz) return launch_hm<MODEL, true, INTEG, false, true>(P, O, h1, multi, grid, block, s);
    if (MODEL == M_GRID3DT || fullx || INTEG != I_RK4) return launch_hm<MODEL, true, INTEG, false, false>(P, O, h1, multi, grid, block, s);
    return launch_hm<MODEL, MODEL == M_GRID3DT || INTEG != I_RK4, INTEG, false, false>(P, O, h1, multi, grid, block, s);
}

// one translation unit per (plasma model, integrator): -DRAPTOR_MODEL=m -DRAPTOR_INTEG=i (build.py, in parallel);
// without the macros, everything in this one
#define RAPTOR_INST(M, I) template cudaError_t launch_model<M, I>(const KP&, const RenderOut&, bool, bool, bool, int, int, cudaStream_t);
#if defined(RAPTOR_MODEL) && defined(RAPTOR_INTEG)
RAPTOR_INST(RAPTOR_MODEL, RAPTOR_INTEG)
#else
#define RAPTOR_INST_ALL(M) RAPTOR_INST(M, I_RK4) RAPTOR_INST(M, I_VERLET) RAPTOR_INST(M, I_VERLET_C) RAPTOR_INST(M, I_RK2)
RAPTOR_INST_ALL(M_VACUUM) RAPTOR_INST_ALL(M_SPHERE) RAPTOR_INST_ALL(M_TORUS)
RAPTOR_INST_ALL(M_GRID2D) RAPTOR_INST_ALL(M_GRID3DT) RAPTOR_INST_ALL(M_SLAB) RAPTOR_INST_ALL(M_DISK)
#endif

}  // namespace raptor
