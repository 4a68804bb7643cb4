// raptor_kernels.cu -- the fused geodesic + radiative-transfer kernel and its satellites (sm_100a).
//
// Design: one ray per thread with the whole state in registers; persistent
// warps pull 8x4-pixel tiles from a global atomic counter (work queue at warp granularity: a warp's
// 32 rays are image neighbours, so they stay in lock-step through vacuum / plasma and end within a
// few steps of each other, while the queue absorbs the 2x spread in ray length between tiles);
// the geometry of a point (exp, sincos) is evaluated once and shared by the transfer update, the
// termination test, the step rule and RK4 stage 1; multi-frequency I/tau live in shared memory.
#include <cuda_runtime.h>
#include <stdint.h>

#include "raptor_device.cuh"
#include "raptor_kernels.h"

namespace raptor {

#ifndef RAPTOR_BLOCK
#define RAPTOR_BLOCK 128
#endif
#ifndef RAPTOR_MIN_BLOCKS
#define RAPTOR_MIN_BLOCKS 3
#endif

// --------------------------------------------------------------------------------------------
// One ray (O4 of DESIGN.md).  I/tau access is abstracted: registers (single frequency) or shared memory.
// --------------------------------------------------------------------------------------------
template <int MODEL, bool H1, bool MULTI>
__device__ __forceinline__ void trace_ray(const KP& P, double alpha, double beta, double* __restrict__ sI,
                                          double* __restrict__ sTau, int sstride, double& I0, double& tau0,
                                          double X[4], double K[4], int& status, int& nsteps, int& nsampled) {
    camera_ray(P, alpha, beta, X, K);
    double I = 0.0, tau = 0.0;
    if (MULTI) {
        for (int k = 0; k < P.n_freq; ++k) { sI[k * sstride] = 0.0; sTau[k * sstride] = 0.0; }
    }
    int n = 0, ns = 0, st = S_RUNNING;
    Geom G;
    geom_eval<H1>(P, X[1], X[2], G);
    for (;;) {
        if (G.r < P.r_in) { st = S_CAPTURED; break; }                         // [A7]
        if (G.r > P.r_out) { st = S_ESCAPED; break; }
        if (n >= P.max_steps) { st = S_MAXSTEPS; break; }
        if (P.use_tau_cutoff) {
            double tmin = tau;
            if (MULTI) {
                tmin = sTau[0];
                for (int k = 1; k < P.n_freq; ++k) tmin = fmin(tmin, sTau[k * sstride]);
            }
            if (tmin > P.tau_cutoff) { st = S_THICK; break; }
        }
        const double h = step_size(P, G, X[2], K[1], K[2], K[3]);
        const double dl = -h;                                                  // backward [A2]
        // ---- RK4, Eq. 7-16 -------------------------------------------------
        double f0, f1, f2, f3;
        double a0, a1, a2, a3;          // sum of stage accelerations  (f_1 + 2 f_2 + 2 f_3 + f_4)
        double b0, b1, b2, b3;          // sum of stage wavevectors    (k_1 + 2 k_2 + 2 k_3 + k_4)
        double k0, k1, k2, k3;          // stage wavevector
        const double hl = 0.5 * dl;
        geodesic_rhs(P, G, K[0], K[1], K[2], K[3], f0, f1, f2, f3);            // stage 1 at (X, K)
        a0 = f0; a1 = f1; a2 = f2; a3 = f3;
        b0 = K[0]; b1 = K[1]; b2 = K[2]; b3 = K[3];
        Geom Gs;
        // stage 2 at X + C1x/2, K + C1k/2
        k0 = fma(hl, f0, K[0]); k1 = fma(hl, f1, K[1]); k2 = fma(hl, f2, K[2]); k3 = fma(hl, f3, K[3]);
        geom_shift<H1>(P, G, X[1], X[2], hl * K[1], hl * K[2], Gs);
        geodesic_rhs(P, Gs, k0, k1, k2, k3, f0, f1, f2, f3);
        a0 = fma(2.0, f0, a0); a1 = fma(2.0, f1, a1); a2 = fma(2.0, f2, a2); a3 = fma(2.0, f3, a3);
        b0 = fma(2.0, k0, b0); b1 = fma(2.0, k1, b1); b2 = fma(2.0, k2, b2); b3 = fma(2.0, k3, b3);
        // stage 3 at X + C2x/2, K + C2k/2   (C2x = dl * stage-2 wavevector)
        {
            const double d1 = hl * k1, d2 = hl * k2;
            k0 = fma(hl, f0, K[0]); k1 = fma(hl, f1, K[1]); k2 = fma(hl, f2, K[2]); k3 = fma(hl, f3, K[3]);
            geom_shift<H1>(P, G, X[1], X[2], d1, d2, Gs);
        }
        geodesic_rhs(P, Gs, k0, k1, k2, k3, f0, f1, f2, f3);
        a0 = fma(2.0, f0, a0); a1 = fma(2.0, f1, a1); a2 = fma(2.0, f2, a2); a3 = fma(2.0, f3, a3);
        b0 = fma(2.0, k0, b0); b1 = fma(2.0, k1, b1); b2 = fma(2.0, k2, b2); b3 = fma(2.0, k3, b3);
        // stage 4 at X + C3x, K + C3k
        {
            const double d1 = dl * k1, d2 = dl * k2;
            k0 = fma(dl, f0, K[0]); k1 = fma(dl, f1, K[1]); k2 = fma(dl, f2, K[2]); k3 = fma(dl, f3, K[3]);
            geom_shift<H1>(P, G, X[1], X[2], d1, d2, Gs);
        }
        geodesic_rhs(P, Gs, k0, k1, k2, k3, f0, f1, f2, f3);
        a0 += f0; a1 += f1; a2 += f2; a3 += f3;
        b0 += k0; b1 += k1; b2 += k2; b3 += k3;
        const double d6 = dl * (1.0 / 6.0);
        const double x1_old = X[1], x2_old = X[2];
        X[0] = fma(d6, b0, X[0]); X[1] = fma(d6, b1, X[1]); X[2] = fma(d6, b2, X[2]); X[3] = fma(d6, b3, X[3]);   // Eq. 15
        K[0] = fma(d6, a0, K[0]); K[1] = fma(d6, a1, K[1]); K[2] = fma(d6, a2, K[2]); K[3] = fma(d6, a3, K[3]);   // Eq. 16
        ++n;
        bool fin = is_finite_bits(X[0]) & is_finite_bits(X[1]) & is_finite_bits(X[2]) & is_finite_bits(X[3]) &
                   is_finite_bits(K[0]) & is_finite_bits(K[1]) & is_finite_bits(K[2]) & is_finite_bits(K[3]);
        if (!fin) { st = S_NONFINITE; break; }
        // ---- new point: geometry shared by transfer, termination, step rule and the next stage 1 ----
        // incremental from the old base; re-evaluated from scratch every 16th step so that the round-off of
        // the increments cannot accumulate (n is warp-uniform: all lanes of a tile start together)
        if ((n & 15) == 0) geom_eval<H1>(P, X[1], X[2], G);
        else { Gs = G; geom_shift<H1>(P, Gs, x1_old, x2_old, d6 * b1, d6 * b2, G); }
        if (MODEL != M_VACUUM && G.r >= P.r_in && G.r <= P.r_out) {            // [A8] end-point sample
            Plasma pl;
            if (plasma_sample<MODEL>(P, G, X, K[0], G.ex * K[1], G.dth * K[2], K[3], pl)) {
                ++ns;
                EmisConst E;
                emis_prepare(P, pl, h, E);
                if (MULTI) {
                    for (int k = 0; k < P.n_freq; ++k) {
                        double Ik = sI[k * sstride], tk = sTau[k * sstride];
                        transfer_one(pl, E, __ldg(P.freq + k), Ik, tk);
                        sI[k * sstride] = Ik; sTau[k * sstride] = tk;
                    }
                } else {
                    transfer_one(pl, E, __ldg(P.freq), I, tau);
                }
            }
        }
    }
    I0 = I; tau0 = tau;
    status = st; nsteps = n; nsampled = ns;
}

// --------------------------------------------------------------------------------------------
// Persistent-warp driver: tiles of 8x4 pixels (render) or 32 consecutive rays (trace) from a global queue.
// --------------------------------------------------------------------------------------------
template <int MODEL, bool H1, bool MULTI>
__global__ void __launch_bounds__(RAPTOR_BLOCK, RAPTOR_MIN_BLOCKS)
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
            const int ty = tile / ntx, tx = tile - ty * ntx;
            const int ix = (tx << 3) + (lane & 7), iy = (ty << 2) + (lane >> 3);
            active = ix < P.nx && iy < P.ny;
            alpha = fma((double)ix + 0.5, P.pix_dx, -0.5 * P.fov);             // pixel centres [A4b]
            beta = fma((double)iy + 0.5, P.pix_dy, -0.5 * P.fov);
            pix = (long long)iy * P.nx + ix;
        }
        if (active) {
            double X[4], K[4], I0, tau0;
            int status, n, ns;
            trace_ray<MODEL, H1, MULTI>(P, alpha, beta, sI, sTau, sstride, I0, tau0, X, K, status, n, ns);
            steps += (unsigned)n; sampled += (unsigned)ns; rays += 1;
            const size_t npix = O.alpha ? (size_t)O.nrays : (size_t)P.nx * P.ny;
            if (O.image) {
                if (MULTI) { for (int k = 0; k < P.n_freq; ++k) O.image[(size_t)k * npix + pix] = sI[k * sstride]; }
                else O.image[pix] = I0;
            }
            if (O.tau) {
                if (MULTI) { for (int k = 0; k < P.n_freq; ++k) O.tau[(size_t)k * npix + pix] = sTau[k * sstride]; }
                else O.tau[pix] = tau0;
            }
            if (O.status) O.status[pix] = status;
            if (O.nsteps) O.nsteps[pix] = n;
            if (O.XK) {
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

template <int MODEL, bool H1, bool MULTI>
static cudaError_t launch_one(const KP& P, const RenderOut& O, int grid, cudaStream_t stream) {
    size_t smem = MULTI ? (size_t)2 * P.n_freq * RAPTOR_BLOCK * sizeof(double) : 0;
    auto kern = k_render<MODEL, H1, MULTI>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    kern<<<grid, RAPTOR_BLOCK, smem, stream>>>(P, O);
    return cudaGetLastError();
}

template <int MODEL>
static cudaError_t launch_model(const KP& P, const RenderOut& O, bool h1, bool multi, int grid, cudaStream_t s) {
    if (h1) return multi ? launch_one<MODEL, true, true>(P, O, grid, s) : launch_one<MODEL, true, false>(P, O, grid, s);
    return multi ? launch_one<MODEL, false, true>(P, O, grid, s) : launch_one<MODEL, false, false>(P, O, grid, s);
}

cudaError_t launch_render(const KP& P, int model, const RenderOut& O, int sm_count, cudaStream_t stream) {
    const bool h1 = (P.omh == 0.0), multi = P.n_freq > 1;
    // persistent grid: RAPTOR_MIN_BLOCKS CTAs per SM (fewer when shared memory for I/tau limits residency)
    int per_sm = RAPTOR_MIN_BLOCKS;
    if (multi) {
        size_t smem = (size_t)2 * P.n_freq * RAPTOR_BLOCK * sizeof(double);
        int fit = (int)((220u * 1024u) / (smem + 1024));
        if (fit < 1) fit = 1;
        if (fit < per_sm) per_sm = fit;
    }
    long long want = ((long long)O.ntiles * 32 + RAPTOR_BLOCK - 1) / RAPTOR_BLOCK;
    int grid = sm_count * per_sm;
    if (want < grid) grid = (int)(want > 0 ? want : 1);
    switch (model) {
        case M_VACUUM: return launch_model<M_VACUUM>(P, O, h1, multi, grid, stream);
        case M_SPHERE: return launch_model<M_SPHERE>(P, O, h1, multi, grid, stream);
        case M_TORUS: return launch_model<M_TORUS>(P, O, h1, multi, grid, stream);
        case M_GRID2D: return launch_model<M_GRID2D>(P, O, h1, multi, grid, stream);
        case M_GRID3DT: return launch_model<M_GRID3DT>(P, O, h1, multi, grid, stream);
        case M_SLAB: return launch_model<M_SLAB>(P, O, h1, multi, grid, stream);
    }
    return cudaErrorInvalidValue;
}

// --------------------------------------------------------------------------------------------
// a7: flux reduction, deterministic (fixed chunking, fixed tree).  O8 of DESIGN.md.
// --------------------------------------------------------------------------------------------
constexpr int kFluxThreads = 256;
constexpr int kFluxChunk = 16384;

__global__ void __launch_bounds__(kFluxThreads) k_flux_partial(const double* __restrict__ image, size_t npix,
                                                               double* __restrict__ partial, int nchunks) {
    __shared__ double sh[kFluxThreads];
    const int k = blockIdx.y, chunk = blockIdx.x;
    const size_t lo = (size_t)chunk * kFluxChunk;
    const size_t hi = lo + kFluxChunk < npix ? lo + kFluxChunk : npix;
    const double* img = image + (size_t)k * npix;
    double acc = 0.0;
    for (size_t i = lo + threadIdx.x; i < hi; i += kFluxThreads) acc += img[i];
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int o = kFluxThreads / 2; o >= 32; o >>= 1) {
        if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x < 32) {
        double v = sh[threadIdx.x];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (threadIdx.x == 0) partial[(size_t)k * nchunks + chunk] = v;
    }
}

__global__ void __launch_bounds__(32) k_flux_final(const double* __restrict__ partial, int nchunks, double scale,
                                                   double* __restrict__ flux) {
    const int k = blockIdx.x;
    double acc = 0.0;
    for (int i = threadIdx.x; i < nchunks; i += 32) acc += partial[(size_t)k * nchunks + i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    if (threadIdx.x == 0) flux[k] = acc * scale;
}

int flux_chunks(size_t npix) { return (int)((npix + kFluxChunk - 1) / kFluxChunk); }

cudaError_t launch_flux(const double* d_image, size_t npix, int n_freq, double scale, double* d_partial,
                        double* d_flux, cudaStream_t stream) {
    const int nchunks = flux_chunks(npix);
    k_flux_partial<<<dim3(nchunks, n_freq), kFluxThreads, 0, stream>>>(d_image, npix, d_partial, nchunks);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    k_flux_final<<<n_freq, 32, 0, stream>>>(d_partial, nchunks, scale, d_flux);
    return cudaGetLastError();
}

// --------------------------------------------------------------------------------------------
// diagnostics: right-hand side at given points
// --------------------------------------------------------------------------------------------
template <bool H1>
__global__ void k_eval_rhs(const __grid_constant__ KP P, int n, const double* __restrict__ XK, double* __restrict__ f) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double* q = XK + (size_t)i * 8;
    Geom G;
    geom_eval<H1>(P, q[1], q[2], G);
    double f0, f1, f2, f3;
    geodesic_rhs(P, G, q[4], q[5], q[6], q[7], f0, f1, f2, f3);
    f[i * 4 + 0] = f0; f[i * 4 + 1] = f1; f[i * 4 + 2] = f2; f[i * 4 + 3] = f3;
}

cudaError_t launch_eval_rhs(const KP& P, int n, const double* d_XK, double* d_f, cudaStream_t stream) {
    int grid = (n + 127) / 128;
    if (P.omh == 0.0) k_eval_rhs<true><<<grid, 128, 0, stream>>>(P, n, d_XK, d_f);
    else k_eval_rhs<false><<<grid, 128, 0, stream>>>(P, n, d_XK, d_f);
    return cudaGetLastError();
}

// --------------------------------------------------------------------------------------------
// FP64 peak probe: 8 independent DFMA chains per thread
// --------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_fp64_peak(int iters, double seed, double* __restrict__ out) {
    double x0 = seed + threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    const double m = 0.999999, c = 1e-9;
#pragma unroll 4
    for (int i = 0; i < iters; ++i) {
        x0 = fma(x0, m, c); x1 = fma(x1, m, c); x2 = fma(x2, m, c); x3 = fma(x3, m, c);
        x4 = fma(x4, m, c); x5 = fma(x5, m, c); x6 = fma(x6, m, c); x7 = fma(x7, m, c);
    }
    double s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (s == 123.456) out[0] = s;      // never true; keeps the chains alive
}

cudaError_t launch_fp64_peak(int iters, int blocks, double* d_out, cudaStream_t stream) {
    k_fp64_peak<<<blocks, 256, 0, stream>>>(iters, 1.0, d_out);
    return cudaGetLastError();
}

}  // namespace raptor
