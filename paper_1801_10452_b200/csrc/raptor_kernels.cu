// raptor_kernels.cu -- launch geometry of the ray kernel (raptor_render.cu) and the satellite kernels:
// deterministic flux reduction (a7), right-hand-side diagnostics, FP64 peak probe (sm_100a).
#include <cuda_runtime.h>
#include <stdint.h>

#include "raptor_device.cuh"
#include "raptor_kernels.h"

namespace raptor {

// Launch shape of the persistent ray kernel.  Single frequency: RAPTOR_MIN_BLOCKS CTAs of RAPTOR_BLOCK threads per
// SM (16 warps, the register limit at 128 registers).  Several frequencies: I/tau take 16 n_freq bytes of shared
// memory per thread, so the (CTAs per SM, warps per CTA) pair with the most resident warps that fits 228 KB per SM
// (1 KB reserved per CTA) and 227 KB per CTA is used -- e.g. 2 x 7 warps at 32 frequencies: 148 x 14 = 2072 warp
// slots, so the 2048 tiles of a 256^2 image (C3) run as a single wave.
static void launch_shape(int n_freq, int& ctas_per_sm, int& warps_per_cta) {
    ctas_per_sm = RAPTOR_MIN_BLOCKS; warps_per_cta = RAPTOR_BLOCK / 32;
    if (n_freq <= 1) return;
    const long long per_warp = 32ll * 16 * n_freq;
    int best = 0;
    for (int c = 1; c <= RAPTOR_MIN_BLOCKS; ++c) {
        long long w = ((228ll * 1024) / c - 1024) / per_warp;
        if (w * per_warp > 227ll * 1024) w = (227ll * 1024) / per_warp;
        if (w > RAPTOR_BLOCK_MULTI / 32) w = RAPTOR_BLOCK_MULTI / 32;
        if (c * w > 16) w = 16 / c;
        if (w >= 1 && c * (int)w >= best) { best = c * (int)w; ctas_per_sm = c; warps_per_cta = (int)w; }
    }
    if (best == 0) { ctas_per_sm = 1; warps_per_cta = 1; }
}

cudaError_t launch_render(const KP& P, int model, const RenderOut& O, int sm_count, cudaStream_t stream) {
    const bool h1 = (P.omh == 0.0), multi = P.n_freq > 1;
    int per_sm, warps;
    launch_shape(P.n_freq, per_sm, warps);
    const int block = warps * 32;
    long long want = ((long long)O.ntiles + warps - 1) / warps;
    int grid = sm_count * per_sm;
    if (want < grid) grid = (int)(want > 0 ? want : 1);
    const bool fullx = O.XK != nullptr || O.null_max != nullptr;
#define RAPTOR_CASE_I(M, I) case I: return launch_model<M, I>(P, O, h1, multi, fullx, grid, block, stream);
#define RAPTOR_CASE_M(M)                                                                          \
    case M:                                                                                       \
        switch (P.integrator) {                                                                   \
            RAPTOR_CASE_I(M, I_RK4) RAPTOR_CASE_I(M, I_VERLET) RAPTOR_CASE_I(M, I_VERLET_C) RAPTOR_CASE_I(M, I_RK2) \
        }                                                                                         \
        break;
    switch (model) {
        RAPTOR_CASE_M(M_VACUUM) RAPTOR_CASE_M(M_SPHERE) RAPTOR_CASE_M(M_TORUS)
        RAPTOR_CASE_M(M_GRID2D) RAPTOR_CASE_M(M_GRID3DT) RAPTOR_CASE_M(M_SLAB) RAPTOR_CASE_M(M_DISK)
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

// Line profile of the thin disk (Fig. 6): bin b of [g_min, g_max) collects I of the pixels whose
// redshift factor falls into it.  Same fixed chunking and tree as the flux => bit-reproducible.
__global__ void __launch_bounds__(kFluxThreads) k_profile_partial(const double* __restrict__ image, const double* __restrict__ red,
                                                                  size_t npix, double g_min, double inv_dg, int nbins,
                                                                  double* __restrict__ partial, int nchunks) {
    __shared__ double sh[kFluxThreads];
    const int b = blockIdx.y, chunk = blockIdx.x;
    const size_t lo = (size_t)chunk * kFluxChunk;
    const size_t hi = lo + kFluxChunk < npix ? lo + kFluxChunk : npix;
    double acc = 0.0;
    for (size_t i = lo + threadIdx.x; i < hi; i += kFluxThreads) {
        const double g = red[i];
        if (g > 0.0 && floor((g - g_min) * inv_dg) == (double)b) acc += image[i];
    }
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
        if (threadIdx.x == 0) partial[(size_t)b * nchunks + chunk] = v;
    }
}

cudaError_t launch_profile(const double* d_image, const double* d_red, size_t npix, int nbins, double g_min, double g_max,
                           double scale, double* d_partial, double* d_hist, cudaStream_t stream) {
    const int nchunks = flux_chunks(npix);
    const double inv_dg = (double)nbins / (g_max - g_min);
    k_profile_partial<<<dim3(nchunks, nbins), kFluxThreads, 0, stream>>>(d_image, d_red, npix, g_min, inv_dg, nbins, d_partial, nchunks);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    k_flux_final<<<nbins, 32, 0, stream>>>(d_partial, nchunks, scale, d_hist);
    return cudaGetLastError();
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

// diagnostics: null condition g_mn k^m k^n (Eq. 4) at given states
template <bool H1>
__global__ void k_null_norm(const __grid_constant__ KP P, int n, const double* __restrict__ XK, double* __restrict__ out,
                            double* __restrict__ elq) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double* q = XK + (size_t)i * 8;
    Geom G;
    geom_eval<H1>(P, q[1], q[2], G);
    Met M;
    met_eval(P, G, M);
    const double kt = q[4], kr = G.ex * q[5], kh = G.dth * q[6], kp = q[7];
    out[i] = ks_dot(M, kt, kr, kh, kp, kt, kr, kh, kp);
    if (elq) {
        // Eq. 38-40: E = -k_t, L = k_phi, Q = k_th^2 + cos^2 th (-a^2 k_t^2 + k_phi^2 / sin^2 th)
        const double k_t = ks_dot(M, kt, kr, kh, kp, 1.0, 0.0, 0.0, 0.0);               // g(k, d_t)
        const double k_p = ks_dot(M, kt, kr, kh, kp, 0.0, 0.0, 0.0, 1.0);               // g(k, d_phi)
        const double k_h = M.Sig * kh;
        elq[i * 3 + 0] = -k_t;
        elq[i * 3 + 1] = k_p;
        elq[i * 3 + 2] = fma(k_h, k_h, G.c * G.c * (k_p * k_p / M.ss - P.a2 * k_t * k_t));
    }
}

cudaError_t launch_null_norm(const KP& P, int n, const double* d_XK, double* d_out, double* d_elq, cudaStream_t stream) {
    int grid = (n + 127) / 128;
    if (P.omh == 0.0) k_null_norm<true><<<grid, 128, 0, stream>>>(P, n, d_XK, d_out, d_elq);
    else k_null_norm<false><<<grid, 128, 0, stream>>>(P, n, d_XK, d_out, d_elq);
    return cudaGetLastError();
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

// FP64 issue-rate probe by operand form: 8 independent chains per thread, 8 warps per sub-partition.
//   0  x = fma(x, imm, imm)     one register source        (the form raptor_fp64_peak times)
//   1  x = fma(y, z, x)         three different register sources
//   2  x = fma(x, y, x)         two different register sources
//   3  x = x * y                DMUL, two register sources
//   4  x = x + z                DADD, two register sources
// Measured on B200 (profiles/fp64_operand_forms_r2.md): forms 0, 2, 3, 4 issue every 2.06 cycles per sub-partition,
// form 1 every 3.17: the register file feeds the FP64 pipe about one 64-bit operand per cycle.
template <int MODE>
__global__ void __launch_bounds__(256) k_fp64_form(int iters, double seed, double* __restrict__ out) {
    double x[8], y[8], z[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { x[i] = seed + threadIdx.x + i; y[i] = 1.0 + 1e-9 * (threadIdx.x + i); z[i] = 1e-9 * i + 1e-12 * threadIdx.x; }
#pragma unroll 2
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            if (MODE == 0) x[i] = fma(x[i], 0.999999, 1e-9);
            if (MODE == 1) x[i] = fma(y[i], z[i], x[i]);
            if (MODE == 2) x[i] = fma(x[i], y[i], x[i]);
            if (MODE == 3) x[i] = x[i] * y[i];
            if (MODE == 4) x[i] = x[i] + z[i];
        }
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i] + y[i] + z[i];
    if (s == 123.456) out[0] = s;      // never true; keeps the chains alive
}

cudaError_t launch_fp64_form(int mode, int iters, int blocks, double* d_out, cudaStream_t stream) {
    switch (mode) {
        case 0: k_fp64_form<0><<<blocks, 256, 0, stream>>>(iters, 1.0, d_out); break;
        case 1: k_fp64_form<1><<<blocks, 256, 0, stream>>>(iters, 1.0, d_out); break;
        case 2: k_fp64_form<2><<<blocks, 256, 0, stream>>>(iters, 1.0, d_out); break;
        case 3: k_fp64_form<3><<<blocks, 256, 0, stream>>>(iters, 1.0, d_out); break;
        case 4: k_fp64_form<4><<<blocks, 256, 0, stream>>>(iters, 1.0, d_out); break;
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

// FP32 peak probe (denominator of the single-precision kernel's roofline): 16 independent FFMA chains per thread
__global__ void __launch_bounds__(256) k_fp32_peak(int iters, float seed, float* __restrict__ out) {
    float x[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = seed + (float)threadIdx.x + (float)i;
    const float m = 0.999999f, c = 1e-6f;
#pragma unroll 2
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = fmaf(x[i], m, c);
    }
    float s = 0.0f;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += x[i];
    if (s == 123.456f) out[0] = s;     // never true; keeps the chains alive
}

cudaError_t launch_fp32_peak(int iters, int blocks, float* d_out, cudaStream_t stream) {
    k_fp32_peak<<<blocks, 256, 0, stream>>>(iters, 1.0f, d_out);
    return cudaGetLastError();
}

cudaError_t launch_fp64_peak(int iters, int blocks, double* d_out, cudaStream_t stream) {
    k_fp64_peak<<<blocks, 256, 0, stream>>>(iters, 1.0, d_out);
    return cudaGetLastError();
}

}  // namespace raptor
