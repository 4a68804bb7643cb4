// raptor_kernels.h -- host-visible launchers of raptor_kernels.cu (internal to the library).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "raptor_device.cuh"

// launch shape of the persistent ray kernel: RAPTOR_BLOCK threads per CTA, RAPTOR_MIN_BLOCKS resident CTAs per SM
#ifndef RAPTOR_BLOCK
#define RAPTOR_BLOCK 128
#endif
// with several frequencies a CTA may have up to RAPTOR_BLOCK_MULTI threads (see launch_shape in raptor_kernels.cu)
#ifndef RAPTOR_BLOCK_MULTI
#define RAPTOR_BLOCK_MULTI 256
#endif
#ifndef RAPTOR_MIN_BLOCKS
#define RAPTOR_MIN_BLOCKS 4
#endif

namespace raptor {

// Outputs and work queue of one launch of the ray kernel.  All pointers are device pointers; any output may be NULL.
struct RenderOut {
    unsigned int* queue;            // tile counter, zeroed before the launch
    unsigned int ntiles;            // tiles this launch processes: global tile = tile_offset + i * tile_stride
    unsigned int tile_offset, tile_stride;
    const unsigned int* order;      // [tiles of one image] tile (ty * ntx + tx) of sequence number k: from the image centre outward; NULL: by rows
    unsigned long long* counters;   // [3] steps, sampled steps, rays (accumulated)
    const double* alpha;            // trace mode: explicit impact parameters [nrays]; NULL = render the pixel grid
    const double* beta;
    long long nrays;
    double* image;                  // [n_freq][npix]
    double* tau;                    // [n_freq][npix]
    int32_t* status;                // [npix]
    int32_t* nsteps;                // [npix]
    double* XK;                     // [npix][8] final state
    double* null_max;               // [npix] max |g(k,k)| over the steps of the ray (Eq. 4), or NULL
    unsigned int frames;            // > 1: light-curve batch, image is [frames][n_freq][npix]; ntiles = frames * tiles_per_frame
    unsigned int tiles_per_frame;
    double t_cam0, dt_frame;        // camera time of frame f: t_cam0 + f dt_frame
};

// Kernel parameters of the single-precision kernel (raptor_render_f32.cu): float copies, computed on the host in
// double and rounded once; only combinations inside the float range (8(f) f1, Table B.1 of the paper).
struct KPf {
    float a, a2, twoa, m, twom, omh, r0;
    float r_cam, sin_i, cos_i, sq1mc2, x1_cam, x2_cam, dth_cam, t_cam, fov;
    float eps, delta, r_in, r_out, tau_cutoff;
    float Lcm, ne_scale, B0, thetae_scale, x1_first, inv_d1, nu_obs;
    const float* grid;          // device, [n1][n2][8] float: (float) of the context's float64 grid
    int nx, ny, max_steps, n1, n2, use_tau_cutoff;
};
cudaError_t launch_render_f32(const KPf& P, const RenderOut& O, int sm_count, cudaStream_t stream);
cudaError_t launch_grid_to_f32(const double* d_src, float* d_dst, size_t n, cudaStream_t stream);

// raptor_render.cu: one explicit instantiation per (plasma model, integrator), one translation unit each
template <int MODEL, int INTEG>
cudaError_t launch_model(const KP& P, const RenderOut& O, bool h1, bool multi, bool fullx, int grid, int block, cudaStream_t s);
cudaError_t launch_render(const KP& P, int model, const RenderOut& O, int sm_count, cudaStream_t stream);
int flux_chunks(size_t npix);
cudaError_t launch_flux(const double* d_image, size_t npix, int n_freq, double scale, double* d_partial,
                        double* d_flux, cudaStream_t stream);
cudaError_t launch_profile(const double* d_image, const double* d_red, size_t npix, int nbins, double g_min, double g_max,
                           double scale, double* d_partial, double* d_hist, cudaStream_t stream);
cudaError_t launch_null_norm(const KP& P, int n, const double* d_XK, double* d_out, double* d_elq, cudaStream_t stream);
cudaError_t launch_eval_rhs(const KP& P, int n, const double* d_XK, double* d_f, cudaStream_t stream);
// raptor_flux_static.cu: the same reduction with its partial sums in a __device__ array of the library (no allocation)
constexpr int kFluxStaticSlots = 16384;      // partial sums the array holds: n_planes * flux_chunks(npix) must fit
cudaError_t launch_flux_static(const double* d_image, size_t npix, int n_planes, double scale, double* d_flux,
                               cudaStream_t stream);
cudaError_t launch_fp64_peak(int iters, int blocks, double* d_out, cudaStream_t stream);
cudaError_t launch_fp32_peak(int iters, int blocks, float* d_out, cudaStream_t stream);
cudaError_t launch_fp64_form(int mode, int iters, int blocks, double* d_out, cudaStream_t stream);

}  // namespace raptor
