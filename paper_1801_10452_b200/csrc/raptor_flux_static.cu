// raptor_flux_static.cu -- flux reduction (a7) for callers that are not allowed to allocate device memory.
//
// The ordinary path (raptor_flux) needs a context, and raptor_create gets the reduction's partial sums from
// cudaMalloc.  Some users of this library cannot do that: a plug-in inside a host program whose memory pool already
// owns all of the device, a service with a fixed device-memory budget signed off in advance, a loop that must not hit
// cudaMalloc's device-wide synchronisation.  For them the partial sums live in the library image itself: a
// file-scope __device__ array that every GPU which loads this library carries from load until the process ends.
//
// Same chunking and the same summation tree as k_flux_partial / k_flux_final of raptor_kernels.cu, so the result is
// the one raptor_flux gives for the same image and scale, bit for bit.
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>

#include "raptor_kernels.h"

namespace raptor {

// The scratch: kFluxStaticSlots partial sums = 128 KiB per GPU, resident until exit.  One slot per
// (image plane, chunk of 16384 pixels); e.g. 64 planes of 2048^2 pixels, or one plane of 2^28 pixels.
static __device__ __align__(256) double g_flux_static_partial[kFluxStaticSlots];

// On the host the NAME g_flux_static_partial is only a handle for the runtime's symbol table, not a device address
// (a kernel handed `g_flux_static_partial` from host code would read host memory or fault).  The address a kernel can
// use comes from cudaGetSymbolAddress, asked once per device with that device current, and is kept here.
constexpr int kMaxDevices = 64;
static double* g_scratch_addr[kMaxDevices] = {nullptr};
static std::mutex g_scratch_lock;

static cudaError_t scratch_of_current_device(double** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> hold(g_scratch_lock);
    if (!g_scratch_addr[dev]) {
        double* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_flux_static_partial);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_scratch_addr[dev] = p;
    }
    *out = g_scratch_addr[dev];
    return cudaSuccess;
}

constexpr int kThreads = 256;       // = kFluxThreads of raptor_kernels.cu
constexpr int kChunk = 16384;       // = kFluxChunk   of raptor_kernels.cu (flux_chunks() counts with it)

// Variant of k_flux_partial: chunk `chunk` of plane k -> partial[k * nchunks + chunk].  Every slot the second kernel
// reads is written here first, in the same call, so what an earlier call left in the array never enters a sum.
__global__ void __launch_bounds__(kThreads) k_flux_partial_static(const double* __restrict__ image, size_t npix,
                                                                  double* __restrict__ partial, int nchunks) {
    __shared__ double sh[kThreads];
    const int k = blockIdx.y, chunk = blockIdx.x;
    const size_t lo = (size_t)chunk * kChunk;
    const size_t hi = lo + kChunk < npix ? lo + kChunk : npix;
    const double* img = image + (size_t)k * npix;
    double acc = 0.0;
    for (size_t i = lo + threadIdx.x; i < hi; i += kThreads) acc += img[i];
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int o = kThreads / 2; o >= 32; o >>= 1) {
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

__global__ void __launch_bounds__(32) k_flux_final_static(const double* __restrict__ partial, int nchunks, double scale,
                                                          double* __restrict__ flux) {
    const int k = blockIdx.x;
    double acc = 0.0;
    for (int i = threadIdx.x; i < nchunks; i += 32) acc += partial[(size_t)k * nchunks + i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    if (threadIdx.x == 0) flux[k] = acc * scale;
}

// Two launches on `stream`, no allocation.  The caller (raptor_flux_static) has checked the sizes.
cudaError_t launch_flux_static(const double* d_image, size_t npix, int n_planes, double scale, double* d_flux,
                               cudaStream_t stream) {
    double* d_partial = nullptr;
    cudaError_t e = scratch_of_current_device(&d_partial);
    if (e != cudaSuccess) return e;
    const int nchunks = flux_chunks(npix);
    k_flux_partial_static<<<dim3(nchunks, n_planes), kThreads, 0, stream>>>(d_image, npix, d_partial, nchunks);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    k_flux_final_static<<<n_planes, 32, 0, stream>>>(d_partial, nchunks, scale, d_flux);
    return cudaGetLastError();
}

}  // namespace raptor
