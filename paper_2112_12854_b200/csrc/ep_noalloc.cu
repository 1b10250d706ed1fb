// ep_noalloc.cu -- ep_weighted_mean_noalloc(): the one entry point of libep that allocates nothing (include/ep.h, README).
//
// Some callers cannot call cudaMalloc: code under CUDA-graph capture, tight serving loops, harnesses that forbid it.  Every
// other call of the library works on an ep_sim handle whose buffers ep_mesh_create() allocated.  This file holds a variant of
// the deterministic two-pass reduction behind ep_mean_vm() (the volume-averaged potential v_bar of PAPER.md:216 / :230) that
// takes caller-owned device arrays and keeps its scratch -- the per-block partial sums -- in a file-scope device array of fixed
// size: 128 KB that every GPU which loads the library holds until the process exits.
//
// The array's name is a DEVICE symbol: in host code it is a host-side stand-in, not a device address, so the host resolves
// it once per device with cudaGetSymbolAddress() (below, with that device current) and passes the result to the kernels.
//
// Every call shares the array and it keeps the previous call's contents.  Nothing in it has to start at zero: pass 1 writes
// the first `blocks` slots of both halves, pass 2 reads exactly those (never a slot an earlier, larger call left behind).  Two
// calls that overlap on the GPU (different streams, or graphs replayed concurrently) race on it; calls on one stream do not.
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <mutex>

#include "../../include/ep.h"

namespace ep {
int set_error(int code, const char* msg);   // ep_api.cu: stores the message ep_last_error() returns, returns `code`
}

namespace {

constexpr int NA_THREADS = 256;
constexpr int NA_PER_THREAD = 16;
constexpr int NA_CHUNK = NA_THREADS * NA_PER_THREAD;   // elements per block: 4,096
constexpr int NA_MAX_BLOCKS = 8192;
static_assert((int64_t)NA_CHUNK * NA_MAX_BLOCKS == EP_NOALLOC_MAX_N, "include/ep.h states the maximum");

// [0, NA_MAX_BLOCKS): partial sums of w v; [NA_MAX_BLOCKS, 2 NA_MAX_BLOCKS): partial sums of w.  2 x 8,192 x 8 B = 128 KB.
static __device__ __align__(256) double ep_noalloc_scratch[2 * NA_MAX_BLOCKS];

// pass 1: block b sums its own chunk [b NA_CHUNK, (b+1) NA_CHUNK) -- the same elements whatever the grid, so the result
// depends on n only
__global__ void __launch_bounds__(NA_THREADS) noalloc_partial_kernel(int64_t n, const double* __restrict__ v,
                                                                     const double* __restrict__ w,
                                                                     double* __restrict__ scratch) {
    __shared__ double sh_wv[NA_THREADS], sh_w[NA_THREADS];
    const int64_t base = (int64_t)blockIdx.x * NA_CHUNK + threadIdx.x;
    double acc_wv = 0.0, acc_w = 0.0;
#pragma unroll
    for (int k = 0; k < NA_PER_THREAD; ++k) {
        const int64_t i = base + (int64_t)k * NA_THREADS;
        if (i < n) {
            const double wi = w[i];
            acc_wv = fma(wi, v[i], acc_wv);
            acc_w += wi;
        }
    }
    sh_wv[threadIdx.x] = acc_wv;
    sh_w[threadIdx.x] = acc_w;
    __syncthreads();
    for (int s = NA_THREADS / 2; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) {
            sh_wv[threadIdx.x] += sh_wv[threadIdx.x + s];
            sh_w[threadIdx.x] += sh_w[threadIdx.x + s];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        scratch[blockIdx.x] = sh_wv[0];
        scratch[NA_MAX_BLOCKS + blockIdx.x] = sh_w[0];
    }
}

// pass 2: one block adds the first `blocks` partial sums of each half in a fixed order
__global__ void __launch_bounds__(1024) noalloc_final_kernel(int blocks, const double* __restrict__ scratch,
                                                             double* __restrict__ out) {
    __shared__ double sh_wv[1024], sh_w[1024];
    double acc_wv = 0.0, acc_w = 0.0;
    for (int j = threadIdx.x; j < blocks; j += 1024) {
        acc_wv += scratch[j];
        acc_w += scratch[NA_MAX_BLOCKS + j];
    }
    sh_wv[threadIdx.x] = acc_wv;
    sh_w[threadIdx.x] = acc_w;
    __syncthreads();
    for (int s = 512; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) {
            sh_wv[threadIdx.x] += sh_wv[threadIdx.x + s];
            sh_w[threadIdx.x] += sh_w[threadIdx.x + s];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        out[0] = sh_wv[0] / sh_w[0];
        out[1] = sh_w[0];
    }
}

// Device address of the scratch array on the CURRENT device, resolved once per device.  cudaGetSymbolAddress allocates
// nothing: the array is part of the module image the device holds from the moment it loads the library.
constexpr int NA_MAX_DEVICES = 64;
std::mutex g_mu;
double* g_scratch[NA_MAX_DEVICES] = {};

int scratch_on_current_device(double** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return ep::set_error(EP_ERR_CUDA, cudaGetErrorString(e));
    if (dev < 0 || dev >= NA_MAX_DEVICES) return ep::set_error(EP_ERR_ARG, "ep_weighted_mean_noalloc: device ordinal above 63");
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, ep_noalloc_scratch);
        if (e != cudaSuccess || !p) {
            char msg[200];
            std::snprintf(msg, sizeof msg, "ep_weighted_mean_noalloc: cudaGetSymbolAddress failed on device %d: %s", dev,
                          cudaGetErrorString(e));
            return ep::set_error(EP_ERR_CUDA, msg);
        }
        g_scratch[dev] = static_cast<double*>(p);
    }
    *out = g_scratch[dev];
    return EP_OK;
}

}  // namespace

extern "C" int ep_weighted_mean_noalloc(const double* v_dev, const double* w_dev, int64_t n, double* out_dev,
                                        void* cuda_stream) {
    if (!v_dev || !w_dev || !out_dev) return ep::set_error(EP_ERR_ARG, "ep_weighted_mean_noalloc: null argument");
    if (n <= 0) return ep::set_error(EP_ERR_ARG, "ep_weighted_mean_noalloc: n must be positive");
    if (n > EP_NOALLOC_MAX_N) {
        char msg[240];
        std::snprintf(msg, sizeof msg,
                      "ep_weighted_mean_noalloc: n = %lld exceeds EP_NOALLOC_MAX_N = %lld (the fixed 128 KB device scratch holds "
                      "one partial sum per 4096 elements); use ep_mean_vm on a handle instead",
                      (long long)n, (long long)EP_NOALLOC_MAX_N);
        return ep::set_error(EP_ERR_ARG, msg);
    }
    double* scratch = nullptr;
    if (int rc = scratch_on_current_device(&scratch)) return rc;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const int blocks = (int)((n + NA_CHUNK - 1) / NA_CHUNK);
    noalloc_partial_kernel<<<blocks, NA_THREADS, 0, s>>>(n, v_dev, w_dev, scratch);
    noalloc_final_kernel<<<1, 1024, 0, s>>>(blocks, scratch, out_dev);
    const cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) return ep::set_error(EP_ERR_CUDA, cudaGetErrorString(e));
    return EP_OK;
}
