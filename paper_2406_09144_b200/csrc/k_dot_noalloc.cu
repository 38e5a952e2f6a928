// k_dot_noalloc.cu -- frs_dot_noalloc (include/frs.h): the fp64 inner product of frs_dot for callers that must not
// allocate device memory.  frs_dot needs a context, and a context allocates (tables at frs_create, gigabytes of scratch on
// first use).  Two kinds of caller cannot live with that: a process in which another allocator already owns the GPU's
// memory (PyTorch's caching allocator sized to fill the 180 GB: a raw cudaMalloc from this library then fails although
// the framework has room), and a latency-bound loop such as the channel-sharded CG, where cudaMalloc / cudaFree stall
// every stream of the device, the NCCL and copy streams included.  This file therefore calls no cudaMalloc, cudaFree or
// other allocating routine: the one piece of scratch the reduction needs, a partial sum per CTA, lives in a
// fixed array inside the library's device image.
//
// The arithmetic and the launch shape are those of dot() in frs_api.cu (256 threads, one float4 per thread and step, fp64
// products and sums, partials summed by one CTA in index order), restated here because ew_kernels.cuh belongs to that
// translation unit; the result has the same bits as frs_dot's.
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <mutex>

#include "../../include/frs.h"

// The scratch: one fp64 partial per CTA, at most kMaxCtas CTAs = 9 472 bytes.  Every GPU that loads libfrs.so carries this
// array from the moment the library's device code is loaded until the process exits, whether or not the entry point is
// ever called -- which is why it is kept this small.
// In HOST code the name below is only a handle for the runtime, not a device address: handing it to a kernel makes
// the kernel fault or, on a system where the GPU can read host memory, quietly work on the wrong memory.  Host code gets
// the real address from cudaGetSymbolAddress (scratch_of_device below); only device code may use the name itself.
static constexpr int kMaxCtas = 1184;   // 148 SMs x 8, the cap of red_blocks() in frs_api.cu
static __device__ __align__(256) double g_dot_noalloc_partials[kMaxCtas];

namespace {

constexpr int kThreads = 256;
constexpr int kMaxDevices = 64;

thread_local char t_err[256] = "no error";
int fail(int code, const char* msg) {
    snprintf(t_err, sizeof(t_err), "%s", msg);
    return code;
}
int cuda_fail(cudaError_t e, const char* where) {
    snprintf(t_err, sizeof(t_err), "frs_dot_noalloc: CUDA error at %s: %s", where, cudaGetErrorString(e));
    return FRS_ECUDA;
}

// Device address of the scratch array on each device, looked up once per device with that device current.
std::mutex g_mu;
double* g_scratch[kMaxDevices] = {};

int scratch_of_device(int device, double** out) {
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch[device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_dot_noalloc_partials);   // the array's copy on the CURRENT device
        if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(g_dot_noalloc_partials)");
        if (!p) return fail(FRS_ECUDA, "frs_dot_noalloc: cudaGetSymbolAddress returned a null address");
        g_scratch[device] = static_cast<double*>(p);
    }
    *out = g_scratch[device];
    return FRS_OK;
}

__device__ __forceinline__ double block_sum(double x) {
    __shared__ double red[32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) red[w] = x;
    __syncthreads();
    double y = 0.0;
    if (w == 0) {
        const int nw = blockDim.x >> 5;
        y = l < nw ? red[l] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) y += __shfl_down_sync(0xffffffffu, y, o);
    }
    return y;   // valid in thread 0
}

// partials[blockIdx.x] = sum over this CTA's slice of a[i] b[i]; `partials` is the scratch array's device address
__global__ void __launch_bounds__(kThreads) dot_partial_noalloc_kernel(const float* __restrict__ a, const float* __restrict__ b,
                                                                        size_t n, double* __restrict__ partials) {
    double acc = 0.0;
    const size_t n4 = n / 4;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
        const float4 x = reinterpret_cast<const float4*>(a)[i], y = reinterpret_cast<const float4*>(b)[i];
        acc += (double)x.x * y.x + (double)x.y * y.y + (double)x.z * y.z + (double)x.w * y.w;
    }
    acc = block_sum(acc);
    if (threadIdx.x == 0) partials[blockIdx.x] = acc;
}

// *out = sum_{i < n} partials[i], fixed order; one CTA.  Reads only the n slots the kernel above has just written, so
// whatever an earlier call left in the rest of the array is never looked at and nothing needs clearing.
__global__ void __launch_bounds__(kThreads) dot_final_noalloc_kernel(const double* __restrict__ partials, int n,
                                                                      double* __restrict__ out) {
    // Device code may name the array itself: a host that passed anything but its address (the host-side handle, say)
    // is told so by a NaN instead of a sum over the wrong memory.
    if (partials != g_dot_noalloc_partials) {
        if (threadIdx.x == 0) *out = __longlong_as_double(0x7ff8000000000000ll);
        return;
    }
    double acc = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) acc += partials[i];
    acc = block_sum(acc);
    if (threadIdx.x == 0) *out = acc;
}

}  // namespace

extern "C" int frs_dot_noalloc(int device, void* stream, const float* a, const float* b, long long n, double* d_out) {
    if (!a || !b || !d_out) return fail(FRS_EINVAL, "frs_dot_noalloc: NULL pointer");
    if (n <= 0 || (n & 3)) return fail(FRS_EINVAL, "frs_dot_noalloc: n must be a positive multiple of 4");
    if (n > FRS_DOT_NOALLOC_MAX_N) {
        snprintf(t_err, sizeof(t_err), "frs_dot_noalloc: n = %lld is beyond the maximum FRS_DOT_NOALLOC_MAX_N = %lld floats this entry point accepts",
                 n, (long long)FRS_DOT_NOALLOC_MAX_N);
        return FRS_EINVAL;
    }
    if ((reinterpret_cast<uintptr_t>(a) & 15u) || (reinterpret_cast<uintptr_t>(b) & 15u) || (reinterpret_cast<uintptr_t>(d_out) & 7u))
        return fail(FRS_EINVAL, "frs_dot_noalloc: a, b must be 16-byte aligned and d_out 8-byte aligned");
    if (device < 0 || device >= kMaxDevices) return fail(FRS_EINVAL, "frs_dot_noalloc: device ordinal out of range");
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) return cuda_fail(e, "cudaSetDevice");
    double* scratch = nullptr;
    const int r = scratch_of_device(device, &scratch);   // first call on this device: looks the address up
    if (r != FRS_OK) return r;
    size_t nb = ((size_t)n / 4 + kThreads - 1) / kThreads;   // red_blocks() of frs_api.cu
    if (nb > (size_t)kMaxCtas) nb = kMaxCtas;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    dot_partial_noalloc_kernel<<<(int)nb, kThreads, 0, st>>>(a, b, (size_t)n, scratch);
    dot_final_noalloc_kernel<<<1, kThreads, 0, st>>>(scratch, (int)nb, d_out);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "kernel launch");
    return FRS_OK;
}

extern "C" const char* frs_dot_noalloc_last_error(void) { return t_err; }
