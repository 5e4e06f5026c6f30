// ov_blas_dot_static: the scalar product <x, y> of include/ov.h's BLAS-1 row ("vector additions and scalar
// products") for callers that must not allocate device memory.
//
// Why this file exists.  ov_blas_dot (blas.cu) is a two-stage reduction: every thread block leaves one partial sum in
// global memory and a second kernel adds them up.  That partial-sum buffer belongs to an ov_ctx and is obtained with
// cudaMalloc -- at ov_create, and again inside the call whenever a larger one is needed.  Some users of this library
// cannot afford that: a lattice code that has already handed every byte of HBM to its own pool (the eigenvector sets
// here are 17-80 GB, so codes size their pools to the last gigabyte and a stray cudaMalloc simply fails), or a solver
// loop that shares the GPU with other streams, where cudaMalloc/cudaFree stall the whole device while they run.  For
// them the partial sums live in a fixed array that is part of the library image itself (g_dot_scratch below); this
// entry point never calls cudaMalloc, cudaFree, cudaMallocHost or any library routine that allocates, and it needs no
// ov_ctx (creating one allocates the gauge copy).
//
// What it costs.  The array is kStaticDotMaxBlocks * 16 B = 512 KiB of device memory on EVERY GPU that loads libov.so,
// from load until the process exits, whether or not this entry point is ever called.  It bounds the vector length:
// n <= kStaticDotMaxBlocks * 1024 = 33 554 432 complex numbers (a 12-component spinor on up to 2 796 202 sites; the
// largest lattice of BASELINE.json, 32^3 x 64, has 2 097 152).  Longer vectors are refused, never truncated.
//
// Sharing.  There is ONE array per GPU, shared by every call from every thread and stream.  A call overwrites entries
// [0, ceil(n/1024)) and its second kernel reads exactly those, so nothing has to be zero beforehand and nothing is
// cleared: whatever an earlier (longer) call left behind the range is never read.  Two calls whose kernels may run on
// the GPU at the same time (different streams without an event between them, or two host threads) race on the array
// and both results are garbage; calls on one stream are ordered and safe.
//
// Set-up.  In host code the name g_dot_scratch is only a handle the runtime knows the array by -- it is not the
// array's device address, and a kernel handed &g_dot_scratch from the host would fault (or, on a system where the
// GPU can reach host memory, quietly scribble over the wrong bytes).  The address is looked up with
// cudaGetSymbolAddress, once per device, with that device current, the first time the entry point is called on it;
// later calls reuse it.  That first call per device should therefore be made before any stream capture is begun.
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "ov.h"
#include "wilson_math.cuh"

namespace {

constexpr int kThreads = 256;                    // same block shape and per-thread work as blas.cu::dot1_kernel,
constexpr int kElemsPerThread = 4;               // so the result agrees with ov_blas_dot to the last bit
constexpr int kBlockElems = kThreads * kElemsPerThread;
constexpr long long kStaticDotMaxBlocks = 32768;  // 512 KiB of partial sums
constexpr long long kStaticDotMaxElems = kStaticDotMaxBlocks * kBlockElems;
constexpr int kMaxDevices = 64;

// the scratch memory: part of the library image, one instance per GPU, never freed (see the header comment)
static __device__ __align__(256) double2 g_dot_scratch[kStaticDotMaxBlocks];

// stage 1: block b leaves sum_{e in its 1024 elements} conj(x[e]) y[e] in partial[b]
__global__ void __launch_bounds__(kThreads) dot_static_kernel(const double2* __restrict__ x, const double2* __restrict__ y,
                                                              long long n, double2* __restrict__ partial) {
    __shared__ double2 sh[kThreads];
    const long long base = (long long)blockIdx.x * kBlockElems + threadIdx.x;
    double2 xv[kElemsPerThread], yv[kElemsPerThread];
#pragma unroll
    for (int m = 0; m < kElemsPerThread; m++) {
        const long long e = base + (long long)m * kThreads;
        xv[m] = (e < n) ? x[e] : make_double2(0.0, 0.0);
        yv[m] = (e < n) ? y[e] : make_double2(0.0, 0.0);
    }
    double2 acc = make_double2(0.0, 0.0);
#pragma unroll
    for (int m = 0; m < kElemsPerThread; m++) ov::cmaddc(acc, xv[m], yv[m]);
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int o = kThreads / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] = ov::cadd(sh[threadIdx.x], sh[threadIdx.x + o]);
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}

// stage 2 (one block): adds partial[0 .. nblocks) in a fixed order and writes (re, im) to out; nblocks = 0 gives 0
__global__ void __launch_bounds__(kThreads) dot_static_reduce_kernel(const double2* __restrict__ partial, long long nblocks,
                                                                     double* __restrict__ out) {
    __shared__ double2 sh[kThreads];
    double2 acc = make_double2(0.0, 0.0);
    for (long long b = threadIdx.x; b < nblocks; b += kThreads) acc = ov::cadd(acc, partial[b]);
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int o = kThreads / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] = ov::cadd(sh[threadIdx.x], sh[threadIdx.x + o]);
        __syncthreads();
    }
    if (threadIdx.x == 0) { out[0] = sh[0].x; out[1] = sh[0].y; }
}

thread_local char t_err[256] = "";

int set_err(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_err, sizeof t_err, fmt, ap);
    va_end(ap);
    return code;
}

std::mutex g_setup_mutex;
double2* g_scratch_addr[kMaxDevices] = {};  // device address of g_dot_scratch on device d (nullptr: not looked up yet)

// device address of the scratch array on the CURRENT device; looks it up on the first call per device
int scratch_on_current_device(double2** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return set_err(OV_ECUDA, "ov_blas_dot_static: cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices)
        return set_err(OV_EINVAL, "ov_blas_dot_static: device ordinal %d outside the supported 0..%d", dev, kMaxDevices - 1);
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_dot_scratch);
        if (e != cudaSuccess || !p)
            return set_err(OV_ECUDA, "ov_blas_dot_static: cudaGetSymbolAddress on device %d: %s", dev, cudaGetErrorString(e));
        g_scratch_addr[dev] = static_cast<double2*>(p);
    }
    *out = g_scratch_addr[dev];
    return OV_OK;
}

}  // namespace

extern "C" {

long long ov_blas_dot_static_max(void) { return kStaticDotMaxElems; }

const char* ov_blas_dot_static_error(void) { return t_err; }

int ov_blas_dot_static(const void* x_dev, const void* y_dev, long long n, void* out_dev, void* cuda_stream) {
    t_err[0] = '\0';
    if (!x_dev || !y_dev || !out_dev) return set_err(OV_EINVAL, "ov_blas_dot_static: null pointer");
    if (n < 0) return set_err(OV_EINVAL, "ov_blas_dot_static: n = %lld is negative", n);
    if (n > kStaticDotMaxElems)
        return set_err(OV_EINVAL,
                       "ov_blas_dot_static: n = %lld complex elements exceeds the fixed scratch array (at most %lld = %lld "
                       "partial sums x %d elements); use ov_blas_dot, which allocates its scratch",
                       n, kStaticDotMaxElems, kStaticDotMaxBlocks, kBlockElems);
    double2* scratch = nullptr;
    const int rc = scratch_on_current_device(&scratch);
    if (rc != OV_OK) return rc;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const long long nblocks = (n + kBlockElems - 1) / kBlockElems;
    if (nblocks > 0)
        dot_static_kernel<<<(unsigned)nblocks, kThreads, 0, stream>>>(static_cast<const double2*>(x_dev),
                                                                      static_cast<const double2*>(y_dev), n, scratch);
    dot_static_reduce_kernel<<<1, kThreads, 0, stream>>>(scratch, nblocks, static_cast<double*>(out_dev));
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return set_err(OV_ECUDA, "ov_blas_dot_static: kernel launch: %s", cudaGetErrorString(e));
    return OV_OK;
}

}  // extern "C"
