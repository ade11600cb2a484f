// mphv_sum_noalloc: the total of a device array (the mass check of f, BJ: conserved to 1e-13)
// for callers that must not allocate device memory. Contract in include/mphv.h.
//
// Who needs this. mphv_sum_f belongs to a context, and mphv_create takes its workspace
// (including the per-block partial sums of the reduction) from cudaMalloc. Two kinds of caller
// cannot go that way: a host code whose own memory manager has already claimed the whole of HBM
// at start-up (a simulation framework with its own arena, or a process whose caching allocator
// holds the device), where a cudaMalloc inside a library simply returns out-of-memory; and a
// caller inside its time loop, where cudaMalloc / cudaFree synchronise the whole device and stall
// every stream that is running. For them the partial sums of this variant live in a file-scope
// __device__ array, which is part of the loaded library image rather than of any heap.
//
// This file shares nothing with the context path in mphv.cu: that path is unchanged.
#include "../../include/mphv.h"

#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdio>
#include <mutex>

namespace {

constexpr int CHUNK = MPHV_SUM_NOALLOC_CHUNK;                               // doubles summed by one CTA
constexpr size_t MAX_COUNT = MPHV_SUM_NOALLOC_MAX_COUNT;
constexpr int MAX_PARTIALS = (int)(MAX_COUNT / (size_t)CHUNK);              // 16384 doubles = 128 KiB
constexpr int THREADS = 256;
constexpr int MAX_DEVICES = 64;

static_assert(MAX_COUNT % (size_t)CHUNK == 0, "the maximum count is a whole number of chunks");

// The scratch: one partial sum per chunk of the input. Every GPU that loads libmphv.so carries these
// 128 KiB from module load until the process exits. All calls on one device share it.
// NOTE for host code below: `g_partials` names a host-side shadow of the symbol, NOT device memory. The
// device address is what cudaGetSymbolAddress returns (scratch_of_current_device); only that may be
// handed to a kernel.
static __device__ __align__(256) double g_partials[MAX_PARTIALS];

std::mutex g_mu;
double *g_partials_dev[MAX_DEVICES];      // device address of g_partials, per CUDA device (nullptr: not resolved yet)

void say(char *err, size_t cap, const char *fmt, ...)
{
    if (!err || !cap) return;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(err, cap, fmt, ap);
    va_end(ap);
}

// Kahan-compensated running sum of one thread, then a fixed-order tree over the CTA: lanes by shuffle,
// warps through shared memory. Fixed order => the same bits on every call and on every GPU.
__device__ __forceinline__ double cta_total(double s, double *red /* [32] */)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) red[wid] = s;
    __syncthreads();
    double t = 0.0;
    if (wid == 0) {
        t = lane < (int)(blockDim.x >> 5) ? red[lane] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
    }
    return t;                                  // valid in thread 0
}

// Stage 1: CTA b owns x[b*CHUNK, min(count, (b+1)*CHUNK)) and writes its total to part[b]. Unlike the
// grid-stride sum_kernel of the context path, the split of the input does not depend on the launch
// shape, so the scratch need is count / CHUNK entries and the result is a function of (x, count) alone.
__global__ void __launch_bounds__(THREADS)
sum_chunks_kernel(const double *__restrict__ x, unsigned long long count, double *__restrict__ part)
{
    __shared__ double red[32];
    const unsigned long long lo = (unsigned long long)blockIdx.x * CHUNK;
    const unsigned long long hi = lo + CHUNK < count ? lo + CHUNK : count;
    double s = 0.0, c = 0.0;
    for (unsigned long long i = lo + threadIdx.x; i < hi; i += THREADS) {
        const double y = x[i] - c;
        const double t = s + y;
        c = (t - s) - y;
        s = t;
    }
    const double tot = cta_total(s, red);
    if (threadIdx.x == 0) part[blockIdx.x] = tot;
}

// Stage 2, one CTA: the total of part[0, nparts). Entries at and beyond nparts are leftovers of earlier
// calls and are never read, which is why nothing in the scratch has to be cleared between calls.
__global__ void __launch_bounds__(THREADS)
sum_partials_kernel(const double *__restrict__ part, int nparts, double *__restrict__ out)
{
    __shared__ double red[32];
    double s = 0.0, c = 0.0;
    for (int i = threadIdx.x; i < nparts; i += THREADS) {
        const double y = part[i] - c;
        const double t = s + y;
        c = (t - s) - y;
        s = t;
    }
    const double tot = cta_total(s, red);
    if (threadIdx.x == 0) *out = tot;
}

// Device address of g_partials on the CURRENT device; resolved once per device, then cached.
// cudaGetSymbolAddress may load the library's module on this device the first time (which is when the
// 128 KiB come into being); it does not take memory from the CUDA heap.
int scratch_of_current_device(double **out, char *err, size_t cap)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { cudaGetLastError(); say(err, cap, "cudaGetDevice: %s", cudaGetErrorString(e)); return MPHV_ERR_CUDA; }
    if (dev < 0 || dev >= MAX_DEVICES) { say(err, cap, "device ordinal %d outside 0..%d", dev, MAX_DEVICES - 1); return MPHV_ERR_ARG; }
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_partials_dev[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_partials);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            say(err, cap, "cudaGetSymbolAddress(scratch) on device %d: %s", dev, cudaGetErrorString(e));
            return e == cudaErrorNoKernelImageForDevice || e == cudaErrorInvalidDeviceFunction ? MPHV_ERR_ARCH : MPHV_ERR_CUDA;
        }
        g_partials_dev[dev] = static_cast<double *>(p);
    }
    *out = g_partials_dev[dev];
    return MPHV_OK;
}

}  // namespace

extern "C" int mphv_sum_noalloc(const double *x_dev, size_t count, double *sum_dev, void *stream,
                                char *err, size_t err_cap)
{
    if (err && err_cap) err[0] = 0;
    if (!sum_dev) { say(err, err_cap, "sum_dev is NULL"); return MPHV_ERR_ARG; }
    if (!x_dev && count) { say(err, err_cap, "x_dev is NULL with count = %zu", count); return MPHV_ERR_ARG; }
    if (((uintptr_t)x_dev | (uintptr_t)sum_dev) & 7) { say(err, err_cap, "x_dev and sum_dev must be 8-byte aligned"); return MPHV_ERR_ARG; }
    if (count > MAX_COUNT) {
        say(err, err_cap, "count = %zu exceeds MPHV_SUM_NOALLOC_MAX_COUNT = %zu doubles: the static scratch holds one partial "
            "per %d-double chunk and has %d entries; sum the array in pieces of at most that many, or use mphv_sum_f",
            count, MAX_COUNT, CHUNK, MAX_PARTIALS);
        return MPHV_ERR_RANGE;
    }
    double *part = nullptr;
    const int st = scratch_of_current_device(&part, err, err_cap);
    if (st != MPHV_OK) return st;

    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const int nparts = (int)((count + (size_t)CHUNK - 1) / (size_t)CHUNK);
    if (nparts > 0) sum_chunks_kernel<<<nparts, THREADS, 0, s>>>(x_dev, (unsigned long long)count, part);
    sum_partials_kernel<<<1, THREADS, 0, s>>>(part, nparts, sum_dev);
    const cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) {
        cudaGetLastError();
        say(err, err_cap, "launch of the sum kernels: %s", cudaGetErrorString(e));
        return e == cudaErrorNoKernelImageForDevice ? MPHV_ERR_ARCH : MPHV_ERR_CUDA;
    }
    return MPHV_OK;
}
