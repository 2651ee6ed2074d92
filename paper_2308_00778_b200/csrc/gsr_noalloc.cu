// gsr_noalloc.cu -- gsr_norm2_noalloc (include/gsr_noalloc.h): the LSQR norm (Eq. 4) for
// callers that must not allocate.  A variant of the handle's k_sumsq + the partial fold of k_scalar
// (gsr_kernels.cuh) whose per-CTA partial sums live in a file-scope __device__ array instead of the
// cudaMalloc'ed sqPartial buffers of a gsr_handle.  Shares no state with gsr.cu.
#include <cstdarg>
#include <cstdio>
#include <cstdint>
#include <mutex>

#include <cuda_runtime.h>

#include "gsr_noalloc.h"

namespace {

constexpr int NA_THREADS = 256;
constexpr int NA_MAX_DEVICES = 64;

// The scratch: one partial sum per first-stage CTA.  Part of the library image, so every GPU that loads
// this module holds its own 128 KiB copy until the process ends.  IN HOST CODE THIS NAME IS ONLY A
// STAND-IN for the symbol, not a device address: handing `g_normPartial` itself to a kernel would make the
// kernel fault (or, on a system where the GPU can reach host memory, quietly scribble over host data).
// Host code must go through cudaGetSymbolAddress (scratch_for below); device code may name it directly.
static __device__ __align__(256) double g_normPartial[GSR_NOALLOC_MAX_PARTIALS];

// Device address of g_normPartial per GPU, looked up once (set-up) and then only read.
std::mutex g_setupLock;
double *g_scratchAddr[NA_MAX_DEVICES] = {};

// Fixed-tree sum over the CTA; valid in thread 0.
__device__ __forceinline__ double na_block_sum(double v)
{
    __shared__ double red[NA_THREADS / 32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();   // red may still be read by the previous use
    if (lane == 0) red[w] = v;
    __syncthreads();
    double r = 0.0;
    if (w == 0) {
        r = lane < NA_THREADS / 32 ? red[lane] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) r += __shfl_xor_sync(0xffffffffu, r, o);
    }
    return r;
}

// Stage 1: CTA c sums the squares of a[c*CHUNK, min(n, (c+1)*CHUNK)) and WRITES (never adds to)
// partial[c]: nothing in the scratch has to be zero beforehand.  Coalesced: consecutive threads read
// consecutive doubles, 256 steps of 2 KiB per CTA.
__global__ void __launch_bounds__(NA_THREADS)
k_sumsq_chunks(const double *__restrict__ a, int64_t n, double *__restrict__ partial)
{
    const int64_t lo = int64_t(blockIdx.x) * GSR_NOALLOC_CHUNK;
    const int64_t hi = lo + GSR_NOALLOC_CHUNK < n ? lo + GSR_NOALLOC_CHUNK : n;
    double s = 0.0;
    for (int64_t j = lo + threadIdx.x; j < hi; j += NA_THREADS) {
        const double t = a[j];
        s = fma(t, t, s);
    }
    s = na_block_sum(s);
    if (threadIdx.x == 0) partial[blockIdx.x] = s;
}

// Stage 2: one CTA folds partial[0, nPartial) in a fixed order and writes the norm.  Entries at and
// beyond nPartial (left over from a longer vector of an earlier call) are never read.
__global__ void __launch_bounds__(NA_THREADS)
k_norm_fold(const double *__restrict__ partial, int nPartial, double *__restrict__ out)
{
    double s = 0.0;
    for (int j = threadIdx.x; j < nPartial; j += NA_THREADS) s += partial[j];
    s = na_block_sum(s);
    if (threadIdx.x == 0) out[0] = sqrt(s);
}

int32_t na_fail(char *err, int64_t errLen, int32_t code, const char *fmt, ...)
{
    if (err && errLen > 0) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(err, size_t(errLen), fmt, ap);
        va_end(ap);
    }
    return code;
}

// Set-up, once per device, with that device current: ask the runtime where g_normPartial lives on it.
cudaError_t scratch_for(int device, double **ptr)
{
    std::lock_guard<std::mutex> guard(g_setupLock);
    if (!g_scratchAddr[device]) {
        double *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void **>(&p), g_normPartial);
        if (e != cudaSuccess) return e;
        g_scratchAddr[device] = p;
    }
    *ptr = g_scratchAddr[device];
    return cudaSuccess;
}

struct DeviceGuard {   // makes `device` current, puts the caller's device back on scope exit
    int prev = -1;
    cudaError_t enter(int device)
    {
        cudaError_t e = cudaGetDevice(&prev);
        if (e != cudaSuccess) { prev = -1; return e; }
        return prev == device ? cudaSuccess : cudaSetDevice(device);
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

}  // namespace

#define NA_CK(call)                                                                                    \
    do {                                                                                               \
        const cudaError_t e_ = (call);                                                                 \
        if (e_ != cudaSuccess) {                                                                       \
            cudaGetLastError();                                                                        \
            return na_fail(err, err_len, GSR_ECUDA, "gsr_norm2_noalloc: %s: %s", #call,                \
                           cudaGetErrorString(e_));                                                    \
        }                                                                                              \
    } while (0)

extern "C" int32_t gsr_norm2_noalloc(const double *a, int64_t n, double *out, int32_t device, void *stream,
                                     char *err, int64_t err_len)
{
    if (n < 0) return na_fail(err, err_len, GSR_EINVAL, "gsr_norm2_noalloc: n = %lld is negative", (long long)n);
    if (n > GSR_NOALLOC_MAX_N)
        return na_fail(err, err_len, GSR_EINVAL,
                       "gsr_norm2_noalloc: n = %lld exceeds GSR_NOALLOC_MAX_N = %lld (the built-in scratch holds "
                       "%d partial sums of %d elements each); split the vector or use a gsr_handle",
                       (long long)n, (long long)GSR_NOALLOC_MAX_N, GSR_NOALLOC_MAX_PARTIALS, GSR_NOALLOC_CHUNK);
    if (!out || (!a && n > 0)) return na_fail(err, err_len, GSR_EINVAL, "gsr_norm2_noalloc: NULL pointer");
    if (device < 0 || device >= NA_MAX_DEVICES)
        return na_fail(err, err_len, GSR_EINVAL, "gsr_norm2_noalloc: device ordinal %d out of range", device);

    DeviceGuard guard;
    NA_CK(guard.enter(device));
    double *scratch = nullptr;
    NA_CK(scratch_for(device, &scratch));

    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int nPartial = int((n + GSR_NOALLOC_CHUNK - 1) / GSR_NOALLOC_CHUNK);
    if (nPartial > 0) k_sumsq_chunks<<<nPartial, NA_THREADS, 0, st>>>(a, n, scratch);
    k_norm_fold<<<1, NA_THREADS, 0, st>>>(scratch, nPartial, out);
    NA_CK(cudaGetLastError());
    NA_CK(cudaStreamSynchronize(st));
    return GSR_OK;
}
