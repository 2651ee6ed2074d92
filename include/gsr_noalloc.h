/*
 * gsr_noalloc.h -- one entry point of libgsr.so for callers that must not allocate.
 *
 * Everything behind gsr.h works on a gsr_handle, and gsr_create / gsr_upload obtain their
 * device storage, scratch included, with cudaMalloc.  Some code that wants one of the solver's
 * building blocks cannot do that:
 *   - a rank whose HBM is already full (the "Large" system keeps about 118 of the 180 GB
 *     resident, and a neighbour process or a framework's memory pool may hold the rest), so a
 *     further cudaMalloc would simply fail;
 *   - code that lives inside a host application which hands out all device memory through its
 *     own pool (torch's caching allocator, an MPI solver's arena) and forbids going around it;
 *   - code on a latency-critical path, or running beside other streams, that cannot accept the
 *     device-wide synchronisation and the unpredictable duration of cudaMalloc / cudaFree.
 * For those callers this header offers the Euclidean norm that LSQR takes of u and v in every
 * iteration (Eq. 4; Alg. 1 l.13-26) as a function that needs no handle and
 * allocates nothing: the caller supplies the input vector and the place for the result, and the
 * only scratch memory -- the per-CTA partial sums of the two-stage reduction -- is a fixed
 * array of GSR_NOALLOC_MAX_PARTIALS doubles (128 KiB) that is part of the library image itself.
 * Every GPU on which the library's device code gets loaded carries that array until the
 * process exits.
 */
#ifndef GSR_NOALLOC_H
#define GSR_NOALLOC_H

#include "gsr.h"

#ifdef __cplusplus
extern "C" {
#endif

/* One CTA of the first stage sums GSR_NOALLOC_CHUNK consecutive elements and leaves one partial
 * sum in the built-in scratch array, which has room for GSR_NOALLOC_MAX_PARTIALS of them.  The
 * longest vector the entry point takes is therefore GSR_NOALLOC_MAX_N = 2^30 elements (8 GiB),
 * twice the row count of the Large config. */
#define GSR_NOALLOC_CHUNK 65536
#define GSR_NOALLOC_MAX_PARTIALS 16384
#define GSR_NOALLOC_MAX_N ((int64_t)GSR_NOALLOC_CHUNK * GSR_NOALLOC_MAX_PARTIALS)

/* out[0] = sqrt(sum_j a[j]^2), the same quantity gsr_lsqr forms for beta = |u| and alpha = |v|
 * (Eq. 4, evaluated without the max-scaling, as the handle's k_sumsq does), in
 * FP64 with a summation order that depends only on n -- not on the GPU model or on earlier
 * calls -- so the result is bit-reproducible.
 *
 *   a       DEVICE pointer to n doubles on GPU `device`; not modified.  May be NULL when n == 0.
 *   n       0 <= n <= GSR_NOALLOC_MAX_N.  n == 0 gives out[0] = 0.
 *   out     DEVICE pointer to one double on the same GPU; the caller owns it.
 *   device  CUDA device ordinal.  The caller's current device is restored before returning.
 *   stream  cudaStream_t of the caller on that device (NULL = legacy default stream).  The two
 *           kernels are queued there and the call waits for them (cudaStreamSynchronize), so
 *           out[0] is valid and every error has been seen when it returns.
 *   err     optional caller-owned buffer of err_len bytes that receives a NUL-terminated
 *           description when the result is not GSR_OK (NULL / 0: no text).
 *
 * Returns GSR_OK; GSR_EINVAL for a NULL pointer, n < 0, or n > GSR_NOALLOC_MAX_N (the text
 * names both numbers; nothing is launched); GSR_ECUDA for a CUDA runtime error.
 *
 * What it does NOT do: it never calls cudaMalloc, cudaFree, cudaMallocHost or any library
 * routine that allocates device or pinned memory, at any n.
 *
 * First call on a device: the function looks up the device address of the built-in scratch
 * array once per GPU (cudaGetSymbolAddress, with that GPU current) and keeps it.  That lookup
 * may make the CUDA runtime create its context on the GPU and load the library's device code,
 * so make the first call per device at start-up, at a point where such one-off work is
 * harmless -- in particular before any stream capture begins.  Later calls only launch.
 *
 * Sharing: all calls on one GPU use the same scratch array, from every thread and every
 * stream, and the array keeps whatever the previous call left in it.  A call reads only the
 * partial sums it has just written, so nothing has to be cleared in between and a stale tail
 * from a longer vector does no harm.  But two calls whose kernels overlap on the GPU -- two
 * host threads, or two streams -- overwrite each other's partial sums: the results are then
 * garbage.  Because the function waits for its own kernels, calls from ONE host thread never
 * overlap; callers with several threads must serialise their calls per GPU themselves.
 */
int32_t gsr_norm2_noalloc(const double *a, int64_t n, double *out, int32_t device, void *stream,
                          char *err, int64_t err_len);

#ifdef __cplusplus
}
#endif
#endif /* GSR_NOALLOC_H */
