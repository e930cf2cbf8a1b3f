/* tvbx_noalloc.h -- ONE entry point of libtvbx.so that allocates nothing.
 *
 * Why: some callers cannot call cudaMalloc -- code under CUDA graph capture, tight serving loops, harnesses that forbid it.
 * Every other call of include/tvbx.h works on a sweep object whose device buffers come from cudaMalloc (through the library's
 * pool).  tvbx_top_k_noalloc is the selection step of tvbx_top_k ("output the best ten fittest simulations";
 * DESIGN.md reading A23b: equal scores go to the lower index) as a call of its own: the caller passes the scores and the two
 * output arrays, all in DEVICE memory; the kernel's scratch -- one "taken" flag per score -- lives in a file-scope
 * `static __device__` array of the library (csrc/tvbx_noalloc.cu), whose device address is looked up once per device with
 * cudaGetSymbolAddress.  The call enqueues one kernel on `cuda_stream` and returns: no cudaMalloc, no cudaFree, no allocating
 * library routine, no synchronisation, no host<->device copy.
 *
 * Limit: at most TVBX_NOALLOC_MAX_SCORES scores per call (1,048,576: the array is 1 MiB, held by every GPU that loads the
 * library until the process exits).  Larger inputs are refused with TVBX_EINVAL and a message that names the limit.
 *
 * Sharing: every call on a device uses the SAME array.  The kernel clears the flags it needs before it uses them, so a
 * call does not depend on what the previous one left behind; but two calls that OVERLAP on the GPU (different streams,
 * no dependency between them) race on the array and return garbage.  Calls on one stream, or ordered by events, are safe.
 *
 * Same conventions as tvbx.h: int32 status (TVBX_OK = 0), thread-local text from tvbx_last_error().
 */
#ifndef TVBX_NOALLOC_H
#define TVBX_NOALLOC_H

#include "tvbx.h"

#ifdef __cplusplus
extern "C" {
#endif

#define TVBX_NOALLOC_MAX_SCORES (1 << 20)

/* The k largest of n scores, best first (ties: the lower index first), selected on the current CUDA device.
 *   scores_dev [n]          float32, DEVICE, read only (e.g. the fcsc / fitness / mean_fc array that tvbx_fc_scores wrote with
 *                           on_device = 1)
 *   n                       1 .. TVBX_NOALLOC_MAX_SCORES
 *   k                       >= 1; min(k, n) entries are written
 *   idx_dev [min(k, n)]     int32, DEVICE, out: positions in scores_dev
 *   val_dev [min(k, n)]     float32, DEVICE, out: the scores at those positions
 *   cuda_stream             cudaStream_t (NULL = the default stream); the results are ready when the stream reaches this point
 * Ownership: all three arrays are the caller's; the library keeps no pointer after the kernel has run.
 * Errors: TVBX_EINVAL (NULL pointer, n < 1, k < 1, n > TVBX_NOALLOC_MAX_SCORES), TVBX_ECUDA (no device; symbol lookup or launch
 * failed).  Nothing is enqueued when an error is returned. */
int32_t tvbx_top_k_noalloc(const float* scores_dev, int32_t n, int32_t k, int32_t* idx_dev, float* val_dev, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* TVBX_NOALLOC_H */
