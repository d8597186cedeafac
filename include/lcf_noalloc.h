/* lcf_noalloc.h -- one allocation-free entry point of liblcf.so, for callers that cannot call cudaMalloc (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid it).  Everything else in include/lcf.h works on a plan, and
 * lcf_plan_create allocates the plan's workspaces.
 *
 *   lcf_gram_global_noalloc: the covariance of the WHOLE field of view, Eq. 1,
 *       R[i][j] = sum_p conj(S[i][p]) S[j][p]        (C^H C of the P x N Casorati matrix; the all-ones-window case of Eq. 12)
 *   -- the first step of the global EVD filter (BASELINE.json config 1) -- in double: fp32 samples widened,
 *   products and sums on the FP64 pipe, per-slice partial sums added in a fixed order (deterministic, no atomics).  It is a
 *   variant of the plan path's CUDA-core Gram kernel (csrc/lcf_gram.cu), whose per-chunk partials live in a workspace that
 *   lcf_plan_create allocates; here they live in a file-scope `static __device__` array of fixed size:
 *
 *       LCF_NOALLOC_SLICES x LCF_NOALLOC_MAX_FRAMES^2 complex doubles = 16 x 128 x 128 x 16 B = 4 MiB
 *
 *   which every GPU that loads liblcf.so holds from module load until the process exits.
 *
 * Arguments: iq_dev  DEVICE, complex64 [N][P] (frame-major, pixels contiguous: the layout of lcf_filter with P = Nx Nz);
 *            N       frames, 1 <= N <= LCF_NOALLOC_MAX_FRAMES;  P pixels, 1 <= P <= 2^30;
 *            R_dev   DEVICE, N x N complex doubles, row-major (re, im interleaved), written in full;
 *            stream  the work is enqueued on it; the call does not synchronise.
 * Ownership: the caller owns iq_dev and R_dev; the library owns the scratch array.
 * Returns  : LCF_OK; LCF_ERR_INVALID_ARG (null pointer, N < 1, P < 1); LCF_ERR_UNSUPPORTED (N or P beyond the maximum: nothing
 *            is launched); LCF_ERR_CUDA (the scratch address could not be taken on this device, or a launch failed).  After a
 *            failure lcf_noalloc_last_error() returns a sentence that says which (for the calling thread).
 * The call makes no cudaMalloc / cudaFree / cudaMallocAsync and calls no library routine that allocates.  Once per device (on the
 * first call with that device current) it takes the scratch array's device address with cudaGetSymbolAddress.
 *
 * Sharing: all calls on a device use the SAME scratch array, and it keeps the contents of the last call.  Nothing in it has to
 * start at zero -- every partial a call reads it has written first -- but two calls whose kernels overlap on the GPU (different
 * streams without an ordering between them, or two host threads) race on it and both results are garbage.  Calls on one stream,
 * or ordered by events, are safe.
 */
#ifndef LCF_NOALLOC_H_
#define LCF_NOALLOC_H_

#include "lcf.h"

#ifdef __cplusplus
extern "C" {
#endif

#define LCF_NOALLOC_MAX_FRAMES 128
#define LCF_NOALLOC_SLICES 16

lcf_status lcf_gram_global_noalloc(const void* iq_dev /* DEVICE */, int N, long long P, double* R_dev /* DEVICE */, cudaStream_t stream);
/* HOST string owned by the library (per thread): why the last lcf_gram_global_noalloc of this thread failed; "" if it did not. */
const char* lcf_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* LCF_NOALLOC_H_ */
