/* allen_velo_noalloc.h — ONE entry point of the library that needs no allocation at all.
 *
 * Why: allen_velo_reconstruct() (allen_velo.h) allocates nothing itself, but it needs a handle (allen_velo_create calls
 * cudaMalloc for the geometry constants) and a caller-allocated workspace.  Some callers cannot allocate: code under
 * CUDA-graph capture, tight serving loops, harnesses that forbid cudaMalloc.  For them the output-compaction step of the
 * path (A9 of SURVEY.md §8(a); "quantities needed to define the grid sizes of individual kernels": the exclusive
 * prefix sum that turns clusters-per-(event, layer) counts into layer_offsets) exists as a variant whose scratch memory
 * — the ticket counter and one status word per tile of the single-pass decoupled-look-back scan — lives in a
 * file-scope `static __device__` array of the library instead of the workspace.
 *
 * Limit: at most ALLEN_VELO_NOALLOC_MAX_COUNTS counts per call (4 194 304 = 65 536 events x 64 layers; the array is
 * 2049 x 8 = 16 392 bytes, held by every GPU that loads the library until the process exits).
 *
 * Sharing: every call on a device uses the SAME array.  The call enqueues a clear of the words it needs before its
 * kernel, so calls that follow each other on one stream (or are otherwise ordered) are independent of what the array
 * held; calls that OVERLAP on the GPU (different streams without ordering, or two host threads at once) race on the
 * array and give wrong results or hang in the look-back.  One call at a time per device.
 */
#ifndef ALLEN_VELO_NOALLOC_H
#define ALLEN_VELO_NOALLOC_H

#include "allen_velo.h"

#ifdef __cplusplus
extern "C" {
#endif

#define ALLEN_VELO_NOALLOC_MAX_COUNTS 4194304u
#define ALLEN_VELO_ERR_TOO_LARGE (-4) /* n exceeds ALLEN_VELO_NOALLOC_MAX_COUNTS: nothing was enqueued */

/* offsets[i] = counts[0] + ... + counts[i-1] for i = 0..n (offsets[n] = total), modulo 2^32 like the path's own scan.
 *   counts       DEVICE [n]    (may be NULL when n == 0)
 *   offsets      DEVICE [n+1]  must not overlap counts
 *   cuda_stream  a cudaStream_t of the CURRENT device (NULL = legacy default stream); the call only enqueues
 *                (one memset of the scratch words + one kernel) and returns without synchronising
 *   error_text   HOST buffer of error_text_bytes bytes or NULL: receives a NUL-terminated message when the call fails
 * Calls no cudaMalloc / cudaFree / allocating library routine.  The first call on a device looks up the device address
 * of the scratch array (cudaGetSymbolAddress, once per device, with that device current): make that first call outside
 * stream capture.
 * Returns ALLEN_VELO_OK, ALLEN_VELO_ERR_INVALID (null pointer with n > 0), ALLEN_VELO_ERR_TOO_LARGE, or
 * ALLEN_VELO_ERR_CUDA (a runtime call failed; the text names it). */
int allen_velo_offsets_noalloc(const uint32_t* counts, uint32_t n, uint32_t* offsets, void* cuda_stream,
                               char* error_text, size_t error_text_bytes);

#ifdef __cplusplus
}
#endif
#endif /* ALLEN_VELO_NOALLOC_H */
