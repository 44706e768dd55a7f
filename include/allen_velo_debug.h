/* allen_velo_debug.h — measurement hooks of the VELO library (not part of the product ABI of allen_velo.h).
 *
 * bench.py uses them for the per-kernel times of its roofline lines and for `gpu_launches`; the
 * tests use the launch count to show that the CUDA path ran.  Same handle, same library.
 */
#ifndef ALLEN_VELO_DEBUG_H
#define ALLEN_VELO_DEBUG_H

#include "allen_velo.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Optional per-kernel timing: keeps a ring of CUDA events for the next `n_calls`
 * reconstruct() calls (n_calls = 0 switches it off and frees the events).  Events are recorded on the caller's
 * stream between the kernels; nothing synchronises. */
int allen_velo_enable_timing(allen_velo_t* handle, uint32_t n_calls);

/* Kernels launched per reconstruct() call and their names (static strings), in launch order. */
uint32_t allen_velo_kernel_count(void);
const char* allen_velo_kernel_name(uint32_t i);

/* Device time in ms of each kernel of call number `call` (0-based since enable_timing, modulo the ring size).
 * out_ms: HOST [allen_velo_kernel_count()].  The caller must have synchronised the stream first. */
int allen_velo_kernel_times(allen_velo_t* handle, uint32_t call, float* out_ms /* HOST out */);

/* Number of kernels the last reconstruct() call launched (bench.py's gpu_launches). */
uint32_t allen_velo_last_launch_count(const allen_velo_t* handle);

/* Bounds checks (the library built with -DVELO_DEBUG: paper_1912_09161_b200/build.py --debug).  1 if this library was
 * built with them.  allen_velo_debug_fault: the highest code of a check that failed since the last call of this function
 * (0 = none; codes in csrc/velo_common.cuh), read from the device (SYNCHRONISES) and cleared. */
int allen_velo_debug_checks_compiled(void);
int allen_velo_debug_fault(allen_velo_t* handle, uint32_t* out /* HOST out */);

/* List sizes of the track search of the last reconstruct() call, copied from the workspace (SYNCHRONISES the device):
 * out[0..2] events searched by the three instances of velo_follow_kernel (at most 256 / 512 / 1024 hits per layer),
 * out[12], out[13] events handed on to the CTA-per-event kernel with 512 / 1024 hits per layer (candidate list or
 * track slots exhausted).  out: HOST [16]. */
int allen_velo_debug_track_counters(allen_velo_t* handle, uint32_t* out /* HOST out */);

#ifdef __cplusplus
}
#endif
#endif /* ALLEN_VELO_DEBUG_H */
