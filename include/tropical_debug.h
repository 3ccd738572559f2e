/*
 * tropical_debug.h -- TEST AND MEASUREMENT HOOKS of libtropical.so.  Not part of the product ABI (include/tropical.h):
 * production callers need none of these.  The two set_* hooks keep process-global state (atomics) that every later
 * tropical_mixed_attention of the process sees; tests reset them in a finally block.
 */
#ifndef TROPICAL_DEBUG_H_
#define TROPICAL_DEBUG_H_

#include "tropical.h"

#ifdef __cplusplus
extern "C" {
#endif

/* The plain CUDA-core (no tensor core, no split-K) attention kernel, same arguments and semantics as
 * tropical_mixed_attention without a workspace.  A device-side cross-check of the tile kernels (CUDA against CUDA: an
 * extra, not parity -- parity is against oracle/); never on a product path. */
int tropical_debug_attention_simt(const tropical_kv_pool_t *pool, const tropical_batch_t *batch,
                                  const void *q, void *out, float *lse, float sm_scale,
                                  void *cuda_stream);

/* Cap the number of CTAs of the persistent step kernel (0 = one per SM, the default), so that small test batches put
 * MANY tiles through each CTA's queues (multi-item sequencing of every role). */
void tropical_debug_set_grid(int num_ctas);

/* Coarsen the decode split size to `pages` pages (rounded up to a multiple of 8; 0 = automatic), so that small test
 * batches exercise multi-block decode units and so that two runs with different head counts can be given the same
 * split boundaries.  It can only raise the split above the automatic value (the workspace bound of
 * tropical_workspace_bytes assumes split >= automatic): a smaller value is ignored. */
void tropical_debug_set_split_pages(int pages);

/* tropical_mixed_step chooses between its fused kernel variant (append inside the step kernel) and the append kernel in
 * front of the plain variant from the batch scalars (prefill-dominated steps fuse).  mode 1 / 0 forces the fused variant
 * on / off for every step, so that tests put every batch shape through both; -1 restores the choice. */
void tropical_debug_set_fused(int mode);

/* Only in special builds (else TROPICAL_ERR_UNSUPPORTED).  Synchronises the device.
 *  -DTROPICAL_WAIT_PROF: cycles spent in and calls of every mbarrier wait of the step kernel, summed over warps,
 *    indexed by the wait's tag (the numbers next to the mbar_wait calls in csrc/); reset != 0 zeroes the counters.
 *  -DTROPICAL_DEBUG_WAIT: instead of trapping, a wait that is stuck for ~0.2 s raises an abort flag that lets every
 *    wait fall through (the step finishes with garbage); cycles[0] = that flag and, for warp w of CTA 0,
 *    cycles[16 + 3 w .. + 2] = tag, parity and aux value of the wait it was stuck in.  The record lives in
 *    host-mapped memory, so it can be read even when the kernel faulted afterwards.
 * cycles / calls are [host] arrays of n <= 512 entries. */
int tropical_debug_wait_profile(uint64_t *cycles, uint64_t *calls, int32_t n, int32_t reset);

/* Role timestamps of the LAST fused step kernel that ran with this workspace (globaltimer nanoseconds): out_ns[0]
 * kernel start (earliest CTA), [1] prefill queue drained (latest softmax warp), [2] latest dedicated decode warp done,
 * [3] latest late-joining decode warp done.  Copies 32 bytes device->host and synchronises the stream. */
int tropical_debug_read_profile(const void *workspace, uint64_t *out_ns, void *cuda_stream);

/* Only in builds with -DTROPICAL_TIMELINE (else TROPICAL_ERR_UNSUPPORTED): global-timer stamps (ns) of the three
 * kernels of the last step(s) since the last reset -- out_ns[0] append start, [1] append end, [2] tile directory start,
 * [3] directory body end, [4] directory end (after its wait on the append), [5] step kernel start, [6] its prologue end
 * (last CTA), [7] its first CTA past griddepcontrol.wait, [8] its end.  Starts are minima over blocks, ends maxima.
 * out_ns [host, nullable] 9 entries; reset != 0 re-arms the stamps.  Synchronises the device.  This is how the overlap
 * of the directory kernel and of the step kernel's prologue with the append was measured (profiles/). */
int tropical_debug_timeline(uint64_t *out_ns, int32_t reset);

#ifdef __cplusplus
}
#endif
#endif /* TROPICAL_DEBUG_H_ */
