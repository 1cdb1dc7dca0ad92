/*
 * xcorr_debug.h -- host-logic introspection of libxcorr.so (no GPU needed, no kernels): the work schedule
 * xcorr_create() builds, for the CPU tests of the decomposition.  xcorr_process()/xcorr_read() never call these.
 */
#ifndef XCORR_DEBUG_H_
#define XCORR_DEBUG_H_

#include <stdint.h>
#include "xcorr.h"

#ifdef __cplusplus
extern "C" {
#endif

/*
 * The host-side work decomposition xcorr_create() would build for `n_workers` CTA pairs (no GPU needed).
 * A work item is a 256 x 256 super-tile (f, I <= J) of the visibility matrix ("computes only upper-triangle
 * tiles", BASELINE.json:north_star (b)); it is cut along time into stages of xcorr_debug_stage_samples()
 * samples and the stages are dealt to workers.
 * Returns the number of segments (>= 0) or XCORR_EINVAL.  With non-NULL outputs writes
 * segments_out[k][7] = {f, I, J, stage_begin, stage_end, tile, slot} (capacity max_segments) and
 * worker_begin_out[n_workers + 1].
 */
int xcorr_debug_schedule(int n_inputs, int n_freq, int t_per_frame, int n_workers,
                         int32_t *segments_out, int max_segments, int32_t *worker_begin_out);

/* Time samples per pipeline stage. */
int xcorr_debug_stage_samples(void);

#ifdef __cplusplus
}
#endif
#endif /* XCORR_DEBUG_H_ */
