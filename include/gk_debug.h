/* gk_debug.h -- instrumentation entry points of libgk used by bench.py and the tests; not part of the hot-path
 * API of gk.h (same library, same conventions). */
#ifndef GK_DEBUG_H
#define GK_DEBUG_H
#include "gk.h"
#ifdef __cplusplus
extern "C" {
#endif

/* Number of kernel launches issued through this context so far (bench.py's gpu_launches). */
long long gk_launch_count(const gk_ctx *ctx);
/* CUDA-event time (ms) spent in the stage kernel since the last call with reset!=0, and the number
 * of stage-kernel launches in that interval; events are recorded on the context stream only while
 * profiling is enabled with gk_set_profiling(ctx, 1).  Synchronises the stream. */
int gk_set_profiling(gk_ctx *ctx, int on);
int gk_stage_kernel_time(gk_ctx *ctx, double *ms_total, long long *launches, int reset);

#ifdef __cplusplus
}
#endif
#endif
