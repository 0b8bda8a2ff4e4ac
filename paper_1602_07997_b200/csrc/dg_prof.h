/* Development-only entry point of libdg (NOT part of include/dg.h and not exported by release builds): present only when
 * the library is built with -DDG_PROF (DG_PROF=1 python -m paper_1602_07997_b200.build --force), which also makes every
 * warp of the tensor-core stage kernel accumulate the cycles it spends in each kind of mbarrier wait (tc3_kernels.cuh,
 * T3_WAIT).  Timings of such a build are not bench numbers. */
#ifndef DG_PROF_H_
#define DG_PROF_H_
#ifdef DG_PROF
#include "../../include/dg.h"
#ifdef __cplusplus
extern "C" {
#endif
/* per-warp wait-cycle counters of the last tensor-core launch of the context's (model, degree):
 * out [296][23][5] int64 = {total cycles, wait kind 0..3} per (CTA, warp); synchronises the device */
int dg_prof_read(dg_ctx *ctx, long long *out);
#ifdef __cplusplus
}
#endif
#endif
#endif /* DG_PROF_H_ */
