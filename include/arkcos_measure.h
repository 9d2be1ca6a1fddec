/*
 * arkcos_measure.h - measurement hooks of arkcos-b200.  NOT part of the product boundary (include/arkcos.h):
 * bench.py and the profiling commands under profiles/ use them to time the two kernels of the hot path and
 * the two classes of work items of step S3 separately (per-kernel roofline evidence).
 */
#ifndef ARKCOS_MEASURE_H_
#define ARKCOS_MEASURE_H_

#include "arkcos.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Flags of arkcos_plan_create_ex: launch only the WIDE (polar / high-latitude rings) or only the NARROW
 * (equatorial band) work items of step S3.  The output rings of the other class are NOT written.  Never
 * set both. */
#define ARKCOS_PLAN_ONLY_WIDE 4u
#define ARKCOS_PLAN_ONLY_NARROW 8u

/* Flag of arkcos_plan_create_ex, EXPERIMENT N1(a) (north_star: tensor cores only "if a ring-pair
 * circulant is recast as a genuinely dense contraction and ncu shows that it wins"): the WIDE work items run on the
 * tensor cores - per stage a banded-Toeplitz GEMM with warp-level mma.m16n8k8 TF32 instructions and a 3-term
 * hi/lo split of both operands that keeps FP32 accuracy (csrc/arkcos_tensor.cuh) - instead of the FFMA kernel.
 * Same plan, same work items, same weights; the result differs from the default path by FP32 rounding only and
 * meets the same tolerance against the oracle.  The NARROW items are not affected. */
#define ARKCOS_PLAN_WIDE_TENSOR 32u

/* Flag of arkcos_plan_create_ex: the scheduler puts EVERY ring into the WIDE class (no band marching), so that the
 * NARROW kernel can be measured against the WIDE kernel - FFMA or, with ARKCOS_PLAN_WIDE_TENSOR, tensor cores - on
 * the same rings.  A complete, correct convolution (the same sum in another order); only slower or faster. */
#define ARKCOS_PLAN_ALL_WIDE 64u

/*
 * arkcos_measure_convolve - one arkcos_convolve_batch on `stream` with CUDA events (created and destroyed
 * inside the call) around each kernel; synchronises the stream and returns the device time of the weight
 * generator (0 for cached plans) and of the convolution kernel, in milliseconds.  Arguments and errors as
 * arkcos_convolve_batch.
 */
arkcos_status arkcos_measure_convolve(const arkcos_plan *plan, const float *d_in, float *d_out, int n_maps,
                                      void *stream, float *ms_generate, float *ms_convolve);

/*
 * arkcos_plan_reserve_host_io_chunks - as arkcos_plan_reserve_host_io (include/arkcos.h), with the number of ring
 * bands of the arkcos_convolve_host pipeline given instead of derived from the map size (0 = derive it; clamped to
 * n_theta).  For tests of the pipeline on small maps and for tuning.  No effect once the staging is reserved.
 */
arkcos_status arkcos_plan_reserve_host_io_chunks(arkcos_plan *plan, int n_chunks);

/*
 * arkcos_plan_item - work item `index` (0 .. arkcos_plan_info.n_items - 1) of the convolution launch, in launch
 * order (heaviest first), so that tests can probe the seams of the schedule.  fields[6] receives:
 *   [0] class: 0 = WIDE (one output ring), 1 = NARROW (a band of rings of one hemisphere)
 *   [1] WIDE: the output ring.  NARROW: the first northern ring of the band
 *   [2] WIDE: 1.  NARROW: rings in the band; negative = the band is the southern mirror of rings [1] .. [1]-[2]-1
 *   [3] first output phi of the tile      [4] outputs of the tile in phi      [5] tap splits (WIDE) / rings per pass (NARROW)
 */
arkcos_status arkcos_plan_item(const arkcos_plan *plan, int index, int *fields);

/*
 * arkcos_plan_validate - re-runs the host-side schedule validation that arkcos_plan_create performs before
 * uploading (every global range and shared-memory offset the kernels form from the plan's descriptors is
 * re-derived and bounds-checked).  `why` (capacity `cap`, may be 0) receives the first failed check.
 * Returns ARKCOS_OK or ARKCOS_EINTERNAL.  Works on host-only plans.
 */
arkcos_status arkcos_plan_validate(const arkcos_plan *plan, char *why, int cap);

#ifdef __cplusplus
}
#endif
#endif /* ARKCOS_MEASURE_H_ */
