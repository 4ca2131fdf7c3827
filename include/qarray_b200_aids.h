/*
 * qarray_b200_aids.h -- measurement and cross-check aids of libqarray_b200.so.  NOT part of the product surface
 * (include/qarray_b200.h): bench.py and the tests use these to time individual kernels, to measure the FP64 issue rate
 * that the ALU roofline divides by, and to force a particular kernel for cross-checks.
 */
#ifndef QARRAY_B200_AIDS_H
#define QARRAY_B200_AIDS_H

#include "qarray_b200.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Sustained FP64 issue rate of the current device: independent DFMA chains on every SM for about `seconds`.
 * Returns FP64 thread-instructions per second (1 DFMA = 1) -- the denominator of the ALU roofline. */
QA_API qa_status qa_measure_fp64_rate(double seconds, double *thread_inst_per_s, void *cuda_stream);

/* Per-kernel timing of a call (per host thread).  While enabled, the ground-state / thermal calls record CUDA events on the
 * call's stream before the first and after every kernel.  qa_get_kernel_timings waits for the last event of the most
 * recent call and returns the device time of each of its kernels in milliseconds, in launch order (names:
 * qa_last_launch_plan).  ms: host, max_kernels floats; *n_kernels: how many were written. */
QA_API qa_status qa_set_kernel_timing(int enable);
QA_API qa_status qa_get_kernel_timings(int max_kernels, float *ms, int *n_kernels);

/* Kernel selection of ONE model (cross-check aid; the results are identical): 0 = the three-kernel path with the
 * exact-compare walk / the generic enumeration for every n_dot, 1 (default) = the production dispatch of DESIGN.md
 * section 5, 2 = as 1, but the open default search of n_dot >= 13 skips the high patterns a rigorous lower bound excludes
 * (same arg min; fewer candidates are scored explicitly), 3 = as 1, but pass 1 of that search bounds every candidate in fp32
 * (packed adds, explicit error bound) and the fp64 pass 2 re-scores the threads the bound cannot exclude: charge map and
 * energies bit-identical to variant 1 (the "fp32 walk, fp64 re-score" path of SURVEY 8(f) NEXT-4), 4 = as 1, but the open
 * default search of a 16-dot Maxwell array without sensor dots runs S1-S7 in ONE persistent kernel that touches no workspace
 * (qa_minplus_fused_kernel; same arithmetic, bit-identical results; measured 4 % slower than the
 * three launches, hence opt-in).  Stored in the model (atomically); calls already enqueued are
 * not affected.  Returns QA_ERR_INVALID_ARG for any other value.  The initial value of every model comes from the
 * environment variable QA_WALK_VARIANT (default 1). */
QA_API qa_status qa_model_set_walk_variant(qa_model *model, int variant);

/* Names of the kernels the last call on this host thread enqueued (comma separated; thread-local storage). */
QA_API const char *qa_last_launch_plan(void);
/* Number of kernels the last call on this host thread enqueued. */
QA_API int qa_last_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* QARRAY_B200_AIDS_H */
