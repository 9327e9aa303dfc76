/*
 * cwo_debug.h -- measurement hooks of libcwo.so for the test and bench harness.  NOT part of the product
 * boundary (include/cwo.h): nothing here changes what a call computes.  With timing on, the propagation calls
 * create and record CUDA events, so they are no longer "enqueue only" (do not capture them into a graph).
 */
#ifndef CWO_DEBUG_H_
#define CWO_DEBUG_H_

#include "cwo.h"

#ifdef __cplusplus
extern "C" {
#endif

/* on = 1: bracket every pass kernel with a CUDA event pair on the plan's stream; 0 (default): off. */
int cwo_debug_set_timing(cwo_plan_t plan, int on);

/* With timing on: synchronises the plan's stream, writes the device time in ms of each pass kernel launched
 * since timing was switched on / since the last call (at most cap entries; tag_out, if not NULL, receives
 * log2(transform length)*16 + kind, kind 0 = row FFT, 1 = row IFFT, 2 = column FFT, 3 = fused column FFT x H x
 * IFFT, 4 = H x column IFFT, 5 = fused line convolution(s) of the separable Fresnel form, 6 = transpose),
 * clears the record and returns the number of launches recorded (may exceed cap), or a negative error. */
int cwo_debug_timings(cwo_plan_t plan, float* ms_out, int* tag_out, int cap);

/* Number of kernels the library has launched through this plan so far (bench accounting). */
long long cwo_debug_launch_count(cwo_plan_t plan);

/* on = 1: cwo_fresnel_conv and cwo_gs (Fresnel) use the three-pass two-dimensional form (row FFT, fused column
 * pass with Cx[k] Cy[l], row IFFT) also for the sizes where the separable line-convolution form exists
 * (256..8192 per axis); 0 (default): separable form where it exists.  Same result either way (comparison runs). */
int cwo_debug_set_fresnel_2d(cwo_plan_t plan, int on);

/* The separable Fresnel form (cwo_fresnel_conv, cwo_fresnel_shifted, cwo_gs) has two ways of switching axes: transpose
 * passes between contiguous line passes, or line passes that gather their lines from the columns of their input.
 * mode -1 (default): chosen by field size (gathering up to 2048 x 2048 samples, where the field stays in L2);
 * 0: always transposing; 1: always gathering.  Same result either way (parity tests run both). */
int cwo_debug_set_fresnel_gather(cwo_plan_t plan, int mode);

#ifdef __cplusplus
}
#endif
#endif /* CWO_DEBUG_H_ */
