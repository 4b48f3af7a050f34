// fpt_inst.cuh -- kernel-pointer tables.  The 2 x (16 + 8) instantiations of the two integrator kernels are split over
// two translation units (fpt_inst64.cu, fpt_inst32.cu) so that they compile in parallel; the API unit only sees these
// lookups.
#pragma once
#include <cstddef>
#include <cuda_runtime.h>

namespace fpt {

// persistent integrator for (model, scheme, amp != 0, nu != 0)
const void* persistent_kernel_f64(int model, int scheme, bool amp, bool ramp);
const void* persistent_kernel_f32(int model, int scheme, bool amp, bool ramp);
// the same with the time-slicing code (ramped bias only: nu != 0)
const void* persistent_sliced_kernel_f64(int model, int scheme, bool amp);
const void* persistent_sliced_kernel_f32(int model, int scheme, bool amp);
const void* persistent_sliced_kernel_f32_fast(int model);
// warp-specialised integrator (drifts with a sine only: amp != 0); dynamic shared memory = *fixed_bytes + consumers x
// *channel_bytes (+ the histogram bins)
const void* specialised_kernel_f64(int model, int scheme, bool ramp, size_t* fixed_bytes, size_t* channel_bytes);
const void* specialised_kernel_f32(int model, int scheme, bool ramp, size_t* fixed_bytes, size_t* channel_bytes);
// single-trajectory tracer (test hook): the same State specialisation the production launch picks
const void* trace_kernel_f64(int model, int scheme, bool amp, bool ramp);
const void* trace_kernel_f32(int model, int scheme, bool amp, bool ramp);

// fp32 state with the hardware sine: scheme 2 (the paper's kernels as printed) with amp != 0 only
const void* persistent_kernel_f32_fast(int model, bool ramp);
const void* trace_kernel_f32_fast(int model, bool ramp);

}  // namespace fpt
