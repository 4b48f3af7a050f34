// fpt_inst.cuh -- kernel-pointer tables.  The 2 x 16 instantiations of the persistent kernel are split over two
// translation units (fpt_inst64.cu, fpt_inst32.cu) so that they compile in parallel; the API unit only sees these
// lookups.
#pragma once
#include <cuda_runtime.h>

namespace fpt {

// persistent integrator for (model, scheme, amp != 0, nu != 0)
const void* persistent_kernel_f64(int model, int scheme, bool amp, bool ramp);
const void* persistent_kernel_f32(int model, int scheme, bool amp, bool ramp);
// single-trajectory tracer (test hook), general amp / ramp code path
const void* trace_kernel_f64(int model, int scheme);
const void* trace_kernel_f32(int model, int scheme);

}  // namespace fpt
