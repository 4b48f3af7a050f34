// fpt_inst64.cu -- instantiations of the integrator kernels and the tracer for the fp64 state (see fpt_inst.cuh).
#include "fpt_inst_impl.cuh"

namespace fpt {

const void* persistent_kernel_f64(int model, int scheme, bool amp, bool ramp) { return Inst<State64>::persistent(model, scheme, amp, ramp); }
const void* persistent_sliced_kernel_f64(int model, int scheme, bool amp) { return Inst<State64>::persistent_sliced(model, scheme, amp); }
const void* specialised_kernel_f64(int model, int scheme, bool ramp, size_t* fixed_bytes, size_t* channel_bytes) {
  return Inst<State64>::specialised(model, scheme, ramp, fixed_bytes, channel_bytes);
}
const void* trace_kernel_f64(int model, int scheme, bool amp, bool ramp) { return Inst<State64>::trace(model, scheme, amp, ramp); }

}  // namespace fpt
