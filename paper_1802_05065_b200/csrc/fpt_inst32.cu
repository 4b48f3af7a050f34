// fpt_inst32.cu -- instantiations of the integrator kernels and the tracer for the fp32 state (see fpt_inst.cuh).
#include "fpt_inst_impl.cuh"

namespace fpt {

const void* persistent_kernel_f32(int model, int scheme, bool amp, bool ramp) { return Inst<State32>::persistent(model, scheme, amp, ramp); }
const void* persistent_sliced_kernel_f32(int model, int scheme, bool amp) { return Inst<State32>::persistent_sliced(model, scheme, amp); }
const void* specialised_kernel_f32(int model, int scheme, bool ramp, size_t* fixed_bytes, size_t* channel_bytes) {
  return Inst<State32>::specialised(model, scheme, ramp, fixed_bytes, channel_bytes);
}
const void* trace_kernel_f32(int model, int scheme, bool amp, bool ramp) { return Inst<State32>::trace(model, scheme, amp, ramp); }

// fp32 state with the hardware sine (FPT_PREC_FP32_FAST): the paper's scheme with a sine only
const void* persistent_kernel_f32_fast(int model, bool ramp) { return Inst<State32Fast>::persistent_paper(model, ramp); }
const void* persistent_sliced_kernel_f32_fast(int model) { return Inst<State32Fast>::persistent_sliced_paper(model); }
const void* trace_kernel_f32_fast(int model, bool ramp) { return Inst<State32Fast>::trace_paper(model, ramp); }

}  // namespace fpt
