// fpt_inst32.cu -- instantiations of the persistent integrator and the tracer for the fp32 state (see fpt_inst.cuh).
#include "fpt_inst.cuh"
#include "fpt_integrator.cuh"

namespace fpt {

namespace {
template <int M, int S, bool A, bool R>
const void* pk() {
  return (const void*)&fpt_persistent_kernel<State32<M, S, A, R>>;
}
template <int M, int S>
const void* pick_ar(bool a, bool r) {
  if (a) return r ? pk<M, S, true, true>() : pk<M, S, true, false>();
  return r ? pk<M, S, false, true>() : pk<M, S, false, false>();
}
}  // namespace

const void* persistent_kernel_f32(int model, int scheme, bool amp, bool ramp) {
  if (model == 0) return scheme == 0 ? pick_ar<0, 0>(amp, ramp) : pick_ar<0, 1>(amp, ramp);
  return scheme == 0 ? pick_ar<1, 0>(amp, ramp) : pick_ar<1, 1>(amp, ramp);
}

const void* trace_kernel_f32(int model, int scheme) {
  if (model == 0)
    return scheme == 0 ? (const void*)&fpt_trace_kernel<State32<0, 0, true, true>>
                       : (const void*)&fpt_trace_kernel<State32<0, 1, true, true>>;
  return scheme == 0 ? (const void*)&fpt_trace_kernel<State32<1, 0, true, true>>
                     : (const void*)&fpt_trace_kernel<State32<1, 1, true, true>>;
}

}  // namespace fpt
