// fpt_inst_impl.cuh -- the lookup tables of fpt_inst.cuh for one state template (State64 or State32).
#pragma once
#include "fpt_inst.cuh"
#include "fpt_integrator.cuh"
#include "fpt_specialised.cuh"

namespace fpt {
namespace {

template <template <int, int, bool, bool> class St>
struct Inst {
  template <int M, int S, bool A, bool R>
  static const void* pk() { return (const void*)&fpt_persistent_kernel<St<M, S, A, R>>; }
  template <int M, int S, bool A, bool R>
  static const void* tk() { return (const void*)&fpt_trace_kernel<St<M, S, A, R>>; }
  template <int M, int S, bool R>
  static const void* sk() { return (const void*)&fpt_specialised_kernel<St<M, S, true, R>>; }

  template <int M, int S>
  static const void* pick_p(bool a, bool r) {
    if (a) return r ? pk<M, S, true, true>() : pk<M, S, true, false>();
    return r ? pk<M, S, false, true>() : pk<M, S, false, false>();
  }
  template <int M, int S>
  static const void* pick_t(bool a, bool r) {
    if (a) return r ? tk<M, S, true, true>() : tk<M, S, true, false>();
    return r ? tk<M, S, false, true>() : tk<M, S, false, false>();
  }
  static const void* persistent(int model, int scheme, bool a, bool r) {
    if (model == 0) return scheme == 0 ? pick_p<0, 0>(a, r) : pick_p<0, 1>(a, r);
    return scheme == 0 ? pick_p<1, 0>(a, r) : pick_p<1, 1>(a, r);
  }
  static const void* trace(int model, int scheme, bool a, bool r) {
    if (model == 0) return scheme == 0 ? pick_t<0, 0>(a, r) : pick_t<0, 1>(a, r);
    return scheme == 0 ? pick_t<1, 0>(a, r) : pick_t<1, 1>(a, r);
  }
  static const void* specialised(int model, int scheme, bool r, size_t* fixed_bytes, size_t* channel_bytes) {
    *fixed_bytes = spec_pool_bytes();
    *channel_bytes = spec_channel_bytes<St<0, 0, true, true>>();      // depends on the precision only
    if (model == 0) {
      if (scheme == 0) return r ? sk<0, 0, true>() : sk<0, 0, false>();
      return r ? sk<0, 1, true>() : sk<0, 1, false>();
    }
    if (scheme == 0) return r ? sk<1, 0, true>() : sk<1, 0, false>();
    return r ? sk<1, 1, true>() : sk<1, 1, false>();
  }
};

}  // namespace
}  // namespace fpt
