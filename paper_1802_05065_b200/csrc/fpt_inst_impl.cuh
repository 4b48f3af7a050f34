// fpt_inst_impl.cuh -- the lookup tables of fpt_inst.cuh for one state template (State64, State32 or State32Fast).
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
  template <int M, int S, bool A>
  static const void* pks() { return (const void*)&fpt_persistent_kernel<St<M, S, A, true>, true>; }      // with time slicing: ramped only
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
  template <int M, int S>
  static const void* pick_s(bool r) { return r ? sk<M, S, true>() : sk<M, S, false>(); }

  // scheme: 0 Euler-Maruyama, 1 stochastic Heun, 2 the paper's kernels as printed
  static const void* persistent(int model, int scheme, bool a, bool r) {
    if (model == 0) return scheme == 0 ? pick_p<0, 0>(a, r) : scheme == 1 ? pick_p<0, 1>(a, r) : pick_p<0, 2>(a, r);
    return scheme == 0 ? pick_p<1, 0>(a, r) : scheme == 1 ? pick_p<1, 1>(a, r) : pick_p<1, 2>(a, r);
  }
  template <int M, int S>
  static const void* pick_ps(bool a) { return a ? pks<M, S, true>() : pks<M, S, false>(); }
  static const void* persistent_sliced(int model, int scheme, bool a) {
    if (model == 0) return scheme == 0 ? pick_ps<0, 0>(a) : scheme == 1 ? pick_ps<0, 1>(a) : pick_ps<0, 2>(a);
    return scheme == 0 ? pick_ps<1, 0>(a) : scheme == 1 ? pick_ps<1, 1>(a) : pick_ps<1, 2>(a);
  }
  static const void* persistent_sliced_paper(int model) { return model == 0 ? pks<0, 2, true>() : pks<1, 2, true>(); }
  static const void* trace(int model, int scheme, bool a, bool r) {
    if (model == 0) return scheme == 0 ? pick_t<0, 0>(a, r) : scheme == 1 ? pick_t<0, 1>(a, r) : pick_t<0, 2>(a, r);
    return scheme == 0 ? pick_t<1, 0>(a, r) : scheme == 1 ? pick_t<1, 1>(a, r) : pick_t<1, 2>(a, r);
  }
  static const void* specialised(int model, int scheme, bool r, size_t* fixed_bytes, size_t* channel_bytes) {
    *fixed_bytes = spec_pool_bytes();
    *channel_bytes = spec_channel_bytes<St<0, 0, true, true>>();      // depends on the precision only
    if (model == 0) return scheme == 0 ? pick_s<0, 0>(r) : scheme == 1 ? pick_s<0, 1>(r) : pick_s<0, 2>(r);
    return scheme == 0 ? pick_s<1, 0>(r) : scheme == 1 ? pick_s<1, 1>(r) : pick_s<1, 2>(r);
  }
  // the paper's scheme only, with a sine (the hardware-sine variant): persistent kernel and tracer
  static const void* persistent_paper(int model, bool r) {
    if (model == 0) return r ? pk<0, 2, true, true>() : pk<0, 2, true, false>();
    return r ? pk<1, 2, true, true>() : pk<1, 2, true, false>();
  }
  static const void* trace_paper(int model, bool r) {
    if (model == 0) return r ? tk<0, 2, true, true>() : tk<0, 2, true, false>();
    return r ? tk<1, 2, true, true>() : tk<1, 2, true, false>();
  }
};

}  // namespace
}  // namespace fpt
