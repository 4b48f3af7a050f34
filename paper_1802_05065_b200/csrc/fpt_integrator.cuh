// fpt_integrator.cuh -- the persistent integrator kernel.
//
// One lane = one trajectory of Eq. (9) at a time, state (phi, v, k) in registers.  Lanes of a warp stay
// converged: every K steps the warp votes on which lanes have finished (first crossing, or the step
// cap klim), finished lanes write their results indexed by trajectory id and take new ids from a
// global counter through ONE atomic per warp ("assigns a new job to the processor as soon as it has
// terminated its task", done here without the host).  The crossing test itself is evaluated after EVERY step as a
// sticky capture (reading R6), so results never depend on K or on the launch geometry.
#pragma once
#include "fpt_math.cuh"

namespace fpt {

constexpr int kStatusEscaped = 0, kStatusCensored = 1, kStatusNan = 2;
constexpr int kMaxFusedBins = 8192;
constexpr int kScheduleDynamic = 0, kScheduleStatic = 1;

struct DevStats {                 // device-side counters, one block of 8 x u64
  unsigned long long next_id;     // the global trajectory counter (S7)
  unsigned long long n_escaped, n_censored, n_nan;
  unsigned long long useful_steps, issued_lane_steps, refill_atomics, migrations;
};

struct KParams {
  // derived on the host in fp64; fp32 kernels read the *_f copies (each rounded once)
  double alpha, amp, gamma0, dgamma, phi0, v0, thr, dt, sigma, h2;
  float alpha_f, amp_f, gamma0_f, nu_f, phi0_f, v0_f, thr_f, dt_f, sigma_f, h2_f;
  unsigned long long n_traj, first_id, n_cap;
  int K;                          // poll interval in steps, a multiple of the macro step
  int hist_of;                    // -1 none, 0 gamma at escape, 1 escape time
  int schedule;                   // kScheduleDynamic (refill from the global counter + drain compaction) | kScheduleStatic
  int nbins;
  double hist_lo, hist_scale;
  double* out_fpt;
  double* out_gamma;
  int* out_status;
  unsigned long long* out_counts;
  DevStats* ws;
  PhiloxKeys keys;
};

// A trajectory parked between two polls (drain-phase lane compaction, see the persistent kernel): everything that is
// not a pure function of (id, k).  The normals of the next macro step and the ramp registers are recomputed on adoption.
struct ParkSlot {
  unsigned long long a, b;        // fp64: bits of phi, v;  fp32: (phi, v) and the Kahan pair (t, c), two floats per word
  unsigned long long kbase, idx;
};

// ---------------------------------------------------------------------------------------------------------------
// S3-S5 fp64 state and the four recurrences.  gamma_j = fma(dgamma, (double)j, gamma0);
// F(phi, j) = fma(-amp, sin phi, gamma_j); AMP == false skips the sine, RAMP == false fixes gamma_j = gamma0 (R15).
template <int MODEL, int SCHEME, bool AMP, bool RAMP>
struct State64 {
  static constexpr int kMacro = 2;            // steps per Philox block
  double phi, v;
  double kd;                                  // (double) k, exact below 2^53; only kept when RAMP
  double g;                                   // gamma_k at the current k; only kept when RAMP

  __device__ __forceinline__ void init(const KParams& P) {
    phi = P.phi0;
    v = P.v0;
    kd = 0.0;
    g = P.gamma0;                             // fma(dgamma, 0, gamma0)
  }
  __device__ __forceinline__ double force(const KParams& P, double x, double gam) const {
    return AMP ? __fma_rn(-P.amp, sin_drift(x), gam) : gam;
  }
  __device__ __forceinline__ void step(const KParams& P, double z) {
    const double g1 = RAMP ? g : P.gamma0;    // gamma_{k-1}
    double g2 = g1;                           // gamma_k
    if (RAMP) {
      kd = __dadd_rn(kd, 1.0);
      g2 = __fma_rn(P.dgamma, kd, P.gamma0);
      g = g2;
    }
    if (MODEL == 0) {
      const double f1 = force(P, phi, g1);
      const double phip = __fma_rn(P.sigma, z, __fma_rn(f1, P.dt, phi));
      if (SCHEME == 0) {
        phi = phip;                           // Euler-Maruyama
      } else {                                // stochastic Heun, additive noise: the same z in both stages
        const double f2 = force(P, phip, g2);
        phi = __fma_rn(P.sigma, z, __fma_rn(P.h2, __dadd_rn(f1, f2), phi));
      }
    } else if (SCHEME == 0) {
      const double a1 = __fma_rn(-P.alpha, v, force(P, phi, g1));
      const double phip = __fma_rn(v, P.dt, phi);                              // both from the OLD state (Alg. 1 l. 11-12)
      const double vp = __fma_rn(P.sigma, z, __fma_rn(a1, P.dt, v));
      phi = phip;
      v = vp;
    } else {
      // Heun: the predictor phi_p does not depend on the first force, so both sines are evaluated side by side
      const double phip = __fma_rn(v, P.dt, phi);
      double f1 = g1, f2 = g2;
      if (AMP) {
        double s1, s2;
        sin_drift2(phi, phip, s1, s2);
        f1 = __fma_rn(-P.amp, s1, g1);
        f2 = __fma_rn(-P.amp, s2, g2);
      }
      const double a1 = __fma_rn(-P.alpha, v, f1);
      const double vp = __fma_rn(P.sigma, z, __fma_rn(a1, P.dt, v));
      const double a2 = __fma_rn(-P.alpha, vp, f2);
      phi = __fma_rn(P.h2, __dadd_rn(v, vp), phi);
      v = __fma_rn(P.sigma, z, __fma_rn(P.h2, __dadd_rn(a1, a2), v));
    }
  }
  __device__ __forceinline__ void park(ParkSlot& s) const {
    s.a = (unsigned long long)__double_as_longlong(phi);
    s.b = (unsigned long long)__double_as_longlong(v);
  }
  // k is a poll boundary; kd and gamma_k are exact functions of k (the running g is always fma(dgamma, kd, gamma0))
  __device__ __forceinline__ void unpark(const KParams& P, const ParkSlot& s, unsigned long long k) {
    phi = __longlong_as_double((long long)s.a);
    v = __longlong_as_double((long long)s.b);
    kd = __ull2double_rn(k);
    g = __fma_rn(P.dgamma, kd, P.gamma0);
  }
  __device__ __forceinline__ bool crossed(const KParams& P) const { return !(phi < P.thr); }   // phi >= thr, or NaN
  __device__ __forceinline__ bool is_nan_hi(int hi) const { return ((unsigned)hi & 0x7fffffffu) > 0x7ff00000u; }
  __device__ __forceinline__ int phi_hi() const { return __double2hiint(phi); }
  __device__ __forceinline__ double phi_as_double() const { return phi; }
  __device__ __forceinline__ double v_as_double() const { return v; }
  // the normals of one Philox block
  __device__ __forceinline__ static void normals(uint32_t o0, uint32_t o1, uint32_t o2, uint32_t o3, double (&z)[2]) {
    normal_pair(o0, o1, o2, o3, z[0], z[1]);
  }
  typedef double real;
};

// fp32 state + Kahan-compensated time: gamma for stage 1 uses t before the Kahan update, stage 2 after.
template <int MODEL, int SCHEME, bool AMP, bool RAMP>
struct State32 {
  static constexpr int kMacro = 4;
  float phi, v;
  float t, c;                                 // Kahan pair; only kept when RAMP

  __device__ __forceinline__ void init(const KParams& P) {
    phi = P.phi0_f;
    v = P.v0_f;
    t = 0.0f;
    c = 0.0f;
  }
  __device__ __forceinline__ float force(const KParams& P, float x, float gam) const {
    return AMP ? __fmaf_rn(-P.amp_f, sin_drift_f(x), gam) : gam;
  }
  __device__ __forceinline__ void step(const KParams& P, float z) {
    float g1 = P.gamma0_f, g2 = P.gamma0_f;
    if (RAMP) {
      g1 = __fmaf_rn(P.nu_f, t, P.gamma0_f);
      const float y = __fadd_rn(P.dt_f, -c);
      const float s = __fadd_rn(t, y);
      c = __fadd_rn(__fadd_rn(s, -t), -y);
      t = s;
      g2 = __fmaf_rn(P.nu_f, t, P.gamma0_f);
    }
    if (MODEL == 0) {
      const float f1 = force(P, phi, g1);
      const float phip = __fmaf_rn(P.sigma_f, z, __fmaf_rn(f1, P.dt_f, phi));
      if (SCHEME == 0) {
        phi = phip;
      } else {
        const float f2 = force(P, phip, g2);
        phi = __fmaf_rn(P.sigma_f, z, __fmaf_rn(P.h2_f, __fadd_rn(f1, f2), phi));
      }
    } else {
      const float a1 = __fmaf_rn(-P.alpha_f, v, force(P, phi, g1));
      const float phip = __fmaf_rn(v, P.dt_f, phi);
      const float vp = __fmaf_rn(P.sigma_f, z, __fmaf_rn(a1, P.dt_f, v));
      if (SCHEME == 0) {
        phi = phip;
        v = vp;
      } else {
        const float a2 = __fmaf_rn(-P.alpha_f, vp, force(P, phip, g2));
        phi = __fmaf_rn(P.h2_f, __fadd_rn(v, vp), phi);
        v = __fmaf_rn(P.sigma_f, z, __fmaf_rn(P.h2_f, __fadd_rn(a1, a2), v));
      }
    }
  }
  __device__ __forceinline__ void park(ParkSlot& s) const {
    s.a = ((unsigned long long)(unsigned)__float_as_int(v) << 32) | (unsigned)__float_as_int(phi);
    s.b = ((unsigned long long)(unsigned)__float_as_int(c) << 32) | (unsigned)__float_as_int(t);
  }
  __device__ __forceinline__ void unpark(const KParams&, const ParkSlot& s, unsigned long long) {
    phi = __int_as_float((int)(unsigned)s.a);
    v = __int_as_float((int)(unsigned)(s.a >> 32));
    t = __int_as_float((int)(unsigned)s.b);
    c = __int_as_float((int)(unsigned)(s.b >> 32));
  }
  __device__ __forceinline__ bool crossed(const KParams& P) const { return !(phi < P.thr_f); }
  __device__ __forceinline__ bool is_nan_hi(int hi) const { return ((unsigned)hi & 0x7fffffffu) > 0x7f800000u; }
  __device__ __forceinline__ int phi_hi() const { return __float_as_int(phi); }
  __device__ __forceinline__ double phi_as_double() const { return (double)phi; }
  __device__ __forceinline__ double v_as_double() const { return (double)v; }
  __device__ __forceinline__ static void normals(uint32_t o0, uint32_t o1, uint32_t o2, uint32_t o3, float (&z)[4]) {
    normal_pair_f(o0, o1, z[0], z[1]);
    normal_pair_f(o2, o3, z[2], z[3]);
  }
  typedef float real;
};

// ---------------------------------------------------------------------------------------------------------------
// S8: bin rule of DESIGN.md 4.11 (R10).  Returns the slot in [under, bins..., over], or -1 for a NaN value.
__device__ __forceinline__ int hist_slot(double x, double lo, double scale, int nbins) {
  const double t = __dmul_rn(__dadd_rn(x, -lo), scale);
  if (t != t) return -1;
  if (t < 0.0) return 0;
  if (t >= (double)nbins) return nbins + 1;
  return 1 + (int)__double2ll_rd(t);
}

// ---------------------------------------------------------------------------------------------------------------
// The persistent kernel.  Grid = (#SM x resident blocks); each warp loops { poll+refill ; K steps } until the global
// counter is exhausted and all of its lanes are idle.
// Launch bounds steer ptxas' scheduler: with a minimum-blocks figure it assumes few resident warps and interleaves the
// independent FP64 chains of a step (two Heun sines, the log / sin / cos polynomials of the next normals), which is
// what a warp needs when it runs nearly alone (drain phase, under-filled configs); without one it serialises every
// chain behind its 8-cycle DFMA latency and relies on other warps.
#ifndef FPT_LB_THREADS
#define FPT_LB_THREADS 256
#endif
#ifndef FPT_LB_MINBLOCKS
#define FPT_LB_MINBLOCKS 1
#endif
#ifndef FPT_UNROLL
#define FPT_UNROLL 4
#endif
constexpr int kUnroll = FPT_UNROLL;     // macro steps per trip of the step loop (a larger basic block schedules better)
constexpr int kMaxWarpsPerBlock = FPT_LB_THREADS / 32;

// Drain-phase lane compaction (per block, shared memory).  Once the global id counter is exhausted a warp cannot refill
// its finished lanes; without help it would keep issuing full-width instructions for its last few trajectories.  Here a
// warp whose live lanes fit into the holes of the block's other warps PARKS them in `slots` and retires; warps with
// holes ADOPT parked trajectories at their next poll.  Invariant (under `lock`): n_parked <= sum of holes[] over the
// live warps that have seen exhaustion, so every parked trajectory is adopted and a warp that finds nothing left to do
// may retire.  Results cannot change: a trajectory's state at a poll boundary is (phi, v[, t, c], k), everything else is
// recomputed from (id, k).
struct DrainPool {
  int lock;
  int n_parked;
  int holes[kMaxWarpsPerBlock];
  ParkSlot slots[FPT_LB_THREADS];
};

#if FPT_LB_MINBLOCKS > 0
#define FPT_LAUNCH_BOUNDS __launch_bounds__(FPT_LB_THREADS, FPT_LB_MINBLOCKS)
#else
#define FPT_LAUNCH_BOUNDS __launch_bounds__(FPT_LB_THREADS)
#endif

template <class S>
__global__ void FPT_LAUNCH_BOUNDS fpt_persistent_kernel(const __grid_constant__ KParams P) {
  extern __shared__ unsigned int smem_hist[];            // nbins + 2 counters when P.hist_of >= 0
  __shared__ DrainPool pool;
  const bool do_hist = P.hist_of >= 0;
  if (do_hist)
    for (int i = threadIdx.x; i < P.nbins + 2; i += blockDim.x) smem_hist[i] = 0u;
  if (threadIdx.x < kMaxWarpsPerBlock) pool.holes[threadIdx.x] = 0;
  if (threadIdx.x == 0) {
    pool.lock = 0;
    pool.n_parked = 0;
  }
  __syncthreads();
  const unsigned lane = threadIdx.x & 31u;
  const int warp_in_block = (int)(threadIdx.x >> 5);
  const int warps_in_block = (int)(blockDim.x >> 5);
  const unsigned lt_mask = (1u << lane) - 1u;
  constexpr int M = S::kMacro;
  const int n_macro = P.K / M;

  S st;
  st.init(P);
  bool active = false;                  // lane holds a live trajectory
  bool exhausted = false;               // warp-uniform: the global counter has run past n_traj
  unsigned long long idx = 0;           // index of the lane's trajectory within this call (id = first_id + idx)
  const unsigned long long lanes_total = (unsigned long long)gridDim.x * blockDim.x;
  unsigned long long next_static = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;   // static schedule only
  unsigned long long kbase = 0;         // steps completed by the lane's trajectory at the last poll
  uint32_t id_lo = 0, id_hi = 0;
  unsigned long long s_useful = 0, s_blocks = 0;
  unsigned s_esc = 0, s_cens = 0, s_nan = 0, s_atom = 0, s_mig = 0;
  // Software pipeline: zc holds the normals of the NEXT macro step to integrate; each loop iteration generates the
  // normals of the one after it (Philox + Box-Muller, independent of the state) alongside the dependent step chain.
  typename S::real zc[M];
#pragma unroll
  for (int s = 0; s < M; ++s) zc[s] = 0;

  for (;;) {
    // ---- S7 poll + S0 claim: idle lanes take new ids, one atomic per warp
    const unsigned want = __ballot_sync(0xffffffffu, !active);
    if (want) {
      if (!exhausted) {
        unsigned long long mine = ~0ull;
        if (P.schedule == kScheduleDynamic) {
          const int leader = __ffs(want) - 1;
          const unsigned cnt = __popc(want);
          unsigned long long base = 0;
          if ((int)lane == leader) {
            base = atomicAdd(&P.ws->next_id, (unsigned long long)cnt);
            ++s_atom;
          }
          base = __shfl_sync(0xffffffffu, base, leader);
          if (!active) mine = base + (unsigned long long)__popc(want & lt_mask);
          exhausted = (base + cnt >= P.n_traj);
        } else {
          // static split of the paper's Appendix A: thread j owns runs j, j + L, j + 2L, ... (L lanes)
          if (!active) {
            mine = next_static;
            next_static += lanes_total;
          }
          exhausted = __all_sync(0xffffffffu, next_static >= P.n_traj);
        }
        if (!active && mine < P.n_traj) {
          idx = mine;
          const unsigned long long id = P.first_id + mine;
          id_lo = (uint32_t)id;
          id_hi = (uint32_t)(id >> 32);
          kbase = 0;
          st.init(P);
          active = true;
          uint32_t o0, o1, o2, o3;                              // normals of block 0 of the new stream
          philox_block(P.keys, 0u, 0u, id_lo, id_hi, o0, o1, o2, o3);
          S::normals(o0, o1, o2, o3, zc);
        }
      }
      // ---- drain: lanes that could not be refilled adopt parked trajectories; a sparse warp parks its own and retires
      const unsigned idle = __ballot_sync(0xffffffffu, !active);
      if (idle && P.schedule != kScheduleDynamic) {         // static split: no hand-over, the warp lives as long as its slowest lane
        if (idle == 0xffffffffu && exhausted) break;
      } else if (idle) {                                    // implies exhausted
        if (lane == 0)
          while (atomicCAS(&pool.lock, 0, 1) != 0) __nanosleep(64);
        __syncwarp();
        __threadfence_block();
        int np = *(volatile int*)&pool.n_parked;
        int na = 32 - __popc(idle);
        const int take = min(32 - na, np);
        bool adopted = false;
        if (!active) {
          const int r = __popc(idle & lt_mask);
          if (r < take) {
            const ParkSlot sl = pool.slots[np - 1 - r];
            idx = sl.idx;
            kbase = sl.kbase;
            st.unpark(P, sl, kbase);
            active = true;
            adopted = true;
          }
        }
        np -= take;
        na += take;
        bool retire = (na == 0);                            // nothing of our own and (then necessarily) nothing parked
        if (!retire && na < 32) {
          int others = 0;
          for (int w = 0; w < warps_in_block; ++w)
            if (w != warp_in_block) others += *(volatile int*)&pool.holes[w];
          if (na <= others - np) {                          // the other warps' holes can take all of ours
            const unsigned live = __ballot_sync(0xffffffffu, active);
            if (active) {
              ParkSlot sl;
              st.park(sl);
              sl.kbase = kbase;
              sl.idx = idx;
              pool.slots[np + __popc(live & lt_mask)] = sl;
              active = false;
              adopted = false;
              ++s_mig;
            }
            np += na;
            retire = true;
          }
        }
        __threadfence_block();
        __syncwarp();
        if (lane == 0) {
          *(volatile int*)&pool.n_parked = np;
          *(volatile int*)&pool.holes[warp_in_block] = retire ? 0 : 32 - na;
          __threadfence_block();
          atomicExch(&pool.lock, 0);
        }
        __syncwarp();
        if (retire) break;
        if (adopted) {                                      // stream position of the adopted trajectory: block kbase / M
          const unsigned long long id = P.first_id + idx;
          id_lo = (uint32_t)id;
          id_hi = (uint32_t)(id >> 32);
          const unsigned long long b = kbase / (unsigned long long)M;
          uint32_t o0, o1, o2, o3;
          philox_block(P.keys, (uint32_t)b, (uint32_t)(b >> 32), id_lo, id_hi, o0, o1, o2, o3);
          S::normals(o0, o1, o2, o3, zc);
        }
      }
    }

    // ---- K steps (S1..S6).  Block index of macro step jj of this poll interval: kbase/M + jj.
    const unsigned long long b0 = kbase / (unsigned long long)M;
    int koff = 0;                       // step offset (1..K) of the first capture in this interval, 0 = none
    int cap_hi = 0;                     // high word of phi at the capture (distinguishes a crossing from a NaN)
    bool captured = false;
#pragma unroll(kUnroll)
    for (int jj = 0; jj < n_macro; ++jj) {
      const unsigned long long bn = b0 + (unsigned long long)(jj + 1);
      uint32_t o0, o1, o2, o3;
      philox_block(P.keys, (uint32_t)bn, (uint32_t)(bn >> 32), id_lo, id_hi, o0, o1, o2, o3);
      typename S::real zn[M];
      S::normals(o0, o1, o2, o3, zn);
#pragma unroll
      for (int s = 0; s < M; ++s) {
        st.step(P, zc[s]);
        const bool hit = st.crossed(P) && !captured;      // sticky per-step test
        if (hit) {
          koff = jj * M + s + 1;
          cap_hi = st.phi_hi();
        }
        captured = captured || hit;
      }
#pragma unroll
      for (int s = 0; s < M; ++s) zc[s] = zn[s];
    }
    ++s_blocks;

    // ---- classify (S6 / cap) and write results by trajectory id
    if (active) {
      const unsigned long long rem = P.n_cap - kbase;     // steps left before the cap, >= 1
      int status = -1;
      unsigned long long k_end = 0;
      if (captured && (unsigned long long)koff <= rem) {
        k_end = kbase + (unsigned long long)koff;
        status = st.is_nan_hi(cap_hi) ? kStatusNan : kStatusEscaped;
      } else if (rem <= (unsigned long long)P.K) {
        k_end = P.n_cap;
        status = kStatusCensored;
      }
      if (status >= 0) {
        const double kf = __ull2double_rn(k_end);          // exact: k_end < 2^53
        double fptv = __dmul_rn(kf, P.dt);
        double gam = __fma_rn(P.dgamma, kf, P.gamma0);
        if (status == kStatusCensored) fptv = -1.0;        // paper's sentinel
        if (status == kStatusNan) {
          fptv = __longlong_as_double(0x7ff8000000000000ll);
          gam = fptv;
        }
        P.out_fpt[idx] = fptv;
        if (P.out_gamma) P.out_gamma[idx] = gam;
        P.out_status[idx] = status;
        if (status == kStatusEscaped) {
          ++s_esc;
          if (do_hist) {
            const int slot = hist_slot(P.hist_of == 0 ? gam : fptv, P.hist_lo, P.hist_scale, P.nbins);
            if (slot >= 0) atomicAdd(&smem_hist[slot], 1u);
          }
        } else if (status == kStatusCensored) {
          ++s_cens;
        } else {
          ++s_nan;
        }
        s_useful += k_end;
        active = false;
      } else {
        kbase += (unsigned long long)P.K;
      }
    }
  }

  // ---- per-warp statistics, S8 merge
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) s_useful += __shfl_xor_sync(0xffffffffu, s_useful, off);
  const unsigned e = __reduce_add_sync(0xffffffffu, s_esc);
  const unsigned c = __reduce_add_sync(0xffffffffu, s_cens);
  const unsigned nn = __reduce_add_sync(0xffffffffu, s_nan);
  s_atom = __reduce_add_sync(0xffffffffu, s_atom);
  s_mig = __reduce_add_sync(0xffffffffu, s_mig);
  if (lane == 0) {
    atomicAdd(&P.ws->useful_steps, s_useful);
    atomicAdd(&P.ws->issued_lane_steps, s_blocks * (unsigned long long)P.K * 32ull);
    atomicAdd(&P.ws->n_escaped, (unsigned long long)e);
    atomicAdd(&P.ws->n_censored, (unsigned long long)c);
    atomicAdd(&P.ws->n_nan, (unsigned long long)nn);
    atomicAdd(&P.ws->refill_atomics, (unsigned long long)s_atom);
    if (s_mig) atomicAdd(&P.ws->migrations, (unsigned long long)s_mig);
  }
  if (do_hist) {
    __syncthreads();
    for (int i = threadIdx.x; i < P.nbins + 2; i += blockDim.x) {
      const unsigned cnt = smem_hist[i];
      if (cnt) atomicAdd(&P.out_counts[i], (unsigned long long)cnt);
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Test hook: one trajectory, one thread, every state recorded (same State code as the persistent kernel).
struct TraceArgs {
  unsigned long long id;
  long long trace_len;
  double* phi;
  double* v;
  int* status;
  unsigned long long* k_end;
};

template <class S>
__global__ void fpt_trace_kernel(const __grid_constant__ KParams P, const TraceArgs T) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  constexpr int M = S::kMacro;
  S st;
  st.init(P);
  if (T.trace_len > 0) {
    T.phi[0] = st.phi_as_double();
    if (T.v) T.v[0] = st.v_as_double();
  }
  int status = kStatusCensored;
  unsigned long long k_end = P.n_cap;
  if (st.crossed(P)) {
    status = st.is_nan_hi(st.phi_hi()) ? kStatusNan : kStatusEscaped;
    k_end = 0;
  } else {
    typename S::real z[M];
    for (unsigned long long k = 1; k <= P.n_cap; ++k) {
      const int s = (int)((k - 1) % (unsigned long long)M);
      if (s == 0) {
        const unsigned long long b = (k - 1) / (unsigned long long)M;
        uint32_t o0, o1, o2, o3;
        philox_block(P.keys, (uint32_t)b, (uint32_t)(b >> 32), (uint32_t)T.id, (uint32_t)(T.id >> 32), o0, o1, o2, o3);
        S::normals(o0, o1, o2, o3, z);
      }
      typename S::real zz = z[0];
#pragma unroll
      for (int i = 1; i < M; ++i) zz = (s == i) ? z[i] : zz;
      st.step(P, zz);
      if ((long long)k < T.trace_len) {
        T.phi[k] = st.phi_as_double();
        if (T.v) T.v[k] = st.v_as_double();
      }
      if (st.crossed(P)) {
        status = st.is_nan_hi(st.phi_hi()) ? kStatusNan : kStatusEscaped;
        k_end = k;
        break;
      }
    }
  }
  if (T.status) *T.status = status;
  if (T.k_end) *T.k_end = k_end;
}

}  // namespace fpt
