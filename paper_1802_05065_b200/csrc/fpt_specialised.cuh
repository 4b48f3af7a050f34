// fpt_specialised.cuh -- the warp-specialised integrator for launches that cannot fill the GPU (SURVEY.md 8(a) rows
// S0..S8, same arithmetic as fpt_integrator.cuh).
//
// A launch lasts at least as long as its longest trajectory ("the overall time is determined by the slowest
// thread"), and a trajectory advances at the latency of its own instruction stream.  Half of that stream does not depend
// on the state: Philox + Box-Muller.  When there are too few trajectories in flight to hide latencies
// behind other warps, the two halves run in DIFFERENT warps from the first step on:
//   * a CONSUMER warp holds 32 trajectories (phi, v, k in registers), reads one normal per step from shared memory and
//     only integrates (S3-S6), polls once per chunk of kChunk steps (S7) and refills finished lanes from the global
//     counter with one atomic per warp;
//   * its PRODUCER warps generate the normals of the consumer's lanes (S1-S2), chunk by chunk, one chunk ahead, into a
//     double buffer in shared memory; producer p of NP takes every NP-th Philox block of a chunk.
// A lane that takes a new trajectory at poll j publishes (id, first chunk = j + 1) in its mailbox slot BEFORE the
// consumer releases buffer j - 1; the producers read the mailbox when they start a chunk, so chunk j + 1 already carries
// the new stream.  The lane idles for the one chunk in between (64 steps; mean trajectory of config 2: 5690).
// Stream positions and arithmetic are those of the persistent kernel, so the outputs are the same bits.
#pragma once
#include "fpt_integrator.cuh"

namespace fpt {

constexpr int kSpecMaxConsumers = 4;
constexpr int kSpecMaxProducers = 3;
constexpr int kSpecMaxThreads = 384;

struct SpecChannel {                                  // one consumer and its producers
  unsigned long long cons_seq;                        // the consumer has polled and is about to consume chunk cons_seq (chunks below
                                                      // are consumed); ~0 before its first poll: only chunk 0 may be produced
  unsigned long long full_seq[kSpecMaxProducers];     // chunks completed by producer p
  int done;                                           // consumer has finished: producers leave
  int pad;
  unsigned long long mail_c0[32];                     // lane's current trajectory starts with chunk mail_c0 (~0: none yet)
  unsigned long long mail_id[32];                     // and has this trajectory id
};

template <class S>
__host__ __device__ constexpr size_t spec_channel_bytes() {
  return sizeof(SpecChannel) + 2 * (size_t)S::kChunk * 32 * sizeof(typename S::real);
}

template <class S>
__global__ void __launch_bounds__(kSpecMaxThreads, 1) fpt_specialised_kernel(const __grid_constant__ KParams P) {
  extern __shared__ __align__(16) unsigned char spec_smem[];
  typedef typename S::real real;
  constexpr int M = S::kMacro;
  constexpr int kChunk = S::kChunk;
  constexpr int kBlocksPerChunk = kChunk / M;
  const int NC = P.spec_consumers, NP = P.spec_producers;
  const unsigned lane = threadIdx.x & 31u;
  const int warp = (int)(threadIdx.x >> 5);
  const bool is_consumer = warp < NC;
  const int chan_id = is_consumer ? warp : (warp - NC) % NC;      // NC == 4: a producer shares its consumer's sub-partition
  const int prod_id = is_consumer ? -1 : (warp - NC) / NC;
  SpecChannel* ch = reinterpret_cast<SpecChannel*>(spec_smem + (size_t)chan_id * spec_channel_bytes<S>());
  real* zbuf = reinterpret_cast<real*>(reinterpret_cast<unsigned char*>(ch) + sizeof(SpecChannel));   // [2][kChunk][32]
  unsigned int* smem_hist = reinterpret_cast<unsigned int*>(spec_smem + (size_t)NC * spec_channel_bytes<S>());
  const bool do_hist = P.hist_of >= 0;
  if (do_hist)
    for (int i = threadIdx.x; i < P.nbins + 2; i += blockDim.x) smem_hist[i] = 0u;
  if (is_consumer) {
    ch->mail_c0[lane] = ~0ull;
    ch->mail_id[lane] = 0ull;
    if (lane == 0) {
      ch->cons_seq = ~0ull;
      ch->done = 0;
      for (int p = 0; p < kSpecMaxProducers; ++p) ch->full_seq[p] = 0ull;
    }
  }
  __syncthreads();

  unsigned long long s_useful = 0, s_chunks = 0, s_help = 0;
  unsigned s_esc = 0, s_cens = 0, s_nan = 0, s_atom = 0;

  if (is_consumer) {
    // ================================================================================================ consumer
    const unsigned lt_mask = (1u << lane) - 1u;
    S st;
    st.init(P);
    bool active = false;                // lane integrates a live trajectory
    bool waiting = false;               // lane has claimed a trajectory whose first chunk is the NEXT one
    bool exhausted = false;             // warp-uniform: the global counter has run past n_traj
    unsigned long long idx = 0, kbase = 0;
    unsigned long long cseq = 0;        // chunk about to be consumed
    for (;;) {
      // ---- S7 poll + S0 claim (before buffer cseq - 1 is released, so the producers see the mailbox in time)
      if (waiting) {                    // claimed one chunk ago: its stream starts with chunk cseq
        st.init(P);
        kbase = 0;
        active = true;
        waiting = false;
      }
      const unsigned want = __ballot_sync(0xffffffffu, !active);
      if (want) {
        if (!exhausted) {
          const int leader = __ffs(want) - 1;
          const unsigned cnt = __popc(want);
          unsigned long long base = 0;
          if ((int)lane == leader) {
            base = atomicAdd(&P.ws->next_id, (unsigned long long)cnt);
            ++s_atom;
          }
          base = __shfl_sync(0xffffffffu, base, leader);
          exhausted = (base + cnt >= P.n_traj);
          if (!active) {
            const unsigned long long mine = base + (unsigned long long)__popc(want & lt_mask);
            if (mine < P.n_traj) {
              idx = mine;
              waiting = true;
              ch->mail_id[lane] = P.first_id + mine;
              ch->mail_c0[lane] = cseq + 1ull;
            }
          }
        }
        if (exhausted && __ballot_sync(0xffffffffu, active || waiting) == 0u) break;
      }
      __threadfence_block();
      __syncwarp();
      if (lane == 0) *(volatile unsigned long long*)&ch->cons_seq = cseq;     // buffer (cseq + 1) & 1 may be refilled
      // ---- wait for chunk cseq
      for (;;) {
        const bool ok = (int)lane >= NP || *(volatile unsigned long long*)&ch->full_seq[lane] > cseq;
        if (__all_sync(0xffffffffu, ok)) break;
        __nanosleep(20);
      }
      __threadfence_block();
      // ---- kChunk steps (S3..S6), sticky per-step escape capture as in the persistent kernel
      int n_alive = 0;
      int cap_hi = 0;
      bool alive = true;
      const real* zb = zbuf + (size_t)(cseq & 1ull) * (kChunk * 32) + lane;
#pragma unroll 8
      for (int s = 0; s < kChunk; ++s) {
        st.step(P, zb[s * 32]);
        if (alive) cap_hi = st.phi_hi();
        alive = alive && !st.crossed(P);
        if (alive) ++n_alive;
      }
      ++cseq;
      ++s_chunks;
      // ---- classify (S6 / cap) and write results by trajectory id
      const unsigned long long rem = P.n_cap - kbase;
      const bool fin = active && (!alive || rem <= (unsigned long long)kChunk);
      if (__any_sync(0xffffffffu, fin)) {
        if (fin) {
          int status = -1;
          unsigned long long k_end = 0;
          const int koff = n_alive + 1;
          if (!alive && (unsigned long long)koff <= rem) {
            k_end = kbase + (unsigned long long)koff;
            status = st.is_nan_hi(cap_hi) ? kStatusNan : kStatusEscaped;
          } else if (rem <= (unsigned long long)kChunk) {
            k_end = P.n_cap;
            status = kStatusCensored;
          }
          if (status >= 0) {
            const double kf = __ull2double_rn(k_end);
            double fptv = __dmul_rn(kf, P.dt);
            double gam = __fma_rn(P.dgamma, kf, P.gamma0);
            if (status == kStatusCensored) fptv = -1.0;
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
          }
        }
      }
      if (active) kbase += (unsigned long long)kChunk;
    }
    if (lane == 0) {
      __threadfence_block();
      *(volatile int*)&ch->done = 1;                                           // releases the producers
    }
  } else if (prod_id < NP) {
    // ================================================================================================ producer
    for (unsigned long long j = 0;; ++j) {
      int stop = 0;
      if (lane == 0) {
        for (;;) {
          if (*(volatile int*)&ch->done) { stop = 1; break; }
          if (j < *(volatile unsigned long long*)&ch->cons_seq + 2ull) break;  // buffer j & 1 is free
          __nanosleep(20);
        }
      }
      stop = __shfl_sync(0xffffffffu, stop, 0);
      if (stop) break;
      __threadfence_block();
      const unsigned long long c0 = *(volatile unsigned long long*)&ch->mail_c0[lane];
      const unsigned long long id = *(volatile unsigned long long*)&ch->mail_id[lane];
      const bool live = c0 <= j;                                               // this lane integrates during chunk j
      if (__any_sync(0xffffffffu, live)) {
        const unsigned long long b0 = live ? (j - c0) * (unsigned long long)kBlocksPerChunk : 0ull;
        const uint32_t id_lo = (uint32_t)id, id_hi = (uint32_t)(id >> 32);
        real* zw = zbuf + (size_t)(j & 1ull) * (kChunk * 32) + lane;
#pragma unroll 2
        for (int m = prod_id; m < kBlocksPerChunk; m += NP) {
          const unsigned long long b = b0 + (unsigned long long)m;
          uint32_t o0, o1, o2, o3;
          philox_block(P.keys, (uint32_t)b, (uint32_t)(b >> 32), id_lo, id_hi, o0, o1, o2, o3);
          real zz[M];
          S::normals(o0, o1, o2, o3, zz);
#pragma unroll
          for (int q = 0; q < M; ++q) zw[(m * M + q) * 32] = zz[q];
          ++s_help;
        }
      }
      __threadfence_block();
      __syncwarp();
      if (lane == 0) *(volatile unsigned long long*)&ch->full_seq[prod_id] = j + 1ull;
    }
  }

  // ---- per-warp statistics, S8 merge
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) s_useful += __shfl_xor_sync(0xffffffffu, s_useful, off);
  const unsigned e = __reduce_add_sync(0xffffffffu, s_esc);
  const unsigned c = __reduce_add_sync(0xffffffffu, s_cens);
  const unsigned nn = __reduce_add_sync(0xffffffffu, s_nan);
  s_atom = __reduce_add_sync(0xffffffffu, s_atom);
  if (lane == 0) {
    if (is_consumer) {
      atomicAdd(&P.ws->useful_steps, s_useful);
      atomicAdd(&P.ws->issued_lane_steps, s_chunks * (unsigned long long)(kChunk * 32));
      atomicAdd(&P.ws->n_escaped, (unsigned long long)e);
      atomicAdd(&P.ws->n_censored, (unsigned long long)c);
      atomicAdd(&P.ws->n_nan, (unsigned long long)nn);
      atomicAdd(&P.ws->refill_atomics, (unsigned long long)s_atom);
    } else if (s_help) {
      atomicAdd(&P.ws->helper_lane_steps, s_help * (unsigned long long)(M * 32));
    }
  }
  if (do_hist) {
    __syncthreads();
    for (int i = threadIdx.x; i < P.nbins + 2; i += blockDim.x) {
      const unsigned cnt = smem_hist[i];
      if (cnt) atomicAdd(&P.out_counts[i], (unsigned long long)cnt);
    }
  }
}

}  // namespace fpt
