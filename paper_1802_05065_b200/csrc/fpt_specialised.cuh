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
// A lane that takes a trajectory at poll j (a new id, or one parked by another consumer) publishes (id, first chunk =
// j + 1, step index there) in its mailbox slot BEFORE the consumer releases buffer j - 1; the producers read the mailbox
// when they start a chunk, so chunk j + 1 already carries the new stream.  The lane idles for the one chunk in between
// (64 steps; mean trajectory of config 2: 5690).
// Measured on B200, Heun underdamped fp64, clk per step: a consumer alone on its SM sub-partition 184,
// against 247 for a warp that also generates its normals; a consumer that shares its sub-partition with a PRODUCER (which
// has the instruction-level parallelism to keep the FP64 pipe busy) 272-286; two consumers sharing one 248.  Hence the warp
// layouts: up to two consumers per SM each have a sub-partition to themselves, and consumers never share one with a producer.
// Once the ids are exhausted the consumers of a block compact their lanes exactly like the warps of the persistent
// kernel (park / adopt through shared memory), so a block is soon down to one consumer and one producer.
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
  unsigned long long mail_id[32];                     // has this trajectory id
  unsigned long long mail_k0[32];                     // and is at this step index when chunk mail_c0 begins (0 unless adopted)
};

struct SpecPool {                                     // drain-phase lane compaction between the consumers of a block
  int lock;
  int n_parked;
  int holes[kSpecMaxConsumers];
  ParkSlot slots[32 * kSpecMaxConsumers];
};

template <class S>
__host__ __device__ constexpr size_t spec_channel_bytes() {
  return sizeof(SpecChannel) + 2 * (size_t)S::kChunk * 32 * sizeof(typename S::real);
}
__host__ __device__ constexpr size_t spec_pool_bytes() { return (sizeof(SpecPool) + 15) / 16 * 16; }

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
  // Warp roles.  Warps are dealt to the four SM sub-partitions round robin (warp w -> sub-partition w mod 4), and a
  // consumer must not share its sub-partition with a producer.  Layout 1 (one producer per consumer): even warps are
  // consumers, odd warps producers, so consumers sit on sub-partitions 0 and 2, producers on 1 and 3.  Layout 0:
  // consumers first (warps 0..NC-1), then the producers (NC <= 2: the consumers have sub-partitions 0 and 1 to themselves
  // when NC * NP <= 2).
  bool is_consumer;
  int chan_id, prod_id;
  if (P.spec_layout == 1) {
    is_consumer = (warp & 1) == 0;
    chan_id = warp >> 1;
    prod_id = is_consumer ? -1 : 0;
  } else {
    is_consumer = warp < NC;
    chan_id = is_consumer ? warp : (warp - NC) % NC;
    prod_id = is_consumer ? -1 : (warp - NC) / NC;
  }
  SpecPool& pool = *reinterpret_cast<SpecPool*>(spec_smem);
  SpecChannel* ch = reinterpret_cast<SpecChannel*>(spec_smem + spec_pool_bytes() + (size_t)chan_id * spec_channel_bytes<S>());
  real* zbuf = reinterpret_cast<real*>(reinterpret_cast<unsigned char*>(ch) + sizeof(SpecChannel));   // [2][kChunk][32]
  unsigned int* smem_hist = reinterpret_cast<unsigned int*>(spec_smem + spec_pool_bytes() + (size_t)NC * spec_channel_bytes<S>());
  const bool do_hist = P.hist_of >= 0;
  if (do_hist)
    for (int i = threadIdx.x; i < P.nbins + 2; i += blockDim.x) smem_hist[i] = 0u;
  if (is_consumer) {
    ch->mail_c0[lane] = ~0ull;
    ch->mail_id[lane] = 0ull;
    ch->mail_k0[lane] = 0ull;
    if (lane == 0) {
      ch->cons_seq = ~0ull;
      ch->done = 0;
      for (int p = 0; p < kSpecMaxProducers; ++p) ch->full_seq[p] = 0ull;
    }
  }
  if (threadIdx.x == 0) {
    pool.lock = 0;
    pool.n_parked = 0;
    for (int i = 0; i < kSpecMaxConsumers; ++i) pool.holes[i] = 0;
  }
  __syncthreads();

  unsigned long long s_useful = 0, s_chunks = 0, s_help = 0;
  unsigned s_esc = 0, s_cens = 0, s_nan = 0, s_atom = 0, s_mig = 0;

  if (is_consumer) {
    // ================================================================================================ consumer
    const unsigned lt_mask = (1u << lane) - 1u;
    S st, st_next;                      // st_next: state of a trajectory taken at this poll, started at the next one
    st.init(P);
    st_next.init(P);
    bool active = false;                // lane integrates a live trajectory
    bool waiting = false;               // lane has taken a trajectory whose first chunk is the NEXT one
    bool exhausted = false;             // warp-uniform: the global counter has run past n_traj
    unsigned long long idx = 0, kbase = 0, kbase_next = 0;
    unsigned long long cseq = 0;        // chunk about to be consumed
    unsigned last_idle = 0;             // idle mask at our last visit of the drain pool
    for (;;) {
      // ---- S7 poll + S0 claim (before buffer cseq - 1 is released, so the producers see the mailbox in time)
      if (waiting) {                    // taken one chunk ago: its stream continues with chunk cseq
        st = st_next;
        kbase = kbase_next;
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
              st_next.init(P);
              kbase_next = 0;
              ch->mail_id[lane] = P.first_id + mine;
              ch->mail_k0[lane] = 0ull;
              ch->mail_c0[lane] = cseq + 1ull;
            }
          }
        }
        // ---- drain: idle lanes adopt parked trajectories; a sparse consumer parks its own and retires (invariant under
        // the lock: n_parked <= sum of holes[] over the live consumers that have seen exhaustion)
        const unsigned idle = __ballot_sync(0xffffffffu, !active && !waiting);
        // the lock is only worth taking when something can happen: our holes changed (or we are empty), something is
        // parked, or the other consumers' holes might now take all of our lanes (lock-free reads: hints, re-read below)
        bool trade = false;
        if (idle && exhausted) {
          int others = 0;
          for (int c = 0; c < NC; ++c)
            if (c != chan_id) others += *(volatile int*)&pool.holes[c];
          const int np_hint = *(volatile int*)&pool.n_parked;
          trade = idle != last_idle || np_hint > 0 || 32 - __popc(idle) <= others - np_hint;
          trade = __shfl_sync(0xffffffffu, trade ? 1 : 0, 0) != 0;
        }
        if (trade) {
          last_idle = idle;
          if (lane == 0)
            while (atomicCAS(&pool.lock, 0, 1) != 0) __nanosleep(64);
          __syncwarp();
          __threadfence_block();
          int np = *(volatile int*)&pool.n_parked;
          int na = 32 - __popc(idle);
          const int take = min(32 - na, np);
          if (!active && !waiting) {
            const int r = __popc(idle & lt_mask);
            if (r < take) {
              const ParkSlot sl = pool.slots[np - 1 - r];
              idx = sl.idx;
              kbase_next = sl.kbase;
              st_next.unpark(P, sl, sl.kbase);
              waiting = true;
              ch->mail_id[lane] = P.first_id + idx;
              ch->mail_k0[lane] = sl.kbase;
              ch->mail_c0[lane] = cseq + 1ull;
            }
          }
          np -= take;
          na += take;
          bool retire = (na == 0);                            // nothing of our own and (then necessarily) nothing parked
          if (!retire && na < 32) {
            int others = 0;
            for (int c = 0; c < NC; ++c)
              if (c != chan_id) others += *(volatile int*)&pool.holes[c];
            if (na <= others - np) {                          // the other consumers' holes can take all of ours
              const unsigned busy = __ballot_sync(0xffffffffu, active || waiting);
              if (active || waiting) {
                ParkSlot sl;
                if (active) {
                  st.park(sl);
                  sl.kbase = kbase;
                } else {
                  st_next.park(sl);
                  sl.kbase = kbase_next;
                }
                sl.idx = idx;
                pool.slots[np + __popc(busy & lt_mask)] = sl;
                active = false;
                waiting = false;
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
            *(volatile int*)&pool.holes[chan_id] = retire ? 0 : 32 - na;
            __threadfence_block();
            atomicExch(&pool.lock, 0);
          }
          __syncwarp();
          if (retire) break;
        }
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
      __syncwarp();                                         // lanes >= NP did not read a counter themselves: order them behind the lanes that did
      __threadfence_block();
      // ---- kChunk steps (S3..S6), sticky per-step escape capture as in the persistent kernel
      EscapeCapture cap;
      cap.reset();
      const real* zb = zbuf + (size_t)(cseq & 1ull) * (kChunk * 32) + lane;
#pragma unroll 8
      for (int s = 0; s < kChunk; ++s) {
        st.template step<true>(P, zb[s * 32]);
        cap.observe(st, P);
      }
      ++cseq;
      ++s_chunks;
      // ---- classify (S6 / cap) and write results by trajectory id
      const unsigned long long rem = P.n_cap - kbase;
      const bool fin = active && (!cap.alive || rem <= (unsigned long long)kChunk);
      if (__any_sync(0xffffffffu, fin)) {
        if (fin) {
          int status = kStatusCensored;
          unsigned long long k_end = P.n_cap;
          const int koff = cap.k_fail();                       // step offset (1..kChunk) of the first crossing in this chunk
          if (!cap.alive && (unsigned long long)koff <= rem) {
            k_end = kbase + (unsigned long long)koff;
            status = st.is_nan_hi(cap.cap_hi) ? kStatusNan : kStatusEscaped;
          }
          const double kf = __ull2double_rn(k_end);           // exact: k_end < 2^53
          double fptv = __dmul_rn(kf, P.dt);
          double gam = __fma_rn(P.dgamma, kf, P.gamma0);
          if (status == kStatusCensored) fptv = -1.0;         // paper's sentinel
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
      if (active) kbase += (unsigned long long)kChunk;
    }
    if (lane == 0) {
      __threadfence_block();
      *(volatile int*)&ch->done = 1;                                           // releases the producers
    }
  } else if (chan_id < NC && prod_id < NP) {
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
      __syncwarp();                                         // only lane 0 observed cons_seq: order the warp's mailbox reads behind it
      __threadfence_block();
      const unsigned long long c0 = *(volatile unsigned long long*)&ch->mail_c0[lane];
      const unsigned long long id = *(volatile unsigned long long*)&ch->mail_id[lane];
      const unsigned long long k0 = *(volatile unsigned long long*)&ch->mail_k0[lane];
      const bool live = c0 <= j;                                               // this lane integrates during chunk j
      if (__any_sync(0xffffffffu, live)) {
        const unsigned long long b0 = live ? k0 / (unsigned long long)M + (j - c0) * (unsigned long long)kBlocksPerChunk : 0ull;
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
  s_mig = __reduce_add_sync(0xffffffffu, s_mig);
  if (lane == 0) {
    if (is_consumer) {
      atomicAdd(&P.ws->useful_steps, s_useful);
      atomicAdd(&P.ws->issued_lane_steps, s_chunks * (unsigned long long)(kChunk * 32));
      atomicAdd(&P.ws->n_escaped, (unsigned long long)e);
      atomicAdd(&P.ws->n_censored, (unsigned long long)c);
      atomicAdd(&P.ws->n_nan, (unsigned long long)nn);
      atomicAdd(&P.ws->refill_atomics, (unsigned long long)s_atom);
      if (s_mig) atomicAdd(&P.ws->migrations, (unsigned long long)s_mig);
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
