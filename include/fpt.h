/* fpt.h -- C ABI of libfpt_b200: first-passage-time Monte Carlo of noisy washboard / RCSJ Langevin
 * trajectories on one NVIDIA B200 (sm_100a).
 *
 * PAPER.md = /root/reference/PAPER.md (arXiv:1802.05065, "Stochastic first passage time accelerated with CUDA").
 * The operations exported here are the paper's two kernels and its output arrays, re-designed for B200:
 *   - Alg. 1 ESCAPETIME: integrate Eq. (9) step by step, "checking at each
 *     time step if a threshold crossing ... has occurred", store the escape time k*h,
 *     or -1 when the step cap klim is reached;
 *   - Alg. 3 SWITCHINGCURRENT: same loop with the bias ramp gamma_k = gamma0 + dgamma*k
 *     (PAPER.md:295), store the bias at the crossing;
 *   - the switching-current histogram;
 *   - "assigns a new job to the processor as soon as it has terminated its task": done inside
 *     the kernel by a warp-aggregated claim on a global trajectory counter.
 * The exact arithmetic (Philox4x32-10 keying, uniforms, Box-Muller, sin/log/sincos algorithms, the four recurrences,
 * cap and sentinel rules) is DESIGN.md section 4 ("MATH SPEC"); readings of silent passages are DESIGN.md section 3.
 *
 * Conventions
 *   - Every pointer named out_*, values, status, counts is DEVICE memory owned by the caller unless the function name
 *     ends in _host.  `p` is HOST memory, read during the call only.  The library keeps no pointer after returning.
 *   - Calls enqueue work on `cuda_stream` (a cudaStream_t passed as void*; NULL = the legacy default stream) of the
 *     CURRENT device and return without synchronising; outputs are valid once the stream has been synchronised.
 *     (_host and fpt_last_stats synchronise before returning.)
 *   - Return value: FPT_OK, or a negative code.  On FPT_E_INVALID nothing has been enqueued or written.
 *     No exceptions, no errno, no printing.  fpt_strerror() gives a static string (for FPT_E_CUDA: the CUDA error
 *     string of the most recent failure on the calling thread).
 *   - Determinism: per-trajectory outputs are a pure function of (params, seed, trajectory id); they do not depend on
 *     launch geometry, on check_every, on any field of fpt_launch_opts (scheduler, tail helper, specialised kernel), on
 *     the GPU, or on which lane integrated which trajectory.
 *   - No state outside a call: the library owns a per-device memory pool and stream pool (caches), nothing a result or a
 *     later call depends on.  Test hooks and the pipe-peak microbenchmarks live in fpt_dbg.h.
 *   - There is no CPU fallback: without a CUDA device every compute entry point returns FPT_E_CUDA.
 */
#ifndef FPT_B200_H_
#define FPT_B200_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FPT_OK          0
#define FPT_E_INVALID (-1)   /* bad argument (see each function)                  */
#define FPT_E_CUDA    (-2)   /* CUDA runtime failure (no device, alloc, launch)   */
#define FPT_E_TOO_LARGE (-3) /* a size beyond an entry point's fixed maximum (fpt_simulate_noalloc); nothing enqueued */

#define FPT_MODEL_OVERDAMPED  0
#define FPT_MODEL_UNDERDAMPED 1
#define FPT_SCHEME_EM    0
#define FPT_SCHEME_HEUN  1
#define FPT_SCHEME_PAPER 2   /* the paper's kernels AS PRINTED (Alg. 1 lines 11-12, Alg. 3 lines 13-16):
                                Euler with the bias gamma_k = gamma0 + dgamma*k taken BEFORE step k (schemes 0, 1: gamma_{k-1}) and
                                the strict crossing test phi_k > threshold (schemes 0, 1: >=).  The paper's threshold pi - phi0
                                (Alg. 1 line 5) is the caller's `threshold`.  Bit-exact against the oracle like schemes 0 and 1. */
#define FPT_PREC_FP64 0
#define FPT_PREC_FP32 1
#define FPT_PREC_FP32_FAST 2 /* fp32 state, and the drift sine taken by the hardware (sin.approx / MUFU.SIN) as in the paper's single
                                precision kernels.  Only with FPT_SCHEME_PAPER and amp != 0.  The hardware sine has
                                no CPU twin: results are NOT bit-comparable with the oracle, only statistically (tests: two-sample KS
                                against the fp32 oracle); everything else is the FPT_PREC_FP32 arithmetic. */

#define FPT_STATUS_ESCAPED  0
#define FPT_STATUS_CENSORED 1
#define FPT_STATUS_NAN      2

/* One simulation's parameters (paper: kernel arguments (V0, beta, gamma, D, h) / (dgamma, V0, beta, D, h),
 * PAPER.md:137-142, 266-271).  4 x int32, 9 x double, 1 x uint64: 96 bytes, no padding. */
typedef struct fpt_params {
  int32_t  model;        /* 0 overdamped : dphi = (gamma(t) - amp*sin phi) dt + sqrt(2*temperature) dW
                            1 underdamped: phi'' + alpha*phi' + amp*sin phi = gamma(t) + sqrt(2*alpha*temperature) xi (Eq. 9) */
  int32_t  scheme;       /* 0 Euler-Maruyama (paper's Euler, Alg. 1 lines 11-12), 1 stochastic Heun, 2 FPT_SCHEME_PAPER */
  int32_t  precision;    /* 0 fp64 state; 1 fp32 state + Kahan-compensated time (outputs stay fp64 functions of k_esc);
                            2 FPT_PREC_FP32_FAST */
  int32_t  check_every;  /* K >= 1: poll/refill interval in steps.  NEVER changes results (the crossing test is per step,
                            PAPER.md:190).  Rounded up to a multiple of the steps per Philox block (2 fp64, 4 fp32).
                            0 = library default (64; 128 for long caps; 512 for ramped trajectories of 2^22 steps or more). */
  double   alpha;        /* damping (paper beta); ignored for model 0 */
  double   temperature;  /* T (paper theta; D = beta*theta).  model 0: the diffusion constant */
  double   amp;          /* amplitude of sin phi; 0 => drifted Brownian motion with mu = gamma0 */
  double   gamma0, nu;   /* bias ramp gamma(t) = gamma0 + nu*t, used as gamma_k = fma(nu*dt, k, gamma0) */
  double   phi0, v0;     /* initial state (paper: arcsin(gamma), 0) */
  double   threshold;    /* escape when phi >= threshold (> with FPT_SCHEME_PAPER; paper: pi - phi0) */
  double   dt;           /* step h */
  uint64_t first_id;     /* trajectory id of element 0 of the outputs (sharding); the Philox stream is keyed by (seed, id) */
} fpt_params;

/* Counters and launch geometry of ONE fpt_simulate* call, written by the call's own kernels (stream ordered) into the
 * caller's device block (fpt_simulate_ex: d_stats) -- nothing is shared between calls. */
typedef struct fpt_stats {
  uint64_t n_traj;             /* trajectories processed                                                  */
  uint64_t n_escaped, n_censored, n_nan;
  uint64_t useful_steps;       /* sum over trajectories of k_end (k_esc, or n_cap when censored)          */
  uint64_t issued_lane_steps;  /* 32 * (steps executed by every warp): lane efficiency = useful / issued   */
  uint64_t refill_atomics;     /* atomics issued on the global trajectory counter                         */
  uint64_t n_cap;              /* step cap used = nearbyint(t_max/dt)                                     */
  int32_t  grid, block;        /* launch geometry used                                                    */
  int32_t  check_every;        /* effective K                                                             */
  int32_t  kernel;             /* FPT_KERNEL_FILL | _PERSISTENT | _SPECIALISED: which kernel integrated    */
  uint64_t migrations;         /* trajectories parked by a sparse warp and adopted by another (drain-phase compaction) */
  uint64_t helper_lane_steps;  /* 32 * (steps whose normals a tail-helper or producer warp generated for another warp);
                                  NOT part of issued_lane_steps                                            */
  uint64_t time_slices;        /* time slicing: quanta after which a trajectory was set aside for a waiting one           */
} fpt_stats;

#define FPT_KERNEL_FILL        0   /* every trajectory decided at k = 0 (phi0 >= threshold) or by n_cap == 0: no integration */
#define FPT_KERNEL_PERSISTENT  1   /* every warp generates its own normals and integrates (filled GPU)                         */
#define FPT_KERNEL_SPECIALISED 2   /* consumer warps integrate, producer warps generate their normals (under-filled GPU)       */

/* Launch options of ONE call (fpt_simulate_ex).  Results never depend on any of them; only the time does.  A zeroed
 * struct (or a NULL pointer) means the library's defaults. */
#define FPT_SCHEDULE_DYNAMIC 0
#define FPT_SCHEDULE_STATIC  1
typedef struct fpt_launch_opts {
  int32_t block;          /* persistent kernel: threads per block, a multiple of 32 in 32..256; 0 = default           */
  int32_t blocks_per_sm;  /* persistent kernel: resident blocks per SM, 0 = default (occupancy / workload heuristic)   */
  int32_t max_blocks;     /* cap on the grid, 0 = none                                                                 */
  int32_t schedule;       /* FPT_SCHEDULE_DYNAMIC (default): a finished lane takes the next id from a global counter at
                             once and sparse warps hand their trajectories over in the drain phase;
                             FPT_SCHEDULE_STATIC: the static split analysed in the paper's Appendix A:
                             lane j of L owns runs j, j+L, j+2L, ...; nothing is handed over, a warp lives as long as its
                             slowest lane (with one run per lane: the paper's own kernel).  It exists to
                             measure what the dynamic scheduler buys (fpt_stats lane efficiency against Eq. (A.5)).       */
  int32_t tail_helper;    /* 0 = default (on), 1 = on, -1 = off.  Persistent kernel: when a block is down to one live warp
                             and nothing is parked, the block's retired warps generate that warp's normals (Philox +
                             Box-Muller) one chunk ahead into shared memory and the survivor only integrates.  Engages only
                             in blocks of >= 3 warps, with a poll interval that is a multiple of 64 steps (fp64) / 32 (fp32),
                             and for drifts with a sine (amp != 0).                                                      */
  int32_t specialise;     /* 0 = automatic (the specialised kernel when the job cannot fill the GPU: fewer than two
                             trajectories-in-flight warps per SM sub-partition), 1 = always, -1 = never.  Needs amp != 0 and
                             the dynamic schedule; otherwise the persistent kernel runs.                                  */
  int32_t consumers;      /* specialised kernel: consumer warps per block, 1..4 (0 = default)                           */
  int32_t producers;      /* specialised kernel: producer warps per consumer, 1..3 (0 = default)                        */
  int32_t time_slice;     /* persistent kernel, dynamic schedule, RAMPED bias (nu != 0: trajectories about equally long), more
                             trajectories than resident lanes: 0 = automatic (jobs of one to three ragged "waves", and fp32
                             jobs of 3 to 3.8 blocks of 128 per SM, which then run 3 blocks per SM), 1 = always, -1 = never.
                             Block b then owns the trajectories b, b + grid, ...; a lane sets its trajectory aside in device
                             memory (32 B per trajectory + 8 B per ring entry, from the call's stream-ordered pool) after a
                             quantum of >= 2048 steps while others of its block's are waiting and takes the one that has
                             waited longest (round robin), so that all trajectories advance at the same rate and no ragged
                             last wave idles the GPU.  Results are the same bits either way.  Ignored for a constant bias
                             (exponentially distributed lengths: the refill balances those).                          */
  int32_t reserved;       /* must be 0 */
} fpt_launch_opts;

/* Fused histogram request of fpt_simulate_ex (as fpt_simulate_hist). */
typedef struct fpt_hist {
  int32_t   of;           /* 0 = bias at escape, 1 = escape time */
  int32_t   nbins;        /* 1..8192 */
  double    lo, hi;
  uint64_t* out_counts;   /* device, nbins + 2, ACCUMULATED into */
} fpt_hist;

/* Integrate trajectories id = first_id .. first_id+n_traj-1 until first passage or the cap n_cap = nearbyint(t_max/dt).
 *   out_fpt[i]     (double, required) k_esc*dt; -1.0 if censored; NaN if status 2
 *   out_gamma_at_escape[i] (double, may be NULL) fma(nu*dt, (double)k_end, gamma0), k_end = k_esc or n_cap; NaN if status 2
 *   out_status[i]  (int32, required) 0 escaped, 1 censored, 2 phi became NaN before any crossing
 * Each array has n_traj elements, device memory.  n_traj == 0 is a successful no-op.
 * FPT_E_INVALID: NULL p / out_fpt / out_status, n_traj < 0, unknown enum, check_every < 0, a non-finite field,
 *   dt <= 0, t_max <= 0, t_max/dt >= 2^53, temperature < 0, alpha < 0 (model 1). */
int fpt_simulate(const fpt_params* p, int64_t n_traj, uint64_t seed, double t_max,
                 double* out_fpt, double* out_gamma_at_escape, int32_t* out_status, void* cuda_stream);

/* As fpt_simulate, and additionally bins the bias at escape of every ESCAPED trajectory (status 0) into
 * out_counts[nbins+2] = [under, bin 0 .. bin nbins-1, over] (device, uint64, ACCUMULATED into: the caller zeroes), through
 * a shared-memory histogram merged once per block.  Bin rule as fpt_histogram.  hist_of: 0 = gamma at
 * escape, 1 = escape time.  Additional FPT_E_INVALID: nbins < 1 or > 8192, hi <= lo, non-finite lo/hi, NULL out_counts. */
int fpt_simulate_hist(const fpt_params* p, int64_t n_traj, uint64_t seed, double t_max,
                      double* out_fpt, double* out_gamma_at_escape, int32_t* out_status,
                      int32_t hist_of, double lo, double hi, int32_t nbins, uint64_t* out_counts, void* cuda_stream);

/* The general entry point: fpt_simulate / fpt_simulate_hist with per-call launch options and per-call statistics, and
 * no state outside the call.  hist: NULL = no histogram.  opts: NULL = defaults.  d_stats (DEVICE memory, may be NULL):
 * receives this call's fpt_stats, written stream-ordered after the integration (valid once cuda_stream has been
 * synchronised).  Calls from any number of host threads on any number of streams are independent.
 * Additional FPT_E_INVALID: a bad field of opts (block not a multiple of 32 in 32..256, negative counts, unknown schedule,
 * consumers > 4, producers > 3, reserved != 0) or of hist (as fpt_simulate_hist). */
int fpt_simulate_ex(const fpt_params* p, int64_t n_traj, uint64_t seed, double t_max,
                    double* out_fpt, double* out_gamma_at_escape, int32_t* out_status,
                    const fpt_hist* hist, const fpt_launch_opts* opts, fpt_stats* d_stats, void* cuda_stream);

/* fpt_simulate for callers that must not allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): same arguments, same results bit for bit (Alg. 1 / Alg. 3; outputs are
 * a function of (params, seed, id) only), but this entry point calls no cudaMalloc / cudaMallocAsync / cudaFree or any other
 * allocating routine, on the first call or later.  It always runs the persistent kernel, and all the scratch memory that
 * kernel needs -- the global id counter and statistics block, and the parking slots and waiting rings of time slicing
 * (fpt_launch_opts.time_slice; used here for ramped jobs with more trajectories than resident lanes) -- lives in ONE
 * file-scope device array of the library, 5.3 MB, which every GPU that loads the library holds until the process exits.
 *   - Limit: n_traj <= FPT_NOALLOC_MAX_TRAJ, else FPT_E_TOO_LARGE (nothing is enqueued or written).  Otherwise argument
 *     checks and FPT_E_INVALID as fpt_simulate.  No fused histogram, no launch options.
 *   - d_stats: NULL, or a caller-owned DEVICE fpt_stats block written at the end of the call (as fpt_simulate_ex).
 *     fpt_last_stats does not see these calls.
 *   - The array is shared by every call and keeps the last call's contents; each call clears, on cuda_stream, what must start
 *     at zero.  Calls that may OVERLAP ON THE GPU (different streams, several host threads) race on it and give wrong
 *     results: issue them on one stream, or order them with events.  One array per device: calls on different GPUs are
 *     independent.
 *   - The first launch of a kernel in a process loads its code (CUDA lazy loading, done by the driver): make one warm-up
 *     call before capturing a graph.  Asynchronous, stream-ordered like fpt_simulate. */
#define FPT_NOALLOC_MAX_TRAJ 131072
int fpt_simulate_noalloc(const fpt_params* p, int64_t n_traj, uint64_t seed, double t_max,
                         double* out_fpt, double* out_gamma_at_escape, int32_t* out_status,
                         fpt_stats* d_stats, void* cuda_stream);

/* Histogram of values[i] over the entries with status[i] == 0 (status may be NULL: all entries):
 *   b = floor((x - lo) * (nbins/(hi-lo))) in fp64, the scale computed once; b < 0 -> under, b >= nbins -> over (x == hi is
 *   "over"), NaN values are not counted.  out_counts[nbins+2] is accumulated into.  Counts are integers, so the result is
 *   independent of the order of accumulation.  FPT_E_INVALID: n < 0, nbins < 1, hi <= lo, NULL values/out_counts. */
int fpt_histogram(const double* values, const int32_t* status, int64_t n,
                  double lo, double hi, int32_t nbins, uint64_t* out_counts, void* cuda_stream);

/* End-to-end convenience: as fpt_simulate but every out_* pointer is HOST memory (pinned or pageable); the call allocates
 * device buffers, runs, copies the results back and synchronises.  h_counts (may be NULL) as in fpt_simulate_hist with
 * hist_of/lo/hi/nbins, host memory, accumulated into. */
int fpt_simulate_host(const fpt_params* p, int64_t n_traj, uint64_t seed, double t_max,
                      double* h_fpt, double* h_gamma_at_escape, int32_t* h_status,
                      int32_t hist_of, double lo, double hi, int32_t nbins, uint64_t* h_counts);

/* Parameter-sweep batch: n_sets independent jobs of n_per_set trajectories each, e.g. the temperature sweep behind the
 * Arrhenius / Kramers plot of the mean escape time (Eqs. (12)-(14), Fig. 10) or a sweep of the bias.
 * Set s uses sets[s] (any field may differ between sets, including model and scheme), the cap t_max[s] and the ids
 * sets[s].first_id + 0 .. n_per_set-1 of the Philox stream `seed`: give the sets disjoint id ranges for independent
 * samples, equal ranges for common random numbers.  Outputs of set s occupy elements [s*n_per_set, (s+1)*n_per_set) of
 * the out_* arrays (device, n_sets*n_per_set elements; out_gamma_at_escape may be NULL).  The sets run CONCURRENTLY as
 * separate persistent launches on an internal pool of streams (a small set cannot fill 148 SMs, and each launch lasts as
 * long as its longest trajectory), forked from and joined back into cuda_stream, so to the caller this is one
 * asynchronous call like fpt_simulate.  Each result is bit-identical to a separate fpt_simulate of that set.
 * sets and t_max are host arrays read during the call.  FPT_E_INVALID as fpt_simulate for any set (nothing is
 * launched then), or NULL sets / t_max, n_sets < 0.  fpt_last_stats afterwards describes the last set. */
int fpt_simulate_sweep(const fpt_params* sets, int32_t n_sets, int64_t n_per_set, uint64_t seed, const double* t_max,
                       double* out_fpt, double* out_gamma_at_escape, int32_t* out_status, void* cuda_stream);

/* DEPRECATED conveniences, kept for one release: defaults for the calls that take no fpt_launch_opts (fpt_simulate,
 * fpt_simulate_hist, fpt_simulate_host, fpt_simulate_sweep) made afterwards BY THE CALLING THREAD (thread-local; no
 * process-wide state).  New code passes fpt_launch_opts to fpt_simulate_ex.  FPT_E_INVALID on a bad value. */
int fpt_set_launch(int32_t block, int32_t blocks_per_sm, int32_t max_blocks);   /* fields of the same names          */
int fpt_set_schedule(int32_t schedule);                                         /* FPT_SCHEDULE_*                    */
int fpt_set_tail_helper(int32_t on);                                            /* 1 on (default), 0 off             */
int fpt_set_specialise(int32_t specialise, int32_t consumers, int32_t producers);

/* DEPRECATED: synchronises the current device and returns the fpt_stats of the most recent fpt_simulate* call the
 * CALLING THREAD made on it (a zeroed struct if it made none).  Concurrent callers pass their own d_stats to
 * fpt_simulate_ex instead. */
int fpt_last_stats(fpt_stats* out);

const char* fpt_strerror(int code);
int fpt_version(void);   /* 10000*major + 100*minor + patch */

#ifdef __cplusplus
}
#endif
#endif /* FPT_B200_H_ */
