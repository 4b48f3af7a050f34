// fpt_api.cu -- the C ABI of include/fpt.h and include/fpt_dbg.h: argument validation, the host-side derived constants
// (DESIGN.md 4.8), launch geometry and kernel choice, the standalone histogram kernel, the roofline microbenchmarks and the
// test hooks.  Nothing a result or a later call depends on is kept between calls: launch options and statistics travel
// with the call (fpt_launch_opts, d_stats); the library owns only caches (a memory pool and a stream pool per device).
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <vector>

#include "../../include/fpt.h"
#include "../../include/fpt_dbg.h"
#include "fpt_inst.cuh"
#include "fpt_integrator.cuh"

namespace {

using namespace fpt;

thread_local cudaError_t g_last_cuda = cudaSuccess;

#define FPT_CUDA(call)                         \
  do {                                         \
    cudaError_t err__ = (call);                \
    if (err__ != cudaSuccess) {                \
      g_last_cuda = err__;                     \
      (void)cudaGetLastError();                \
      return FPT_E_CUDA;                       \
    }                                          \
  } while (0)

constexpr int kMaxDevices = 64;
// default poll interval in steps: measured on B200, a poll costs about as much as 1.3 steps in fp64 and 3 in fp32 (the
// software pipeline of the step loop drains and refills around it), and a finished lane idles K/2 steps on average, so
// the best K grows with the square root of the trajectory length.  The cap is all the host knows about that length:
// fp64 64, and 128 from caps of 2^21 steps (configs 3 and 5: +0.5 %, +1 %; config 2, cap 10^6 and mean 5700: -0.4 %);
// fp32 64, and 128 from caps of 2^16 steps (config 4 twin: +3.8 % over 32; 256 is no better)
constexpr int kDefaultK = 64, kDefaultKLong = 128;
constexpr unsigned long long kLongCap64 = 1ull << 21, kLongCap32 = 1ull << 16;
// ramped bias: a trajectory switches before the tilt reaches the critical one, after about (amp - gamma0) / (nu dt) steps,
// so its length is known in advance to within the switching width.  From 2^22 steps a poll every 512 costs a finished lane
// 256 idle steps in millions and saves three quarters of the polls (measured on B200 against 128: config 4's geometry
// +1.2 % issued-lane throughput, config 3 as stated +0.2 %; 2048: +0.5 % on config 3, no better in fp32)
constexpr int kDefaultKRampLong = 512;
constexpr double kRampLongSteps = 4194304.0;
// specialised kernel (fpt_specialised.cuh): hand-over chunk = its poll interval; limits of fpt_launch_opts
constexpr int kSpecChunk64 = 64, kSpecChunk32 = 32;
constexpr int kSpecMaxConsumersHost = 4, kSpecMaxProducersHost = 3;

// Defaults of the calls that take no fpt_launch_opts: per THREAD (the deprecated fpt_set_* shims write them).
thread_local fpt_launch_opts t_opts = {};
thread_local unsigned long long t_dbg_seq0 = 0;
thread_local unsigned long long t_dbg_slice_q = 0;

constexpr int kSweepStreams = 8;
constexpr int kLastSlots = 256;   // ring of "last call" statistics blocks per device (fpt_last_stats shim)

struct DeviceCtx {          // per device: caches only
  std::mutex mu;                 // serialises fpt_simulate_sweep's use of the stream pool
  cudaStream_t pool[kSweepStreams] = {};
  bool pool_ready = false;
  cudaMemPool_t mem = nullptr;   // the library's own stream-ordered pool: freed blocks stay cached across synchronisations
  fpt_stats* d_last = nullptr;   // kLastSlots blocks; a call writes its statistics into slot (ticket % kLastSlots)
  unsigned long long* d_ticket = nullptr;   // ticket of the call that owns each slot
  std::atomic<unsigned long long> next_ticket{1};
  int sm_count = 0;
  std::atomic<bool> ready{false};
};
DeviceCtx g_ctx[kMaxDevices];
std::mutex g_init_mu;

struct ThreadLast {         // ticket of the calling thread's most recent call, per device
  unsigned long long ticket[kMaxDevices] = {};
};
thread_local ThreadLast t_last;

int device_ctx(DeviceCtx** out, int* dev_out = nullptr) {
  int dev = 0;
  FPT_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return FPT_E_CUDA;
  DeviceCtx& c = g_ctx[dev];
  if (!c.ready.load(std::memory_order_acquire)) {
    std::lock_guard<std::mutex> lk(g_init_mu);
    if (!c.ready.load(std::memory_order_relaxed)) {
      FPT_CUDA(cudaMalloc(&c.d_last, sizeof(fpt_stats) * kLastSlots));
      FPT_CUDA(cudaMemset(c.d_last, 0, sizeof(fpt_stats) * kLastSlots));
      FPT_CUDA(cudaMalloc(&c.d_ticket, sizeof(unsigned long long) * kLastSlots));
      FPT_CUDA(cudaMemset(c.d_ticket, 0, sizeof(unsigned long long) * kLastSlots));
      FPT_CUDA(cudaDeviceGetAttribute(&c.sm_count, cudaDevAttrMultiProcessorCount, dev));
      // per-call workspaces come from a private memory pool that never trims (release threshold = max): with the device's
      // default pool every stream synchronisation hands the memory back to the driver and the next call pays a real
      // allocation (hundreds of microseconds, sometimes milliseconds) between the caller's event and the kernel launch
      cudaMemPoolProps props{};
      props.allocType = cudaMemAllocationTypePinned;
      props.handleTypes = cudaMemHandleTypeNone;
      props.location.type = cudaMemLocationTypeDevice;
      props.location.id = dev;
      FPT_CUDA(cudaMemPoolCreate(&c.mem, &props));
      unsigned long long keep = ~0ull;
      FPT_CUDA(cudaMemPoolSetAttribute(c.mem, cudaMemPoolAttrReleaseThreshold, &keep));
      c.ready.store(true, std::memory_order_release);
    }
  }
  *out = &c;
  if (dev_out) *dev_out = dev;
  return FPT_OK;
}

bool finite_all(const double* x, int n) {
  for (int i = 0; i < n; ++i)
    if (!std::isfinite(x[i])) return false;
  return true;
}

int validate(const fpt_params* p, int64_t n_traj, double t_max) {
  if (!p || n_traj < 0) return FPT_E_INVALID;
  if (p->model < 0 || p->model > 1 || p->scheme < 0 || p->scheme > 2 || p->precision < 0 || p->precision > 2) return FPT_E_INVALID;
  // the hardware-sine variant exists for the paper's own kernels only (single precision, Euler as printed, a sine to take)
  if (p->precision == FPT_PREC_FP32_FAST && (p->scheme != FPT_SCHEME_PAPER || p->amp == 0.0)) return FPT_E_INVALID;
  if (p->check_every < 0) return FPT_E_INVALID;
  const double f[] = {p->alpha, p->temperature, p->amp, p->gamma0, p->nu, p->phi0, p->v0, p->threshold, p->dt, t_max};
  if (!finite_all(f, 10)) return FPT_E_INVALID;
  if (!(p->dt > 0.0) || !(t_max > 0.0) || p->temperature < 0.0) return FPT_E_INVALID;
  if (p->model == 1 && p->alpha < 0.0) return FPT_E_INVALID;
  if (!(t_max / p->dt < 0x1p53)) return FPT_E_INVALID;
  return FPT_OK;
}

int validate_opts(const fpt_launch_opts* o) {
  if (!o) return FPT_OK;
  if (o->block != 0 && (o->block < 32 || o->block > 256 || (o->block % 32) != 0)) return FPT_E_INVALID;
  if (o->blocks_per_sm < 0 || o->blocks_per_sm > 64 || o->max_blocks < 0) return FPT_E_INVALID;
  if (o->schedule != FPT_SCHEDULE_DYNAMIC && o->schedule != FPT_SCHEDULE_STATIC) return FPT_E_INVALID;
  if (o->tail_helper < -1 || o->tail_helper > 1 || o->specialise < -1 || o->specialise > 1) return FPT_E_INVALID;
  if (o->time_slice < -1 || o->time_slice > 1 || o->reserved != 0) return FPT_E_INVALID;
  if (o->consumers < 0 || o->consumers > kSpecMaxConsumersHost || o->producers < 0 || o->producers > kSpecMaxProducersHost)
    return FPT_E_INVALID;
  return FPT_OK;
}

int validate_hist(const fpt_hist* h) {
  if (!h) return FPT_OK;
  if (!h->out_counts || h->nbins < 1 || h->nbins > kMaxFusedBins || !std::isfinite(h->lo) || !std::isfinite(h->hi) || !(h->hi > h->lo))
    return FPT_E_INVALID;
  if (h->of < 0 || h->of > 1) return FPT_E_INVALID;
  return FPT_OK;
}

// derived constants, fp64, left-to-right products; the fp32 copies are each rounded once.
void derive(const fpt_params& p, double t_max, uint64_t seed, KParams& P) {
  std::memset(&P, 0, sizeof(P));
  P.alpha = p.alpha;
  P.amp = p.amp;
  P.gamma0 = p.gamma0;
  P.dgamma = p.nu * p.dt;
  P.phi0 = p.phi0;
  P.v0 = p.v0;
  P.thr = p.threshold;
  P.dt = p.dt;
  P.sigma = (p.model == 1) ? std::sqrt(2.0 * p.alpha * p.temperature * p.dt) : std::sqrt(2.0 * p.temperature * p.dt);
  P.h2 = 0.5 * p.dt;
  P.alpha_f = (float)p.alpha;
  P.amp_f = (float)p.amp;
  P.gamma0_f = (float)p.gamma0;
  P.nu_f = (float)p.nu;
  P.phi0_f = (float)p.phi0;
  P.v0_f = (float)p.v0;
  P.thr_f = (float)p.threshold;
  P.dt_f = (float)p.dt;
  P.sigma_f = (float)P.sigma;
  P.h2_f = (float)P.h2;
  P.first_id = p.first_id;
  P.n_cap = (unsigned long long)std::nearbyint(t_max / p.dt);
  const int macro = p.precision != FPT_PREC_FP64 ? 4 : 2;
  const unsigned long long long_cap = p.precision != FPT_PREC_FP64 ? kLongCap32 : kLongCap64;
  int K = p.check_every > 0 ? p.check_every : (P.n_cap >= long_cap ? kDefaultKLong : kDefaultK);
  if (p.check_every <= 0 && p.nu > 0.0 && p.amp > p.gamma0 &&
      std::fmin((double)P.n_cap, (p.amp - p.gamma0) / (p.nu * p.dt)) >= kRampLongSteps)
    K = kDefaultKRampLong;
  K = ((K + macro - 1) / macro) * macro;
  P.K = K;
  P.hist_of = -1;
  P.keys = philox_round_keys(seed);
}

// Trajectories that are decided at k = 0 (phi0 >= threshold: escaped at once, PAPER.md:166 applied to the initial state)
// or by n_cap == 0 (censored at once) are the same for every id: written by a fill kernel, no integration.
__global__ void fpt_fill_kernel(KParams P, int status, double fptv, double gam) {
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < P.n_traj; i += stride) {
    P.out_fpt[i] = fptv;
    if (P.out_gamma) P.out_gamma[i] = gam;
    P.out_status[i] = status;
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    if (status == kStatusEscaped) {
      P.ws->n_escaped = P.n_traj;
      if (P.hist_of >= 0) {
        const int slot = hist_slot(P.hist_of == 0 ? gam : fptv, P.hist_lo, P.hist_scale, P.nbins);
        if (slot >= 0) atomicAdd(&P.out_counts[slot], P.n_traj);
      }
    } else {
      P.ws->n_censored = P.n_traj;
      P.ws->useful_steps = 0;
    }
  }
}

// The call's statistics: counters of its workspace + the geometry the host chose, written to the caller's block (may be
// NULL) and to the call's slot of the per-device ring behind the deprecated fpt_last_stats.
__global__ void fpt_export_stats_kernel(const DevStats* ws, fpt_stats geo, fpt_stats* user, fpt_stats* slot,
                                        unsigned long long* slot_ticket, unsigned long long ticket) {
  geo.n_escaped = ws->n_escaped;
  geo.n_censored = ws->n_censored;
  geo.n_nan = ws->n_nan;
  geo.useful_steps = ws->useful_steps;
  geo.issued_lane_steps = ws->issued_lane_steps;
  geo.refill_atomics = ws->refill_atomics;
  geo.migrations = ws->migrations;
  geo.helper_lane_steps = ws->helper_lane_steps;
  geo.time_slices = ws->time_slices;
  if (user) *user = geo;
  *slot = geo;
  *slot_ticket = ticket;
}

struct WsGuard {            // the per-call workspaces go back to the pool on every path, stream ordered
  DevStats* ws = nullptr;
  void* slice = nullptr;    // time slicing: n_traj parking slots + the waiting ring
  cudaStream_t stream = nullptr;
  ~WsGuard() {
    if (slice) (void)cudaFreeAsync(slice, stream);
    if (ws) (void)cudaFreeAsync(ws, stream);
  }
};



// Opt in to more than 48 KB of shared memory when a launch needs it (fused histograms of many bins next to the drain pool
// and the tail helper's buffer; the specialised kernel's hand-over rings).  FPT_E_INVALID when it cannot fit at all.
int ensure_dynamic_smem(const void* fn, size_t dyn_bytes, int dev) {
  cudaFuncAttributes a{};
  FPT_CUDA(cudaFuncGetAttributes(&a, fn));
  if (a.sharedSizeBytes + dyn_bytes <= 48 * 1024) return FPT_OK;
  int optin = 0;
  FPT_CUDA(cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
  if (a.sharedSizeBytes + dyn_bytes > (size_t)optin) return FPT_E_INVALID;
  if ((size_t)a.maxDynamicSharedSizeBytes >= dyn_bytes) return FPT_OK;
  FPT_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn_bytes));
  return FPT_OK;
}

// the persistent kernel with the time-slicing code (ramped-bias states only)
const void* sliced_kernel(const fpt_params* p, bool amp) {
  if (p->precision == FPT_PREC_FP32_FAST) return persistent_sliced_kernel_f32_fast(p->model);
  return p->precision != FPT_PREC_FP64 ? persistent_sliced_kernel_f32(p->model, p->scheme, amp)
                                       : persistent_sliced_kernel_f64(p->model, p->scheme, amp);
}

int simulate_impl(const fpt_params* p, int64_t n_traj, uint64_t seed, double t_max, double* out_fpt, double* out_gamma,
                  int32_t* out_status, const fpt_hist* hist, const fpt_launch_opts* opts_in, fpt_stats* d_stats,
                  void* cuda_stream) {
  int rc = validate(p, n_traj, t_max);
  if (rc != FPT_OK) return rc;
  if (n_traj > 0 && (!out_fpt || !out_status)) return FPT_E_INVALID;   // empty outputs may be NULL
  if ((rc = validate_hist(hist)) != FPT_OK) return rc;
  if ((rc = validate_opts(opts_in)) != FPT_OK) return rc;
  if (n_traj == 0) return FPT_OK;
  const fpt_launch_opts cfg = opts_in ? *opts_in : t_opts;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  DeviceCtx* ctx = nullptr;
  int dev = 0;
  rc = device_ctx(&ctx, &dev);
  if (rc != FPT_OK) return rc;

  KParams P;
  derive(*p, t_max, seed, P);
  P.n_traj = (unsigned long long)n_traj;
  P.out_fpt = out_fpt;
  P.out_gamma = out_gamma;
  P.out_status = out_status;
  P.dbg_seq0 = t_dbg_seq0;
  const bool with_hist = hist != nullptr;
  if (with_hist) {
    P.hist_of = hist->of;
    P.nbins = hist->nbins;
    P.hist_lo = hist->lo;
    P.hist_scale = (double)hist->nbins / (hist->hi - hist->lo);
    P.out_counts = (unsigned long long*)hist->out_counts;
  }
  WsGuard guard;
  guard.stream = stream;
  FPT_CUDA(cudaMallocFromPoolAsync(&guard.ws, sizeof(DevStats), ctx->mem, stream));
  DevStats* ws = guard.ws;
  FPT_CUDA(cudaMemsetAsync(ws, 0, sizeof(DevStats), stream));
  P.ws = ws;

  int grid = 1, block = 128, kernel = FPT_KERNEL_FILL;
  const bool fp32 = p->precision != FPT_PREC_FP64;
  const bool fast_sine = p->precision == FPT_PREC_FP32_FAST;
  const int sms = ctx->sm_count;
  // the crossing test applied to the initial state: >= (strict > for the paper's scheme), in the state's precision
  const bool strict = p->scheme == FPT_SCHEME_PAPER;
  const bool at_once_escaped = fp32 ? (strict ? !((float)p->phi0 <= (float)p->threshold) : !((float)p->phi0 < (float)p->threshold))
                                    : (strict ? !(p->phi0 <= p->threshold) : !(p->phi0 < p->threshold));
  if (at_once_escaped || P.n_cap == 0) {
    block = 256;
    grid = (int)std::min<int64_t>((n_traj + block - 1) / block, (int64_t)sms * 8);
    const int status = at_once_escaped ? kStatusEscaped : kStatusCensored;
    const double fptv = at_once_escaped ? 0.0 : -1.0;
    const double gam = std::fma(P.dgamma, at_once_escaped ? 0.0 : (double)P.n_cap, P.gamma0);
    fpt_fill_kernel<<<grid, block, 0, stream>>>(P, status, fptv, gam);
    FPT_CUDA(cudaGetLastError());
  } else {
    const bool amp = p->amp != 0.0, ramp = p->nu != 0.0;
    const size_t hist_bytes = with_hist ? (size_t)(hist->nbins + 2) * sizeof(unsigned int) : 0;
    const long long unit = 128LL * sms;                         // one warp per SM sub-partition everywhere
    // ---- which kernel.  The specialised kernel (consumers integrate, producers generate the normals) is for launches
    // that cannot fill the GPU: a warp that runs (nearly) alone advances at the latency of its own instruction stream, and
    // splitting that stream over two warps on different sub-partitions shortens it (measured on B200, clk per step of a
    // lone warp, persistent -> specialised: Heun underdamped 247 -> 184, Heun overdamped 360 -> 310, Euler overdamped
    // 210 -> 172, Euler underdamped 178 -> 170, fp32 Heun underdamped 119 -> 91).  Up to two consumers per SM every
    // consumer has a sub-partition to itself and every variant gains (10-25 % at 5000 trajectories); with four per SM only
    // the fp64 Heun variants still gain (2-6 %), the others lose.  Trajectories in flight: the persistent kernel would
    // keep n_traj / 5 of a constant-bias job in flight (below), all of a ramped one.
    const bool explicit_geometry = cfg.block > 0 || cfg.blocks_per_sm > 0;
    // consumers per SM wanted: all trajectories of a ramped job, a fifth of a constant-bias job but at least two
    // consumers' worth (below that every consumer is alone on its sub-partition anyway)
    const long long lanes_wanted = ramp ? n_traj : std::max<long long>(n_traj / 5, std::min<long long>(n_traj, 64LL * sms));
    const long long nc_wanted = (lanes_wanted + 32LL * sms - 1) / (32LL * sms);
    const bool spec_pays = nc_wanted <= 2 || (nc_wanted <= 8 && !fp32 && p->scheme == FPT_SCHEME_HEUN);
    const bool spec = amp && !fast_sine && cfg.schedule == FPT_SCHEDULE_DYNAMIC && cfg.specialise >= 0 &&
                      (cfg.specialise == 1 || (!explicit_geometry && spec_pays));
    const void* fn = nullptr;
    size_t smem = hist_bytes;
    long long blocks = 0;
    bool want_slice = cfg.time_slice == 1 && ramp;     // the slicing kernels exist for the ramped-bias states only
    if (spec) {
      size_t fixed = 0, chan = 0;
      fn = fp32 ? specialised_kernel_f32(p->model, p->scheme, ramp, &fixed, &chan)
                : specialised_kernel_f64(p->model, p->scheme, ramp, &fixed, &chan);
      int NC = cfg.consumers > 0 ? cfg.consumers : (int)std::min<long long>(4, std::max<long long>(1, nc_wanted));
      const int NP = cfg.producers > 0 ? cfg.producers : 1;
      P.spec_consumers = NC;
      P.spec_producers = NP;
      // a consumer must not share its SM sub-partition with a producer (fpt_specialised.cuh): with one producer each and
      // more than two consumers, even warps consume and odd warps produce
      P.spec_layout = (NP == 1 && NC > 2) ? 1 : 0;
      P.K = fp32 ? kSpecChunk32 : kSpecChunk64;                   // one poll per hand-over chunk
      block = 32 * NC * (1 + NP);
      smem = fixed + (size_t)NC * chan + hist_bytes;
      rc = ensure_dynamic_smem(fn, smem, dev);
      if (rc != FPT_OK) return rc;
      int per_sm = 0;
      FPT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, block, smem));
      if (per_sm < 1) return FPT_E_CUDA;
      per_sm = cfg.blocks_per_sm > 0 ? std::min(per_sm, cfg.blocks_per_sm) : 1;
      blocks = (long long)per_sm * sms;
      const long long needed = (n_traj + 32LL * NC - 1) / (32LL * NC);
      if (blocks > needed) blocks = needed;
      kernel = FPT_KERNEL_SPECIALISED;
    } else {
      fn = fast_sine ? persistent_kernel_f32_fast(p->model, ramp)
           : fp32    ? persistent_kernel_f32(p->model, p->scheme, amp, ramp)
                     : persistent_kernel_f64(p->model, p->scheme, amp, ramp);
      rc = ensure_dynamic_smem(fn, smem, dev);
      if (rc != FPT_OK) return rc;
      auto max_blocks_per_sm = [&](int blk, int* out) -> cudaError_t {
        return cudaOccupancyMaxActiveBlocksPerMultiprocessor(out, fn, blk, smem);
      };
      if (explicit_geometry) {
        // explicit geometry: block x min(blocks_per_sm, occupancy limit) per SM
        block = cfg.block > 0 ? cfg.block : 128;
        int per_sm = 0;
        FPT_CUDA(max_blocks_per_sm(block, &per_sm));
        if (per_sm < 1) return FPT_E_CUDA;
        if (cfg.blocks_per_sm > 0) per_sm = std::min(per_sm, cfg.blocks_per_sm);
        blocks = (long long)per_sm * sms;
      } else {
        // Default geometry.  Resident lanes = n_traj / R, at least one warp per SM sub-partition (128 lanes per SM) and at
        // most what the registers allow.  R = 1 for a ramped bias (nu != 0: switching happens in a narrow window, all
        // trajectories are about equally long, so throughput is everything); R = 5 for a constant bias (escape is a
        // Poisson process, lengths are exponential: a launch lasts at least as long as its longest trajectory, and that
        // one runs fastest when few warps share its SM sub-partition; the refills keep the lanes busy meanwhile).
        const long long R = ramp ? 1 : 5;
        // ramped: round UP, so that a job that fits resident at once runs as one wave (C4: 65536 equal-length trajectories
        // on 4 x 128 lanes per SM, not 3 x 128 plus a straggler wave); constant bias: round down, more refills per lane
        long long units = ramp ? (n_traj + unit - 1) / unit : n_traj / (R * unit);
        if (n_traj >= unit && units >= 1) {
          int per_sm128 = 0;
          FPT_CUDA(max_blocks_per_sm(128, &per_sm128));
          if (per_sm128 < 1) return FPT_E_CUDA;
          // Time slicing (fpt_integrator.cuh): equal-length trajectories that do not fill a whole number of waves.  Between
          // one and three waves with the last one ragged by more than 5 %: slice at full occupancy (beyond three waves the
          // spread of the escape times blends the waves by itself, measured on config 4's twin at 3.46 waves: slicing costs
          // 2 % there).  fp32, between 3 and 3.8 blocks of 128 per SM (config 4: 3.46): 3 blocks per SM + slicing instead of
          // 4 and 3 blocks side by side -- measured on B200, a sub-partition with 3 warps does 95 % of the work of one with
          // 4, so 3 everywhere for n / (3 x 128 x #SM) "waves" beats waiting for the SMs that got 4 (0.509 -> 0.572).
          if (ramp && cfg.time_slice >= 0 && cfg.schedule == FPT_SCHEDULE_DYNAMIC) {
            const double f = (double)n_traj / (double)unit;
            const double waves = f / (double)per_sm128;
            if (waves > 1.0 && waves < 3.0 && std::ceil(waves) > 1.05 * waves) want_slice = true;
            else if (fp32 && per_sm128 >= 4 && f > 3.0 && f < 3.8) { want_slice = true; units = 3; }
          }
          units = std::min<long long>(units, per_sm128);
          if (!fp32 && units >= 2 && (units % 2) == 0) {          // fp64: pairs of 128 as one 256-thread block (compaction
                                                                  // works over more lanes; measured +3 %, fp32: -20 %)
            int per_sm256 = 0;
            FPT_CUDA(max_blocks_per_sm(256, &per_sm256));
            if (per_sm256 >= units / 2) { block = 256; blocks = (units / 2) * sms; }
          }
          if (blocks == 0) { block = 128; blocks = units * sms; }
        } else {
          const long long lanes = std::min<long long>(n_traj, unit);
          block = (int)std::min<long long>(128, std::max<long long>(32, ((lanes + sms - 1) / sms + 31) / 32 * 32));
          blocks = (lanes + block - 1) / block;
        }
      }
      const long long needed = (n_traj + block - 1) / block;      // never more lanes than trajectories
      if (blocks > needed) blocks = needed;
      kernel = FPT_KERNEL_PERSISTENT;
    }
    if (cfg.max_blocks > 0 && blocks > cfg.max_blocks) blocks = cfg.max_blocks;
    grid = (int)blocks;
    if (want_slice && !spec && cfg.schedule == FPT_SCHEDULE_DYNAMIC && (long long)grid * block < n_traj &&
        (cfg.time_slice == 1 || P.n_cap >= (1ull << 15))) {
      // quantum: a power of two of steps, a multiple of K, at least 2048 (a hand-over costs a warp about as much as ten
      // steps) and at least 1/2048 of the cap
      unsigned long long q = 2048;
      while (q < (unsigned long long)P.K || q * 2048ull < P.n_cap) q <<= 1;
      if (t_dbg_slice_q != 0ull) {                                  // test hook (fpt_dbg.h)
        q = t_dbg_slice_q;
        while (q < (unsigned long long)P.K) q <<= 1;
      }
      if ((q % (unsigned long long)P.K) != 0ull) q *= (unsigned long long)P.K;       // K not a power of two: any multiple will do
      if ((q & (q - 1ull)) == 0ull) {
        fn = sliced_kernel(p, amp);                                 // the variant of the kernel that holds the slicing code
        rc = ensure_dynamic_smem(fn, smem, dev);
        if (rc != FPT_OK) return rc;
        int per_sm_s = 0;
        FPT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm_s, fn, block, smem));
        if (per_sm_s < 1) return FPT_E_CUDA;
        if ((long long)per_sm_s * sms < (long long)grid) grid = per_sm_s * sms;       // all blocks resident (slicing balances any grid)
        P.slice_cap = ((unsigned long long)n_traj + (unsigned long long)grid - 1ull) / (unsigned long long)grid;
        const size_t slot_bytes = (size_t)n_traj * sizeof(ParkSlot);
        const size_t ring_bytes = (size_t)grid * (size_t)P.slice_cap * sizeof(unsigned long long);
        FPT_CUDA(cudaMallocFromPoolAsync(&guard.slice, slot_bytes + ring_bytes, ctx->mem, stream));
        P.slice_slots = (ParkSlot*)guard.slice;
        P.slice_ring = (unsigned long long*)((char*)guard.slice + slot_bytes);
        FPT_CUDA(cudaMemsetAsync(P.slice_ring, 0, ring_bytes, stream));
        P.slice_mask = q - 1ull;
      }
    }
    P.schedule = cfg.schedule;
    P.tail_helper = cfg.tail_helper >= 0 ? 1 : 0;
    void* args[] = {(void*)&P};
    FPT_CUDA(cudaLaunchKernel(fn, dim3(grid), dim3(block), args, smem, stream));
  }
  // this call's statistics -> the caller's block and the call's slot of the "last call" ring; then release the workspace
  fpt_stats geo{};
  geo.n_traj = (uint64_t)n_traj;
  geo.n_cap = P.n_cap;
  geo.grid = grid;
  geo.block = block;
  geo.check_every = P.K;
  geo.kernel = kernel;
  const unsigned long long ticket = ctx->next_ticket.fetch_add(1);
  const int slot = (int)(ticket % kLastSlots);
  fpt_export_stats_kernel<<<1, 1, 0, stream>>>(ws, geo, d_stats, ctx->d_last + slot, ctx->d_ticket + slot, ticket);
  FPT_CUDA(cudaGetLastError());
  t_last.ticket[dev] = ticket;
  return FPT_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// Standalone histogram (S8 / DESIGN.md 4.11): shared-memory bins per block when they fit, global atomics otherwise.
__global__ void fpt_histogram_kernel(const double* __restrict__ values, const int* __restrict__ status, long long n,
                                     double lo, double scale, int nbins, unsigned long long* counts, int use_smem) {
  extern __shared__ unsigned int sh[];
  if (use_smem) {
    for (int i = threadIdx.x; i < nbins + 2; i += blockDim.x) sh[i] = 0u;
    __syncthreads();
  }
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    if (status && status[i] != 0) continue;
    const int slot = hist_slot(values[i], lo, scale, nbins);
    if (slot < 0) continue;
    if (use_smem) atomicAdd(&sh[slot], 1u);
    else atomicAdd(&counts[slot], 1ull);
  }
  if (use_smem) {
    __syncthreads();
    for (int i = threadIdx.x; i < nbins + 2; i += blockDim.x) {
      const unsigned c = sh[i];
      if (c) atomicAdd(&counts[i], (unsigned long long)c);
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Roofline denominators: independent fma chains, 8 per thread, every SM full.  The SM clock is read from clock64 (a
// per-SM counter): every block records its start and end into its SM's slot, the host takes the longest span.
constexpr int kMaxSm = 256;
struct PeakClocks {
  long long t_min[kMaxSm];
  long long t_max[kMaxSm];
};

template <typename T>
__global__ void __launch_bounds__(256) fpt_peak_kernel(T* sink, int iters, PeakClocks* clk) {
  T a[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) a[i] = (T)(threadIdx.x + i) * (T)1e-3;
  const T m = (T)0.999, c = (T)1e-3;
  const long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        if constexpr (sizeof(T) == 8) a[i] = __fma_rn(a[i], m, c);
        else a[i] = __fmaf_rn(a[i], m, c);
      }
    }
  }
  const long long t1 = clock64();
  T s = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += a[i];
  if (s == (T)123456.789) sink[0] = s;
  if (threadIdx.x == 0) {
    unsigned smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    if (smid < (unsigned)kMaxSm) {
      atomicMin(&clk->t_min[smid], t0);
      atomicMax(&clk->t_max[smid], t1);
    }
  }
}

template <typename T>
int peak_impl(double seconds, double* inst_per_s, double* sm_clock_hz) {
  if (!inst_per_s || !(seconds > 0.0) || seconds > 30.0) return FPT_E_INVALID;
  DeviceCtx* ctx = nullptr;
  int rc = device_ctx(&ctx);
  if (rc != FPT_OK) return rc;
  T* sink = nullptr;
  PeakClocks* d_clk = nullptr;
  FPT_CUDA(cudaMalloc(&sink, sizeof(T)));
  FPT_CUDA(cudaMalloc(&d_clk, sizeof(PeakClocks)));
  cudaEvent_t e0, e1;
  FPT_CUDA(cudaEventCreate(&e0));
  FPT_CUDA(cudaEventCreate(&e1));
  const int block = 256, grid = ctx->sm_count * 8;            // 2048 threads per SM, one wave
  const int iters = sizeof(T) == 8 ? 4096 : 16384;
  const double inst_per_launch = (double)grid * block * (double)iters * 64.0;
  std::vector<long long> h(2 * kMaxSm);
  auto reset_clk = [&]() {
    for (int i = 0; i < kMaxSm; ++i) { h[i] = 0x7fffffffffffffffll; h[kMaxSm + i] = 0; }
    return cudaMemcpy(d_clk, h.data(), sizeof(PeakClocks), cudaMemcpyHostToDevice);
  };
  FPT_CUDA(reset_clk());
  fpt_peak_kernel<T><<<grid, block>>>(sink, iters, d_clk);   // warm-up
  FPT_CUDA(cudaDeviceSynchronize());
  double total_ms = 0.0;
  float ms = 0.f;
  int launches = 0;
  // load the GPU for `seconds`, then report the LAST launch: the sustained rate and clock under this load
  do {
    FPT_CUDA(reset_clk());
    FPT_CUDA(cudaEventRecord(e0));
    fpt_peak_kernel<T><<<grid, block>>>(sink, iters, d_clk);
    FPT_CUDA(cudaEventRecord(e1));
    FPT_CUDA(cudaEventSynchronize(e1));
    FPT_CUDA(cudaEventElapsedTime(&ms, e0, e1));
    total_ms += ms;
    ++launches;
  } while (total_ms < seconds * 1e3 && launches < 100000);
  *inst_per_s = inst_per_launch / (ms * 1e-3);
  FPT_CUDA(cudaMemcpy(h.data(), d_clk, sizeof(PeakClocks), cudaMemcpyDeviceToHost));
  long long span = 0;
  for (int i = 0; i < kMaxSm; ++i)
    if (h[kMaxSm + i] > h[i]) span = std::max(span, h[kMaxSm + i] - h[i]);
  if (sm_clock_hz) *sm_clock_hz = (double)span / (ms * 1e-3);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  cudaFree(d_clk);
  return FPT_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// test-hook kernels
__global__ void dbg_philox_kernel(PhiloxKeys K, unsigned long long id0, long long n, unsigned long long block, uint32_t* out) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const unsigned long long id = id0 + (unsigned long long)i;
  uint32_t o0, o1, o2, o3;
  philox_block(K, (uint32_t)block, (uint32_t)(block >> 32), (uint32_t)id, (uint32_t)(id >> 32), o0, o1, o2, o3);
  out[4 * i] = o0; out[4 * i + 1] = o1; out[4 * i + 2] = o2; out[4 * i + 3] = o3;
}
__global__ void dbg_normals64_kernel(PhiloxKeys K, unsigned long long id, unsigned long long b0, long long n, double* out) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const unsigned long long b = b0 + (unsigned long long)i;
  uint32_t o0, o1, o2, o3;
  philox_block(K, (uint32_t)b, (uint32_t)(b >> 32), (uint32_t)id, (uint32_t)(id >> 32), o0, o1, o2, o3);
  double za, zb;
  normal_pair(o0, o1, o2, o3, za, zb);
  out[2 * i] = za; out[2 * i + 1] = zb;
}
__global__ void dbg_normals32_kernel(PhiloxKeys K, unsigned long long id, unsigned long long b0, long long n, float* out) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const unsigned long long b = b0 + (unsigned long long)i;
  uint32_t o0, o1, o2, o3;
  philox_block(K, (uint32_t)b, (uint32_t)(b >> 32), (uint32_t)id, (uint32_t)(id >> 32), o0, o1, o2, o3);
  float z0, z1, z2, z3;
  normal_pair_f(o0, o1, z0, z1);
  normal_pair_f(o2, o3, z2, z3);
  out[4 * i] = z0; out[4 * i + 1] = z1; out[4 * i + 2] = z2; out[4 * i + 3] = z3;
}
__global__ void dbg_unary64_kernel(int which, const double* x, double* y, long long n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  y[i] = which == 0 ? sin_drift(x[i]) : neg2log(x[i]);
}
__global__ void dbg_unary32_kernel(int which, const float* x, float* y, long long n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  y[i] = which == 0 ? sin_drift_f(x[i]) : neg2log_f(x[i]);
}
__global__ void dbg_sincos64_kernel(const unsigned long long* Y, double* c, double* s, long long n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double cc, ss;
  sincos_turns((uint32_t)(Y[i] >> 32), (uint32_t)Y[i], cc, ss);
  c[i] = cc; s[i] = ss;
}
__global__ void dbg_sincos32_kernel(const uint32_t* o, float* c, float* s, long long n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  float cc, ss;
  sincos_turns_f(o[i], cc, ss);
  c[i] = cc; s[i] = ss;
}

// guard-free division / square root against nvcc's builtins on operands drawn from the real pipeline
// (Philox block -> u1 -> m -> (m-1)/(m+1); w = -2 ln u1 -> sqrt w), fp64 and fp32: out[0..3] = mismatch counts
__global__ void dbg_selfcheck_kernel(PhiloxKeys K, unsigned long long id0, int blocks_per_thread, unsigned long long* out) {
  const unsigned long long id = id0 + (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  unsigned bad_div = 0, bad_sqrt = 0, bad_divf = 0, bad_sqrtf = 0;
  for (int b = 0; b < blocks_per_thread; ++b) {
    uint32_t o0, o1, o2, o3;
    philox_block(K, (uint32_t)b, 0u, (uint32_t)id, (uint32_t)(id >> 32), o0, o1, o2, o3);
    {
      const double d = __hiloint2double((int)(0x3FF00000u | (o0 >> 12)), (int)__funnelshift_r(o1, o0, 12));
      const double u1 = __dadd_rn(__dadd_rn(d, -1.0), 0x1p-53);
      const uint32_t hi2 = (uint32_t)__double2hiint(u1) + (0x3FF00000u - 0x3FE6A09Eu);
      const double m = __hiloint2double((int)((hi2 & 0x000FFFFFu) + 0x3FE6A09Eu), __double2loint(u1));
      const double a = __dadd_rn(m, -1.0), bb = __dadd_rn(m, 1.0);
      if (__double_as_longlong(div_rn_inrange(a, bb)) != __double_as_longlong(__ddiv_rn(a, bb))) ++bad_div;
      const double w = neg2log(u1);
      if (__double_as_longlong(sqrt_rn_inrange(w)) != __double_as_longlong(__dsqrt_rn(w))) ++bad_sqrt;
      // a second, denser family: w straight from the random bits, spread over [2^-52, 128)
      const double w2 = __hiloint2double((int)(0x3CB00000u + (o2 % 0x03B00000u)), (int)o3);
      if (__double_as_longlong(sqrt_rn_inrange(w2)) != __double_as_longlong(__dsqrt_rn(w2))) ++bad_sqrt;
    }
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const uint32_t o = h ? o2 : o0;
      const float u1 = __fmaf_rn(__uint2float_rn(o), 0x1p-32f, 0x1p-33f);
      const uint32_t ix2 = (uint32_t)__float_as_int(u1) + (0x3f800000u - 0x3f3504f3u);
      const float m = __int_as_float((int)((ix2 & 0x007fffffu) + 0x3f3504f3u));
      const float a = __fadd_rn(m, -1.0f), bb = __fadd_rn(m, 1.0f);
      if (__float_as_int(div_rn_inrange_f(a, bb)) != __float_as_int(__fdiv_rn(a, bb))) ++bad_divf;
      const float w = neg2log_f(u1);
      if (__float_as_int(sqrt_rn_inrange_f(w)) != __float_as_int(__fsqrt_rn(w))) ++bad_sqrtf;
      const float w2 = __int_as_float((int)(0x33000000u + ((h ? o3 : o1) % 0x10000000u)));      // [2^-25, 2^7)
      if (__float_as_int(sqrt_rn_inrange_f(w2)) != __float_as_int(__fsqrt_rn(w2))) ++bad_sqrtf;
    }
  }
  if (bad_div) atomicAdd(&out[0], (unsigned long long)bad_div);
  if (bad_sqrt) atomicAdd(&out[1], (unsigned long long)bad_sqrt);
  if (bad_divf) atomicAdd(&out[2], (unsigned long long)bad_divf);
  if (bad_sqrtf) atomicAdd(&out[3], (unsigned long long)bad_sqrtf);
}

inline int grid_for(long long n, int block) { return (int)((n + block - 1) / block); }

}  // namespace

// =================================================================================================================
extern "C" {

int fpt_simulate(const fpt_params* p, int64_t n_traj, uint64_t seed, double t_max, double* out_fpt,
                 double* out_gamma_at_escape, int32_t* out_status, void* cuda_stream) {
  return simulate_impl(p, n_traj, seed, t_max, out_fpt, out_gamma_at_escape, out_status, nullptr, nullptr, nullptr, cuda_stream);
}

int fpt_simulate_hist(const fpt_params* p, int64_t n_traj, uint64_t seed, double t_max, double* out_fpt,
                      double* out_gamma_at_escape, int32_t* out_status, int32_t hist_of, double lo, double hi,
                      int32_t nbins, uint64_t* out_counts, void* cuda_stream) {
  const fpt_hist h{hist_of, nbins, lo, hi, out_counts};
  return simulate_impl(p, n_traj, seed, t_max, out_fpt, out_gamma_at_escape, out_status, &h, nullptr, nullptr, cuda_stream);
}

int fpt_simulate_ex(const fpt_params* p, int64_t n_traj, uint64_t seed, double t_max, double* out_fpt,
                    double* out_gamma_at_escape, int32_t* out_status, const fpt_hist* hist, const fpt_launch_opts* opts,
                    fpt_stats* d_stats, void* cuda_stream) {
  return simulate_impl(p, n_traj, seed, t_max, out_fpt, out_gamma_at_escape, out_status, hist, opts, d_stats, cuda_stream);
}

int fpt_histogram(const double* values, const int32_t* status, int64_t n, double lo, double hi, int32_t nbins,
                  uint64_t* out_counts, void* cuda_stream) {
  if (!values || !out_counts || n < 0 || nbins < 1 || !std::isfinite(lo) || !std::isfinite(hi) || !(hi > lo)) return FPT_E_INVALID;
  if (n == 0) return FPT_OK;
  DeviceCtx* ctx = nullptr;
  int rc = device_ctx(&ctx);
  if (rc != FPT_OK) return rc;
  const double scale = (double)nbins / (hi - lo);
  const int block = 256;
  const int grid = (int)std::min<long long>(grid_for(n, block), (long long)ctx->sm_count * 8);
  const int use_smem = nbins <= kMaxFusedBins ? 1 : 0;
  const size_t smem = use_smem ? (size_t)(nbins + 2) * sizeof(unsigned int) : 0;
  fpt_histogram_kernel<<<grid, block, smem, (cudaStream_t)cuda_stream>>>(values, status, (long long)n, lo, scale, nbins,
                                                                         (unsigned long long*)out_counts, use_smem);
  FPT_CUDA(cudaGetLastError());
  return FPT_OK;
}

int fpt_simulate_host(const fpt_params* p, int64_t n_traj, uint64_t seed, double t_max, double* h_fpt, double* h_gamma,
                      int32_t* h_status, int32_t hist_of, double lo, double hi, int32_t nbins, uint64_t* h_counts) {
  int rc = validate(p, n_traj, t_max);
  if (rc != FPT_OK) return rc;
  if (n_traj == 0) return FPT_OK;
  if (!h_fpt || !h_status) return FPT_E_INVALID;
  if (h_counts && nbins < 1) return FPT_E_INVALID;
  DeviceCtx* hctx = nullptr;
  rc = device_ctx(&hctx);
  if (rc != FPT_OK) return rc;
  cudaStream_t stream = nullptr;
  FPT_CUDA(cudaStreamCreateWithFlags(&stream, cudaStreamNonBlocking));
  const size_t n = (size_t)n_traj;
  const size_t cnt_bytes = h_counts ? (size_t)(nbins + 2) * 8 : 0;
  const size_t bytes = n * (8 + (h_gamma ? 8 : 0) + 4) + cnt_bytes;
  char* d = nullptr;
  cudaError_t e = cudaMallocFromPoolAsync((void**)&d, bytes, hctx->mem, stream);
  if (e != cudaSuccess) { g_last_cuda = e; (void)cudaGetLastError(); cudaStreamDestroy(stream); return FPT_E_CUDA; }
  double* d_fpt = (double*)d;
  double* d_gam = h_gamma ? d_fpt + n : nullptr;
  uint64_t* d_cnt = h_counts ? (uint64_t*)(d + n * (8 + (h_gamma ? 8 : 0))) : nullptr;
  int32_t* d_st = (int32_t*)(d + n * (8 + (h_gamma ? 8 : 0)) + cnt_bytes);
  // every copy is checked; the first failure is reported after the buffer has been released and the stream drained
  auto note = [&](cudaError_t err) { if (err != cudaSuccess && e == cudaSuccess) e = err; };
  if (h_counts) {
    note(cudaMemcpyAsync(d_cnt, h_counts, cnt_bytes, cudaMemcpyHostToDevice, stream));
    if (e == cudaSuccess) rc = fpt_simulate_hist(p, n_traj, seed, t_max, d_fpt, d_gam, d_st, hist_of, lo, hi, nbins, d_cnt, stream);
  } else {
    rc = fpt_simulate(p, n_traj, seed, t_max, d_fpt, d_gam, d_st, stream);
  }
  if (rc == FPT_OK && e == cudaSuccess) {
    note(cudaMemcpyAsync(h_fpt, d_fpt, n * 8, cudaMemcpyDeviceToHost, stream));
    if (h_gamma) note(cudaMemcpyAsync(h_gamma, d_gam, n * 8, cudaMemcpyDeviceToHost, stream));
    note(cudaMemcpyAsync(h_status, d_st, n * 4, cudaMemcpyDeviceToHost, stream));
    if (h_counts) note(cudaMemcpyAsync(h_counts, d_cnt, cnt_bytes, cudaMemcpyDeviceToHost, stream));
  }
  note(cudaFreeAsync(d, stream));
  note(cudaStreamSynchronize(stream));
  cudaStreamDestroy(stream);
  if (rc == FPT_OK && e != cudaSuccess) { g_last_cuda = e; (void)cudaGetLastError(); return FPT_E_CUDA; }
  return rc;
}

int fpt_simulate_sweep(const fpt_params* sets, int32_t n_sets, int64_t n_per_set, uint64_t seed, const double* t_max,
                       double* out_fpt, double* out_gamma_at_escape, int32_t* out_status, void* cuda_stream) {
  if (!sets || !t_max || n_sets < 0 || n_per_set < 0) return FPT_E_INVALID;
  for (int32_t i = 0; i < n_sets; ++i) {                       // nothing is launched unless every set is valid
    const int rc = validate(&sets[i], n_per_set, t_max[i]);
    if (rc != FPT_OK) return rc;
  }
  if (n_sets == 0 || n_per_set == 0) return FPT_OK;
  if (!out_fpt || !out_status) return FPT_E_INVALID;
  DeviceCtx* ctx = nullptr;
  int rc = device_ctx(&ctx);
  if (rc != FPT_OK) return rc;
  // one sweep at a time per device on the stream pool (the launches of two sweeps would interleave on it otherwise); the
  // section only enqueues, so the lock is held for microseconds per set
  std::lock_guard<std::mutex> lk(ctx->mu);
  if (!ctx->pool_ready) {
    for (int i = 0; i < kSweepStreams; ++i) FPT_CUDA(cudaStreamCreateWithFlags(&ctx->pool[i], cudaStreamNonBlocking));
    ctx->pool_ready = true;
  }
  cudaStream_t caller = (cudaStream_t)cuda_stream;
  const int used = n_sets < kSweepStreams ? n_sets : kSweepStreams;
  // per-call events: recorded, waited on and destroyed here (the runtime defers the destruction until they complete)
  cudaEvent_t fork = nullptr, done[kSweepStreams] = {};
  cudaError_t e = cudaEventCreateWithFlags(&fork, cudaEventDisableTiming);
  for (int i = 0; i < used && e == cudaSuccess; ++i) e = cudaEventCreateWithFlags(&done[i], cudaEventDisableTiming);
  int forked = 0;
  // fork: the pool streams start after everything already queued on the caller's stream
  if (e == cudaSuccess) e = cudaEventRecord(fork, caller);
  for (int i = 0; i < used && e == cudaSuccess; ++i) {
    e = cudaStreamWaitEvent(ctx->pool[i], fork, 0);
    if (e == cudaSuccess) forked = i + 1;
  }
  // the sets run side by side: when together they fill the GPU no warp runs alone, and the persistent kernel (every warp
  // self-sufficient, little shared memory, several blocks per SM) is the one to use for each of them
  fpt_launch_opts opts = t_opts;
  if (opts.specialise == 0 && (long long)n_sets * n_per_set >= 256LL * ctx->sm_count) opts.specialise = -1;
  for (int32_t i = 0; i < n_sets && rc == FPT_OK && e == cudaSuccess; ++i) {
    const size_t off = (size_t)i * (size_t)n_per_set;
    rc = simulate_impl(&sets[i], n_per_set, seed, t_max[i], out_fpt + off, out_gamma_at_escape ? out_gamma_at_escape + off : nullptr,
                       out_status + off, nullptr, &opts, nullptr, ctx->pool[i % kSweepStreams]);
  }
  // join, ALWAYS (also after a failed launch): the caller's stream continues when every forked pool stream is done
  for (int i = 0; i < forked; ++i) {
    cudaError_t e2 = cudaEventRecord(done[i], ctx->pool[i]);
    if (e2 == cudaSuccess) e2 = cudaStreamWaitEvent(caller, done[i], 0);
    if (e2 != cudaSuccess && e == cudaSuccess) e = e2;
  }
  if (fork) cudaEventDestroy(fork);
  for (int i = 0; i < used; ++i)
    if (done[i]) cudaEventDestroy(done[i]);
  if (rc == FPT_OK && e != cudaSuccess) { g_last_cuda = e; (void)cudaGetLastError(); return FPT_E_CUDA; }
  return rc;
}

int fpt_set_launch(int32_t block, int32_t blocks_per_sm, int32_t max_blocks) {
  fpt_launch_opts o = t_opts;
  o.block = block;
  o.blocks_per_sm = blocks_per_sm;
  o.max_blocks = max_blocks;
  if (validate_opts(&o) != FPT_OK) return FPT_E_INVALID;
  t_opts = o;
  return FPT_OK;
}

int fpt_set_schedule(int32_t schedule) {
  if (schedule != FPT_SCHEDULE_DYNAMIC && schedule != FPT_SCHEDULE_STATIC) return FPT_E_INVALID;
  t_opts.schedule = schedule;
  return FPT_OK;
}

int fpt_set_tail_helper(int32_t on) {
  if (on != 0 && on != 1) return FPT_E_INVALID;
  t_opts.tail_helper = on ? 1 : -1;
  return FPT_OK;
}

int fpt_set_specialise(int32_t specialise, int32_t consumers, int32_t producers) {
  fpt_launch_opts o = t_opts;
  o.specialise = specialise;
  o.consumers = consumers;
  o.producers = producers;
  if (validate_opts(&o) != FPT_OK) return FPT_E_INVALID;
  t_opts = o;
  return FPT_OK;
}

int fpt_last_stats(fpt_stats* out) {
  if (!out) return FPT_E_INVALID;
  DeviceCtx* ctx = nullptr;
  int dev = 0;
  int rc = device_ctx(&ctx, &dev);
  if (rc != FPT_OK) return rc;
  std::memset(out, 0, sizeof(*out));
  const unsigned long long ticket = t_last.ticket[dev];
  if (ticket == 0) return FPT_OK;                              // this thread has made no call on this device
  FPT_CUDA(cudaDeviceSynchronize());
  const int slot = (int)(ticket % kLastSlots);
  unsigned long long owner = 0;
  FPT_CUDA(cudaMemcpy(&owner, ctx->d_ticket + slot, sizeof(owner), cudaMemcpyDeviceToHost));
  if (owner != ticket) return FPT_OK;                          // kLastSlots later calls have recycled the slot: zeros
  FPT_CUDA(cudaMemcpy(out, ctx->d_last + slot, sizeof(*out), cudaMemcpyDeviceToHost));
  return FPT_OK;
}

int fpt_fp64_peak(double seconds, double* inst_per_s, double* sm_clock_hz) { return peak_impl<double>(seconds, inst_per_s, sm_clock_hz); }
int fpt_fp32_peak(double seconds, double* inst_per_s, double* sm_clock_hz) { return peak_impl<float>(seconds, inst_per_s, sm_clock_hz); }

const char* fpt_strerror(int code) {
  switch (code) {
    case FPT_OK: return "ok";
    case FPT_E_INVALID: return "invalid argument";
    case FPT_E_CUDA: return g_last_cuda != cudaSuccess ? cudaGetErrorString(g_last_cuda) : "CUDA failure";
    case FPT_E_TOO_LARGE: return "size beyond the fixed maximum of this entry point (fpt_simulate_noalloc: FPT_NOALLOC_MAX_TRAJ trajectories)";
    default: return "unknown error code";
  }
}

int fpt_version(void) { return 200; }

// ---- test hooks
int fpt_dbg_philox(uint64_t seed, uint64_t id0, int64_t n_ids, uint64_t block, uint32_t* out, void* s) {
  if (!out || n_ids < 0) return FPT_E_INVALID;
  if (n_ids == 0) return FPT_OK;
  dbg_philox_kernel<<<grid_for(n_ids, 128), 128, 0, (cudaStream_t)s>>>(philox_round_keys(seed), id0, n_ids, block, out);
  FPT_CUDA(cudaGetLastError());
  return FPT_OK;
}
int fpt_dbg_normals_f64(uint64_t seed, uint64_t id, uint64_t b0, int64_t nblocks, double* out, void* s) {
  if (!out || nblocks < 0) return FPT_E_INVALID;
  if (nblocks == 0) return FPT_OK;
  dbg_normals64_kernel<<<grid_for(nblocks, 128), 128, 0, (cudaStream_t)s>>>(philox_round_keys(seed), id, b0, nblocks, out);
  FPT_CUDA(cudaGetLastError());
  return FPT_OK;
}
int fpt_dbg_normals_f32(uint64_t seed, uint64_t id, uint64_t b0, int64_t nblocks, float* out, void* s) {
  if (!out || nblocks < 0) return FPT_E_INVALID;
  if (nblocks == 0) return FPT_OK;
  dbg_normals32_kernel<<<grid_for(nblocks, 128), 128, 0, (cudaStream_t)s>>>(philox_round_keys(seed), id, b0, nblocks, out);
  FPT_CUDA(cudaGetLastError());
  return FPT_OK;
}
int fpt_dbg_unary_f64(int32_t which, const double* x, double* y, int64_t n, void* s) {
  if (!x || !y || n < 0 || which < 0 || which > 1) return FPT_E_INVALID;
  if (n == 0) return FPT_OK;
  dbg_unary64_kernel<<<grid_for(n, 128), 128, 0, (cudaStream_t)s>>>(which, x, y, n);
  FPT_CUDA(cudaGetLastError());
  return FPT_OK;
}
int fpt_dbg_unary_f32(int32_t which, const float* x, float* y, int64_t n, void* s) {
  if (!x || !y || n < 0 || which < 0 || which > 1) return FPT_E_INVALID;
  if (n == 0) return FPT_OK;
  dbg_unary32_kernel<<<grid_for(n, 128), 128, 0, (cudaStream_t)s>>>(which, x, y, n);
  FPT_CUDA(cudaGetLastError());
  return FPT_OK;
}
int fpt_dbg_sincos_f64(const uint64_t* Y, double* c, double* sn, int64_t n, void* s) {
  if (!Y || !c || !sn || n < 0) return FPT_E_INVALID;
  if (n == 0) return FPT_OK;
  dbg_sincos64_kernel<<<grid_for(n, 128), 128, 0, (cudaStream_t)s>>>((const unsigned long long*)Y, c, sn, n);
  FPT_CUDA(cudaGetLastError());
  return FPT_OK;
}
int fpt_dbg_sincos_f32(const uint32_t* o, float* c, float* sn, int64_t n, void* s) {
  if (!o || !c || !sn || n < 0) return FPT_E_INVALID;
  if (n == 0) return FPT_OK;
  dbg_sincos32_kernel<<<grid_for(n, 128), 128, 0, (cudaStream_t)s>>>(o, c, sn, n);
  FPT_CUDA(cudaGetLastError());
  return FPT_OK;
}
int fpt_dbg_selfcheck(uint64_t seed, uint64_t id0, int64_t n_threads, int32_t blocks_per_thread, uint64_t* out4, void* s) {
  if (!out4 || n_threads < 0 || blocks_per_thread < 1 || (n_threads % 128) != 0) return FPT_E_INVALID;
  if (n_threads == 0) return FPT_OK;
  dbg_selfcheck_kernel<<<(int)(n_threads / 128), 128, 0, (cudaStream_t)s>>>(philox_round_keys(seed), id0, blocks_per_thread,
                                                                          (unsigned long long*)out4);
  FPT_CUDA(cudaGetLastError());
  return FPT_OK;
}
int fpt_dbg_set_helper_seq0(uint64_t seq0) {
  t_dbg_seq0 = seq0;
  return FPT_OK;
}
int fpt_dbg_set_slice_quantum(uint64_t steps) {
  if (steps != 0 && (steps & (steps - 1)) != 0) return FPT_E_INVALID;
  t_dbg_slice_q = steps;
  return FPT_OK;
}
int fpt_dbg_trace(const fpt_params* p, uint64_t seed, uint64_t id, double t_max, int64_t trace_len, double* trace_phi,
                  double* trace_v, int32_t* out_status, uint64_t* out_k_end, void* s) {
  int rc = validate(p, 0, t_max);
  if (rc != FPT_OK) return rc;
  if (trace_len < 0 || (trace_len > 0 && !trace_phi)) return FPT_E_INVALID;
  KParams P;
  derive(*p, t_max, seed, P);
  TraceArgs T{id, trace_len, trace_phi, trace_v, out_status, (unsigned long long*)out_k_end};
  // the same State specialisation as the production launch of these parameters (R15 shortcuts included)
  const bool amp = p->amp != 0.0, ramp = p->nu != 0.0;
  const void* fn = p->precision == FPT_PREC_FP32_FAST ? trace_kernel_f32_fast(p->model, ramp)
                   : p->precision == FPT_PREC_FP32    ? trace_kernel_f32(p->model, p->scheme, amp, ramp)
                                                 : trace_kernel_f64(p->model, p->scheme, amp, ramp);
  void* args[] = {(void*)&P, (void*)&T};
  FPT_CUDA(cudaLaunchKernel(fn, dim3(1), dim3(32), args, 0, (cudaStream_t)s));
  return FPT_OK;
}

}  // extern "C"

// =================================================================================================================
// fpt_simulate_noalloc (fpt.h): the persistent kernel with ALL its scratch memory in one file-scope device array, for callers
// that must not allocate (no cudaMalloc / cudaMallocAsync / cudaFree / memory-pool call on this path, ever; it does not
// touch device_ctx(), whose first call per device allocates).  The array is part of the library's image: every GPU that
// loads the library holds it (5.3 MB) until the process exits.  It is shared by all calls and keeps the last call's
// contents; what must start at zero (the counters, the ring entries this call will use) is cleared on the caller's stream
// at the start of every call.  Two calls that overlap on the GPU would share the id counter and the parking slots: they race.
namespace {

constexpr unsigned long long kNoAllocMaxTraj = FPT_NOALLOC_MAX_TRAJ;
constexpr unsigned long long kNoAllocMaxGrid = 1024;               // ceil(max n_traj / 128): never more lanes than trajectories
constexpr size_t kNoAllocHeader = 512;                             // DevStats (128 B) | fpt_stats sink (104 B) | ticket sink (8 B)
constexpr size_t kNoAllocSlotsOff = kNoAllocHeader;
constexpr size_t kNoAllocRingOff = kNoAllocSlotsOff + (size_t)kNoAllocMaxTraj * sizeof(ParkSlot);
constexpr size_t kNoAllocRingEntries = (size_t)(kNoAllocMaxTraj + kNoAllocMaxGrid);      // grid x ceil(n / grid) <= n + grid - 1
constexpr size_t kNoAllocBytes = kNoAllocRingOff + kNoAllocRingEntries * sizeof(unsigned long long);
static_assert(sizeof(DevStats) <= 128 && sizeof(fpt_stats) <= 256 - 8, "header layout");
static_assert(kNoAllocBytes < (6u << 20), "the scratch array is meant to stay modest");

static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocBytes];

struct NoAllocCtx {           // per device: the array's DEVICE address (the name above is only a host-side handle) and the SM count
  std::atomic<bool> ready{false};
  unsigned char* base = nullptr;
  int sm_count = 0;
};
NoAllocCtx g_noalloc[kMaxDevices];
std::mutex g_noalloc_mu;

int noalloc_ctx(NoAllocCtx** out) {
  int dev = 0;
  FPT_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return FPT_E_CUDA;
  NoAllocCtx& c = g_noalloc[dev];
  if (!c.ready.load(std::memory_order_acquire)) {
    std::lock_guard<std::mutex> lk(g_noalloc_mu);
    if (!c.ready.load(std::memory_order_relaxed)) {
      void* ptr = nullptr;                                          // with device `dev` current: this device's copy of the array
      FPT_CUDA(cudaGetSymbolAddress(&ptr, g_noalloc_scratch));
      if (!ptr) return FPT_E_CUDA;
      c.base = (unsigned char*)ptr;
      FPT_CUDA(cudaDeviceGetAttribute(&c.sm_count, cudaDevAttrMultiProcessorCount, dev));
      c.ready.store(true, std::memory_order_release);
    }
  }
  *out = &c;
  return FPT_OK;
}

}  // namespace

extern "C" int fpt_simulate_noalloc(const fpt_params* p, int64_t n_traj, uint64_t seed, double t_max, double* out_fpt,
                                    double* out_gamma, int32_t* out_status, fpt_stats* d_stats, void* cuda_stream) {
  int rc = validate(p, n_traj, t_max);
  if (rc != FPT_OK) return rc;
  if (n_traj > 0 && (!out_fpt || !out_status)) return FPT_E_INVALID;
  if ((unsigned long long)n_traj > kNoAllocMaxTraj) return FPT_E_TOO_LARGE;
  if (n_traj == 0) return FPT_OK;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  NoAllocCtx* ctx = nullptr;
  if ((rc = noalloc_ctx(&ctx)) != FPT_OK) return rc;
  const int sms = ctx->sm_count;

  KParams P;
  derive(*p, t_max, seed, P);
  P.n_traj = (unsigned long long)n_traj;
  P.out_fpt = out_fpt;
  P.out_gamma = out_gamma;
  P.out_status = out_status;
  DevStats* ws = (DevStats*)ctx->base;
  fpt_stats* sink = (fpt_stats*)(ctx->base + 128);
  unsigned long long* sink_ticket = (unsigned long long*)(ctx->base + 256 - 8);
  FPT_CUDA(cudaMemsetAsync(ws, 0, 128, stream));                    // id counter and statistics start at zero
  P.ws = ws;

  int grid = 1, block = 128, kernel = FPT_KERNEL_FILL;
  const bool fp32 = p->precision != FPT_PREC_FP64;
  const bool strict = p->scheme == FPT_SCHEME_PAPER;
  const bool at_once_escaped = fp32 ? (strict ? !((float)p->phi0 <= (float)p->threshold) : !((float)p->phi0 < (float)p->threshold))
                                    : (strict ? !(p->phi0 <= p->threshold) : !(p->phi0 < p->threshold));
  if (at_once_escaped || P.n_cap == 0) {
    block = 256;
    grid = (int)std::min<int64_t>((n_traj + block - 1) / block, (int64_t)sms * 8);
    const double gam = std::fma(P.dgamma, at_once_escaped ? 0.0 : (double)P.n_cap, P.gamma0);
    fpt_fill_kernel<<<grid, block, 0, stream>>>(P, at_once_escaped ? kStatusEscaped : kStatusCensored, at_once_escaped ? 0.0 : -1.0, gam);
    FPT_CUDA(cudaGetLastError());
  } else {
    const bool amp = p->amp != 0.0, ramp = p->nu != 0.0;
    const void* fn = p->precision == FPT_PREC_FP32_FAST ? persistent_kernel_f32_fast(p->model, ramp)
                     : fp32                            ? persistent_kernel_f32(p->model, p->scheme, amp, ramp)
                                                       : persistent_kernel_f64(p->model, p->scheme, amp, ramp);
    int per_sm = 0;
    FPT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, block, 0));
    if (per_sm < 1) return FPT_E_CUDA;
    // blocks of 128: all trajectories of a ramped job in flight if they fit, a fifth of a constant-bias job (as the
    // allocating path, without its refinements), at least one block per SM, never more lanes than trajectories
    const long long unit = 128LL * sms;
    long long units = ramp ? (n_traj + unit - 1) / unit : n_traj / (5 * unit);
    units = std::max<long long>(1, std::min<long long>(units, per_sm));
    const long long blocks = std::min<long long>(units * sms, (n_traj + block - 1) / block);
    grid = (int)blocks;
    kernel = FPT_KERNEL_PERSISTENT;
    // equal-length trajectories on fewer lanes: rotate them through the parking slots of the array (time slicing)
    if (ramp && (long long)grid * block < n_traj && P.n_cap >= (1ull << 15)) {
      unsigned long long q = 2048;
      while (q < (unsigned long long)P.K || q * 2048ull < P.n_cap) q <<= 1;
      if ((q % (unsigned long long)P.K) != 0ull) q *= (unsigned long long)P.K;
      const unsigned long long cap = ((unsigned long long)n_traj + (unsigned long long)grid - 1ull) / (unsigned long long)grid;
      const void* fn_s = sliced_kernel(p, amp);
      int per_sm_s = 0;
      FPT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm_s, fn_s, block, 0));
      if ((q & (q - 1ull)) == 0ull && (unsigned long long)grid * cap <= kNoAllocRingEntries && (long long)per_sm_s * sms >= (long long)grid) {
        fn = fn_s;
        P.slice_cap = cap;
        P.slice_slots = (ParkSlot*)(ctx->base + kNoAllocSlotsOff);
        P.slice_ring = (unsigned long long*)(ctx->base + kNoAllocRingOff);
        FPT_CUDA(cudaMemsetAsync(P.slice_ring, 0, (size_t)grid * (size_t)cap * sizeof(unsigned long long), stream));   // 0 = not published
        P.slice_mask = q - 1ull;
      }
    }
    P.schedule = FPT_SCHEDULE_DYNAMIC;
    P.tail_helper = 1;
    void* args[] = {(void*)&P};
    FPT_CUDA(cudaLaunchKernel(fn, dim3(grid), dim3(block), args, 0, stream));
  }
  fpt_stats geo{};
  geo.n_traj = (uint64_t)n_traj;
  geo.n_cap = P.n_cap;
  geo.grid = grid;
  geo.block = block;
  geo.check_every = P.K;
  geo.kernel = kernel;
  fpt_export_stats_kernel<<<1, 1, 0, stream>>>(ws, geo, d_stats, sink, sink_ticket, 0ull);
  FPT_CUDA(cudaGetLastError());
  return FPT_OK;
}
