/* fpt_dbg.h -- test hooks and roofline microbenchmarks of libfpt_b200 (NOT part of the product API of fpt.h).
 *
 * The device functions of the hot path, exposed one by one so that tests can compare bits with the
 * oracle, and the two pipe-peak microbenchmarks bench.py uses as roofline denominators.  All pointers are device memory
 * unless stated; work is enqueued on cuda_stream (a cudaStream_t passed as void*).  Return codes as in fpt.h.
 */
#ifndef FPT_B200_DBG_H_
#define FPT_B200_DBG_H_

#include "fpt.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Roofline denominators measured live: a kernel of independent DFMA (fp64) or FFMA (fp32) chains on every SM, run
 * repeatedly for about `seconds`; *inst_per_s = thread-instructions per second, *sm_clock_hz = SM clock seen by the
 * kernel (clock64 ticks / elapsed time; may be NULL).  Host pointers; synchronises. */
int fpt_fp64_peak(double seconds, double* inst_per_s, double* sm_clock_hz);
int fpt_fp32_peak(double seconds, double* inst_per_s, double* sm_clock_hz);

/* out[4*i..4*i+3] = Philox4x32-10 block `block` of stream (seed, id0+i) */
int fpt_dbg_philox(uint64_t seed, uint64_t id0, int64_t n_ids, uint64_t block, uint32_t* out, void* cuda_stream);
/* normals of blocks b0..b0+nblocks-1 of stream (seed, id): fp64 2 per block (z_a, z_b); fp32 4 per block */
int fpt_dbg_normals_f64(uint64_t seed, uint64_t id, uint64_t b0, int64_t nblocks, double* out, void* cuda_stream);
int fpt_dbg_normals_f32(uint64_t seed, uint64_t id, uint64_t b0, int64_t nblocks, float* out, void* cuda_stream);
/* elementwise: which = 0 sin_drift(x), 1 neg2log(x) (x in (0,1)) */
int fpt_dbg_unary_f64(int32_t which, const double* x, double* y, int64_t n, void* cuda_stream);
int fpt_dbg_unary_f32(int32_t which, const float* x, float* y, int64_t n, void* cuda_stream);
/* cos, sin of the Box-Muller angle from the raw 64-bit (fp64) / 32-bit (fp32) word */
int fpt_dbg_sincos_f64(const uint64_t* Y, double* c, double* s, int64_t n, void* cuda_stream);
int fpt_dbg_sincos_f32(const uint32_t* o, float* c, float* s, int64_t n, void* cuda_stream);
/* the guard-free division / square-root sequences of csrc/fpt_math.cuh against nvcc's IEEE builtins, on operands drawn
 * from the real pipeline (n_threads streams, a multiple of 128, x blocks_per_thread Philox blocks each):
 * out4[0..3] += number of bit mismatches {fp64 div, fp64 sqrt, fp32 div, fp32 sqrt} (device, uint64, caller zeroes). */
int fpt_dbg_selfcheck(uint64_t seed, uint64_t id0, int64_t n_threads, int32_t blocks_per_thread, uint64_t* out4,
                      void* cuda_stream);
/* First value of the tail helper's hand-over sequence counters for the calls the CALLING THREAD makes afterwards (0 = the
 * product's value).  The counters are 64-bit; a test presets them just below 2^32 to run across the point where 32-bit
 * counters would wrap. */
int fpt_dbg_set_helper_seq0(uint64_t seq0);
/* Quantum of the time slicing (fpt_launch_opts.time_slice) for the calls the CALLING THREAD makes afterwards: a power of
 * two of steps (it is raised to the call's poll interval K when smaller), 0 = the product's value (>= 2048).  A test
 * sets 64 to drive thousands of hand-overs through a small job.  FPT_E_INVALID when not 0 or a power of two. */
int fpt_dbg_set_slice_quantum(uint64_t steps);
/* one trajectory (id) with its states recorded: trace_phi[k], trace_v[k] for k = 0..min(k_end, trace_len-1) (as double),
 * out_status[0], out_k_end[0]; entries past k_end are left untouched. */
int fpt_dbg_trace(const fpt_params* p, uint64_t seed, uint64_t id, double t_max, int64_t trace_len,
                  double* trace_phi, double* trace_v, int32_t* out_status, uint64_t* out_k_end, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* FPT_B200_DBG_H_ */
