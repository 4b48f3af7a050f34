// fpt_oracle.cpp -- the ORACLE: a plain, slow, one-trajectory-at-a-time CPU integrator.
//
// THIS IS TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no
// code, header, table or constant generator with the CUDA path under paper_1802_05065_b200/;
// the two meet only in the written definition DESIGN.md section 4 ("MATH SPEC").
//
// What it computes (citations: PAPER.md = /root/reference/PAPER.md, arXiv:1802.05065):
//   * Alg. 1 ESCAPETIME and Alg. 3 SWITCHINGCURRENT: one
//     realisation of the noisy washboard Langevin equation, Eq. (9)-(11), is
//     integrated step by step until phi first reaches a threshold ("checking at each time step
//     if a threshold crossing ... has occurred"); the escape time k*h
//     or the bias at escape gamma_k is stored per run; -1 marks a run that hit the
//     step cap.
//   * nrand(): Box-Muller normals from uniform deviates.
//   * BASELINE.json north_star overrides the paper on: Philox4x32-10 keyed by (seed, trajectory id)
//     instead of the per-thread Mersenne Twister, stochastic Heun beside Euler,
//     the overdamped limit, fp64 first with an fp32 + Kahan-compensated-time variant.
//   Every reading of a silent/garbled passage is DESIGN.md section 3 (R1..R13).
//
// Arithmetic contract: only +, -, *, fma, IEEE sqrt, IEEE /, integer ops.
// Compile with -ffp-contract=off -fno-fast-math so the ONLY fused operations are the explicit
// std::fma calls below.  No blocking, no vectorisation, no reordering: a reader can check each
// function against the passage it cites by eye.
//
// Parity pins (tests/, -m "not gpu"): Philox known answers; each transcendental against mpmath;
// normal moments/KS; inverse-Gaussian FPT law (config 1); deterministic escape at gamma>1; exact
// MFPT quadrature / Kramers scaling; brute-force enumeration with injected +-1 noise; 50-digit
// mpmath recomputation of whole short paths; SURVEY.md P10 worked examples.  Nothing here is
// "parity unpinned"; the *distribution* of the underdamped noisy configs (2-4) is pinned only
// statistically (equipartition, Smoluchowski limit, an independent numpy sample) -- DESIGN.md 5.

#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ---------------------------------------------------------------------------------------------
// bit casts
inline double   f64_from_bits(uint64_t b) { double d; std::memcpy(&d, &b, 8); return d; }
inline uint64_t bits_from_f64(double d)   { uint64_t b; std::memcpy(&b, &d, 8); return b; }
inline float    f32_from_bits(uint32_t b) { float f; std::memcpy(&f, &b, 4); return f; }
inline uint32_t bits_from_f32(float f)    { uint32_t b; std::memcpy(&b, &f, 4); return b; }

// ---------------------------------------------------------------------------------------------
// O1. Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11; mandated by BASELINE.json north_star in
// place of PAPER.md Alg. 2).  One round on counter (c0,c1,c2,c3) and key (k0,k1):
//   (c0,c1,c2,c3) <- ( hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0) )
// ten rounds, the key bumped by the Weyl constants (W0,W1) between rounds.
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    const uint64_t p0 = (uint64_t)M0 * (uint64_t)c0;
    const uint64_t p1 = (uint64_t)M1 * (uint64_t)c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    const uint32_t n1 = (uint32_t)p1;
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    const uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += W0; k1 += W1;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Keying (reading R1): key = (seed lo, seed hi); counter = (block lo, block hi, id lo, id hi).
void philox_block(uint64_t seed, uint64_t id, uint64_t block, uint32_t out[4]) {
  const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  const uint32_t ctr[4] = {(uint32_t)block, (uint32_t)(block >> 32), (uint32_t)id, (uint32_t)(id >> 32)};
  philox4x32_10(ctr, key, out);
}

// ---------------------------------------------------------------------------------------------
// O4 (fp64). Constants: every one is a closed form rounded to nearest double.
const double INV_PI = 0x1.45f306dc9c883p-2;    // RN(1/pi)
const double PI_HI  = 0x1.921fb54442d18p+1;    // RN(pi)
const double PI_LO  = 0x1.1a62633145c07p-53;   // RN(pi - PI_HI)
const double MAGIC  = 0x1.8p+52;               // 1.5 * 2^52
// SIN_C[j] = RN((-1)^j / (2j+1)!), j = 1..10  (Taylor coefficients of sin, r^3 .. r^21)
const double SIN_C[11] = {
    1.0,
    -0x1.5555555555555p-3,  0x1.1111111111111p-7,  -0x1.a01a01a01a01ap-13, 0x1.71de3a556c734p-19,
    -0x1.ae64567f544e4p-26, 0x1.6124613a86d09p-33, -0x1.ae7f3e733b81fp-41, 0x1.952c77030ad4ap-49,
    -0x1.2f49b46814157p-57, 0x1.71b8ef6dcf572p-66};
// COS_C[j] = RN((-1)^j / (2j)!), j = 1..8  (x^2 .. x^16)
const double COS_C[9] = {
    1.0,
    -0x1.0000000000000p-1,  0x1.5555555555555p-5,  -0x1.6c16c16c16c17p-10, 0x1.a01a01a01a01ap-16,
    -0x1.27e4fb7789f5cp-22, 0x1.1eed8eff8d898p-29, -0x1.93974a8c07c9dp-37, 0x1.ae7f3e733b81fp-45};
// LOG_C[j] = RN(-4 / (2j+1)), j = 0..10 : -2 ln m = -4 atanh(s) = s * sum_j LOG_C[j] s^(2j)
const double LOG_C[11] = {
    -0x1.0000000000000p+2, -0x1.5555555555555p+0, -0x1.999999999999ap-1, -0x1.2492492492492p-1,
    -0x1.c71c71c71c71cp-2, -0x1.745d1745d1746p-2, -0x1.3b13b13b13b14p-2, -0x1.1111111111111p-2,
    -0x1.e1e1e1e1e1e1ep-3, -0x1.af286bca1af28p-3, -0x1.8618618618618p-3};
const double M2LN2_HI = -0x1.62e42fefa39efp+0;  // RN(-2 ln 2)
const double M2LN2_LO = -0x1.abc9e3b39803fp-55; // RN(-2 ln 2 - M2LN2_HI)
const double TWO_PI_S = 0x1.921fb54442d18p-51;  // RN(2 pi) * 2^-53 (exact scaling)

// sin(phi) for the drift term -sin(phi) of Eq. (9) (Alg. 1 line 12 PAPER.md:164).
// n = rint(phi/pi) by the magic-add; r = phi - n*pi in two fma; odd Taylor polynomial to r^21;
// sign flipped when n is odd.
double sin_drift(double phi) {
  const double t = std::fma(phi, INV_PI, MAGIC);
  const double n = t - MAGIC;
  double r = std::fma(-n, PI_HI, phi);
  r = std::fma(-n, PI_LO, r);
  const double z = r * r;
  double p = SIN_C[10];
  for (int j = 9; j >= 1; --j) p = std::fma(p, z, SIN_C[j]);
  const double rz = r * z;
  double res = std::fma(rz, p, r);
  if (bits_from_f64(t) & 1ull) res = f64_from_bits(bits_from_f64(res) ^ 0x8000000000000000ull);
  return res;
}

// O2: u1 = (2*(X>>12)+1) * 2^-53, built without an int->fp conversion.
double uniform_open(uint64_t X) {
  const double d = f64_from_bits(0x3FF0000000000000ull | (X >> 12));  // in [1,2)
  return (d - 1.0) + 0x1p-53;                                          // both operations exact
}

// w = -2 ln(u) for u in (0,1): exponent/mantissa split with m in [1/sqrt2, sqrt2),
// s = (m-1)/(m+1), -2 ln m = s * P(s^2), w = e*(-2 ln2) + (-2 ln m).
double neg2log(double u) {
  const uint64_t ub = bits_from_f64(u);
  const uint32_t hi = (uint32_t)(ub >> 32), lo = (uint32_t)ub;
  const uint32_t hi2 = hi + (0x3FF00000u - 0x3FE6A09Eu);
  const int e = (int)(hi2 >> 20) - 1023;
  const uint32_t mhi = (hi2 & 0x000FFFFFu) + 0x3FE6A09Eu;
  const double m = f64_from_bits(((uint64_t)mhi << 32) | lo);
  const double a = m - 1.0;
  const double b = m + 1.0;
  const double s = a / b;
  const double z = s * s;
  double p = LOG_C[10];
  for (int j = 9; j >= 0; --j) p = std::fma(p, z, LOG_C[j]);
  const double wm = s * p;
  const double ed = (double)e;
  return std::fma(ed, M2LN2_HI, std::fma(ed, M2LN2_LO, wm));
}

// cos and sin of the angle 2*pi*f, f = (Y>>11) * 2^-53 turns: nearest quarter turn q and signed
// remainder rho in integer arithmetic (exact), x = rho * 2pi*2^-53 in [-pi/4, pi/4].
void sincos_turns(uint64_t Y, double* c, double* s) {
  const uint64_t A = (Y >> 11) + (1ull << 50);
  const unsigned q = (unsigned)(A >> 51) & 3u;
  const uint64_t low = A & ((1ull << 51) - 1ull);
  const double d = f64_from_bits(0x4330000000000000ull | low);  // 2^52 + low
  const double rho = d - (0x1p52 + 0x1p50);                     // low - 2^50, exact
  const double x = rho * TWO_PI_S;
  const double z = x * x;
  double ps = SIN_C[8];
  for (int j = 7; j >= 1; --j) ps = std::fma(ps, z, SIN_C[j]);
  const double xz = x * z;
  const double sx = std::fma(xz, ps, x);
  double pc = COS_C[8];
  for (int j = 7; j >= 1; --j) pc = std::fma(pc, z, COS_C[j]);
  const double cx = std::fma(z, pc, 1.0);
  switch (q) {
    case 0: *c = cx;  *s = sx;  break;
    case 1: *c = -sx; *s = cx;  break;
    case 2: *c = -cx; *s = -sx; break;
    default: *c = sx; *s = -cx; break;
  }
}

// O3. Box-Muller: r = sqrt(-2 ln u1), (z_a, z_b) = r (cos, sin)(2 pi f).
void normal_pair(const uint32_t o[4], double* za, double* zb, double* u1_out, double* f_out) {
  const uint64_t X = ((uint64_t)o[0] << 32) | o[1];
  const uint64_t Y = ((uint64_t)o[2] << 32) | o[3];
  const double u1 = uniform_open(X);
  const double r = std::sqrt(neg2log(u1));
  double c, s;
  sincos_turns(Y, &c, &s);
  *za = r * c;
  *zb = r * s;
  if (u1_out) *u1_out = u1;
  if (f_out) *f_out = (double)(Y >> 11) * 0x1p-53;
}

// ---------------------------------------------------------------------------------------------
// O10 (fp32 variant). Same shapes in float.
const float INV_PI_F = 0x1.45f306p-2f;
const float PI_HI_F  = 0x1.921fb6p+1f;
const float PI_LO_F  = -0x1.777a5cp-24f;
const float MAGIC_F  = 0x1.8p+23f;
const float SIN_CF[7] = {1.0f, -0x1.555556p-3f, 0x1.111112p-7f, -0x1.a01a02p-13f, 0x1.71de3ap-19f,
                         -0x1.ae6456p-26f, 0x1.612462p-33f};
const float COS_CF[6] = {1.0f, -0x1.0p-1f, 0x1.555556p-5f, -0x1.6c16c2p-10f, 0x1.a01a02p-16f, -0x1.27e4fcp-22f};
const float LOG_CF[5] = {-0x1.0p+2f, -0x1.555556p+0f, -0x1.99999ap-1f, -0x1.24924ap-1f, -0x1.c71c72p-2f};
const float M2LN2_HI_F = -0x1.62e43p+0f;
const float M2LN2_LO_F = 0x1.05c61p-28f;
const float TWO_PI_SF  = 0x1.921fb6p-30f;  // RN_f(2 pi) * 2^-32

float sin_drift_f(float phi) {   // odd Taylor polynomial to r^13
  const float t = std::fmaf(phi, INV_PI_F, MAGIC_F);
  const float n = t - MAGIC_F;
  float r = std::fmaf(-n, PI_HI_F, phi);
  r = std::fmaf(-n, PI_LO_F, r);
  const float z = r * r;
  float p = SIN_CF[6];
  for (int j = 5; j >= 1; --j) p = std::fmaf(p, z, SIN_CF[j]);
  const float rz = r * z;
  float res = std::fmaf(rz, p, r);
  if (bits_from_f32(t) & 1u) res = f32_from_bits(bits_from_f32(res) ^ 0x80000000u);
  return res;
}

float uniform_open_f(uint32_t o) {   // one IEEE int->float rounding, then an exact-scale fma
  return std::fmaf((float)o, 0x1p-32f, 0x1p-33f);
}

float neg2log_f(float u) {
  const uint32_t ix = bits_from_f32(u);
  const uint32_t ix2 = ix + (0x3f800000u - 0x3f3504f3u);
  const int e = (int)(ix2 >> 23) - 127;
  const float m = f32_from_bits((ix2 & 0x007fffffu) + 0x3f3504f3u);
  const float a = m - 1.0f;
  const float b = m + 1.0f;
  const float s = a / b;
  const float z = s * s;
  float p = LOG_CF[4];
  for (int j = 3; j >= 0; --j) p = std::fmaf(p, z, LOG_CF[j]);
  const float wm = s * p;
  const float ed = (float)e;
  return std::fmaf(ed, M2LN2_HI_F, std::fmaf(ed, M2LN2_LO_F, wm));
}

void sincos_turns_f(uint32_t o, float* c, float* s) {   // sin to x^9, cos to x^10
  const uint32_t A = o + (1u << 29);                    // wraps mod 2^32 == quarter turns mod 4
  const unsigned q = A >> 30;
  const int32_t rho_i = (int32_t)(A & ((1u << 30) - 1u)) - (int32_t)(1 << 29);
  const float rho = (float)rho_i;                       // one IEEE rounding
  const float x = rho * TWO_PI_SF;
  const float z = x * x;
  float ps = SIN_CF[4];
  for (int j = 3; j >= 1; --j) ps = std::fmaf(ps, z, SIN_CF[j]);
  const float xz = x * z;
  const float sx = std::fmaf(xz, ps, x);
  float pc = COS_CF[5];
  for (int j = 4; j >= 1; --j) pc = std::fmaf(pc, z, COS_CF[j]);
  const float cx = std::fmaf(z, pc, 1.0f);
  switch (q) {
    case 0: *c = cx;  *s = sx;  break;
    case 1: *c = -sx; *s = cx;  break;
    case 2: *c = -cx; *s = -sx; break;
    default: *c = sx; *s = -cx; break;
  }
}

// one Philox block -> two Box-Muller pairs -> four normals (cosA, sinA, cosB, sinB)
void normal_quad_f(const uint32_t o[4], float z[4]) {
  for (int h = 0; h < 2; ++h) {
    const float u1 = uniform_open_f(o[2 * h]);
    const float r = std::sqrt(neg2log_f(u1));
    float c, s;
    sincos_turns_f(o[2 * h + 1], &c, &s);
    z[2 * h] = r * c;
    z[2 * h + 1] = r * s;
  }
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// The parameter block of one simulation (the oracle's own declaration; the CUDA library has its own).
extern "C" {

struct oracle_params {
  int32_t model;        // 0 overdamped: dphi = (gamma(t) - amp sin phi) dt + sqrt(2 temperature) dW
                        // 1 underdamped: phi'' + alpha phi' + amp sin phi = gamma(t) + sqrt(2 alpha temperature) xi
  int32_t scheme;       // 0 Euler-Maruyama (paper's Euler), 1 stochastic Heun,
                        // 2 the paper's kernels AS PRINTED (Alg. 1 / Alg. 3): Euler with the bias
                        //   gamma_k = gamma0 + dgamma*k taken BEFORE the step (Alg. 3 line 13 precedes lines 14-15) and the
                        //   strict comparison phi_k > th (Alg. 1 line 12, Alg. 3 line 16); reading R17
  int32_t precision;    // 0 fp64 state, 1 fp32 state + Kahan-compensated time
  int32_t reserved;
  double alpha, temperature, amp, gamma0, nu, phi0, v0, threshold, dt;
  uint64_t first_id;
};

}  // extern "C"

namespace {

struct derived {          // O5: host-side derived constants, fp64
  double sigma, dgamma, h2;
  uint64_t n_cap;
};

derived derive(const oracle_params& p, double t_max) {
  derived d;
  if (p.model == 1) d.sigma = std::sqrt(2.0 * p.alpha * p.temperature * p.dt);   // sigma = sqrt(2 D h), D = beta*theta
  else              d.sigma = std::sqrt(2.0 * p.temperature * p.dt);
  d.dgamma = p.nu * p.dt;                                                        // delta-gamma per step
  d.h2 = 0.5 * p.dt;
  d.n_cap = (uint64_t)std::nearbyint(t_max / p.dt);                               // klim, reading R8
  return d;
}

struct normal_source {    // Philox stream of one trajectory, or an injected array (test hook, pin P6)
  uint64_t seed, id;
  const double* injected;   // nullptr -> Philox
  uint64_t n_injected;
  double za, zb;
  float zq[4];
  // normal for step k (1-based), fp64: block (k-1) div 2, cos-branch for odd k, sin-branch for even k (R4)
  double next64(uint64_t k) {
    if (injected) return (k - 1 < n_injected) ? injected[k - 1] : 0.0;
    if (((k - 1) & 1ull) == 0) {
      uint32_t o[4];
      philox_block(seed, id, (k - 1) >> 1, o);
      normal_pair(o, &za, &zb, nullptr, nullptr);
      return za;
    }
    return zb;
  }
  // fp32: block (k-1) div 4, normals (cosA, sinA, cosB, sinB) for steps 4b+1..4b+4 (O10)
  float next32(uint64_t k) {
    if (injected) return (k - 1 < n_injected) ? (float)injected[k - 1] : 0.0f;
    const unsigned j = (unsigned)((k - 1) & 3ull);
    if (j == 0) {
      uint32_t o[4];
      philox_block(seed, id, (k - 1) >> 2, o);
      normal_quad_f(o, zq);
    }
    return zq[j];
  }
};

// result of one trajectory
struct traj_result {
  int32_t status;       // 0 escaped, 1 censored, 2 state became NaN
  uint64_t k_end;       // k_esc if escaped, n_cap if censored, the step at which phi became NaN for status 2
  double phi_end, v_end;
};

// O6-O8, fp64 state.  gamma_j = fma(dgamma, (double) j, gamma0) (reading R11: gamma_{k-1} at the start
// of step k, gamma_k in Heun's second stage);  F(phi, j) = fma(-amp, sin(phi), gamma_j), and
// F = gamma_j without evaluating sin when amp == 0; gamma_j = gamma0 when nu == 0.
traj_result run_f64(const oracle_params& p, const derived& d, normal_source& ns,
                    uint64_t trace_len, double* trace_phi, double* trace_v) {
  const double A = p.amp, alpha = p.alpha, dt = p.dt, sigma = d.sigma, h2 = d.h2, thr = p.threshold;
  auto gamma_at = [&](uint64_t j) { return (p.nu == 0.0) ? p.gamma0 : std::fma(d.dgamma, (double)j, p.gamma0); };
  auto F = [&](double phi, uint64_t j) { return (A == 0.0) ? gamma_at(j) : std::fma(-A, sin_drift(phi), gamma_at(j)); };
  double phi = p.phi0, v = p.v0;
  traj_result res{1, d.n_cap, phi, v};
  if (trace_len > 0) { trace_phi[0] = phi; if (trace_v) trace_v[0] = v; }
  if (phi != phi) { res.status = 2; res.k_end = 0; return res; }
  // scheme 2 compares strictly (paper: "if phi_k > th"); schemes 0 and 1 with >= (reading R7)
  auto crossed = [&](double x) { return p.scheme == 2 ? (x > thr) : (x >= thr); };
  if (crossed(phi)) { res.status = 0; res.k_end = 0; return res; }         // O7: check at k = 0
  for (uint64_t k = 1; k <= d.n_cap; ++k) {
    const double z = ns.next64(k);
    if (p.scheme == 2) {                   // the paper's Euler as printed: gamma_k, not gamma_{k-1}, in step k
      if (p.model == 0) {
        const double f = F(phi, k);
        phi = std::fma(sigma, z, std::fma(f, dt, phi));
      } else {                             // Alg. 3 lines 13-15 (Alg. 1 lines 11-12 when dgamma = 0): both from the OLD state
        const double a = std::fma(-alpha, v, F(phi, k));
        const double phin = std::fma(v, dt, phi);
        const double vn = std::fma(sigma, z, std::fma(a, dt, v));
        phi = phin; v = vn;
      }
    } else if (p.model == 0) {
      if (p.scheme == 0) {                 // Euler-Maruyama, overdamped
        const double f = F(phi, k - 1);
        phi = std::fma(sigma, z, std::fma(f, dt, phi));
      } else {                             // stochastic Heun, overdamped (additive noise, same z in both stages)
        const double f1 = F(phi, k - 1);
        const double phip = std::fma(sigma, z, std::fma(f1, dt, phi));
        const double f2 = F(phip, k);
        phi = std::fma(sigma, z, std::fma(h2, f1 + f2, phi));
      }
    } else {
      if (p.scheme == 0) {                 // paper's Euler, Alg. 1 lines 11-12: both updates from the OLD state
        const double a = std::fma(-alpha, v, F(phi, k - 1));
        const double phin = std::fma(v, dt, phi);
        const double vn = std::fma(sigma, z, std::fma(a, dt, v));
        phi = phin; v = vn;
      } else {                             // stochastic Heun, underdamped
        const double a1 = std::fma(-alpha, v, F(phi, k - 1));
        const double phip = std::fma(v, dt, phi);
        const double vp = std::fma(sigma, z, std::fma(a1, dt, v));
        const double a2 = std::fma(-alpha, vp, F(phip, k));
        const double phin = std::fma(h2, v + vp, phi);
        const double vn = std::fma(sigma, z, std::fma(h2, a1 + a2, v));
        phi = phin; v = vn;
      }
    }
    if (k < trace_len) { trace_phi[k] = phi; if (trace_v) trace_v[k] = v; }
    if (phi != phi) { res.status = 2; res.k_end = k; break; }
    if (crossed(phi)) { res.status = 0; res.k_end = k; break; }            // O7: first k with phi_k >= threshold (> for scheme 2)
  }
  res.phi_end = phi; res.v_end = v;
  return res;
}

// O10: fp32 state, Kahan-compensated time (t, c); gamma for a stage = fmaf(nu_f, t, gamma0_f) with the t
// before (stage 1) / after (stage 2) the Kahan update; gamma = gamma0_f when nu == 0.
traj_result run_f32(const oracle_params& p, const derived& d, normal_source& ns,
                    uint64_t trace_len, double* trace_phi, double* trace_v) {
  const float A = (float)p.amp, alpha = (float)p.alpha, dt = (float)p.dt, sigma = (float)d.sigma,
              h2 = (float)d.h2, thr = (float)p.threshold, g0 = (float)p.gamma0, nu = (float)p.nu;
  const bool ramp = (p.nu != 0.0);
  auto F = [&](float phi, float g) { return (p.amp == 0.0) ? g : std::fmaf(-A, sin_drift_f(phi), g); };
  float phi = (float)p.phi0, v = (float)p.v0;
  float t = 0.0f, c = 0.0f;
  traj_result res{1, d.n_cap, phi, v};
  if (trace_len > 0) { trace_phi[0] = phi; if (trace_v) trace_v[0] = v; }
  if (phi != phi) { res.status = 2; res.k_end = 0; return res; }
  auto crossed = [&](float x) { return p.scheme == 2 ? (x > thr) : (x >= thr); };
  if (crossed(phi)) { res.status = 0; res.k_end = 0; return res; }
  for (uint64_t k = 1; k <= d.n_cap; ++k) {
    const float z = ns.next32(k);
    const float g1 = ramp ? std::fmaf(nu, t, g0) : g0;
    {                                       // Kahan step: t <- t + dt
      const float y = dt - c;
      const float s = t + y;
      c = (s - t) - y;
      t = s;
    }
    const float g2 = ramp ? std::fmaf(nu, t, g0) : g0;
    if (p.scheme == 2) {                   // the paper's Euler as printed: the bias AFTER the time update (gamma_k)
      if (p.model == 0) {
        const float f = F(phi, g2);
        phi = std::fmaf(sigma, z, std::fmaf(f, dt, phi));
      } else {
        const float a = std::fmaf(-alpha, v, F(phi, g2));
        const float phin = std::fmaf(v, dt, phi);
        const float vn = std::fmaf(sigma, z, std::fmaf(a, dt, v));
        phi = phin; v = vn;
      }
    } else if (p.model == 0) {
      if (p.scheme == 0) {
        const float f = F(phi, g1);
        phi = std::fmaf(sigma, z, std::fmaf(f, dt, phi));
      } else {
        const float f1 = F(phi, g1);
        const float phip = std::fmaf(sigma, z, std::fmaf(f1, dt, phi));
        const float f2 = F(phip, g2);
        phi = std::fmaf(sigma, z, std::fmaf(h2, f1 + f2, phi));
      }
    } else {
      if (p.scheme == 0) {
        const float a = std::fmaf(-alpha, v, F(phi, g1));
        const float phin = std::fmaf(v, dt, phi);
        const float vn = std::fmaf(sigma, z, std::fmaf(a, dt, v));
        phi = phin; v = vn;
      } else {
        const float a1 = std::fmaf(-alpha, v, F(phi, g1));
        const float phip = std::fmaf(v, dt, phi);
        const float vp = std::fmaf(sigma, z, std::fmaf(a1, dt, v));
        const float a2 = std::fmaf(-alpha, vp, F(phip, g2));
        const float phin = std::fmaf(h2, v + vp, phi);
        const float vn = std::fmaf(sigma, z, std::fmaf(h2, a1 + a2, v));
        phi = phin; v = vn;
      }
    }
    if (k < trace_len) { trace_phi[k] = phi; if (trace_v) trace_v[k] = v; }
    if (phi != phi) { res.status = 2; res.k_end = k; break; }
    if (crossed(phi)) { res.status = 0; res.k_end = k; break; }
  }
  res.phi_end = phi; res.v_end = v;
  return res;
}

bool params_ok(const oracle_params* p, double t_max) {
  if (!p) return false;
  if (p->model < 0 || p->model > 1 || p->scheme < 0 || p->scheme > 2 || p->precision < 0 || p->precision > 1) return false;
  const double f[] = {p->alpha, p->temperature, p->amp, p->gamma0, p->nu, p->phi0, p->v0, p->threshold, p->dt, t_max};
  for (double x : f) if (!std::isfinite(x)) return false;
  if (!(p->dt > 0.0) || !(t_max > 0.0) || p->temperature < 0.0) return false;
  if (p->model == 1 && p->alpha < 0.0) return false;
  if (!(t_max / p->dt < 0x1p53)) return false;
  return true;
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// C entry points (loaded with ctypes by oracle/__init__.py)
extern "C" {

void oracle_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }
void oracle_philox_block(uint64_t seed, uint64_t id, uint64_t block, uint32_t* out) { philox_block(seed, id, block, out); }

double oracle_sin_drift(double x) { return sin_drift(x); }
double oracle_uniform_open(uint64_t X) { return uniform_open(X); }
double oracle_neg2log(double u) { return neg2log(u); }
void oracle_sincos_turns(uint64_t Y, double* c, double* s) { sincos_turns(Y, c, s); }
float oracle_sin_drift_f(float x) { return sin_drift_f(x); }
float oracle_uniform_open_f(uint32_t o) { return uniform_open_f(o); }
float oracle_neg2log_f(float u) { return neg2log_f(u); }
void oracle_sincos_turns_f(uint32_t o, float* c, float* s) { sincos_turns_f(o, c, s); }

// vectorised conveniences for the accuracy pins
void oracle_sin_drift_v(const double* x, double* y, int64_t n) { for (int64_t i = 0; i < n; ++i) y[i] = sin_drift(x[i]); }
void oracle_neg2log_v(const double* x, double* y, int64_t n) { for (int64_t i = 0; i < n; ++i) y[i] = neg2log(x[i]); }
void oracle_sincos_turns_v(const uint64_t* Y, double* c, double* s, int64_t n) { for (int64_t i = 0; i < n; ++i) sincos_turns(Y[i], c + i, s + i); }
void oracle_sin_drift_fv(const float* x, float* y, int64_t n) { for (int64_t i = 0; i < n; ++i) y[i] = sin_drift_f(x[i]); }
void oracle_neg2log_fv(const float* x, float* y, int64_t n) { for (int64_t i = 0; i < n; ++i) y[i] = neg2log_f(x[i]); }
void oracle_sincos_turns_fv(const uint32_t* o, float* c, float* s, int64_t n) { for (int64_t i = 0; i < n; ++i) sincos_turns_f(o[i], c + i, s + i); }

// normals of blocks b0 .. b0+nblocks-1 of stream (seed, id): fp64 -> 2 per block (z_a, z_b), plus optional u1, f
void oracle_normals_f64(uint64_t seed, uint64_t id, uint64_t b0, int64_t nblocks, double* z, double* u1, double* f) {
  for (int64_t i = 0; i < nblocks; ++i) {
    uint32_t o[4];
    philox_block(seed, id, b0 + (uint64_t)i, o);
    normal_pair(o, z + 2 * i, z + 2 * i + 1, u1 ? u1 + i : nullptr, f ? f + i : nullptr);
  }
}
// fp32 -> 4 per block
void oracle_normals_f32(uint64_t seed, uint64_t id, uint64_t b0, int64_t nblocks, float* z) {
  for (int64_t i = 0; i < nblocks; ++i) {
    uint32_t o[4];
    philox_block(seed, id, b0 + (uint64_t)i, o);
    normal_quad_f(o, z + 4 * i);
  }
}
// first normal pair of many ids (block 0) -- bulk statistics
void oracle_normals_ids_f64(uint64_t seed, uint64_t id0, int64_t nids, uint64_t block, double* z) {
  for (int64_t i = 0; i < nids; ++i) {
    uint32_t o[4];
    philox_block(seed, id0 + (uint64_t)i, block, o);
    normal_pair(o, z + 2 * i, z + 2 * i + 1, nullptr, nullptr);
  }
}

uint64_t oracle_n_cap(const oracle_params* p, double t_max) { return params_ok(p, t_max) ? derive(*p, t_max).n_cap : 0; }

// Simulate trajectories id = first_id .. first_id + n_traj - 1.  Outputs follow DESIGN.md 2 (boundary):
//   out_status 0 escaped / 1 censored / 2 NaN state;  out_fpt = k_esc*dt, -1 if censored, NaN if status 2;
//   out_gamma  = fma(nu*dt, (double)k_end, gamma0) (k_end = n_cap when censored), NaN if status 2;
//   out_k (optional) = k_end;  out_phi_end / out_v_end (optional) = state at k_end (test hook for Wald's identity).
// nthreads: 1 = single thread; 0 = all cores (OpenMP over trajectories -- the reported CPU baseline).
// returns 0, or -1 on invalid parameters (nothing written).
int oracle_simulate(const oracle_params* p, int64_t n_traj, uint64_t seed, double t_max,
                    double* out_fpt, double* out_gamma, int32_t* out_status,
                    uint64_t* out_k, double* out_phi_end, double* out_v_end, int nthreads) {
  if (!params_ok(p, t_max) || n_traj < 0) return -1;
  const derived d = derive(*p, t_max);
  const double nan = std::numeric_limits<double>::quiet_NaN();
#ifdef _OPENMP
  const int nt = nthreads > 0 ? nthreads : omp_get_max_threads();
#pragma omp parallel for schedule(dynamic, 8) num_threads(nt)
#endif
  for (int64_t i = 0; i < n_traj; ++i) {
    normal_source ns{seed, p->first_id + (uint64_t)i, nullptr, 0, 0.0, 0.0, {0, 0, 0, 0}};
    const traj_result r = (p->precision == 0) ? run_f64(*p, d, ns, 0, nullptr, nullptr)
                                              : run_f32(*p, d, ns, 0, nullptr, nullptr);
    if (out_status) out_status[i] = r.status;
    const double g = std::fma(d.dgamma, (double)r.k_end, p->gamma0);
    if (out_fpt) out_fpt[i] = r.status == 0 ? (double)r.k_end * p->dt : (r.status == 1 ? -1.0 : nan);
    if (out_gamma) out_gamma[i] = r.status == 2 ? nan : g;
    if (out_k) out_k[i] = r.k_end;
    if (out_phi_end) out_phi_end[i] = r.phi_end;
    if (out_v_end) out_v_end[i] = r.v_end;
  }
  return 0;
}

// One trajectory with its states recorded: trace_phi[k], trace_v[k] for k = 0 .. min(k_end, trace_len-1).
// normals == nullptr: Philox stream (seed, id); else step k uses normals[k-1] (0 beyond n_normals) -- pin P6.
int oracle_trace(const oracle_params* p, uint64_t seed, uint64_t id, double t_max,
                 const double* normals, uint64_t n_normals,
                 uint64_t trace_len, double* trace_phi, double* trace_v,
                 int32_t* status, uint64_t* k_end) {
  if (!params_ok(p, t_max)) return -1;
  const derived d = derive(*p, t_max);
  normal_source ns{seed, id, normals, n_normals, 0.0, 0.0, {0, 0, 0, 0}};
  const traj_result r = (p->precision == 0) ? run_f64(*p, d, ns, trace_len, trace_phi, trace_v)
                                            : run_f32(*p, d, ns, trace_len, trace_phi, trace_v);
  if (status) *status = r.status;
  if (k_end) *k_end = r.k_end;
  return 0;
}

// O9. Histogram of values[i] over status[i]==0 (status may be null: all counted):
// b = floor((x-lo) * (nbins/(hi-lo))); b<0 -> counts[0] (under), b>=nbins -> counts[nbins+1] (over, so x==hi is "over"),
// else counts[1+b].  Accumulates into counts (caller zeroes).
int oracle_histogram(const double* values, const int32_t* status, int64_t n, double lo, double hi, int32_t nbins,
                     uint64_t* counts) {
  if (nbins < 1 || !(hi > lo) || n < 0) return -1;
  const double scale = (double)nbins / (hi - lo);
  for (int64_t i = 0; i < n; ++i) {
    if (status && status[i] != 0) continue;
    const double t = (values[i] - lo) * scale;
    if (t != t) continue;                      // NaN value: not counted
    if (t < 0.0) counts[0] += 1;
    else if (t >= (double)nbins) counts[nbins + 1] += 1;
    else counts[1 + (int64_t)std::floor(t)] += 1;
  }
  return 0;
}

int oracle_omp_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
