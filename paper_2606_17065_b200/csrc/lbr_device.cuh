// lbr_device.cuh -- device-side math for the fused LBR implied-volatility kernel (sm_100a).
//
// Per-row solver in normalised Black coordinates (eq.(4)-(5); :359-363 A.5 stages 1-5):
//   x = ln(F/K) reduced to x <= 0, s = sigma sqrt(tau), h = x/s, t = s/2, beta = time value / sqrt(FK),
//   b(x,s) = e^{x/2} Phi(h+t) - e^{-x/2} Phi(h-t),  b' = phi0 exp(-E), E = (h^2+t^2)/2,  b_max = e^{x/2}.
// Everything is expressed through the ratios  W = b/b'  and  Wbar = (b_max-b)/b', built on erfcx of NON-NEGATIVE
// arguments only  (z1 = (|h|-t)/sqrt2, z2 = (|h|+t)/sqrt2, c = sqrt(pi/2)):
//   z1 >= 0:  W    = c [erfcx(z1) - erfcx(z2)]                       Wbar = b_max/b' - W
//   z1 <  0:  Wbar = c [erfcx(-z1) + erfcx(z2)]                      W    = b_max/b' - Wbar
//   t < 0.1:  W    = 2 sum_j w^(2j+1)(h) t^(2j+1)/(2j+1)!,  w(z) = Phi(z)/phi(z) = c erfcx(-z/sqrt2)   (no cancellation)
// The solve is split in passes so that the kernel can regroup rows in shared memory between them (pivot_iv.cu):
// lbr_seed_head (boundary point, node, zone, middle-zone seeds), lbr_seed_tail0 / _tail3 (tail seeds) and lbr_refine
// (Householder(3) steps).
//
// Precision tiers (template parameter FULL).  FULL = false, the default instantiation: the seed and every Householder
// step but the last run at "seed grade" -- fp32 erfcx, MUFU exp / log, one-Newton reciprocals, and the rational-cubic
// interpolants in fp32 on O(1) quantities (the NORMALISED form below); the status decision, the normalisation, ln(beta),
// the last Householder step and b' at the final s run at full fp64.  FULL = true (PIVOT_FWD_FP64_ONLY): the same
// formulas with every special function and reciprocal at full fp64, for the A/B that bounds the tiering.
//
// Normalised rational cubic.  The Delbourgo-Gregory interpolant is affine invariant, so every seed interpolates
// Y(u) on [0,1] with Y(0) = 0, Y(1) = 1, end slopes Dl, Dr and end curvature DD (all dimensionless):
//   Y(u) = u G(u),  G = [u (u + (r - Dr)(1-u)) + (1-u)^2 Dl] / [1 + (r-3) u (1-u)],
//   r = (DD/2 + Dr - Dl)/(Dr - 1) (curvature fitted at u = 1), floored for monotonicity.
// In these variables the exponentials of the tail maps f_low, f_up cancel analytically (see lbr_seed_tail0/3), which is
// what lets the interpolants run in fp32 for every |x| <= 693.
//
// exp / log / log1p / erfcx / reciprocals are this file's own, with coefficients in constant memory (gen_coeffs.py):
// no slow paths, no 64-bit immediates.  See DESIGN.md section 5.
// This file shares nothing with oracle/ (the CPU checker).
#pragma once
#include <cstdint>
#include <type_traits>
#include <cuda_runtime.h>

#include "coeffs.cuh"

namespace pivot {

// Scalar constants live in constant memory: an fp64 instruction takes a c[bank][offset] operand for free, whereas a
// 64-bit immediate costs two extra MOV/UMOV issue slots (16.6 % of all issued instructions in the v3 capture,
// profiles/r1a_forward_v3_ncu_full.md).
static __constant__ double kInvSqrt2 = 0.70710678118654752440;       // 1/sqrt(2)
static __constant__ double kSqrtPiOver2 = 1.2533141373155002512;      // sqrt(pi/2)
static __constant__ double kSqrt2Pi = 2.5066282746310005024;          // sqrt(2 pi)
static __constant__ double kPhi0 = 0.39894228040143267794;            // 1/sqrt(2 pi)
static __constant__ double kLnPhi0 = -0.91893853320467274178;         // ln(1/sqrt(2 pi))
static __constant__ double kTwoThirdsLnPhi0 = -0.61262568880311516119;  // (2/3) ln(1/sqrt(2 pi))
static __constant__ double kInvSqrt3 = 0.57735026918962576451;        // 1/sqrt(3)
static __constant__ double kLog2e = 1.4426950408889634074;            // 1/ln 2
static __constant__ double kLn2 = 0.69314718055994530942;             // ln 2 (nearest double)
static __constant__ double kLn2Lo = 2.3190468138462995584e-17;        // ln 2 - (double)ln 2
static __constant__ double kSmallT = 0.1;                              // |h| - t below -kSmallT: sum form of eval_W; t_c below it: series for s_l
static __constant__ double kSqrt2 = 1.4142135623730950488;            // sqrt(2)
static __constant__ double kSqrt2m1 = 0.41421356237309504880;         // sqrt(2) - 1
static __constant__ double kSeriesC[5] = {1.0 / 6.0, 1.0 / 120.0, 1.0 / 5040.0, 1.0 / 362880.0, 1.0 / 39916800.0};
static __constant__ double kNinvCut = -1.0651;                         // ln 0.345: domain of the Phi^-1 tail fit

enum : int { KIND_LOWER = 0, KIND_LINEAR = 1, KIND_UPPER = 2 };

__device__ __forceinline__ int hi32(double v) { return __double2hiint(v); }
__device__ __forceinline__ int lo32(double v) { return __double2loint(v); }
__device__ __forceinline__ bool is_fin(double v) { return (hi32(v) & 0x7fffffff) < 0x7ff00000; }   // not NaN, not +-inf
// 0 < v < inf (false for NaN): two fp64 compares
__device__ __forceinline__ bool pos_fin(double v) { return v > 0.0 && v < __longlong_as_double(0x7ff0000000000000LL); }
__device__ __forceinline__ double canonical_nan() { return __longlong_as_double(0x7ff8000000000000LL); }
// max / min of two ordinary numbers (no NaN propagation rules to honour: one compare, one select)
__device__ __forceinline__ double dmax_nn(double a, double b) { return a > b ? a : b; }
__device__ __forceinline__ double dmin_nn(double a, double b) { return a < b ? a : b; }

// 1/x from MUFU.RCP64H (about 20 bits, full fp64 exponent range, no slow path) plus Newton steps.
__device__ __forceinline__ double rcp_raw(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  return r;
}
__device__ __forceinline__ double rcp_nr1(double x) {  // relative error ~1e-12: seeds only
  double r = rcp_raw(x);
  r = fma(r, fma(-x, r, 1.0), r);
  return r;
}
// relative error ~1 ulp: ONE third-order step from the MUFU value r0 (9e-7):  e = 1 - x r0,  1/x = r0 (1 + e + e^2) (1 + O(e^3)).
// Three dependent fp64 instructions (two Newton steps take four).
__device__ __forceinline__ double rcp_nr2(double x) {
  const double r0 = rcp_raw(x);
  const double e = fma(-x, r0, 1.0);
  return fma(r0, fma(e, e, e), r0);
}
// a/b to ~1 ulp (b normal, finite, non-zero)
__device__ __forceinline__ double div_fast(double a, double b) {
  const double r = rcp_nr1(b);   // 1e-12: the residual correction below squares it
  const double q = a * r;
  return fma(fma(-b, q, a), r, q);
}
__device__ __forceinline__ float rcpf(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

// exp(a), |a| < ~745; error ~1 ulp.  n = rint(a log2 e) through the 1.5*2^52 shift, Cody-Waite reduction by fma,
// degree-11 polynomial (coeffs.cuh), exponent add.
__device__ __forceinline__ double exp_fast(double a) {
  const double sh = 6755399441055744.0;
  const double tt = fma(a, kLog2e, sh);
  const int n = __double2loint(tt);
  const double nf = tt - sh;
  double r = fma(nf, -kLn2, a);
  r = fma(nf, -kLn2Lo, r);
  double p = kExpP[kExpN];
#pragma unroll
  for (int k = kExpN - 1; k >= 0; --k) p = fma(p, r, kExpP[k]);
  if ((unsigned)(n + 1020) > 2040u) {  // result leaves the normal range: two-step scaling / saturation
    if (n > 1020)
      return (n > 1024) ? __longlong_as_double(0x7ff0000000000000LL)
                        : p * 0x1p512 * __hiloint2double((n - 512 + 1023) << 20, 0);
    if (n < -1080) return 0.0;
    return p * __hiloint2double((n + 128 + 1023) << 20, 0) * 0x1p-128;
  }
  return __hiloint2double(__double2hiint(p) + (n << 20), __double2loint(p));
}

// ef ln2 + 2 atanh(num/den), |num/den| <= 0.175
__device__ __forceinline__ double log_core(double num, double den, double ef) {
  const double r = rcp_nr1(den);   // 1e-12: the residual correction of f below squares it
  const double f0 = num * r;
  const double f = fma(fma(-den, f0, num), r, f0);
  const double w = f * f;
  double G = kAtanhG[kAtanhN];
#pragma unroll
  for (int k = kAtanhN - 1; k >= 0; --k) G = fma(G, w, kAtanhG[k]);
  const double two_f = f + f;
  const double tail = fma(ef, kLn2Lo, two_f * w * G);
  return fma(ef, kLn2, two_f) + tail;
}

// ln(v), v positive and normal; error ~1 ulp
__device__ __forceinline__ double log_fast(double v) {
  int hi = __double2hiint(v);
  int e = (hi >> 20) - 1023;
  hi = (hi & 0x000fffff) | 0x3ff00000;
  if (hi > 0x3ff6a09e) { hi -= 0x00100000; e += 1; }  // m in (sqrt2/2, sqrt2]
  const double m = __hiloint2double(hi, __double2loint(v));
  const double num = m - 1.0;
  return log_core(num, num + 2.0, (double)e);
}

// ln(1 + q), q >= 0 finite; relative error ~1 ulp also for tiny q
__device__ __forceinline__ double log1p_fast(double q) {
  const double u = 1.0 + q;
  int hi = __double2hiint(u);
  int e = (hi >> 20) - 1023;
  hi = (hi & 0x000fffff) | 0x3ff00000;
  if (hi > 0x3ff6a09e) { hi -= 0x00100000; e += 1; }
  const double m = __hiloint2double(hi, __double2loint(u));
  const double num = (q < kSqrt2m1) ? q : m - 1.0;  // q < sqrt2 - 1  =>  e == 0 and q itself is the exact numerator
  return log_core(num, num + 2.0, (double)e);
}

// erfcx(z1), erfcx(z2) for z1, z2 >= 0:  erfcx(z) = (2C/(z+C)) Q((z-C)/(z+C)), one shared reciprocal.
__device__ __forceinline__ void erfcx_pair(double z1, double z2, double& e1, double& e2) {
  const double d1 = z1 + kErfcxC, d2 = z2 + kErfcxC;
  const double r12 = rcp_nr2(d1 * d2);
  const double r1 = r12 * d2, r2 = r12 * d1;
  const double y1 = fma(-2.0 * kErfcxC, r1, 1.0), y2 = fma(-2.0 * kErfcxC, r2, 1.0);
  double q1 = kErfcxQ[kErfcxN], q2 = kErfcxQ[kErfcxN];
#pragma unroll
  for (int k = kErfcxN - 1; k >= 0; --k) {
    q1 = fma(q1, y1, kErfcxQ[k]);
    q2 = fma(q2, y2, kErfcxQ[k]);
  }
  e1 = (2.0 * kErfcxC) * r1 * q1;
  e2 = (2.0 * kErfcxC) * r2 * q2;
}

// erfcx(z), z >= 0 (single evaluation, same polynomial as erfcx_pair)
__device__ __forceinline__ double erfcx_one(double z) {
  const double r = rcp_nr2(z + kErfcxC);
  const double y = fma(-2.0 * kErfcxC, r, 1.0);
  double q = kErfcxQ[kErfcxN];
#pragma unroll
  for (int k = kErfcxN - 1; k >= 0; --k) q = fma(q, y, kErfcxQ[k]);
  return (2.0 * kErfcxC) * r * q;
}

// ---- fp32-grade helpers for the seeds (relative error ~1e-6; results carried as double where the range needs it) ----
__device__ __forceinline__ float ex2_approx(float f) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(f)); return r; }
__device__ __forceinline__ float lg2_approx(float f) { float r; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(f)); return r; }

// exp(a) for |a| < 700, relative error ~2e-7
__device__ __forceinline__ double exp_seed(double a) {
  const double tt = a * kLog2e;
  const double n = rint(tt);
  const float m = ex2_approx(__double2float_rn(tt - n));
  const int e = (int)n;
  return (double)m * __hiloint2double((e + 1023) << 20, 0);
}
// exp(a) for a float in [-87, 87]
__device__ __forceinline__ float expf_seed(float a) { return ex2_approx(a * 1.4426950408889634f); }
__device__ __forceinline__ float logf_seed(float v) { return lg2_approx(v) * 0.6931471805599453f; }

// ln(v) for v > 0, absolute error ~1e-7 * max(1, |ln v|)
__device__ __forceinline__ double log_seed(double v) {
  int adj = 1023;
  if (v < 2.2250738585072014e-308) { v *= 0x1p64; adj += 64; }  // subnormal
  const int hi = __double2hiint(v);
  const int e = (hi >> 20) - adj;
  const double m = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, __double2loint(v));  // [1,2)
  return ((double)e + (double)lg2_approx(__double2float_rn(m))) * kLn2;
}

// erfcx(z), z >= 0, fp32
__device__ __forceinline__ float erfcx_seed(float z) {
  const float r = rcpf(z + kErfcxCf);
  const float y = fmaf(-2.0f * kErfcxCf, r, 1.0f);
  float q = kErfcxQf[kErfcxNf];
#pragma unroll
  for (int k = kErfcxNf - 1; k >= 0; --k) q = fmaf(q, y, kErfcxQf[k]);
  return 2.0f * kErfcxCf * r * q;
}

// -Phi^-1(p) from lnp = ln p, p <= 0.345: u = sqrt(-2 ln p), z = u - R(1/(1+u)); relative error ~2e-5
__device__ __forceinline__ float ninv_tail_seed(float lnp) {
  const float u = sqrtf(-2.0f * lnp);
  const float w = rcpf(1.0f + u);
  float R = kNinvR[kNinvN];
#pragma unroll
  for (int k = kNinvN - 1; k >= 0; --k) R = fmaf(R, w, kNinvR[k]);
  return u - R;
}
// ... refined at full fp64 by two Newton steps on ln Phi(-z) = ln(erfcx(z/sqrt2)/2) - z^2/2 (FULL instantiation only)
__device__ __forceinline__ double ninv_tail_full(double lnp) {
  double z = (double)ninv_tail_seed(__double2float_rn(lnp));
#pragma unroll 1
  for (int it = 0; it < 2; ++it) {
    const double e = erfcx_one(z * kInvSqrt2);
    const double f = log_fast(0.5 * e) - 0.5 * z * z - lnp;
    z = fma(f, kSqrtPiOver2 * e, z);   // z - f/f',  f' = -1/(c erfcx(z/sqrt2))
  }
  return z;
}

// sqrt(v), v >= 0, relative error ~1e-12 (MUFU.RSQ64H + one Newton step); seeds only
__device__ __forceinline__ double sqrt_nr1(double v) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(v));
  y = y * fma(-0.5 * v, y * y, 1.5);
  return (v > 0.0) ? v * y : 0.0;
}

// sqrt(v) and 1/sqrt(v), v > 0 normal, ~1 ulp, no slow path: MUFU.RSQ64H + two Newton steps + one residual correction
__device__ __forceinline__ double sqrt_nr2(double v, double& rinv) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(v));
  const double hv = -0.5 * v;
  y = y * fma(hv, y * y, 1.5);
  y = y * fma(hv, y * y, 1.5);
  const double s = v * y;
  rinv = y;
  return fma(fma(-s, s, v), 0.5 * y, s);
}

__device__ __forceinline__ double sqrt_nr2(double v) { double r; return sqrt_nr2(v, r); }

// 1/sqrt(v), v positive normal, ~1 ulp: ONE third-order step from the MUFU value y0 (~1e-6):  e = 1 - v y0^2,
// 1/sqrt(v) = y0 (1 + e/2 + 3 e^2/8) (1 + O(e^3)).  Five dependent fp64 instructions (two Newton steps take seven).
__device__ __forceinline__ double rsqrt_c3(double v) {
  double y0;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(v));
  const double e = fma(-(v * y0), y0, 1.0);
  return fma(y0 * e, fma(0.375, e, 0.5), y0);
}

// sqrt(v) to ~1 ulp with 1/sqrt(v) only to ~1e-12: one Newton step + the residual correction (which squares the error of the
// Newton value).  For callers that use the reciprocal root only inside residual-corrected quotients (lbr_normalise).
__device__ __forceinline__ double sqrt_nr1c(double v, double& rinv) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(v));
  y = y * fma(-0.5 * v, y * y, 1.5);
  const double s = v * y;
  rinv = y;
  return fma(fma(-s, s, v), 0.5 * y, s);
}

// grade-dependent primitives
// seed-grade reciprocal: MUFU.RCP64H alone (9e-7 relative, measured: tests/test_gpu_mathlib.py), no Newton step -- every consumer is a
// rational-seed quantity that is rounded to fp32 or only has to land the seed within ~1e-3
template <bool FULL> __device__ __forceinline__ double g_rcp(double x) { return FULL ? rcp_nr2(x) : rcp_raw(x); }
template <bool FULL> __device__ __forceinline__ double g_exp(double a) { return FULL ? exp_fast(a) : exp_seed(a); }
template <bool FULL> __device__ __forceinline__ double g_log(double v) { return FULL ? log_fast(v) : log_seed(v); }
template <bool FULL> __device__ __forceinline__ double g_erfcx(double z) {
  return FULL ? erfcx_one(z) : (double)erfcx_seed(__double2float_rn(z));
}

// ---------------------------------------------------------------------------------------------------------------
// erfcx(z1) - erfcx(z2) and erfcx(z1) + erfcx(z2) for z1 >= kErfcxZmin, z2 = z1 + delta, delta >= 0 handed in as formed by
// the caller WITHOUT cancellation.  With r = 1/(z + C), y = 1 - 2C r, erfcx(z) = 2C r Q(y) and the divided difference
// DQ = Q[y1, y2] (one Horner-type recurrence beside the one of Q(y1): c_k = b_{k+1} + y2 c_{k+1}; no division):
//   y2 - y1 = 2C delta r1 r2,        Q(y2) = Q(y1) + (y2 - y1) DQ,
//   erfcx(z1) - erfcx(z2) = 2C delta r1 r2 [Q(y1) - 2C r2 DQ]     a PRODUCT: full relative accuracy however small delta is
//   erfcx(z1) + erfcx(z2) = 2C [r1 Q(y1) + r2 Q(y2)]
// (Q - 2C r Q' = -erfcx'(z) (z + C)^2 / 2C runs from 2.26 at z = 0 to 1/(2C sqrt(pi)) at infinity with both terms positive:
// no cancellation inside the bracket either.)  Same cost as two independent erfcx evaluations, and it replaces the
// small-t Taylor series of W that round 1 needed where the plain difference cancels.
// ---------------------------------------------------------------------------------------------------------------
// Two adjacent doubles of a __constant__ table, loaded into ordinary registers where they are used.  sm_100a instructions
// take no constant-bank operand: every constant passes through a register, the compiler hoists all such loads out of the pass
// loops into UNIFORM registers, and once those run out (the fp64 erfcx table alone needs 50) it parks the overflow in vector
// registers and swaps it in and out through MOV.SPILL / R2UR (3.7 % of the issued instructions, ~12 vector registers).
// `vary` is a per-thread byte offset that is always 0 but that the compiler cannot prove uniform: the load then is a plain
// LDC.128 into vector registers, outside the uniform register file.
__device__ __forceinline__ void ldc_pair(const double* p, unsigned vary, double& lo, double& hi) {
  asm volatile("ld.const.v2.f64 {%0, %1}, [%2];" : "=d"(lo), "=d"(hi) : "l"(__cvta_generic_to_constant(p) + vary));
}

// INPLACE = true: the table is read in place (ldc_pair: the tile kernel, whose pass loops overflow the uniform registers);
// false: ordinary constant operands (the row-per-thread kernel and the single-use callers).  Same arithmetic, same bits.
template <bool INPLACE = false>
__device__ __forceinline__ double erfcx_dd(double z1, double z2, double delta, bool want_sum) {
  static_assert(kErfcxN % 2 == 0, "the pairs (k-2, k-1) start at even indices");
  const double d1 = z1 + kErfcxC, d2 = z2 + kErfcxC;
  const double r12 = rcp_nr2(d1 * d2);            // = r1 r2
  const double r1 = r12 * d2, r2 = r12 * d1;
  const double y1 = fma(-2.0 * kErfcxC, r1, 1.0), y2 = fma(-2.0 * kErfcxC, r2, 1.0);
  const unsigned vary = ((unsigned)__double2hiint(d2) >> 31) << 4;   // sign bit of d2 = z2 + C >= 3.9: always 0
  double b = kErfcxQ[kErfcxN], c = 0.0;
#pragma unroll
  for (int k = kErfcxN; k >= 2; k -= 2) {
    double q0, q1;
    if (INPLACE) { ldc_pair(&kErfcxQ[k - 2], vary, q0, q1); } else { q0 = kErfcxQ[k - 2]; q1 = kErfcxQ[k - 1]; }
    c = fma(c, y2, b);
    b = fma(b, y1, q1);
    c = fma(c, y2, b);
    b = fma(b, y1, q0);
  }
  const double p = (2.0 * kErfcxC) * delta * r12;  // y2 - y1
  const double diff = p * fma(-2.0 * kErfcxC, r2 * c, b);
  const double sum = (2.0 * kErfcxC) * fma(r1, b, r2 * fma(p, c, b));
  return want_sum ? sum : diff;
}

// ... at seed grade: fp32, on the FMA pipe (relative error ~2e-6 in either result)
__device__ __forceinline__ float erfcx_dd_seed(float z1, float z2, float delta, bool want_sum) {
  const float d1 = z1 + kErfcxCf, d2 = z2 + kErfcxCf;
  const float r12 = rcpf(d1 * d2);
  const float r1 = r12 * d2, r2 = r12 * d1;
  const float y1 = fmaf(-2.0f * kErfcxCf, r1, 1.0f), y2 = fmaf(-2.0f * kErfcxCf, r2, 1.0f);
  float b = kErfcxQf[kErfcxNf], c = 0.0f;
#pragma unroll
  for (int k = kErfcxNf - 1; k >= 0; --k) {
    c = fmaf(c, y2, b);
    b = fmaf(b, y1, kErfcxQf[k]);
  }
  const float p = (2.0f * kErfcxCf) * delta * r12;
  const float diff = p * fmaf(-2.0f * kErfcxCf, r2 * c, b);
  const float sum = (2.0f * kErfcxCf) * fmaf(r1, b, r2 * fmaf(p, c, b));
  return want_sum ? sum : diff;
}

// ---------------------------------------------------------------------------------------------------------------
// W-evaluation shared by the node stage and the Householder stages: at the point s returns
//   have_W = true : Wd = W = b/b'     = c [erfcx(z1) - erfcx(z2)]    (z1 >= -0.1/sqrt2: the difference form, by erfcx_dd)
//   have_W = false: Wd = Wbar = (b_max-b)/b' = c [erfcx(-z1) + erfcx(z2)]   (z1 < -0.1/sqrt2, which implies t > 0.1)
// together with h = x/s, 1/s and E = (h^2+t^2)/2.   z1 = (|h| - t)/sqrt2, z2 = (|h| + t)/sqrt2.
// The gap delta of erfcx_dd is sqrt2 t (difference form) or sqrt2 |h| (sum form: z2 - (-z1)), both formed directly.
// ---------------------------------------------------------------------------------------------------------------
struct WEval {
  double Wd, E, h, rs;
  bool have_W;
};

// SEED = true: the erfcx pair in fp32 on the FMA pipe (~2e-6): enough for the node of the seed interpolant and for every
// Householder step but the last.
template <bool SEED = false, bool INPLACE = false>
__device__ __forceinline__ WEval eval_W(double x, double s) {
  WEval w;
  w.rs = SEED ? rcp_nr1(s) : rcp_nr2(s);
  w.h = x * w.rs;  // <= 0
  const double t = 0.5 * s;
  const double ah = -w.h;
  w.E = 0.5 * fma(w.h, w.h, t * t);
  const double dz = ah - t;            // sqrt2 z1
  const bool sum = dz < -kSmallT;      // z1 < -0.0707 (> kErfcxZmin)
  w.have_W = !sum;
  if (SEED) {
    const float ahf = __double2float_rn(ah), tf = __double2float_rn(t);
    const float dzf = ahf - tf;
    const float e = erfcx_dd_seed((sum ? -dzf : dzf) * 0.70710678f, (ahf + tf) * 0.70710678f, (sum ? ahf : tf) * 1.41421356f, sum);
    w.Wd = (double)(1.2533141f * e);
  } else {
    w.Wd = kSqrtPiOver2 * erfcx_dd<INPLACE>((sum ? -dz : dz) * kInvSqrt2, (ah + t) * kInvSqrt2, (sum ? ah : t) * kSqrt2, sum);
  }
  return w;
}

// ---------------------------------------------------------------------------------------------------------------
// Normalised rational cubic (header comment): R = float at seed grade, double in the FULL instantiation.
// ---------------------------------------------------------------------------------------------------------------
template <typename R> __device__ __forceinline__ R r_rcp(R x);
template <> __device__ __forceinline__ float r_rcp<float>(float x) { return rcpf(x); }
template <> __device__ __forceinline__ double r_rcp<double>(double x) { return rcp_nr2(x); }
template <typename R> __device__ __forceinline__ R r_max(R a, R b) { return a > b ? a : b; }
template <> __device__ __forceinline__ float r_max<float>(float a, float b) { return fmaxf(a, b); }
template <typename R> __device__ __forceinline__ R r_abs(R a) { return a < R(0) ? -a : a; }
template <> __device__ __forceinline__ float r_abs<float>(float a) { return fabsf(a); }
template <> __device__ __forceinline__ double r_abs<double>(double a) { return fabs(a); }

// control parameter: curvature DD fitted at u = 1; floored by the monotonicity / convexity bounds
// (Delta = 1 in these variables); +inf = linear interpolant
template <typename R>
__device__ __forceinline__ R rcn_control(R Dl, R Dr, R DD) {
  const R dR = Dr - R(1), dL = R(1) - Dl, span = Dr - Dl;
  const R rR = r_rcp<R>(dR), rL = r_rcp<R>(dL);
  R r = fma(R(0.5), DD, span) * rR;
  R rmin = r_max<R>(R(-0.999), Dl + Dr);
  if (dR != R(0)) rmin = r_max<R>(rmin, r_abs<R>(span * rR));
  if (dL != R(0)) rmin = r_max<R>(rmin, r_abs<R>(span * rL));
  if (dR == R(0)) r = R(3e38);
  return (r > rmin) ? r : rmin;     // a NaN r falls to rmin
}

// G(u) = Y(u)/u
template <typename R>
__device__ __forceinline__ R rcn_G(R u, R omu, R Dl, R Dr, R r) {
  if (!(r < R(1e30))) return R(1);
  const R num = fma(u, fma(r - Dr, omu, u), omu * omu * Dl);
  return num * r_rcp<R>(fma(r - R(3), u * omu, R(1)));
}

// ---------------------------------------------------------------------------------------------------------------
// Pass 1 of the solve (A.5 stage 4): boundary point, zone, rational seed.  Split in two so that the
// kernel can regroup rows by zone in between:
//   lbr_seed_head : x, boundary point s_c, node (s_l or s_u), zone.  The two middle zones (1, 2: s(beta) interpolated
//                   between the node and the inflection point) are finished here; the tails only hand over their node.
//   lbr_seed_tail0 / lbr_seed_tail3 : the lower / upper tail maps f_low, f_up, their rational-cubic interpolant in beta
//                   and its inversion.
// Result of the pass: x = -ln(1+qrel) <= 0, the seed s0, the objective kind and its two parameters
//        KIND_LOWER : p1 = ln beta,          p2 unused       g = 1/ln b - 1/ln beta
//        KIND_LINEAR: p1 = beta,             p2 = bbar       g = b - beta
//        KIND_UPPER : p1 = ln(b_max - beta), p2 unused       g = ln((b_max - beta)/(b_max - b))
// ---------------------------------------------------------------------------------------------------------------
struct SeedHead {
  int zone;        // 0: tail pending, v = (x, s_n, beta, pack(W_n, beta/b_n));  3: tail pending, v = (x, s_n, bbar,
                   // pack(Wbar_n, bbar/bbar_n));  1, 2: v = (x, pack(-+s_n, wq), beta, pack(Dr, Dl)) for lbr_seed_mid (sign
                   // bit of the first float set: zone 1); FULL tier: finished, v = (x, s0, beta, bbar)
  double v0, v1, v2, v3;
};

__device__ __forceinline__ double pack2f(float a, float b) {
  return __hiloint2double(__float_as_int(b), __float_as_int(a));
}
__device__ __forceinline__ void unpack2f(double p, float& a, float& b) {
  a = __int_as_float(__double2loint(p));
  b = __int_as_float(__double2hiint(p));
}

template <bool FULL>
__device__ __forceinline__ SeedHead lbr_seed_head(double qrel, double beta, double bbar, double bmax) {
  SeedHead o;
  const double x = -log1p_fast(qrel);
  const double a = -x;
  o.v0 = x;
  const double sc = sqrt_nr1(2.0 * a);        // inflection point of b(x, .)
  const double vc = kPhi0 * bmax;             // b'(x, s_c) = phi0 e^{-|x|/2}
  // at s_c: |h| = t = s_c/2, so z1 = 0, z2 = sqrt(|x|):  W_c = c (1 - erfcx(sqrt|x|)), and the tangent at the inflection
  // point hits 0 at s_l = s_c - W_c.  For small s_c that difference cancels (s_l ~ 0.63 s_c^2), so there s_l comes from
  // the small-t series of W itself:  W_c = s_c (w1 + t^2 w3/6 + t^4 w5/120 + ...), w1 = 1 - t w0  =>
  //   s_l = s_c (t w0 - t^2 w3/6 - t^4 w5/120 - t^6 w7/5040),  w(.) at h = -t, w0 = c erfcx(t/sqrt2)
  const double tc = 0.5 * sc;
  const bool small_c = tc < kSmallT;
  const double ec = g_erfcx<FULL>((small_c ? tc : sc) * kInvSqrt2);
  double Wc, sl;
  if (small_c) {
    const double w0 = kSqrtPiOver2 * ec;
    const double w1 = fma(-tc, w0, 1.0);
    const double w2 = fma(-tc, w1, w0);
    const double w3 = fma(-tc, w2, 2.0 * w1);
    const double w4 = fma(-tc, w3, 3.0 * w2);
    const double w5 = fma(-tc, w4, 4.0 * w3);
    const double w6 = fma(-tc, w5, 5.0 * w4);
    const double w7 = fma(-tc, w6, 6.0 * w5);
    const double t2 = tc * tc;
    const double tail = t2 * fma(t2, fma(t2, w7 * kSeriesC[2], w5 * kSeriesC[1]), w3 * kSeriesC[0]);
    sl = sc * fma(tc, w0, -tail);
    Wc = sc - sl;
  } else {
    Wc = kSqrtPiOver2 * (1.0 - ec);
    sl = sc - Wc;
  }
  const double Wbc = kSqrt2Pi - Wc;           // (b_max - b_c)/b'(s_c)
  const double bc = vc * Wc;
  const bool lower = beta < bc;
  o.v2 = beta; o.v3 = bbar;
  if (lower && !(sl > 1e-30)) {  // rounding / fp32-range guard, |x| below ~1e-30: linear seed
    o.zone = 1;
    const double lin = beta * rcp_nr1(bc);
    if (FULL) {
      o.v1 = sc * lin;
    } else {   // the same linear seed through lbr_seed_mid: node at s = 0, Dl = Dr = 1 (G = 1)
      o.v1 = pack2f(-0.0f, __double2float_rn(lin));
      o.v3 = pack2f(1.0f, 1.0f);
    }
    return o;
  }
  const double sn = lower ? sl : sc + Wbc;    // s_l, or s_u where the tangent at the inflection point hits b_max
  const WEval w = eval_W<!FULL>(x, sn);
  const double vn = kPhi0 * g_exp<FULL>(-w.E);  // b'(s_n)
  const double wv = w.Wd * vn;
  const double bn = w.have_W ? wv : bmax - wv;       // b(s_n)
  const double bbn = w.have_W ? bmax - wv : wv;      // b_max - b(s_n)
  if (lower ? (beta < bn) : (beta > bn)) {   // a tail: hand the node over
    // W_n (lower) or Wbar_n (upper), and the interpolation abscissa beta/b_n or bbar/bbar_n, as floats
    const double den = lower ? bn : bbn;
    const double rden = g_rcp<FULL>(den);
    const double Wn = (lower == w.have_W) ? w.Wd : den * g_rcp<FULL>(vn);
    o.zone = lower ? 0 : 3;
    o.v1 = sn;
    o.v2 = lower ? beta : bbar;
    o.v3 = pack2f(__double2float_rn(Wn), __double2float_rn((lower ? beta : bbar) * rden));
    return o;
  }
  // zones 1 and 2: s(beta) from the node (u = 0) to the inflection point (u = 1), s'' = 0 at the inflection point.
  // With kappa = b'(s_c)/b'(s_n) = exp(E_n - |x|/2) and rho = b_n/b_c (lower) or (b_max-b_n)/(b_max-b_c) (upper):
  //   Dr = 1 - rho = |b_c - b_n| / (b_c or b_max - b_c),  Dl = kappa (1 - rho),  DD = 0.
  // The interpolant is evaluated from the end with the SMALLER s (the node s_l below the inflection point, the inflection
  // point itself above it), so that s keeps its relative accuracy when s_c -> 0 (|x| -> 0): wq is the abscissa measured from
  // that end.  Default tier: only the three dimensionless parameters (wq, Dr, Dl) are formed here, where ~9 of 32 lanes are
  // middle-zone rows; the fp32 rational cubic itself runs in lbr_seed_mid on warps that hold middle-zone rows only.
  o.zone = lower ? 1 : 2;
  const double bbc = vc * Wbc;
  const double H = bc - bn;                         // > 0 below the inflection point, < 0 above it
  const double aH = fabs(H), den = lower ? bc : bbc;
  const double rHD = g_rcp<FULL>(aH * den);
  const double rH = rHD * den;                      // 1/|H|
  const double Drd = aH * (rHD * aH);               // |H| / den
  const double kappa = vc * g_rcp<FULL>(vn);
  const double wqd = (lower ? beta - bn : beta - bc) * rH;
  const double Dld = dmin_nn(kappa * Drd, 1e30);
  if (!FULL) {
    const float snf = __double2float_rn(sn);
    o.v1 = pack2f(lower ? -snf : snf, __double2float_rn(wqd));
    o.v3 = pack2f(__double2float_rn(Drd), __double2float_rn(Dld));
    return o;
  }
  const double r = rcn_control<double>(Dld, Drd, 0.0);
  const double Y = wqd * rcn_G<double>(wqd, 1.0 - wqd, lower ? Dld : Drd, lower ? Drd : Dld, r);
  const double s = fma(fabs(sc - sn), Y, lower ? sn : sc);
  o.v1 = (s > 0.0 && is_fin(s)) ? s : sc;   // a failed interpolant falls back to the inflection point
  return o;
}

struct Seed {
  double x, s, p1, p2;
  int kind, zone;
};

// zones 1, 2 (default tier): the fp32 rational cubic on the parameters lbr_seed_head packed (header comment there).
// The objective is LINEAR with p1 = beta; p2 = b_max - beta is rebuilt here (in these zones b_max - beta >= 0.1 b_max:
// at s_u, Phi(-(h+t)) >= Phi(-1.3), so the subtraction costs at most 3 bits of a quantity that only enters where
// Wbar is the ratio at hand).
__device__ __forceinline__ Seed lbr_seed_mid(double x, double packed_sn_wq, double beta, double packed_D) {
  Seed o;
  o.x = x; o.kind = KIND_LINEAR; o.p1 = beta;
  float sns, wq, Dr, Dl;
  unpack2f(packed_sn_wq, sns, wq);
  unpack2f(packed_D, Dr, Dl);
  const bool lower = __float_as_int(sns) < 0;
  o.zone = lower ? 1 : 2;
  const double sn = (double)fabsf(sns);
  const double sc = sqrt_nr1(-2.0 * x);
  const float r = rcn_control<float>(Dl, Dr, 0.0f);
  const float Y = wq * rcn_G<float>(wq, 1.0f - wq, lower ? Dl : Dr, lower ? Dr : Dl, r);
  const double s = fma(fabs(sc - sn), (double)Y, lower ? sn : sc);
  o.s = (s > 0.0 && is_fin(s)) ? s : sc;   // a failed interpolant falls back to the inflection point
  o.p2 = exp_fast(0.5 * x) - beta;
  return o;
}

// zone 0: f_low(s) = (2 pi |x| / 3 sqrt3) Phi(-z)^3, z = |x| / (sqrt3 s), as a function of beta on [0, b_l].
// In normalised variables (u = beta/b_l, Y = f/f_low(s_l)) with q = |x|/s_l = sqrt3 z, omega = W_l/s_l,
// Ym = Phi(-z)/phi(z) (Mills ratio), m = 1/Ym, every exponential of f', f'' cancels against b(s_l) = W_l phi0 e^{-E}:
//   Dl = 3 sqrt3 omega m^3 e^{-s_l^2/8} / q,   Dr = sqrt3 q omega m,
//   DD = (sqrt3/12) q [(3 (s_l^2 - 8) - 8 q^2) Ym + 8 sqrt3 q] (omega m)^2,
// and  ln Phi(-z(beta)) = ln Ym + (2/3) ln phi0 + s_l^2/24 + (ln beta - ln W_l + ln G(u))/3.
template <bool FULL>
__device__ __forceinline__ Seed lbr_seed_tail0(double x, double sn, double beta, double packed) {
  typedef typename std::conditional<FULL, double, float>::type R;
  const double a = -x;
  Seed o;
  o.x = x; o.zone = 0; o.kind = KIND_LOWER; o.p2 = 0.0;
  o.p1 = log_fast(beta);     // ln beta: the objective's target, full precision
  R Wn, u;
  if (FULL) {
    const WEval w = eval_W<false>(x, sn);        // have_W holds at s_l (z1 > 0 below the inflection point)
    const double bn = w.Wd * kPhi0 * exp_fast(-w.E);
    Wn = (R)w.Wd; u = (R)(beta * rcp_nr2(bn));
  } else {
    float fw, fu; unpack2f(packed, fw, fu); Wn = (R)fw; u = (R)fu;
  }
  const R snr = (R)sn, ar = (R)a;
  const R rs = r_rcp<R>(snr);
  const R q = ar * rs;
  const R Ym = (R)kSqrtPiOver2 * (R)g_erfcx<FULL>((double)(q * R(0.40824829046386301637)));   // z/sqrt2 = q/sqrt6
  const R m = r_rcp<R>(Ym);
  const R om = Wn * rs * m;
  const R sn2 = snr * snr;
  const R iB = FULL ? (R)exp_fast(-0.125 * (double)sn2) : (R)expf_seed(-0.125f * (float)sn2);
  const R Dr = R(1.7320508075688772935) * q * om;
  const R DD = R(0.14433756729740644113) * q * om * om *
               fma(fma(R(3), sn2, fma(R(-8), q * q, R(-24))), Ym, R(13.856406460551018348) * q);
  const R Dl = R(5.1961524227066318806) * om * m * m * iB * (snr * r_rcp<R>(ar));
  const R r = rcn_control<R>(Dl, Dr, DD);
  R G = rcn_G<R>(u, R(1) - u, Dl, Dr, r);
  if (!(G > R(0))) G = fma(Dl, R(1) - u, u);
  const double lnWG = FULL ? log_fast((double)G * rcp_nr2((double)Wn)) : (double)logf_seed((float)G * rcpf((float)Wn));
  const double lnY = FULL ? log_fast((double)Ym) : (double)logf_seed((float)Ym);
  const double lnp = dmin_nn(lnY + kTwoThirdsLnPhi0 + (double)sn2 * (1.0 / 24.0) + (o.p1 + lnWG) * (1.0 / 3.0), kNinvCut);
  const double zz = FULL ? ninv_tail_full(lnp) : (double)ninv_tail_seed(__double2float_rn(lnp));
  double s = a * kInvSqrt3 * g_rcp<FULL>(zz);
  if (!(s > 0.0) || !is_fin(s)) s = sn;
  o.s = s;
  return o;
}

// zone 3: f_up(s) = Phi(-s/2) as a function of beta on [b_u, b_max].  Interpolated from the b_max end (v = 0, f = 0) to
// the node (v = 1): v = bbar/bbar_u, Ybar = f/f_up(s_u) = v G(v), with h = x/s_u, e = erfcx(s_u/(2 sqrt2)):
//   slope at the node  Dn = Wbar_u phi0 / e,   slope at b_max  Dm = Dn e^{-h^2/2},
//   curvature at the node  DDn = 2 c (h^2/s_u) Wbar_u phi0 Dn,
// and  ln f = ln bbar + h^2/2 + ln(G(v) / (2 Dn)).
template <bool FULL>
__device__ __forceinline__ Seed lbr_seed_tail3(double x, double sn, double bbar, double packed) {
  typedef typename std::conditional<FULL, double, float>::type R;
  const double bmax = exp_fast(0.5 * x);   // e^{x/2} (the handover carries four words: beta = b_max - bbar)
  Seed o;
  o.x = x; o.zone = 3;
  const bool upper = bbar < 0.5 * bmax;
  double lnbbar;
  if (upper) {
    o.kind = KIND_UPPER; o.p1 = log_fast(bbar); o.p2 = 0.0; lnbbar = o.p1;
  } else {
    o.kind = KIND_LINEAR; o.p1 = bmax - bbar; o.p2 = bbar; lnbbar = g_log<FULL>(bbar);
  }
  const double rs = g_rcp<FULL>(sn);
  const double h = x * rs;
  const double hh2 = 0.5 * h * h;
  R Wbn, v;
  if (FULL) {
    const WEval w = eval_W<false>(x, sn);        // z1 < 0 above the inflection point: Wd = Wbar
    const double bbn = w.Wd * kPhi0 * exp_fast(-w.E);
    Wbn = (R)w.Wd; v = (R)(bbar * rcp_nr2(bbn));
  } else {
    float fw, fv; unpack2f(packed, fw, fv); Wbn = (R)fw; v = (R)fv;
  }
  const R e = (R)g_erfcx<FULL>(0.5 * sn * kInvSqrt2);
  const R Dn = Wbn * (R)kPhi0 * r_rcp<R>(e);
  const R Dm = Dn * (R)g_exp<FULL>(-hh2);
  const R DDn = R(5.0132565492620010048) * (R)(hh2 * rs) * Wbn * (R)kPhi0 * Dn;     // 2c h^2/s = 4c (h^2/2)/s
  const R r = rcn_control<R>(Dm, Dn, DDn);
  R G = rcn_G<R>(v, R(1) - v, Dm, Dn, r);
  if (!(G > R(0))) G = fma(Dm, R(1) - v, v);
  const double lnG = FULL ? log_fast((double)G * rcp_nr2(2.0 * (double)Dn)) : (double)logf_seed((float)G * rcpf(2.0f * (float)Dn));
  const double lnf = dmin_nn(lnbbar + hh2 + lnG, kNinvCut);
  double s = 2.0 * (FULL ? ninv_tail_full(lnf) : (double)ninv_tail_seed(__double2float_rn(lnf)));
  if (!(s > 0.0) || !is_fin(s)) s = sn;
  o.s = s;
  return o;
}

// one-call form (row-per-thread kernel)
template <bool FULL>
__device__ __forceinline__ Seed lbr_seed(double qrel, double beta, double bbar, double bmax) {
  const SeedHead hd = lbr_seed_head<FULL>(qrel, beta, bbar, bmax);
  if (hd.zone == 0) return lbr_seed_tail0<FULL>(hd.v0, hd.v1, hd.v2, hd.v3);
  if (hd.zone == 3) return lbr_seed_tail3<FULL>(hd.v0, hd.v1, hd.v2, hd.v3);
  if (!FULL) return lbr_seed_mid(hd.v0, hd.v1, hd.v2, hd.v3);
  Seed o;
  o.x = hd.v0; o.s = hd.v1; o.p1 = hd.v2; o.p2 = hd.v3; o.kind = KIND_LINEAR; o.zone = hd.zone;
  return o;
}

// ---------------------------------------------------------------------------------------------------------------
// Pass 2 of the solve (A.5 stage 5): NITER Householder(3) steps on the zone's objective, then
// b'(x, s) = phi0 exp(-E) at the final s for the vega (eq.(14)).
//   ds = nu (1 + h2 nu / 2) / (1 + nu (h2 + h3 nu / 6)),  nu = -g/g', h2 = g''/g', h3 = g'''/g',  ds >= -s/2.
// Each step needs W or Wbar (one erfcx pair or the small-t series) and ONE of exp / log:
//   LINEAR: 1/b' = sqrt(2 pi) e^E;   LOWER: ln W;   UPPER: ln Wbar
// (plus the exp when the available ratio is not the one the objective wants).
// ---------------------------------------------------------------------------------------------------------------
struct NormSolve {
  double s;     // total volatility after NITER Householder steps
  double s1;    // ... after NITER - 1 steps (diagnostics)
  double vfin;  // b'(x, s) at that s
};

// One Householder(3) step.  SEED = true evaluates W, exp and log at seed grade (fp32 erfcx pair, MUFU exp / log,
// ~1e-6 relative in the step): enough for every step but the last, because the step is fourth order and the last step
// then takes an iterate that is good to ~1e-6 to ~1e-24.  In EVERY step the factors that multiply the residual (the reciprocals
// inside nu, h2, h3 and the final quotient) use the one-Newton reciprocal (1e-12 relative): the step ds is at most 1e-4 s in the
// last step, so they enter s at 1e-16; the residual itself (W, exp E, ln W, ln beta) is what carries the full precision.
// The seed-grade step takes them from MUFU.RCP64H alone (9e-7).  (EXACT_RCP: the all-fp64 tier keeps two-Newton reciprocals.)
template <bool SEED, bool INPLACE, bool EXACT_RCP = false>
__device__ __forceinline__ double householder_step(double x, double s, double p1, double p2, int kind) {
  const WEval w = eval_W<SEED, INPLACE>(x, s);
  if (SEED && !EXACT_RCP) {
    // Seed-grade step: only the residual nu stays in fp64 (it is a cancelling difference); the third-order correction factor
    // is assembled in fp32 in SCALED variables n = nu/s, h2 s, h3 s^2, which are O(h^2) = O(1e3) at most for every s:
    //   ds/s = n (1 + h2s n/2) / (1 + n (h2s + h3s n/6)),  (b2/b1) s = h^2 - s^2/4,  (b3/b1) s^2 = ((b2/b1) s)^2 - 3 h^2 - s^2/4
    // (b1, b2, b3: first to third derivative of b in s).
    const float hf = __double2float_rn(w.h), sf = __double2float_rn(s);
    const float hh = hf * hf, sq = 0.25f * sf * sf;
    const float b2 = hh - sq;
    const float b3 = fmaf(b2, b2, fmaf(-3.0f, hh, -sq));
    double nu;
    float h2s, h3s;
    if (kind == KIND_LINEAR) {
      const double inv_v = kSqrt2Pi * exp_seed(w.E);
      nu = w.have_W ? fma(p1, inv_v, -w.Wd) : fma(-p2, inv_v, w.Wd);
      h2s = b2;
      h3s = b3;
    } else {
      const bool want_W = kind == KIND_LOWER;
      double R = w.Wd;
      // rare; one exponential of the summed exponent (relative error |x/2 + E| 2^-53 <= 1e-13: seed grade)
      if (want_W != w.have_W) R = fma(kSqrt2Pi, exp_fast(fma(0.5, x, w.E)), -w.Wd);
      const double L = kLnPhi0 - w.E + log_seed(R);
      const float u = __double2float_rn(s * rcp_raw(R));   // s/W or s/Wbar: O(h^2 + s^2)
      if (want_W) {
        const float lam = rcpf(__double2float_rn(L));
        const float k2 = fmaf(2.0f, lam, 1.0f);
        nu = (p1 - L) * (L * rcp_raw(p1)) * R;
        h2s = fmaf(-u, k2, b2);
        h3s = fmaf(u * u, fmaf(6.0f * lam, 1.0f + lam, 2.0f), fmaf(-3.0f * b2 * u, k2, b3));
      } else {
        nu = (L - p1) * R;
        h2s = b2 + u;
        h3s = fmaf(u, fmaf(2.0f, u, 3.0f * b2), b3);
      }
    }
    const float n = __double2float_rn(nu * w.rs);
    const float den = fmaf(n, fmaf(h3s * (1.0f / 6.0f), n, h2s), 1.0f);
    float f = n * fmaf(0.5f * h2s, n, 1.0f) * rcpf(den);
    if (!(f > -0.5f)) f = -0.5f;
    return fma(s, (double)f, s);
  }
  const double hr = w.h * w.rs;
  const double B2 = fma(w.h, hr, -0.25 * s);                  // second derivative of b over b'
  const double B3 = fma(B2, B2, fma(-3.0 * hr, hr, -0.25));   // third derivative of b over b'
  double nu, h2, h3;
  if (kind == KIND_LINEAR) {
    // g = b - beta:  nu = (beta - b)/b'  (p1 = beta, p2 = bbar)
    const double inv_v = kSqrt2Pi * (SEED ? exp_seed(w.E) : exp_fast(w.E));
    nu = w.have_W ? fma(p1, inv_v, -w.Wd) : fma(-p2, inv_v, w.Wd);
    h2 = B2;
    h3 = B3;
  } else {
    const bool want_W = kind == KIND_LOWER;
    double R = w.Wd;  // the ratio the objective wants: W (lower tail) or Wbar (upper tail)
    if (want_W != w.have_W) R = fma(exp_fast(0.5 * x) * kSqrt2Pi, exp_fast(w.E), -w.Wd);   // rare: b_max = e^{x/2} rebuilt here
    const double L = kLnPhi0 - w.E + (SEED ? log_seed(R) : log_fast(R));  // ln b (lower) or ln(b_max - b) (upper)
    if (want_W) {
      // g = 1/ln b - 1/ln beta  (p1 = ln beta)
      const double rLW = EXACT_RCP ? rcp_nr2(L * R) : (SEED ? rcp_raw(L * R) : rcp_nr1(L * R));
      const double lam = rLW * R, ub = rLW * L;  // 1/L, b'/b = 1/W
      const double k2 = fma(2.0, lam, 1.0);
      nu = (p1 - L) * (L * (EXACT_RCP ? rcp_nr2(p1) : (SEED ? rcp_raw(p1) : rcp_nr1(p1)))) * R;
      h2 = fma(-ub, k2, B2);
      h3 = fma(ub * ub, fma(6.0 * lam, 1.0 + lam, 2.0), fma(-3.0 * B2 * ub, k2, B3));
    } else {
      // g = ln((b_max - beta)/(b_max - b)):  g' = 1/Wbar  (p1 = ln(b_max - beta))
      const double gp = EXACT_RCP ? rcp_nr2(R) : (SEED ? rcp_raw(R) : rcp_nr1(R));
      nu = (L - p1) * R;
      h2 = B2 + gp;
      h3 = fma(gp, fma(2.0, gp, 3.0 * B2), B3);
    }
  }
  const double den = fma(nu, fma(h3 * (1.0 / 6.0), nu, h2), 1.0);
  double ds = nu * fma(0.5 * h2, nu, 1.0) * (EXACT_RCP ? rcp_nr2(den) : (SEED ? rcp_raw(den) : rcp_nr1(den)));
  if (!(ds > -0.5 * s)) ds = -0.5 * s;
  return s + ds;
}

template <int NITER, bool FULL, bool INPLACE = false>
__device__ __forceinline__ NormSolve lbr_refine(double x, double s, double p1, double p2, int kind) {
#pragma unroll 1
  for (int it = 0; it < NITER - 1; ++it) s = householder_step<!FULL, INPLACE, FULL>(x, s, p1, p2, kind);
  NormSolve o;
  o.s1 = s;
  s = householder_step<false, INPLACE, FULL>(x, s, p1, p2, kind);
  const double rs = rcp_nr2(s);
  const double h = x * rs, t = 0.5 * s;
  o.s = s;
  o.vfin = kPhi0 * exp_fast(-0.5 * fma(h, h, t * t));
  return o;
}

// ---------------------------------------------------------------------------------------------------------------
// Row prelude (Alg.1 l.1 and l.3; A.5 stages 1-2): validity and status for EVERY row.
//
// EXACT form (lbr_prelude_exact; the definition, and the path of unusual rows): only correctly rounded IEEE operations
// issued through intrinsics, so the decision cannot be contracted into FMAs and is bit-reproducible against any
// IEEE-754 implementation of the same sequence; no division:
//   beta = RN(tv / rootFK) < DBL_MIN   <=>   tv * 2^1022 < rootFK     (exact: the scaling is exact, and for doubles
//   bmax = RN(lo / rootFK) >= 2^-500   <=>   lo * 2^500 >= rootFK      a < b implies a <= b - ulp(b) < b (1 - 2^-53))
//
// FAST form (lbr_prelude): the same decision for the COMMON case, classified on the high words:
//   F (or S e^{(r-q)tau}), K in [2^-400, 2^400), tau positive normal, P (B) finite, flag = +-1  [, D in [2^-300, 2^300)].
// Then sqrt(FK) is in [2^-400, 2^400), so  lo 2^500 >= sqrt(FK)  holds and sqrt(FK) is positive finite;  tv <= 0  =>
// AT_INTRINSIC;  and  tv 2^1022 < sqrt(FK)  is decided from the exponents of tv, F and K except in a band two binades wide
// around beta = 2^-1022 (kD2Solve / kD2Zero below).  So no square root is needed to decide the status; rows outside the
// common case, and rows inside that band, take the exact form (status 5 = "rare" asks the caller to do so).  The remaining operations (F-K, U-B, lo-(U-B), B-iota and
// the comparisons) are the exact form's own, operation for operation, with U = the strike-side bound and O = the other
// one of (F, K):  iota = max(U - O, 0),  in the money <=> U > O,  lo = O and hi = U when in the money.
// BSM mode: F = S e^{(r-q)tau}, D = e^{-r tau}, B = P/D with this file's exp_fast / div_fast (<= 1 ulp) on the fast path
// and CUDA's exp / IEEE division on the exact path (reading 17: each side of the parity uses its own exp).
// ---------------------------------------------------------------------------------------------------------------
struct Prelude {
  double U;       // upper bound of the undiscounted price: F (call) or K (put)
  double O;       // the other one of (F, K)
  double B;       // undiscounted price (BSM: P / D)
  double D;       // discount factor (1 in Black-76 mode)
  int status;     // 0..4; lbr_prelude only: 5 = rare, take lbr_prelude_exact
};

template <bool BSM>
static __device__ __noinline__ Prelude lbr_prelude_exact(double SorF, double K, double tau, double r, double q, double P,
                                                  double flag) {
  Prelude p;
  bool bad = !pos_fin(SorF) || !pos_fin(K) || !pos_fin(tau) || !is_fin(P) || !(flag == 1.0 || flag == -1.0);
  double F = SorF, D = 1.0, B = P;
  if (BSM) {
    if (!is_fin(r) || !is_fin(q)) bad = true;
    if (!bad) {
      F = __dmul_rn(SorF, exp(__dmul_rn(__dsub_rn(r, q), tau)));
      D = exp(__dmul_rn(-r, tau));
      B = __ddiv_rn(P, D);
      if (!pos_fin(F) || !pos_fin(D) || !is_fin(B)) bad = true;
    }
  }
  const double rootFK = __dsqrt_rn(__dmul_rn(F, K));
  const double lo = fmin(F, K);
  if (!pos_fin(rootFK) || !(__dmul_rn(lo, 0x1p500) >= rootFK)) bad = true;
  const bool call = flag > 0.0;
  const double iota = fmax(call ? __dsub_rn(F, K) : __dsub_rn(K, F), 0.0);
  const double U = call ? F : K;
  const double hi = fmax(F, K);
  // time value (reading 18): B - iota where iota = F - K is exact (hi <= 2 lo, or out of the money), else
  // lo - (U - B), which does not inherit the half-ulp-of-hi rounding of iota (U - iota = lo exactly, U - B exact)
  const double tv = (iota > 0.0 && hi > __dmul_rn(2.0, lo)) ? __dsub_rn(lo, __dsub_rn(U, B)) : __dsub_rn(B, iota);
  int st = 0;
  if (bad) st = 3;
  else if (B < iota) st = 1;
  else if (B >= U) st = 2;
  else if (__dmul_rn(tv, 0x1p1022) < rootFK) st = 4;
  p.status = st;
  p.U = U;
  p.O = call ? K : F;
  p.B = B;
  p.D = D;
  return p;
}

constexpr unsigned kExpLo400 = (1023u - 400u) << 20;   // high word of 2^-400
constexpr unsigned kExpSpan800 = 800u << 20;
constexpr unsigned kExpLo300 = (1023u - 300u) << 20;
constexpr unsigned kExpSpan600 = 600u << 20;
// AT_INTRINSIC band on the high words.  With L(v) = hi32(v)/2^20 - 1023:  L(v) <= log2 v <= L(v) + 0.0861 for normal v,
// and log2 v <= L(v) + 1 for subnormal v.  d2 = hi32(tv) - (hi32(F) + hi32(K))/2 therefore brackets
// log2(tv / sqrt(FK)) = log2(beta):   d2 >= kD2Solve and tv normal  =>  beta > 2^-1022 (the row solves);
//                                     d2 <= kD2Zero   =>  beta < 2^-1022 (AT_INTRINSIC);  in between: the exact form decides.
constexpr int kD2Solve = -(1022 << 20) + (1 << 19);
constexpr int kD2Zero = -(1023 << 20) - (1 << 19);

template <bool BSM>
__device__ __forceinline__ Prelude lbr_prelude(double SorF, double K, double tau, double r, double q, double P,
                                               double flag) {
  Prelude p;
  const int hf = hi32(flag), hK = hi32(K);
  bool common = ((unsigned)(hK - (int)kExpLo400) < kExpSpan800) & ((unsigned)(hi32(tau) - 0x00100000) < 0x7fe00000u) &
                ((hf & 0x7fffffff) == 0x3ff00000) & (lo32(flag) == 0);
  double F = SorF, B = P, D = 1.0;
  if (BSM) {
    common = common & is_fin(r) & is_fin(q) & ((unsigned)(hi32(SorF) - (int)kExpLo400) < kExpSpan800);
    F = __dmul_rn(SorF, exp_fast(__dmul_rn(__dsub_rn(r, q), tau)));
    D = exp_fast(__dmul_rn(-r, tau));
    common = common & ((unsigned)(hi32(D) - (int)kExpLo300) < kExpSpan600);
    B = div_fast(P, D);
  }
  const int hF = hi32(F);
  common = common & ((unsigned)(hF - (int)kExpLo400) < kExpSpan800) & is_fin(B);
  const bool call = hf >= 0;
  const double U = call ? F : K, O = call ? K : F;
  const double d = __dsub_rn(U, O);
  const bool itm = d > 0.0;
  const double iota = itm ? d : 0.0;
  const double ub = __dsub_rn(U, B);
  const bool big = itm & (U > __dadd_rn(O, O));
  const double tv = big ? __dsub_rn(O, ub) : __dsub_rn(B, iota);
  const int d2 = hi32(tv) - (int)(((unsigned)hF + (unsigned)hK) >> 1);
  int st = ((d2 >= kD2Solve) & (hi32(tv) >= 0x00100000)) ? 0 : ((d2 <= kD2Zero) ? 4 : 5);   // the lower bound needs a normal tv
  st = (tv > 0.0) ? st : 4;
  st = (B >= U) ? 2 : st;
  st = (B < iota) ? 1 : st;
  p.status = common ? st : 5;
  p.U = U; p.O = O; p.B = B; p.D = D;
  return p;
}

// Normalised solver inputs of a row that reached the solver (A.5 stage 2), from (U, O, B) of the prelude.
// Quotients by reciprocal + one residual correction (~1 ulp, no slow path).  Common rows: sqrt(FK) and 1/sqrt(FK) from
// MUFU.RSQ64H + Newton (FK in [2^-800, 2^800): normal);  rare rows (flag set by the prelude): the IEEE square root, since
// FK may be subnormal there, and sqrt(FK) in [2^-537, 2^512].
struct Norm {
  double qrel;    // (hi - lo)/lo, hi = max(F,K), lo = min(F,K):  x = -log1p(qrel)
  double beta;    // time value / sqrt(FK)
  double bbar;    // (U - B)/sqrt(FK) = b_max - beta, formed without cancellation
  double bmax;    // lo / sqrt(FK) = e^{x/2}
  double rootFK;  // sqrt(F K)
};

__device__ __forceinline__ Norm lbr_normalise(double U, double O, double B, bool rare) {
  Norm n;
  const double d = __dsub_rn(U, O);
  const bool itm = d > 0.0;
  const double iota = itm ? d : 0.0;
  const double ub = __dsub_rn(U, B);
  const bool big = itm && (U > __dadd_rn(O, O));
  const double tv = big ? __dsub_rn(O, ub) : __dsub_rn(B, iota);   // as in the prelude
  const double lo = itm ? O : U, hi = itm ? U : O;
  const double dabs = fabs(d);
  const double FK = __dmul_rn(U, O);
  double r, rl;
  if (rare) {
    n.rootFK = __dsqrt_rn(FK);
    r = rcp_nr2(n.rootFK);
  } else {
    n.rootFK = sqrt_nr1c(FK, r);   // r to 1e-12: every quotient below carries its own residual correction; b_max is seed-grade
  }
  n.bmax = lo * r;   // seed-grade consumers only (the boundary point and the node of the seed); no residual correction
  double q = tv * r;
  n.beta = fma(fma(-n.rootFK, q, tv), r, q);
  q = ub * r;
  n.bbar = fma(fma(-n.rootFK, q, ub), r, q);
  if (rare) rl = r * rcp_nr2(n.bmax);   // ~ 1/lo, formed without inverting lo (may be subnormal)
  else rl = r * r * hi;                 // 1/lo = hi/(lo hi)
  q = dabs * rl;
  n.qrel = fma(fma(-lo, q, dabs), rl, q);
  return n;
}

struct RowOut {
  double sigma, vega;
  double s0, s1;      // total volatility of the seed and after the first Householder step (diagnostics)
  uint8_t status;
  int8_t zone;
};

// Full row (Alg.1 l.1-3).  BSM = true: (S,K,tau,r,q,P,flag); false: Black-76 with discount factor 1.
template <bool BSM, int NITER, bool FULL, bool INPLACE = false>
__device__ __forceinline__ RowOut lbr_row(double SorF, double K, double tau, double r, double q, double P, double flag) {
  RowOut o;
  Prelude p = lbr_prelude<BSM>(SorF, K, tau, r, q, P, flag);
  const bool rare = p.status == 5;
  if (rare) p = lbr_prelude_exact<BSM>(SorF, K, tau, r, q, P, flag);
  o.sigma = (p.status == 4) ? 0.0 : canonical_nan();
  o.vega = 0.0;
  o.zone = -1;
  o.s0 = o.s1 = 0.0;
  o.status = (uint8_t)p.status;
  if (p.status == 0) {
    const Norm nm = lbr_normalise(p.U, p.O, p.B, rare);
    const Seed sd = lbr_seed<FULL>(nm.qrel, nm.beta, nm.bbar, nm.bmax);
    const NormSolve ns = lbr_refine<NITER, FULL, INPLACE>(sd.x, sd.s, sd.p1, sd.p2, sd.kind);
    // as the tile kernel: MUFU.RSQ64H + one third-order step for the common rows, the library rsqrt for rare ones
    const double rinv = rare ? rsqrt(tau) : rsqrt_c3(tau);
    o.sigma = ns.s * rinv;
    o.vega = (BSM ? p.D * nm.rootFK : nm.rootFK) * ns.vfin * (tau * rinv);
    o.zone = (int8_t)sd.zone;
    o.s0 = sd.s; o.s1 = ns.s1;
  }
  return o;
}

}  // namespace pivot
