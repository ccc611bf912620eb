// lbr_device.cuh -- device-side fp64 math for the fused LBR implied-volatility kernel (sm_100a).
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
// lbr_seed_head (boundary point, node, zone), lbr_seed_tail0 / _tail3 (tail seeds) and lbr_refine (Householder(3) steps).
// Precision tiers: the seed and every Householder step but the last run at "seed grade" (fp32 erfcx, MUFU exp / log,
// one-Newton reciprocals); the normalisation, ln(beta), the last step and b' at the final s run at full fp64.
// exp / log / log1p / erfcx / reciprocals are this file's own, with coefficients in constant memory (gen_coeffs.py):
// no slow paths, no 64-bit immediates.  See DESIGN.md section 5.
// This file shares nothing with oracle/ (the CPU checker).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "coeffs.cuh"

namespace pivot {

// Scalar constants live in constant memory: an fp64 instruction takes a c[bank][offset] operand for free, whereas a
// 64-bit immediate costs two extra MOV/UMOV issue slots (16.6 % of all issued instructions in the v3 capture,
// profiles/r1a_forward_v3_ncu_full.md).
__constant__ double kInvSqrt2 = 0.70710678118654752440;       // 1/sqrt(2)
__constant__ double kSqrtPiOver2 = 1.2533141373155002512;      // sqrt(pi/2)
__constant__ double kSqrt2Pi = 2.5066282746310005024;          // sqrt(2 pi)
__constant__ double kPhi0 = 0.39894228040143267794;            // 1/sqrt(2 pi)
__constant__ double kLnPhi0 = -0.91893853320467274178;         // ln(1/sqrt(2 pi))
__constant__ double kSqrt3 = 1.7320508075688772935;            // sqrt(3)
__constant__ double kInvSqrt3 = 0.57735026918962576451;        // 1/sqrt(3)
__constant__ double kTwoPi = 6.2831853071795864769;            // 2 pi
__constant__ double kTwoPiOver3Sqrt3 = 1.2091995761561452337;  // 2 pi / (3 sqrt 3)
__constant__ double kPiOver6 = 0.52359877559829887308;         // pi/6
__constant__ double kLog2e = 1.4426950408889634074;            // 1/ln 2
__constant__ double kLn2 = 0.69314718055994530942;             // ln 2 (nearest double)
__constant__ double kLn2Lo = 2.3190468138462995584e-17;        // ln 2 - (double)ln 2
__constant__ double kSmallT = 0.1;                              // series / erfcx switch-over
__constant__ double kSqrt2m1 = 0.41421356237309504880;         // sqrt(2) - 1
__constant__ double kEightSqrt3 = 13.856406460551018348;       // 8 sqrt 3
__constant__ double kSeriesC[5] = {1.0 / 6.0, 1.0 / 120.0, 1.0 / 5040.0, 1.0 / 362880.0, 1.0 / 39916800.0};

enum : int { KIND_LOWER = 0, KIND_LINEAR = 1, KIND_UPPER = 2 };

__device__ __forceinline__ bool is_fin(double v) { return fabs(v) < __longlong_as_double(0x7ff0000000000000LL); }
// 0 < v < inf (false for NaN): two fp64 compares
__device__ __forceinline__ bool pos_fin(double v) { return v > 0.0 && v < __longlong_as_double(0x7ff0000000000000LL); }
__device__ __forceinline__ double canonical_nan() { return __longlong_as_double(0x7ff8000000000000LL); }

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
__device__ __forceinline__ double rcp_nr2(double x) {  // relative error ~1 ulp
  double r = rcp_nr1(x);
  r = fma(r, fma(-x, r, 1.0), r);
  return r;
}
__device__ __forceinline__ double rcp_pos(double x) { return rcp_nr2(x); }
// a/b to ~1 ulp (b normal, finite, non-zero)
__device__ __forceinline__ double div_fast(double a, double b) {
  const double r = rcp_nr2(b);
  const double q = a * r;
  return fma(fma(-b, q, a), r, q);
}

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
  const double r = rcp_nr2(den);
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
  const double r12 = rcp_pos(d1 * d2);
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

// ---- fp32-grade helpers for the seeds (relative error ~1e-6; results carried as double for range) ----
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
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(z + kErfcxCf));
  const float y = fmaf(-2.0f * kErfcxCf, r, 1.0f);
  float q = kErfcxQf[kErfcxNf];
#pragma unroll
  for (int k = kErfcxNf - 1; k >= 0; --k) q = fmaf(q, y, kErfcxQf[k]);
  return 2.0f * kErfcxCf * r * q;
}

// -Phi^-1(p) from lnp = ln p, p <= 0.345: u = sqrt(-2 ln p), z = u - R(1/(1+u)); relative error ~2e-5
__device__ __forceinline__ double ninv_tail_seed(double lnp) {
  const float u = sqrtf(__double2float_rn(-2.0 * lnp));
  float w;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(w) : "f"(1.0f + u));
  float R = kNinvR[kNinvN];
#pragma unroll
  for (int k = kNinvN - 1; k >= 0; --k) R = fmaf(R, w, kNinvR[k]);
  return (double)(u - R);
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

// sqrt(v), v >= 0, relative error ~1e-12 (MUFU.RSQ64H + one Newton step); seeds only
__device__ __forceinline__ double sqrt_nr1(double v) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(v));
  y = y * fma(-0.5 * v, y * y, 1.5);
  return (v > 0.0) ? v * y : 0.0;
}

// ---------------------------------------------------------------------------------------------------------------
// W-evaluation shared by the node stage and the Householder stages: at the point s returns
//   have_W = true : Wd = W = b/b'            (z1 >= 0, or the small-t series)
//   have_W = false: Wd = Wbar = (b_max-b)/b' (z1 < 0)
// together with h = x/s, 1/s and E = (h^2+t^2)/2.
// ---------------------------------------------------------------------------------------------------------------
struct WEval {
  double Wd, E, h, rs;
  bool have_W;
};

// SEED = true: the erfcx pair in fp32 on the FMA pipe (2e-7): enough for the node of the seed interpolant, where
// z1 = O(1) by construction (no cancellation in e1 - e2) and |h| ~ 0.8 whenever the small-t series is taken.
template <bool SEED = false>
__device__ __forceinline__ WEval eval_W(double x, double s) {
  WEval w;
  w.rs = SEED ? rcp_nr1(s) : rcp_nr2(s);
  w.h = x * w.rs;  // <= 0
  const double t = 0.5 * s;
  const double ah = -w.h;
  w.E = 0.5 * fma(w.h, w.h, t * t);
  const bool small = t < kSmallT;
  const double z1 = (ah - t) * kInvSqrt2;
  const bool neg = z1 < 0.0;
  double e1, e2;
  if (SEED) {
    e1 = (double)erfcx_seed(__double2float_rn(small ? ah * kInvSqrt2 : fabs(z1)));
    e2 = (double)erfcx_seed(__double2float_rn((ah + t) * kInvSqrt2));
  } else {
    erfcx_pair(small ? ah * kInvSqrt2 : fabs(z1), (ah + t) * kInvSqrt2, e1, e2);
  }
  w.have_W = small || !neg;
  if (small) {
    const double h = w.h;
    const double w0 = kSqrtPiOver2 * e1;
    const double w1 = fma(h, w0, 1.0);
    const double w2 = fma(h, w1, w0);
    const double w3 = fma(h, w2, 2.0 * w1);
    const double w4 = fma(h, w3, 3.0 * w2);
    const double w5 = fma(h, w4, 4.0 * w3);
    const double t2 = t * t;
    double acc = w5 * kSeriesC[1];
    if (!SEED) {   // seed grade stops at the t^5 term (t < 0.1: the next one is below 1e-8)
      const double w6 = fma(h, w5, 5.0 * w4);
      const double w7 = fma(h, w6, 6.0 * w5);
      const double w8 = fma(h, w7, 7.0 * w6);
      const double w9 = fma(h, w8, 8.0 * w7);
      const double w10 = fma(h, w9, 9.0 * w8);
      const double w11 = fma(h, w10, 10.0 * w9);
      acc = w11 * kSeriesC[4];
      acc = fma(acc, t2, w9 * kSeriesC[3]);
      acc = fma(acc, t2, w7 * kSeriesC[2]);
      acc = fma(acc, t2, w5 * kSeriesC[1]);
    }
    acc = fma(acc, t2, w3 * kSeriesC[0]);
    acc = fma(acc, t2, w1);
    w.Wd = s * acc;  // 2 t acc
  } else {
    w.Wd = kSqrtPiOver2 * (neg ? e1 + e2 : e1 - e2);
  }
  return w;
}

// sqrt(v), v > 0 normal, ~1 ulp, no slow path: MUFU.RSQ64H + two Newton steps + one residual correction
__device__ __forceinline__ double sqrt_nr2(double v) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(v));
  y = y * fma(-0.5 * v, y * y, 1.5);
  y = y * fma(-0.5 * v, y * y, 1.5);
  const double s = v * y;
  return fma(fma(-s, s, v), 0.5 * y, s);
}

// Rational cubic on [0,1] (Delbourgo-Gregory form), H = interval width, u and omu = 1-u both supplied.
// Seed-grade arithmetic: reciprocals carry ~1e-12.
__device__ __forceinline__ double rc_eval(double u, double omu, double H, double yl, double yr, double dl, double dr,
                                          double r) {
  if (!(r < 1e300)) return fma(yr, u, yl * omu);
  const double c2 = fma(r, yr, -H * dr), c1 = fma(r, yl, H * dl);
  const double num = fma(u * u, fma(yr, u, c2 * omu), omu * omu * fma(c1, u, yl * omu));
  return num * rcp_nr1(fma(r - 3.0, u * omu, 1.0));
}

// control parameter: fit the second derivative `dd` at the left (side = 0) or right (side = 1) end, floored by the
// monotonicity / convexity bounds.  rH = 1/H.
__device__ __forceinline__ double rc_control(int side, double H, double rH, double yl, double yr, double dl, double dr,
                                             double dd) {
  const double Delta = (yr - yl) * rH;
  const double dR = dr - Delta, dL = Delta - dl;
  const double rR = rcp_nr1(dR), rL = rcp_nr1(dL), rD = rcp_nr1(Delta);
  const double span = dr - dl;
  const double den = side ? dR : dL;
  double r = fma(0.5 * H, dd, span) * (side ? rR : rL);
  double rmin = -1.0 + 1e-9;
  if (Delta != 0.0) rmin = fmax(rmin, (dl + dr) * rD);
  if (dR != 0.0) rmin = fmax(rmin, fabs(span * rR));
  if (dL != 0.0) rmin = fmax(rmin, fabs(span * rL));
  if (den == 0.0) r = __longlong_as_double(0x7ff0000000000000LL);
  return (r > rmin) ? r : rmin;
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
// Everything here only has to deliver a seed good to ~1e-3 (Householder(3) is fourth order), so reciprocals and
// square roots carry ~1e-12 and the tail maps use fp32-grade exp / log / erfcx / Phi^-1 on MUFU.
// ---------------------------------------------------------------------------------------------------------------
struct SeedHead {
  int zone;        // 0: tail pending, v = (x, s_n, b_n, beta);  3: tail pending, v = (x, s_n, b_n, bbar);
                   // 1, 2: finished, v = (x, s0, beta, bbar)
  double v0, v1, v2, v3;
};

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
  const double ec = (double)erfcx_seed(__double2float_rn(small_c ? tc * kInvSqrt2 : sc * kInvSqrt2));   // seed grade (2e-7)
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
  const double bc = vc * Wc;
  const double su = sc + (kSqrt2Pi - Wc);     // ... and the tangent hits b_max at s_u
  const bool lower = beta < bc;
  o.v2 = beta; o.v3 = bbar;
  if (lower && !(sl > 0.0)) {  // rounding guard, |x| below ~1e-30: linear seed
    o.zone = 1;
    o.v1 = sc * beta * rcp_nr1(bc);
    return o;
  }
  const double sn = lower ? sl : su;
  const WEval w = eval_W<true>(x, sn);
  const double vn = kPhi0 * exp_seed(-w.E);  // b'(s_n), seed grade
  const double bn = w.have_W ? w.Wd * vn : fma(-w.Wd, vn, bmax);
  if (lower ? (beta < bn) : (beta > bn)) {   // a tail: hand the node over
    o.zone = lower ? 0 : 3;
    o.v1 = sn; o.v2 = bn; o.v3 = lower ? beta : bbar;
    return o;
  }
  // zones 1 and 2: s(beta) between the node and the inflection point, s'' = 0 at the inflection point
  o.zone = lower ? 1 : 2;
  const double inv_vn = rcp_nr1(vn), rvc = kSqrt2Pi * rcp_nr1(bmax);
  const double xl = lower ? bn : bc, xr = lower ? bc : bn;
  const double yl = lower ? sn : sc, yr = lower ? sc : sn;
  const double dl = lower ? inv_vn : rvc, dr = lower ? rvc : inv_vn;
  const double H = xr - xl, rH = rcp_nr1(H);
  const double r = rc_control(lower ? 1 : 0, H, rH, yl, yr, dl, dr, 0.0);
  const double s = rc_eval((beta - xl) * rH, (xr - beta) * rH, H, yl, yr, dl, dr, r);
  o.v1 = (s > 0.0 && is_fin(s)) ? s : sc;   // a failed interpolant falls back to the inflection point
  return o;
}

struct Seed {
  double x, s, p1, p2;
  int kind, zone;
};

// zone 0: f_low(s) = (2 pi |x| / 3 sqrt3) Phi(-z)^3, z = |x| / (sqrt3 s), as a function of beta on [0, b_l]
__device__ __forceinline__ Seed lbr_seed_tail0(double x, double sn, double bn, double beta) {
  const double a = -x;
  const double rs = rcp_nr1(sn);
  const double z = a * rs * kInvSqrt3;
  const double Y = kSqrtPiOver2 * (double)erfcx_seed(__double2float_rn(z * kInvSqrt2));  // Phi(-z)/phi(z)
  const double Yp = Y * kPhi0;
  const double A = exp_seed(-0.5 * z * z), B = exp_seed(0.125 * sn * sn);
  const double Phz = Yp * A;
  const double sn2 = sn * sn;
  const double rA = rcp_nr1(A);
  const double yr = kTwoPiOver3Sqrt3 * a * Phz * Phz * Phz;
  const double dr = kTwoPi * z * z * Yp * Yp * B;
  const double dd = kPiOver6 * (z * z * rs * rs * rs) * Yp *
                    fma(fma(3.0 * sn2, sn2 - 8.0, -8.0 * a * a), Y, kEightSqrt3 * sn * a) * (B * B) * (rA * rA * rA);
  const double H = bn, rH = rcp_nr1(bn);
  const double r = rc_control(1, H, rH, 0.0, yr, 1.0, dr, dd);
  const double u = beta * rH, omu = (bn - beta) * rH;
  double y = rc_eval(u, omu, H, 0.0, yr, 1.0, dr, r);
  if (!(y > 0.0)) y = fma(yr, u, bn * omu) * u;
  // Phi(-z) = (f/c)^{1/3}  ->  ln p = ln(f/c)/3
  const double lnp = fmin(log_seed(y * rcp_nr1(kTwoPiOver3Sqrt3 * a)) * (1.0 / 3.0), -1.0651);
  double s = a * kInvSqrt3 * rcp_nr1(ninv_tail_seed(lnp));
  if (!(s > 0.0) || !is_fin(s)) s = sn;
  Seed o;
  o.x = x; o.s = s; o.zone = 0;
  o.kind = KIND_LOWER; o.p1 = log_fast(beta); o.p2 = 0.0;   // b_max = e^{x/2} is rebuilt by lbr_refine if ever needed
  return o;
}

// zone 3: f_up(s) = Phi(-s/2) as a function of beta on [b_u, b_max]
__device__ __forceinline__ Seed lbr_seed_tail3(double x, double sn, double bn, double bbar) {
  const double bmax = exp_fast(0.5 * x);   // e^{x/2} (the handover carries four words: beta = b_max - bbar)
  const double beta = bmax - bbar;
  const double rs = rcp_nr1(sn);
  const double h = x * rs;
  const double hu2 = h * h;
  const double tn = 0.5 * sn;
  const double A = exp_seed(0.5 * hu2), B = exp_seed(0.125 * sn * sn);
  const double yl = 0.5 * (double)erfcx_seed(__double2float_rn(tn * kInvSqrt2)) * rcp_nr1(B);  // Phi(-t)
  const double dl = -0.5 * A;
  const double dd = kSqrtPiOver2 * (A * A) * B * hu2 * rs;
  const double H = bmax - bn, rH = rcp_nr1(H);
  const double r = rc_control(0, H, rH, yl, 0.0, dl, -0.5, dd);
  const double u = (beta - bn) * rH, omu = bbar * rH;
  double y = rc_eval(u, omu, H, yl, 0.0, dl, -0.5, r);
  if (!(y > 0.0)) y = fma(yl, omu, 0.5 * H * u) * omu;
  double s = 2.0 * ninv_tail_seed(fmin(log_seed(y), -1.0651));
  if (!(s > 0.0) || !is_fin(s)) s = sn;
  Seed o;
  o.x = x; o.s = s; o.zone = 3;
  if (bbar < 0.5 * bmax) {
    o.kind = KIND_UPPER; o.p1 = log_fast(bbar); o.p2 = 0.0;
  } else {
    o.kind = KIND_LINEAR; o.p1 = beta; o.p2 = bbar;
  }
  return o;
}

// one-call form (row-per-thread kernel)
__device__ __forceinline__ Seed lbr_seed(double qrel, double beta, double bbar, double bmax) {
  const SeedHead hd = lbr_seed_head(qrel, beta, bbar, bmax);
  if (hd.zone == 0) return lbr_seed_tail0(hd.v0, hd.v1, hd.v2, hd.v3);
  if (hd.zone == 3) return lbr_seed_tail3(hd.v0, hd.v1, hd.v2, hd.v3);
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
  double vfin;  // b'(x, s) at that s
};

// One Householder(3) step.  SEED = true evaluates W, exp and log at seed grade (fp32 erfcx pair, MUFU exp / log,
// ~1e-6 relative in the step): enough for every step but the last, because the step is fourth order and the last step
// then takes an iterate that is good to ~1e-6 to ~1e-24.
template <bool SEED>
__device__ __forceinline__ double householder_step(double x, double s, double p1, double p2, int kind) {
  const WEval w = eval_W<SEED>(x, s);
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
      const double rLW = (SEED ? rcp_nr1(L * R) : rcp_nr2(L * R));
      const double lam = rLW * R, ub = rLW * L;  // 1/L, b'/b = 1/W
      const double k2 = fma(2.0, lam, 1.0);
      nu = (p1 - L) * (L * (SEED ? rcp_nr1(p1) : rcp_nr2(p1))) * R;
      h2 = fma(-ub, k2, B2);
      h3 = fma(ub * ub, fma(6.0 * lam, 1.0 + lam, 2.0), fma(-3.0 * B2 * ub, k2, B3));
    } else {
      // g = ln((b_max - beta)/(b_max - b)):  g' = 1/Wbar  (p1 = ln(b_max - beta))
      const double gp = SEED ? rcp_nr1(R) : rcp_nr2(R);
      nu = (L - p1) * R;
      h2 = B2 + gp;
      h3 = fma(gp, fma(2.0, gp, 3.0 * B2), B3);
    }
  }
  const double den = fma(nu, fma(h3 * (1.0 / 6.0), nu, h2), 1.0);
  double ds = nu * fma(0.5 * h2, nu, 1.0) * (SEED ? rcp_nr1(den) : rcp_nr2(den));
  if (!(ds > -0.5 * s)) ds = -0.5 * s;
  return s + ds;
}

template <int NITER>
__device__ __forceinline__ NormSolve lbr_refine(double x, double s, double p1, double p2, int kind) {
#pragma unroll 1
  for (int it = 0; it < NITER - 1; ++it) s = householder_step<true>(x, s, p1, p2, kind);
  s = householder_step<false>(x, s, p1, p2, kind);
  const double rs = rcp_nr2(s);
  const double h = x * rs, t = 0.5 * s;
  NormSolve o;
  o.s = s;
  o.vfin = kPhi0 * exp_fast(-0.5 * fma(h, h, t * t));
  return o;
}

// one-call form (row-per-thread kernel): seed + refine
template <int NITER>
__device__ __forceinline__ NormSolve lbr_solve(double qrel, double beta, double bmax, double bbar, int& zone) {
  const Seed sd = lbr_seed(qrel, beta, bbar, bmax);
  zone = sd.zone;
  return lbr_refine<NITER>(sd.x, sd.s, sd.p1, sd.p2, sd.kind);
}

// Row prelude (Alg.1 l.1 and l.3; A.5 stages 1-2): validity and status for EVERY row, with no division:
//   beta = RN(tv / rootFK) < DBL_MIN   <=>   tv * 2^1022 < rootFK     (exact: the scaling is exact, and for doubles
//   bmax = RN(lo / rootFK) >= 2^-500   <=>   lo * 2^500 >= rootFK      a < b implies a <= b - ulp(b) < b (1 - 2^-53))
// so the status byte equals the one obtained from the correctly rounded quotients, bit for bit, and rows that leave
// here (57.8 % of config 1/4) cost no division (a zero numerator would even take the divide's slow path).
// The status decision uses only correctly rounded IEEE operations issued through intrinsics, so it cannot be
// contracted into FMAs and is bit-reproducible against any IEEE-754 implementation of the same sequence.
struct Prelude {
  double F;       // forward (BSM: S e^{(r-q) tau})
  double B;       // undiscounted price (BSM: P / D)
  double rootFK;  // sqrt(F K)
  double scale;   // D sqrt(FK): vega = scale * b'(x,s) * sqrt(tau)
  int status;
  bool call;
};

template <bool BSM>
__device__ __forceinline__ Prelude lbr_prelude(double SorF, double K, double tau, double r, double q, double P,
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
  p.F = F;
  p.B = B;
  p.rootFK = rootFK;
  p.scale = BSM ? D * rootFK : rootFK;
  p.call = call;
  return p;
}

// Normalised solver inputs of a row that reached the solver (A.5 stage 2).  Quotients by Newton
// reciprocal + one residual correction (~1 ulp, no slow path): sqrt(FK) lies in [2^-537, 2^512] and b_max in
// [2^-500, 1], so the MUFU reciprocal seeds never leave the normal range; lo itself is never inverted.
struct Norm {
  double qrel;    // (hi - lo)/lo, hi = max(F,K), lo = min(F,K):  x = -log1p(qrel)
  double beta;    // time value / sqrt(FK)
  double bbar;    // (U - B)/sqrt(FK) = b_max - beta, formed without cancellation
  double bmax;    // lo / sqrt(FK) = e^{x/2}
};

__device__ __forceinline__ Norm lbr_normalise(double F, double K, double B, double rootFK, bool call) {
  Norm n;
  const double lo = fmin(F, K), hi = fmax(F, K);
  const double iota = fmax(call ? __dsub_rn(F, K) : __dsub_rn(K, F), 0.0);
  const double U = call ? F : K;
  const double ub = __dsub_rn(U, B), d = __dsub_rn(hi, lo);
  const double tv = (iota > 0.0 && hi > __dmul_rn(2.0, lo)) ? __dsub_rn(lo, ub) : __dsub_rn(B, iota);  // as in lbr_prelude
  const double r = rcp_nr2(rootFK);
  double q = lo * r;
  n.bmax = fma(fma(-rootFK, q, lo), r, q);
  q = tv * r;
  n.beta = fma(fma(-rootFK, q, tv), r, q);
  q = ub * r;
  n.bbar = fma(fma(-rootFK, q, ub), r, q);
  const double rl = r * rcp_nr2(n.bmax);  // ~ 1/lo, formed without inverting lo
  q = d * rl;
  n.qrel = fma(fma(-lo, q, d), rl, q);
  return n;
}

struct RowOut {
  double sigma, vega;
  uint8_t status;
  int8_t zone;
};

// Full row (Alg.1 l.1-3).  BSM = true: (S,K,tau,r,q,P,flag); false: Black-76 with discount factor 1.
template <bool BSM, int NITER>
__device__ __forceinline__ RowOut lbr_row(double SorF, double K, double tau, double r, double q, double P, double flag) {
  RowOut o;
  const Prelude p = lbr_prelude<BSM>(SorF, K, tau, r, q, P, flag);
  o.sigma = (p.status == 4) ? 0.0 : canonical_nan();
  o.vega = 0.0;
  o.zone = -1;
  o.status = (uint8_t)p.status;
  if (p.status == 0) {
    int zone;
    const Norm nm = lbr_normalise(p.F, K, p.B, p.rootFK, p.call);
    const NormSolve ns = lbr_solve<NITER>(nm.qrel, nm.beta, nm.bmax, nm.bbar, zone);
    const double rinv = rsqrt(tau);
    o.sigma = ns.s * rinv;
    o.vega = p.scale * ns.vfin * (tau * rinv);
    o.zone = (int8_t)zone;
  }
  return o;
}

}  // namespace pivot
