// lbr_device.cuh -- device-side fp64 math for the fused LBR implied-volatility kernel (sm_100a).
//
// Per-row solver in normalised Black coordinates (eq.(4)-(5); :359-363 A.5 stages 1-5):
//   x = ln(F/K) reduced to x <= 0, s = sigma sqrt(tau), h = x/s, t = s/2, beta = time value / sqrt(FK),
//   b(x,s) = e^{x/2} Phi(h+t) - e^{-x/2} Phi(h-t),  b' = phi0 exp(-(h^2+t^2)/2),  b_max = e^{x/2}.
// Everything is expressed through the ratios  W = b/b'  and  Wbar = (b_max-b)/b', built on erfcx:
//   W    = sqrt(pi/2) [erfcx((|h|-t)/sqrt2) - erfcx((|h|+t)/sqrt2)]      (odd Taylor series in t for t < 0.1)
//   Wbar = sqrt(pi/2) [erfcx((t-|h|)/sqrt2) + erfcx((t+|h|)/sqrt2)]
// so the lower-tail objective needs no exp at all (ln b = ln b' + ln W) and the upper-tail objective no subtraction.
// This file shares nothing with oracle/ (the CPU checker); see DESIGN.md section 5 for the derivations.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace pivot {

// constants (correctly rounded decimal expansions)
__device__ constexpr double kInvSqrt2 = 0.70710678118654752440;   // 1/sqrt(2)
__device__ constexpr double kSqrtPiOver2 = 1.2533141373155002512;  // sqrt(pi/2)
__device__ constexpr double kSqrt2Pi = 2.5066282746310005024;      // sqrt(2 pi)
__device__ constexpr double kPhi0 = 0.39894228040143267794;        // 1/sqrt(2 pi)
__device__ constexpr double kLnPhi0 = -0.91893853320467274178;     // ln(1/sqrt(2 pi))
__device__ constexpr double kSqrt3 = 1.7320508075688772935;        // sqrt(3)
__device__ constexpr double kInvSqrt3 = 0.57735026918962576451;    // 1/sqrt(3)
__device__ constexpr double kTwoPi = 6.2831853071795864769;        // 2 pi
__device__ constexpr double kTwoPiOver3Sqrt3 = 1.2091995761561452337;  // 2 pi / (3 sqrt 3)
__device__ constexpr double kPiOver6 = 0.52359877559829887308;     // pi/6
__device__ constexpr double kSmallT = 0.1;                          // series / erfcx switch-over

enum : int { KIND_LOWER = 0, KIND_LINEAR = 1, KIND_UPPER = 2 };

__device__ __forceinline__ bool is_fin(double v) { return fabs(v) < __longlong_as_double(0x7ff0000000000000LL); }
__device__ __forceinline__ double canonical_nan() { return __longlong_as_double(0x7ff8000000000000LL); }

// W(h,t) = b/b' for h <= 0, t >= 0.
//   t < 0.1 : 2 sum_{j=0..5} w^{(2j+1)}(h) t^{2j+1}/(2j+1)!,  w(z) = Phi(z)/phi(z),  w' = 1 + z w,
//             w^{(n+1)} = z w^{(n)} + n w^{(n-1)}   (truncation < 1e-17 relative at t = 0.1)
//   else    : difference of two erfcx
__device__ __forceinline__ double W_ratio(double h, double t) {
  if (t < kSmallT) {
    const double w0 = kSqrtPiOver2 * erfcx(-h * kInvSqrt2);
    const double w1 = fma(h, w0, 1.0);
    const double w2 = fma(h, w1, w0);
    const double w3 = fma(h, w2, 2.0 * w1);
    const double w4 = fma(h, w3, 3.0 * w2);
    const double w5 = fma(h, w4, 4.0 * w3);
    const double w6 = fma(h, w5, 5.0 * w4);
    const double w7 = fma(h, w6, 6.0 * w5);
    const double w8 = fma(h, w7, 7.0 * w6);
    const double w9 = fma(h, w8, 8.0 * w7);
    const double w10 = fma(h, w9, 9.0 * w8);
    const double w11 = fma(h, w10, 10.0 * w9);
    const double t2 = t * t;
    double acc = w11 * (1.0 / 39916800.0);
    acc = fma(acc, t2, w9 * (1.0 / 362880.0));
    acc = fma(acc, t2, w7 * (1.0 / 5040.0));
    acc = fma(acc, t2, w5 * (1.0 / 120.0));
    acc = fma(acc, t2, w3 * (1.0 / 6.0));
    acc = fma(acc, t2, w1);
    return 2.0 * t * acc;
  }
  return kSqrtPiOver2 * (erfcx((-h - t) * kInvSqrt2) - erfcx((t - h) * kInvSqrt2));
}

__device__ __forceinline__ double Wbar_ratio(double h, double t) {
  return kSqrtPiOver2 * (erfcx((h + t) * kInvSqrt2) + erfcx((t - h) * kInvSqrt2));
}

// (h^2 + t^2)/2
__device__ __forceinline__ double half_sq(double h, double t) { return 0.5 * fma(h, h, t * t); }

// Rational cubic on [0,1] (Delbourgo-Gregory form), H = interval width, u and omu = 1-u both supplied.
__device__ __forceinline__ double rc_eval(double u, double omu, double H, double yl, double yr, double dl, double dr,
                                          double r) {
  if (!(r < 1e300)) return fma(yr, u, yl * omu);
  const double c2 = fma(r, yr, -H * dr), c1 = fma(r, yl, H * dl);
  const double num = fma(u * u, fma(yr, u, c2 * omu), omu * omu * fma(c1, u, yl * omu));
  return num / fma(r - 3.0, u * omu, 1.0);
}

// control parameter: fit the second derivative `dd` at the left (side = 0) or right (side = 1) end, floored by the
// monotonicity / convexity bounds
__device__ __forceinline__ double rc_control(int side, double H, double yl, double yr, double dl, double dr, double dd) {
  const double Delta = (yr - yl) / H;
  const double den = side ? (dr - Delta) : (Delta - dl);
  const double span = dr - dl;
  double r = fma(0.5 * H, dd, span) / den;  // den == 0 -> inf/NaN, handled by the max below
  double rmin = -1.0 + 1e-9;
  if (Delta != 0.0) rmin = fmax(rmin, (dl + dr) / Delta);
  if (dr != Delta) rmin = fmax(rmin, fabs(span / (dr - Delta)));
  if (Delta != dl) rmin = fmax(rmin, fabs(span / (Delta - dl)));
  if (den == 0.0) r = __longlong_as_double(0x7ff0000000000000LL);
  return (r > rmin) ? r : rmin;
}

struct NormSolve {
  double s;
  int zone;
};

// Solve b(x,s) = beta, x <= 0, 0 < beta < bmax; bbar = bmax - beta supplied exactly.  NITER Householder(3) steps.
template <int NITER>
__device__ __forceinline__ NormSolve lbr_solve(double x, double beta, double bmax, double bbar) {
  const double a = -x;
  // boundary point: inflection s_c = sqrt(2|x|) (h = -t there), tangent hits 0 at s_l and b_max at s_u
  const double sc = sqrt(2.0 * a);
  const double vc = kPhi0 * bmax;
  const double Wc = W_ratio(-0.5 * sc, 0.5 * sc);
  const double bc = vc * Wc;
  const bool lower = beta < bc;
  const double sl = sc - Wc;
  const double su = sc + (kSqrt2Pi - Wc);
  double s;
  int zone;
  if (lower && !(sl > 0.0)) {  // rounding guard, |x| below ~1e-30
    s = sc * (beta / bc);
    zone = 1;
  } else {
    // the one extra node this row needs: (s_l, b_l, v_l) or (s_u, b_u, v_u)
    const double sn = lower ? sl : su;
    const double hn = (a == 0.0) ? 0.0 : x / sn;
    const double tn = 0.5 * sn;
    const double vn = kPhi0 * exp(-half_sq(hn, tn));
    const double bn = vn * W_ratio(hn, tn);
    // interpolation data: x-range [xl,xr] in beta, values y, slopes d, second derivative dd fitted at `side`
    double xl, xr, yl, yr, dl, dr, dd;
    int side;
    if (lower) {
      if (beta < bn) {
        zone = 0;  // f_low(s) = (2 pi |x| / 3 sqrt3) Phi(-z)^3, z = |x| / (sqrt3 s), as a function of beta on [0, b_l]
        const double z = a * kInvSqrt3 / sl;
        const double Y = kSqrtPiOver2 * erfcx(z * kInvSqrt2);  // Phi(-z)/phi(z)
        const double Yp = Y * kPhi0;
        const double Phz = Yp * exp(-0.5 * z * z);
        const double sl2 = sl * sl;
        xl = 0.0; xr = bn; yl = 0.0; dl = 1.0;
        yr = kTwoPiOver3Sqrt3 * a * Phz * Phz * Phz;
        dr = kTwoPi * z * z * Yp * Yp * exp(0.125 * sl2);
        dd = kPiOver6 * (z * z / (sl2 * sl)) * Yp *
             fma(fma(3.0 * sl2, sl2 - 8.0, -8.0 * a * a), Y, 8.0 * kSqrt3 * sl * a) * exp(fma(1.5 * z, z, 0.25 * sl2));
        side = 1;
      } else {
        zone = 1;  // s(beta) on [b_l, b_c], s'' = 0 at b_c
        xl = bn; xr = bc; yl = sl; yr = sc; dl = 1.0 / vn; dr = 1.0 / vc; dd = 0.0; side = 1;
      }
    } else {
      if (beta <= bn) {
        zone = 2;  // s(beta) on [b_c, b_u], s'' = 0 at b_c
        xl = bc; xr = bn; yl = sc; yr = su; dl = 1.0 / vc; dr = 1.0 / vn; dd = 0.0; side = 0;
      } else {
        zone = 3;  // f_up(s) = Phi(-s/2) as a function of beta on [b_u, b_max]
        const double hu2 = hn * hn;
        xl = bn; xr = bmax; yl = 0.5 * erfc(tn * kInvSqrt2); yr = 0.0;
        dl = -0.5 * exp(0.5 * hu2); dr = -0.5;
        dd = kSqrtPiOver2 * exp(fma(0.125 * su, su, hu2)) * hu2 / su;
        side = 0;
      }
    }
    const double H = xr - xl;
    const double r = rc_control(side, H, yl, yr, dl, dr, dd);
    const double u = (beta - xl) / H;
    const double omu = (zone == 3) ? bbar / H : (xr - beta) / H;
    double y = rc_eval(u, omu, H, yl, yr, dl, dr, r);
    if (zone == 0) {
      if (!(y > 0.0)) y = fma(yr, u, xr * omu) * u;
      double p = cbrt(y / (kTwoPiOver3Sqrt3 * a));
      p = fmin(p, 0.5);
      const double zi = -normcdfinv(p);
      s = (zi > 0.0) ? a * kInvSqrt3 / zi : sl;
    } else if (zone == 3) {
      if (!(y > 0.0)) y = fma(yl, omu, 0.5 * H * u) * omu;
      s = -2.0 * normcdfinv(y);
    } else {
      s = y;
    }
  }
  if (!(s > 0.0) || !is_fin(s)) s = (sc > 0.0) ? sc : 1.0;

  const int kind = (zone == 0) ? KIND_LOWER : ((zone == 3 && beta > 0.5 * bmax) ? KIND_UPPER : KIND_LINEAR);
  const double ln_target = (kind == KIND_LOWER) ? log(beta) : 0.0;

#pragma unroll
  for (int it = 0; it < NITER; ++it) {
    const double rs = 1.0 / s;
    const double h = x * rs;
    const double t = 0.5 * s;
    const double hr = h * rs;
    const double B2 = fma(h, hr, -0.25 * s);               // b''/b'
    const double B3 = fma(B2, B2, fma(-3.0 * hr, hr, -0.25));  // b'''/b'
    const double E = half_sq(h, t);
    double nu, h2, h3;
    if (kind == KIND_UPPER) {
      // g = ln((b_max - beta)/(b_max - b)):  g' = 1/Wbar
      const double Wb = Wbar_ratio(h, t);
      const double gp = 1.0 / Wb;
      nu = (kLnPhi0 - E + log(Wb / bbar)) * Wb;
      h2 = B2 + gp;
      h3 = fma(gp, fma(2.0, gp, 3.0 * B2), B3);
    } else {
      const double W = W_ratio(h, t);
      if (kind == KIND_LOWER) {
        // g = 1/ln b - 1/ln beta, ln b = ln phi0 - E + ln W
        const double L = kLnPhi0 - E + log(W);
        const double lam = 1.0 / L;
        const double ub = 1.0 / W;  // b'/b
        const double k2 = fma(2.0, lam, 1.0);
        nu = (ln_target - L) * (L / ln_target) * W;
        h2 = fma(-ub, k2, B2);
        h3 = fma(ub * ub, fma(6.0 * lam, 1.0 + lam, 2.0), fma(-3.0 * B2 * ub, k2, B3));
      } else {
        // g = b - beta
        const double v = kPhi0 * exp(-E);
        nu = (beta - v * W) / v;
        h2 = B2;
        h3 = B3;
      }
    }
    double ds = nu * fma(0.5 * h2, nu, 1.0) / fma(nu, fma(h3 * (1.0 / 6.0), nu, h2), 1.0);
    if (!(ds > -0.5 * s)) ds = -0.5 * s;
    s += ds;
  }
  return NormSolve{s, zone};
}

struct RowOut {
  double sigma, vega;
  uint8_t status;
  int8_t zone;
};

// Full row (Alg.1 l.1-3).  BSM = true: (S,K,tau,r,q,P,flag); false: Black-76 with discount factor 1.
// The status decision uses only correctly rounded IEEE operations issued through intrinsics, so it cannot be
// contracted into FMAs and is bit-reproducible against any IEEE-754 implementation of the same sequence.
template <bool BSM, int NITER>
__device__ __forceinline__ RowOut lbr_row(double SorF, double K, double tau, double r, double q, double P, double flag) {
  RowOut o;
  o.sigma = canonical_nan();
  o.vega = 0.0;
  o.zone = -1;
  bool bad = !(is_fin(SorF) && SorF > 0.0) || !(is_fin(K) && K > 0.0) || !(is_fin(tau) && tau > 0.0) || !is_fin(P) ||
             !(flag == 1.0 || flag == -1.0);
  double F = SorF, D = 1.0, B = P;
  if (BSM) {
    if (!is_fin(r) || !is_fin(q)) bad = true;
    if (!bad) {
      F = __dmul_rn(SorF, exp(__dmul_rn(__dsub_rn(r, q), tau)));
      D = exp(__dmul_rn(-r, tau));
      B = __ddiv_rn(P, D);
      if (!(is_fin(F) && F > 0.0) || !(is_fin(D) && D > 0.0) || !is_fin(B)) bad = true;
    }
  }
  if (bad) { o.status = 3; return o; }
  const double rootFK = __dsqrt_rn(__dmul_rn(F, K));
  if (!(is_fin(rootFK) && rootFK > 0.0)) { o.status = 3; return o; }
  const double lo = fmin(F, K), hi = fmax(F, K);
  const double bmax = __ddiv_rn(lo, rootFK);
  if (!(bmax >= 0x1p-500)) { o.status = 3; return o; }
  const bool call = flag > 0.0;
  const double iota = fmax(call ? __dsub_rn(F, K) : __dsub_rn(K, F), 0.0);
  const double U = call ? F : K;
  if (B < iota) { o.status = 1; return o; }
  if (B >= U) { o.status = 2; return o; }
  const double tv = __dsub_rn(B, iota);
  const double beta = __ddiv_rn(tv, rootFK);
  if (beta < 2.2250738585072014e-308) { o.status = 4; o.sigma = 0.0; return o; }
  const double x = -log1p(__ddiv_rn(__dsub_rn(hi, lo), lo));
  const double bbar = __ddiv_rn(__dsub_rn(U, B), rootFK);
  const NormSolve ns = lbr_solve<NITER>(x, beta, bmax, bbar);
  const double s = ns.s;
  const double rt = sqrt(tau);
  const double h = (x == 0.0) ? 0.0 : x / s;
  o.sigma = s / rt;
  o.vega = D * rootFK * kPhi0 * exp(-half_sq(h, 0.5 * s)) * rt;
  o.status = 0;
  o.zone = (int8_t)ns.zone;
  return o;
}

}  // namespace pivot
