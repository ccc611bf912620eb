// oracle/lbr_oracle.hpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, scalar CPU implementation of the PIVOT hot path (arxiv/paper_2606_17065):
// price -> implied volatility by Jaeckel's "Let's Be Rational" (LBR) construction, fused
// vega + status, and the gated implicit backward rule.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may build, link or call this.  It shares
// no code, header, table or constant generator with paper_2606_17065_b200/csrc (the CUDA path).
//
// What it follows (PAPER.md = /root/reference/PAPER.md; SURVEY = /root/repo/SURVEY.md):
//   O1 normalise            PAPER.md:96 (Alg.1 l.1), :360 (A.5 stage 2), eq.(1) :47
//   O2 validity / status    PAPER.md:98 (Alg.1 l.3), :125, :363; readings 5-7 in DESIGN.md
//   O3 put-call reduction   PAPER.md:359 (A.5 stage 1), fn.2 :86
//   O4 stable b(x,s)        PAPER.md:67 eq.(4), :73 eq.(5), :361 (A.5 stage 3)
//   O5/O6 boundary + seed   PAPER.md:362 (A.5 stage 4), :111
//   O7 Householder(3)       PAPER.md:363 (A.5 stage 5), :111, :347
//   O8 sigma, vega          PAPER.md:97 (Alg.1 l.2), :322 eq.(14)
//   O9 backward + gates     PAPER.md:107 eq.(7), :131 eq.(8), :144 eq.(9), :150 eq.(10)
// The paper delegates the LBR internals to its refs [12],[17]; the formulas used
// here are the ones listed (and machine-checked) in SURVEY.md section 8(c) O4-O7; each is re-pinned
// by tests/test_oracle_*.py (finite differences, mpmath, __float128 bisection, closed forms).
//
// Notation: x = ln(F/K) = -k of the paper, reduced to x <= 0 (OTM call); s = sigma*sqrt(tau)
// (paper's sigma_tau); h = x/s; t = s/2; beta = undiscounted time value / sqrt(FK);
// b(x,s) = e^{x/2} Phi(h+t) - e^{-x/2} Phi(h-t)   (eq.(4) with k = -x);   b_max = e^{x/2} (eq.(5)).
//
// Everything is templated on the scalar type T (double = the timed fp64 oracle, long double = a
// tighter second opinion).  No blocking, fusion or reordering beyond what the formulas state.
#pragma once
#include <cfloat>
#include <cmath>
#include <cstdint>
#include <limits>

namespace lbr_oracle {

enum Status : uint8_t {
  ST_OK = 0,
  ST_BELOW_INTRINSIC = 1,
  ST_ABOVE_MAX = 2,
  ST_BAD_INPUT = 3,
  ST_AT_INTRINSIC = 4
};

// ---------------------------------------------------------------------------------------------
// Special functions.  erfcx and the inverse normal CDF are evaluated in x87 long double from
// libm's expl/erfcl/logl; no coefficient tables.
// ---------------------------------------------------------------------------------------------

// erfcx(z) = exp(z^2) erfc(z).  For z < 25 the product is formed in long double (64-bit mantissa:
// the rounding of z*z costs <= z^2 * 2^-64 <= 3.4e-17 relative); for z >= 25 the divergent
// asymptotic series erfcx(z) ~ 1/(z sqrt(pi)) * sum_k (-1)^k (2k-1)!! / (2 z^2)^k is summed to
// its k = 10 term (< 1e-23 relative at z = 25).
inline long double erfcx_ld(long double z) {
  if (z < 25.0L) return expl(z * z) * erfcl(z);
  const long double inv = 1.0L / (2.0L * z * z);
  long double term = 1.0L, sum = 1.0L;
  for (int k = 1; k <= 10; ++k) {
    term *= -(2.0L * k - 1.0L) * inv;
    sum += term;
  }
  return sum / (z * sqrtl(acosl(-1.0L)));
}

// Phi(z) = erfc(-z/sqrt2)/2 in long double.
inline long double Phi_ld(long double z) { return 0.5L * erfcl(-z / sqrtl(2.0L)); }

// Inverse normal CDF by Newton's method on ln Phi(z) = ln p (concave, so globally convergent).
inline long double ninv_ld(long double p) {
  if (!(p > 0.0L)) return -std::numeric_limits<long double>::infinity();
  if (!(p < 1.0L)) return std::numeric_limits<long double>::infinity();
  if (p > 0.5L) return -ninv_ld(1.0L - p);
  const long double lp = logl(p);
  const long double root2pi = sqrtl(2.0L * acosl(-1.0L));
  long double z = -sqrtl(-2.0L * lp);
  for (int it = 0; it < 100; ++it) {
    const long double Ph = Phi_ld(z);
    const long double ph = expl(-0.5L * z * z) / root2pi;
    const long double dz = (logl(Ph) - lp) * Ph / ph;
    z -= dz;
    if (fabsl(dz) <= 2e-19L * fabsl(z) || fabsl(dz) < 1e-40L) break;
  }
  return z;
}

template <class T> inline T erfcx_(T z) { return (T)erfcx_ld((long double)z); }
template <class T> inline T ninv_(T p) { return (T)ninv_ld((long double)p); }

template <class T> struct K {
  static T pi() { using std::acos; return acos(T(-1)); }
  static T sqrt2() { using std::sqrt; return sqrt(T(2)); }
  static T sqrt3() { using std::sqrt; return sqrt(T(3)); }
  static T phi0() { using std::sqrt; return T(1) / sqrt(T(2) * pi()); }        // 1/sqrt(2 pi)
  static T sqrt_pi_2() { using std::sqrt; return sqrt(pi() / T(2)); }          // sqrt(pi/2)
};

// Phi(z) via erfc (eq.(4)'s Phi).
template <class T> inline T Phi_(T z) { using std::erfc; return T(0.5) * erfc(-z / K<T>::sqrt2()); }

// ---------------------------------------------------------------------------------------------
// O4: the normalised Black function and its relatives, for x <= 0.
//   v(x,s)   = db/ds = phi0 * exp(-(h^2+t^2)/2)                          ("b'")
//   W(h,t)   = b / v     = w(h+t) - w(h-t),   w(z) = Phi(z)/phi(z) = sqrt(pi/2) erfcx(-z/sqrt2)
//   Wbar(h,t)= (b_max-b)/v = w(-h-t) + w(h-t)                            (complementary, no cancellation)
// ---------------------------------------------------------------------------------------------
template <class T> inline T ln_v(T h, T t) {
  using std::log;
  return log(K<T>::phi0()) - T(0.5) * (h * h + t * t);
}

// O4(iii): Taylor series in t about h,  W = 2 * sum_{j>=0} w^{(2j+1)}(h) t^{2j+1} / (2j+1)!,
// with w' = 1 + z w and w^{(n+1)} = z w^{(n)} + n w^{(n-1)}.
template <class T> inline T W_series(T h, T t, int nterms = 8) {
  const T w0 = K<T>::sqrt_pi_2() * erfcx_<T>(-h / K<T>::sqrt2());
  T wm1 = w0;            // w^{(n-1)}
  T wn = T(1) + h * w0;  // w^{(n)}, n = 1
  int n = 1;
  const T t2 = t * t;
  T tpow = t, fact = T(1);
  T sum = wn * tpow;
  for (int j = 1; j < nterms; ++j) {
    const T w2 = h * wn + T(n) * wm1;       // w^{(n+1)}
    const T w3 = h * w2 + T(n + 1) * wn;    // w^{(n+2)}
    n += 2;
    wm1 = w2;
    wn = w3;
    tpow *= t2;
    fact *= T(n - 1) * T(n);
    sum += wn * tpow / fact;
  }
  return T(2) * sum;
}

// Threshold below which the series replaces the erfcx difference (anywhere in [1e-2,1e-1]).
template <class T> inline T small_t() { return T(0.1); }

template <class T> inline T W_ratio(T h, T t) {
  if (!(t > T(0))) return T(0);
  if (t < small_t<T>()) return W_series<T>(h, t);
  // O4(ii): b = (1/2) e^{-(h^2+t^2)/2} [erfcx((|h|-t)/sqrt2) - erfcx((|h|+t)/sqrt2)],  h <= 0
  const T r2 = K<T>::sqrt2();
  return K<T>::sqrt_pi_2() * (erfcx_<T>((-h - t) / r2) - erfcx_<T>((-h + t) / r2));
}

template <class T> inline T Wbar_ratio(T h, T t) {
  const T r2 = K<T>::sqrt2();
  return K<T>::sqrt_pi_2() * (erfcx_<T>((t + h) / r2) + erfcx_<T>((t - h) / r2));
}

// b(x,s), x <= 0.  O4(i): when t - |h| is large the erfcx form overflows, so use eq.(4) directly.
template <class T> inline T norm_black(T x, T s) {
  using std::exp;
  if (!(s > T(0))) return T(0);
  const T h = (x == T(0)) ? T(0) : x / s;
  const T t = T(0.5) * s;
  if (t + h > T(10)) {
    const T bmax = exp(T(0.5) * x);
    return bmax * Phi_<T>(h + t) - Phi_<T>(h - t) / bmax;
  }
  return exp(ln_v<T>(h, t)) * W_ratio<T>(h, t);
}

template <class T> inline T norm_vega(T x, T s) {
  using std::exp;
  if (!(s > T(0))) return (x == T(0)) ? K<T>::phi0() : T(0);
  const T h = (x == T(0)) ? T(0) : x / s;
  return exp(ln_v<T>(h, T(0.5) * s));
}

// ---------------------------------------------------------------------------------------------
// O6: rational cubic interpolation on [xl, xr] (values yl, yr; slopes dl, dr; control r):
//   y(u) = [yr u^3 + (r yr - H dr) u^2 (1-u) + (r yl + H dl) u (1-u)^2 + yl (1-u)^3] / [1 + (r-3) u (1-u)]
// u and 1-u are both passed so that either end keeps full relative precision.
// ---------------------------------------------------------------------------------------------
template <class T> inline T rational_cubic(T u, T omu, T H, T yl, T yr, T dl, T dr, T r) {
  if (!(r < T(1e300))) return yr * u + yl * omu;  // r -> infinity: linear
  const T num = yr * u * u * u + (r * yr - H * dr) * u * u * omu + (r * yl + H * dl) * u * omu * omu +
                yl * omu * omu * omu;
  return num / (T(1) + (r - T(3)) * u * omu);
}

// Shape-preservation lower bound on r (monotone: (dl+dr)/Delta; convex/concave: the two ratios).
template <class T> inline T min_control(T dl, T dr, T Delta) {
  using std::fabs;
  T r = T(-1) + T(1e-9);  // r > -1 always
  if (Delta != T(0)) {
    const T r1 = (dl + dr) / Delta;
    if (r1 > r) r = r1;
  }
  if (dr != Delta) {
    const T r2 = fabs((dr - dl) / (dr - Delta));
    if (r2 > r) r = r2;
  }
  if (Delta != dl) {
    const T r3 = fabs((dr - dl) / (Delta - dl));
    if (r3 > r) r = r3;
  }
  return r;
}

// r matching a prescribed second derivative at the left / right end, floored by min_control.
template <class T> inline T control_fit_left(T H, T yl, T yr, T dl, T dr, T ddl) {
  const T Delta = (yr - yl) / H;
  const T den = Delta - dl;
  T r = (den != T(0)) ? (T(0.5) * H * ddl + (dr - dl)) / den : std::numeric_limits<T>::infinity();
  const T rmin = min_control<T>(dl, dr, Delta);
  return (r > rmin) ? r : rmin;  // NaN -> rmin
}
template <class T> inline T control_fit_right(T H, T yl, T yr, T dl, T dr, T ddr) {
  const T Delta = (yr - yl) / H;
  const T den = dr - Delta;
  T r = (den != T(0)) ? (T(0.5) * H * ddr + (dr - dl)) / den : std::numeric_limits<T>::infinity();
  const T rmin = min_control<T>(dl, dr, Delta);
  return (r > rmin) ? r : rmin;
}

// O6, zone 0 end point: f_low(s) = (2 pi |x| / (3 sqrt3)) Phi(-z)^3, z = |x|/(sqrt3 s), and its first and
// second derivative with respect to beta = b(x,s) at s:
//   f'  = 2 pi z^2 Phi(-z)^2 e^{z^2 + s^2/8}
//   f'' = (pi/6)(z^2/s^3) Phi(-z) [8 sqrt3 s |x| + (3 s^2 (s^2-8) - 8 x^2) Phi(-z)/phi(z)] e^{2 z^2 + s^2/4}
// written with Y = Phi(-z)/phi(z) = sqrt(pi/2) erfcx(z/sqrt2) so that no e^{z^2} is formed on its own.
template <class T> inline void f_low_end(T a, T s, T* f, T* d, T* dd) {
  using std::exp;
  const T phi0 = K<T>::phi0(), pi = K<T>::pi(), r3 = K<T>::sqrt3();
  const T z = a / (r3 * s);
  const T c = T(2) * pi * a / (T(3) * r3);
  const T Y = K<T>::sqrt_pi_2() * erfcx_<T>(z / K<T>::sqrt2());
  const T Phz = Y * phi0 * exp(-T(0.5) * z * z);  // Phi(-z)
  *f = c * Phz * Phz * Phz;
  *d = T(2) * pi * z * z * (Y * phi0) * (Y * phi0) * exp(s * s / T(8));
  *dd = (pi / T(6)) * (z * z / (s * s * s)) * (Y * phi0) *
        (T(8) * r3 * s * a + (T(3) * s * s * (s * s - T(8)) - T(8) * a * a) * Y) * exp(T(1.5) * z * z + s * s / T(4));
}

// O6, zone 3 end point: f_up(s) = Phi(-s/2);  f' = -e^{h^2/2}/2;  f'' = sqrt(pi/2) e^{h^2 + s^2/8} h^2/s  (w.r.t. beta).
template <class T> inline void f_up_end(T x, T s, T* f, T* d, T* dd) {
  using std::exp;
  const T h = x / s;
  *f = Phi_<T>(-T(0.5) * s);
  *d = -T(0.5) * exp(T(0.5) * h * h);
  *dd = K<T>::sqrt_pi_2() * exp(h * h + s * s / T(8)) * h * h / s;
}

// ---------------------------------------------------------------------------------------------
// Normalised problem: solve b(x,s) = beta for s, x <= 0, 0 < beta < b_max.
// bbar_beta = b_max - beta is passed separately (computed in price space, exact near the bound).
// ---------------------------------------------------------------------------------------------
template <class T> struct Seed {
  int zone;   // 0..3
  T s0;       // rational initial guess
  T sl, sc, su, bl, bc, bu;
};

template <class T> inline Seed<T> lbr_seed(T x, T beta, T bmax, T bbar_beta) {
  using std::cbrt; using std::exp; using std::fabs; using std::sqrt;
  Seed<T> sd{};
  const T a = -x;
  const T phi0 = K<T>::phi0(), pi = K<T>::pi(), r3 = K<T>::sqrt3();
  // O5: inflection point s_c = sqrt(2|x|) (there h = -t), tangent there hits 0 at s_l, b_max at s_u.
  const T sc = sqrt(T(2) * a);
  const T vc = phi0 * bmax;                       // b'(x,s_c) = phi0 e^{-|x|/2}
  const T Wc = W_ratio<T>(-T(0.5) * sc, T(0.5) * sc);
  const T bc = vc * Wc;
  const T sl = sc - bc / vc;
  const T su = sc + (bmax - bc) / vc;
  sd.sc = sc; sd.bc = bc; sd.sl = sl; sd.su = su; sd.bl = T(0); sd.bu = T(0);

  if (beta < bc) {
    if (!(sl > T(0))) {  // unreachable in exact arithmetic (s_l ~ 0.63 s_c^2 > 0); rounding guard
      sd.zone = 1;
      sd.s0 = sc * beta / bc;
      return sd;
    }
    const T bl = norm_black<T>(x, sl);
    const T vl = norm_vega<T>(x, sl);
    sd.bl = bl;
    if (beta < bl) {
      // Z0: f_low(s) = (2 pi |x| / (3 sqrt3)) Phi(-z)^3, z = |x|/(sqrt3 s); interpolate f(beta).
      sd.zone = 0;
      const T c = T(2) * pi * a / (T(3) * r3);
      T fl, d_fl, dd_fl;
      f_low_end<T>(a, sl, &fl, &d_fl, &dd_fl);
      const T r = control_fit_right<T>(bl, T(0), fl, T(1), d_fl, dd_fl);
      const T u = beta / bl;
      T f = rational_cubic<T>(u, T(1) - u, bl, T(0), fl, T(1), d_fl, r);
      if (!(f > T(0))) f = (fl * u + bl * (T(1) - u)) * u;
      T pz = cbrt(f / c);
      if (!(pz < T(0.5))) pz = T(0.5);
      const T zi = -ninv_<T>(pz);
      sd.s0 = (zi > T(0)) ? a / (r3 * zi) : sl;
    } else {
      // Z1: s(beta) through (b_l, s_l, 1/v_l), (b_c, s_c, 1/v_c), s'' = 0 at the right end.
      sd.zone = 1;
      const T H = bc - bl;
      const T r = control_fit_right<T>(H, sl, sc, T(1) / vl, T(1) / vc, T(0));
      const T u = (beta - bl) / H;
      sd.s0 = rational_cubic<T>(u, (bc - beta) / H, H, sl, sc, T(1) / vl, T(1) / vc, r);
    }
  } else {
    const T bu = norm_black<T>(x, su);
    const T vu = norm_vega<T>(x, su);
    sd.bu = bu;
    if (beta <= bu) {
      // Z2: s(beta) through (b_c, s_c, 1/v_c), (b_u, s_u, 1/v_u), s'' = 0 at the left end.
      sd.zone = 2;
      const T H = bu - bc;
      const T r = control_fit_left<T>(H, sc, su, T(1) / vc, T(1) / vu, T(0));
      const T u = (beta - bc) / H;
      sd.s0 = rational_cubic<T>(u, (bu - beta) / H, H, sc, su, T(1) / vc, T(1) / vu, r);
    } else {
      // Z3: interpolate f_up(s(beta)) through (b_u, f_up(s_u)) and (b_max, 0, slope -1/2), f'' matched at the left.
      sd.zone = 3;
      T fu, d_fu, dd_fu;
      f_up_end<T>(x, su, &fu, &d_fu, &dd_fu);
      const T H = bmax - bu;
      const T r = control_fit_left<T>(H, fu, T(0), d_fu, -T(0.5), dd_fu);
      const T u = (beta - bu) / H;
      const T omu = bbar_beta / H;
      T f = rational_cubic<T>(u, omu, H, fu, T(0), d_fu, -T(0.5), r);
      if (!(f > T(0))) f = (fu * omu + T(0.5) * H * u) * omu;
      sd.s0 = -T(2) * ninv_<T>(f);
    }
  }
  return sd;
}

// O7: the zone's objective g(s) (for reference / finite-difference pins) ...
//   Z0: g = 1/ln b - 1/ln beta;   Z1, Z2, Z3 with beta <= b_max/2: g = b - beta;
//   Z3 with beta > b_max/2: g = ln((b_max - beta)/(b_max - b)).
template <class T> inline int objective_kind(int zone, T beta, T bmax) {
  if (zone == 0) return 0;
  if (zone == 3 && beta > T(0.5) * bmax) return 2;
  return 1;
}

template <class T> inline T objective_g(int kind, T x, T s, T beta, T bbar_beta) {
  using std::exp; using std::log;
  const T h = (x == T(0)) ? T(0) : x / s;
  const T t = T(0.5) * s;
  if (kind == 0) return T(1) / (ln_v<T>(h, t) + log(W_ratio<T>(h, t))) - T(1) / log(beta);
  if (kind == 2) return log(bbar_beta) - (ln_v<T>(h, t) + log(Wbar_ratio<T>(h, t)));
  return norm_black<T>(x, s) - beta;
}

// ... and the three ratios the Householder(3) step needs: nu = -g/g1, h2 = g2/g1, h3 = g3/g1
// (g1, g2, g3 = first, second, third derivative of g in s).
template <class T>
inline void householder_terms(int kind, T x, T s, T beta, T bbar_beta, T* nu_, T* h2_, T* h3_) {
  using std::exp; using std::log;
  const T h = (x == T(0)) ? T(0) : x / s;
  const T t = T(0.5) * s;
  const T B2 = h * h / s - s / T(4);                               // b''/b'
  const T B3 = B2 * B2 - T(3) * (h / s) * (h / s) - T(0.25);       // b'''/b'
  T nu, h2, h3;
  if (kind == 0) {
    const T W = W_ratio<T>(h, t);
    const T L = ln_v<T>(h, t) + log(W);      // ln b
    const T lb = log(beta);
    const T u = T(1) / W;                    // b'/b
    const T lam = T(1) / L;
    nu = (lb - L) * (L / lb) / u;
    h2 = B2 - u * (T(1) + T(2) * lam);
    h3 = B3 + u * u * (T(2) + T(6) * lam * (T(1) + lam)) - T(3) * B2 * u * (T(1) + T(2) * lam);
  } else if (kind == 2) {
    const T Wb = Wbar_ratio<T>(h, t);
    const T gp = T(1) / Wb;                  // g' = b'/(b_max - b)
    nu = (ln_v<T>(h, t) + log(Wb) - log(bbar_beta)) / gp;
    h2 = B2 + gp;
    h3 = B3 + gp * (T(2) * gp + T(3) * B2);
  } else {
    const T v = exp(ln_v<T>(h, t));
    if (bbar_beta < beta) {
      // beta > b_max/2: beta - b = (b_max - b) - (b_max - beta), both terms in their complementary form (O4, O2);
      // b - beta itself would lose eps * b_max / (b_max - beta) as beta approaches b_max
      nu = Wbar_ratio<T>(h, t) - bbar_beta / v;
    } else {
      const T b = (t + h > T(10)) ? norm_black<T>(x, s) : v * W_ratio<T>(h, t);
      nu = (beta - b) / v;
    }
    h2 = B2;
    h3 = B3;
  }
  *nu_ = nu; *h2_ = h2; *h3_ = h3;
}

// One Householder(3) step: ds = nu (1 + h2 nu/2) / (1 + nu (h2 + h3 nu/6)), clamped to ds >= -s/2.
template <class T> inline T householder_step(int zone, T x, T s, T beta, T bmax, T bbar_beta) {
  T nu, h2, h3;
  householder_terms<T>(objective_kind<T>(zone, beta, bmax), x, s, beta, bbar_beta, &nu, &h2, &h3);
  T ds = nu * (T(1) + T(0.5) * h2 * nu) / (T(1) + nu * (h2 + h3 * nu / T(6)));
  if (!(ds > -T(0.5) * s)) ds = -T(0.5) * s;  // also catches NaN
  return ds;
}

template <class T> struct NormResult { T s; int zone; int iters; T s0; };

// fixed_iters > 0: exactly that many steps (GPU-like); otherwise until |ds| <= eps*s, cap 4.
template <class T>
inline NormResult<T> lbr_solve_normalised(T x, T beta, T bmax, T bbar_beta, int fixed_iters = 0) {
  using std::fabs;
  const Seed<T> sd = lbr_seed<T>(x, beta, bmax, bbar_beta);
  T s = sd.s0;
  if (!(s > T(0)) || !(s < T(1e300))) s = (sd.sc > T(0)) ? sd.sc : T(1);  // paranoia: never start at <= 0 / inf
  const int cap = fixed_iters > 0 ? fixed_iters : 4;
  int it = 0;
  for (; it < cap; ++it) {
    const T ds = householder_step<T>(sd.zone, x, s, beta, bmax, bbar_beta);
    s += ds;
    if (fixed_iters <= 0 && fabs(ds) <= std::numeric_limits<T>::epsilon() * s) { ++it; break; }
  }
  return NormResult<T>{s, sd.zone, it, sd.s0};
}

// ---------------------------------------------------------------------------------------------
// Full row: O1-O3, O8.  r,q both null => Black-76 with discount factor 1.
// ---------------------------------------------------------------------------------------------
template <class T> struct RowResult {
  T sigma, vega;
  uint8_t status;
  int zone, iters;
  T x, beta, s0;
};

template <class T> inline bool finite_(T v) { using std::isfinite; return isfinite(v); }

template <class T>
inline RowResult<T> lbr_row(T SorF, T Kk, T tau, const T* r, const T* q, T P, T flag, int fixed_iters = 0) {
  using std::exp; using std::log1p; using std::sqrt;
  RowResult<T> out{};
  const T nan = std::numeric_limits<T>::quiet_NaN();
  out.sigma = nan; out.vega = T(0); out.zone = -1; out.iters = 0; out.x = nan; out.beta = nan; out.s0 = nan;
  // O1
  T F = SorF, D = T(1), B = P;
  bool bad = !(finite_(SorF) && SorF > T(0)) || !(finite_(Kk) && Kk > T(0)) || !(finite_(tau) && tau > T(0)) ||
             !finite_(P) || !(flag == T(1) || flag == T(-1));
  if (r && q) {
    if (!finite_(*r) || !finite_(*q)) bad = true;
    if (!bad) {
      F = SorF * exp((*r - *q) * tau);
      D = exp(-(*r) * tau);
      B = P / D;
      if (!(finite_(F) && F > T(0)) || !(finite_(D) && D > T(0)) || !finite_(B)) bad = true;
    }
  }
  if (bad) { out.status = ST_BAD_INPUT; return out; }
  const T rootFK = sqrt(F * Kk);
  if (!(finite_(rootFK) && rootFK > T(0))) { out.status = ST_BAD_INPUT; return out; }
  // supported moneyness: b_max = min(F,K)/sqrt(FK) = e^{-|x|/2} >= 2^-500 (|x| <= 693); beyond it every normalised
  // price sits next to the fp64 underflow threshold (reading 17)
  if (!(((F < Kk) ? F : Kk) / rootFK >= T(0x1p-500))) { out.status = ST_BAD_INPUT; return out; }
  // O2 (exact IEEE operations only from here to the status decision)
  T iota = (flag > T(0)) ? (F - Kk) : (Kk - F);
  if (iota < T(0)) iota = T(0);
  const T U = (flag > T(0)) ? F : Kk;
  if (B < iota) { out.status = ST_BELOW_INTRINSIC; return out; }
  if (B >= U) { out.status = ST_ABOVE_MAX; return out; }
  // Time value (reading 18).  Out of the money (iota == 0) it is B itself.  In the money:
  //   max(F,K) <= 2 min(F,K): iota = F - K is exact (Sterbenz) and so is B - iota: the textbook form;
  //   max(F,K) >  2 min(F,K): iota carries half an ulp of max(F,K), which is eps e^{|x|/2} / beta relative to the time
  //     value (1e-11 at |x| = 12); but U - iota = min(F,K) holds exactly and U - B is exact (B >= iota > U/2, Sterbenz),
  //     so tv = min(F,K) - (U - B) has a single rounding at the scale of min(F,K), and beta + (b_max - beta) = b_max
  //     holds to rounding.  Pinned against the __float128 bisection by
  //     test_lbr_in_the_money_large_moneyness_against_truth.  A tv that comes out <= 0 is AT_INTRINSIC.
  const T lo = (F < Kk) ? F : Kk, hi = (F < Kk) ? Kk : F;
  const T tv = (iota > T(0) && hi > T(2) * lo) ? lo - (U - B) : B - iota;
  const T beta = tv / rootFK;
  out.beta = beta;
  if (beta < T(DBL_MIN)) { out.status = ST_AT_INTRINSIC; out.sigma = T(0); return out; }
  // O3: OTM call, x = -|ln(F/K)| (log1p of the exact difference keeps |x| accurate near the money)
  const T x = -log1p((hi - lo) / lo);
  const T bmax = lo / rootFK;              // e^{x/2}
  const T bbar_beta = (U - B) / rootFK;    // b_max - beta
  out.x = x;
  const NormResult<T> nr = lbr_solve_normalised<T>(x, beta, bmax, bbar_beta, fixed_iters);
  const T s = nr.s;
  out.zone = nr.zone; out.iters = nr.iters; out.s0 = nr.s0;
  // O8
  const T rt = sqrt(tau);
  out.sigma = s / rt;
  const T h = (x == T(0)) ? T(0) : x / s;
  out.vega = D * rootFK * K<T>::phi0() * exp(-T(0.5) * (h * h + T(0.25) * s * s)) * rt;
  out.status = ST_OK;
  return out;
}

// O9: backward rule.  mode 0 = MASK 1{|V| > floor}, mode 1 = ATTENUATE V^2/(V^2+floor^2).
// mode 2 = STRICT ("Rows outside G_tau return a zero cotangent when the upstream gradient is
// already zero, and return NaN when a loss explicitly asks for an ill-conditioned gradient"; :418 uses it with the floor
// 1e-14): on G_tau = {OK and |V| > floor} the exact sigma_bar / V, elsewhere +0 if sigma_bar == 0 else NaN.
template <class T> inline T backward_row(T gsigma, T vega, uint8_t status, T floor_, int mode) {
  using std::fabs;
  if (mode == 2) {
    if (status == ST_OK && fabs(vega) > floor_) return gsigma / vega;
    return (gsigma == T(0)) ? T(0) : std::numeric_limits<T>::quiet_NaN();
  }
  if (status != ST_OK) return T(0);
  if (mode == 0) return (fabs(vega) > floor_) ? gsigma / vega : T(0);
  const T den = vega * vega + floor_ * floor_;
  return (den > T(0)) ? gsigma * vega / den : T(0);
}

// Black price via the OTM-normalised form + intrinsic (eq.(2)/(3) rearranged).
template <class T> inline T black_price(T SorF, T Kk, T tau, const T* r, const T* q, T sigma, T flag) {
  using std::exp; using std::log1p; using std::sqrt;
  T F = SorF, D = T(1);
  if (r && q) { F = SorF * exp((*r - *q) * tau); D = exp(-(*r) * tau); }
  T iota = (flag > T(0)) ? (F - Kk) : (Kk - F);
  if (iota < T(0)) iota = T(0);
  const T lo = (F < Kk) ? F : Kk, hi = (F < Kk) ? Kk : F;
  const T x = -log1p((hi - lo) / lo);
  const T s = sigma * sqrt(tau);
  return D * (iota + sqrt(F * Kk) * norm_black<T>(x, s));
}

// eq.(14), first form: V = F e^{-r tau} phi(d1) sqrt(tau), d1 = (ln(F/K) + s^2/2)/s.
template <class T> inline T black_vega_eq14(T SorF, T Kk, T tau, const T* r, const T* q, T sigma) {
  using std::exp; using std::log; using std::sqrt;
  T F = SorF, D = T(1);
  if (r && q) { F = SorF * exp((*r - *q) * tau); D = exp(-(*r) * tau); }
  const T s = sigma * sqrt(tau);
  const T d1 = (log(F / Kk) + T(0.5) * s * s) / s;
  return F * D * K<T>::phi0() * exp(-T(0.5) * d1 * d1) * sqrt(tau);
}

// ---------------------------------------------------------------------------------------------
// the second half of eq.(8):  xi_bar = -(sigma_bar / V) dP/dxi
// at sigma = sigma_imp, with the gate of eq.(9)/(10) applied to the common factor exactly as in
// backward_row.  The paper obtains dP/dxi "by ordinary autograd through the analytic Black price
// helper"; written out, for the discounted price of eq.(2)
//   P = theta [ S e^{-q tau} Phi(theta d1) - K e^{-r tau} Phi(theta d2) ],
//   d1,2 = [ln(S/K) + (r - q) tau +- s^2/2] / s,  s = sigma sqrt(tau):
//   dP/dS   =  theta e^{-q tau} Phi(theta d1)
//   dP/dK   = -theta e^{-r tau} Phi(theta d2)
//   dP/dtau =  theta [ -q S e^{-q tau} Phi(theta d1) + r K e^{-r tau} Phi(theta d2) ] + V sigma / (2 tau)
//   dP/dr   =  theta K tau e^{-r tau} Phi(theta d2)
//   dP/dq   = -theta S tau e^{-q tau} Phi(theta d1)
// (the phi(d1), phi(d2) terms of dP/dS, dP/dK, dP/dr, dP/dq cancel through S e^{-q tau} phi(d1) =
// K e^{-r tau} phi(d2); in dP/dtau they leave V sigma / (2 tau), V = S e^{-q tau} phi(d1) sqrt(tau),
// eq.(14)).  Black-76 with D = 1 (r = q = NULL): the same with S -> F, r = q = 0; only dF, dK, dtau.
// These five formulas are pinned in tests/test_oracle_pins.py by central differences of black_price.
// ---------------------------------------------------------------------------------------------
template <class T> struct Greeks { T dS, dK, dtau, dr, dq; };

template <class T>
inline Greeks<T> black_greeks(T SorF, T Kk, T tau, const T* r, const T* q, T sigma, T flag) {
  using std::exp; using std::log; using std::sqrt;
  const T rr = (r && q) ? *r : T(0), qq = (r && q) ? *q : T(0);
  const T s = sigma * sqrt(tau);
  const T d1 = (log(SorF / Kk) + (rr - qq) * tau + T(0.5) * s * s) / s;
  const T d2 = d1 - s;
  const T th = (flag > T(0)) ? T(1) : T(-1);
  const T Dq = exp(-qq * tau), Dr = exp(-rr * tau);
  const T N1 = Phi_<T>(th * d1), N2 = Phi_<T>(th * d2);
  const T V = SorF * Dq * K<T>::phi0() * exp(-T(0.5) * d1 * d1) * sqrt(tau);
  Greeks<T> g;
  g.dS = th * Dq * N1;
  g.dK = -th * Dr * N2;
  g.dtau = th * (-qq * SorF * Dq * N1 + rr * Kk * Dr * N2) + V * sigma / (T(2) * tau);
  g.dr = (r && q) ? th * Kk * tau * Dr * N2 : T(0);    // Black-76 with D = 1 has no rate inputs
  g.dq = (r && q) ? -th * SorF * tau * Dq * N1 : T(0);
  return g;
}

// xi_bar = -(gated sigma_bar / V) dP/dxi; the gated factor is backward_row's grad_P.
template <class T>
inline Greeks<T> backward_inputs_row(T gsigma, T vega, uint8_t status, T floor_, int mode, T SorF, T Kk, T tau,
                                     const T* r, const T* q, T sigma, T flag) {
  Greeks<T> z{T(0), T(0), T(0), T(0), T(0)};
  const T gP = backward_row<T>(gsigma, vega, status, floor_, mode);
  using std::fabs;
  if (mode == 2 && !(status == ST_OK && fabs(vega) > floor_)) {  // STRICT, off the gate: every component is 0 or NaN with grad_P
    z.dS = z.dK = z.dtau = z.dr = z.dq = gP;
    if (!(r && q)) z.dr = z.dq = T(0);
    return z;
  }
  if (status != ST_OK || gP == T(0)) return z;
  const Greeks<T> g = black_greeks<T>(SorF, Kk, tau, r, q, sigma, flag);
  z.dS = -gP * g.dS; z.dK = -gP * g.dK; z.dtau = -gP * g.dtau; z.dr = -gP * g.dr; z.dq = -gP * g.dq;
  return z;
}

}  // namespace lbr_oracle
