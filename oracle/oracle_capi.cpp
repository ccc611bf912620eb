// oracle/oracle_capi.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
// extern "C" drivers over lbr_oracle.hpp (double / long double) and the __float128 truth solver,
// called through ctypes by oracle/pyoracle.py.  OpenMP `parallel for` over rows (the
// timed CPU baseline is this oracle as it stands on the host's cores).
#include <omp.h>
#include <quadmath.h>

#include <cstdint>
#include <vector>

#include "lbr_oracle.hpp"

using namespace lbr_oracle;

namespace {

template <class T>
void forward_impl(int64_t n, const double* SorF, const double* Kk, const double* tau, const double* r,
                  const double* q, const double* P, const double* flag, double* sigma, double* vega,
                  uint8_t* status, int8_t* zone, int8_t* iters, double* s0, int fixed_iters, int nthreads) {
  if (nthreads <= 0) nthreads = omp_get_max_threads();
#pragma omp parallel for schedule(static) num_threads(nthreads)
  for (int64_t i = 0; i < n; ++i) {
    T rr = r ? (T)r[i] : T(0), qq = q ? (T)q[i] : T(0);
    RowResult<T> o = lbr_row<T>((T)SorF[i], (T)Kk[i], (T)tau[i], (r && q) ? &rr : nullptr,
                                (r && q) ? &qq : nullptr, (T)P[i], (T)flag[i], fixed_iters);
    sigma[i] = (double)o.sigma;
    vega[i] = (double)o.vega;
    status[i] = o.status;
    if (zone) zone[i] = (int8_t)o.zone;
    if (iters) iters[i] = (int8_t)o.iters;
    if (s0) s0[i] = (double)o.s0;
  }
}

template <class T>
void price_impl(int64_t n, const double* SorF, const double* Kk, const double* tau, const double* r,
                const double* q, const double* sig, const double* flag, double* out) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    T rr = r ? (T)r[i] : T(0), qq = q ? (T)q[i] : T(0);
    out[i] = (double)black_price<T>((T)SorF[i], (T)Kk[i], (T)tau[i], (r && q) ? &rr : nullptr,
                                    (r && q) ? &qq : nullptr, (T)sig[i], (T)flag[i]);
  }
}

// ------------------------------------------------------------------------------------------
// O-truth: the plain definition (eq.(6)): the unique sigma with
//   D * theta * [F Phi(theta d1) - K Phi(theta d2)] = P,   d1,2 = (ln(F/K) +- s^2/2)/s   (eq.(3)),
// by bisection in __float128 with Phi(z) = erfcq(-z/sqrt2)/2.  Literal eq.(3), no stable rearrangement.
// ------------------------------------------------------------------------------------------
__float128 Phi_q(__float128 z) { return 0.5Q * erfcq(-z / sqrtq(2.0Q)); }

__float128 black_literal_q(__float128 F, __float128 Kk, __float128 D, __float128 tau, __float128 sigma,
                           __float128 theta) {
  const __float128 s = sigma * sqrtq(tau);
  const __float128 lx = logq(F / Kk);
  const __float128 d1 = (lx + 0.5Q * s * s) / s, d2 = (lx - 0.5Q * s * s) / s;
  return D * theta * (F * Phi_q(theta * d1) - Kk * Phi_q(theta * d2));
}

double truth_row(double SorF, double Kk, double tau, const double* r, const double* q, double P, double flag) {
  __float128 F = SorF, D = 1.0Q;
  if (r && q) {
    F = (__float128)SorF * expq(((__float128)*r - (__float128)*q) * (__float128)tau);
    D = expq(-(__float128)*r * (__float128)tau);
  }
  const __float128 th = flag, K = Kk, T = tau, Pq = P;
  __float128 iota = th * (F - K);
  if (iota < 0) iota = 0;
  const __float128 U = (flag > 0) ? F : K;
  if (!(Pq > D * iota) || !(Pq < D * U)) return NAN;
  __float128 lo = 0.0Q, hi = 1.0Q;
  int guard = 0;
  while (black_literal_q(F, K, D, T, hi, th) < Pq && guard++ < 2000) { lo = hi; hi *= 2.0Q; }
  for (int it = 0; it < 400; ++it) {
    const __float128 mid = 0.5Q * (lo + hi);
    if (mid == lo || mid == hi) break;
    if (black_literal_q(F, K, D, T, mid, th) < Pq) lo = mid; else hi = mid;
    if (hi - lo <= 1e-32Q * hi) break;
  }
  return (double)(0.5Q * (lo + hi));
}

}  // namespace

extern "C" {

int oracle_max_threads(void) { return omp_get_max_threads(); }

// prec: 0 = double (the timed oracle), 1 = long double.
void oracle_forward(int prec, int64_t n, const double* SorF, const double* Kk, const double* tau,
                    const double* r, const double* q, const double* P, const double* flag, double* sigma,
                    double* vega, uint8_t* status, int8_t* zone, int8_t* iters, double* s0, int fixed_iters,
                    int nthreads) {
  if (prec == 0)
    forward_impl<double>(n, SorF, Kk, tau, r, q, P, flag, sigma, vega, status, zone, iters, s0, fixed_iters, nthreads);
  else
    forward_impl<long double>(n, SorF, Kk, tau, r, q, P, flag, sigma, vega, status, zone, iters, s0, fixed_iters, nthreads);
}

void oracle_backward(int64_t n, const double* gsigma, const double* vega, const uint8_t* status,
                     double vega_floor, int mode, double* gP) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) gP[i] = backward_row<double>(gsigma[i], vega[i], status[i], vega_floor, mode);
}

void oracle_black_price(int prec, int64_t n, const double* SorF, const double* Kk, const double* tau,
                        const double* r, const double* q, const double* sig, const double* flag, double* out) {
  if (prec == 0) price_impl<double>(n, SorF, Kk, tau, r, q, sig, flag, out);
  else price_impl<long double>(n, SorF, Kk, tau, r, q, sig, flag, out);
}

void oracle_vega_eq14(int64_t n, const double* SorF, const double* Kk, const double* tau, const double* r,
                      const double* q, const double* sig, double* out) {
  for (int64_t i = 0; i < n; ++i) {
    long double rr = r ? r[i] : 0, qq = q ? q[i] : 0;
    out[i] = (double)black_vega_eq14<long double>(SorF[i], Kk[i], tau[i], (r && q) ? &rr : nullptr,
                                                  (r && q) ? &qq : nullptr, sig[i]);
  }
}

void oracle_truth_iv(int64_t n, const double* SorF, const double* Kk, const double* tau, const double* r,
                     const double* q, const double* P, const double* flag, double* out) {
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t i = 0; i < n; ++i)
    out[i] = truth_row(SorF[i], Kk[i], tau[i], (r && q) ? &r[i] : nullptr, (r && q) ? &q[i] : nullptr, P[i], flag[i]);
}

// Literal eq.(3) price in __float128, rounded to double (pins black_price).
void oracle_black_literal_q(int64_t n, const double* F, const double* Kk, const double* D, const double* tau,
                            const double* sig, const double* flag, double* out) {
  for (int64_t i = 0; i < n; ++i) out[i] = (double)black_literal_q(F[i], Kk[i], D[i], tau[i], sig[i], flag[i]);
}

// ---- elementary pieces, exposed for the pins in tests/ (prec as above) ----
void oracle_erfcx(int64_t n, const double* z, double* out) { for (int64_t i = 0; i < n; ++i) out[i] = erfcx_<double>(z[i]); }
void oracle_ninv(int64_t n, const double* p, double* out) { for (int64_t i = 0; i < n; ++i) out[i] = ninv_<double>(p[i]); }

void oracle_norm_black(int prec, int64_t n, const double* x, const double* s, double* b, double* v) {
  for (int64_t i = 0; i < n; ++i) {
    if (prec == 0) { b[i] = norm_black<double>(x[i], s[i]); v[i] = norm_vega<double>(x[i], s[i]); }
    else { b[i] = (double)norm_black<long double>(x[i], s[i]); v[i] = (double)norm_vega<long double>(x[i], s[i]); }
  }
}
void oracle_W(int prec, int64_t n, const double* h, const double* t, double* W, double* Wbar) {
  for (int64_t i = 0; i < n; ++i) {
    if (prec == 0) { W[i] = W_ratio<double>(h[i], t[i]); Wbar[i] = Wbar_ratio<double>(h[i], t[i]); }
    else { W[i] = (double)W_ratio<long double>(h[i], t[i]); Wbar[i] = (double)Wbar_ratio<long double>(h[i], t[i]); }
  }
}
void oracle_W_series(int64_t n, const double* h, const double* t, int nterms, double* W) {
  for (int64_t i = 0; i < n; ++i) W[i] = W_series<double>(h[i], t[i], nterms);
}
void oracle_rational_cubic(int64_t n, const double* u, double H, double yl, double yr, double dl, double dr,
                           double r, double* out) {
  for (int64_t i = 0; i < n; ++i)
    out[i] = (double)rational_cubic<long double>(u[i], 1.0L - (long double)u[i], H, yl, yr, dl, dr, r);
}
double oracle_control_fit(int side, double H, double yl, double yr, double dl, double dr, double dd, int floor_it) {
  // floor_it = 0 returns the raw second-derivative fit (no shape floor) for the pin.
  const long double Delta = ((long double)yr - yl) / H;
  if (!floor_it) {
    if (side == 0) return (double)((0.5L * H * dd + ((long double)dr - dl)) / (Delta - dl));
    return (double)((0.5L * H * dd + ((long double)dr - dl)) / (dr - Delta));
  }
  return side == 0 ? (double)control_fit_left<long double>(H, yl, yr, dl, dr, dd)
                   : (double)control_fit_right<long double>(H, yl, yr, dl, dr, dd);
}
// zone-0 / zone-3 end-point value, slope and second derivative of the transformed seed functions (long double)
void oracle_f_low_end(double a, double s, double* out3) {
  long double f, d, dd; f_low_end<long double>(a, s, &f, &d, &dd); out3[0] = (double)f; out3[1] = (double)d; out3[2] = (double)dd;
}
void oracle_f_up_end(double x, double s, double* out3) {
  long double f, d, dd; f_up_end<long double>(x, s, &f, &d, &dd); out3[0] = (double)f; out3[1] = (double)d; out3[2] = (double)dd;
}
// normalised solve: (x <= 0, beta, bmax, bbar) -> s, zone, seed and boundary points
void oracle_solve_normalised(int prec, int64_t n, const double* x, const double* beta, const double* bmax,
                             const double* bbar, int fixed_iters, double* s, int8_t* zone, double* s0,
                             double* nodes /* n x 6: sl sc su bl bc bu, may be null */) {
  for (int64_t i = 0; i < n; ++i) {
    if (prec == 0) {
      NormResult<double> o = lbr_solve_normalised<double>(x[i], beta[i], bmax[i], bbar[i], fixed_iters);
      s[i] = o.s; zone[i] = (int8_t)o.zone; s0[i] = o.s0;
      if (nodes) { Seed<double> sd = lbr_seed<double>(x[i], beta[i], bmax[i], bbar[i]);
        double* p = nodes + 6 * i; p[0] = sd.sl; p[1] = sd.sc; p[2] = sd.su; p[3] = sd.bl; p[4] = sd.bc; p[5] = sd.bu; }
    } else {
      NormResult<long double> o = lbr_solve_normalised<long double>(x[i], beta[i], bmax[i], bbar[i], fixed_iters);
      s[i] = (double)o.s; zone[i] = (int8_t)o.zone; s0[i] = (double)o.s0;
      if (nodes) { Seed<long double> sd = lbr_seed<long double>(x[i], beta[i], bmax[i], bbar[i]);
        double* p = nodes + 6 * i; p[0] = sd.sl; p[1] = sd.sc; p[2] = sd.su; p[3] = sd.bl; p[4] = sd.bc; p[5] = sd.bu; }
    }
  }
}
// objective value and Householder ratios (long double), kind 0/1/2 as objective_kind().
void oracle_householder_terms(int64_t n, const int* kind, const double* x, const double* s, const double* beta,
                              const double* bbar, double* g, double* nu, double* h2, double* h3) {
  for (int64_t i = 0; i < n; ++i) {
    long double a, b, c;
    householder_terms<long double>(kind[i], x[i], s[i], beta[i], bbar[i], &a, &b, &c);
    g[i] = (double)objective_g<long double>(kind[i], x[i], s[i], beta[i], bbar[i]);
    nu[i] = (double)a; h2[i] = (double)b; h3[i] = (double)c;
  }
}

// prec: 0 = double, 1 = long double.  out5 = dP/dS, dP/dK, dP/dtau, dP/dr, dP/dq (n each, row-major blocks).
void oracle_black_greeks(int prec, int64_t n, const double* SorF, const double* Kk, const double* tau, const double* r,
                         const double* q, const double* sig, const double* flag, double* dS, double* dK, double* dtau,
                         double* dr, double* dq) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    if (prec == 0) {
      double rr = r ? r[i] : 0, qq = q ? q[i] : 0;
      const Greeks<double> g = black_greeks<double>(SorF[i], Kk[i], tau[i], (r && q) ? &rr : nullptr, (r && q) ? &qq : nullptr, sig[i], flag[i]);
      dS[i] = g.dS; dK[i] = g.dK; dtau[i] = g.dtau; dr[i] = g.dr; dq[i] = g.dq;
    } else {
      long double rr = r ? r[i] : 0, qq = q ? q[i] : 0;
      const Greeks<long double> g = black_greeks<long double>(SorF[i], Kk[i], tau[i], (r && q) ? &rr : nullptr, (r && q) ? &qq : nullptr, sig[i], flag[i]);
      dS[i] = (double)g.dS; dK[i] = (double)g.dK; dtau[i] = (double)g.dtau; dr[i] = (double)g.dr; dq[i] = (double)g.dq;
    }
  }
}

void oracle_backward_inputs(int64_t n, const double* gsigma, const double* vega, const uint8_t* status, double vega_floor,
                            int mode, const double* SorF, const double* Kk, const double* tau, const double* r,
                            const double* q, const double* sig, const double* flag, double* gS, double* gK, double* gtau,
                            double* gr, double* gq) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    double rr = r ? r[i] : 0, qq = q ? q[i] : 0;
    const Greeks<double> g = backward_inputs_row<double>(gsigma[i], vega[i], status[i], vega_floor, mode, SorF[i], Kk[i],
                                                        tau[i], (r && q) ? &rr : nullptr, (r && q) ? &qq : nullptr, sig[i], flag[i]);
    gS[i] = g.dS; gK[i] = g.dK; gtau[i] = g.dtau;
    if (gr) gr[i] = g.dr;
    if (gq) gq[i] = g.dq;
  }
}

// the two PIVOT objectives as plain sums.
//   eq.(11)  L_price = (1/|B|) sum_i ((P_BS(xi_i, sigma_hat_i; theta_i) - P*_i) / ((1/|B|) sum_j |P*_j|))^2
//   eq.(12)  L_rt    = (1/|B|) sum_i w_tau(V_hat_i) (JaeckelIV(P~_i) - sigma*_i)^2,   w_tau(V) = V^2/(V^2 + tau^2) (eq.(10)),
//            P~_i = model price where |V_hat_i| > tau, else the sentinel market price P*_i
// Returned as raw sums so that the caller normalises: price: out = {sum (P_model - P*)^2, sum |P*|, rows used};
// round trip: out = {sum w (sigma_rt - sigma*)^2, sum w, rows used}.  Rows whose sigma_hat or model price is not finite
// are skipped in both; rows whose round-trip inversion is not OK or whose sigma* is not finite are skipped in (12).
void oracle_loss_price(int64_t n, const double* SorF, const double* Kk, const double* tau, const double* r, const double* q,
                       const double* Pstar, const double* flag, const double* sig_hat, double* out3) {
  long double s2 = 0, s1 = 0, cnt = 0;
  for (int64_t i = 0; i < n; ++i) {
    long double rr = r ? r[i] : 0, qq = q ? q[i] : 0;
    const long double pm = black_price<long double>(SorF[i], Kk[i], tau[i], (r && q) ? &rr : nullptr, (r && q) ? &qq : nullptr,
                                                    sig_hat[i], flag[i]);
    if (!std::isfinite(sig_hat[i]) || !std::isfinite((double)pm) || !std::isfinite(Pstar[i])) continue;
    const long double d = pm - (long double)Pstar[i];
    s2 += d * d; s1 += fabsl((long double)Pstar[i]); cnt += 1;
  }
  out3[0] = (double)s2; out3[1] = (double)s1; out3[2] = (double)cnt;
}

void oracle_loss_roundtrip(int64_t n, const double* SorF, const double* Kk, const double* tau, const double* r,
                           const double* q, const double* Pstar, const double* flag, const double* sig_hat,
                           const double* sig_star, double vega_floor, double* out3) {
  long double acc = 0, wsum = 0, cnt = 0;
  for (int64_t i = 0; i < n; ++i) {
    double rr = r ? r[i] : 0, qq = q ? q[i] : 0;
    const double* pr = (r && q) ? &rr : nullptr; const double* pq = (r && q) ? &qq : nullptr;
    const double pm = black_price<double>(SorF[i], Kk[i], tau[i], pr, pq, sig_hat[i], flag[i]);
    const double vh = black_vega_eq14<double>(SorF[i], Kk[i], tau[i], pr, pq, sig_hat[i]);
    if (!std::isfinite(sig_hat[i]) || !std::isfinite(pm) || !std::isfinite(vh) || !std::isfinite(sig_star[i])) continue;
    const double pt = (std::fabs(vh) > vega_floor) ? pm : Pstar[i];
    const RowResult<double> o = lbr_row<double>(SorF[i], Kk[i], tau[i], pr, pq, pt, flag[i]);
    if (o.status != ST_OK) continue;
    const long double w = (long double)vh * vh / ((long double)vh * vh + (long double)vega_floor * vega_floor);
    const long double d = (long double)o.sigma - (long double)sig_star[i];
    acc += w * d * d; wsum += w; cnt += 1;
  }
  out3[0] = (double)acc; out3[1] = (double)wsum; out3[2] = (double)cnt;
}

// ---------------------------------------------------------------------------------------------
// Gradients of the two objectives with respect to sigma_hat, row by row (plain loops).
// eq.(11):  d/d sigma_hat_i (P_model_i - P*_i)^2 = 2 (P_model_i - P*_i) V_hat_i.
// eq.(12) per-row term T_i = w(V_hat_i) (sigma_rt_i - sigma*_i)^2, sigma_rt = IV(P~):
//   on the gate (|V_hat| > tau: P~ = P_model(sigma_hat)), by eq.(17)
//     dT/d sigma_hat = w 2 (sigma_rt - sigma*) (1/V_rt) V_hat  +  w'(V_hat) (sigma_rt - sigma*)^2 dV_hat/d sigma_hat,
//   with the inverse channel 1/V_rt under the MASK rule at the same floor (backward_row mode 0);
//   off the gate (P~ = the sentinel P*, which carries no gradient) only the w' term.
//   w'(V) = 2 V tau^2 / (V^2 + tau^2)^2,  dV/d sigma = V d1 d2 / sigma (Black vomma).
// NAIVE composition (Fig.6: no gate, no sentinel, no sanitisation): T_i = (IV(P_model) - sigma*)^2 and
//   dT/d sigma_hat = STRICT(2 (sigma_rt - sigma*), V_rt; floor) V_hat  (backward_row mode 2: NaN off the gate unless the
//   cotangent is 0); a row whose inversion returns NaN has a NaN term and a NaN gradient.
// The results are NOT normalised by |B|.  Rows skipped by the loss (non-finite sigma_hat / price / sigma*, or, gated only,
// an inversion that is not OK) have gradient 0 in the gated form.
// ---------------------------------------------------------------------------------------------
static double vomma_of(double SorF, double Kk, double tau, const double* r, const double* q, double sigma, double vh) {
  double F = SorF;
  if (r && q) F = SorF * std::exp((*r - *q) * tau);
  const double s = sigma * std::sqrt(tau);
  if (!(s > 0.0)) return 0.0;
  const double d1 = (std::log(F / Kk) + 0.5 * s * s) / s, d2 = d1 - s;
  return vh * d1 * d2 / sigma;
}

void oracle_loss_price_grad(int64_t n, const double* SorF, const double* Kk, const double* tau, const double* r, const double* q,
                            const double* Pstar, const double* flag, const double* sig_hat, double* g) {
  for (int64_t i = 0; i < n; ++i) {
    double rr = r ? r[i] : 0, qq = q ? q[i] : 0;
    const double* pr = (r && q) ? &rr : nullptr; const double* pq = (r && q) ? &qq : nullptr;
    const double pm = black_price<double>(SorF[i], Kk[i], tau[i], pr, pq, sig_hat[i], flag[i]);
    const double vh = black_vega_eq14<double>(SorF[i], Kk[i], tau[i], pr, pq, sig_hat[i]);
    g[i] = 0.0;
    if (!std::isfinite(sig_hat[i]) || !std::isfinite(pm) || !std::isfinite(Pstar[i])) continue;
    g[i] = 2.0 * (pm - Pstar[i]) * vh;
  }
}

void oracle_loss_roundtrip_grad(int64_t n, const double* SorF, const double* Kk, const double* tau, const double* r,
                                const double* q, const double* Pstar, const double* flag, const double* sig_hat,
                                const double* sig_star, double vega_floor, int naive, double* g, double* term) {
  const double nan = std::numeric_limits<double>::quiet_NaN();
  for (int64_t i = 0; i < n; ++i) {
    double rr = r ? r[i] : 0, qq = q ? q[i] : 0;
    const double* pr = (r && q) ? &rr : nullptr; const double* pq = (r && q) ? &qq : nullptr;
    const double pm = black_price<double>(SorF[i], Kk[i], tau[i], pr, pq, sig_hat[i], flag[i]);
    const double vh = black_vega_eq14<double>(SorF[i], Kk[i], tau[i], pr, pq, sig_hat[i]);
    const bool usable = std::isfinite(sig_hat[i]) && std::isfinite(pm) && std::isfinite(vh) && std::isfinite(sig_star[i]);
    g[i] = 0.0; if (term) term[i] = 0.0;
    if (naive) {
      if (!usable) { g[i] = nan; if (term) term[i] = nan; continue; }
      const RowResult<double> o = lbr_row<double>(SorF[i], Kk[i], tau[i], pr, pq, pm, flag[i]);
      const double d = o.sigma - sig_star[i];                 // NaN for status 1-3, -sigma* for AT_INTRINSIC (sigma = +0)
      if (term) term[i] = d * d;
      g[i] = backward_row<double>(2.0 * d, o.vega, o.status, vega_floor, 2) * vh;
      continue;
    }
    if (!usable) continue;
    const bool on = std::fabs(vh) > vega_floor;
    const RowResult<double> o = lbr_row<double>(SorF[i], Kk[i], tau[i], pr, pq, on ? pm : Pstar[i], flag[i]);
    if (o.status != ST_OK) continue;
    const double f2 = vega_floor * vega_floor, v2 = vh * vh;
    const double w = v2 / (v2 + f2);
    const double wp = (v2 + f2 > 0.0) ? 2.0 * vh * f2 / ((v2 + f2) * (v2 + f2)) : 0.0;
    const double d = o.sigma - sig_star[i];
    if (term) term[i] = w * d * d;
    double gi = wp * d * d * vomma_of(SorF[i], Kk[i], tau[i], pr, pq, sig_hat[i], vh);
    if (on) gi += w * backward_row<double>(2.0 * d, o.vega, o.status, vega_floor, 0) * vh;
    g[i] = gi;
  }
}

}  // extern "C"
