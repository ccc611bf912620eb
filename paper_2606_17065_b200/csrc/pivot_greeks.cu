// pivot_greeks.cu -- the "next" rows of the hot path, sm_100a:
//   pivot_iv_black_price        the smooth Black price node P_BSM(xi, sigma; theta) and its vega (eq.(2)/(3),
//                            :322 eq.(14)) -- what L_price eq.(11) and the round trip of eq.(12) evaluate;
//   pivot_iv_backward_inputs the full VJP of eq.(8): grad_P and xi_bar = -(sigma_bar/V) dP/dxi with
//                            analytic Greeks instead of autograd through a price helper, same gate as pivot_iv_backward.
// Both are streaming elementwise kernels (one thread per row, coalesced 8-byte accesses, every element touched once).
#include <cuda_runtime.h>

#include <cstdint>

#include "../../include/pivot_iv.h"
#include "lbr_device.cuh"

namespace pivot {

constexpr int kEwThreads = 256;
#ifndef PIVOT_EW_MIN_CTAS
#define PIVOT_EW_MIN_CTAS 4
#endif
#ifndef PIVOT_RT_MIN_CTAS
#define PIVOT_RT_MIN_CTAS 4
#endif

// Black price through the OTM-normalised form: P = D (intrinsic + sqrt(FK) b(x, s)), b from the same W / Wbar ratios as
// the solver (no cancellation for deep in-the-money rows).  sigma == 0 gives the discounted intrinsic value; NaN / negative
// sigma or bad inputs give NaN.
template <bool BSM>
__device__ __forceinline__ void black_row(double SorF, double K, double tau, double r, double q, double sigma, double flag,
                                          double& price, double& vega, double* d1d2 = nullptr) {
  price = canonical_nan();
  vega = canonical_nan();
  if (d1d2) *d1d2 = 0.0;
  bool bad = !pos_fin(SorF) || !pos_fin(K) || !pos_fin(tau) || !(sigma >= 0.0) || !is_fin(sigma) ||
             !(flag == 1.0 || flag == -1.0);
  double F = SorF, D = 1.0;
  if (BSM) {
    if (!is_fin(r) || !is_fin(q)) bad = true;
    if (!bad) {
      F = SorF * exp((r - q) * tau);
      D = exp(-r * tau);
      if (!pos_fin(F) || !pos_fin(D)) bad = true;
    }
  }
  const double FK = F * K;
  const double lo = fmin(F, K), hi = fmax(F, K);
  const double rootFK = (FK >= 0x1p-1000 && FK <= 0x1p1000) ? sqrt_nr2(FK) : sqrt(FK);
  if (!pos_fin(rootFK) || !(lo * 0x1p500 >= rootFK)) bad = true;   // same domain as the forward pass
  if (bad) return;
  const bool call = flag > 0.0;
  const double iota = fmax(call ? F - K : K - F, 0.0);
  const double rt = (tau >= 0x1p-1000 && tau <= 0x1p1000) ? sqrt_nr2(tau) : sqrt(tau);
  const double s = sigma * rt;
  double b = 0.0, v = 0.0;
  if (s > 0.0) {
    // b_max = lo / sqrt(FK) and qrel = (hi - lo)/lo by Newton reciprocals (as lbr_normalise: lo is never inverted)
    const double r = rcp_nr2(rootFK);
    double qq = lo * r;
    const double bmax = fma(fma(-rootFK, qq, lo), r, qq);
    const double rl = r * rcp_nr2(bmax), d = hi - lo;
    qq = d * rl;
    const double x = -log1p_fast(fma(fma(-lo, qq, d), rl, qq));
    const WEval w = eval_W<false, true>(x, s);   // table read in place: these kernels are grid-stride loops
    v = kPhi0 * exp_fast(-w.E);
    b = w.have_W ? w.Wd * v : fma(-w.Wd, v, bmax);
    if (d1d2) *d1d2 = fma(w.h, w.h, -0.25 * s * s);   // d1 d2 = h^2 - t^2 (sign of x does not matter)
  }
  price = D * fma(rootFK, b, iota);
  vega = D * rootFK * v * rt;
}

template <bool BSM>
__global__ void __launch_bounds__(kEwThreads, PIVOT_EW_MIN_CTAS)
black_price_kernel(pivot_iv_inputs in, const double* __restrict__ sigma, int64_t n, double* __restrict__ price,
                   double* __restrict__ vega) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const double r = BSM ? __ldcs(in.r + i) : 0.0, q = BSM ? __ldcs(in.q + i) : 0.0;
    double p, v;
    black_row<BSM>(__ldcs(in.S_or_F + i), __ldcs(in.K + i), __ldcs(in.tau + i), r, q, __ldcs(sigma + i),
                   __ldcs(in.flag + i), p, v);
    __stcs(price + i, p);
    if (vega) __stcs(vega + i, v);
  }
}

// Phi(z1), Phi(z2) from one erfcx pair and two exps: Phi(-|z|) = erfcx(|z|/sqrt2) exp(-z^2/2) / 2.
__device__ __forceinline__ void Phi_pair(double z1, double z2, double& P1, double& P2) {
  double e1, e2;
  erfcx_pair(fabs(z1) * kInvSqrt2, fabs(z2) * kInvSqrt2, e1, e2);
  const double t1 = 0.5 * e1 * exp_fast(-0.5 * z1 * z1), t2 = 0.5 * e2 * exp_fast(-0.5 * z2 * z2);
  P1 = (z1 < 0.0) ? t1 : 1.0 - t1;
  P2 = (z2 < 0.0) ? t2 : 1.0 - t2;
}

// Each warp walks blocks of 128 consecutive rows.  Pass 1 (all rows, coalesced): the gated common factor c = grad_P (exactly
// pivot_iv_backward's arithmetic) and the outputs of the rows that need no Greeks; the rows that do (OK, on the gate, c != 0:
// 26 % of config 4, scattered) are appended to a per-warp list in shared memory.  Pass 2 (dense over that list): the analytic
// Greeks, one listed row per lane -- in one pass they ran at ~8 of 32 lanes.
template <bool BSM, int MODE>
__global__ void __launch_bounds__(kEwThreads)
backward_inputs_kernel(pivot_iv_inputs in, const double* __restrict__ sigma, const double* __restrict__ vega,
                       const uint8_t* __restrict__ status, const double* __restrict__ gs, double floor_, int64_t n,
                       double* __restrict__ gP, double* __restrict__ gS, double* __restrict__ gK, double* __restrict__ gT,
                       double* __restrict__ gR, double* __restrict__ gQ) {
  constexpr int kBlockRows = 128, kWarps = kEwThreads / 32;
  __shared__ double c_list[kWarps][kBlockRows];
  __shared__ uint8_t i_list[kWarps][kBlockRows];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const double floor2 = __dmul_rn(floor_, floor_);
  const int64_t nblocks = (n + kBlockRows - 1) / kBlockRows;
  const int64_t wstride = (int64_t)gridDim.x * kWarps;
  for (int64_t blk = (int64_t)blockIdx.x * kWarps + warp; blk < nblocks; blk += wstride) {
    const int64_t base = blk * kBlockRows;
    int count = 0;
#pragma unroll
    for (int k = 0; k < kBlockRows / 32; ++k) {
      const int64_t i = base + k * 32 + lane;
      bool heavy = false;
      double c = 0.0;
      if (i < n) {
        const double V = __ldcs(vega + i), g = __ldcs(gs + i);
        const uint8_t st = status[i];
        bool strict_off = false;
        if (MODE == PIVOT_GATE_MASK) {
          c = ((st == PIVOT_ST_OK) && (fabs(V) > floor_)) ? __ddiv_rn(g, V) : 0.0;
        } else if (MODE == PIVOT_GATE_STRICT) {
          const bool on = (st == PIVOT_ST_OK) && (fabs(V) > floor_);
          c = on ? __ddiv_rn(g, V) : ((g == 0.0) ? 0.0 : canonical_nan());
          strict_off = !on;
        } else {
          const double den = __dadd_rn(__dmul_rn(V, V), floor2);
          c = ((st == PIVOT_ST_OK) && (den > 0.0)) ? __ddiv_rn(__dmul_rn(g, V), den) : 0.0;
        }
        heavy = !strict_off && st == PIVOT_ST_OK && c != 0.0;
        __stcs(gP + i, c);
        if (!heavy) {
          const double z = strict_off ? c : 0.0;   // 0, or NaN with grad_P under the strict contract
          __stcs(gS + i, z);
          __stcs(gK + i, z);
          __stcs(gT + i, z);
          if (BSM) {
            __stcs(gR + i, z);
            __stcs(gQ + i, z);
          }
        }
      }
      const unsigned m = __ballot_sync(0xffffffffu, heavy);
      if (heavy) {
        const int e = count + __popc(m & ((1u << lane) - 1u));
        c_list[warp][e] = c;
        i_list[warp][e] = (uint8_t)(k * 32 + lane);
      }
      count += __popc(m);
    }
    __syncwarp();
    for (int e = lane; e < count; e += 32) {
      const int64_t i = base + i_list[warp][e];
      const double c = c_list[warp][e];
      const double V = __ldcs(vega + i);
      const double S = __ldcs(in.S_or_F + i), K = __ldcs(in.K + i), tau = __ldcs(in.tau + i), sg = __ldcs(sigma + i);
      const double th = (__ldcs(in.flag + i) > 0.0) ? 1.0 : -1.0;
      const double r = BSM ? __ldcs(in.r + i) : 0.0, q = BSM ? __ldcs(in.q + i) : 0.0;
      const double s = sg * sqrt(tau);
      const double d1 = (log_fast(S / K) + (r - q) * tau + 0.5 * s * s) / s;
      const double d2 = d1 - s;
      double N1, N2;
      Phi_pair(th * d1, th * d2, N1, N2);
      const double Dq = BSM ? exp_fast(-q * tau) : 1.0, Dr = BSM ? exp_fast(-r * tau) : 1.0;
      const double a1 = th * Dq * N1, a2 = th * Dr * N2;   // dP/dS, -dP/dK
      __stcs(gS + i, -c * a1);
      __stcs(gK + i, c * a2);
      __stcs(gT + i, -c * (fma(-q * S, a1, r * K * a2) + V * sg / (2.0 * tau)));
      if (BSM) {
        __stcs(gR + i, -c * (K * tau * a2));
        __stcs(gQ + i, c * (S * tau * a1));
      }
    }
    __syncwarp();
  }
}

// ---------------------------------------------------------------------------------------------------------------
// The two PIVOT objectives as sums (eq.(11), eq.(12)).
// ---------------------------------------------------------------------------------------------------------------
// adds (a, b, c) over the CTA into out[0..2]: warp shuffles, one shared-memory hop, three fp64 atomics per CTA
__device__ __forceinline__ void block_add3(double a, double b, double c, double* __restrict__ out) {
  __shared__ double red[3][kEwThreads / 32];
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) {
    a += __shfl_down_sync(0xffffffffu, a, d);
    b += __shfl_down_sync(0xffffffffu, b, d);
    c += __shfl_down_sync(0xffffffffu, c, d);
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) { red[0][warp] = a; red[1][warp] = b; red[2][warp] = c; }
  __syncthreads();
  if (warp == 0) {
    a = (lane < kEwThreads / 32) ? red[0][lane] : 0.0;
    b = (lane < kEwThreads / 32) ? red[1][lane] : 0.0;
    c = (lane < kEwThreads / 32) ? red[2][lane] : 0.0;
#pragma unroll
    for (int d = 4; d > 0; d >>= 1) {
      a += __shfl_down_sync(0xffffffffu, a, d);
      b += __shfl_down_sync(0xffffffffu, b, d);
      c += __shfl_down_sync(0xffffffffu, c, d);
    }
    if (lane == 0) { atomicAdd(out + 0, a); atomicAdd(out + 1, b); atomicAdd(out + 2, c); }
  }
}

// eq.(11): out += { sum (P_model - P*)^2, sum |P*|, rows used };  GRAD: grad[i] = grad_scale 2 (P_model - P*) V_hat
// (0 for rows the sum skips)
template <bool BSM, bool GRAD>
__global__ void __launch_bounds__(kEwThreads, PIVOT_EW_MIN_CTAS)
loss_price_kernel(pivot_iv_inputs in, const double* __restrict__ sigma_hat, int64_t n, double* __restrict__ out,
                  double* __restrict__ grad, double grad_scale) {
  double s2 = 0.0, s1 = 0.0, cnt = 0.0;
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const double r = BSM ? __ldcs(in.r + i) : 0.0, q = BSM ? __ldcs(in.q + i) : 0.0;
    double pm, v;
    black_row<BSM>(__ldcs(in.S_or_F + i), __ldcs(in.K + i), __ldcs(in.tau + i), r, q, __ldcs(sigma_hat + i),
                   __ldcs(in.flag + i), pm, v);
    const double ps = __ldcs(in.P + i);
    double g = 0.0;
    if (is_fin(pm) && is_fin(ps)) {
      const double d = pm - ps;
      s2 = fma(d, d, s2); s1 += fabs(ps); cnt += 1.0;
      g = grad_scale * (2.0 * d * v);
    }
    if (GRAD) __stcs(grad + i, g);
  }
  block_add3(s2, s1, cnt, out);
}

// eq.(12), fused: price node P_model(sigma_hat), V_hat  ->  P~ (model price on the gate, the sentinel P* off it)  ->  the LBR
// inversion (the forward kernel's own per-row arithmetic: lbr_prelude, lbr_normalise, lbr_seed, lbr_refine)  ->  weighted
// residual and, GRAD, its gradient by eq.(17) -- one pass over the inputs, no HBM workspace.
//   MODE = PIVOT_RT_GATED: out += { sum w (sigma_rt - sigma*)^2, sum w, rows used },  w = V_hat^2 / (V_hat^2 + floor^2) (eq.(10));
//       grad[i] = grad_scale { [on the gate] w 2 (sigma_rt - sigma*) MASK(1/V_rt) V_hat  +  w'(V_hat) (sigma_rt - sigma*)^2 V_hat' },
//       w' = 2 V floor^2 / (V^2 + floor^2)^2,  V_hat' = dV/dsigma = V_hat d1 d2 / sigma_hat;  0 for rows the sum skips.
//   MODE = PIVOT_RT_NAIVE (no gate, no sentinel, no sanitisation): out += { sum (sigma_rt - sigma*)^2, rows, rows };
//       grad[i] = grad_scale STRICT(2 (sigma_rt - sigma*), V_rt; floor) V_hat -- NaN wherever the inverse channel is singular.
// Organisation: each warp walks blocks of 32 consecutive rows (grid-stride).  Pass 1 (every row, coalesced): price node, P~ and
// the status prelude of the inversion; a row the prelude finishes is accounted for at once, a row that needs the solver is
// pushed on a per-warp stack in shared memory (U, O, B, tau, sigma*, V_hat, the vomma term, row index: 64 B/row, 72 B in BSM
// mode).  As soon as the stack holds 32 rows the warp solves its top 32, one per lane: FULL warps whatever share of the rows
// solves (in a single pass the inversion ran at 16 of 32 lanes on the mixed workload); what is left is flushed after the warp's
// last block.  Warp-synchronous: no CTA barrier but the one of the final sum.
constexpr int kRtCap = 64;   // stack capacity per warp: at most 31 rows left over + one block of 32

template <bool BSM, int MODE, bool GRAD>
__global__ void __launch_bounds__(kEwThreads, PIVOT_RT_MIN_CTAS)
loss_roundtrip_kernel(pivot_iv_inputs in, const double* __restrict__ sigma_hat, const double* __restrict__ sigma_star,
                      double floor_, int64_t n, double* __restrict__ out, double* __restrict__ grad, double grad_scale) {
  constexpr int kWarps = kEwThreads / 32;
  __shared__ double qU[kWarps][kRtCap], qO[kWarps][kRtCap], qB[kWarps][kRtCap], qT[kWarps][kRtCap], qS[kWarps][kRtCap],
      qV[kWarps][kRtCap], qG[kWarps][kRtCap], qD[BSM ? kWarps : 1][BSM ? kRtCap : 1];
  __shared__ long long qI[kWarps][kRtCap];   // row index; bit 62: rare row (exact prelude), bit 61: on the gate
  double acc = 0.0, wsum = 0.0, cnt = 0.0;
  const double f2 = floor_ * floor_;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int64_t nblocks = (n + 31) >> 5;
  const int64_t wstride = (int64_t)gridDim.x * kWarps;
  int64_t blk = (int64_t)blockIdx.x * kWarps + warp;
  int count = 0;   // rows on the warp's stack (warp-uniform)
  for (;;) {
    const bool more = blk < nblocks;   // warp-uniform
    if (more) {
      // ---- pass 1: one row per lane
      const int64_t i = (blk << 5) + lane;
      blk += wstride;
      bool push = false;
      double eU = 0.0, eO = 0.0, eB = 0.0, eD = 1.0, eT = 0.0, eS = 0.0, eV = 0.0, eG = 0.0;
      long long eI = i;
      if (i < n) {
        const double r = BSM ? __ldcs(in.r + i) : 0.0, q = BSM ? __ldcs(in.q + i) : 0.0;
        const double S = __ldcs(in.S_or_F + i), K = __ldcs(in.K + i), tau = __ldcs(in.tau + i), flag = __ldcs(in.flag + i);
        const double sh = __ldcs(sigma_hat + i), ss = __ldcs(sigma_star + i);
        double pm, vh, dd;
        black_row<BSM>(S, K, tau, r, q, sh, flag, pm, vh, &dd);
        const bool usable = is_fin(pm) && is_fin(vh) && is_fin(ss);     // a non-finite sigma_hat gives a NaN price
        double g = 0.0, pt = pm;
        bool on = true;
        if (MODE == PIVOT_RT_NAIVE) {
          if (!usable) { acc += canonical_nan(); cnt += 1.0; g = canonical_nan(); }
        } else if (usable) {
          on = fabs(vh) > floor_;
          if (!on) pt = __ldcs(in.P + i);
        }
        if (usable) {
          Prelude p = lbr_prelude<BSM>(S, K, tau, r, q, pt, flag);
          const bool rare = p.status == 5;
          if (rare) p = lbr_prelude_exact<BSM>(S, K, tau, r, q, pt, flag);
          push = p.status == 0;
          if (push) {
            eU = p.U; eO = p.O; eB = p.B; eD = p.D; eT = tau; eS = ss; eV = vh;
            eI |= (rare ? (1LL << 62) : 0LL) | (on ? (1LL << 61) : 0LL);
            if (MODE == PIVOT_RT_GATED && GRAD) {
              const double den = fma(vh, vh, f2);
              const double wp = (den > 0.0) ? 2.0 * vh * f2 / (den * den) : 0.0;
              eG = wp * ((sh > 0.0) ? vh * dd / sh : 0.0);   // w'(V_hat) V_hat'
            }
          } else if (MODE == PIVOT_RT_NAIVE) {
            // the inversion stops at the prelude: sigma_rt = 0 (AT_INTRINSIC) or NaN, no usable vega
            const double d = ((p.status == 4) ? 0.0 : canonical_nan()) - ss;
            acc = fma(d, d, acc); cnt += 1.0;
            g = grad_scale * (((2.0 * d == 0.0) ? 0.0 : canonical_nan()) * vh);
          }
        }
        if (GRAD && !push) __stcs(grad + i, g);
      }
      const unsigned m = __ballot_sync(0xffffffffu, push);
      if (push) {
        const int e = count + __popc(m & ((1u << lane) - 1u));
        qU[warp][e] = eU; qO[warp][e] = eO; qB[warp][e] = eB; qT[warp][e] = eT; qS[warp][e] = eS; qV[warp][e] = eV;
        if (MODE == PIVOT_RT_GATED && GRAD) qG[warp][e] = eG;
        if (BSM) qD[warp][e] = eD;
        qI[warp][e] = eI;
      }
      count += __popc(m);
      __syncwarp();
    }
    if (count >= 32 || (!more && count > 0)) {
      // ---- pass 2: the top min(count, 32) rows of the stack, one per lane
      const int take = count < 32 ? count : 32;
      count -= take;
      if (lane < take) {
        const int e = count + lane;
        const long long ei = qI[warp][e];
        const bool rare = (ei >> 62) & 1, on = (ei >> 61) & 1;
        const int64_t i = ei & ((1LL << 61) - 1);
        const double tau = qT[warp][e], ss = qS[warp][e], vh = qV[warp][e];
        const Norm nm = lbr_normalise(qU[warp][e], qO[warp][e], qB[warp][e], rare);
        const Seed sd = lbr_seed<false>(nm.qrel, nm.beta, nm.bbar, nm.bmax);
        const NormSolve ns = lbr_refine<2, false, true>(sd.x, sd.s, sd.p1, sd.p2, sd.kind);
        const double rinv = rare ? rsqrt(tau) : rsqrt_c3(tau);   // as lbr_row
        const double sig = ns.s * rinv;
        const double veg = (BSM ? qD[warp][e] * nm.rootFK : nm.rootFK) * ns.vfin * (tau * rinv);
        const double d = sig - ss;
        double g;
        if (MODE == PIVOT_RT_NAIVE) {
          acc = fma(d, d, acc); cnt += 1.0;
          const double up = 2.0 * d;
          g = grad_scale * (((fabs(veg) > floor_) ? __ddiv_rn(up, veg) : ((up == 0.0) ? 0.0 : canonical_nan())) * vh);
        } else {
          const double v2 = vh * vh, den = v2 + f2;
          const double w = v2 / den;
          acc = fma(w * d, d, acc); wsum += w; cnt += 1.0;
          double gi = 0.0;
          if (GRAD) {
            gi = qG[warp][e] * (d * d);
            if (on && fabs(veg) > floor_) gi += w * __ddiv_rn(2.0 * d, veg) * vh;
          }
          g = grad_scale * gi;
        }
        if (GRAD) __stcs(grad + i, g);
      }
      __syncwarp();
    }
    if (!more && count == 0) break;
  }
  if (MODE == PIVOT_RT_NAIVE) wsum = cnt;
  block_add3(acc, wsum, cnt, out);
}

// Status histogram (optional diagnostics): out[k] += rows with status k, k = 0..4; out[5] += any other byte.
// 16 status bytes per load where the pointer allows it, four bytes classified at a time (bit-sliced masks + popc), one warp reduction
// in shared memory and at most six 64-bit global atomics per CTA (per warp they cost 113 us of contention at 2^26 rows).
__device__ __forceinline__ void hist_byte(unsigned st, unsigned long long (&c)[6]) {
#pragma unroll
  for (unsigned k = 0; k < 5; ++k) c[k] += (st == k) ? 1ull : 0ull;
  c[5] += (st > 4u) ? 1ull : 0ull;
}

__global__ void __launch_bounds__(kEwThreads) status_histogram_kernel(const uint8_t* __restrict__ status, int64_t n,
                                                                      unsigned long long* __restrict__ out) {
  unsigned long long c[6] = {0, 0, 0, 0, 0, 0};
  const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, nthreads = (int64_t)gridDim.x * blockDim.x;
  const int64_t head = (16 - (int64_t)(reinterpret_cast<uintptr_t>(status) & 15u)) & 15;   // bytes before the first 16-byte boundary
  const int64_t h = head < n ? head : n;
  const int64_t nvec = (n - h) / 16;
  const uint4* __restrict__ v = reinterpret_cast<const uint4*>(status + h);
  for (int64_t i = tid; i < nvec; i += nthreads) {
    const uint4 w = __ldcs(v + i);
    const unsigned words[4] = {w.x, w.y, w.z, w.w};
    unsigned p[5] = {0u, 0u, 0u, 0u, 0u};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      // bit-sliced: per byte b0, b1, b2 = the three low bits and hi = "any of bits 3..7" as one flag bit each (0x01 per byte);
      // status 0..4 = 000, 001, 010, 011, 100 with hi clear
      const unsigned w_ = words[k], m = 0x01010101u;
      const unsigned b0 = w_ & m, b1 = (w_ >> 1) & m, b2 = (w_ >> 2) & m;
      const unsigned t = (w_ >> 3) & 0x1f1f1f1fu;
      const unsigned hi = ((t + 0x7f7f7f7fu) >> 7) & m;     // t <= 0x1f per byte: no carry into the next byte
      const unsigned n12h = ~(b1 | b2 | hi), n0 = ~b0;
      p[0] += (unsigned)__popc(n0 & n12h & m);
      p[1] += (unsigned)__popc(b0 & n12h);
      p[2] += (unsigned)__popc(b1 & n0 & ~(b2 | hi));
      p[3] += (unsigned)__popc(b0 & b1 & ~(b2 | hi));
      p[4] += (unsigned)__popc(b2 & n0 & ~(b1 | hi));
    }
    const unsigned known = p[0] + p[1] + p[2] + p[3] + p[4];
#pragma unroll
    for (int b = 0; b < 5; ++b) c[b] += p[b];
    c[5] += 16u - known;
  }
  for (int64_t i = tid; i < h; i += nthreads) hist_byte(status[i], c);
  for (int64_t i = h + nvec * 16 + tid; i < n; i += nthreads) hist_byte(status[i], c);
  __shared__ unsigned long long red[6];
  if (threadIdx.x < 6) red[threadIdx.x] = 0ull;
  __syncthreads();
#pragma unroll
  for (int k = 0; k < 6; ++k) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) c[k] += __shfl_down_sync(0xffffffffu, c[k], d);
    if ((threadIdx.x & 31) == 0 && c[k]) atomicAdd(&red[k], c[k]);
  }
  __syncthreads();
  if (threadIdx.x < 6 && red[threadIdx.x]) atomicAdd(out + threadIdx.x, red[threadIdx.x]);   // six global atomics per CTA at most
}

inline int ew_blocks(int64_t n) {
  int dev = 0, sms = 0;   // per call: the current device may differ between calls (cudaDeviceGetAttribute is a cached lookup)
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) {
    (void)cudaGetLastError();
    sms = 148;
  }
  int64_t blocks = (n + kEwThreads - 1) / kEwThreads;
  const int64_t cap = (int64_t)sms * 8 * 4;  // 8 resident CTAs of 256 threads per SM, 4 waves' worth; grid-stride beyond
  return (int)(blocks < cap ? blocks : cap);
}

}  // namespace pivot

using namespace pivot;

extern "C" {

int pivot_iv_black_price(const pivot_iv_inputs* in, const double* sigma, int64_t n, double* price, double* vega,
                      pivot_iv_stream stream) {
  if (!in) return PIVOT_ERR_NULL;
  if (n < 0) return PIVOT_ERR_BAD_N;
  if ((in->r == nullptr) != (in->q == nullptr)) return PIVOT_ERR_MIXED_RQ;
  if (n == 0) return PIVOT_OK;
  if (!in->S_or_F || !in->K || !in->tau || !in->flag || !sigma || !price) return PIVOT_ERR_NULL;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  if (in->r)
    black_price_kernel<true><<<ew_blocks(n), kEwThreads, 0, st>>>(*in, sigma, n, price, vega);
  else
    black_price_kernel<false><<<ew_blocks(n), kEwThreads, 0, st>>>(*in, sigma, n, price, vega);
  return cudaGetLastError() == cudaSuccess ? PIVOT_OK : PIVOT_ERR_CUDA;
}

int pivot_iv_status_histogram(const uint8_t* status, int64_t n, unsigned long long* counts6, pivot_iv_stream stream) {
  if (n < 0) return PIVOT_ERR_BAD_N;
  if (!counts6) return PIVOT_ERR_NULL;
  if (n == 0) return PIVOT_OK;
  if (!status) return PIVOT_ERR_NULL;
  status_histogram_kernel<<<ew_blocks((n + 15) / 16), kEwThreads, 0, reinterpret_cast<cudaStream_t>(stream)>>>(status, n, counts6);
  return cudaGetLastError() == cudaSuccess ? PIVOT_OK : PIVOT_ERR_CUDA;
}

int pivot_iv_backward_inputs(const pivot_iv_inputs* in, const double* sigma, const double* vega, const uint8_t* status,
                             const double* grad_sigma, double vega_floor, int mode, int64_t n, double* grad_P,
                             double* grad_S_or_F, double* grad_K, double* grad_tau, double* grad_r, double* grad_q,
                             pivot_iv_stream stream) {
  if (!in) return PIVOT_ERR_NULL;
  if (n < 0) return PIVOT_ERR_BAD_N;
  if (mode != PIVOT_GATE_MASK && mode != PIVOT_GATE_ATTENUATE && mode != PIVOT_GATE_STRICT) return PIVOT_ERR_BAD_MODE;
  if (!(vega_floor >= 0.0)) return PIVOT_ERR_BAD_FLOOR;
  if ((in->r == nullptr) != (in->q == nullptr)) return PIVOT_ERR_MIXED_RQ;
  if (n == 0) return PIVOT_OK;
  const bool bsm = in->r != nullptr;
  if (!in->S_or_F || !in->K || !in->tau || !in->flag || !sigma || !vega || !status || !grad_sigma || !grad_P ||
      !grad_S_or_F || !grad_K || !grad_tau || (bsm && (!grad_r || !grad_q)))
    return PIVOT_ERR_NULL;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const int blocks = ew_blocks(n);
#define PIVOT_LAUNCH_BI(B, M)                                                                                         \
  backward_inputs_kernel<B, M><<<blocks, kEwThreads, 0, st>>>(*in, sigma, vega, status, grad_sigma, vega_floor, n,    \
                                                              grad_P, grad_S_or_F, grad_K, grad_tau, grad_r, grad_q)
  if (bsm) {
    if (mode == PIVOT_GATE_MASK) PIVOT_LAUNCH_BI(true, PIVOT_GATE_MASK);
    else if (mode == PIVOT_GATE_STRICT) PIVOT_LAUNCH_BI(true, PIVOT_GATE_STRICT);
    else PIVOT_LAUNCH_BI(true, PIVOT_GATE_ATTENUATE);
  } else {
    if (mode == PIVOT_GATE_MASK) PIVOT_LAUNCH_BI(false, PIVOT_GATE_MASK);
    else if (mode == PIVOT_GATE_STRICT) PIVOT_LAUNCH_BI(false, PIVOT_GATE_STRICT);
    else PIVOT_LAUNCH_BI(false, PIVOT_GATE_ATTENUATE);
  }
#undef PIVOT_LAUNCH_BI
  return cudaGetLastError() == cudaSuccess ? PIVOT_OK : PIVOT_ERR_CUDA;
}

int pivot_iv_loss_price(const pivot_iv_inputs* in, const double* sigma_hat, int64_t n, double* out3, double* grad_sigma_hat,
                        double grad_scale, pivot_iv_stream stream) {
  if (!in) return PIVOT_ERR_NULL;
  if (n < 0) return PIVOT_ERR_BAD_N;
  if ((in->r == nullptr) != (in->q == nullptr)) return PIVOT_ERR_MIXED_RQ;
  if (n == 0) return PIVOT_OK;
  if (!in->S_or_F || !in->K || !in->tau || !in->flag || !in->P || !sigma_hat || !out3) return PIVOT_ERR_NULL;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const int blocks = ew_blocks(n);
  if (in->r) {
    if (grad_sigma_hat) loss_price_kernel<true, true><<<blocks, kEwThreads, 0, st>>>(*in, sigma_hat, n, out3, grad_sigma_hat, grad_scale);
    else loss_price_kernel<true, false><<<blocks, kEwThreads, 0, st>>>(*in, sigma_hat, n, out3, nullptr, 0.0);
  } else {
    if (grad_sigma_hat) loss_price_kernel<false, true><<<blocks, kEwThreads, 0, st>>>(*in, sigma_hat, n, out3, grad_sigma_hat, grad_scale);
    else loss_price_kernel<false, false><<<blocks, kEwThreads, 0, st>>>(*in, sigma_hat, n, out3, nullptr, 0.0);
  }
  return cudaGetLastError() == cudaSuccess ? PIVOT_OK : PIVOT_ERR_CUDA;
}

int pivot_iv_loss_roundtrip(const pivot_iv_inputs* in, const double* sigma_hat, const double* sigma_star, double vega_floor,
                            int mode, int64_t n, double* out3, double* grad_sigma_hat, double grad_scale,
                            pivot_iv_stream stream) {
  if (!in) return PIVOT_ERR_NULL;
  if (n < 0) return PIVOT_ERR_BAD_N;
  if (mode != PIVOT_RT_GATED && mode != PIVOT_RT_NAIVE) return PIVOT_ERR_BAD_MODE;
  if (!(vega_floor >= 0.0)) return PIVOT_ERR_BAD_FLOOR;
  if ((in->r == nullptr) != (in->q == nullptr)) return PIVOT_ERR_MIXED_RQ;
  if (n == 0) return PIVOT_OK;
  if (!in->S_or_F || !in->K || !in->tau || !in->flag || !in->P || !sigma_hat || !sigma_star || !out3) return PIVOT_ERR_NULL;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const int blocks = ew_blocks(n);
#define PIVOT_LAUNCH_RT(B, M, G)                                                                                        \
  loss_roundtrip_kernel<B, M, G><<<blocks, kEwThreads, 0, st>>>(*in, sigma_hat, sigma_star, vega_floor, n, out3,        \
                                                                grad_sigma_hat, grad_scale)
  const bool bsm = in->r != nullptr, g = grad_sigma_hat != nullptr;
  if (mode == PIVOT_RT_GATED) {
    if (bsm) { if (g) PIVOT_LAUNCH_RT(true, PIVOT_RT_GATED, true); else PIVOT_LAUNCH_RT(true, PIVOT_RT_GATED, false); }
    else { if (g) PIVOT_LAUNCH_RT(false, PIVOT_RT_GATED, true); else PIVOT_LAUNCH_RT(false, PIVOT_RT_GATED, false); }
  } else {
    if (bsm) { if (g) PIVOT_LAUNCH_RT(true, PIVOT_RT_NAIVE, true); else PIVOT_LAUNCH_RT(true, PIVOT_RT_NAIVE, false); }
    else { if (g) PIVOT_LAUNCH_RT(false, PIVOT_RT_NAIVE, true); else PIVOT_LAUNCH_RT(false, PIVOT_RT_NAIVE, false); }
  }
#undef PIVOT_LAUNCH_RT
  return cudaGetLastError() == cudaSuccess ? PIVOT_OK : PIVOT_ERR_CUDA;
}

}  // extern "C"
