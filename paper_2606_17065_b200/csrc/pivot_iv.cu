// pivot_iv.cu -- kernels and C ABI (include/pivot_iv.h) of the PIVOT implied-volatility hot path, sm_100a.
//
// Forward: one fused kernel; every intermediate of the per-row LBR solve lives in registers or shared memory, HBM is
// touched once per element (57 B/row Black-76, 73 B/row BSM).  Two organisations of the same per-row arithmetic:
// forward_kernel_tile (rows compacted and regrouped by LBR zone in shared memory; the default) and
// forward_kernel_scalar (one row per thread).  Backward: one streaming elementwise kernel (25 B/row).
// No tensor cores: the path is an fp64 transcendental chain, not a contraction.
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <new>

#include "../../include/pivot_iv.h"
#include "lbr_device.cuh"

namespace pivot {

constexpr int kFwdThreads = 128;
constexpr int kBwdThreads = 256;
constexpr int kHouseholderSteps = 2;  // north_star: two Householder(3) steps

// ---------------------------------------------------------------------------------------------------------------
// Forward kernel, one row per thread (PIVOT_FWD_ROWWISE): no shared memory, no barriers; coalesced 8-byte accesses.
// Best when nearly every row solves and neighbouring rows are alike (option chains in strike order).
// ---------------------------------------------------------------------------------------------------------------
template <bool BSM, bool ZONES>
__device__ __forceinline__ void solve_and_store(int64_t i, double S, double K, double tau, double r, double q, double P,
                                                double flag, double* __restrict__ sigma, double* __restrict__ vega,
                                                uint8_t* __restrict__ status, int8_t* __restrict__ zone) {
  const RowOut o = lbr_row<BSM, kHouseholderSteps>(S, K, tau, r, q, P, flag);
  __stcs(sigma + i, o.sigma);
  __stcs(vega + i, o.vega);
  status[i] = o.status;
  if (ZONES) zone[i] = o.zone;
}

// SEL = false: one launch covers the rows (grid = ceil(n / 128)).  SEL = true (pivot_iv_forward_auto): small grid-stride
// grid that first reads the probe's decision and returns at once when the other organisation was chosen.
template <bool BSM, bool ZONES, bool SEL = false>
__global__ void __launch_bounds__(kFwdThreads)
forward_kernel_scalar(pivot_iv_inputs in, int64_t begin, int64_t n, double* __restrict__ sigma,
                      double* __restrict__ vega, uint8_t* __restrict__ status, int8_t* __restrict__ zone,
                      const int* __restrict__ sel, int want) {
  if (SEL) {
    if (*sel != want) return;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = begin + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
      const double r = BSM ? __ldcs(in.r + i) : 0.0, q = BSM ? __ldcs(in.q + i) : 0.0;
      solve_and_store<BSM, ZONES>(i, __ldcs(in.S_or_F + i), __ldcs(in.K + i), __ldcs(in.tau + i), r, q, __ldcs(in.P + i),
                                  __ldcs(in.flag + i), sigma, vega, status, zone);
    }
  } else {
    const int64_t i = begin + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double r = BSM ? __ldcs(in.r + i) : 0.0, q = BSM ? __ldcs(in.q + i) : 0.0;
    solve_and_store<BSM, ZONES>(i, __ldcs(in.S_or_F + i), __ldcs(in.K + i), __ldcs(in.tau + i), r, q, __ldcs(in.P + i),
                                __ldcs(in.flag + i), sigma, vega, status, zone);
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Forward kernel, "tile compaction".  A CTA owns a tile of kTileRows consecutive rows.
//   Phase A  (all rows, coalesced 8-byte loads): prelude -> status, with exact IEEE operations and no division.  Rows
//            that need the solver are appended to a compact queue in shared memory (one warp prefix scan and one shared
//            atomic per warp per tile); the others get their final sigma / vega straight away.  For queued rows the
//            staged output slots carry tau and D sqrt(FK) meanwhile.
//   Phase B1 (queued rows, DENSE warps): lbr_normalise + lbr_seed_head: x, boundary point, node, zone; the middle zones
//            get their seed here; rows are regrouped by zone class (warp ballots + three shared counters).
//   Phase B2 (queued rows, grouped zone 0 / middle / zone 3): the tail seeds (lbr_seed_tail0 / _tail3) fused with the
//            two Householder(3) steps (lbr_refine); sigma and vega into the staged output slots of the row.
//   Phase C: the staged sigma, vega and status of the tile are streamed out with coalesced stores.
// Every row still touches HBM exactly once (57 B Black-76, 73 B BSM); both partitions cost shared-memory traffic only.
// The ncu capture of the one-row-per-thread kernel (profiles/r1a_*, r1d_ab_*) shows ~11 of 32 lanes active because more
// than half of config 1/4's rows leave at the validity check; here the solver's warps are full (26.6 of 32).
// ---------------------------------------------------------------------------------------------------------------
constexpr int kTileThreads = 256;
// RPT rows per thread: 4 (1024-row tiles, 55 KB of shared memory, 4 CTAs per SM at 64 registers) for large n; 1 (256-row tiles) for
// small n, so that a launch of 65,536 rows still spreads over every SM.

template <int RPT>
struct TileSmem {
  static constexpr int kTileRows = kTileThreads * RPT;
  double sig[kTileRows];      // phase A: tau (queued rows) or final sigma;  phase B2: final sigma
  double veg[kTileRows];      // phase A: D sqrt(FK) (queued rows) or 0;      phase B2: final vega
  double q0[kTileRows];       // compact queue.  after A: F, K, B, sqrt(FK);  after B1: x, s0, p1, p2 (lbr_seed)
  double q1[kTileRows];
  double q2[kTileRows];
  double q3[kTileRows];
  uint16_t pos[kTileRows];    // tile position of the queued row; bit 15 = call
  uint16_t perm[kTileRows];   // queue indices: zone 0 rows from the front, finished middle-zone rows from the back
  uint16_t permU[kTileRows];  // ... and zone 3 rows
  uint8_t status[kTileRows];
  unsigned long long nclass;  // rows per class, three 21-bit fields: zone 0 | zones 1-2 << 21 | zone 3 << 42
  int count;                  // queued rows
};

template <bool BSM, bool ZONES, int RPT, bool SEL = false>
__global__ void __launch_bounds__(kTileThreads, BSM ? 3 : 4)
forward_kernel_tile(pivot_iv_inputs in, int64_t n, double* __restrict__ sigma, double* __restrict__ vega,
                    uint8_t* __restrict__ status, int8_t* __restrict__ zone, const int* __restrict__ sel, int want) {
  if (SEL && *sel != want) return;   // pivot_iv_forward_auto: the probe chose the other organisation
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int kTileRows = kTileThreads * RPT;
  TileSmem<RPT>& sm = *reinterpret_cast<TileSmem<RPT>*>(smem_raw);
  const int tid = threadIdx.x;
  const int lane = tid & 31;
  const int64_t base = (int64_t)blockIdx.x * kTileRows;
  const int rows = (int)((n - base < kTileRows) ? (n - base) : kTileRows);
  if (tid == 0) { sm.count = 0; sm.nclass = 0ull; }
  __syncthreads();

  // ---- phase A: all rows of the tile; every load of the thread's rows is issued before the first use
  const double* __restrict__ gF = in.S_or_F + base;
  const double* __restrict__ gK = in.K + base;
  const double* __restrict__ gT = in.tau + base;
  const double* __restrict__ gP = in.P + base;
  const double* __restrict__ gf = in.flag + base;
  const double* __restrict__ gr = BSM ? in.r + base : nullptr;
  const double* __restrict__ gq = BSM ? in.q + base : nullptr;
  double vF[RPT], vK[RPT], vT[RPT], vP[RPT],
      vf[RPT], vr[RPT], vq[RPT];
#pragma unroll
  for (int k = 0; k < RPT; ++k) {
    const int p = k * kTileThreads + tid;
    const bool live = p < rows;
    // dead rows read as flag = 0 -> BAD_INPUT, never stored
    vF[k] = live ? __ldcs(gF + p) : 0.0;
    vK[k] = live ? __ldcs(gK + p) : 0.0;
    vT[k] = live ? __ldcs(gT + p) : 0.0;
    vP[k] = live ? __ldcs(gP + p) : 0.0;
    vf[k] = live ? __ldcs(gf + p) : 0.0;
    vr[k] = (BSM && live) ? __ldcs(gr + p) : 0.0;
    vq[k] = (BSM && live) ? __ldcs(gq + p) : 0.0;
  }
  unsigned qmask = 0, cmask = 0;  // bit k: row k of this thread is queued / is a call
#pragma unroll
  for (int k = 0; k < RPT; ++k) {
    const int p = k * kTileThreads + tid;
    const Prelude pr = lbr_prelude<BSM>(vF[k], vK[k], vT[k], vr[k], vq[k], vP[k], vf[k]);
    const bool queued = pr.status == 0;
    if (p < rows) {
      sm.status[p] = (uint8_t)pr.status;
      sm.sig[p] = queued ? vT[k] : (pr.status == 4 ? 0.0 : canonical_nan());
      sm.veg[p] = queued ? pr.scale : 0.0;
      if (ZONES && !queued) zone[base + p] = -1;
    }
    qmask |= queued ? (1u << k) : 0u;
    cmask |= pr.call ? (1u << k) : 0u;
    vF[k] = pr.F; vP[k] = pr.B; vT[k] = pr.rootFK;  // what the solver pass needs: F, K, B, sqrt(FK)
  }
  {
    // one warp scan and one shared atomic per warp for the whole tile
    const int c = __popc(qmask);
    int incl = c;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const int v = __shfl_up_sync(0xffffffffu, incl, d);
      if (lane >= d) incl += v;
    }
    int wbase = 0;
    if (lane == 31 && incl > 0) wbase = atomicAdd(&sm.count, incl);
    int slot = __shfl_sync(0xffffffffu, wbase, 31) + incl - c;
#pragma unroll
    for (int k = 0; k < RPT; ++k) {
      if (qmask & (1u << k)) {
        sm.q0[slot] = vF[k];
        sm.q1[slot] = vK[k];
        sm.q2[slot] = vP[k];
        sm.q3[slot] = vT[k];
        sm.pos[slot] = (uint16_t)((k * kTileThreads + tid) | ((cmask >> k) & 1u ? 0x8000 : 0));
        ++slot;
      }
    }
  }
  __syncthreads();

  // ---- phase B1a: x, boundary point, node, zone; middle zones (1, 2) finished; rows regrouped by zone class
  //      lists: zone 0 (-> LOWER) from the front of perm, finished LINEAR rows from the back, zone 3 in permU
  const int cnt = sm.count;
  for (int j0 = 0; j0 < cnt; j0 += kTileThreads) {   // j0 is CTA-uniform: every lane reaches the ballots
    const int j = j0 + tid;
    int cls = -1;  // 0: zone 0, 1: finished (zones 1, 2), 2: zone 3
    if (j < cnt) {
      const Norm nm = lbr_normalise(sm.q0[j], sm.q1[j], sm.q2[j], sm.q3[j], (sm.pos[j] & 0x8000) != 0);
      const SeedHead hd = lbr_seed_head(nm.qrel, nm.beta, nm.bbar, nm.bmax);
      sm.q0[j] = hd.v0; sm.q1[j] = hd.v1; sm.q2[j] = hd.v2; sm.q3[j] = hd.v3;
      cls = (hd.zone == 0) ? 0 : ((hd.zone == 3) ? 2 : 1);
      if (ZONES) zone[base + (sm.pos[j] & 0x3fff)] = (int8_t)hd.zone;
    }
    const unsigned m0 = __ballot_sync(0xffffffffu, cls == 0);
    const unsigned m1 = __ballot_sync(0xffffffffu, cls == 1);
    const unsigned m2 = __ballot_sync(0xffffffffu, cls == 2);
    // one 64-bit shared atomic per warp hands out the three list offsets at once
    unsigned long long base3 = 0ull;
    if (lane == 0)
      base3 = atomicAdd(&sm.nclass, (unsigned long long)__popc(m0) | ((unsigned long long)__popc(m1) << 21) |
                                        ((unsigned long long)__popc(m2) << 42));
    base3 = __shfl_sync(0xffffffffu, base3, 0);
    const int b0 = (int)(base3 & 0x1fffffu), b1 = (int)((base3 >> 21) & 0x1fffffu), b2 = (int)(base3 >> 42);
    const unsigned lt = (1u << lane) - 1u;
    if (cls == 0) sm.perm[b0 + __popc(m0 & lt)] = (uint16_t)j;
    else if (cls == 1) sm.perm[kTileRows - 1 - (b1 + __popc(m1 & lt))] = (uint16_t)j;
    else if (cls == 2) sm.permU[b2 + __popc(m2 & lt)] = (uint16_t)j;
  }
  __syncthreads();

  // ---- phase B2: the tail seeds (zone 0 rows, zone 3 rows) fused with the Householder steps; rows ordered zone 0
  //      (LOWER), finished middle rows (LINEAR), zone 3 (UPPER or LINEAR): a warp sees one zone and one objective kind
  //      except at the two group boundaries
  const int n0 = (int)(sm.nclass & 0x1fffffu), n1 = (int)((sm.nclass >> 21) & 0x1fffffu);
  for (int k = tid; k < cnt; k += kTileThreads) {
    int j, kind;
    double x, s0, p1, p2;
    if (k < n0) {
      j = sm.perm[k];
      const Seed sd = lbr_seed_tail0(sm.q0[j], sm.q1[j], sm.q2[j], sm.q3[j]);
      x = sd.x; s0 = sd.s; p1 = sd.p1; p2 = sd.p2; kind = KIND_LOWER;
    } else if (k < n0 + n1) {
      j = sm.perm[kTileRows - 1 - (k - n0)];
      x = sm.q0[j]; s0 = sm.q1[j]; p1 = sm.q2[j]; p2 = sm.q3[j]; kind = KIND_LINEAR;
    } else {
      j = sm.permU[k - n0 - n1];
      const Seed sd = lbr_seed_tail3(sm.q0[j], sm.q1[j], sm.q2[j], sm.q3[j]);
      x = sd.x; s0 = sd.s; p1 = sd.p1; p2 = sd.p2; kind = sd.kind;
    }
    const NormSolve ns = lbr_refine<kHouseholderSteps>(x, s0, p1, p2, kind);
    const int p = sm.pos[j] & 0x3fff;
    const double tau = sm.sig[p];
    const double rinv = rsqrt(tau);
    sm.sig[p] = ns.s * rinv;
    sm.veg[p] = sm.veg[p] * ns.vfin * (tau * rinv);
  }
  __syncthreads();

  // ---- phase C
#pragma unroll 4
  for (int k = 0; k < RPT; ++k) {
    const int p = k * kTileThreads + tid;
    if (p < rows) {
      __stcs(sigma + base + p, sm.sig[p]);
      __stcs(vega + base + p, sm.veg[p]);
    }
  }
  if (rows == kTileRows && ((reinterpret_cast<uintptr_t>(status + base) & 15u) == 0)) {
    if (tid < kTileRows / 16) __stcs(reinterpret_cast<uint4*>(status + base) + tid, reinterpret_cast<const uint4*>(sm.status)[tid]);
  } else {
    for (int p = tid; p < rows; p += kTileThreads) status[base + p] = sm.status[p];
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Backward kernel: grad_P = gate * grad_sigma / vega  (eq.(8)-(10)); 25 B/row, HBM-bound.
// ---------------------------------------------------------------------------------------------------------------
template <int MODE>
__device__ __forceinline__ double backward_row(double gs, double V, uint8_t st, double floor_, double floor2) {
  if (MODE == PIVOT_GATE_MASK) {
    const bool on = (st == PIVOT_ST_OK) && (fabs(V) > floor_);
    return on ? __ddiv_rn(gs, V) : 0.0;
  } else if (MODE == PIVOT_GATE_STRICT) {
    const bool on = (st == PIVOT_ST_OK) && (fabs(V) > floor_);
    return on ? __ddiv_rn(gs, V) : ((gs == 0.0) ? 0.0 : canonical_nan());
  } else {
    const double den = __dadd_rn(__dmul_rn(V, V), floor2);
    const bool on = (st == PIVOT_ST_OK) && (den > 0.0);
    return on ? __ddiv_rn(__dmul_rn(gs, V), den) : 0.0;
  }
}

// 4 rows per thread per iteration (two 16-byte loads per fp64 array, one 4-byte status load), grid-stride.
template <int MODE>
__global__ void __launch_bounds__(kBwdThreads)
backward_kernel_vec4(const double* __restrict__ gs, const double* __restrict__ vega, const uint8_t* __restrict__ status,
                     double floor_, int64_t n4, double* __restrict__ gP) {
  const double floor2 = __dmul_rn(floor_, floor_);
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j < n4; j += stride) {
    const double2 g0 = __ldcs(reinterpret_cast<const double2*>(gs) + 2 * j);
    const double2 g1 = __ldcs(reinterpret_cast<const double2*>(gs) + 2 * j + 1);
    const double2 v0 = __ldcs(reinterpret_cast<const double2*>(vega) + 2 * j);
    const double2 v1 = __ldcs(reinterpret_cast<const double2*>(vega) + 2 * j + 1);
    const uchar4 st = __ldcs(reinterpret_cast<const uchar4*>(status) + j);
    double2 o0, o1;
    o0.x = backward_row<MODE>(g0.x, v0.x, st.x, floor_, floor2);
    o0.y = backward_row<MODE>(g0.y, v0.y, st.y, floor_, floor2);
    o1.x = backward_row<MODE>(g1.x, v1.x, st.z, floor_, floor2);
    o1.y = backward_row<MODE>(g1.y, v1.y, st.w, floor_, floor2);
    __stcs(reinterpret_cast<double2*>(gP) + 2 * j, o0);
    __stcs(reinterpret_cast<double2*>(gP) + 2 * j + 1, o1);
  }
}

template <int MODE>
__global__ void __launch_bounds__(kBwdThreads)
backward_kernel_scalar(const double* __restrict__ gs, const double* __restrict__ vega, const uint8_t* __restrict__ status,
                       double floor_, int64_t begin, int64_t n, double* __restrict__ gP) {
  const double floor2 = __dmul_rn(floor_, floor_);
  const int64_t i = begin + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) gP[i] = backward_row<MODE>(gs[i], vega[i], status[i], floor_, floor2);
}

// fp64-pipe probe: 8 independent DFMA chains per thread
__global__ void __launch_bounds__(256) dfma_probe_kernel(int64_t iters, double* sink) {
  double a0 = 1.0 + threadIdx.x * 1e-9, a1 = a0 + 1e-3, a2 = a0 + 2e-3, a3 = a0 + 3e-3, a4 = a0 + 4e-3, a5 = a0 + 5e-3,
         a6 = a0 + 6e-3, a7 = a0 + 7e-3;
  const double m = 0.999999999, c = 1e-9;
  for (int64_t i = 0; i < iters; ++i) {
    a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
    a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
  }
  const double sum = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
  if (sum == 123.456) sink[0] = sum;  // never true; keeps the chains alive
}

// ---------------------------------------------------------------------------------------------------------------
// Probe of pivot_iv_forward_auto: 2048 sampled (row, next row) pairs.  ws[0] = 1 (row-per-thread organisation) when at
// least 95 % of the sampled rows reach the solver AND at least 90 % of the pairs are the same contract up to 2 % in F|S
// and K (an option chain in strike order: warps are zone-uniform by themselves); else 0 (compaction).  ws[1..3] = rows
// that solve, alike pairs, samples.
// ---------------------------------------------------------------------------------------------------------------
constexpr int kProbePairs = 2048;
constexpr int kProbeBlocks = 8;   // 8 x 256 threads: one pair per thread, every load of the probe is in flight at once
template <bool BSM>
__global__ void __launch_bounds__(256) forward_probe_kernel(pivot_iv_inputs in, int64_t n, int* __restrict__ ws) {
  // ws[1], ws[2] accumulate; ws[4] is the ticket; the last CTA to arrive decides and resets the accumulators' ticket
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t i = (int64_t)(((n - 2) / kProbePairs) * (int64_t)k);
  const double F0 = in.S_or_F[i], K0 = in.K[i], F1 = in.S_or_F[i + 1], K1 = in.K[i + 1];
  const double r = BSM ? in.r[i] : 0.0, q = BSM ? in.q[i] : 0.0;
  const Prelude pr = lbr_prelude<BSM>(F0, K0, in.tau[i], r, q, in.P[i], in.flag[i]);
  const unsigned mo = __ballot_sync(0xffffffffu, pr.status == PIVOT_ST_OK);
  const unsigned ma = __ballot_sync(0xffffffffu, fabs(K1 - K0) <= 0.02 * K0 && fabs(F1 - F0) <= 0.02 * F0);
  __shared__ int last;
  if ((threadIdx.x & 31) == 0) {
    atomicAdd(&ws[5], __popc(mo));
    atomicAdd(&ws[6], __popc(ma));
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    last = atomicAdd(&ws[4], 1) == kProbeBlocks - 1;
  }
  __syncthreads();
  if (last && threadIdx.x == 0) {
    __threadfence();
    const int ok = atomicAdd(&ws[5], 0), alike = atomicAdd(&ws[6], 0);
    ws[1] = ok; ws[2] = alike; ws[3] = kProbePairs;
    ws[0] = (ok * 100 >= 95 * kProbePairs && alike * 100 >= 90 * kProbePairs) ? 1 : 0;
    ws[4] = 0; ws[5] = 0; ws[6] = 0;   // ready for the next call on this stream
  }
}

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

}  // namespace pivot

// ===============================================================================================================
// C ABI
// ===============================================================================================================
using namespace pivot;

namespace {

// Kernel choice.  PIVOT_FWD_AUTO follows the environment variable PIVOT_IV_FWD_KERNEL (=rowwise: one row per thread;
// anything else / unset: tile compaction), read once; it exists for the ncu A/B studies of DESIGN.md section 8.
bool env_rowwise() {
  static const bool v = [] {
    const char* e = std::getenv("PIVOT_IV_FWD_KERNEL");
    return e && e[0] == 'r';
  }();
  return v;
}

template <bool BSM, bool ZONES>
int launch_forward_t(const pivot_iv_inputs& in, int64_t n, double* sigma, double* vega, uint8_t* status, int8_t* zone,
                     int kernel, cudaStream_t st) {
  const bool rowwise = kernel == PIVOT_FWD_ROWWISE || (kernel == PIVOT_FWD_AUTO && env_rowwise());
  if (rowwise) {
    const int64_t blocks = (n + kFwdThreads - 1) / kFwdThreads;
    forward_kernel_scalar<BSM, ZONES><<<(unsigned)blocks, kFwdThreads, 0, st>>>(in, 0, n, sigma, vega, status, zone, nullptr, 0);
  } else {
    // small launches use 256-row tiles so that the grid still covers the chip (n <= 2^19: at most 2048 CTAs)
    if (n <= ((int64_t)1 << 19)) {
      static const cudaError_t attr = cudaFuncSetAttribute(forward_kernel_tile<BSM, ZONES, 1>,
                                                           cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(TileSmem<1>));
      if (attr != cudaSuccess) return PIVOT_ERR_CUDA;
      const int64_t blocks = (n + kTileThreads - 1) / kTileThreads;
      forward_kernel_tile<BSM, ZONES, 1><<<(unsigned)blocks, kTileThreads, sizeof(TileSmem<1>), st>>>(in, n, sigma, vega, status, zone, nullptr, 0);
    } else {
      static const cudaError_t attr = cudaFuncSetAttribute(forward_kernel_tile<BSM, ZONES, 4>,
                                                           cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(TileSmem<4>));
      if (attr != cudaSuccess) return PIVOT_ERR_CUDA;
      const int64_t blocks = (n + 4 * kTileThreads - 1) / (4 * kTileThreads);
      forward_kernel_tile<BSM, ZONES, 4><<<(unsigned)blocks, kTileThreads, sizeof(TileSmem<4>), st>>>(in, n, sigma, vega, status, zone, nullptr, 0);
    }
  }
  return cudaGetLastError() == cudaSuccess ? PIVOT_OK : PIVOT_ERR_CUDA;
}

int forward_impl(const pivot_iv_inputs* in, int64_t n, double* sigma, double* vega, uint8_t* status, int8_t* zone,
                 bool zones, cudaStream_t st, int kernel = PIVOT_FWD_AUTO) {
  if (!in) return PIVOT_ERR_NULL;
  if (kernel != PIVOT_FWD_AUTO && kernel != PIVOT_FWD_COMPACT && kernel != PIVOT_FWD_ROWWISE) return PIVOT_ERR_BAD_ARG;
  if (n < 0) return PIVOT_ERR_BAD_N;
  if ((in->r == nullptr) != (in->q == nullptr)) return PIVOT_ERR_MIXED_RQ;
  if (n == 0) return PIVOT_OK;
  if (!in->S_or_F || !in->K || !in->tau || !in->P || !in->flag || !sigma || !vega || !status || (zones && !zone))
    return PIVOT_ERR_NULL;
  if (n > ((int64_t)1 << 37)) return PIVOT_ERR_BAD_N;  // grid.x limit
  const bool bsm = in->r != nullptr;
  if (bsm) return zones ? launch_forward_t<true, true>(*in, n, sigma, vega, status, zone, kernel, st)
                        : launch_forward_t<true, false>(*in, n, sigma, vega, status, zone, kernel, st);
  return zones ? launch_forward_t<false, true>(*in, n, sigma, vega, status, zone, kernel, st)
               : launch_forward_t<false, false>(*in, n, sigma, vega, status, zone, kernel, st);
}

int g_sm_count = 0;
int sm_count() {
  if (g_sm_count == 0) {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0)
      sms = 148;
    g_sm_count = sms;
  }
  return g_sm_count;
}

// pivot_iv_forward_auto: probe, then both organisations are enqueued and the one the probe did not choose returns at
// once (the row-per-thread kernel as a small grid-stride grid, so that its early exit costs microseconds).
template <bool BSM>
int launch_forward_auto_t(const pivot_iv_inputs& in, int64_t n, double* sigma, double* vega, uint8_t* status, int* ws,
                          cudaStream_t st) {
  static const cudaError_t attr = cudaFuncSetAttribute(forward_kernel_tile<BSM, false, 4, true>,
                                                       cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(TileSmem<4>));
  if (attr != cudaSuccess) return PIVOT_ERR_CUDA;
  forward_probe_kernel<BSM><<<kProbeBlocks, kProbePairs / kProbeBlocks, 0, st>>>(in, n, ws);
  const int64_t rblocks = (n + kFwdThreads - 1) / kFwdThreads;
  const int64_t rcap = (int64_t)sm_count() * 6 * 8;    // 80 registers: 6 resident CTAs of 128 threads per SM; 8 waves' worth, grid-stride
  forward_kernel_scalar<BSM, false, true><<<(unsigned)(rblocks < rcap ? rblocks : rcap), kFwdThreads, 0, st>>>(
      in, 0, n, sigma, vega, status, nullptr, ws, 1);
  const int64_t tblocks = (n + 4 * kTileThreads - 1) / (4 * kTileThreads);
  forward_kernel_tile<BSM, false, 4, true><<<(unsigned)tblocks, kTileThreads, sizeof(TileSmem<4>), st>>>(in, n, sigma, vega,
                                                                                                       status, nullptr, ws, 0);
  return cudaGetLastError() == cudaSuccess ? PIVOT_OK : PIVOT_ERR_CUDA;
}

template <int MODE>
int launch_backward_t(const double* gs, const double* vega, const uint8_t* status, double floor_, int64_t n, double* gP,
                      cudaStream_t st) {
  const bool vec = aligned16(gs) && aligned16(vega) && aligned16(gP) && ((reinterpret_cast<uintptr_t>(status) & 3u) == 0);
  int64_t done = 0;
  if (vec && n >= 4) {
    const int64_t n4 = n / 4;
    int64_t blocks = (n4 + kBwdThreads - 1) / kBwdThreads;
    const int64_t cap = (int64_t)sm_count() * 8 * 4;  // 8 resident CTAs of 256 threads per SM, 4 waves' worth
    if (blocks > cap) blocks = cap;
    backward_kernel_vec4<MODE><<<(unsigned)blocks, kBwdThreads, 0, st>>>(gs, vega, status, floor_, n4, gP);
    done = 4 * n4;
  }
  if (done < n) {
    const int64_t rem = n - done;
    const int64_t blocks = (rem + kBwdThreads - 1) / kBwdThreads;
    backward_kernel_scalar<MODE><<<(unsigned)blocks, kBwdThreads, 0, st>>>(gs, vega, status, floor_, done, n, gP);
  }
  return cudaGetLastError() == cudaSuccess ? PIVOT_OK : PIVOT_ERR_CUDA;
}

int backward_impl(const double* gs, const double* vega, const uint8_t* status, double floor_, int mode, int64_t n,
                  double* gP, cudaStream_t st) {
  if (n < 0) return PIVOT_ERR_BAD_N;
  if (mode != PIVOT_GATE_MASK && mode != PIVOT_GATE_ATTENUATE && mode != PIVOT_GATE_STRICT) return PIVOT_ERR_BAD_MODE;
  if (!(floor_ >= 0.0)) return PIVOT_ERR_BAD_FLOOR;
  if (n == 0) return PIVOT_OK;
  if (!gs || !vega || !status || !gP) return PIVOT_ERR_NULL;
  if (n > ((int64_t)1 << 38)) return PIVOT_ERR_BAD_N;
  if (mode == PIVOT_GATE_MASK) return launch_backward_t<PIVOT_GATE_MASK>(gs, vega, status, floor_, n, gP, st);
  if (mode == PIVOT_GATE_STRICT) return launch_backward_t<PIVOT_GATE_STRICT>(gs, vega, status, floor_, n, gP, st);
  return launch_backward_t<PIVOT_GATE_ATTENUATE>(gs, vega, status, floor_, n, gP, st);
}

}  // namespace

extern "C" {

int pivot_iv_forward(const pivot_iv_inputs* in, int64_t n, double* sigma, double* vega, uint8_t* status,
                     pivot_iv_stream stream) {
  return forward_impl(in, n, sigma, vega, status, nullptr, false, reinterpret_cast<cudaStream_t>(stream));
}

int pivot_iv_forward_ex(const pivot_iv_inputs* in, int64_t n, double* sigma, double* vega, uint8_t* status, int kernel,
                        pivot_iv_stream stream) {
  return forward_impl(in, n, sigma, vega, status, nullptr, false, reinterpret_cast<cudaStream_t>(stream), kernel);
}

int64_t pivot_iv_forward_auto_workspace_bytes(void) { return 64; }

int pivot_iv_forward_auto(const pivot_iv_inputs* in, int64_t n, double* sigma, double* vega, uint8_t* status,
                          void* workspace, pivot_iv_stream stream) {
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  if (!in) return PIVOT_ERR_NULL;
  if (n < ((int64_t)1 << 23))   // no probe below 2^23 rows (probe + the unused launch cost ~30 us); workspace not used
    return forward_impl(in, n, sigma, vega, status, nullptr, false, st, PIVOT_FWD_COMPACT);
  if (!workspace) return PIVOT_ERR_NULL;
  if ((in->r == nullptr) != (in->q == nullptr)) return PIVOT_ERR_MIXED_RQ;
  if (!in->S_or_F || !in->K || !in->tau || !in->P || !in->flag || !sigma || !vega || !status) return PIVOT_ERR_NULL;
  if (n > ((int64_t)1 << 37)) return PIVOT_ERR_BAD_N;
  if ((reinterpret_cast<uintptr_t>(workspace) & 3u) != 0) return PIVOT_ERR_BAD_ARG;
  int* ws = static_cast<int*>(workspace);
  return in->r ? launch_forward_auto_t<true>(*in, n, sigma, vega, status, ws, st)
               : launch_forward_auto_t<false>(*in, n, sigma, vega, status, ws, st);
}

int pivot_iv_forward_zones(const pivot_iv_inputs* in, int64_t n, double* sigma, double* vega, uint8_t* status,
                           int8_t* zone, pivot_iv_stream stream) {
  return forward_impl(in, n, sigma, vega, status, zone, true, reinterpret_cast<cudaStream_t>(stream));
}

int pivot_iv_backward(const double* grad_sigma, const double* vega, const uint8_t* status, double vega_floor, int mode,
                      int64_t n, double* grad_P, pivot_iv_stream stream) {
  return backward_impl(grad_sigma, vega, status, vega_floor, mode, n, grad_P, reinterpret_cast<cudaStream_t>(stream));
}

int pivot_iv_probe_dfma(int64_t iters, double* sink, double* fma_count_out, pivot_iv_stream stream) {
  if (!sink || !fma_count_out) return PIVOT_ERR_NULL;
  if (iters <= 0) return PIVOT_ERR_BAD_ARG;
  const int blocks = sm_count() * 8, threads = 256;
  dfma_probe_kernel<<<blocks, threads, 0, reinterpret_cast<cudaStream_t>(stream)>>>(iters, sink);
  *fma_count_out = (double)iters * 8.0 * (double)blocks * (double)threads;
  return cudaGetLastError() == cudaSuccess ? PIVOT_OK : PIVOT_ERR_CUDA;
}

int pivot_iv_launches_per_forward(void) { return 1; }
int pivot_iv_launches_per_backward(void) { return 1; }

const char* pivot_iv_strerror(int code) {
  switch (code) {
    case PIVOT_OK: return "ok";
    case PIVOT_ERR_NULL: return "a required pointer is NULL";
    case PIVOT_ERR_BAD_N: return "n is negative or too large";
    case PIVOT_ERR_BAD_MODE: return "mode must be PIVOT_GATE_MASK (0), PIVOT_GATE_ATTENUATE (1) or PIVOT_GATE_STRICT (2)";
    case PIVOT_ERR_BAD_FLOOR: return "vega_floor must be a non-negative number";
    case PIVOT_ERR_MIXED_RQ: return "r and q must both be NULL (Black-76) or both non-NULL (BSM)";
    case PIVOT_ERR_CUDA: return "CUDA runtime error";
    case PIVOT_ERR_BAD_ARG: return "invalid argument";
    default: return "unknown pivot_iv error code";
  }
}

int pivot_iv_version(void) { return PIVOT_IV_VERSION; }

}  // extern "C"

// ===============================================================================================================
// Host-buffer pipeline: chunked H2D -> forward [-> backward] -> D2H, one stream per slot so that the copy engines
// and the SMs overlap across chunks (streaming label generation over batches of rows).
// ===============================================================================================================
struct pivot_iv_pipeline {
  int device = 0;
  int64_t chunk = 0;
  int nslots = 0;
  int fwd_kernel = PIVOT_FWD_AUTO;
  cudaStream_t streams[8] = {};
  double* dbl[8] = {};   // per slot: 11 fp64 arrays of `chunk` rows: S,K,tau,r,q,P,flag,sigma,vega,gs,gP
  uint8_t* st[8] = {};   // per slot: status bytes
};

namespace {

#define PIVOT_CUDA_TRY(expr)                    \
  do {                                          \
    if ((expr) != cudaSuccess) {                \
      (void)cudaGetLastError();                 \
      return PIVOT_ERR_CUDA;                    \
    }                                           \
  } while (0)

int pipeline_run(pivot_iv_pipeline* p, const pivot_iv_inputs* in, const double* gs, double floor_, int mode, bool bwd,
                 int64_t n, double* sigma, double* vega, uint8_t* status, double* gP) {
  if (!p || !in) return PIVOT_ERR_NULL;
  if (n < 0) return PIVOT_ERR_BAD_N;
  if ((in->r == nullptr) != (in->q == nullptr)) return PIVOT_ERR_MIXED_RQ;
  if (bwd) {
    if (mode != PIVOT_GATE_MASK && mode != PIVOT_GATE_ATTENUATE && mode != PIVOT_GATE_STRICT) return PIVOT_ERR_BAD_MODE;
    if (!(floor_ >= 0.0)) return PIVOT_ERR_BAD_FLOOR;
  }
  if (n == 0) return PIVOT_OK;
  if (!in->S_or_F || !in->K || !in->tau || !in->P || !in->flag || !sigma || !vega || !status) return PIVOT_ERR_NULL;
  if (bwd && (!gs || !gP)) return PIVOT_ERR_NULL;
  int prev = 0;
  PIVOT_CUDA_TRY(cudaGetDevice(&prev));
  PIVOT_CUDA_TRY(cudaSetDevice(p->device));
  const bool bsm = in->r != nullptr;
  const int64_t C = p->chunk;
  int rc = PIVOT_OK;
  int64_t c = 0;
  for (int64_t off = 0; off < n && rc == PIVOT_OK; off += C, ++c) {
    const int slot = (int)(c % p->nslots);
    const int64_t m = (n - off < C) ? (n - off) : C;
    cudaStream_t s = p->streams[slot];
    double* base = p->dbl[slot];
    double* d[11];
    for (int k = 0; k < 11; ++k) d[k] = base + (int64_t)k * C;
    const size_t bytes = (size_t)m * sizeof(double);
    const double* src[7] = {in->S_or_F, in->K, in->tau, in->r, in->q, in->P, in->flag};
    for (int k = 0; k < 7; ++k) {
      if (!src[k]) continue;
      if (cudaMemcpyAsync(d[k], src[k] + off, bytes, cudaMemcpyHostToDevice, s) != cudaSuccess) rc = PIVOT_ERR_CUDA;
    }
    if (bwd && cudaMemcpyAsync(d[9], gs + off, bytes, cudaMemcpyHostToDevice, s) != cudaSuccess) rc = PIVOT_ERR_CUDA;
    if (rc != PIVOT_OK) break;
    pivot_iv_inputs din{d[0], d[1], d[2], bsm ? d[3] : nullptr, bsm ? d[4] : nullptr, d[5], d[6]};
    rc = forward_impl(&din, m, d[7], d[8], p->st[slot], nullptr, false, s, p->fwd_kernel);
    if (rc == PIVOT_OK && bwd) rc = backward_impl(d[9], d[8], p->st[slot], floor_, mode, m, d[10], s);
    if (rc != PIVOT_OK) break;
    if (cudaMemcpyAsync(sigma + off, d[7], bytes, cudaMemcpyDeviceToHost, s) != cudaSuccess ||
        cudaMemcpyAsync(vega + off, d[8], bytes, cudaMemcpyDeviceToHost, s) != cudaSuccess ||
        cudaMemcpyAsync(status + off, p->st[slot], (size_t)m, cudaMemcpyDeviceToHost, s) != cudaSuccess ||
        (bwd && cudaMemcpyAsync(gP + off, d[10], bytes, cudaMemcpyDeviceToHost, s) != cudaSuccess))
      rc = PIVOT_ERR_CUDA;
  }
  for (int k = 0; k < p->nslots; ++k)
    if (cudaStreamSynchronize(p->streams[k]) != cudaSuccess) rc = PIVOT_ERR_CUDA;
  if (rc == PIVOT_ERR_CUDA) (void)cudaGetLastError();
  (void)cudaSetDevice(prev);
  return rc;
}

}  // namespace

extern "C" {

int pivot_iv_pipeline_create(pivot_iv_pipeline** out, int device, int64_t chunk_rows, int n_slots) {
  if (!out) return PIVOT_ERR_NULL;
  *out = nullptr;
  if (chunk_rows <= 0 || n_slots < 1 || n_slots > 8) return PIVOT_ERR_BAD_ARG;
  int prev = 0;
  PIVOT_CUDA_TRY(cudaGetDevice(&prev));
  if (device < 0) device = prev;
  if (cudaSetDevice(device) != cudaSuccess) { (void)cudaGetLastError(); return PIVOT_ERR_BAD_ARG; }
  pivot_iv_pipeline* p = new (std::nothrow) pivot_iv_pipeline();
  if (!p) { (void)cudaSetDevice(prev); return PIVOT_ERR_CUDA; }
  p->device = device;
  p->chunk = (chunk_rows + 1) & ~(int64_t)1;  // even, keeps every array of a slot 16-byte aligned
  p->nslots = n_slots;
  int rc = PIVOT_OK;
  for (int k = 0; k < n_slots && rc == PIVOT_OK; ++k) {
    if (cudaStreamCreateWithFlags(&p->streams[k], cudaStreamNonBlocking) != cudaSuccess ||
        cudaMalloc(&p->dbl[k], (size_t)p->chunk * 11 * sizeof(double)) != cudaSuccess ||
        cudaMalloc(&p->st[k], (size_t)p->chunk) != cudaSuccess)
      rc = PIVOT_ERR_CUDA;
  }
  (void)cudaSetDevice(prev);
  if (rc != PIVOT_OK) { (void)cudaGetLastError(); pivot_iv_pipeline_destroy(p); return rc; }
  *out = p;
  return PIVOT_OK;
}

int pivot_iv_pipeline_set_forward_kernel(pivot_iv_pipeline* p, int kernel) {
  if (!p) return PIVOT_ERR_NULL;
  if (kernel != PIVOT_FWD_AUTO && kernel != PIVOT_FWD_COMPACT && kernel != PIVOT_FWD_ROWWISE) return PIVOT_ERR_BAD_ARG;
  p->fwd_kernel = kernel;
  return PIVOT_OK;
}

int pivot_iv_pipeline_destroy(pivot_iv_pipeline* p) {
  if (!p) return PIVOT_OK;
  int prev = 0;
  (void)cudaGetDevice(&prev);
  (void)cudaSetDevice(p->device);
  for (int k = 0; k < 8; ++k) {
    if (p->streams[k]) { (void)cudaStreamSynchronize(p->streams[k]); (void)cudaStreamDestroy(p->streams[k]); }
    if (p->dbl[k]) (void)cudaFree(p->dbl[k]);
    if (p->st[k]) (void)cudaFree(p->st[k]);
  }
  (void)cudaSetDevice(prev);
  delete p;
  return PIVOT_OK;
}

int pivot_iv_forward_host(pivot_iv_pipeline* p, const pivot_iv_inputs* in, int64_t n, double* sigma, double* vega,
                          uint8_t* status) {
  return pipeline_run(p, in, nullptr, 0.0, 0, false, n, sigma, vega, status, nullptr);
}

int pivot_iv_forward_backward_host(pivot_iv_pipeline* p, const pivot_iv_inputs* in, const double* grad_sigma,
                                   double vega_floor, int mode, int64_t n, double* sigma, double* vega,
                                   uint8_t* status, double* grad_P) {
  return pipeline_run(p, in, grad_sigma, vega_floor, mode, true, n, sigma, vega, status, grad_P);
}

}  // extern "C"
