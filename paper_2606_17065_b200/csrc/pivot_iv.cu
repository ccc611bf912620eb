// pivot_iv.cu -- kernels and C ABI (include/pivot_iv.h) of the PIVOT implied-volatility hot path, sm_100a.
//
// Forward: one fused kernel; every intermediate of the per-row LBR solve lives in registers or shared memory, HBM is
// touched once per element (57 B/row Black-76, 73 B/row BSM).  Two organisations of the same per-row arithmetic:
// forward_kernel_tile (rows compacted and regrouped by LBR zone in shared memory; the default) and
// forward_kernel_scalar (one row per thread).  Backward: one streaming elementwise kernel (25 B/row).
// No tensor cores: the path is an fp64 transcendental chain, not a contraction.
#include <cuda_runtime.h>

#include <atomic>
#include <cstddef>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <mutex>
#include <new>

#include "../../include/pivot_iv.h"
#include "lbr_device.cuh"

// -DPIVOT_BOUNDS_CHECK (build.py build(bounds_check=True) -> libpivot_iv_boundscheck.so): every shared-memory index of the
// tile kernel is asserted in range on the device (compute-sanitizer is not available on this pool; tests/test_gpu_boundscheck.py
// runs the ragged / edge / BSM cases through this build).  Compiled out of the product library.
#ifdef PIVOT_BOUNDS_CHECK
#include <cassert>
#define PIVOT_ASSERT(c) assert(c)
#else
#define PIVOT_ASSERT(c) ((void)0)
#endif

namespace pivot {

constexpr int kFwdThreads = 256;
constexpr int kBwdThreads = 256;
constexpr int kHouseholderSteps = 2;  // north_star: two Householder(3) steps

// optional per-row diagnostics of the forward kernels (pivot_iv_forward_diag): any pointer may be null
struct DiagOut {
  int8_t* zone;   // LBR zone 0..3, -1 for rows that never reach the solver
  double* s0;     // total volatility of the rational seed
  double* s1;     // ... after the first (seed-grade) Householder step
};

// ---------------------------------------------------------------------------------------------------------------
// Forward kernel, one row per thread (PIVOT_FWD_ROWWISE): no shared memory, no barriers; coalesced 8-byte accesses.
// Best when nearly every row solves and neighbouring rows are alike (option chains in strike order).
// ---------------------------------------------------------------------------------------------------------------
template <bool BSM, bool DIAG, bool FULL>
__global__ void __launch_bounds__(kFwdThreads, (FULL || DIAG) ? 1 : 4)
forward_kernel_scalar(pivot_iv_inputs in, int64_t n, double* __restrict__ sigma, double* __restrict__ vega,
                      uint8_t* __restrict__ status, DiagOut dg) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double r = BSM ? __ldcs(in.r + i) : 0.0, q = BSM ? __ldcs(in.q + i) : 0.0;
  const RowOut o = lbr_row<BSM, kHouseholderSteps, FULL>(__ldcs(in.S_or_F + i), __ldcs(in.K + i), __ldcs(in.tau + i), r, q,
                                                         __ldcs(in.P + i), __ldcs(in.flag + i));
  __stcs(sigma + i, o.sigma);
  __stcs(vega + i, o.vega);
  status[i] = o.status;
  if (DIAG) {
    if (dg.zone) dg.zone[i] = o.zone;
    if (dg.s0) dg.s0[i] = o.s0;
    if (dg.s1) dg.s1[i] = o.s1;
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Forward kernel, "tile compaction".  A CTA owns a tile of kTileRows consecutive rows.
//   Phase A  (all rows, coalesced 8-byte loads): lbr_prelude -> status, decided on the high words and five exact
//            subtractions / comparisons; no square root, no division.  Rows that need the solver are appended to a
//            compact queue (U, O, B) in shared memory (one ballot per 32 rows and one shared atomic per warp per stage --
//            1024-row tiles run phase A in two stages of two rows per thread; slots in row order within the warp); the others get their final sigma / vega straight away.  For queued rows the staged sigma
//            slot carries tau meanwhile (and the vega slot the discount factor in BSM mode).
//   Phase B1 (queued rows, DENSE warps): lbr_normalise (sqrt(FK) and the four quotients) + lbr_seed_head: x, boundary
//            point, node, zone, and four handover words per row (tails: the node; middle zones: the three fp32 parameters
//            of their rational cubic); rows are regrouped by zone class (warp ballots + two shared counters).
//   Phase B2 (queued rows, grouped zone 0 / middle / zone 3): the seed of the row's zone (lbr_seed_tail0 / _mid / _tail3)
//            fused with the two Householder(3) steps (lbr_refine); sigma and vega into the staged output slots of the row.
//   Phase C: the staged sigma, vega and status of the tile are streamed out with coalesced stores.
// Every row still touches HBM exactly once (57 B Black-76, 73 B BSM); both partitions cost shared-memory traffic only.
// ---------------------------------------------------------------------------------------------------------------
constexpr int kTileThreads = 256;
#ifndef PIVOT_PREFETCH_DIST
#define PIVOT_PREFETCH_DIST 222
#endif
// RPT rows per thread: 4 (1024-row tiles, 55 KB of shared memory, 4 CTAs per SM at 64 registers, both modes) for large n;
// 2 (512-row tiles) up to 2^20 rows and 1 (256-row tiles) up to 2^17, so that a small launch still spreads over every SM.

template <int RPT>
struct TileSmem {
  static constexpr int kTileRows = kTileThreads * RPT;
  double sig[kTileRows];      // phase A: tau (queued rows) or final sigma;  phase B2: final sigma
  double veg[kTileRows];      // phase A: D (queued rows, BSM) or 0; phase B1: D sqrt(FK); phase B2: final vega
  double q0[kTileRows];       // compact queue.  after A: U, O, B;  after B1: the four handover words of lbr_seed_head
  double q1[kTileRows];
  double q2[kTileRows];
  double q3[kTileRows];
  uint16_t pos[kTileRows];    // tile position of the queued row; bit 15 = rare row (exact prelude, IEEE square root)
  uint16_t perm[kTileRows];   // queue indices: zone 0 rows from the front, middle-zone rows from the back
  uint16_t permU[kTileRows];  // ... and zone 3 rows
  uint8_t status[kTileRows];
  unsigned n01;               // rows per class: zone 0 | zones 1-2 << 16  (one native 32-bit shared atomic per warp)
  unsigned n2;                // ... zone 3
  unsigned count;             // queued rows
};

// Shared-memory atomic add issued by ONE lane.  For an atomic on a warp-uniform address ptxas emits its warp-aggregation
// sequence (vote / find-leader / popc / multiply / shuffle: ~25 instructions) even when a single lane is active; `vary` is a
// per-thread byte offset that is always 0 but that the compiler cannot prove uniform (a hash of tid x a bit of n that is never set), which
// leaves the plain predicated ATOMS.ADD.
__device__ __forceinline__ unsigned smem_atomic_add(unsigned* addr, unsigned vary, unsigned v) {
  unsigned old;
  asm volatile("atom.shared.add.u32 %0, [%1], %2;"
               : "=r"(old) : "r"((unsigned)__cvta_generic_to_shared(addr) + vary), "r"(v) : "memory");
  return old;
}

// A row the fast prelude could not classify (status 5): lbr_prelude_exact on its inputs, staged outputs, and its own
// queue slot (flagged: lbr_normalise then takes the IEEE square root).
template <bool BSM, bool DIAG, int RPT>
static __device__ __noinline__ void tile_rare_row(pivot_iv_inputs in, int64_t base, int p, TileSmem<RPT>& sm, DiagOut dg) {
  const int64_t i = base + p;
  const double tau = in.tau[i];
  const Prelude pr = lbr_prelude_exact<BSM>(in.S_or_F[i], in.K[i], tau, BSM ? in.r[i] : 0.0, BSM ? in.q[i] : 0.0, in.P[i],
                                            in.flag[i]);
  const bool queued = pr.status == 0;
  sm.status[p] = (uint8_t)pr.status;
  sm.sig[p] = queued ? tau : (pr.status == 4 ? 0.0 : canonical_nan());
  sm.veg[p] = queued ? pr.D : 0.0;
  if (queued) {
    const int slot = (int)atomicAdd(&sm.count, 1u);
    PIVOT_ASSERT(slot >= 0 && slot < TileSmem<RPT>::kTileRows && p >= 0 && p < TileSmem<RPT>::kTileRows);
    sm.q0[slot] = pr.U;
    sm.q1[slot] = pr.O;
    sm.q2[slot] = pr.B;
    sm.pos[slot] = (uint16_t)(p | 0x8000);
  } else if (DIAG) {
    if (dg.zone) dg.zone[i] = -1;
    if (dg.s0) dg.s0[i] = 0.0;
    if (dg.s1) dg.s1[i] = 0.0;
  }
}

template <bool BSM, bool DIAG, int RPT, bool FULL>
__global__ void __launch_bounds__(kTileThreads, (FULL || DIAG) ? 3 : 4)
forward_kernel_tile(pivot_iv_inputs in, int64_t n, double* __restrict__ sigma, double* __restrict__ vega,
                    uint8_t* __restrict__ status, DiagOut dg) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int kTileRows = kTileThreads * RPT;
  TileSmem<RPT>& sm = *reinterpret_cast<TileSmem<RPT>*>(smem_raw);
  const int tid = threadIdx.x;
  const int lane = tid & 31;
  const unsigned vary = ((unsigned)tid * 40503u >> 3) * (unsigned)((uint64_t)n >> 62) * 4u;   // 0 (n < 2^38); see smem_atomic_add
  const int64_t base = (int64_t)blockIdx.x * kTileRows;
  const int rows = (int)((n - base < kTileRows) ? (n - base) : kTileRows);
  if (tid == 0) { sm.count = 0u; sm.n01 = 0u; sm.n2 = 0u; }
  {
    // L2 prefetch for a CTA that starts within the next residency (blockIdx.x + PIVOT_PREFETCH_DIST; 592 CTAs are resident at a
    // time; distances of 148 ... 296 measure alike, 592 is 0.3 % slower, 1184 1 % slower, none 2 % slower): its phase A
    // then finds its 40 (56) KB of inputs in L2 instead of waiting for HBM while nothing else of that CTA can run
    const int64_t pbase = base + (int64_t)PIVOT_PREFETCH_DIST * kTileRows;
    constexpr int kLines = kTileRows * 8 / 128;   // 128-byte lines per input array of a tile
    if (tid < kLines && pbase + kTileRows <= n) {
      const int64_t o = pbase + (int64_t)tid * 16;
      asm volatile("prefetch.global.L2 [%0];" ::"l"(in.S_or_F + o));
      asm volatile("prefetch.global.L2 [%0];" ::"l"(in.K + o));
      asm volatile("prefetch.global.L2 [%0];" ::"l"(in.tau + o));
      asm volatile("prefetch.global.L2 [%0];" ::"l"(in.P + o));
      asm volatile("prefetch.global.L2 [%0];" ::"l"(in.flag + o));
      if (BSM) {
        asm volatile("prefetch.global.L2 [%0];" ::"l"(in.r + o));
        asm volatile("prefetch.global.L2 [%0];" ::"l"(in.q + o));
      }
    }
  }
  __syncthreads();

  // ---- phase A: all rows of the tile.  1024-row tiles take it in two stages of two rows per thread (a rolled loop): half the
  //      code of four unrolled rows (the kernel's hot code has to fit the 32 KB instruction cache of the SM: hit rate 95.4 ->
  //      97.6 %, -2.4 % time on mixed rows) and half the registers in flight (no spills in BSM mode); the second stage's
  //      load latency is covered by the other CTAs of the SM.  Four stages of one row, and two stages on the 512-row tiles,
  //      measure slower.  Every load of a stage is issued before the first use.
  const double* __restrict__ gF = in.S_or_F + base;
  const double* __restrict__ gK = in.K + base;
  const double* __restrict__ gT = in.tau + base;
  const double* __restrict__ gP = in.P + base;
  const double* __restrict__ gf = in.flag + base;
  const double* __restrict__ gr = BSM ? in.r + base : nullptr;
  const double* __restrict__ gq = BSM ? in.q + base : nullptr;
  constexpr int NST = (RPT >= 4) ? 2 : 1;   // stages
  constexpr int HR = RPT / NST;             // rows per thread per stage
  unsigned rmask = 0;   // bit: row of this thread that needs the exact prelude
#pragma unroll 1
  for (int h = 0; h < NST; ++h) {
    double vF[HR], vK[HR], vT[HR], vP[HR], vf[HR], vr[HR], vq[HR];
    const int p0 = h * HR * kTileThreads + tid;
    if (rows == kTileRows) {   // full tile (all but the last one): plain loads
#pragma unroll
      for (int k = 0; k < HR; ++k) {
        const int p = p0 + k * kTileThreads;
        vF[k] = __ldcs(gF + p); vK[k] = __ldcs(gK + p); vT[k] = __ldcs(gT + p); vP[k] = __ldcs(gP + p); vf[k] = __ldcs(gf + p);
        vr[k] = BSM ? __ldcs(gr + p) : 0.0; vq[k] = BSM ? __ldcs(gq + p) : 0.0;
      }
    } else {
#pragma unroll
      for (int k = 0; k < HR; ++k) {
        const int p = p0 + k * kTileThreads;
        const bool live = p < rows;   // dead rows read as flag = 0: "rare" by the fast prelude, dropped below (p < rows)
        vF[k] = live ? __ldcs(gF + p) : 0.0; vK[k] = live ? __ldcs(gK + p) : 0.0; vT[k] = live ? __ldcs(gT + p) : 0.0;
        vP[k] = live ? __ldcs(gP + p) : 0.0; vf[k] = live ? __ldcs(gf + p) : 0.0;
        vr[k] = (BSM && live) ? __ldcs(gr + p) : 0.0; vq[k] = (BSM && live) ? __ldcs(gq + p) : 0.0;
      }
    }
    unsigned qmask = 0;   // bit k: row k of this stage is queued
#pragma unroll
    for (int k = 0; k < HR; ++k) {
      const int p = p0 + k * kTileThreads;
      const Prelude pr = lbr_prelude<BSM>(vF[k], vK[k], vT[k], vr[k], vq[k], vP[k], vf[k]);
      const bool queued = pr.status == 0;
      // staged unconditionally: the slots of dead rows (p >= rows) are never read, those of rare rows (status 5) are rewritten
      // by tile_rare_row below, and the vega slot of a queued row is rewritten in phase B1
      sm.status[p] = (uint8_t)pr.status;
      sm.sig[p] = queued ? vT[k] : (pr.status == 4 ? 0.0 : canonical_nan());
      sm.veg[p] = (BSM && queued) ? pr.D : 0.0;
      if (DIAG && !queued && p < rows && pr.status != 5) {
        if (dg.zone) dg.zone[base + p] = -1;
        if (dg.s0) dg.s0[base + p] = 0.0;
        if (dg.s1) dg.s1[base + p] = 0.0;
      }
      qmask |= queued ? (1u << k) : 0u;
      rmask |= (pr.status == 5 && p < rows) ? (1u << (h * HR + k)) : 0u;
      vF[k] = pr.U; vK[k] = pr.O; vP[k] = pr.B;   // what the solver pass needs
    }
    // Queue slots, warp by warp: within a warp and a stage the order is k-major then lane, so that a run of 32 CONSECUTIVE rows
    // stays contiguous in the queue (on option chains in strike order the dense warps of phase B1 then see neighbouring rows:
    // one zone).  HR ballots and one shared atomic per warp per stage.
    unsigned bal[HR];
    int total = 0;
#pragma unroll
    for (int k = 0; k < HR; ++k) {
      bal[k] = __ballot_sync(0xffffffffu, (qmask >> k) & 1u);
      total += __popc(bal[k]);
    }
    unsigned wbase = 0u;
    if (lane == 0 && total > 0) wbase = smem_atomic_add(&sm.count, vary, (unsigned)total);
    int slot = (int)__shfl_sync(0xffffffffu, wbase, 0);
    const unsigned lt = (1u << lane) - 1u;
#pragma unroll
    for (int k = 0; k < HR; ++k) {
      if ((qmask >> k) & 1u) {
        const int j = slot + __popc(bal[k] & lt);
        PIVOT_ASSERT(j >= 0 && j < kTileRows);
        sm.q0[j] = vF[k];
        sm.q1[j] = vK[k];
        sm.q2[j] = vP[k];
        sm.pos[j] = (uint16_t)(p0 + k * kTileThreads);
      }
      slot += __popc(bal[k]);
    }
  }
  if (rmask) {   // unusual rows: the exact prelude decides, from the row's inputs re-read (rare, divergent)
#pragma unroll 1
    for (int k = 0; k < RPT; ++k)
      if ((rmask >> k) & 1u) tile_rare_row<BSM, DIAG, RPT>(in, base, k * kTileThreads + tid, sm, dg);
  }
  __syncthreads();

  // ---- phase B1: normalisation, x, boundary point, node, zone; middle zones (1, 2) finished; rows regrouped by zone class
  //      lists: zone 0 (-> LOWER) from the front of perm, finished LINEAR rows from the back, zone 3 in permU
  const int cnt = (int)sm.count;
  for (int j0 = 0; j0 < cnt; j0 += kTileThreads) {   // j0 is CTA-uniform: every lane reaches the ballots
    const int j = j0 + tid;
    int cls = -1;  // 0: zone 0, 1: finished (zones 1, 2), 2: zone 3
    if (j < cnt) {
      const int pj = sm.pos[j];
      const Norm nm = lbr_normalise(sm.q0[j], sm.q1[j], sm.q2[j], (pj & 0x8000) != 0);
      const SeedHead hd = lbr_seed_head<FULL>(nm.qrel, nm.beta, nm.bbar, nm.bmax);
      sm.q0[j] = hd.v0; sm.q1[j] = hd.v1; sm.q2[j] = hd.v2; sm.q3[j] = hd.v3;
      const int p = pj & 0x3fff;
      PIVOT_ASSERT(p < rows);
      sm.veg[p] = BSM ? sm.veg[p] * nm.rootFK : nm.rootFK;    // D sqrt(FK)
      cls = (hd.zone == 0) ? 0 : ((hd.zone == 3) ? 2 : 1);
      if (DIAG && dg.zone) dg.zone[base + p] = (int8_t)hd.zone;
    }
    const unsigned m0 = __ballot_sync(0xffffffffu, cls == 0);
    const unsigned m1 = __ballot_sync(0xffffffffu, cls == 1);
    const unsigned m2 = __ballot_sync(0xffffffffu, cls == 2);
    // native 32-bit shared atomics hand out the list offsets: one for zone 0 / middle, one for zone 3 (if any)
    unsigned base01 = 0u, base2 = 0u;
    if (lane == 0) {
      base01 = smem_atomic_add(&sm.n01, vary, (unsigned)__popc(m0) | ((unsigned)__popc(m1) << 16));
      if (m2) base2 = smem_atomic_add(&sm.n2, vary, (unsigned)__popc(m2));
    }
    base01 = __shfl_sync(0xffffffffu, base01, 0);
    base2 = __shfl_sync(0xffffffffu, base2, 0);
    const int b0 = (int)(base01 & 0xffffu), b1 = (int)(base01 >> 16), b2 = (int)base2;
    const unsigned lt = (1u << lane) - 1u;
    PIVOT_ASSERT(cls != 0 || (b0 + __popc(m0 & lt) >= 0 && b0 + __popc(m0 & lt) < kTileRows));
    PIVOT_ASSERT(cls != 1 || (kTileRows - 1 - (b1 + __popc(m1 & lt)) >= 0 && b0 + b1 + __popc(m1 & lt) < kTileRows));
    PIVOT_ASSERT(cls != 2 || (b2 + __popc(m2 & lt) >= 0 && b2 + __popc(m2 & lt) < kTileRows));
    {
      // one store: perm and permU are adjacent (permU[i] = perm[kTileRows + i])
      static_assert(offsetof(TileSmem<RPT>, permU) == offsetof(TileSmem<RPT>, perm) + sizeof(uint16_t) * kTileRows, "perm | permU");
      const int r = __popc((cls == 0 ? m0 : (cls == 1 ? m1 : m2)) & lt);
      const int idx = (cls == 0) ? b0 + r : ((cls == 1) ? kTileRows - 1 - b1 - r : kTileRows + b2 + r);
      if (cls >= 0) sm.perm[idx] = (uint16_t)j;
    }
  }
  __syncthreads();

  // ---- phase B2: the tail seeds (zone 0 rows, zone 3 rows) fused with the Householder steps; rows ordered zone 0
  //      (LOWER), finished middle rows (LINEAR), zone 3 (UPPER or LINEAR): a warp sees one zone and one objective kind
  //      except at the two group boundaries
  const int n0 = (int)(sm.n01 & 0xffffu), n1 = (int)(sm.n01 >> 16);
  for (int k = tid; k < cnt; k += kTileThreads) {
    int j, kind;
    double x, s0, p1, p2;
    if (k < n0) {
      j = sm.perm[k];
      const Seed sd = lbr_seed_tail0<FULL>(sm.q0[j], sm.q1[j], sm.q2[j], sm.q3[j]);
      x = sd.x; s0 = sd.s; p1 = sd.p1; p2 = sd.p2; kind = KIND_LOWER;
    } else if (k < n0 + n1) {
      j = sm.perm[kTileRows - 1 - (k - n0)];
      if (FULL) {
        x = sm.q0[j]; s0 = sm.q1[j]; p1 = sm.q2[j]; p2 = sm.q3[j];
      } else {
        const Seed sd = lbr_seed_mid(sm.q0[j], sm.q1[j], sm.q2[j], sm.q3[j]);
        x = sd.x; s0 = sd.s; p1 = sd.p1; p2 = sd.p2;
      }
      kind = KIND_LINEAR;
    } else {
      j = sm.permU[k - n0 - n1];
      const Seed sd = lbr_seed_tail3<FULL>(sm.q0[j], sm.q1[j], sm.q2[j], sm.q3[j]);
      x = sd.x; s0 = sd.s; p1 = sd.p1; p2 = sd.p2; kind = sd.kind;
    }
    PIVOT_ASSERT(j >= 0 && j < cnt && cnt <= rows && n0 + n1 + (int)sm.n2 == cnt);
    const NormSolve ns = lbr_refine<kHouseholderSteps, FULL, true>(x, s0, p1, p2, kind);
    const int p = sm.pos[j] & 0x3fff;
    PIVOT_ASSERT(p < rows);
    const double tau = sm.sig[p];
    // 1/sqrt(tau): MUFU.RSQ64H + one third-order step for the common rows (tau positive normal, checked by the prelude); a rare row may carry
    // a subnormal tau and takes the library rsqrt
    const double rinv = (sm.pos[j] & 0x8000) ? rsqrt(tau) : rsqrt_c3(tau);
    sm.sig[p] = ns.s * rinv;
    sm.veg[p] = sm.veg[p] * ns.vfin * (tau * rinv);
    if (DIAG) {
      if (dg.s0) dg.s0[base + p] = s0;
      if (dg.s1) dg.s1[base + p] = ns.s1;
    }
  }
  __syncthreads();

  // ---- phase C
  if (rows == kTileRows) {   // full tile: no bounds tests, one address per array
    double* __restrict__ gs = sigma + base + tid;
    double* __restrict__ gv = vega + base + tid;
#pragma unroll
    for (int k = 0; k < RPT; ++k) {
      __stcs(gs + k * kTileThreads, sm.sig[k * kTileThreads + tid]);
      __stcs(gv + k * kTileThreads, sm.veg[k * kTileThreads + tid]);
    }
  } else {
#pragma unroll 1
    for (int p = tid; p < rows; p += kTileThreads) {
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
// Launch probe of PIVOT_FWD_AUTO (large launches only; see launch_auto): ONE warp looks at kProbeSegs groups of 32 consecutive
// rows spread over the arrays and counts the neighbour pairs that sit close to each other in (moneyness, time value over
// min(S, K), tau, carry): such rows follow the same branches of the solver, and row-per-thread is then the faster organisation
// (option chains in strike order).  Density does not enter: dense RANDOM rows are 12-19 % faster
// regrouped.  Close pairs of 124 on the workloads of DESIGN.md section 6: BSM chains 124, every other workload 0 ... 3.
// The test works on the raw inputs (BSM: S for F and P for P / D: along a chain carry and discount factor are common factors
// of neighbouring rows).  The verdict goes to the IF / ELSE node of the launch graph (handle) and / or to *verdict.
// ---------------------------------------------------------------------------------------------------------------
constexpr int kProbeSegs = 4;
constexpr int kProbeClosePairs = 93;   // of 31 kProbeSegs = 124: three quarters

template <bool BSM>
__global__ void __launch_bounds__(32) forward_probe_kernel(pivot_iv_inputs in, int64_t n, cudaGraphConditionalHandle handle,
                                                           int use_handle, int* verdict) {
  const int lane = threadIdx.x;
  int close_pairs = 0;
  if (n >= 32 * 2 * kProbeSegs) {
#pragma unroll
    for (int s = 0; s < kProbeSegs; ++s) {
      const int64_t i = ((((int64_t)(2 * s + 1) * (n / (2 * kProbeSegs))) >> 5) << 5) + lane;   // i + (31 - lane) < n
      const double F = in.S_or_F[i], K = in.K[i], T = in.tau[i], P = in.P[i], f = in.flag[i];
      const double c = BSM ? (in.r[i] - in.q[i]) * T : 0.0;
      const double lo = fmin(F, K), hi = fmax(F, K), iota = fmax(f * (F - K), 0.0);
      // fp32 is plenty; the quotients are formed in double first (F, K may lie outside the fp32 range).  NaN / Inf compare false.
      const float a = (float)(lo / hi), b = (float)((P - iota) / lo), t = (float)T, cf = (float)c;
      const float an = __shfl_down_sync(0xffffffffu, a, 1), bn = __shfl_down_sync(0xffffffffu, b, 1),
                  tn = __shfl_down_sync(0xffffffffu, t, 1), cn = __shfl_down_sync(0xffffffffu, cf, 1);
      const bool close = (lane < 31) & (fabsf(a - an) <= 0.05f) & (fabsf(b - bn) <= 0.05f) & (fabsf(t - tn) <= 0.125f * t) &
                         (fabsf(cf - cn) <= 0.05f);
      close_pairs += __popc(__ballot_sync(0xffffffffu, close));
    }
  }
  if (lane == 0) {
    const unsigned rowwise = close_pairs >= kProbeClosePairs ? 1u : 0u;
    if (use_handle) cudaGraphSetConditional(handle, rowwise);
    if (verdict) *verdict = (int)rowwise;
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
// grad_P may alias grad_sigma (include/pivot_iv.h).  INPLACE = false (distinct buffers): both pointers are __restrict__, so
// the loads of the next iteration may be hoisted over the stores of this one.  INPLACE = true (grad_P == grad_sigma):
// neither is, and a thread loads its rows before it stores them.
template <int MODE, bool INPLACE>
__global__ void __launch_bounds__(kBwdThreads)
backward_kernel_vec4(const double* gs_, const double* __restrict__ vega, const uint8_t* __restrict__ status,
                     double floor_, int64_t n4, double* gP_) {
  typedef const double* __restrict__ RIn;
  typedef double* __restrict__ ROut;
  const double* gs = INPLACE ? gs_ : static_cast<RIn>(gs_);
  double* gP = INPLACE ? gP_ : static_cast<ROut>(gP_);
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
backward_kernel_scalar(const double* gs, const double* __restrict__ vega, const uint8_t* __restrict__ status,
                       double floor_, int64_t begin, int64_t n, double* gP) {
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

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

}  // namespace pivot

// ===============================================================================================================
// C ABI
// ===============================================================================================================
using namespace pivot;

namespace {

constexpr int kMaxDevices = 64;

// cudaFuncSetAttribute applies to the CURRENT device only: remember per kernel and per device ordinal where the dynamic
// shared-memory opt-in has been made (a failure is not cached, it is retried by the next call).
template <auto Kernel>
int ensure_dynamic_smem(int bytes) {
  static std::atomic<unsigned long long> done{0ull};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return PIVOT_ERR_CUDA;
  if (dev >= 0 && dev < kMaxDevices && ((done.load(std::memory_order_relaxed) >> dev) & 1ull)) return PIVOT_OK;
  if (cudaFuncSetAttribute(Kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes) != cudaSuccess) {
    (void)cudaGetLastError();
    return PIVOT_ERR_CUDA;
  }
  if (dev >= 0 && dev < kMaxDevices) done.fetch_or(1ull << dev, std::memory_order_relaxed);
  return PIVOT_OK;
}

// SM count of the current device (cached per device ordinal)
int sm_count() {
  static std::atomic<int> cache[kMaxDevices];
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { (void)cudaGetLastError(); return 148; }
  if (dev >= 0 && dev < kMaxDevices) {
    const int c = cache[dev].load(std::memory_order_relaxed);
    if (c > 0) return c;
  }
  int sms = 0;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) {
    (void)cudaGetLastError();
    return 148;
  }
  if (dev >= 0 && dev < kMaxDevices) cache[dev].store(sms, std::memory_order_relaxed);
  return sms;
}

template <bool BSM, bool DIAG, int RPT, bool FULL>
int launch_tile(const pivot_iv_inputs& in, int64_t n, double* sigma, double* vega, uint8_t* status, const DiagOut& dg,
                cudaStream_t st) {
  const int rc = ensure_dynamic_smem<forward_kernel_tile<BSM, DIAG, RPT, FULL>>((int)sizeof(TileSmem<RPT>));
  if (rc != PIVOT_OK) return rc;
  const int64_t blocks = (n + RPT * kTileThreads - 1) / (RPT * kTileThreads);
  forward_kernel_tile<BSM, DIAG, RPT, FULL><<<(unsigned)blocks, kTileThreads, sizeof(TileSmem<RPT>), st>>>(in, n, sigma, vega,
                                                                                                         status, dg);
  return PIVOT_OK;
}

constexpr int64_t kAutoMinRows = PIVOT_AUTO_MIN_ROWS;
static_assert(kAutoMinRows == ((int64_t)3 << 23), "PIVOT_AUTO_MIN_ROWS");
template <bool BSM>
int launch_auto(const pivot_iv_inputs& in, int64_t n, double* sigma, double* vega, uint8_t* status, cudaStream_t st,
                bool* launched);   // below

template <bool BSM, bool DIAG, bool FULL>
int launch_forward_t(const pivot_iv_inputs& in, int64_t n, double* sigma, double* vega, uint8_t* status, const DiagOut& dg,
                     bool rowwise, bool autosel, cudaStream_t st) {
  int rc = PIVOT_OK;
  if (!DIAG && !FULL && autosel && n >= kAutoMinRows) {
    bool launched = false;
    rc = launch_auto<BSM>(in, n, sigma, vega, status, st, &launched);
    if (rc != PIVOT_OK || launched) return rc;
  }
  if (rowwise) {
    const int64_t blocks = (n + kFwdThreads - 1) / kFwdThreads;
    forward_kernel_scalar<BSM, DIAG, FULL><<<(unsigned)blocks, kFwdThreads, 0, st>>>(in, n, sigma, vega, status, dg);
  } else if (!DIAG && !FULL && n <= ((int64_t)1 << 17)) {
    // small launches use smaller tiles so that the grid still covers the chip and no SM is left with one long CTA:
    // 256-row tiles up to 2^17 rows, 512-row tiles up to 2^20 (kernel time from a CUDA graph, mixed / 1-solve rows, in us:
    // 2^18: 256-row 12.8 / 15.6, 512-row 10.5 / 17.0, 1024-row 11.9 / 18.6;  2^19: 22.8 / 28.0, 16.7 / 27.0, 18.4 / 31.3;
    // 2^20: 41.5 / 53.1, 29.9 / 50.0, 30.0 / 51.1)
    rc = launch_tile<BSM, false, 1, false>(in, n, sigma, vega, status, dg, st);
  } else if (!DIAG && !FULL && n <= ((int64_t)1 << 20)) {
    rc = launch_tile<BSM, false, 2, false>(in, n, sigma, vega, status, dg, st);
  } else {
    rc = launch_tile<BSM, DIAG, 4, FULL>(in, n, sigma, vega, status, dg, st);
  }
  if (rc != PIVOT_OK) return rc;
  return cudaGetLastError() == cudaSuccess ? PIVOT_OK : PIVOT_ERR_CUDA;
}

// ---------------------------------------------------------------------------------------------------------------
// PIVOT_FWD_AUTO on large launches (n >= kAutoMinRows): ONE graph launch = forward_probe_kernel -> IF / ELSE node ->
// forward_kernel_scalar (rows that follow each other closely) | forward_kernel_tile (everything else).  The choice is made on
// the device, between two separate kernels: every way tried to make it INSIDE one kernel cost the tile kernel more than it
// gained, because its hot code already fills the 32 KB instruction cache of the SM.  The graph costs
// ~20 us on the GPU time line (probe + conditional node + launch of the body: 1.519 -> 1.540 ms at 2^26 mixed rows, where the
// row-per-thread branch saves 9 % on option chains) and ~3 us of host time per call (three parameter updates + launch), hence
// the size limit: <= 3.5 % of a launch of kAutoMinRows rows.  One executable graph per device and mode, built on first use;
// calls are serialised by a mutex around update + launch (the launches themselves are asynchronous as ever; CUDA runs two launches
// of one executable graph one after the other, also from different streams: at these sizes each fills the GPU anyway).  During stream
// capture (a graph launch cannot be captured) and after any failure to build the graph the call takes the tile kernel.
// ---------------------------------------------------------------------------------------------------------------

struct AutoGraph {
  std::mutex mu;
  bool failed = false;
  cudaGraph_t graph = nullptr;
  cudaGraphExec_t exec = nullptr;
  cudaGraphNode_t probe = nullptr, row = nullptr, tile = nullptr;
  cudaGraphConditionalHandle handle{};
};

struct AutoArgs {   // argument storage the kernel-node parameter arrays point into
  pivot_iv_inputs in;
  int64_t n;
  double* sigma;
  double* vega;
  uint8_t* status;
  DiagOut dg;
  cudaGraphConditionalHandle handle;
  int use_handle;
  int* verdict;
};

template <bool BSM>
void auto_node_params(AutoArgs& a, void** pargs, void** fargs, cudaKernelNodeParams& kprobe, cudaKernelNodeParams& krow,
                      cudaKernelNodeParams& ktile) {
  pargs[0] = &a.in; pargs[1] = &a.n; pargs[2] = &a.handle; pargs[3] = &a.use_handle; pargs[4] = &a.verdict;
  fargs[0] = &a.in; fargs[1] = &a.n; fargs[2] = &a.sigma; fargs[3] = &a.vega; fargs[4] = &a.status; fargs[5] = &a.dg;
  kprobe = cudaKernelNodeParams{};
  kprobe.func = reinterpret_cast<void*>(forward_probe_kernel<BSM>);
  kprobe.gridDim = dim3(1); kprobe.blockDim = dim3(32); kprobe.kernelParams = pargs;
  krow = cudaKernelNodeParams{};
  krow.func = reinterpret_cast<void*>(forward_kernel_scalar<BSM, false, false>);
  krow.gridDim = dim3((unsigned)((a.n + kFwdThreads - 1) / kFwdThreads)); krow.blockDim = dim3(kFwdThreads); krow.kernelParams = fargs;
  ktile = cudaKernelNodeParams{};
  ktile.func = reinterpret_cast<void*>(forward_kernel_tile<BSM, false, 4, false>);
  ktile.gridDim = dim3((unsigned)((a.n + 4 * kTileThreads - 1) / (4 * kTileThreads))); ktile.blockDim = dim3(kTileThreads);
  ktile.sharedMemBytes = (unsigned)sizeof(TileSmem<4>); ktile.kernelParams = fargs;
}

// returns PIVOT_OK and *launched = true when the graph has been enqueued; *launched = false: the caller takes the tile kernel
template <bool BSM>
int launch_auto(const pivot_iv_inputs& in, int64_t n, double* sigma, double* vega, uint8_t* status, cudaStream_t st,
                bool* launched) {
  static AutoGraph graphs[kMaxDevices];
  *launched = false;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) { (void)cudaGetLastError(); return PIVOT_OK; }
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(st, &cs) != cudaSuccess) { (void)cudaGetLastError(); return PIVOT_OK; }
  if (cs != cudaStreamCaptureStatusNone) return PIVOT_OK;
  const int rc = ensure_dynamic_smem<forward_kernel_tile<BSM, false, 4, false>>((int)sizeof(TileSmem<4>));
  if (rc != PIVOT_OK) return rc;
  AutoGraph& g = graphs[dev];
  std::lock_guard<std::mutex> lock(g.mu);
  if (g.failed) return PIVOT_OK;
  AutoArgs a{in, n, sigma, vega, status, DiagOut{nullptr, nullptr, nullptr}, g.handle, 1, nullptr};
  void* pargs[5];
  void* fargs[6];
  cudaKernelNodeParams kprobe, krow, ktile;
  if (!g.exec) {
    bool ok = cudaGraphCreate(&g.graph, 0) == cudaSuccess &&
              cudaGraphConditionalHandleCreate(&g.handle, g.graph, 0, cudaGraphCondAssignDefault) == cudaSuccess;
    if (ok) {
      a.handle = g.handle;
      auto_node_params<BSM>(a, pargs, fargs, kprobe, krow, ktile);
      ok = cudaGraphAddKernelNode(&g.probe, g.graph, nullptr, 0, &kprobe) == cudaSuccess;
    }
    cudaGraphNodeParams cp{};
    if (ok) {
      cp.type = cudaGraphNodeTypeConditional;
      cp.conditional.handle = g.handle;
      cp.conditional.type = cudaGraphCondTypeIf;
      cp.conditional.size = 2;   // [0]: condition != 0 (row per thread), [1]: else (tile)
      cudaGraphNode_t cond = nullptr;
      ok = cudaGraphAddNode(&cond, g.graph, &g.probe, 1, &cp) == cudaSuccess;
    }
    ok = ok && cudaGraphAddKernelNode(&g.row, cp.conditional.phGraph_out[0], nullptr, 0, &krow) == cudaSuccess &&
         cudaGraphAddKernelNode(&g.tile, cp.conditional.phGraph_out[1], nullptr, 0, &ktile) == cudaSuccess &&
         cudaGraphInstantiate(&g.exec, g.graph, 0) == cudaSuccess;
    if (!ok) {
      (void)cudaGetLastError();
      if (g.graph) (void)cudaGraphDestroy(g.graph);
      g.graph = nullptr; g.exec = nullptr; g.failed = true;
      return PIVOT_OK;
    }
  } else {
    auto_node_params<BSM>(a, pargs, fargs, kprobe, krow, ktile);
    if (cudaGraphExecKernelNodeSetParams(g.exec, g.probe, &kprobe) != cudaSuccess ||
        cudaGraphExecKernelNodeSetParams(g.exec, g.row, &krow) != cudaSuccess ||
        cudaGraphExecKernelNodeSetParams(g.exec, g.tile, &ktile) != cudaSuccess) {
      (void)cudaGetLastError();
      g.failed = true;   // the executable graph may hold a partial update: never launched again
      return PIVOT_OK;
    }
  }
  if (cudaGraphLaunch(g.exec, st) != cudaSuccess) {   // e.g. after cudaDeviceReset: the plain launch reports what is really wrong
    (void)cudaGetLastError();
    g.failed = true;
    return PIVOT_OK;
  }
  *launched = true;
  return PIVOT_OK;
}

int forward_impl(const pivot_iv_inputs* in, int64_t n, double* sigma, double* vega, uint8_t* status, const DiagOut* dg,
                 cudaStream_t st, int kernel = PIVOT_FWD_AUTO) {
  if (!in) return PIVOT_ERR_NULL;
  const int org = kernel & ~PIVOT_FWD_FP64_ONLY;
  if (kernel < 0 || (org != PIVOT_FWD_AUTO && org != PIVOT_FWD_COMPACT && org != PIVOT_FWD_ROWWISE)) return PIVOT_ERR_BAD_ARG;
  if (n < 0) return PIVOT_ERR_BAD_N;
  if ((in->r == nullptr) != (in->q == nullptr)) return PIVOT_ERR_MIXED_RQ;
  if (n == 0) return PIVOT_OK;
  if (!in->S_or_F || !in->K || !in->tau || !in->P || !in->flag || !sigma || !vega || !status) return PIVOT_ERR_NULL;
  if (n > ((int64_t)1 << 37)) return PIVOT_ERR_BAD_N;  // grid.x limit
  const bool bsm = in->r != nullptr, full = (kernel & PIVOT_FWD_FP64_ONLY) != 0, rowwise = org == PIVOT_FWD_ROWWISE,
             autosel = org == PIVOT_FWD_AUTO;
  const DiagOut none{nullptr, nullptr, nullptr};
  const DiagOut& d = dg ? *dg : none;
#define PIVOT_DISPATCH(B, G, F) return launch_forward_t<B, G, F>(*in, n, sigma, vega, status, d, rowwise, autosel, st)
  if (dg) {
    if (bsm) { if (full) PIVOT_DISPATCH(true, true, true); PIVOT_DISPATCH(true, true, false); }
    if (full) PIVOT_DISPATCH(false, true, true);
    PIVOT_DISPATCH(false, true, false);
  }
  if (bsm) { if (full) PIVOT_DISPATCH(true, false, true); PIVOT_DISPATCH(true, false, false); }
  if (full) PIVOT_DISPATCH(false, false, true);
  PIVOT_DISPATCH(false, false, false);
#undef PIVOT_DISPATCH
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
    // overlapping but unequal ranges are the caller's error (the header allows grad_P == grad_sigma only)
    if (gs == gP) backward_kernel_vec4<MODE, true><<<(unsigned)blocks, kBwdThreads, 0, st>>>(gs, vega, status, floor_, n4, gP);
    else backward_kernel_vec4<MODE, false><<<(unsigned)blocks, kBwdThreads, 0, st>>>(gs, vega, status, floor_, n4, gP);
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
  return forward_impl(in, n, sigma, vega, status, nullptr, reinterpret_cast<cudaStream_t>(stream));
}

int pivot_iv_forward_ex(const pivot_iv_inputs* in, int64_t n, double* sigma, double* vega, uint8_t* status, int kernel,
                        pivot_iv_stream stream) {
  return forward_impl(in, n, sigma, vega, status, nullptr, reinterpret_cast<cudaStream_t>(stream), kernel);
}

int pivot_iv_forward_zones(const pivot_iv_inputs* in, int64_t n, double* sigma, double* vega, uint8_t* status,
                           int8_t* zone, pivot_iv_stream stream) {
  if (n > 0 && !zone) return PIVOT_ERR_NULL;
  const DiagOut dg{zone, nullptr, nullptr};
  return forward_impl(in, n, sigma, vega, status, &dg, reinterpret_cast<cudaStream_t>(stream));
}

int pivot_iv_forward_diag(const pivot_iv_inputs* in, int64_t n, double* sigma, double* vega, uint8_t* status,
                          int8_t* zone, double* s_seed, double* s_step1, int kernel, pivot_iv_stream stream) {
  const DiagOut dg{zone, s_seed, s_step1};
  return forward_impl(in, n, sigma, vega, status, &dg, reinterpret_cast<cudaStream_t>(stream), kernel);
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

int pivot_iv_forward_launches(int64_t n, int kernel) {
  return ((kernel & ~PIVOT_FWD_FP64_ONLY) == PIVOT_FWD_AUTO && !(kernel & PIVOT_FWD_FP64_ONLY) && n >= kAutoMinRows) ? 2 : 1;
}

int pivot_iv_forward_probe(const pivot_iv_inputs* in, int64_t n, int* rowwise, pivot_iv_stream stream) {
  if (!in || !rowwise) return PIVOT_ERR_NULL;
  if (n < 0) return PIVOT_ERR_BAD_N;
  if ((in->r == nullptr) != (in->q == nullptr)) return PIVOT_ERR_MIXED_RQ;
  if (!in->S_or_F || !in->K || !in->tau || !in->P || !in->flag) return PIVOT_ERR_NULL;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  if (in->r) forward_probe_kernel<true><<<1, 32, 0, st>>>(*in, n, cudaGraphConditionalHandle{}, 0, rowwise);
  else forward_probe_kernel<false><<<1, 32, 0, st>>>(*in, n, cudaGraphConditionalHandle{}, 0, rowwise);
  return cudaGetLastError() == cudaSuccess ? PIVOT_OK : PIVOT_ERR_CUDA;
}
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
    case PIVOT_ERR_STATIC_MAX: return "n exceeds PIVOT_STATIC_MAX_ROWS (65536), the capacity of the static staging of pivot_iv_forward_host_static";
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
  int host_access = PIVOT_HOST_AUTO;
  int last_path = PIVOT_HOST_STAGED;   // path of the last *_host call: PIVOT_HOST_STAGED or PIVOT_HOST_DIRECT
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

// Device alias of the pinned, device-accessible host range [h, h + bytes), or nullptr: pageable memory, memory the device cannot
// reach, or a range that does not lie inside one pinned allocation (both ends are looked up and must map consistently).
template <typename T>
T* mapped_alias(T* h, size_t bytes) {
  if (!h || bytes == 0) return nullptr;
  cudaPointerAttributes a0{}, a1{};
  const char* hb = reinterpret_cast<const char*>(h);
  if (cudaPointerGetAttributes(&a0, hb) != cudaSuccess || cudaPointerGetAttributes(&a1, hb + bytes - 1) != cudaSuccess) {
    (void)cudaGetLastError();
    return nullptr;
  }
  if (a0.type != cudaMemoryTypeHost || a1.type != cudaMemoryTypeHost || !a0.devicePointer || !a1.devicePointer) return nullptr;
  if (static_cast<const char*>(a1.devicePointer) - static_cast<const char*>(a0.devicePointer) != (ptrdiff_t)(bytes - 1)) return nullptr;
  return reinterpret_cast<T*>(a0.devicePointer);
}

// pivot_iv_forward_host without staging: ONE forward launch whose loads and stores go to the caller's pinned host arrays over
// PCIe (unified addressing: the kernels are the device path's own).  No cudaMemcpyAsync, no chunks, both link directions busy
// from one kernel: 4,194,304 labels 3.75 -> 3.40 ms, one 65,536-row batch 0.129 -> 0.069 ms (per-copy overhead gone).
// `applied` says whether the path was taken (every array pinned and device-accessible); if so the return value is the call's.
int pipeline_run_zero_copy(pivot_iv_pipeline* p, const pivot_iv_inputs* in, int64_t n, double* sigma, double* vega,
                           uint8_t* status, bool* applied) {
  *applied = false;
  const size_t bytes = (size_t)n * sizeof(double);
  pivot_iv_inputs din{mapped_alias(in->S_or_F, bytes), mapped_alias(in->K, bytes), mapped_alias(in->tau, bytes),
                      mapped_alias(in->r, bytes), mapped_alias(in->q, bytes), mapped_alias(in->P, bytes),
                      mapped_alias(in->flag, bytes)};
  double* dsig = mapped_alias(sigma, bytes);
  double* dveg = mapped_alias(vega, bytes);
  uint8_t* dst = mapped_alias(status, (size_t)n);
  const bool bsm = in->r != nullptr;
  if (!din.S_or_F || !din.K || !din.tau || !din.P || !din.flag || (bsm && (!din.r || !din.q)) || !dsig || !dveg || !dst) return PIVOT_OK;
  *applied = true;
  // PCIe-bound whatever the organisation; the row-per-thread kernel streams more evenly (49 against 47 GB/s) -- an explicit
  // choice of the caller is kept
  const int flags = p->fwd_kernel & PIVOT_FWD_FP64_ONLY, org = p->fwd_kernel & ~PIVOT_FWD_FP64_ONLY;
  const int kernel = ((org == PIVOT_FWD_AUTO) ? PIVOT_FWD_ROWWISE : org) | flags;
  cudaStream_t s = p->streams[0];
  int rc = forward_impl(&din, n, dsig, dveg, dst, nullptr, s, kernel);
  if (cudaStreamSynchronize(s) != cudaSuccess) { (void)cudaGetLastError(); rc = PIVOT_ERR_CUDA; }
  return rc;
}

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
  if (!bwd && p->host_access == PIVOT_HOST_AUTO) {   // every array pinned and reachable from the device: no staging at all
    bool applied = false;
    rc = pipeline_run_zero_copy(p, in, n, sigma, vega, status, &applied);
    if (applied) {
      p->last_path = PIVOT_HOST_DIRECT;
      (void)cudaSetDevice(prev);
      return rc;
    }
  }
  p->last_path = PIVOT_HOST_STAGED;
  // Chunks of more than 2^19 rows ramp up (2^19 or C/8 rows first, then doubling) and down again (halving what is left):
  // nothing overlaps the first chunk's H2D copies and the last chunk's D2H copies, so those two are kept short, while the
  // chunks in between stay large -- every cudaMemcpyAsync costs ~8 us of idle link (2^26 rows, forward + backward: 40 GB/s H2D
  // with 2^18-row chunks, 49 GB/s with 2^22; raw duplex link: 52.6).  Below 2^19 rows the extra copies cost more than they save.
  constexpr int64_t kRampFloor = (int64_t)1 << 19;
  const int64_t Cmin = (C <= kRampFloor) ? C : ((C / 8 > kRampFloor) ? ((C / 8) & ~(int64_t)1) : kRampFloor);
  int64_t c = 0, m = 0, up = Cmin;
  for (int64_t off = 0; off < n && rc == PIVOT_OK; off += m, ++c) {
    const int slot = (int)(c % p->nslots);
    const int64_t left = n - off;
    m = (up < C) ? up : C;
    up = (up < C) ? up * 2 : C;
    if (left < 2 * m) m = (left > Cmin) ? (((left + 1) / 2 + 1) & ~(int64_t)1) : left;   // tail: halve what is left (even sizes)
    if (m > left) m = left;
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
    rc = forward_impl(&din, m, d[7], d[8], p->st[slot], nullptr, s, p->fwd_kernel);
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
  const int org = kernel & ~PIVOT_FWD_FP64_ONLY;
  if (kernel < 0 || (org != PIVOT_FWD_AUTO && org != PIVOT_FWD_COMPACT && org != PIVOT_FWD_ROWWISE)) return PIVOT_ERR_BAD_ARG;
  p->fwd_kernel = kernel;
  return PIVOT_OK;
}

int pivot_iv_pipeline_set_host_access(pivot_iv_pipeline* p, int mode) {
  if (!p) return PIVOT_ERR_NULL;
  if (mode != PIVOT_HOST_AUTO && mode != PIVOT_HOST_STAGED) return PIVOT_ERR_BAD_ARG;
  p->host_access = mode;
  return PIVOT_OK;
}

int pivot_iv_pipeline_last_host_path(const pivot_iv_pipeline* p) { return p ? p->last_path : PIVOT_ERR_NULL; }

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

// ===============================================================================================================
// pivot_iv_forward_host_static: the host-array forward call for callers that must not allocate (code under CUDA graph
// capture, tight serving loops, harnesses that forbid cudaMalloc).  The device staging that a pipeline object obtains
// from cudaMalloc is here a file-scope array, held by every GPU that loads the library until the process exits:
// PIVOT_STATIC_MAX_ROWS rows of 9 doubles (S_or_F, K, tau, r, q, P, flag, sigma, vega) + 1 status byte = 4,784,128 B.
// In host code `g_static_stage` is a host-side stand-in for the symbol, NOT a device address: the address comes from
// cudaGetSymbolAddress, once per device, with that device current.
// Nothing in the array has to start at zero: every input byte the kernel reads is written by this call's own H2D copies
// first, and the kernel writes all n rows of the three outputs before they are copied back; rows n ... MAX keep the last
// call's contents and are never read.  Every call shares the array, so two calls that overlap on the GPU (different
// streams, no dependency between them) race; calls on one stream are ordered by the stream.
// ===============================================================================================================
static __device__ __align__(256) unsigned char g_static_stage[(size_t)PIVOT_STATIC_MAX_ROWS * (9 * sizeof(double) + 1)];

namespace {

// device address of g_static_stage on the CURRENT device (looked up once per device ordinal, then cached)
int static_stage_address(unsigned char** out) {
  static std::atomic<unsigned char*> cache[kMaxDevices];
  int dev = 0;
  PIVOT_CUDA_TRY(cudaGetDevice(&dev));
  if (dev >= 0 && dev < kMaxDevices) {
    unsigned char* c = cache[dev].load(std::memory_order_acquire);
    if (c) { *out = c; return PIVOT_OK; }
  }
  unsigned char* ptr = nullptr;
  PIVOT_CUDA_TRY(cudaGetSymbolAddress((void**)&ptr, g_static_stage));
  if (!ptr) return PIVOT_ERR_CUDA;
  if (dev >= 0 && dev < kMaxDevices) cache[dev].store(ptr, std::memory_order_release);
  *out = ptr;
  return PIVOT_OK;
}

}  // namespace

extern "C" {

int pivot_iv_forward_host_static(const pivot_iv_inputs* in, int64_t n, double* sigma, double* vega, uint8_t* status,
                                 pivot_iv_stream stream) {
  if (!in) return PIVOT_ERR_NULL;
  if (n < 0) return PIVOT_ERR_BAD_N;
  if (n > PIVOT_STATIC_MAX_ROWS) return PIVOT_ERR_STATIC_MAX;
  if ((in->r == nullptr) != (in->q == nullptr)) return PIVOT_ERR_MIXED_RQ;
  if (n == 0) return PIVOT_OK;
  if (!in->S_or_F || !in->K || !in->tau || !in->P || !in->flag || !sigma || !vega || !status) return PIVOT_ERR_NULL;
  unsigned char* stage = nullptr;
  const int rc0 = static_stage_address(&stage);
  if (rc0 != PIVOT_OK) return rc0;
  cudaStream_t s = reinterpret_cast<cudaStream_t>(stream);
  double* d[9];
  for (int k = 0; k < 9; ++k) d[k] = reinterpret_cast<double*>(stage) + (size_t)k * PIVOT_STATIC_MAX_ROWS;
  uint8_t* dst = stage + (size_t)9 * PIVOT_STATIC_MAX_ROWS * sizeof(double);
  const bool bsm = in->r != nullptr;
  const size_t bytes = (size_t)n * sizeof(double);
  const double* src[7] = {in->S_or_F, in->K, in->tau, in->r, in->q, in->P, in->flag};
  for (int k = 0; k < 7; ++k)
    if (src[k]) PIVOT_CUDA_TRY(cudaMemcpyAsync(d[k], src[k], bytes, cudaMemcpyHostToDevice, s));
  const pivot_iv_inputs din{d[0], d[1], d[2], bsm ? d[3] : nullptr, bsm ? d[4] : nullptr, d[5], d[6]};
  // an explicit organisation: the default call's probe + graph launch starts far above PIVOT_STATIC_MAX_ROWS anyway
  const int rc = forward_impl(&din, n, d[7], d[8], dst, nullptr, s, PIVOT_FWD_COMPACT);
  if (rc != PIVOT_OK) return rc;
  PIVOT_CUDA_TRY(cudaMemcpyAsync(sigma, d[7], bytes, cudaMemcpyDeviceToHost, s));
  PIVOT_CUDA_TRY(cudaMemcpyAsync(vega, d[8], bytes, cudaMemcpyDeviceToHost, s));
  PIVOT_CUDA_TRY(cudaMemcpyAsync(status, dst, (size_t)n, cudaMemcpyDeviceToHost, s));
  return PIVOT_OK;
}

}  // extern "C"
