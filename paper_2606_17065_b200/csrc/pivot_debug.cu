// pivot_debug.cu -- test-only export of the device math library (lbr_device.cuh): pivot_iv_debug_math evaluates one
// function elementwise so that tests/test_gpu_mathlib.py can measure its error against mpmath on the device itself
// (FMA contraction, MUFU seeds and the range branches included).  Not on the hot path.
#include <cuda_runtime.h>

#include <cstdint>

#include "../../include/pivot_iv.h"
#include "lbr_device.cuh"

namespace pivot {

__global__ void __launch_bounds__(256)
debug_math_kernel(int fn, const double* __restrict__ a, const double* __restrict__ b, int64_t n, double* __restrict__ out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double x = a[i], y = b ? b[i] : 0.0;
  double r = 0.0, e1, e2;
  switch (fn) {
    case PIVOT_DBG_ERFCX_ONE: r = erfcx_one(x); break;
    case PIVOT_DBG_ERFCX_PAIR_1: erfcx_pair(x, y, e1, e2); r = e1; break;
    case PIVOT_DBG_ERFCX_PAIR_2: erfcx_pair(x, y, e1, e2); r = e2; break;
    case PIVOT_DBG_ERFCX_SEED: r = (double)erfcx_seed(__double2float_rn(x)); break;
    case PIVOT_DBG_EXP_FAST: r = exp_fast(x); break;
    case PIVOT_DBG_EXP_SEED: r = exp_seed(x); break;
    case PIVOT_DBG_LOG_FAST: r = log_fast(x); break;
    case PIVOT_DBG_LOG_SEED: r = log_seed(x); break;
    case PIVOT_DBG_LOG1P_FAST: r = log1p_fast(x); break;
    case PIVOT_DBG_RCP_NR1: r = rcp_nr1(x); break;
    case PIVOT_DBG_RCP_NR2: r = rcp_nr2(x); break;
    case PIVOT_DBG_DIV_FAST: r = div_fast(x, y); break;
    case PIVOT_DBG_SQRT_NR1: r = sqrt_nr1(x); break;
    case PIVOT_DBG_SQRT_NR2: r = sqrt_nr2(x); break;
    case PIVOT_DBG_RSQRT_NR2: (void)sqrt_nr2(x, r); break;
    case PIVOT_DBG_NINV_TAIL_SEED: r = (double)ninv_tail_seed(__double2float_rn(x)); break;
    case PIVOT_DBG_NINV_TAIL_FULL: r = ninv_tail_full(x); break;
    case PIVOT_DBG_EXPF_SEED: r = (double)expf_seed(__double2float_rn(x)); break;
    case PIVOT_DBG_LOGF_SEED: r = (double)logf_seed(__double2float_rn(x)); break;
    case PIVOT_DBG_ERFCX_DD_DIFF: r = erfcx_dd(x, x + y, y, false); break;
    case PIVOT_DBG_ERFCX_DD_SUM: r = erfcx_dd(x, x + y, y, true); break;
    case PIVOT_DBG_ERFCX_DD_SEED_DIFF:
    case PIVOT_DBG_ERFCX_DD_SEED_SUM: {
      const float z1 = __double2float_rn(x), d = __double2float_rn(y);
      r = (double)erfcx_dd_seed(z1, z1 + d, d, fn == PIVOT_DBG_ERFCX_DD_SEED_SUM);
      break;
    }
    case PIVOT_DBG_W_FULL: { const WEval w = eval_W<false>(x, y); r = w.have_W ? w.Wd : -w.Wd; break; }
    case PIVOT_DBG_W_SEED: { const WEval w = eval_W<true>(x, y); r = w.have_W ? w.Wd : -w.Wd; break; }
    case PIVOT_DBG_RCP_RAW: r = rcp_raw(x); break;
    case PIVOT_DBG_RSQRT_C3: r = rsqrt_c3(x); break;
    default: r = canonical_nan(); break;
  }
  out[i] = r;
}

}  // namespace pivot

extern "C" int pivot_iv_debug_math(int fn, const double* a, const double* b, int64_t n, double* out, pivot_iv_stream stream) {
  if (n < 0) return PIVOT_ERR_BAD_N;
  if (fn < 0 || fn >= PIVOT_DBG_COUNT) return PIVOT_ERR_BAD_ARG;
  if (n == 0) return PIVOT_OK;
  if (!a || !out) return PIVOT_ERR_NULL;
  const bool two = fn == PIVOT_DBG_ERFCX_PAIR_1 || fn == PIVOT_DBG_ERFCX_PAIR_2 || fn == PIVOT_DBG_DIV_FAST ||
                   (fn >= PIVOT_DBG_ERFCX_DD_DIFF && fn <= PIVOT_DBG_W_SEED);
  if (two && !b) return PIVOT_ERR_NULL;
  const int64_t blocks = (n + 255) / 256;
  if (blocks > 0x7fffffff) return PIVOT_ERR_BAD_N;
  pivot::debug_math_kernel<<<(unsigned)blocks, 256, 0, reinterpret_cast<cudaStream_t>(stream)>>>(fn, a, two ? b : nullptr, n, out);
  return cudaGetLastError() == cudaSuccess ? PIVOT_OK : PIVOT_ERR_CUDA;
}
