/* include/pivot_iv.h -- C ABI of the PIVOT implied-volatility hot path for NVIDIA B200 (sm_100a).
 *
 * One data-parallel path (arxiv/paper_2606_17065, "PIVOT"): batched, row-independent fp64 inversion of
 * Black-76 / Black-Scholes-Merton prices to implied volatility with the "Let's Be Rational" construction in
 * the forward pass, fused with the Black vega and a status byte; and a separate fused elementwise backward
 * pass  grad_P = gate * grad_sigma / vega  by implicit differentiation (never through the solver branches).
 * Citations are /root/reference/PAPER.md line numbers (section / equation given alongside).
 *
 * Conventions for every entry point
 *   - plain C, no C++ exceptions cross the boundary; returns 0 (PIVOT_OK) or a negative PIVOT_ERR_* code;
 *   - per-row numerical problems are never error codes, they are `status` values;
 *   - the library never allocates, frees or retains caller memory, keeps no global mutable state that changes a result
 *     (state lives inside an explicit pivot_iv_pipeline object; per device ordinal it caches, thread-safely, what it would
 *     otherwise look up on every call: kernel attributes, the SM count, the launch graph of the default forward call, the
 *     address of the static staging array of pivot_iv_forward_host_static), reads no environment variable, and the device
 *     entry points never synchronise the host:
 *     work is enqueued on `stream` (a cudaStream_t passed as an opaque pointer; NULL = the legacy default stream);
 *   - all arrays are SoA, contiguous, length n, fp64 unless stated; pointers need only their natural alignment
 *     (8 B for double): the forward kernel uses 8-byte accesses throughout, the backward kernel has a 16-B-aligned
 *     vector path and a scalar path; there is no CPU fallback;
 *   - n == 0 is a successful no-op.
 */
#ifndef PIVOT_IV_H_
#define PIVOT_IV_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PIVOT_IV_VERSION 100 /* major*10000 + minor*100 + patch */

/* error codes */
#define PIVOT_OK 0
#define PIVOT_ERR_NULL (-1)      /* a required pointer is NULL */
#define PIVOT_ERR_BAD_N (-2)     /* n < 0 */
#define PIVOT_ERR_BAD_MODE (-3)  /* mode not PIVOT_GATE_MASK / PIVOT_GATE_ATTENUATE / PIVOT_GATE_STRICT */
#define PIVOT_ERR_BAD_FLOOR (-4) /* vega_floor is NaN or negative */
#define PIVOT_ERR_MIXED_RQ (-5)  /* exactly one of r, q is NULL */
#define PIVOT_ERR_CUDA (-6)      /* CUDA runtime error (launch, copy, allocation inside a pipeline) */
#define PIVOT_ERR_BAD_ARG (-7)   /* other invalid argument (pipeline geometry, device index) */
#define PIVOT_ERR_STATIC_MAX (-8) /* pivot_iv_forward_host_static: n > PIVOT_STATIC_MAX_ROWS */

/* per-row status byte written by the forward pass (PAPER.md:98 Alg.1 l.3, :125, :363; readings in DESIGN.md) */
#define PIVOT_ST_OK 0              /* sigma, vega valid */
#define PIVOT_ST_BELOW_INTRINSIC 1 /* undiscounted price < max(theta (F-K), 0)        -> sigma = NaN, vega = 0 */
#define PIVOT_ST_ABOVE_MAX 2       /* undiscounted price >= F (call) or >= K (put)     -> sigma = NaN, vega = 0 */
#define PIVOT_ST_BAD_INPUT 3       /* tau <= 0, non-finite or non-positive S|F, K, non-finite P, r, q, flag not +-1,
                                      or |ln(F/K)| > 693, or F K overflows / underflows in fp64 (sqrt(F K) must be a
                                      positive normal number: e.g. F = K = 2e154 is rejected) -> sigma = NaN, vega = 0 */
#define PIVOT_ST_AT_INTRINSIC 4    /* time value is zero or subnormal after normalisation -> sigma = +0, vega = 0 */

/* gate modes of the backward pass (eq.(9), :148-150 eq.(10)) */
#define PIVOT_GATE_MASK 0      /* hard mask 1{|V| > vega_floor} */
#define PIVOT_GATE_ATTENUATE 1 /* smooth gate w(V) = V^2 / (V^2 + vega_floor^2) */
#define PIVOT_GATE_STRICT 2    /* exact gradient on {OK, |V| > vega_floor}; elsewhere +0 if the upstream
                                  cotangent is 0, NaN otherwise (an ill-conditioned gradient was explicitly asked for) */

/* Row tuple as parallel arrays (PAPER.md:123 "every input is treated as a tensor"; :51 xi = (S,K,tau,r,q), theta).
 * For the device entry points these are DEVICE pointers; for the *_host entry points HOST pointers. */
typedef struct pivot_iv_inputs {
  const double* S_or_F; /* spot S (BSM mode) or forward F (Black-76 mode) */
  const double* K;      /* strike */
  const double* tau;    /* time to expiry in years */
  const double* r;      /* risk-free rate;   r and q both NULL => Black-76 with discount factor 1 */
  const double* q;      /* dividend yield;   r and q both non-NULL => BSM: F = S e^{(r-q) tau}, D = e^{-r tau} */
  const double* P;      /* observed (discounted) option price P* */
  const double* flag;   /* theta: +1.0 call, -1.0 put; anything else => PIVOT_ST_BAD_INPUT */
} pivot_iv_inputs;

typedef struct CUstream_st* pivot_iv_stream; /* == cudaStream_t */

/* Forward pass, one fused kernel (PAPER.md:94-98 Alg.1 l.1-3; :359-363 A.5 stages 1-5; :322 eq.(14)).
 * Per row: normalise (F = S e^{(r-q)tau}, x = ln(F/K), beta = e^{r tau} P / sqrt(FK)); validity -> status; reduce to an
 * OTM call (x <= 0); LBR boundary point and four-zone rational initial guess; two Householder(3) steps on the zone's
 * transformed objective; sigma = s / sqrt(tau); vega = dP/dsigma = D sqrt(FK) phi0 exp(-(h^2+t^2)/2) sqrt(tau).
 *   in      device pointers (see pivot_iv_inputs), read only
 *   n       number of rows, >= 0
 *   sigma   [out, device, n doubles] implied volatility; canonical quiet NaN (0x7ff8000000000000) for status 1-3, +0 for 4
 *   vega    [out, device, n doubles] Black vega (per unit of sigma, not per 1%); 0 when status != 0
 *   status  [out, device, n bytes]   PIVOT_ST_*
 *   stream  CUDA stream the kernel is enqueued on
 * Outputs must not alias inputs.  Returns PIVOT_ERR_NULL / _BAD_N / _MIXED_RQ / _CUDA. */
int pivot_iv_forward(const pivot_iv_inputs* in, int64_t n, double* sigma, double* vega, uint8_t* status,
                     pivot_iv_stream stream);

/* Forward pass with an explicit kernel organisation and precision tier:
 *   PIVOT_FWD_COMPACT  rows that need the solver are compacted and regrouped by LBR zone in shared memory before the
 *                      solver passes run: best when the batch is mixed (degenerate / invalid rows, zones in random order);
 *   PIVOT_FWD_ROWWISE  one row per thread, no shared memory, no barriers: best when nearly every row solves and
 *                      neighbouring rows are alike (option chains in strike order);
 *   PIVOT_FWD_AUTO     what pivot_iv_forward uses: COMPACT below PIVOT_AUTO_MIN_ROWS rows; from there on the choice is made
 *                      on the device, inside ONE graph launch: a one-warp probe kernel reads 4 x 32 rows spread over the
 *                      arrays and an IF / ELSE graph node runs ROWWISE if at least three quarters of the neighbour pairs
 *                      sit close to each other in (moneyness, time value, tau, carry), else COMPACT (~20 us on the GPU time
 *                      line, ~3 us of host time; serialised per device by a mutex around the launch).  A call made while
 *                      the stream is being captured takes COMPACT (a graph launch cannot be captured).
 * COMPACT and ROWWISE run the same per-row arithmetic: bit-identical results, whichever AUTO picks.
 *   PIVOT_FWD_FP64_ONLY (flag, OR it into any of the three): every special function, reciprocal and interpolant of the
 *                      seed and of the first Householder step at full fp64 instead of "seed grade" (fp32 erfcx, MUFU
 *                      exp / log, fp32 rational cubics).  The default tiering only has to land inside the basin of the
 *                      last, full-precision Householder step (PAPER.md:125 says fp64 throughout; DESIGN.md section 5
 *                      bounds what the tiering changes: the two agree to <= 1e-13 relative in sigma).  Diagnostic / A-B.
 * Returns PIVOT_ERR_BAD_ARG for any other value. */
#define PIVOT_FWD_AUTO 0
#define PIVOT_FWD_COMPACT 1
#define PIVOT_FWD_ROWWISE 2
#define PIVOT_FWD_FP64_ONLY 4
#define PIVOT_AUTO_MIN_ROWS 25165824 /* 3 * 2^23 */
int pivot_iv_forward_ex(const pivot_iv_inputs* in, int64_t n, double* sigma, double* vega, uint8_t* status, int kernel,
                        pivot_iv_stream stream);

/* As pivot_iv_forward, additionally writing the LBR zone taken by each OK row (0 lower tail, 1 lower middle,
 * 2 upper middle, 3 upper tail; -1 when status != 0).  Diagnostics only: zone edges are transcendental, so this
 * byte is not bit-reproducible across implementations and is not part of `status`. */
int pivot_iv_forward_zones(const pivot_iv_inputs* in, int64_t n, double* sigma, double* vega, uint8_t* status,
                           int8_t* zone, pivot_iv_stream stream);

/* Diagnostics of the solve (rational seed, then Householder(3) steps), per row, in total
 * volatility s = sigma sqrt(tau):
 *   zone     [out, device, n bytes or NULL]    as pivot_iv_forward_zones
 *   s_seed   [out, device, n doubles or NULL]  the rational initial guess s0 (0 when status != 0)
 *   s_step1  [out, device, n doubles or NULL]  the iterate after the first Householder(3) step, i.e. what the last,
 *                                              full-precision step starts from (0 when status != 0)
 *   kernel   PIVOT_FWD_* as in pivot_iv_forward_ex
 * sigma / vega / status as pivot_iv_forward (same bits).  Used by the tests that bound the seed-grade tier. */
int pivot_iv_forward_diag(const pivot_iv_inputs* in, int64_t n, double* sigma, double* vega, uint8_t* status,
                          int8_t* zone, double* s_seed, double* s_step1, int kernel, pivot_iv_stream stream);

/* Backward pass, one fused elementwise kernel (PAPER.md:100-103 Alg.1 l.4-6; :107 eq.(7); :131 eq.(8) first half;
 * :144 eq.(9); :150 eq.(10)).  Reads only what the forward emitted: 25 B per row.
 *   MASK:      grad_P = grad_sigma / vega                              if status == OK and |vega| > vega_floor (strict)
 *   ATTENUATE: grad_P = grad_sigma * vega / (vega^2 + vega_floor^2)    if status == OK   (= w(V) grad_sigma / V)
 *   otherwise  grad_P = +0.0 exactly (by select, so 0*NaN never leaks).
 *   STRICT:    grad_P = grad_sigma / vega if status == OK and |vega| > vega_floor; else +0.0 if grad_sigma == 0, else NaN.
 *   grad_sigma, vega [in, device, n doubles]; status [in, device, n bytes]; grad_P [out, device, n doubles], may
 *   alias grad_sigma.  Returns PIVOT_ERR_NULL / _BAD_N / _BAD_MODE / _BAD_FLOOR / _CUDA. */
int pivot_iv_backward(const double* grad_sigma, const double* vega, const uint8_t* status, double vega_floor,
                      int mode, int64_t n, double* grad_P, pivot_iv_stream stream);

/* ---- next rows of the path ---- */
/* The smooth Black price node P_BSM(xi, sigma; theta) and its vega (eq.(2)/(3); :322 eq.(14)): what the
 * price loss eq.(11) and the round trip of eq.(12) evaluate.  Evaluated as
 * D (intrinsic + sqrt(FK) b(x, sigma sqrt(tau))) so that deep in-the-money rows keep their time value.
 *   in      device pointers; in->P is not read and may be NULL; r = q = NULL selects Black-76 with D = 1
 *   sigma   [in, device, n doubles] volatility; 0 gives the discounted intrinsic value; negative / NaN / bad inputs give NaN
 *   price   [out, device, n doubles]; vega [out, device, n doubles] may be NULL.
 * Returns PIVOT_ERR_NULL / _BAD_N / _MIXED_RQ / _CUDA. */
int pivot_iv_black_price(const pivot_iv_inputs* in, const double* sigma, int64_t n, double* price, double* vega,
                      pivot_iv_stream stream);

/* Full vector-Jacobian product of eq.(8), one fused elementwise kernel:
 *   grad_P = gate * grad_sigma / vega            (exactly pivot_iv_backward's value, same gate and modes)
 *   xi_bar = -grad_P * dP/dxi at sigma = sigma_imp, xi = (S, K, tau, r, q) in BSM mode, (F, K, tau) in Black-76 mode,
 * with the analytic derivatives of the discounted price eq.(2) (the paper differentiates a price helper by autograd):
 *   dP/dS = theta e^{-q tau} Phi(theta d1), dP/dK = -theta e^{-r tau} Phi(theta d2), dP/dr = theta K tau e^{-r tau} Phi(theta d2),
 *   dP/dq = -theta S tau e^{-q tau} Phi(theta d1), dP/dtau = theta[-q S e^{-q tau} Phi(theta d1) + r K e^{-r tau} Phi(theta d2)] + V sigma/(2 tau).
 * Rows that are not OK or off-gate get exactly +0.0 in every output.
 *   in, sigma, vega, status  the forward's inputs and outputs (device); in->P is not read
 *   grad_sigma [in, n]; grad_P, grad_S_or_F, grad_K, grad_tau [out, n]; grad_r, grad_q [out, n] required iff BSM mode.
 * Returns PIVOT_ERR_NULL / _BAD_N / _BAD_MODE / _BAD_FLOOR / _MIXED_RQ / _CUDA. */
int pivot_iv_backward_inputs(const pivot_iv_inputs* in, const double* sigma, const double* vega, const uint8_t* status,
                             const double* grad_sigma, double vega_floor, int mode, int64_t n, double* grad_P,
                             double* grad_S_or_F, double* grad_K, double* grad_tau, double* grad_r, double* grad_q,
                             pivot_iv_stream stream);

/* The two PIVOT objectives as sums, so that the caller normalises by the rows used, each fused with its
 * gradient with respect to sigma_hat in the same pass (one kernel each; every intermediate in registers, no workspace):
 *   eq.(11)  L_price = (out3[0]/out3[2]) / (out3[1]/out3[2])^2,  out3 += { sum (P_BS(xi, sigma_hat) - P*)^2, sum |P*|, rows used }
 *            grad_sigma_hat[i] = grad_scale * 2 (P_BS - P*) V_hat           (V_hat = vega at sigma_hat; eq.(14))
 *   eq.(12)  L_rt    =  out3[0]/out3[2],                         out3 += { sum w (JaeckelIV(P~) - sigma*)^2, sum w, rows used },
 *            w = V_hat^2/(V_hat^2 + vega_floor^2) (eq.(10)), P~ = the model price where |V_hat| > vega_floor, else the sentinel
 *            market price P* (in->P), which carries no gradient; the inversion is the forward pass's own per-row arithmetic.
 *            grad_sigma_hat[i] = grad_scale * { [|V_hat| > floor] w 2 (sigma_rt - sigma*) (1/V_rt) V_hat
 *                                               + w'(V_hat) (sigma_rt - sigma*)^2 dV_hat/dsigma_hat }
 *            -- eq.(17): the 1/V_rt of the inverse channel (MASK rule at vega_floor) against the V_hat of the
 *            price node; w' = 2 V floor^2/(V^2 + floor^2)^2, dV/dsigma = V d1 d2 / sigma.
 *   mode PIVOT_RT_NAIVE (the NaN-poisoning diagnostic): no gate, no sentinel, no sanitisation:
 *            out3 += { sum (JaeckelIV(P_BS(sigma_hat)) - sigma*)^2, rows, rows },
 *            grad_sigma_hat[i] = grad_scale * STRICT(2 (sigma_rt - sigma*), V_rt; vega_floor) V_hat: NaN wherever the inverse channel is
 *            singular (|V_rt| <= vega_floor or the inversion is not OK) unless the cotangent is exactly 0; a row with a non-finite
 *            sigma_hat contributes NaN to the sum and to its gradient.
 * Rows with a non-finite model price or P* are skipped by (11); rows whose inversion is not OK or whose sigma* is not finite
 * by the gated (12); skipped rows have gradient +0.
 *   out3 [device, 3 doubles] is ACCUMULATED into (zero it first).  sigma_hat, sigma_star [in, device, n doubles].
 *   grad_sigma_hat [out, device, n doubles] or NULL (sums only); grad_scale: the caller's normalisation, e.g. 1/(|B| m^2) with
 *   m = mean |P*| for eq.(11), 1/|B| for eq.(12).
 * Returns PIVOT_ERR_NULL / _BAD_N / _BAD_FLOOR / _BAD_MODE / _MIXED_RQ / _CUDA. */
#define PIVOT_RT_GATED 0
#define PIVOT_RT_NAIVE 1
int pivot_iv_loss_price(const pivot_iv_inputs* in, const double* sigma_hat, int64_t n, double* out3, double* grad_sigma_hat,
                        double grad_scale, pivot_iv_stream stream);
int pivot_iv_loss_roundtrip(const pivot_iv_inputs* in, const double* sigma_hat, const double* sigma_star, double vega_floor,
                            int mode, int64_t n, double* out3, double* grad_sigma_hat, double grad_scale,
                            pivot_iv_stream stream);

/* Status histogram (diagnostics): counts6[k] += number of rows with status k for k = PIVOT_ST_OK ..
 * PIVOT_ST_AT_INTRINSIC (0..4), counts6[5] += rows with any other byte.
 *   status  [in, device, n bytes], any alignment;  counts6 [device, 6 x uint64] is ACCUMULATED into (zero it first).
 * Asynchronous on `stream`.  Returns PIVOT_ERR_BAD_N / PIVOT_ERR_NULL / PIVOT_ERR_CUDA. */
int pivot_iv_status_histogram(const uint8_t* status, int64_t n, unsigned long long* counts6, pivot_iv_stream stream);

/* ---- host-buffer pipeline (the streaming label-generation setting: batches of rows, H2D included) ----
 * A pipeline owns `n_slots` device staging slots of `chunk_rows` rows each, one CUDA stream per slot and pinned
 * bounce buffers are NOT used: host arrays are copied directly (pin them for full PCIe speed).  The *_host calls split
 * the n rows into chunks of at most `chunk_rows` rows (with chunk_rows > 2^19 the first chunks ramp up from 2^19 or
 * chunk_rows/8 rows by doubling and the last ones halve what is left, so that the copies nothing overlaps stay short),
 * overlap H2D copy, kernels and D2H copy across slots, and return after the last byte of output is in host memory (they
 * synchronise).  Not thread-safe per pipeline object. */
typedef struct pivot_iv_pipeline pivot_iv_pipeline;

/* Creates a pipeline on CUDA device `device` (-1 = current).  chunk_rows > 0, 1 <= n_slots <= 8. */
int pivot_iv_pipeline_create(pivot_iv_pipeline** out, int device, int64_t chunk_rows, int n_slots);
int pivot_iv_pipeline_destroy(pivot_iv_pipeline* p);
/* Kernel organisation the pipeline's forward launches use (PIVOT_FWD_*; default AUTO). */
int pivot_iv_pipeline_set_forward_kernel(pivot_iv_pipeline* p, int kernel);
/* How pivot_iv_forward_host reaches the caller's host arrays (default PIVOT_HOST_AUTO):
 *   PIVOT_HOST_AUTO    if EVERY input and output array is pinned (cudaHostAlloc / cudaHostRegister) and addressable from the
 *                      pipeline's device, ONE forward launch loads and stores the host arrays directly over PCIe (unified
 *                      addressing; the device path's own kernels, same bits; row-per-thread unless
 *                      pivot_iv_pipeline_set_forward_kernel chose otherwise): no staging, no cudaMemcpyAsync, no chunks.
 *                      Otherwise (any array pageable) the staged path below.
 *   PIVOT_HOST_STAGED  always the chunked H2D copy -> kernels -> D2H copy path through the staging slots.
 * pivot_iv_forward_backward_host always takes the staged path (the backward reads what the forward wrote: vega and status
 * stay in device memory between the two kernels).  Returns PIVOT_ERR_NULL / PIVOT_ERR_BAD_ARG. */
#define PIVOT_HOST_AUTO 0
#define PIVOT_HOST_STAGED 1
#define PIVOT_HOST_DIRECT 2   /* reported only: the last call ran straight on the host arrays */
int pivot_iv_pipeline_set_host_access(pivot_iv_pipeline* p, int mode);
/* Path the last *_host call of this pipeline took: PIVOT_HOST_STAGED or PIVOT_HOST_DIRECT (PIVOT_ERR_NULL for p == NULL). */
int pivot_iv_pipeline_last_host_path(const pivot_iv_pipeline* p);

/* Forward on HOST arrays: `in`, sigma, vega, status are host pointers (length n). */
int pivot_iv_forward_host(pivot_iv_pipeline* p, const pivot_iv_inputs* in, int64_t n, double* sigma, double* vega,
                          uint8_t* status);

/* Forward + backward on HOST arrays: additionally reads grad_sigma (host, n) and writes grad_P (host, n). */
int pivot_iv_forward_backward_host(pivot_iv_pipeline* p, const pivot_iv_inputs* in, const double* grad_sigma,
                                   double vega_floor, int mode, int64_t n, double* sigma, double* vega,
                                   uint8_t* status, double* grad_P);

/* Forward on HOST arrays without any allocation (for callers that cannot call cudaMalloc: code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it).  Same operation and same bits as pivot_iv_forward (Alg.1 l.1-3);
 * the device staging is a file-scope `static __device__` array of the library instead of a pipeline's cudaMalloc buffers:
 * PIVOT_STATIC_MAX_ROWS rows x (9 doubles + 1 byte) = 4,784,128 B, held by every GPU that loads the library until exit.
 *   in       host pointers, n doubles each (r = q = NULL: Black-76); pin them for copies that are asynchronous to the host
 *   n        0 <= n <= PIVOT_STATIC_MAX_ROWS, else PIVOT_ERR_STATIC_MAX (nothing is enqueued)
 *   sigma, vega [out, host, n doubles], status [out, host, n bytes]
 *   stream   the H2D copies, the kernel and the D2H copies are enqueued on it, on the current device; the call does NOT
 *            synchronise: the outputs are valid once the caller has synchronised the stream (or waited on an event)
 * Calls no cudaMalloc / cudaFree / allocating library routine; the first call on a device looks the array's address up
 * (cudaGetSymbolAddress) and opts the kernel in to its shared-memory size.  Every call shares the one array per GPU, which keeps
 * the previous call's contents: nothing in it has to start at zero (the call overwrites every byte it reads), but two calls
 * that overlap on the GPU -- different streams without a dependency, several host threads -- race on it; calls on one stream
 * are ordered.  Returns PIVOT_ERR_NULL / _BAD_N / _STATIC_MAX / _MIXED_RQ / _CUDA. */
#define PIVOT_STATIC_MAX_ROWS 65536
int pivot_iv_forward_host_static(const pivot_iv_inputs* in, int64_t n, double* sigma, double* vega, uint8_t* status,
                                 pivot_iv_stream stream);

/* ---- measurement helpers ---- */
/* Dependent-DFMA-chain microbenchmark on `stream`: every thread of a full-occupancy grid runs `iters` rounds of 8
 * independent fused multiply-adds.  Writes the number of fp64 FMA instructions (per thread, summed over threads)
 * to *fma_count_out (host); the caller times it with CUDA events to obtain the fp64-pipe peak.
 * `sink` is a device buffer of at least 8 bytes. */
int pivot_iv_probe_dfma(int64_t iters, double* sink, double* fma_count_out, pivot_iv_stream stream);

/* Test-only: evaluates ONE function of the device math library elementwise, out[i] = fn(a[i] [, b[i]]), so that its error
 * can be measured on the device against a multiprecision reference (tests/test_gpu_mathlib.py; DESIGN.md section 5 lists
 * the measured bounds).  a, b, out: device, n doubles; b is read only by the two-argument functions (erfcx pair: the pair
 * is erfcx(a), erfcx(b); div_fast: a / b; erfcx_dd: z1 = a, gap b; W: x = a, s = b).  fp32-grade functions take and return doubles (converted inside).
 * Returns PIVOT_ERR_BAD_ARG for an unknown fn, PIVOT_ERR_NULL / _BAD_N / _CUDA as usual. */
#define PIVOT_DBG_ERFCX_ONE 0      /* erfcx(a), a >= -0.0708, fp64 (degree-24 form) */
#define PIVOT_DBG_ERFCX_PAIR_1 1   /* first of erfcx_pair(a, b) */
#define PIVOT_DBG_ERFCX_PAIR_2 2   /* second of erfcx_pair(a, b) */
#define PIVOT_DBG_ERFCX_SEED 3     /* erfcx(a), fp32 seed grade */
#define PIVOT_DBG_EXP_FAST 4       /* exp(a), full range incl. the under / overflow branches */
#define PIVOT_DBG_EXP_SEED 5       /* exp(a), |a| < 700, MUFU.EX2 grade */
#define PIVOT_DBG_LOG_FAST 6       /* ln(a), a positive normal */
#define PIVOT_DBG_LOG_SEED 7       /* ln(a), a > 0 incl. subnormal, MUFU.LG2 grade */
#define PIVOT_DBG_LOG1P_FAST 8     /* ln(1 + a), a >= 0 */
#define PIVOT_DBG_RCP_NR1 9        /* 1/a, one Newton step */
#define PIVOT_DBG_RCP_NR2 10       /* 1/a, two Newton steps */
#define PIVOT_DBG_DIV_FAST 11      /* a / b */
#define PIVOT_DBG_SQRT_NR1 12      /* sqrt(a), one Newton step */
#define PIVOT_DBG_SQRT_NR2 13      /* sqrt(a), a positive normal */
#define PIVOT_DBG_RSQRT_NR2 14     /* 1/sqrt(a) as returned beside sqrt_nr2 */
#define PIVOT_DBG_NINV_TAIL_SEED 15 /* -Phi^-1(e^a), a <= ln 0.345, fp32 seed grade */
#define PIVOT_DBG_NINV_TAIL_FULL 16 /* ... refined by two Newton steps at fp64 */
#define PIVOT_DBG_EXPF_SEED 17     /* exp(a) in fp32 (MUFU.EX2), |a| <= 87 */
#define PIVOT_DBG_LOGF_SEED 18     /* ln(a) in fp32 (MUFU.LG2) */
#define PIVOT_DBG_ERFCX_DD_DIFF 19 /* erfcx(a) - erfcx(a + b), a >= -0.0708, b >= 0: divided-difference form, fp64 */
#define PIVOT_DBG_ERFCX_DD_SUM 20  /* erfcx(a) + erfcx(a + b), same evaluation */
#define PIVOT_DBG_ERFCX_DD_SEED_DIFF 21 /* ... fp32 seed grade */
#define PIVOT_DBG_ERFCX_DD_SEED_SUM 22
#define PIVOT_DBG_W_FULL 23        /* eval_W at x = a <= 0, s = b > 0: W = b/b' if the difference form was taken, else -Wbar */
#define PIVOT_DBG_W_SEED 24        /* ... at seed grade */
#define PIVOT_DBG_RCP_RAW 25       /* 1/a from MUFU.RCP64H alone (seed grade) */
#define PIVOT_DBG_RSQRT_C3 26     /* 1/sqrt(a), a positive normal: MUFU.RSQ64H + one third-order step */
#define PIVOT_DBG_COUNT 27
int pivot_iv_debug_math(int fn, const double* a, const double* b, int64_t n, double* out, pivot_iv_stream stream);

/* Number of kernels a call launches (for bench.py's `gpu_launches` bookkeeping): pivot_iv_launches_per_forward is the
 * count of an explicit organisation (and of PIVOT_FWD_AUTO below PIVOT_AUTO_MIN_ROWS); pivot_iv_forward_launches(n, kernel)
 * is the count of pivot_iv_forward_ex(..., kernel, ...) on n rows outside stream capture: 2 (probe + chosen kernel, one
 * graph launch) for PIVOT_FWD_AUTO at n >= PIVOT_AUTO_MIN_ROWS, else 1. */
int pivot_iv_launches_per_forward(void);
int pivot_iv_launches_per_backward(void);
int pivot_iv_forward_launches(int64_t n, int kernel);

/* The launch probe of PIVOT_FWD_AUTO on its own (diagnostic; tests): *rowwise = 1 if the rows follow each other closely enough
 * for the row-per-thread organisation, else 0 (n < 256: 0).
 *   in       as pivot_iv_forward (P is read)
 *   rowwise  [out, device, one int]
 * Returns PIVOT_ERR_NULL / _BAD_N / _MIXED_RQ / _CUDA. */
int pivot_iv_forward_probe(const pivot_iv_inputs* in, int64_t n, int* rowwise, pivot_iv_stream stream);

const char* pivot_iv_strerror(int code);
int pivot_iv_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PIVOT_IV_H_ */
