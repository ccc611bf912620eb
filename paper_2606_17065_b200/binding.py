"""ctypes binding of include/pivot_iv.h: argument marshalling only (same names as the C entry points)."""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Tuple

import torch  # loads libcudart first, so the library shares torch's CUDA runtime / primary context

HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(HERE, "libpivot_iv.so")

GATE_MASK = 0
GATE_ATTENUATE = 1
GATE_STRICT = 2
FWD_AUTO = 0
FWD_COMPACT = 1
FWD_ROWWISE = 2
FWD_FP64_ONLY = 4   # flag: OR into FWD_AUTO / FWD_COMPACT / FWD_ROWWISE
HOST_AUTO = 0       # Pipeline.set_host_access
HOST_STAGED = 1
HOST_DIRECT = 2     # Pipeline.last_host_path only

# every symbol include/pivot_iv.h declares
EXPORTS = (
    "pivot_iv_forward", "pivot_iv_forward_zones", "pivot_iv_backward", "pivot_iv_pipeline_create",
    "pivot_iv_pipeline_destroy", "pivot_iv_forward_host", "pivot_iv_forward_backward_host", "pivot_iv_probe_dfma",
    "pivot_iv_launches_per_forward", "pivot_iv_launches_per_backward", "pivot_iv_strerror", "pivot_iv_version",
    "pivot_iv_black_price", "pivot_iv_backward_inputs", "pivot_iv_loss_price", "pivot_iv_loss_roundtrip",
    "pivot_iv_forward_ex", "pivot_iv_pipeline_set_forward_kernel",
    "pivot_iv_forward_diag", "pivot_iv_debug_math", "pivot_iv_forward_launches", "pivot_iv_forward_probe",
    "pivot_iv_forward_host_static", "pivot_iv_pipeline_set_host_access", "pivot_iv_pipeline_last_host_path", "pivot_iv_status_histogram",
)


class PivotError(RuntimeError):
    pass


class _Inputs(C.Structure):
    _fields_ = [(name, C.c_void_p) for name in ("S_or_F", "K", "tau", "r", "q", "P", "flag")]


_lib = None


def library_path() -> str:
    return _SO


def load_library():
    """Loads libpivot_iv.so; raises (never falls back) if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_SO):
        raise PivotError(f"{_SO} is missing: build it with `python paper_2606_17065_b200/build.py` "
                         "(or __graft_entry__.build()); there is no CPU fallback")
    lib = C.CDLL(_SO)
    vp, i64, dbl, cint = C.c_void_p, C.c_int64, C.c_double, C.c_int
    lib.pivot_iv_forward.argtypes = [C.POINTER(_Inputs), i64, vp, vp, vp, vp]
    lib.pivot_iv_forward_ex.argtypes = [C.POINTER(_Inputs), i64, vp, vp, vp, cint, vp]
    lib.pivot_iv_forward_probe.argtypes = [C.POINTER(_Inputs), i64, vp, vp]
    lib.pivot_iv_forward_launches.argtypes = [i64, cint]
    lib.pivot_iv_pipeline_set_forward_kernel.argtypes = [vp, cint]
    lib.pivot_iv_pipeline_set_host_access.argtypes = [vp, cint]
    lib.pivot_iv_pipeline_last_host_path.argtypes = [vp]
    lib.pivot_iv_status_histogram.argtypes = [vp, i64, vp, vp]
    lib.pivot_iv_debug_math.argtypes = [cint, vp, vp, i64, vp, vp]
    lib.pivot_iv_forward_diag.argtypes = [C.POINTER(_Inputs), i64, vp, vp, vp, vp, vp, vp, cint, vp]
    lib.pivot_iv_forward_zones.argtypes = [C.POINTER(_Inputs), i64, vp, vp, vp, vp, vp]
    lib.pivot_iv_backward.argtypes = [vp, vp, vp, dbl, cint, i64, vp, vp]
    lib.pivot_iv_pipeline_create.argtypes = [C.POINTER(vp), cint, i64, cint]
    lib.pivot_iv_pipeline_destroy.argtypes = [vp]
    lib.pivot_iv_forward_host.argtypes = [vp, C.POINTER(_Inputs), i64, vp, vp, vp]
    lib.pivot_iv_forward_host_static.argtypes = [C.POINTER(_Inputs), i64, vp, vp, vp, vp]
    lib.pivot_iv_forward_backward_host.argtypes = [vp, C.POINTER(_Inputs), vp, dbl, cint, i64, vp, vp, vp, vp]
    lib.pivot_iv_probe_dfma.argtypes = [i64, vp, C.POINTER(dbl), vp]
    lib.pivot_iv_black_price.argtypes = [C.POINTER(_Inputs), vp, i64, vp, vp, vp]
    lib.pivot_iv_backward_inputs.argtypes = [C.POINTER(_Inputs), vp, vp, vp, vp, dbl, cint, i64, vp, vp, vp, vp, vp, vp, vp]
    lib.pivot_iv_strerror.argtypes = [cint]
    lib.pivot_iv_strerror.restype = C.c_char_p
    lib.pivot_iv_loss_price.argtypes = [C.POINTER(_Inputs), vp, i64, vp, vp, dbl, vp]
    lib.pivot_iv_loss_roundtrip.argtypes = [C.POINTER(_Inputs), vp, vp, dbl, cint, i64, vp, vp, dbl, vp]
    for name in EXPORTS:
        if name != "pivot_iv_strerror":
            getattr(lib, name).restype = cint
    _lib = lib
    return lib


def pivot_iv_strerror(code: int) -> str:
    return load_library().pivot_iv_strerror(int(code)).decode()


def pivot_iv_version() -> int:
    return int(load_library().pivot_iv_version())


def _check(code: int):
    if code != 0:
        raise PivotError(f"pivot_iv error {code}: {pivot_iv_strerror(code)}")


def _dev(t: Optional[torch.Tensor], name: str, dtype=torch.float64) -> Optional[int]:
    if t is None:
        return None
    if not (t.is_cuda and t.dtype == dtype and t.is_contiguous() and t.dim() == 1):
        raise PivotError(f"{name}: expected a contiguous 1-D CUDA tensor of {dtype}")
    return t.data_ptr()


def _same_len(n: int, **tensors):
    """Every tensor given must hold exactly n elements (None is skipped)."""
    for nm, t in tensors.items():
        if t is not None and t.numel() != n:
            raise PivotError(f"{nm}: length {t.numel()} != {n}")


def _same_device(ref: torch.Tensor, **tensors):
    for nm, t in tensors.items():
        if t is not None and t.device != ref.device:
            raise PivotError(f"{nm}: on {t.device}, expected {ref.device}")


def _stream_ptr(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


class _NoGuard:
    def __enter__(self):
        return None

    def __exit__(self, *a):
        return False


_NOGUARD = _NoGuard()


def _guard(device):
    """Device guard around a launch; skipped (it costs several microseconds per call) when `device` is already current."""
    idx = device.index
    if idx is None or idx == torch.cuda.current_device():
        return _NOGUARD
    return torch.cuda.device(device)


def _require_cuda():
    if not torch.cuda.is_available():
        raise PivotError("no CUDA device: the PIVOT path runs only on the GPU (no CPU fallback)")


_F64, _U8 = torch.float64, torch.uint8


def _ptr(t, name, n, dev, dtype=_F64):
    """data_ptr() of a contiguous 1-D CUDA tensor of `dtype` with n elements on `dev` (one pass: this sits on the per-call path)."""
    if not isinstance(t, torch.Tensor):
        raise PivotError(f"{name}: expected a contiguous 1-D CUDA tensor of {dtype}")
    if t.dtype is not dtype or t.device != dev or t.dim() != 1 or t.shape[0] != n or not t.is_contiguous():
        if not (t.is_cuda and t.dtype == dtype and t.is_contiguous() and t.dim() == 1):
            raise PivotError(f"{name}: expected a contiguous 1-D CUDA tensor of {dtype}")
        if t.numel() != n:
            raise PivotError(f"{name}: length {t.numel()} != {n}")
        raise PivotError(f"{name}: on {t.device}, expected {dev}")
    return t.data_ptr()


def _forward(SorF, K, tau, P, flag, r, q, out, stream, zones, kernel=None):
    _require_cuda()
    lib = load_library()
    if not (isinstance(SorF, torch.Tensor) and SorF.is_cuda and SorF.dim() == 1):
        raise PivotError("S_or_F: expected a contiguous 1-D CUDA tensor of torch.float64")
    n = SorF.shape[0]
    dev = SorF.device
    inp = _Inputs(_ptr(SorF, "S_or_F", n, dev), _ptr(K, "K", n, dev), _ptr(tau, "tau", n, dev),
                  None if r is None else _ptr(r, "r", n, dev), None if q is None else _ptr(q, "q", n, dev),
                  _ptr(P, "P", n, dev), _ptr(flag, "flag", n, dev))
    if out is None:
        sigma = torch.empty(n, dtype=_F64, device=dev)
        vega = torch.empty(n, dtype=_F64, device=dev)
        status = torch.empty(n, dtype=_U8, device=dev)
    else:
        sigma, vega, status = out[:3]
    ps, pv_, pst = _ptr(sigma, "out[0]", n, dev), _ptr(vega, "out[1]", n, dev), _ptr(status, "out[2]", n, dev, _U8)
    sp = _stream_ptr(stream)
    with _guard(dev):
        if zones:
            zone = torch.empty(n, dtype=torch.int8, device=dev) if out is None or len(out) < 4 else out[3]
            _check(lib.pivot_iv_forward_zones(C.byref(inp), n, ps, pv_, pst, _ptr(zone, "out[3]", n, dev, torch.int8), sp))
            return sigma, vega, status, zone
        if kernel is not None:
            _check(lib.pivot_iv_forward_ex(C.byref(inp), n, ps, pv_, pst, int(kernel), sp))
        else:
            _check(lib.pivot_iv_forward(C.byref(inp), n, ps, pv_, pst, sp))
    return sigma, vega, status


def pivot_iv_forward(S_or_F, K, tau, P, flag, r=None, q=None, out=None, stream=None
                     ) -> Tuple[torch.Tensor, torch.Tensor, torch.Tensor]:
    """(sigma, vega, status) = pivot_iv_forward(...) on CUDA fp64 tensors; r = q = None selects Black-76 with D = 1.
    `out` = (sigma, vega, status) preallocated tensors; `stream` = torch.cuda.Stream (default: current)."""
    return _forward(S_or_F, K, tau, P, flag, r, q, out, stream, False)


def pivot_iv_forward_ex(S_or_F, K, tau, P, flag, kernel: int, r=None, q=None, out=None, stream=None):
    """pivot_iv_forward with an explicit kernel organisation: FWD_AUTO, FWD_COMPACT or FWD_ROWWISE (same results)."""
    return _forward(S_or_F, K, tau, P, flag, r, q, out, stream, False, kernel=kernel)


AUTO_MIN_ROWS = 3 << 23   # PIVOT_AUTO_MIN_ROWS: from here on FWD_AUTO chooses on the device (probe kernel + IF / ELSE graph node)


def pivot_iv_forward_probe(S_or_F, K, tau, P, flag, r=None, q=None, stream=None) -> torch.Tensor:
    """The launch probe of FWD_AUTO on its own: a one-element int32 CUDA tensor, 1 if the rows follow each other closely
    enough for the row-per-thread organisation (option chains in strike order), else 0."""
    _require_cuda()
    lib = load_library()
    n = S_or_F.shape[0]
    dev = S_or_F.device
    inp = _Inputs(_ptr(S_or_F, "S_or_F", n, dev), _ptr(K, "K", n, dev), _ptr(tau, "tau", n, dev),
                  None if r is None else _ptr(r, "r", n, dev), None if q is None else _ptr(q, "q", n, dev),
                  _ptr(P, "P", n, dev), _ptr(flag, "flag", n, dev))
    verdict = torch.zeros(1, dtype=torch.int32, device=dev)
    with _guard(dev):
        _check(lib.pivot_iv_forward_probe(C.byref(inp), n, verdict.data_ptr(), _stream_ptr(stream)))
    return verdict


def pivot_iv_forward_launches(n: int, kernel: int = FWD_AUTO) -> int:
    """Kernels launched by one forward call on n rows with this organisation (2 = probe + chosen kernel, one graph launch)."""
    return int(load_library().pivot_iv_forward_launches(int(n), int(kernel)))


def pivot_iv_forward_diag(S_or_F, K, tau, P, flag, r=None, q=None, kernel: int = FWD_AUTO, stream=None):
    """(sigma, vega, status, zone, s_seed, s_step1): pivot_iv_forward plus the per-row diagnostics of the solve (LBR
    zone, rational seed, iterate after the first Householder step; total volatilities)."""
    _require_cuda()
    lib = load_library()
    n = S_or_F.numel()
    _same_len(n, K=K, tau=tau, P=P, flag=flag, r=r, q=q)
    inp = _Inputs(_dev(S_or_F, "S_or_F"), _dev(K, "K"), _dev(tau, "tau"), _dev(r, "r"), _dev(q, "q"), _dev(P, "P"),
                  _dev(flag, "flag"))
    dev = S_or_F.device
    sigma, vega, s0, s1 = (torch.empty(n, dtype=torch.float64, device=dev) for _ in range(4))
    status = torch.empty(n, dtype=torch.uint8, device=dev)
    zone = torch.empty(n, dtype=torch.int8, device=dev)
    with torch.cuda.device(dev):
        _check(lib.pivot_iv_forward_diag(C.byref(inp), n, sigma.data_ptr(), vega.data_ptr(), status.data_ptr(),
                                         zone.data_ptr(), s0.data_ptr(), s1.data_ptr(), int(kernel), _stream_ptr(stream)))
    return sigma, vega, status, zone, s0, s1


DBG = {name: i for i, name in enumerate((
    "erfcx_one", "erfcx_pair_1", "erfcx_pair_2", "erfcx_seed", "exp_fast", "exp_seed", "log_fast", "log_seed", "log1p_fast",
    "rcp_nr1", "rcp_nr2", "div_fast", "sqrt_nr1", "sqrt_nr2", "rsqrt_nr2", "ninv_tail_seed", "ninv_tail_full", "expf_seed",
    "logf_seed", "erfcx_dd_diff", "erfcx_dd_sum", "erfcx_dd_seed_diff", "erfcx_dd_seed_sum", "w_full", "w_seed", "rcp_raw", "rsqrt_c3"))}


def pivot_iv_debug_math(fn: str, a: torch.Tensor, b: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    """Test-only: out = fn(a [, b]) evaluated by the device math library (see PIVOT_DBG_* in include/pivot_iv.h)."""
    _require_cuda()
    n = a.numel()
    _same_len(n, b=b)
    out = torch.empty_like(a)
    with _guard(a.device):
        _check(load_library().pivot_iv_debug_math(DBG[fn], _dev(a, "a"), _dev(b, "b"), n, _dev(out, "out"),
                                                  _stream_ptr(stream)))
    return out


def pivot_iv_forward_zones(S_or_F, K, tau, P, flag, r=None, q=None, out=None, stream=None):
    """As pivot_iv_forward, also returning the LBR zone per row (diagnostics)."""
    return _forward(S_or_F, K, tau, P, flag, r, q, out, stream, True)


def pivot_iv_backward(grad_sigma, vega, status, vega_floor: float, mode: int, out=None, stream=None) -> torch.Tensor:
    """grad_P = gate * grad_sigma / vega (mode GATE_MASK or GATE_ATTENUATE); `out` may alias grad_sigma."""
    _require_cuda()
    lib = load_library()
    n = grad_sigma.numel()
    _same_len(n, vega=vega, status=status, out=out)
    _same_device(grad_sigma, vega=vega, status=status, out=out)
    gP = torch.empty_like(grad_sigma) if out is None else out
    with _guard(grad_sigma.device):
        _check(lib.pivot_iv_backward(_dev(grad_sigma, "grad_sigma"), _dev(vega, "vega"),
                                     _dev(status, "status", torch.uint8), float(vega_floor), int(mode), n,
                                     _dev(gP, "grad_P"), _stream_ptr(stream)))
    return gP


def pivot_iv_status_histogram(status, out=None, stream=None) -> torch.Tensor:
    """Rows per status code: an int64 CUDA tensor of 6 counts (status 0..4, anything else); `out` is accumulated into."""
    _require_cuda()
    n = status.numel()
    counts = torch.zeros(6, dtype=torch.int64, device=status.device) if out is None else out
    if not (counts.is_cuda and counts.dtype == torch.int64 and counts.numel() == 6 and counts.is_contiguous()):
        raise PivotError("out: expected a contiguous CUDA int64 tensor of 6 elements")
    _same_device(status, out=counts)
    with _guard(status.device):
        _check(load_library().pivot_iv_status_histogram(_dev(status, "status", torch.uint8), n, counts.data_ptr(),
                                                        _stream_ptr(stream)))
    return counts


def pivot_iv_black_price(S_or_F, K, tau, sigma, flag, r=None, q=None, with_vega=True, stream=None):
    """(price, vega) of the Black-76 / BSM price eq.(2)/(3) at `sigma` (CUDA fp64 tensors); vega is None if not asked."""
    _require_cuda()
    lib = load_library()
    n = S_or_F.numel()
    _same_len(n, K=K, tau=tau, sigma=sigma, flag=flag, r=r, q=q)
    _same_device(S_or_F, K=K, tau=tau, sigma=sigma, flag=flag, r=r, q=q)
    inp = _Inputs(_dev(S_or_F, "S_or_F"), _dev(K, "K"), _dev(tau, "tau"), _dev(r, "r"), _dev(q, "q"), None,
                  _dev(flag, "flag"))
    price = torch.empty(n, dtype=torch.float64, device=S_or_F.device)
    vega = torch.empty(n, dtype=torch.float64, device=S_or_F.device) if with_vega else None
    with _guard(S_or_F.device):
        _check(lib.pivot_iv_black_price(C.byref(inp), _dev(sigma, "sigma"), n, _dev(price, "price"), _dev(vega, "vega"),
                                     _stream_ptr(stream)))
    return price, vega


def pivot_iv_backward_inputs(S_or_F, K, tau, flag, sigma, vega, status, grad_sigma, vega_floor: float, mode: int,
                             r=None, q=None, stream=None):
    """Full VJP of eq.(8): returns (grad_P, grad_S_or_F, grad_K, grad_tau, grad_r, grad_q); the last two are None in
    Black-76 mode (r = q = None)."""
    _require_cuda()
    lib = load_library()
    n = S_or_F.numel()
    _same_len(n, K=K, tau=tau, flag=flag, sigma=sigma, vega=vega, status=status, grad_sigma=grad_sigma, r=r, q=q)
    _same_device(S_or_F, K=K, tau=tau, flag=flag, sigma=sigma, vega=vega, status=status, grad_sigma=grad_sigma, r=r, q=q)
    inp = _Inputs(_dev(S_or_F, "S_or_F"), _dev(K, "K"), _dev(tau, "tau"), _dev(r, "r"), _dev(q, "q"), None,
                  _dev(flag, "flag"))
    outs = [torch.empty(n, dtype=torch.float64, device=S_or_F.device) for _ in range(4)]
    outs += [torch.empty(n, dtype=torch.float64, device=S_or_F.device) if r is not None else None for _ in range(2)]
    with _guard(S_or_F.device):
        _check(lib.pivot_iv_backward_inputs(C.byref(inp), _dev(sigma, "sigma"), _dev(vega, "vega"),
                                            _dev(status, "status", torch.uint8), _dev(grad_sigma, "grad_sigma"),
                                            float(vega_floor), int(mode), n, *[_dev(o, "grad") for o in outs],
                                            _stream_ptr(stream)))
    return tuple(outs)


RT_GATED = 0
RT_NAIVE = 1


def pivot_iv_loss_price(S_or_F, K, tau, P_star, flag, sigma_hat, r=None, q=None, grad_scale: Optional[float] = None,
                        stream=None):
    """eq.(11) as sums: returns a CUDA tensor [sum (P_model - P*)^2, sum |P*|, rows used]; with grad_scale also the
    gradient grad_scale * 2 (P_model - P*) V_hat with respect to sigma_hat: (sums, grad)."""
    _require_cuda()
    lib = load_library()
    n = S_or_F.numel()
    _same_len(n, K=K, tau=tau, P_star=P_star, flag=flag, sigma_hat=sigma_hat, r=r, q=q)
    _same_device(S_or_F, K=K, tau=tau, P_star=P_star, flag=flag, sigma_hat=sigma_hat, r=r, q=q)
    inp = _Inputs(_dev(S_or_F, "S_or_F"), _dev(K, "K"), _dev(tau, "tau"), _dev(r, "r"), _dev(q, "q"), _dev(P_star, "P"),
                  _dev(flag, "flag"))
    out = torch.zeros(3, dtype=torch.float64, device=S_or_F.device)
    grad = torch.empty(n, dtype=torch.float64, device=S_or_F.device) if grad_scale is not None else None
    with _guard(S_or_F.device):
        _check(lib.pivot_iv_loss_price(C.byref(inp), _dev(sigma_hat, "sigma_hat"), n, _dev(out, "out"), _dev(grad, "grad"),
                                       float(grad_scale or 0.0), _stream_ptr(stream)))
    return out if grad is None else (out, grad)


def pivot_iv_loss_roundtrip(S_or_F, K, tau, P_star, flag, sigma_hat, sigma_star, vega_floor: float, r=None, q=None,
                            mode: int = RT_GATED, grad_scale: Optional[float] = None, stream=None):
    """eq.(12) as sums (mode RT_GATED) or the naive ungated composition (RT_NAIVE): returns a CUDA tensor
    [sum w (IV(P~) - sigma*)^2, sum w, rows used]; with grad_scale also the gradient w.r.t. sigma_hat: (sums, grad)."""
    _require_cuda()
    lib = load_library()
    n = S_or_F.numel()
    _same_len(n, K=K, tau=tau, P_star=P_star, flag=flag, sigma_hat=sigma_hat, sigma_star=sigma_star, r=r, q=q)
    _same_device(S_or_F, K=K, tau=tau, P_star=P_star, flag=flag, sigma_hat=sigma_hat, sigma_star=sigma_star, r=r, q=q)
    inp = _Inputs(_dev(S_or_F, "S_or_F"), _dev(K, "K"), _dev(tau, "tau"), _dev(r, "r"), _dev(q, "q"), _dev(P_star, "P"),
                  _dev(flag, "flag"))
    out = torch.zeros(3, dtype=torch.float64, device=S_or_F.device)
    grad = torch.empty(n, dtype=torch.float64, device=S_or_F.device) if grad_scale is not None else None
    with _guard(S_or_F.device):
        _check(lib.pivot_iv_loss_roundtrip(C.byref(inp), _dev(sigma_hat, "sigma_hat"), _dev(sigma_star, "sigma_star"),
                                           float(vega_floor), int(mode), n, _dev(out, "out"), _dev(grad, "grad"),
                                           float(grad_scale or 0.0), _stream_ptr(stream)))
    return out if grad is None else (out, grad)


def pivot_iv_probe_dfma(iters: int, stream=None) -> float:
    """Enqueues the DFMA-chain probe; returns the number of fp64 FMAs it executes (time it with CUDA events)."""
    _require_cuda()
    sink = torch.zeros(8, dtype=torch.float64, device="cuda")
    cnt = C.c_double(0.0)
    _check(load_library().pivot_iv_probe_dfma(int(iters), sink.data_ptr(), C.byref(cnt), _stream_ptr(stream)))
    return float(cnt.value)


def _host(t: Optional[torch.Tensor], name: str, dtype=torch.float64) -> Optional[int]:
    if t is None:
        return None
    if t.is_cuda or t.dtype != dtype or not t.is_contiguous() or t.dim() != 1:
        raise PivotError(f"{name}: expected a contiguous 1-D CPU tensor of {dtype}")
    return t.data_ptr()


class Pipeline:
    """Host-buffer pipeline (pivot_iv_pipeline_*): chunked H2D -> kernels -> D2H over `n_slots` streams.
    Pass pinned CPU tensors for full PCIe bandwidth."""

    def __init__(self, chunk_rows: int = 1 << 20, n_slots: int = 3, device: int = -1):
        _require_cuda()
        self._lib = load_library()
        self._h = C.c_void_p()
        _check(self._lib.pivot_iv_pipeline_create(C.byref(self._h), int(device), int(chunk_rows), int(n_slots)))

    def set_forward_kernel(self, kernel: int):
        _check(self._lib.pivot_iv_pipeline_set_forward_kernel(self._h, int(kernel)))

    def set_host_access(self, mode: int):
        """HOST_AUTO (default): forward_host on pinned tensors runs ONE launch straight on the host arrays (no staging);
        HOST_STAGED: always the chunked copy path."""
        _check(self._lib.pivot_iv_pipeline_set_host_access(self._h, int(mode)))

    def last_host_path(self) -> int:
        """HOST_STAGED or HOST_DIRECT: how the last forward_host / forward_backward_host call reached the host arrays."""
        return int(self._lib.pivot_iv_pipeline_last_host_path(self._h))

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.pivot_iv_pipeline_destroy(self._h)
            self._h = C.c_void_p()

    __del__ = close

    def forward_host(self, S_or_F, K, tau, P, flag, r=None, q=None, out=None):
        n = S_or_F.numel()
        _same_len(n, K=K, tau=tau, P=P, flag=flag, r=r, q=q)
        if out is not None:
            _same_len(n, **{f"out[{i}]": t for i, t in enumerate(out)})
        if out is None:
            out = (torch.empty(n, dtype=torch.float64), torch.empty(n, dtype=torch.float64),
                   torch.empty(n, dtype=torch.uint8))
        sigma, vega, status = out
        inp = _Inputs(_host(S_or_F, "S_or_F"), _host(K, "K"), _host(tau, "tau"), _host(r, "r"), _host(q, "q"),
                      _host(P, "P"), _host(flag, "flag"))
        _check(self._lib.pivot_iv_forward_host(self._h, C.byref(inp), n, _host(sigma, "sigma"), _host(vega, "vega"),
                                               _host(status, "status", torch.uint8)))
        return sigma, vega, status

    def forward_backward_host(self, S_or_F, K, tau, P, flag, grad_sigma, vega_floor, mode, r=None, q=None, out=None):
        n = S_or_F.numel()
        _same_len(n, K=K, tau=tau, P=P, flag=flag, grad_sigma=grad_sigma, r=r, q=q)
        if out is not None:
            _same_len(n, **{f"out[{i}]": t for i, t in enumerate(out)})
        if out is None:
            out = (torch.empty(n, dtype=torch.float64), torch.empty(n, dtype=torch.float64),
                   torch.empty(n, dtype=torch.uint8), torch.empty(n, dtype=torch.float64))
        sigma, vega, status, gP = out
        inp = _Inputs(_host(S_or_F, "S_or_F"), _host(K, "K"), _host(tau, "tau"), _host(r, "r"), _host(q, "q"),
                      _host(P, "P"), _host(flag, "flag"))
        _check(self._lib.pivot_iv_forward_backward_host(self._h, C.byref(inp), _host(grad_sigma, "grad_sigma"),
                                                        float(vega_floor), int(mode), n, _host(sigma, "sigma"),
                                                        _host(vega, "vega"), _host(status, "status", torch.uint8),
                                                        _host(gP, "grad_P")))
        return sigma, vega, status, gP


STATIC_MAX_ROWS = 65536   # PIVOT_STATIC_MAX_ROWS


def pivot_iv_forward_host_static(S_or_F, K, tau, P, flag, r=None, q=None, out=None, stream=None, sync=True):
    """Forward on HOST tensors with no device allocation (pivot_iv_forward_host_static): the device staging is a static array
    of the library (at most STATIC_MAX_ROWS rows per call).  `out` = (sigma, vega, status) host tensors, allocated here (on the
    host) if not given -- pass them, pinned, from a loop that must not allocate at all.  The C call only enqueues on `stream`;
    with sync=True (default) this wrapper waits for the stream before it returns.  Calls that overlap on the GPU race on the
    shared staging array."""
    _require_cuda()
    lib = load_library()
    n = S_or_F.numel()
    _same_len(n, K=K, tau=tau, P=P, flag=flag, r=r, q=q)
    if out is None:
        out = (torch.empty(n, dtype=torch.float64), torch.empty(n, dtype=torch.float64), torch.empty(n, dtype=torch.uint8))
    _same_len(n, **{f"out[{i}]": t for i, t in enumerate(out)})
    sigma, vega, status = out
    inp = _Inputs(_host(S_or_F, "S_or_F"), _host(K, "K"), _host(tau, "tau"), _host(r, "r"), _host(q, "q"),
                  _host(P, "P"), _host(flag, "flag"))
    if stream is None:
        stream = torch.cuda.current_stream()
    _check(lib.pivot_iv_forward_host_static(C.byref(inp), n, _host(sigma, "sigma"), _host(vega, "vega"),
                                            _host(status, "status", torch.uint8), int(stream.cuda_stream)))
    if sync:
        stream.synchronize()
    return sigma, vega, status


class ShardedPipeline:
    """Row-sharded label generation over several GPUs from ONE process: one
    pivot_iv_pipeline per device, each fed a contiguous shard (sharding.shard_rows) of the same host arrays by its own
    host thread (the C call releases the GIL).  Rows are independent: no collective, results land in the caller's arrays.
    With one process per GPU (torchrun) each rank simply runs a Pipeline on shard_rows(n, rank, world) instead."""

    def __init__(self, devices, chunk_rows: int = 1 << 19, n_slots: int = 4):
        from .sharding import shard_rows
        self._shard_rows = shard_rows
        self.devices = list(devices)
        if not self.devices:
            raise PivotError("ShardedPipeline needs at least one device")
        self.pipes = [Pipeline(chunk_rows=chunk_rows, n_slots=n_slots, device=int(d)) for d in self.devices]

    def close(self):
        for p in self.pipes:
            p.close()

    def shards(self, n: int):
        return [self._shard_rows(n, k, len(self.pipes)) for k in range(len(self.pipes))]

    def forward_host(self, S_or_F, K, tau, P, flag, r=None, q=None, out=None):
        import threading
        n = S_or_F.numel()
        _same_len(n, K=K, tau=tau, P=P, flag=flag, r=r, q=q)
        if out is None:
            out = (torch.empty(n, dtype=torch.float64), torch.empty(n, dtype=torch.float64),
                   torch.empty(n, dtype=torch.uint8))
        _same_len(n, **{f"out[{i}]": t for i, t in enumerate(out)})
        errs = []

        def work(k, b, e):
            try:
                sl = lambda t: None if t is None else t[b:e]
                self.pipes[k].forward_host(sl(S_or_F), sl(K), sl(tau), sl(P), sl(flag), r=sl(r), q=sl(q),
                                           out=tuple(t[b:e] for t in out))
            except Exception as ex:   # surfaced to the caller below
                errs.append(ex)
        threads = [threading.Thread(target=work, args=(k, b, e)) for k, (b, e) in enumerate(self.shards(n)) if e > b]
        for t in threads:
            t.start()
        for t in threads:
            t.join()
        if errs:
            raise errs[0]
        return out
