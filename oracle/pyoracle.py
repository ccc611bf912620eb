"""oracle/pyoracle.py -- TEST INFRASTRUCTURE.  ctypes front end of oracle/liblbr_oracle.so (numpy in, numpy out).

Nothing here is on the product path; paper_2606_17065_b200 never imports it.
"""
import ctypes as C

import numpy as np

from . import build as _build

_lib = None

_D = C.POINTER(C.c_double)
_U8 = C.POINTER(C.c_uint8)
_I8 = C.POINTER(C.c_int8)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.oracle_max_threads.restype = C.c_int
        _lib.oracle_control_fit.restype = C.c_double
        _lib.oracle_control_fit.argtypes = [C.c_int] + [C.c_double] * 6 + [C.c_int]
    return _lib


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a, t=_D):
    return None if a is None else a.ctypes.data_as(t)


def max_threads():
    return int(lib().oracle_max_threads())


def forward(SorF, K, tau, P, flag, r=None, q=None, prec=0, fixed_iters=0, nthreads=0, debug=False):
    """LBR forward. Returns (sigma, vega, status[, zone, iters, s0])."""
    SorF, K, tau, P, flag = map(_d, (SorF, K, tau, P, flag))
    r = None if r is None else _d(r)
    q = None if q is None else _d(q)
    n = SorF.size
    sigma = np.empty(n); vega = np.empty(n); status = np.empty(n, dtype=np.uint8)
    zone = np.empty(n, dtype=np.int8) if debug else None
    iters = np.empty(n, dtype=np.int8) if debug else None
    s0 = np.empty(n) if debug else None
    lib().oracle_forward(C.c_int(prec), C.c_int64(n), _p(SorF), _p(K), _p(tau), _p(r), _p(q), _p(P), _p(flag),
                         _p(sigma), _p(vega), _p(status, _U8), _p(zone, _I8), _p(iters, _I8), _p(s0),
                         C.c_int(fixed_iters), C.c_int(nthreads))
    if debug:
        return sigma, vega, status, zone, iters, s0
    return sigma, vega, status


def backward(gsigma, vega, status, vega_floor, mode):
    gsigma, vega = _d(gsigma), _d(vega)
    status = np.ascontiguousarray(status, dtype=np.uint8)
    out = np.empty(gsigma.size)
    lib().oracle_backward(C.c_int64(gsigma.size), _p(gsigma), _p(vega), _p(status, _U8), C.c_double(vega_floor),
                          C.c_int(mode), _p(out))
    return out


def black_price(SorF, K, tau, sigma, flag, r=None, q=None, prec=1):
    SorF, K, tau, sigma, flag = map(_d, (SorF, K, tau, sigma, flag))
    r = None if r is None else _d(r)
    q = None if q is None else _d(q)
    out = np.empty(SorF.size)
    lib().oracle_black_price(C.c_int(prec), C.c_int64(SorF.size), _p(SorF), _p(K), _p(tau), _p(r), _p(q), _p(sigma),
                             _p(flag), _p(out))
    return out


def vega_eq14(SorF, K, tau, sigma, r=None, q=None):
    SorF, K, tau, sigma = map(_d, (SorF, K, tau, sigma))
    r = None if r is None else _d(r)
    q = None if q is None else _d(q)
    out = np.empty(SorF.size)
    lib().oracle_vega_eq14(C.c_int64(SorF.size), _p(SorF), _p(K), _p(tau), _p(r), _p(q), _p(sigma), _p(out))
    return out


def truth_iv(SorF, K, tau, P, flag, r=None, q=None):
    """__float128 bisection on the literal eq.(3)/(6) definition."""
    SorF, K, tau, P, flag = map(_d, (SorF, K, tau, P, flag))
    r = None if r is None else _d(r)
    q = None if q is None else _d(q)
    out = np.empty(SorF.size)
    lib().oracle_truth_iv(C.c_int64(SorF.size), _p(SorF), _p(K), _p(tau), _p(r), _p(q), _p(P), _p(flag), _p(out))
    return out


def black_literal_q(F, K, D, tau, sigma, flag):
    F, K, D, tau, sigma, flag = map(_d, (F, K, D, tau, sigma, flag))
    out = np.empty(F.size)
    lib().oracle_black_literal_q(C.c_int64(F.size), _p(F), _p(K), _p(D), _p(tau), _p(sigma), _p(flag), _p(out))
    return out


def erfcx(z):
    z = _d(z); out = np.empty(z.size)
    lib().oracle_erfcx(C.c_int64(z.size), _p(z), _p(out))
    return out


def ninv(p):
    p = _d(p); out = np.empty(p.size)
    lib().oracle_ninv(C.c_int64(p.size), _p(p), _p(out))
    return out


def norm_black(x, s, prec=0):
    x, s = _d(x), _d(s)
    b = np.empty(x.size); v = np.empty(x.size)
    lib().oracle_norm_black(C.c_int(prec), C.c_int64(x.size), _p(x), _p(s), _p(b), _p(v))
    return b, v


def W(h, t, prec=0):
    h, t = _d(h), _d(t)
    w = np.empty(h.size); wb = np.empty(h.size)
    lib().oracle_W(C.c_int(prec), C.c_int64(h.size), _p(h), _p(t), _p(w), _p(wb))
    return w, wb


def W_series(h, t, nterms=8):
    h, t = _d(h), _d(t)
    w = np.empty(h.size)
    lib().oracle_W_series(C.c_int64(h.size), _p(h), _p(t), C.c_int(nterms), _p(w))
    return w


def rational_cubic(u, H, yl, yr, dl, dr, r):
    u = _d(u); out = np.empty(u.size)
    lib().oracle_rational_cubic(C.c_int64(u.size), _p(u), *(C.c_double(v) for v in (H, yl, yr, dl, dr, r)), _p(out))
    return out


def control_fit(side, H, yl, yr, dl, dr, dd, floor_it=True):
    return float(lib().oracle_control_fit(int(side), H, yl, yr, dl, dr, dd, int(floor_it)))


def solve_normalised(x, beta, bmax=None, bbar=None, prec=0, fixed_iters=0, nodes=False):
    x, beta = _d(x), _d(beta)
    bmax = np.exp(0.5 * x) if bmax is None else _d(bmax)
    bbar = (bmax - beta) if bbar is None else _d(bbar)
    n = x.size
    s = np.empty(n); zone = np.empty(n, dtype=np.int8); s0 = np.empty(n)
    nd = np.empty((n, 6)) if nodes else None
    lib().oracle_solve_normalised(C.c_int(prec), C.c_int64(n), _p(x), _p(beta), _p(bmax), _p(bbar),
                                  C.c_int(fixed_iters), _p(s), _p(zone, _I8), _p(s0), _p(nd))
    return (s, zone, s0, nd) if nodes else (s, zone, s0)


def householder_terms(kind, x, s, beta, bbar):
    kind = np.ascontiguousarray(kind, dtype=np.int32)
    x, s, beta, bbar = map(_d, (x, s, beta, bbar))
    n = x.size
    g = np.empty(n); nu = np.empty(n); h2 = np.empty(n); h3 = np.empty(n)
    lib().oracle_householder_terms(C.c_int64(n), kind.ctypes.data_as(C.POINTER(C.c_int)), _p(x), _p(s), _p(beta),
                                   _p(bbar), _p(g), _p(nu), _p(h2), _p(h3))
    return g, nu, h2, h3


def f_low_end(a, s):
    out = (C.c_double * 3)()
    lib().oracle_f_low_end(C.c_double(a), C.c_double(s), out)
    return tuple(out)


def f_up_end(x, s):
    out = (C.c_double * 3)()
    lib().oracle_f_up_end(C.c_double(x), C.c_double(s), out)
    return tuple(out)


OP_NAMES = ("add", "mul", "div", "sqrt", "exp", "log", "log1p", "erfc", "erfcx", "ninv", "cbrt")


def count_ops(SorF, K, tau, P, flag, r=None, q=None, fixed_iters=2):
    """Algorithmic fp64 operation counts of the oracle (op-counting scalar type), per LBR zone.
    Returns (counts[5, 11] uint64, rows[5]): classes 0..3 = zone of OK rows, 4 = non-OK rows; columns OP_NAMES."""
    SorF, K, tau, P, flag = map(_d, (SorF, K, tau, P, flag))
    r = None if r is None else _d(r)
    q = None if q is None else _d(q)
    nc = int(lib().oracle_count_ops_ncounters())
    counts = np.zeros((5, nc), dtype=np.uint64); rows = np.zeros(5, dtype=np.uint64)
    lib().oracle_count_ops(C.c_int64(SorF.size), _p(SorF), _p(K), _p(tau), _p(r), _p(q), _p(P), _p(flag),
                           C.c_int(fixed_iters), counts.ctypes.data_as(C.c_void_p), rows.ctypes.data_as(C.c_void_p))
    return counts, rows


def black_greeks(SorF, K, tau, sigma, flag, r=None, q=None, prec=1):
    """dP/dS (or dF), dP/dK, dP/dtau, dP/dr, dP/dq of the discounted Black price."""
    SorF, K, tau, sigma, flag = map(_d, (SorF, K, tau, sigma, flag))
    r = None if r is None else _d(r)
    q = None if q is None else _d(q)
    outs = [np.empty(SorF.size) for _ in range(5)]
    lib().oracle_black_greeks(C.c_int(prec), C.c_int64(SorF.size), _p(SorF), _p(K), _p(tau), _p(r), _p(q), _p(sigma),
                              _p(flag), *[_p(o) for o in outs])
    return tuple(outs)


def backward_inputs(gsigma, vega, status, vega_floor, mode, SorF, K, tau, sigma, flag, r=None, q=None):
    """xi_bar = -(gated sigma_bar / V) dP/dxi (eq.(8) second half): returns (gS|gF, gK, gtau, gr, gq)."""
    gsigma, vega, SorF, K, tau, sigma, flag = map(_d, (gsigma, vega, SorF, K, tau, sigma, flag))
    status = np.ascontiguousarray(status, dtype=np.uint8)
    r = None if r is None else _d(r)
    q = None if q is None else _d(q)
    outs = [np.empty(SorF.size) for _ in range(5)]
    lib().oracle_backward_inputs(C.c_int64(SorF.size), _p(gsigma), _p(vega), _p(status, _U8), C.c_double(vega_floor),
                                 C.c_int(mode), _p(SorF), _p(K), _p(tau), _p(r), _p(q), _p(sigma), _p(flag),
                                 *[_p(o) for o in outs])
    return tuple(outs)


def loss_price(SorF, K, tau, Pstar, flag, sigma_hat, r=None, q=None):
    """eq.(11) as raw sums: (sum (P_model - P*)^2, sum |P*|, rows used)."""
    SorF, K, tau, Pstar, flag, sigma_hat = map(_d, (SorF, K, tau, Pstar, flag, sigma_hat))
    r = None if r is None else _d(r)
    q = None if q is None else _d(q)
    out = np.empty(3)
    lib().oracle_loss_price(C.c_int64(SorF.size), _p(SorF), _p(K), _p(tau), _p(r), _p(q), _p(Pstar), _p(flag),
                            _p(sigma_hat), _p(out))
    return out


def loss_roundtrip(SorF, K, tau, Pstar, flag, sigma_hat, sigma_star, vega_floor, r=None, q=None):
    """eq.(12) as raw sums: (sum w (IV(P~) - sigma*)^2, sum w, rows used)."""
    SorF, K, tau, Pstar, flag, sigma_hat, sigma_star = map(_d, (SorF, K, tau, Pstar, flag, sigma_hat, sigma_star))
    r = None if r is None else _d(r)
    q = None if q is None else _d(q)
    out = np.empty(3)
    lib().oracle_loss_roundtrip(C.c_int64(SorF.size), _p(SorF), _p(K), _p(tau), _p(r), _p(q), _p(Pstar), _p(flag),
                                _p(sigma_hat), _p(sigma_star), C.c_double(vega_floor), _p(out))
    return out


def loss_price_grad(SorF, K, tau, Pstar, flag, sigma_hat, r=None, q=None):
    """d/d sigma_hat_i of (P_model_i - P*_i)^2 (eq.(11), unnormalised): 2 (P_model - P*) V_hat."""
    SorF, K, tau, Pstar, flag, sigma_hat = map(_d, (SorF, K, tau, Pstar, flag, sigma_hat))
    r = None if r is None else _d(r)
    q = None if q is None else _d(q)
    g = np.empty(SorF.size)
    lib().oracle_loss_price_grad(C.c_int64(SorF.size), _p(SorF), _p(K), _p(tau), _p(r), _p(q), _p(Pstar), _p(flag),
                                 _p(sigma_hat), _p(g))
    return g


def loss_roundtrip_grad(SorF, K, tau, Pstar, flag, sigma_hat, sigma_star, vega_floor, naive=False, r=None, q=None):
    """(d T_i / d sigma_hat_i, T_i) of the per-row round-trip terms of eq.(12) (gated) or of the naive composition."""
    SorF, K, tau, Pstar, flag, sigma_hat, sigma_star = map(_d, (SorF, K, tau, Pstar, flag, sigma_hat, sigma_star))
    r = None if r is None else _d(r)
    q = None if q is None else _d(q)
    g = np.empty(SorF.size); term = np.empty(SorF.size)
    lib().oracle_loss_roundtrip_grad(C.c_int64(SorF.size), _p(SorF), _p(K), _p(tau), _p(r), _p(q), _p(Pstar), _p(flag),
                                     _p(sigma_hat), _p(sigma_star), C.c_double(vega_floor), C.c_int(int(naive)), _p(g),
                                     _p(term))
    return g, term
