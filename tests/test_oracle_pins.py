"""Pins for the CPU oracle (oracle/): everything here runs without a GPU (-m "not gpu").

The paper prints no worked values for this path (tests/golden/README.md), so the oracle is pinned by what the paper
and the mathematics fix: eq.(4) evaluated literally in mpmath at 50 digits, mpmath derivatives of the transformed
objectives, the ATM closed form, a __float128 bisection of the literal definition eq.(3)/(6), price round trips,
put-call symmetries, monotonicity, the NaN domain, eq.(14) two ways and finite differences.
Each check is chosen so that a dropped term, wrong sign/index or transposed operand in oracle/lbr_oracle.hpp fails it.
"""
import math

import mpmath as mp
import numpy as np
import pytest

from oracle import pyoracle as po

mp.mp.dps = 50
EPS = np.finfo(np.float64).eps


# ------------------------------------------------------------------ mpmath definitions (independent of oracle/)
def mp_Phi(z):
    return mp.erfc(-z / mp.sqrt(2)) / 2


def mp_b(x, s):
    """eq.(4), with k = -x."""
    x, s = mp.mpf(x), mp.mpf(s)
    h, t = x / s, s / 2
    return mp.exp(x / 2) * mp_Phi(h + t) - mp.exp(-x / 2) * mp_Phi(h - t)


def mp_bprime(x, s):
    x, s = mp.mpf(x), mp.mpf(s)
    h, t = x / s, s / 2
    return mp.exp(-(h * h + t * t) / 2) / mp.sqrt(2 * mp.pi)


GRID_X = [0.0, -1e-9, -1e-4, -0.01, -0.3, -1.0, -2.5, -5.0]
GRID_S = [1e-4, 3e-3, 0.05, 0.099, 0.1, 0.101, 0.2, 0.5, 1.0, 2.0, 3.5, 5.0, 9.0, 30.0]


def _grid():
    pts = []
    for x in GRID_X:
        for s in GRID_S:
            if abs(x) / s <= 37.0:
                pts.append((x, s))
    return pts


# ------------------------------------------------------------------ special functions
def test_erfcx_matches_mpmath():
    z = np.concatenate([np.linspace(-5, 30, 141), [1e-8, 24.999, 25.0, 25.001, 60.0, 1e3, 1e7]])
    got = po.erfcx(z)
    ref = np.array([float(mp.exp(mp.mpf(v) ** 2) * mp.erfc(mp.mpf(v))) for v in z])
    assert np.max(np.abs(got / ref - 1)) <= 2 * EPS


def test_ninv_matches_mpmath():
    p = np.array([1e-300, 1e-100, 1e-20, 1e-5, 0.02, 0.3, 0.5, 0.7, 0.98, 1 - 1e-10])
    got = po.ninv(p)
    for pi, zi in zip(p, got):
        ref = mp.findroot(lambda z: mp_Phi(z) - mp.mpf(pi), mp.mpf(zi))
        assert abs(zi - float(ref)) <= 4 * EPS * max(1.0, abs(float(ref)))
    assert po.ninv(np.array([0.5]))[0] == pytest.approx(0.0, abs=1e-18)


# ------------------------------------------------------------------ O4: b, b', W, Wbar
def test_norm_black_matches_eq4():
    """sigma-equivalent error |b - b_eq4| / (s b') of the fp64 oracle stays at a few ulps in every regime
    (series t < 0.1, erfcx difference, direct eq.(4) for t - |h| > 10)."""
    pts = _grid()
    x = np.array([p[0] for p in pts]); s = np.array([p[1] for p in pts])
    b, v = po.norm_black(x, s, prec=0)
    worst = 0.0
    for xi, si, bi, vi in zip(x, s, b, v):
        bref, vref = mp_b(xi, si), mp_bprime(xi, si)
        if float(bref) < 1e-300:
            continue
        assert abs(vi / float(vref) - 1) <= 8 * EPS * (1 + (xi / si) ** 2 / 2 + si * si / 8)
        sig_equiv = abs((mp.mpf(bi) - bref) / (mp.mpf(si) * vref))
        rel = abs(mp.mpf(bi) / bref - 1)
        worst = max(worst, float(min(sig_equiv, rel)))
    assert worst <= 16 * EPS, worst


def test_W_and_Wbar_identities():
    """W = b/b', Wbar = (b_max - b)/b' against eq.(4)/(5)."""
    for x, s in _grid():
        if s > 20:
            continue
        h, t = (x / s if x != 0 else 0.0), s / 2
        w, wb = po.W(np.array([h]), np.array([t]), prec=1)
        bref, vref = mp_b(x, s), mp_bprime(x, s)
        if float(vref) < 1e-280:
            continue
        assert abs(w[0] / float(bref / vref) - 1) <= 2e-13 * (1 + h * h)
        bbar = mp.exp(mp.mpf(x) / 2) - bref
        assert abs(wb[0] / float(bbar / vref) - 1) <= 4 * EPS * (1 + h * h)


def test_series_and_erfcx_forms_agree_at_switch():
    h = -np.array([0.0, 0.5, 2.0, 7.0, 20.0])
    for t in (0.0999, 0.1001):
        ser = po.W_series(h, np.full_like(h, t), nterms=8)
        ref = np.array([float((mp_b(2 * hh * t, 2 * t)) / mp_bprime(2 * hh * t, 2 * t)) for hh in h])
        assert np.max(np.abs(ser / ref - 1) / (1 + h * h)) <= 8 * EPS
    # truncation: 6 terms are exact to fp64 at t = 0.1 and visibly short at t = 0.4
    h0 = np.array([-0.3])
    assert abs(po.W_series(h0, np.array([0.1]), 6)[0] / po.W_series(h0, np.array([0.1]), 10)[0] - 1) < 4 * EPS
    assert abs(po.W_series(h0, np.array([0.4]), 6)[0] / po.W_series(h0, np.array([0.4]), 12)[0] - 1) > 1e-12


def test_vega_ratio_derivatives():
    """b''/b' = h^2/s - s/4 and b'''/b' via the kind-1 Householder terms vs mpmath derivatives of eq.(4)."""
    for x, s in [(-0.3, 0.4), (-2.0, 1.1), (-1e-3, 0.02), (-4.0, 3.0)]:
        beta = float(mp_b(x, s)) * 1.01
        g, nu, h2, h3 = po.householder_terms([1], [x], [s], [beta], [math.exp(x / 2) - beta])
        f = lambda ss: mp_b(x, ss) - mp.mpf(beta)
        d1, d2, d3 = (mp.diff(f, mp.mpf(s), n) for n in (1, 2, 3))
        assert abs(g[0] / float(f(mp.mpf(s))) - 1) < 1e-10
        assert abs(nu[0] / float(-f(mp.mpf(s)) / d1) - 1) < 1e-10
        assert abs(h2[0] / float(d2 / d1) - 1) < 1e-12
        assert abs(h3[0] / float(d3 / d1) - 1) < 1e-12


# ------------------------------------------------------------------ O7: transformed objectives
@pytest.mark.parametrize("kind,x,s,rel", [(0, -1.0, 0.35, 0.9), (0, -3.0, 0.8, 1.2), (0, -0.02, 0.01, 0.95),
                                          (2, -0.5, 3.0, 0.97), (2, -2.0, 4.5, 1.05), (2, 0.0, 2.9, 1.01)])
def test_householder_terms_match_mpmath_derivatives(kind, x, s, rel):
    """nu = -g/g', h2 = g''/g', h3 = g'''/g' for g = 1/ln b - 1/ln beta (zone 0) and g = ln((b_max-beta)/(b_max-b))."""
    bmax = mp.exp(mp.mpf(x) / 2)
    b_here = mp_b(x, s)
    if kind == 0:
        beta = b_here * rel
        g = lambda ss: 1 / mp.log(mp_b(x, ss)) - 1 / mp.log(beta)
    else:
        beta = bmax - (bmax - b_here) * rel
        g = lambda ss: mp.log((bmax - beta) / (bmax - mp_b(x, ss)))
    d0 = g(mp.mpf(s)); d1, d2, d3 = (mp.diff(g, mp.mpf(s), n) for n in (1, 2, 3))
    gg, nu, h2, h3 = po.householder_terms([kind], [x], [s], [float(beta)], [float(bmax - beta)])
    assert abs(gg[0] / float(d0) - 1) < 1e-9
    assert abs(nu[0] / float(-d0 / d1) - 1) < 1e-9
    assert abs(h2[0] / float(d2 / d1) - 1) < 1e-11
    assert abs(h3[0] / float(d3 / d1) - 1) < 1e-11


# ------------------------------------------------------------------ O5/O6: boundary points and interpolants
def test_inflection_and_tangent_points():
    """s_c = sqrt(2|x|) is the inflection of b (b''(s_c) = 0); the tangent there meets 0 at s_l and b_max at s_u."""
    for x in (-0.05, -1.0, -4.0):
        beta = 0.5 * float(mp_b(x, math.sqrt(-2 * x)))
        _, _, _, nd = po.solve_normalised([x], [beta], nodes=True, prec=1)
        sl, sc, su, bl, bc, bu = nd[0]
        assert sc == pytest.approx(math.sqrt(-2 * x), rel=1e-15)
        assert abs(float(mp.diff(lambda ss: mp_b(x, ss), mp.sqrt(-2 * mp.mpf(x)), 2))) < 1e-40
        vc = float(mp_bprime(x, sc)); bcr = float(mp_b(x, sc))
        assert bc == pytest.approx(bcr, rel=1e-14)
        assert sl == pytest.approx(sc - bcr / vc, rel=1e-12)
        assert su == pytest.approx(sc + (math.exp(x / 2) - bcr) / vc, rel=1e-13)
        assert bl == pytest.approx(float(mp_b(x, sl)), rel=1e-13)


def test_rational_cubic_end_conditions():
    """End values, end slopes, and the control parameter reproducing a prescribed second derivative."""
    H, yl, yr, dl, dr = 0.7, 0.2, 1.3, 0.9, 2.8
    for side, dd in ((0, 1.7), (1, 3.1)):
        r = po.control_fit(side, H, yl, yr, dl, dr, dd, floor_it=False)
        f = lambda u: po.rational_cubic(np.atleast_1d(u), H, yl, yr, dl, dr, r)
        assert f(0.0)[0] == pytest.approx(yl, rel=1e-15) and f(1.0)[0] == pytest.approx(yr, rel=1e-15)
        e = 1e-6
        assert (f(e)[0] - f(0.0)[0]) / (e * H) == pytest.approx(dl, rel=1e-4)
        assert (f(1.0)[0] - f(1 - e)[0]) / (e * H) == pytest.approx(dr, rel=1e-4)
        e = 1e-4
        u0 = 0.0 if side == 0 else 1.0
        sg = 1 if side == 0 else -1
        # one-sided second difference at the end point
        d2 = (2 * f(u0)[0] - 5 * f(u0 + sg * e)[0] + 4 * f(u0 + 2 * sg * e)[0] - f(u0 + 3 * sg * e)[0]) / (e * H) ** 2
        assert d2 == pytest.approx(dd, rel=2e-3)
    # r -> large: linear interpolation
    assert po.rational_cubic(np.array([0.25]), H, yl, yr, dl, dr, 1e301)[0] == pytest.approx(yl + 0.25 * (yr - yl))
    # shape floor keeps a monotone convex data set monotone
    r = po.control_fit(0, 1.0, 0.0, 1.0, 0.1, 5.0, -50.0, floor_it=True)
    y = po.rational_cubic(np.linspace(0, 1, 101), 1.0, 0.0, 1.0, 0.1, 5.0, r)
    assert np.all(np.diff(y) > 0)


def _shape_ok(kind, H, yl, yr, dl, dr, r, m=4001):
    u = np.linspace(0.0, 1.0, m)
    y = po.rational_cubic(u, H, yl, yr, dl, dr, r)
    if not np.all(np.isfinite(y)):
        return False
    if kind == "monotone":
        return bool(np.all(np.diff(y) > 0))
    d2 = np.diff(y, 2)
    tol = 1e-13 * np.max(np.abs(y))
    return bool(np.all(d2 >= -tol)) if kind == "convex" else bool(np.all(d2 <= tol))


def test_shape_floor_is_the_smallest_shape_preserving_control():
    """min_control (the floor under every fitted control parameter) pinned by brute force on the interpolant itself,
    not by its formula: for convex / concave data the floor must be the smallest r whose rational cubic keeps the shape on a
    fine grid (found by bisection on r: the second derivative at one end changes sign there), on data sets in which each of the
    two ratio terms is the binding one; for monotone data with an inflection (where the (dl + dr)/Delta term binds) the floor
    keeps the interpolant monotone and a control of a tenth of that size does not.  A dropped or mis-signed term fails one of these."""
    cases = [("convex", 1.0, 0.0, 1.0, 0.2, 1.1),     # dr close to Delta: |dr - dl| / (dr - Delta) binds
             ("convex", 0.7, 0.3, 1.0, 0.9, 4.0),     # dl close to Delta: |dr - dl| / (Delta - dl) binds
             ("convex", 2.0, -1.0, 3.0, 0.5, 3.0),
             ("concave", 1.0, 0.0, 1.0, 3.0, 0.8),
             ("concave", 0.5, 2.0, 2.6, 1.3, 0.1)]
    binding = set()
    for kind, H, yl, yr, dl, dr in cases:
        Delta = (yr - yl) / H
        rmin = po.control_fit(0, H, yl, yr, dl, dr, -1e300 if Delta > dl else 1e300, floor_it=True)   # fitted r -> -inf: the floor
        assert rmin == po.control_fit(1, H, yl, yr, dl, dr, -1e300 if dr > Delta else 1e300, floor_it=True)
        assert _shape_ok(kind, H, yl, yr, dl, dr, rmin * (1 + 1e-6))
        lo, hi = 0.0, rmin * (1 + 1e-6)           # bisection for the smallest shape-preserving r
        assert not _shape_ok(kind, H, yl, yr, dl, dr, lo + 1e-3)
        for _ in range(60):
            mid = 0.5 * (lo + hi)
            lo, hi = (lo, mid) if _shape_ok(kind, H, yl, yr, dl, dr, mid) else (mid, hi)
        assert hi == pytest.approx(rmin, rel=2e-3), (kind, H, yl, yr, dl, dr, hi, rmin)
        binding.add(abs(dr - Delta) < abs(Delta - dl))
    assert binding == {True, False}
    # monotone data with an inflection: slopes on both sides above the secant slope
    for H, yl, yr, dl, dr in [(1.0, 0.0, 1.0, 2.0, 2.0), (0.4, 1.0, 1.2, 1.5, 0.9), (1.0, 0.0, 1.0, 5.0, 5.0)]:
        Delta = (yr - yl) / H
        rmin = po.control_fit(0, H, yl, yr, dl, dr, 1e300 if Delta < dl else -1e300, floor_it=True)
        assert rmin >= (dl + dr) / Delta * (1 - 1e-12)
        assert _shape_ok("monotone", H, yl, yr, dl, dr, rmin)
        assert not _shape_ok("monotone", H, yl, yr, dl, dr, 0.1 * rmin)   # far below the floor the interpolant overshoots


def test_seed_transform_end_derivatives():
    """f_low, f_up and their first/second derivatives w.r.t. beta vs mpmath differentiation of f(s(beta))."""
    for x, s in [(-0.4, 0.5), (-2.0, 1.2), (-4.5, 2.0)]:
        a = -x
        flow = lambda ss: (2 * mp.pi * a / (3 * mp.sqrt(3))) * mp_Phi(-a / (mp.sqrt(3) * ss)) ** 3
        fup = lambda ss: mp_Phi(-ss / 2)
        for fun, got in ((flow, po.f_low_end(a, s)), (fup, po.f_up_end(x, s))):
            d1 = lambda ss: mp.diff(fun, ss) / mp.diff(lambda q: mp_b(x, q), ss)          # df/dbeta
            d2 = mp.diff(d1, mp.mpf(s)) / mp.diff(lambda q: mp_b(x, q), mp.mpf(s))          # d2f/dbeta2
            assert got[0] == pytest.approx(float(fun(mp.mpf(s))), rel=1e-14)
            assert got[1] == pytest.approx(float(d1(mp.mpf(s))), rel=1e-12)
            assert got[2] == pytest.approx(float(d2), rel=1e-10)


def test_seed_quality_and_zone_continuity():
    """The rational seed is within 12% (zone 0) / 1% (zones 1-3) of the root, and continuous across b_l, b_c, b_u."""
    rng = np.random.default_rng(5)
    n = 20000
    x = -rng.uniform(0, 5, n)
    s = np.exp(rng.uniform(np.log(1e-3), np.log(6), n))
    s = np.maximum(s, np.abs(x) / 30)
    b, _ = po.norm_black(x, s, prec=1)
    keep = b > 1e-290
    x, s, b = x[keep], s[keep], b[keep]
    sol, zone, s0 = po.solve_normalised(x, b, prec=0)
    assert set(np.unique(zone)) == {0, 1, 2, 3}
    err = np.abs(s0 / s - 1)
    assert err[zone == 0].max() < 0.12 and err[zone != 0].max() < 1e-2
    for xx in (-0.2, -1.5, -4.0):
        _, _, _, nd = po.solve_normalised([xx, xx], [1e-12, 0.99 * math.exp(xx / 2)], nodes=True)
        sl, sc, su, bl, bc, _ = nd[0]
        bu = nd[1][5]
        for bnode, snode in ((bl, sl), (bc, sc), (bu, su)):
            lo, hi = bnode * (1 - 1e-9), bnode * (1 + 1e-9)
            _, z, seeds = po.solve_normalised([xx, xx], [lo, hi])
            assert z[0] + 1 == z[1]
            assert seeds[0] == pytest.approx(snode, rel=1e-6) and seeds[1] == pytest.approx(snode, rel=1e-6)


# ------------------------------------------------------------------ whole solver
def test_atm_closed_form():
    """x = 0: sigma = -2 Phi^-1((1-beta)/2)/sqrt(T) (north_star; from eq.(4): b(0,s) = 1 - 2 Phi(-s/2))."""
    F = 100.0
    T = np.array([0.01, 0.25, 1.0, 2.0, 1.0, 0.5])
    beta = np.array([1e-6, 0.02, 0.15, 0.4, 0.9, 0.999999])
    P = beta * F
    sig, vega, st = po.forward(np.full(6, F), np.full(6, F), T, P, np.array([1.0, -1, 1, -1, 1, -1]))
    assert np.all(st == 0)
    for i in range(6):
        ref = -2 * mp.findroot(lambda z: mp_Phi(z) - (1 - mp.mpf(float(P[i])) / F) / 2, 0) / mp.sqrt(mp.mpf(float(T[i])))
        assert sig[i] == pytest.approx(float(ref), rel=8 * EPS)


def _rows(n, seed, otm_only=True, smin=1e-4):
    rng = np.random.default_rng(seed)
    x = rng.uniform(-5, 5, n)
    s = np.exp(rng.uniform(np.log(smin), np.log(6), n))
    s = np.maximum(s, np.abs(x) / 34)
    T = np.exp(rng.uniform(np.log(1 / 365), np.log(2), n))
    F = np.full(n, 100.0); K = F * np.exp(-x)
    otm = np.where(K >= F, 1.0, -1.0)
    flag = otm if otm_only else np.where(rng.random(n) < 0.5, 1.0, -1.0)
    sig = s / np.sqrt(T)
    tv = po.black_price(F, K, T, sig, otm, prec=1)
    P = np.maximum(flag * (F - K), 0.0) + tv
    return F, K, T, P, flag, sig, s, x


def test_truth_solver_against_mpmath_root():
    """The __float128 bisection is itself pinned by mpmath.findroot on the literal eq.(3) price."""
    F, K, T, P, flag, sig, s, x = _rows(12, 11)
    tr = po.truth_iv(F, K, T, P, flag)
    for i in range(12):
        th = mp.mpf(float(flag[i])); Fi, Ki, Ti = mp.mpf(float(F[i])), mp.mpf(float(K[i])), mp.mpf(float(T[i]))
        def price(v):
            st = v * mp.sqrt(Ti); d1 = (mp.log(Fi / Ki) + st * st / 2) / st; d2 = d1 - st
            return th * (Fi * mp_Phi(th * d1) - Ki * mp_Phi(th * d2)) - mp.mpf(float(P[i]))
        ref = mp.findroot(price, mp.mpf(float(sig[i])), tol=1e-40, maxsteps=100)
        assert tr[i] == pytest.approx(float(ref), rel=2 * EPS)


def test_truth_solver_bsm_branch_against_mpmath_root_of_eq2():
    """The (S, K, tau, r, q) branch of the __float128 bisection pinned by mpmath.findroot on the literal SPOT form of eq.(2)
    (PAPER.md:55-57): theta (S e^{-q tau} Phi(theta d1) - K e^{-r tau} Phi(theta d2)), d1 = (ln(S/K) + (r - q + sigma^2/2) tau) /
    (sigma sqrt(tau)) -- a different arrangement from the forward / discount-factor form the oracle evaluates, so a wrong sign of
    r or q, a missing discount factor or a swapped carry term shows; calls and puts, in and out of the money, r < q included."""
    rng = np.random.default_rng(21)
    n = 16
    S = rng.lognormal(np.log(100.0), 0.2, n); K = S * rng.uniform(0.6, 1.5, n)
    tau = np.exp(rng.uniform(np.log(5 / 365), np.log(2.5), n)); r = rng.uniform(-0.01, 0.08, n); q = rng.uniform(0.0, 0.06, n)
    sig = rng.uniform(0.08, 0.9, n); flag = np.where(rng.random(n) < 0.5, 1.0, -1.0)
    P = np.empty(n)
    for i in range(n):
        Si, Ki, Ti, ri, qi, th = (mp.mpf(float(v)) for v in (S[i], K[i], tau[i], r[i], q[i], flag[i]))
        def price(v, Si=Si, Ki=Ki, Ti=Ti, ri=ri, qi=qi, th=th):
            st = v * mp.sqrt(Ti); d1 = (mp.log(Si / Ki) + (ri - qi + v * v / 2) * Ti) / st; d2 = d1 - st
            return th * (Si * mp.exp(-qi * Ti) * mp_Phi(th * d1) - Ki * mp.exp(-ri * Ti) * mp_Phi(th * d2))
        P[i] = float(price(mp.mpf(float(sig[i]))))
    tr = po.truth_iv(S, K, tau, P, flag, r=r, q=q)
    assert (r < q).any() and (flag > 0).any() and (flag < 0).any()
    for i in range(n):
        Si, Ki, Ti, ri, qi, th = (mp.mpf(float(v)) for v in (S[i], K[i], tau[i], r[i], q[i], flag[i]))
        def resid(v):
            st = v * mp.sqrt(Ti); d1 = (mp.log(Si / Ki) + (ri - qi + v * v / 2) * Ti) / st; d2 = d1 - st
            return th * (Si * mp.exp(-qi * Ti) * mp_Phi(th * d1) - Ki * mp.exp(-ri * Ti) * mp_Phi(th * d2)) - mp.mpf(float(P[i]))
        ref = mp.findroot(resid, mp.mpf(float(sig[i])), tol=1e-40, maxsteps=100)
        assert tr[i] == pytest.approx(float(ref), rel=2 * EPS), i
        # and the oracle's own forward pass agrees with that root (conditioning: sigma moves by ~ eps P / (V sigma))
        sg, vega, st_ = po.forward(S[i:i + 1], K[i:i + 1], tau[i:i + 1], P[i:i + 1], flag[i:i + 1], r=r[i:i + 1], q=q[i:i + 1])
        assert st_[0] == 0 and abs(sg[0] / float(ref) - 1) <= 8 * EPS * (1 + P[i] / (vega[0] * float(ref)))


def test_lbr_matches_float128_bisection_all_zones():
    """>= 1e4 tiny-input rows over 4 zones x b-regimes: fp64 O-LBR agrees with the definition's root to a few ulps
    (OTM rows, where the time value is an input and not a rounded subtraction)."""
    F, K, T, P, flag, sig, s, x = _rows(12000, 12)
    o = po.forward(F, K, T, P, flag, prec=0, debug=True)
    ok = o[2] == 0
    assert ok.mean() > 0.95
    assert all((o[3][ok] == z).sum() > 300 for z in range(4))
    tr = po.truth_iv(F, K, T, P, flag)
    err = np.abs(o[0][ok] / tr[ok] - 1)
    assert err.max() <= 24 * EPS, err.max()
    # exactly two Householder steps (the GPU's count) reach the same accuracy
    o2 = po.forward(F, K, T, P, flag, prec=0, fixed_iters=2)
    assert np.abs(o2[0][ok] / tr[ok] - 1).max() <= 24 * EPS
    # one step does not (so the step is doing real work and the seed is not secretly exact)
    o1 = po.forward(F, K, T, P, flag, prec=0, fixed_iters=1)
    assert np.abs(o1[0][ok] / tr[ok] - 1).max() > 1e-9


def test_lbr_zone_edges_and_extremes():
    """beta at the zone boundaries +-1 ulp, beta -> 0, beta -> b_max, tiny |x|."""
    rows = []
    for x in (-1e-12, -1e-6, -0.1, -2.0, -5.0):
        bmax = math.exp(x / 2)
        _, _, _, nd = po.solve_normalised([x, x], [1e-14, 0.99 * bmax], nodes=True)
        sl, sc, su, bl, bc, _ = nd[0]
        bu = nd[1][5]
        for bnode in (bl, bc, bu):
            rows += [(x, np.nextafter(bnode, 0)), (x, bnode), (x, np.nextafter(bnode, 1))]
        rows += [(x, 1e-300), (x, 1e-100), (x, bmax * (1 - 1e-9)), (x, bmax * 0.5)]
    F = 100.0
    for x, beta in rows:
        K = F * math.exp(-x)
        P = beta * math.sqrt(F * K)
        if not P < F:
            continue
        sig, _, st = po.forward([F], [K], [1.0], [P], [1.0])
        tr = po.truth_iv([F], [K], [1.0], [P], [1.0])
        assert st[0] == 0
        # relative conditioning of the root w.r.t. the rounded P near b_max is ~ eps * b / (s b')
        b, v = po.norm_black([math.log(F / K)], [sig[0]], prec=1)
        cond = max(1.0, min(beta, math.sqrt(F / K) - beta) / (sig[0] * max(v[0], 1e-300)))
        assert abs(sig[0] / tr[0] - 1) <= 32 * EPS * cond, (x, beta, sig[0], tr[0])


def test_price_round_trip():
    """Black price of the returned sigma equals P to 1e-13 relative to P (north_star; paper Q50 1.1e-13)."""
    F, K, T, P, flag, sig, s, x = _rows(20000, 13, otm_only=False)
    sg, vega, st = po.forward(F, K, T, P, flag)
    ok = st == 0
    back = po.black_price(F[ok], K[ok], T[ok], sg[ok], flag[ok], prec=1)
    # sigma itself is only known to ~eps relative, which moves the price by (vega sigma / P) * eps: in the far tail the
    # elasticity vega*sigma/P ~ h^2 reaches ~1e3, so the 1e-13 bar applies where the elasticity is <= 100 and scales beyond
    elast = vega[ok] * sg[ok] / P[ok]
    rel = np.abs(back / P[ok] - 1)
    assert np.max(rel[elast <= 100]) <= 1e-13
    assert np.max(rel / np.maximum(1.0, elast)) <= 4 * EPS
    # and the oracle's own pricer agrees with the literal eq.(3) in __float128
    lit = po.black_literal_q(F[ok], K[ok], np.ones(ok.sum()), T[ok], sg[ok], flag[ok])
    assert np.max(np.abs(back / lit - 1)) <= 1e-13


def test_bsm_mode_round_trip_and_truth():
    """(S,K,tau,r,q,P) path: F = S e^{(r-q)tau}, beta = e^{r tau} P / sqrt(FK)."""
    rng = np.random.default_rng(14)
    n = 3000
    S = rng.lognormal(np.log(4000), 0.25, n); K = S * rng.uniform(0.5, 1.6, n)
    tau = np.exp(rng.uniform(np.log(1 / 365), np.log(3), n)); r = rng.uniform(0, 0.05, n); q = rng.uniform(0, 0.02, n)
    sig = rng.uniform(0.1, 0.6, n)
    Fw = S * np.exp((r - q) * tau)
    flag = np.where(K >= Fw, 1.0, -1.0)
    P = po.black_price(S, K, tau, sig, flag, r=r, q=q, prec=1)
    good = P > 1e-200
    sg, vega, st = po.forward(S, K, tau, P, flag, r=r, q=q)
    assert np.all(st[good] == 0)
    tr = po.truth_iv(S, K, tau, P, flag, r=r, q=q)
    # F and D carry one rounding each: sigma moves by ~ eps * 1.25 / s
    s = sig * np.sqrt(tau)
    assert np.max(np.abs(sg[good] / tr[good] - 1) * np.minimum(s[good], 1.0)) <= 16 * EPS
    lit = po.vega_eq14(S, K, tau, sg, r=r, q=q)
    assert np.max(np.abs(vega[good] / lit[good] - 1)) <= 1e-12


def test_reflection_symmetry_is_bit_exact():
    """IV(F,K,put,P) == IV(K,F,call,P) bit for bit (O2/O3 are symmetric in (F,K) under theta -> -theta)."""
    F, K, T, P, flag, sig, s, x = _rows(5000, 15, otm_only=False)
    a = po.forward(F, K, T, P, flag)
    b = po.forward(K, F, T, P, -flag)
    assert np.array_equal(a[2], b[2])
    assert np.array_equal(a[0].view(np.uint64), b[0].view(np.uint64))
    assert np.array_equal(a[1].view(np.uint64), b[1].view(np.uint64))


def test_put_call_parity():
    """IV(call C) == IV(put C - (F-K)) at D = 1, on rows where both subtractions are benign."""
    F, K, T, P, flag, sig, s, x = _rows(5000, 16, smin=0.05)
    m = np.abs(x) < 0.5
    F, K, T, P, flag = F[m], K[m], T[m], P[m], flag[m]
    other = P + (-flag) * (K - F) * -1.0  # theta' = -theta: P' = P - theta (F - K)
    other = P - flag * (F - K)
    a = po.forward(F, K, T, P, flag)
    b = po.forward(F, K, T, other, -flag)
    ok = (a[2] == 0) & (b[2] == 0)
    assert ok.mean() > 0.9
    cond = np.maximum(1.0, np.abs(other[ok]) / P[ok])
    assert np.max(np.abs(a[0][ok] / b[0][ok] - 1) / cond) <= 64 * EPS


def test_monotone_in_price():
    for x in (-2.0, -0.3, 0.0):
        F = 100.0; K = F * math.exp(-x)
        P = np.exp(np.linspace(np.log(1e-250), np.log(F * 0.999999), 4001))
        sig, _, st = po.forward(np.full_like(P, F), np.full_like(P, K), np.full_like(P, 0.7), P, np.ones_like(P))
        assert np.all(st == 0)
        assert np.all(np.diff(sig) >= -4 * EPS * sig[1:])


def test_nan_domain_and_status_codes():
    """NaN iff P < intrinsic, P >= upper bound or bad input; never NaN inside (DESIGN.md readings)."""
    F, K = 100.0, 90.0
    nan, inf = float("nan"), float("inf")
    cases = [  # (F, K, T, P, flag) -> status
        ((F, K, 1.0, 9.999, 1.0), 1), ((F, K, 1.0, 10.0, 1.0), 4), ((F, K, 1.0, np.nextafter(10.0, 11), 1.0), 0),
        ((F, K, 1.0, 99.99, 1.0), 0), ((F, K, 1.0, 100.0, 1.0), 2), ((F, K, 1.0, 101.0, 1.0), 2),
        ((F, K, 1.0, -1e-9, -1.0), 1), ((F, K, 1.0, 0.0, -1.0), 4), ((F, K, 1.0, 1e-320, -1.0), 4),
        ((F, K, 1.0, 89.9, -1.0), 0), ((F, K, 1.0, 90.0, -1.0), 2),
        ((F, K, 0.0, 12.0, 1.0), 3), ((F, K, -1.0, 12.0, 1.0), 3), ((F, K, nan, 12.0, 1.0), 3), ((F, K, inf, 12.0, 1.0), 3),
        ((0.0, K, 1.0, 12.0, 1.0), 3), ((F, -K, 1.0, 12.0, 1.0), 3), ((nan, K, 1.0, 12.0, 1.0), 3),
        ((F, K, 1.0, nan, 1.0), 3), ((F, K, 1.0, inf, 1.0), 3), ((F, K, 1.0, 12.0, 0.0), 3), ((F, K, 1.0, 12.0, 2.0), 3),
    ]
    arr = np.array([c[0] for c in cases])
    sig, vega, st = po.forward(arr[:, 0], arr[:, 1], arr[:, 2], arr[:, 3], arr[:, 4])
    assert list(st) == [c[1] for c in cases]
    for s_, v_, code in zip(sig, vega, st):
        if code in (1, 2, 3):
            assert np.isnan(s_) and v_ == 0.0
        elif code == 4:
            assert s_ == 0.0 and v_ == 0.0
        else:
            assert np.isfinite(s_) and s_ > 0 and v_ >= 0
    # inside the open interval it is never NaN
    F_, K_, T_, P_, fl, *_ = _rows(20000, 17, otm_only=False)
    sg, vg, st = po.forward(F_, K_, T_, P_, fl)
    assert not np.isnan(sg[st == 0]).any() and np.all(np.isin(st, (0, 4)))
    # BSM mode: non-finite r / q is bad input
    _, _, st = po.forward([100.0] * 2, [90.0] * 2, [1.0] * 2, [12.0] * 2, [1.0] * 2, r=[nan, 0.01], q=[0.0, inf])
    assert list(st) == [3, 3]


def test_extreme_log_moneyness_is_bad_input():
    """|x| > 693 (b_max = e^{-|x|/2} < 2^-500): every normalised price sits at the fp64 underflow edge -> BAD_INPUT,
    never an OK row carrying NaN (reading 17); |x| ~ 600 still solves."""
    sig, vega, st = po.forward([1e-300, 1e300, 1e-130, 1e-100], [1e300, 1e-300, 1e130, 1e100], [1.0] * 4,
                               [1e-301, 1e299, 1e-135, 1e-101], [1.0, -1.0, 1.0, 1.0])
    assert list(st) == [3, 3, 0, 0]
    assert np.isnan(sig[:2]).all() and np.isfinite(sig[2:]).all()
    tr = po.truth_iv([1e-130, 1e-100], [1e130, 1e100], [1.0] * 2, [1e-135, 1e-101], [1.0, 1.0])
    assert np.max(np.abs(sig[2:] / tr - 1)) <= 1e-13


def test_vega_two_ways_and_finite_difference():
    """eq.(14): F e^{-r tau} phi(d1) sqrt(tau) == normalised form sqrt(FK) b' sqrt(tau); and d(price)/d(sigma) by central FD."""
    F, K, T, P, flag, sig, s, x = _rows(4000, 18, otm_only=False, smin=0.02)
    sg, vega, st = po.forward(F, K, T, P, flag)
    ok = (st == 0) & (vega > 1e-200)
    v14 = po.vega_eq14(F[ok], K[ok], T[ok], sg[ok])
    st_ = sg[ok] * np.sqrt(T[ok])
    expo = 0.5 * ((x[ok] / st_) ** 2 + st_ ** 2 / 4)      # |exponent| of phi(d1): its rounding is the error budget
    assert np.max(np.abs(vega[ok] / v14 - 1) / (1 + expo)) <= 8 * EPS
    m = ok & (vega > 1e-3)
    e = 1e-4 * sg[m]
    fd = (po.black_price(F[m], K[m], T[m], sg[m] + e, flag[m]) - po.black_price(F[m], K[m], T[m], sg[m] - e, flag[m])) / (2 * e)
    assert np.max(np.abs(fd / vega[m] - 1)) <= 5e-6 and np.median(np.abs(fd / vega[m] - 1)) <= 1e-7


def test_implicit_gradient_vs_central_fd():
    """d sigma / d P = 1/V (eq.(7)) against central FD of the oracle in P, h in {1e-6, 1e-3}."""
    F, K, T, P, flag, sig, s, x = _rows(4000, 19, otm_only=True, smin=0.05)
    sg, vega, st = po.forward(F, K, T, P, flag)
    band = (st == 0) & (vega > 1.0) & (P > 0.5) & (P < 0.9 * np.minimum(F, K))
    assert band.sum() > 300
    for h, tol in ((1e-6, 2e-6), (1e-3, 2e-5)):
        up = po.forward(F[band], K[band], T[band], P[band] + h, flag[band])[0]
        dn = po.forward(F[band], K[band], T[band], P[band] - h, flag[band])[0]
        fd = (up - dn) / (2 * h)
        rel = np.abs(fd * vega[band] - 1)
        assert np.median(rel) <= tol and np.quantile(rel, 0.99) <= 100 * tol


def test_backward_gate_truth_table():
    """O9 / eq.(8)-(10): MASK -> gs/V iff OK and |V| > floor (strict), else exactly +0; ATTENUATE -> gs V/(V^2+floor^2)."""
    floor = 1e-8
    vegas = [0.0, 1e-300, np.nextafter(floor, 0), floor, np.nextafter(floor, 1), 1e-3, 7.5]
    for status in (0, 1, 2, 3, 4):
        for V in vegas:
            for gs in (0.0, -2.5, 1e300, float("nan"), float("inf")):
                for mode in (0, 1):
                    out = po.backward([gs], [V], [status], floor, mode)[0]
                    if status != 0:
                        assert out == 0.0 and not np.signbit(out)
                    elif mode == 0:
                        if abs(V) > floor:
                            exp = gs / V
                            assert (np.isnan(exp) and np.isnan(out)) or out == exp
                        else:
                            assert out == 0.0 and not np.signbit(out)
                    else:
                        exp = gs * V / (V * V + floor * floor)
                        assert (np.isnan(exp) and np.isnan(out)) or out == exp
    # attenuate == w_tau(V) * gs / V  (eq.(10)) and -> gs/V for V >> floor
    V = np.array([1e-9, 1e-8, 1e-6, 0.3]); gs = np.array([1.0, -2.0, 3.0, 0.5])
    att = po.backward(gs, V, np.zeros(4, np.uint8), floor, 1)
    w = V ** 2 / (V ** 2 + floor ** 2)
    assert np.allclose(att, w * gs / V, rtol=1e-15)
    assert att[3] == pytest.approx(gs[3] / V[3], rel=1e-12)
    # STRICT: exact gradient on the gate, +0 off the gate iff the upstream cotangent is 0, else NaN
    for status in (0, 1, 2, 3, 4):
        for V in vegas:
            for gs in (0.0, -0.0, -2.5, 1e300, float("nan"), float("inf")):
                out = po.backward([gs], [V], [status], floor, 2)[0]
                if status == 0 and abs(V) > floor:
                    exp = gs / V
                    assert (np.isnan(exp) and np.isnan(out)) or out == exp
                elif gs == 0.0:
                    assert out == 0.0 and not np.signbit(out)
                else:
                    assert np.isnan(out)
    # floor = 0: attenuate at V = 0 stays finite (0), mask at V = 0 is off-gate
    assert po.backward([1.0], [0.0], [0], 0.0, 1)[0] == 0.0 and po.backward([1.0], [0.0], [0], 0.0, 0)[0] == 0.0


# ------------------------------------------------------------------ input gradients, eq.(8) second half
def _bsm_rows(n, seed):
    rng = np.random.default_rng(seed)
    S = np.exp(rng.normal(np.log(4000.0), 0.25, n))
    K = S * rng.uniform(0.7, 1.4, n)
    tau = np.exp(rng.uniform(np.log(10 / 365), np.log(2.0), n))
    r = rng.uniform(0.0, 0.05, n)
    q = rng.uniform(0.0, 0.02, n)
    sig = rng.uniform(0.1, 0.6, n)
    flag = np.where(rng.random(n) < 0.5, 1.0, -1.0)
    return S, K, tau, r, q, sig, flag


def test_black_greeks_against_mpmath_derivatives_of_eq2():
    """Each of the five closed forms against mpmath's numerical derivative of the literal eq.(2) price (50 digits):
    a wrong sign, a dropped discount factor or a swapped d1/d2 fails it."""
    S, K, tau, r, q, sig, flag = _bsm_rows(40, 5)

    def price(S_, K_, t_, r_, q_, sg_, th):
        s = sg_ * mp.sqrt(t_)
        d1 = (mp.log(S_ / K_) + (r_ - q_) * t_ + s * s / 2) / s
        d2 = d1 - s
        return th * (S_ * mp.exp(-q_ * t_) * mp_Phi(th * d1) - K_ * mp.exp(-r_ * t_) * mp_Phi(th * d2))

    g = po.black_greeks(S, K, tau, sig, flag, r=r, q=q, prec=1)
    for i in range(S.size):
        a = [mp.mpf(float(v[i])) for v in (S, K, tau, r, q)]
        sg, th = mp.mpf(float(sig[i])), int(flag[i])
        for j in range(5):
            f = lambda z, j=j: price(*[z if m == j else a[m] for m in range(5)], sg, th)
            ref = mp.diff(f, a[j])
            got = mp.mpf(float(g[j][i]))
            scale = max(abs(ref), mp.mpf(1e-3) * abs(price(*a, sg, th)) / abs(a[j]) if a[j] != 0 else 0)
            assert abs(got - ref) <= 1e-12 * scale + 1e-15, (i, j, got, ref)


def test_black76_greeks_reduce_to_forward_form():
    """r = q = NULL: dP/dF = theta Phi(theta d1), dP/dK = -theta Phi(theta d2), dP/dtau = V sigma/(2 tau); dr = dq = 0."""
    S, K, tau, r, q, sig, flag = _bsm_rows(500, 6)
    g = po.black_greeks(S, K, tau, sig, flag, prec=1)
    e = 1e-5
    pF = (po.black_price(S * (1 + e), K, tau, sig, flag) - po.black_price(S * (1 - e), K, tau, sig, flag)) / (2 * e * S)
    pK = (po.black_price(S, K * (1 + e), tau, sig, flag) - po.black_price(S, K * (1 - e), tau, sig, flag)) / (2 * e * K)
    pT = (po.black_price(S, K, tau * (1 + e), sig, flag) - po.black_price(S, K, tau * (1 - e), sig, flag)) / (2 * e * tau)
    assert np.max(np.abs(g[0] - pF)) <= 1e-7
    assert np.max(np.abs(g[1] - pK)) <= 1e-7
    assert np.all(np.abs(g[2] - pT) <= 1e-6 * np.abs(g[2]) + 1e-6)
    assert np.all(g[3] == 0) and np.all(g[4] == 0)
    assert np.allclose(g[2], po.vega_eq14(S, K, tau, sig) * sig / (2 * tau), rtol=1e-13, atol=0)


def test_input_gradients_are_the_implicit_derivatives_of_the_solver():
    """xi_bar for sigma_bar = 1 must equal d sigma_imp / d xi of the oracle's own inversion (implicit function theorem,
    eq.(8)): central differences of po.forward in S, K, tau, r, q at fixed observed price."""
    S, K, tau, r, q, sig, flag = _bsm_rows(600, 8)
    P = po.black_price(S, K, tau, sig, flag, r=r, q=q)
    s0, v0, st = po.forward(S, K, tau, P, flag, r=r, q=q)
    m = (st == 0) & (v0 > 50.0)
    assert m.sum() > 300
    S, K, tau, r, q, flag, P, s0, v0, st = (a[m] for a in (S, K, tau, r, q, flag, P, s0, v0, st))
    gin = po.backward_inputs(np.ones_like(s0), v0, st, 1e-8, 0, S, K, tau, s0, flag, r=r, q=q)
    args = [S, K, tau, r, q]
    for j, h in enumerate((1e-6, 1e-6, 1e-6, 1e-7, 1e-7)):
        up = list(args); dn = list(args)
        step = h * np.maximum(np.abs(args[j]), 1.0 if j >= 3 else 0.0)
        up[j] = args[j] + step; dn[j] = args[j] - step
        su = po.forward(up[0], up[1], up[2], P, flag, r=up[3], q=up[4])[0]
        sd = po.forward(dn[0], dn[1], dn[2], P, flag, r=dn[3], q=dn[4])[0]
        fd = (su - sd) / (2 * step)
        err = np.abs(fd - gin[j]) / np.maximum(np.abs(gin[j]), 1e-3 * np.abs(s0 / args[j]) if j < 3 else 1e-3)
        assert np.median(err) <= 1e-6 and np.quantile(err, 0.99) <= 1e-4, (j, np.median(err), np.quantile(err, 0.99))


def test_input_gradient_gate_follows_grad_P():
    """Off-gate / invalid rows give exactly +0 in every component, in both modes; on-gate rows scale with -grad_P."""
    S, K, tau, r, q, sig, flag = _bsm_rows(200, 9)
    P = po.black_price(S, K, tau, sig, flag, r=r, q=q)
    s0, v0, st = po.forward(S, K, tau, P, flag, r=r, q=q)
    st2 = st.copy(); st2[::5] = 1
    gs = np.random.default_rng(1).standard_normal(S.size)
    for mode in (0, 1):
        floor = float(np.median(v0))
        gP = po.backward(gs, v0, st2, floor, mode)
        gin = po.backward_inputs(gs, v0, st2, floor, mode, S, K, tau, s0, flag, r=r, q=q)
        greeks = po.black_greeks(S, K, tau, s0, flag, r=r, q=q, prec=0)
        off = gP == 0
        assert off.sum() > 20 and (~off).sum() > 20
        for j in range(5):
            assert np.array_equal(gin[j][off].view(np.uint64), np.zeros(off.sum()).view(np.uint64))
            assert np.allclose(gin[j][~off], -gP[~off] * greeks[j][~off], rtol=1e-14, atol=0)


def test_lbr_in_the_money_large_moneyness_against_truth():
    """In-the-money rows at |x| up to 12: the time value must not inherit the rounding of F - K (reading 18).
    With tv = B - fl(F - K) the oracle sat 1e-11 away from the __float128 bisection of the literal price here."""
    rng = np.random.default_rng(321)
    n = 600
    x = rng.choice([-1.0, 1.0], n) * rng.uniform(3.0, 12.0, n)
    F = np.exp(rng.uniform(np.log(0.5), np.log(5e3), n)); K = F * np.exp(-x)
    T = np.exp(rng.uniform(np.log(0.05), np.log(20), n))
    s = rng.uniform(0.5, 1.6, n) * np.sqrt(2 * np.abs(x))
    flag = np.where(K >= F, -1.0, 1.0)   # in the money
    P = po.black_price(F, K, T, s / np.sqrt(T), flag, prec=1)
    sg, vega, st = po.forward(F, K, T, P, flag)
    ok = st == 0
    assert ok.sum() > 500
    tr = po.truth_iv(F[ok], K[ok], T[ok], P[ok], flag[ok])
    # what is left is the rounding of the quoted price itself: eps * P / (time value) relative to the time value,
    # times the elasticity of sigma to the time value (<= ~1 here)
    tvq = P[ok] - np.maximum(np.where(flag[ok] > 0, F[ok] - K[ok], K[ok] - F[ok]), 0)
    rel = np.abs(sg[ok] / tr - 1)
    assert np.all(rel <= 2e-13 + 4 * EPS * np.minimum(F, K)[ok] / tvq), float(rel.max())


# ------------------------------------------------------------------ the two objectives, eq.(11) / eq.(12)
def test_loss_price_closed_forms():
    """eq.(11): with P* = P_model + delta the sums are sum delta^2 and sum |P*| (numpy, independent of the oracle's loop);
    sigma_hat = sigma_true gives exactly 0."""
    S, K, tau, r, q, sig, flag = _bsm_rows(5000, 12)
    pm = po.black_price(S, K, tau, sig, flag, r=r, q=q, prec=1)
    z = po.loss_price(S, K, tau, pm, flag, sig, r=r, q=q)
    assert z[0] <= 1e-20 * np.sum(pm ** 2) and z[2] == S.size
    delta = np.random.default_rng(2).standard_normal(S.size) * 0.01 * pm
    out = po.loss_price(S, K, tau, pm + delta, flag, sig, r=r, q=q)
    assert out[0] == pytest.approx(np.sum(delta ** 2), rel=1e-9)
    assert out[1] == pytest.approx(np.sum(np.abs(pm + delta)), rel=1e-14)
    L = (out[0] / out[2]) / (out[1] / out[2]) ** 2
    assert L == pytest.approx(np.mean((delta / np.mean(np.abs(pm + delta))) ** 2), rel=1e-9)


def test_loss_roundtrip_against_direct_formula():
    """eq.(12): on gate-on rows IV(P_model(sigma_hat)) = sigma_hat, so the sum must equal sum w(V_hat)(sigma_hat - sigma*)^2
    computed without any inversion; gate-off rows use the sentinel P*, whose IV is sigma* itself, and contribute 0."""
    S, K, tau, r, q, sig_star, flag = _bsm_rows(4000, 13)
    Pstar = po.black_price(S, K, tau, sig_star, flag, r=r, q=q, prec=1)
    sstar, _, st0 = po.forward(S, K, tau, Pstar, flag, r=r, q=q)
    keep = (st0 == 0) & (np.abs(sstar / sig_star - 1) < 1e-6)        # rows whose market IV is recoverable
    assert keep.sum() > 3500
    S, K, tau, r, q, sig_star, flag, Pstar, sstar = (a[keep] for a in (S, K, tau, r, q, sig_star, flag, Pstar, sstar))
    sig_hat = sig_star * (1 + 0.05 * np.random.default_rng(3).standard_normal(S.size))
    vh = po.vega_eq14(S, K, tau, sig_hat, r=r, q=q)
    floor = float(np.quantile(vh, 0.3))                 # 30 % of the rows fall off the gate
    out = po.loss_roundtrip(S, K, tau, Pstar, flag, sig_hat, sstar, floor, r=r, q=q)
    w = vh ** 2 / (vh ** 2 + floor ** 2)
    on = vh > floor
    direct = np.sum(w[on] * (sig_hat[on] - sstar[on]) ** 2)
    assert out[2] == S.size
    assert out[0] == pytest.approx(direct, rel=1e-9)
    assert out[1] == pytest.approx(np.sum(w), rel=1e-13)
    # sigma_hat = sigma*: zero
    z = po.loss_roundtrip(S, K, tau, Pstar, flag, sstar, sstar, floor, r=r, q=q)
    assert z[0] <= 1e-24 * S.size


# ------------------------------------------------------- gradients of the objectives: eq.(11), eq.(12), eq.(17)
def test_loss_price_grad_against_central_differences():
    """d/d sigma_hat (P_model - P*)^2 = 2 (P_model - P*) V_hat: central differences of the literal long-double price."""
    S, K, tau, r, q, sig, flag = _bsm_rows(3000, 21)
    rng = np.random.default_rng(4)
    Pstar = po.black_price(S, K, tau, sig, flag, r=r, q=q, prec=1) * (1 + 0.02 * rng.standard_normal(S.size))
    sig_hat = sig * (1 + 0.1 * rng.standard_normal(S.size))
    g = po.loss_price_grad(S, K, tau, Pstar, flag, sig_hat, r=r, q=q)
    h = 1e-6 * sig_hat
    fp = (po.black_price(S, K, tau, sig_hat + h, flag, r=r, q=q, prec=1) - Pstar) ** 2
    fm = (po.black_price(S, K, tau, sig_hat - h, flag, r=r, q=q, prec=1) - Pstar) ** 2
    fd = (fp - fm) / (2 * h)
    f = np.maximum(fp, fm)                                  # rounding of the prices entering the difference quotient:
    noise = 16 * EPS * (f + np.sqrt(f) * np.abs(Pstar)) / h  # d(res^2) = 2 res dP with dP ~ eps P
    assert np.all(np.abs(g - fd) <= 1e-5 * np.abs(g) + noise)
    resolved = np.abs(g) > 100 * noise                        # rows on which the difference quotient resolves the slope
    assert resolved.sum() > 2000 and np.max(np.abs(g[resolved] / fd[resolved] - 1)) < 1e-3
    assert np.count_nonzero(g) > 2900


def test_loss_roundtrip_grad_against_central_differences_and_eq17():
    """eq.(12) per-row term T = w(V_hat)(IV(P~) - sigma*)^2: its gradient (eq.(17) chain 1/V * V_hat on the gate, plus the
    w' V_hat' term; off the gate only the latter) against central differences of the oracle's own term; the sentinel
    carries no gradient; and the eq.(17) cancellation in closed form: on the gate IV(P_model(sigma_hat)) = sigma_hat, so
    the naive composition's gradient 2 (sigma_rt - sigma*) V_hat / V_rt equals 2 (sigma_hat - sigma*)."""
    S, K, tau, r, q, sig_star, flag = _bsm_rows(3000, 22)
    rng = np.random.default_rng(5)
    Pstar = po.black_price(S, K, tau, sig_star, flag, r=r, q=q, prec=1)
    sstar, _, st0 = po.forward(S, K, tau, Pstar, flag, r=r, q=q)
    vh0 = po.vega_eq14(S, K, tau, sig_star, r=r, q=q)
    keep = (st0 == 0) & (np.abs(sstar / sig_star - 1) < 1e-7) & (vh0 > 1e-3 * S)
    S, K, tau, r, q, flag, Pstar, sstar = (a[keep] for a in (S, K, tau, r, q, flag, Pstar, sstar))
    assert S.size > 1500
    sig_hat = sstar * (1 + 0.05 * rng.standard_normal(S.size))
    vh = po.vega_eq14(S, K, tau, sig_hat, r=r, q=q)
    floor = float(np.quantile(vh, 0.3))
    g, term = po.loss_roundtrip_grad(S, K, tau, Pstar, flag, sig_hat, sstar, floor, r=r, q=q)
    h = 1e-6 * sig_hat
    _, tp = po.loss_roundtrip_grad(S, K, tau, Pstar, flag, sig_hat + h, sstar, floor, r=r, q=q)
    _, tm = po.loss_roundtrip_grad(S, K, tau, Pstar, flag, sig_hat - h, sstar, floor, r=r, q=q)
    vp = po.vega_eq14(S, K, tau, sig_hat + h, r=r, q=q); vm = po.vega_eq14(S, K, tau, sig_hat - h, r=r, q=q)
    same_side = ((vp > floor) == (vh > floor)) & ((vm > floor) == (vh > floor))    # the FD stencil must not straddle the gate
    fd = (tp - tm) / (2 * h)
    scale = np.abs(g) + 1e-7 * (np.abs(term) / np.abs(h) + 1e-12)
    err = np.abs(g - fd)[same_side] / scale[same_side]
    assert same_side.sum() > 0.95 * S.size and err.max() < 2e-4, float(err.max())
    on = vh > floor
    assert on.sum() > 100 and (~on).sum() > 100
    # off the gate the sentinel carries no gradient: only the w' term, tiny because IV(P*) = sigma*
    assert np.max(np.abs(g[~on])) <= 1e-12 * np.max(np.abs(g[on]))
    # loss sums agree with the per-row terms
    sums = po.loss_roundtrip(S, K, tau, Pstar, flag, sig_hat, sstar, floor, r=r, q=q)
    assert sums[0] == pytest.approx(term.sum(), rel=1e-12)
    # eq.(17): 1/V * V = 1 on the well-conditioned rows
    gn, tn = po.loss_roundtrip_grad(S, K, tau, Pstar, flag, sig_hat, sstar, 1e-14, naive=True, r=r, q=q)
    assert np.max(np.abs(gn / (2 * (sig_hat - sstar)) - 1)) < 1e-9
    assert np.all(np.abs(tn - (sig_hat - sstar) ** 2) <= 1e-9 * (sig_hat - sstar) ** 2 + 1e-11 * sstar * np.abs(sig_hat - sstar))


def test_naive_roundtrip_gradient_follows_the_strict_contract():
    """without the gate the inverse channel returns NaN wherever |V_rt| <= 1e-14 or the inversion is
    not OK (unless the cotangent is exactly 0); with the gate every gradient is finite."""
    rng = np.random.default_rng(6)
    n = 4000
    F = np.full(n, 100.0); k = rng.uniform(-2.5, 2.5, n); K = F * np.exp(k)
    tau = np.exp(rng.uniform(np.log(1e-8), np.log(10 ** -0.5), n))
    sig_star = rng.uniform(0.1, 0.6, n)
    flag = np.where(K >= F, 1.0, -1.0)
    Pstar = po.black_price(F, K, tau, sig_star, flag, prec=1)
    sstar = np.where(np.isfinite(sig_star), sig_star, 0.0)
    sig_hat = np.full(n, 0.3)
    vrt = po.vega_eq14(F, K, tau, sig_hat)
    gn, tn = po.loss_roundtrip_grad(F, K, tau, Pstar, flag, sig_hat, sstar, 1e-14, naive=True)
    gg, tg = po.loss_roundtrip_grad(F, K, tau, Pstar, flag, sig_hat, sstar, 1e-6, naive=False)
    assert np.isfinite(gg).all() and np.isfinite(tg).all()
    dead = vrt <= 1e-14
    assert dead.mean() > 0.8
    assert np.isnan(gn[dead]).all()                       # sigma_hat != sigma*: the cotangent is not zero
    alive = vrt > 1e-10
    assert np.isfinite(gn[alive]).all()
