"""-m gpu: the device math library of csrc/lbr_device.cuh, function by function, against mpmath at 40 digits ON THE DEVICE
(pivot_iv_debug_math): the errors DESIGN.md section 5 quotes are measured here, FMA contraction, MUFU seeds and the range
branches included, not taken from the coefficient fit."""
import mpmath as mp
import numpy as np
import pytest
import torch

import paper_2606_17065_b200 as pv

pytestmark = pytest.mark.gpu
mp.mp.dps = 40
EPS = 2.0 ** -52


def _run(fn, a, b=None):
    ta = torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()
    tb = None if b is None else torch.from_numpy(np.ascontiguousarray(b, dtype=np.float64)).cuda()
    return pv.pivot_iv_debug_math(fn, ta, tb).cpu().numpy()


def _relerr(got, ref_mp):
    """max |got/ref - 1| with ref in mpmath (got is exact as a double)."""
    worst = mp.mpf(0)
    for g, r in zip(got, ref_mp):
        if r == 0:
            assert g == 0.0
            continue
        e = abs(mp.mpf(float(g)) / r - 1)
        worst = max(worst, e)
    return float(worst)


def _erfcx(z):
    z = mp.mpf(float(z))
    return mp.exp(z * z) * mp.erfc(z)


def _lu(rng, lo, hi, n):
    return np.exp(rng.uniform(np.log(lo), np.log(hi), n))


def test_erfcx_fp64_and_seed():
    rng = np.random.default_rng(1)
    z = np.concatenate([[0.0, 1e-300, 1e-17, 0.5, 1.0, 4.0, 26.0, 1e3, 1e8, -0.0708, -0.05, -1e-9], rng.uniform(0, 8, 1500),
                        _lu(rng, 1e-6, 1e3, 1500), rng.uniform(-0.0708, 0, 200)])
    ref = [_erfcx(v) for v in z]
    e_one = _relerr(_run("erfcx_one", z), ref)
    z2 = z[::-1].copy()
    e_p1 = _relerr(_run("erfcx_pair_1", z, z2), ref)
    e_p2 = _relerr(_run("erfcx_pair_2", z2, z), ref)
    e_seed = _relerr(_run("erfcx_seed", z), ref)
    print(f"erfcx_one {e_one:.2e}  pair {max(e_p1, e_p2):.2e}  seed {e_seed:.2e}")
    assert e_one <= 8 * EPS and e_p1 <= 8 * EPS and e_p2 <= 8 * EPS      # fit error 5.7e-16 + evaluation rounding
    assert e_seed <= 6e-7


def test_erfcx_divided_difference_forms():
    """erfcx(z1) -/+ erfcx(z1 + d) from the divided difference of the fitted polynomial (lbr_device.cuh: erfcx_dd): the
    difference keeps its RELATIVE accuracy however small the gap d is (it replaced the small-t Taylor series of W)."""
    rng = np.random.default_rng(11)
    n = 4000
    z1 = np.concatenate([rng.uniform(-0.0708, 1, n // 4), rng.uniform(0, 30, n // 4), _lu(rng, 1e-8, 50, n // 4),
                         rng.uniform(-0.0708, 0.0, n // 4)])
    d = _lu(rng, 1e-12, 60, n)
    d[:50] = 0.0
    z2 = z1 + d
    d = z2 - z1                                   # the gap the device sees (exact)
    ref_d = [_erfcx(a) - _erfcx(b) for a, b in zip(z1, z2)]
    ref_s = [_erfcx(a) + _erfcx(b) for a, b in zip(z1, z2)]
    e_d = _relerr(_run("erfcx_dd_diff", z1, d), ref_d)
    e_s = _relerr(_run("erfcx_dd_sum", z1, d), ref_s)
    # the seed-grade form sees float-rounded arguments
    z1f, df = z1.astype(np.float32).astype(np.float64), d.astype(np.float32).astype(np.float64)
    z1f = np.maximum(z1f, -0.0708)
    ref_df = [_erfcx(a) - _erfcx(mp.mpf(float(a)) + mp.mpf(float(g))) for a, g in zip(z1f, df)]
    ref_sf = [_erfcx(a) + _erfcx(mp.mpf(float(a)) + mp.mpf(float(g))) for a, g in zip(z1f, df)]
    e_df = _relerr(_run("erfcx_dd_seed_diff", z1f, df), ref_df)
    e_sf = _relerr(_run("erfcx_dd_seed_sum", z1f, df), ref_sf)
    print(f"erfcx_dd diff {e_d:.2e} sum {e_s:.2e}  seed diff {e_df:.2e} seed sum {e_sf:.2e}")
    assert e_d <= 16 * EPS and e_s <= 8 * EPS
    assert e_df <= 2e-5 and e_sf <= 2e-6


def test_eval_W_against_the_definition():
    """eval_W (the ratio every Householder step is built on) against W = b/b', Wbar = (b_max - b)/b' from the literal
    eq.(4) in mpmath, over small and large t, |h| from 0 to 36, both sides of the difference / sum switch."""
    rng = np.random.default_rng(12)
    n = 3000
    s = _lu(rng, 1e-6, 40, n)
    h = -np.concatenate([rng.uniform(0, 36, n // 2), _lu(rng, 1e-8, 5, n // 2)])
    x = h * s
    x[:20] = 0.0
    keep = (np.abs(x) < 600)
    x, s = x[keep], s[keep]

    def W_ref(xv, sv):
        xv, sv = mp.mpf(float(xv)), mp.mpf(float(sv))
        hh, t = xv / sv, sv / 2
        Phi = lambda z: mp.erfc(-z / mp.sqrt(2)) / 2
        bmax = mp.exp(xv / 2)
        b = bmax * Phi(hh + t) - Phi(hh - t) / bmax
        bp = mp.exp(-(hh * hh + t * t) / 2) / mp.sqrt(2 * mp.pi)
        return b / bp, (bmax - b) / bp

    old = mp.mp.dps
    mp.mp.dps = 400          # b underflows against b_max at 40 digits when |h| is large
    try:
        refs = [W_ref(a, b) for a, b in zip(x, s)]
    finally:
        mp.mp.dps = old
    for name, tol in (("w_full", 3e-14), ("w_seed", 3e-5)):
        got = _run(name, x, s)
        worst = 0.0
        for g, (W, Wb), xv, sv in zip(got, refs, x, s):
            ref = W if g > 0 else -Wb
            worst = max(worst, float(abs(mp.mpf(float(g)) / ref - 1)))
        print(f"{name} max rel err {worst:.2e}")
        assert worst <= tol, name


def test_exp_fast_full_range_and_seed():
    rng = np.random.default_rng(2)
    a = np.concatenate([[0.0, -0.0, 1e-300, -1e-300, 709.7, 709.78, -708.3, -708.5, -745.0, -745.2, -750.0, 710.0, 1e4, -1e4,
                         0.5 * np.log(2.0), -0.5 * np.log(2.0)],
                        rng.uniform(-745.1, 709.78, 3000), rng.uniform(-1, 1, 1000)])
    got = _run("exp_fast", a)
    worst = 0.0
    for x, g in zip(a, got):
        r = mp.exp(mp.mpf(float(x)))
        if x > 709.782712893384:
            assert g == np.inf
        elif r < mp.mpf(2) ** -1074 / 2:
            assert g == 0.0
        elif r < mp.mpf(2) ** -1022:          # subnormal result: absolute error within one subnormal ulp
            assert abs(mp.mpf(float(g)) - r) <= mp.mpf(2) ** -1074
        else:
            worst = max(worst, float(abs(mp.mpf(float(g)) / r - 1)))
    print(f"exp_fast max rel err (normal range) {worst:.2e}")
    assert worst <= 4 * EPS                 # polynomial 1.5e-16 + reduction + evaluation rounding
    b = rng.uniform(-700, 700, 3000)
    e_seed = _relerr(_run("exp_seed", b), [mp.exp(mp.mpf(float(x))) for x in b])
    c = rng.uniform(-87, 87, 2000)
    e_f = _relerr(_run("expf_seed", c), [mp.exp(mp.mpf(float(np.float32(x)))) for x in c])
    print(f"exp_seed {e_seed:.2e}  expf_seed {e_f:.2e}")
    assert e_seed <= 1e-6 and e_f <= 2e-5     # fp32 argument rounding: |a| 6e-8 relative => up to 87 * 6e-8 in the result


def test_log_and_log1p():
    rng = np.random.default_rng(3)
    v = np.concatenate([[1.0, 2.0, 0.5, np.sqrt(2.0), 1 / np.sqrt(2.0), 2.2250738585072014e-308, 1.7976931348623157e308,
                         1 + 2 ** -52, 1 - 2 ** -53], _lu(rng, 1e-307, 1e307, 3000), rng.uniform(0.5, 2.0, 2000)])
    got = _run("log_fast", v)
    worst = 0.0
    for x, g in zip(v, got):
        r = mp.log(mp.mpf(float(x)))
        err = abs(mp.mpf(float(g)) - r)
        worst = max(worst, float(err / max(abs(r), mp.mpf(2) ** -60)))
        assert err <= 2 * EPS * max(abs(r), mp.mpf(1e-16)) + mp.mpf(2) ** -70 or err <= 1.2e-16 * abs(x - 1), (x, g)
    print(f"log_fast max rel err {worst:.2e}")
    q = np.concatenate([[0.0, 1e-300, 1e-17, np.sqrt(2.0) - 1, 0.41421356, 0.41421357, 1.0, 1e10, 1e300],
                        _lu(rng, 1e-20, 1e3, 3000), rng.uniform(0.3, 0.5, 1000)])
    e_l1p = _relerr(_run("log1p_fast", q), [mp.log1p(mp.mpf(float(x))) for x in q])
    print(f"log1p_fast max rel err {e_l1p:.2e}")
    assert e_l1p <= 3 * EPS
    s = np.concatenate([[5e-324, 1e-310], _lu(rng, 1e-300, 1e300, 2000)])
    gs = _run("log_seed", s)
    for x, g in zip(s, gs):
        r = mp.log(mp.mpf(float(x)))
        assert abs(mp.mpf(float(g)) - r) <= 2e-7 * max(1, abs(r)), (x, g)
    f = _lu(rng, 1e-30, 1e30, 2000)
    gf = _run("logf_seed", f)
    for x, g in zip(f, gf):
        r = mp.log(mp.mpf(float(np.float32(x))))
        assert abs(mp.mpf(float(g)) - r) <= 2e-6 * max(1, abs(r)), (x, g)


def test_reciprocal_division_sqrt():
    rng = np.random.default_rng(4)
    x = np.concatenate([_lu(rng, 1e-300, 1e300, 3000), -_lu(rng, 1e-300, 1e300, 500), [1.0, 3.0, 2.0 ** -1000, 2.0 ** 1000]])
    ref = [1 / mp.mpf(float(v)) for v in x]
    e1, e2 = _relerr(_run("rcp_nr1", x), ref), _relerr(_run("rcp_nr2", x), ref)
    e0 = _relerr(_run("rcp_raw", x), ref)
    a = rng.standard_normal(3504) * _lu(rng, 1e-100, 1e100, 3504)
    xb = np.sign(x) * np.exp(np.log(np.abs(x)) * 0.5)          # 1e-150 .. 1e150: the quotient stays in the normal range
    ed = _relerr(_run("div_fast", a, xb), [mp.mpf(float(p)) / mp.mpf(float(q)) for p, q in zip(a, xb)])
    v = np.concatenate([_lu(rng, 2.3e-308, 1e308, 3000), [1.0, 2.0, 4.0, 2.0 ** -800, 2.0 ** 800]])
    rs = [mp.sqrt(mp.mpf(float(t))) for t in v]
    es1, es2 = _relerr(_run("sqrt_nr1", v), rs), _relerr(_run("sqrt_nr2", v), rs)
    er = _relerr(_run("rsqrt_nr2", v), [1 / t for t in rs])
    er3 = _relerr(_run("rsqrt_c3", v), [1 / t for t in rs])
    assert _run("sqrt_nr1", np.array([0.0]))[0] == 0.0
    print(f"rcp_raw {e0:.2e} rcp_nr1 {e1:.2e} rcp_nr2 {e2:.2e} div_fast {ed:.2e} sqrt_nr1 {es1:.2e} sqrt_nr2 {es2:.2e} rsqrt_nr2 {er:.2e} rsqrt_c3 {er3:.2e}")
    assert e0 <= 2.0 ** -19 and e1 <= 1e-11 and e2 <= 2 * EPS and ed <= 1.5 * EPS
    assert es1 <= 1e-11 and es2 <= 1.5 * EPS and er <= 4 * EPS and er3 <= 4 * EPS


def test_ninv_tail():
    rng = np.random.default_rng(5)
    lnp = np.concatenate([[-1.0651, -1.07, -700.0, -50.0], -_lu(rng, 1.0651, 700, 3000)])
    ref = [-mp.sqrt(2) * mp.erfinv(2 * mp.exp(mp.mpf(float(t))) - 1) if t > -30 else None for t in lnp]

    def z_of(t):
        """-Phi^-1(e^t) for very negative t: solve ln Phi(-z) = t by Newton on the erfc form."""
        t = mp.mpf(float(t))
        z = mp.sqrt(-2 * t)
        for _ in range(60):
            f = mp.log(mp.erfc(z / mp.sqrt(2)) / 2) - t
            fp = -mp.exp(-z * z / 2) / mp.sqrt(2 * mp.pi) / (mp.erfc(z / mp.sqrt(2)) / 2)
            z = z - f / fp
        return z
    ref = [z_of(t) for t in lnp]
    es = _relerr(_run("ninv_tail_seed", lnp), ref)
    ef = _relerr(_run("ninv_tail_full", lnp), ref)
    print(f"ninv_tail_seed {es:.2e}  ninv_tail_full {ef:.2e}")
    assert es <= 5e-5 and ef <= 1e-12
