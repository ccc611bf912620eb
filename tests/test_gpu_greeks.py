"""GPU parity (-m gpu) of the "next" rows SURVEY.md 8(f1)/(f2): pivot_iv_black_price and pivot_iv_backward_inputs
against the CPU oracle on the same seeded inputs, element by element."""
import numpy as np
import pytest
import torch

import workloads as wl
import paper_2606_17065_b200 as pv
from oracle import pyoracle as po
from tests.parity_util import KEYS, to_device, to_numpy

pytestmark = pytest.mark.gpu
EPS = np.finfo(np.float64).eps


def _expo(c, sigma):
    """h^2 + s^2/4 + |h|/s: what amplifies rounding in exp(-E), E = (h^2 + t^2)/2.  The first two terms are the vega
    tolerance of tests/parity_util.py (relative error of s); |h|/s is the effect of a one-ulp change of x = ln(F/K)
    (dE = h dx / s), which the two sides do incur: the forward F = S exp((r - q) tau) is rounded differently."""
    F = c["SorF"] * np.exp((c["r"] - c["q"]) * c["tau"]) if c.get("r") is not None else c["SorF"]
    s = sigma * np.sqrt(c["tau"])
    with np.errstate(divide="ignore", invalid="ignore"):
        h = np.log(np.minimum(F, c["K"]) / np.maximum(F, c["K"])) / s
    return np.nan_to_num(h * h + 0.25 * s * s + np.abs(h) / s, nan=0.0, posinf=0.0)


@pytest.mark.parametrize("cfgname", ["config0", "config2"])
def test_black_price_matches_oracle(cfgname):
    """Price and vega of a given sigma (eq.(2)/(3), eq.(14)); includes sigma = 0 (intrinsic) and NaN sigma rows."""
    cfg = wl.config0(200_003, seed=21) if cfgname == "config0" else wl.config2(days=12, seed=22)
    d, c = to_device(cfg), to_numpy(cfg)
    n = c["K"].size
    sig = c["sigma_true"].copy() if "sigma_true" in c and c["sigma_true"] is not None else np.random.default_rng(3).uniform(0.05, 1.0, n)
    sig[::1001] = 0.0
    sig[5::2003] = np.nan
    sg = torch.from_numpy(sig).cuda()
    price, vega = pv.pivot_iv_black_price(d["SorF"], d["K"], d["tau"], sg, d["flag"], r=d.get("r"), q=d.get("q"))
    price, vega = price.cpu().numpy(), vega.cpu().numpy()
    ok = np.isfinite(sig)
    assert np.isnan(price[~ok]).all() and np.isnan(vega[~ok]).all()
    sig_or = np.where(ok, sig, 0.1)
    ref = po.black_price(c["SorF"], c["K"], c["tau"], sig_or, c["flag"], r=c.get("r"), q=c.get("q"), prec=1)
    vref = po.vega_eq14(c["SorF"], c["K"], c["tau"], np.where(sig_or > 0, sig_or, 0.1), r=c.get("r"), q=c.get("q"))
    tol = 1e-12 + 16 * EPS * _expo(c, sig_or)
    F = c["SorF"] * np.exp((c["r"] - c["q"]) * c["tau"]) if c.get("r") is not None else c["SorF"]
    scale = np.maximum(np.abs(ref), 1e-300)
    assert np.all(np.abs(price[ok] - ref[ok]) <= tol[ok] * scale[ok]), float(np.max(np.abs(price[ok] - ref[ok]) / scale[ok]))
    pos = ok & (sig > 0)
    assert np.all(np.abs(vega[pos] - vref[pos]) <= tol[pos] * vref[pos] + 1e-300)   # subnormal vegas: absolute slack
    z = ok & (sig == 0)
    assert z.sum() > 50 and np.all(vega[z] == 0)
    D = np.exp(-c["r"] * c["tau"]) if c.get("r") is not None else 1.0
    intr = np.maximum(np.where(c["flag"] > 0, F - c["K"], c["K"] - F), 0.0) * D
    assert np.allclose(price[z], intr[z], rtol=1e-15, atol=0)


def test_price_round_trip_through_the_gpu_path():
    """P -> pivot_iv_forward -> sigma -> pivot_iv_black_price reproduces P to 1e-13 relative on solved rows (the round
    trip of eq.(12); PAPER.md:385 reports Q50 1.1e-13 on SPX)."""
    cfg = wl.config0(300_000, seed=23, invalid_frac=0.0)
    d = to_device(cfg)
    sig, vega, st = pv.pivot_iv_forward(*[d[k] for k in KEYS])
    ok = st == 0
    price, _ = pv.pivot_iv_black_price(d["SorF"], d["K"], d["tau"], torch.where(ok, sig, torch.zeros_like(sig)), d["flag"])
    rel = (price[ok] / d["P"][ok] - 1).abs()
    assert ok.sum().item() > 200_000
    # sigma is known to ~eps relative, which moves the price by (vega sigma / P) eps: the 1e-13 bar applies where that
    # elasticity is <= 100 and scales with it beyond (same rule as the oracle's own round-trip pin)
    elast = (vega[ok] * sig[ok] / d["P"][ok])
    assert rel[elast <= 100].max().item() <= 1e-13, rel[elast <= 100].max().item()
    # beyond it: the two fixed Householder steps leave sigma good to ~1e-14 relative (measured max 1.2e-14 vs the oracle)
    assert (rel / elast.clamp(min=1.0)).max().item() <= 5e-14


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("bsm", [False, True])
def test_backward_inputs_matches_oracle(mode, bsm):
    cfg = wl.config2(days=10, seed=31) if bsm else wl.config3(1 << 18, seed=32)
    d, c = to_device(cfg), to_numpy(cfg)
    n = c["K"].size
    sig, vega, st = pv.pivot_iv_forward(*[d[k] for k in KEYS], r=d.get("r"), q=d.get("q"))
    gs = torch.randn(n, dtype=torch.float64, device="cuda", generator=torch.Generator(device="cuda").manual_seed(5))
    floor = 1e-8
    outs = pv.pivot_iv_backward_inputs(d["SorF"], d["K"], d["tau"], d["flag"], sig, vega, st, gs, floor, mode,
                                       r=d.get("r"), q=d.get("q"))
    gP_ref_gpu = pv.pivot_iv_backward(gs, vega, st, floor, mode)
    assert torch.equal(outs[0], gP_ref_gpu), "grad_P must be bit-identical to pivot_iv_backward"
    assert (outs[4] is None) == (not bsm) and (outs[5] is None) == (not bsm)
    g = [o.cpu().numpy() if o is not None else None for o in outs]
    sig_h, vega_h, st_h, gs_h = sig.cpu().numpy(), vega.cpu().numpy(), st.cpu().numpy(), gs.cpu().numpy()
    # oracle on the GPU's own sigma / vega (the forward's parity is tested elsewhere)
    sig_in = np.where(st_h == 0, sig_h, 0.1)
    ref = po.backward_inputs(gs_h, vega_h, st_h, floor, mode, c["SorF"], c["K"], c["tau"], sig_in, c["flag"],
                             r=c.get("r"), q=c.get("q"))
    gPh = g[0]
    off = gPh == 0
    greeks = po.black_greeks(c["SorF"], c["K"], c["tau"], sig_in, c["flag"], r=c.get("r"), q=c.get("q"), prec=1)
    tolrow = 1e-12 + 64 * EPS * _expo(c, sig_in)
    # scale of each component: |grad_P| times the largest term of the derivative (dtau is a sum of terms that may cancel)
    S, K, tau = c["SorF"], c["K"], c["tau"]
    rr = c["r"] if bsm else np.zeros(n); qq = c["q"] if bsm else np.zeros(n)
    term_tau = np.abs(qq * S * greeks[0]) + np.abs(rr * K * greeks[1]) + np.abs(vega_h * sig_in / (2 * tau))
    scales = [np.abs(greeks[0]), np.abs(greeks[1]), term_tau, np.abs(greeks[3]), np.abs(greeks[4])]
    for j in range(5):
        if g[j + 1] is None:
            continue
        got, want = g[j + 1], ref[j]
        assert np.array_equal(got[off].view(np.uint64), np.zeros(off.sum()).view(np.uint64)), f"component {j}: off-gate rows must be +0.0"
        on = ~off
        err = np.abs(got[on] - want[on])
        bound = tolrow[on] * np.maximum(np.abs(want[on]), np.abs(gPh[on]) * scales[j][on])
        assert np.all(err <= bound + 1e-300), (j, float(np.max(err / (bound + 1e-300))))
    assert (~off).sum() > 0.5 * n


def test_strict_gate_mode_matches_oracle():
    """on the gate the exact gradient, off the gate +0 iff the upstream cotangent is
    0 else NaN -- in pivot_iv_backward and in every component of pivot_iv_backward_inputs, bit for bit vs the oracle."""
    cfg = wl.config3(1 << 18, seed=41)
    d, c = to_device(cfg), to_numpy(cfg)
    n = c["K"].size
    sig, vega, st = pv.pivot_iv_forward(*[d[k] for k in KEYS])
    gs = torch.randn(n, dtype=torch.float64, device="cuda", generator=torch.Generator(device="cuda").manual_seed(6))
    gs[::3] = 0.0
    gs[1::97] = float("nan")
    floor = 1e-14
    gP = pv.pivot_iv_backward(gs, vega, st, floor, pv.GATE_STRICT).cpu().numpy()
    vega_h, st_h, gs_h = vega.cpu().numpy(), st.cpu().numpy(), gs.cpu().numpy()
    ref = po.backward(gs_h, vega_h, st_h, floor, 2)
    assert np.array_equal(np.isnan(gP), np.isnan(ref))
    fin = ~np.isnan(ref)
    assert np.array_equal(gP[fin].view(np.uint64), ref[fin].view(np.uint64))
    off = ~((st_h == 0) & (np.abs(vega_h) > floor))
    assert off.sum() > 1000 and np.isnan(gP[off & (gs_h != 0)]).all() and np.all(gP[off & (gs_h == 0)] == 0)
    outs = pv.pivot_iv_backward_inputs(d["SorF"], d["K"], d["tau"], d["flag"], sig, vega, st, gs, floor, pv.GATE_STRICT)
    assert np.array_equal(outs[0].cpu().numpy().view(np.uint64)[fin], ref.view(np.uint64)[fin])
    for j in (1, 2, 3):
        g = outs[j].cpu().numpy()
        assert np.isnan(g[off & (gs_h != 0)]).all() and np.all(g[off & (gs_h == 0)] == 0)
        on = ~off & np.isfinite(gs_h)
        assert np.isfinite(g[on]).all()


@pytest.mark.parametrize("bsm", [False, True])
def test_losses_match_oracle(bsm):
    """the sums of eq.(11) and eq.(12) against the oracle's plain loops (different summation order:
    tolerance 1e-11 relative), including gate-off rows (sentinel price) and rows that are skipped."""
    cfg = wl.config2(days=6, seed=51) if bsm else wl.config0(200_000, seed=52)
    d, c = to_device(cfg), to_numpy(cfg)
    n = c["K"].size
    rq = dict(r=d.get("r"), q=d.get("q"))
    rqh = dict(r=c.get("r"), q=c.get("q"))
    sstar, vstar, st = pv.pivot_iv_forward(*[d[k] for k in KEYS], **rq)
    sstar_h = sstar.cpu().numpy()
    rng = np.random.default_rng(7)
    base = np.where(np.isfinite(sstar_h) & (sstar_h > 0), sstar_h, 0.3)
    sig_hat = base * (1 + 0.05 * rng.standard_normal(n))
    sig_hat[::997] = np.nan                                   # skipped rows
    sh = torch.from_numpy(sig_hat).cuda()
    vh = pv.pivot_iv_black_price(d["SorF"], d["K"], d["tau"], torch.nan_to_num(sh, nan=0.3), d["flag"], **rq)[1]
    floor = float(torch.quantile(vh[torch.isfinite(vh)][:1_000_000], 0.3).item())
    got_p = pv.pivot_iv_loss_price(d["SorF"], d["K"], d["tau"], d["P"], d["flag"], sh, **rq).cpu().numpy()
    ref_p = po.loss_price(c["SorF"], c["K"], c["tau"], c["P"], c["flag"], sig_hat, **rqh)
    assert got_p[2] == ref_p[2] and 0 < ref_p[2] < n
    assert got_p[0] == pytest.approx(ref_p[0], rel=1e-11) and got_p[1] == pytest.approx(ref_p[1], rel=1e-12)
    got_r = pv.pivot_iv_loss_roundtrip(d["SorF"], d["K"], d["tau"], d["P"], d["flag"], sh, sstar, floor, **rq).cpu().numpy()
    ref_r = po.loss_roundtrip(c["SorF"], c["K"], c["tau"], c["P"], c["flag"], sig_hat, sstar_h, floor, **rqh)
    assert abs(got_r[2] - ref_r[2]) <= 2 and ref_r[2] > 0.5 * n      # a row at a status boundary may differ
    assert got_r[1] == pytest.approx(ref_r[1], rel=1e-9)
    assert got_r[0] == pytest.approx(ref_r[0], rel=1e-9)
    # sigma_hat = sigma*: the round-trip loss vanishes (every row inverts back to sigma* or uses the sentinel)
    zero = pv.pivot_iv_loss_roundtrip(d["SorF"], d["K"], d["tau"], d["P"], d["flag"], sstar, sstar, floor, **rq).cpu().numpy()
    assert zero[0] <= 1e-22 * max(zero[2], 1.0)


# ------------------------------------------------------------------ gradients of the objectives; eq.(17); the diagnostic
@pytest.mark.parametrize("bsm", [False, True])
def test_loss_gradients_match_oracle(bsm):
    """pivot_iv_loss_price / pivot_iv_loss_roundtrip with grad_scale: the per-row gradients with respect to sigma_hat against the
    oracle's plain loops (pinned by finite differences in tests/test_oracle_pins.py), gated and naive, including the NaN mask of
    the naive composition bit for bit, and the sums of the fused round trip against the oracle's."""
    cfg = wl.config2(days=5, seed=61) if bsm else wl.config3(150_000, seed=62)
    d, c = to_device(cfg), to_numpy(cfg)
    n = c["K"].size
    rq = dict(r=d.get("r"), q=d.get("q")); rqh = dict(r=c.get("r"), q=c.get("q"))
    sstar, vstar, st = pv.pivot_iv_forward(*[d[k] for k in KEYS], **rq)
    sstar_h = sstar.cpu().numpy()
    rng = np.random.default_rng(8)
    base = np.where(np.isfinite(sstar_h) & (sstar_h > 0), sstar_h, 0.3)
    sig_hat = base * (1 + 0.05 * rng.standard_normal(n))
    sig_hat[::991] = np.nan
    sstar_h = np.where(np.isfinite(sstar_h), sstar_h, 0.25)
    sh, ss = torch.from_numpy(sig_hat).cuda(), torch.from_numpy(sstar_h).cuda()
    a = [d[k] for k in ("SorF", "K", "tau", "P", "flag")]
    ah = [c[k] for k in ("SorF", "K", "tau", "P", "flag")]
    scale = 0.37
    # eq.(11)
    sums, g = pv.pivot_iv_loss_price(*a, sh, grad_scale=scale, **rq)
    ref = scale * po.loss_price_grad(*ah, sig_hat, **rqh)
    g = g.cpu().numpy()
    vh = po.vega_eq14(c["SorF"], c["K"], c["tau"], np.nan_to_num(sig_hat, nan=0.3), **rqh)
    assert np.array_equal(g == 0, ref == 0) or np.mean((g == 0) != (ref == 0)) < 1e-4
    Fh = c["SorF"] * (np.exp((c["r"] - c["q"]) * c["tau"]) if bsm else 1.0)
    s_hat = np.nan_to_num(sig_hat, nan=0.3) * np.sqrt(c["tau"])
    expo = (np.log(Fh / c["K"]) / s_hat) ** 2 + 0.25 * s_hat ** 2       # vega = C exp(-expo/2): its own tolerance (parity_util)
    hos = np.abs(np.log(Fh / c["K"])) / s_hat ** 2                      # |h|/s: one ulp of x = ln(F/K) in the exponent
    tol = (1e-11 + 32 * EPS * expo) * np.abs(ref) + \
        scale * 2 * vh * np.abs(c["P"]) * (1e-12 + 32 * EPS * (expo + hos))   # + the price tolerance on the cancelling residual
    assert np.all(np.abs(g - ref) <= tol + 1e-300)
    # eq.(12), gated
    floor = float(np.quantile(vh[np.isfinite(vh)], 0.3))
    sums_r, gr = pv.pivot_iv_loss_roundtrip(*a, sh, ss, floor, mode=pv.RT_GATED, grad_scale=scale, **rq)
    ref_g, term = po.loss_roundtrip_grad(*ah, sig_hat, sstar_h, floor, naive=False, **rqh)
    ref_sums = po.loss_roundtrip(*ah, sig_hat, sstar_h, floor, **rqh)
    sums_r = sums_r.cpu().numpy()
    assert abs(sums_r[2] - ref_sums[2]) <= 2 and sums_r[0] == pytest.approx(ref_sums[0], rel=1e-9)
    assert sums_r[1] == pytest.approx(ref_sums[1], rel=1e-9)
    gr = gr.cpu().numpy()
    assert np.isfinite(gr).all()
    big = np.abs(ref_g) > 1e-6 * np.max(np.abs(ref_g))
    assert np.max(np.abs(gr[big] / (scale * ref_g[big]) - 1)) < 1e-8
    assert np.max(np.abs(gr - scale * ref_g)) <= 1e-8 * np.max(np.abs(scale * ref_g))
    # naive composition at the strict floor 1e-14: same NaN mask, same finite values
    sums_n, gn = pv.pivot_iv_loss_roundtrip(*a, sh, ss, 1e-14, mode=pv.RT_NAIVE, grad_scale=scale, **rq)
    ref_n, term_n = po.loss_roundtrip_grad(*ah, sig_hat, sstar_h, 1e-14, naive=True, **rqh)
    gn = gn.cpu().numpy()
    # the NaN mask hangs on exact ties (a cotangent of exactly 0, a time value of exactly 0, |V_rt| against 1e-14): identical up to
    # the rows where the two sides round such a tie differently
    assert np.mean(np.isnan(gn) != np.isnan(ref_n)) < 2e-3 and np.isnan(ref_n).sum() > 0
    fin = np.isfinite(ref_n) & np.isfinite(gn) & (np.abs(ref_n) > 1e-6 * np.nanmax(np.abs(ref_n)))
    v_rt = po.vega_eq14(c["SorF"], c["K"], c["tau"], np.nan_to_num(sig_hat, nan=0.3), **rqh)
    well = fin & (v_rt > 1e-8 * c["K"])
    assert np.max(np.abs(gn[well] / (scale * ref_n[well]) - 1)) < 1e-8
    # eq.(17): on well-conditioned rows the composed factor (1/V_rt) V_hat is 1: the naive gradient is 2 (sigma_hat - sigma*)
    # (where the price -> sigma -> price round trip itself is well conditioned: elasticity P / (V sigma) <= 100)
    cond = well & (np.abs(c["P"]) <= 100 * v_rt * np.nan_to_num(sig_hat, nan=1.0)) & (np.abs(sig_hat - sstar_h) > 1e-3 * sstar_h)
    assert cond.sum() > 0.2 * n
    assert np.max(np.abs(gn[cond] / (scale * 2 * (sig_hat[cond] - sstar_h[cond])) - 1)) < 1e-9
    assert np.isnan(sums_n[0].item())                     # the NaN sigma_hat rows poison the naive sum


@pytest.mark.parametrize("bsm", [False, True])
def test_roundtrip_ragged_sizes_and_row_independence(bsm):
    """The fused round trip walks 32-row blocks per warp and solves from a per-warp stack: sizes around the block and the stack
    capacity (empty, 1, 31 ... 97 rows, a ragged tail, one size that wraps the grid-stride loop) must give, row for row, the
    bits of the full-size call (a row's arithmetic does not depend on where it sits in a stack), and sums that match the
    oracle's on the same slice; mixed rows (config 4: most rows never reach the solver) and BSM chains (all do)."""
    cfg = wl.config2(days=1, expiries=4, strikes=2000, seed=71) if bsm else wl.config4(1_300_000, seed=72)
    d, c = to_device(cfg), to_numpy(cfg)
    n = c["K"].size
    names = ("SorF", "K", "tau", "P", "flag") + (("r", "q") if bsm else ())
    sstar, _, _ = pv.pivot_iv_forward(*[d[k] for k in KEYS], r=d.get("r"), q=d.get("q"))
    sstar_h = np.where(np.isfinite(sstar.cpu().numpy()), sstar.cpu().numpy(), 0.25)
    rng = np.random.default_rng(9)
    sig_hat = np.where(sstar_h > 0, sstar_h, 0.3) * (1 + 0.05 * rng.standard_normal(n))
    sig_hat[::613] = np.nan
    sh, ss = torch.from_numpy(sig_hat).cuda(), torch.from_numpy(sstar_h).cuda()
    floor = 1e-6

    def call(m, mode):
        a = [d[k][:m] for k in names[:5]]
        rq = dict(r=d["r"][:m], q=d["q"][:m]) if bsm else {}
        sums, g = pv.pivot_iv_loss_roundtrip(*a, sh[:m], ss[:m], floor, mode=mode, grad_scale=0.5, **rq)
        return sums.cpu().numpy(), g.cpu().numpy()

    for mode in (pv.RT_GATED, pv.RT_NAIVE):
        sums_full, g_full = call(n, mode)
        assert g_full.shape == (n,)
        for m in (0, 1, 31, 32, 33, 63, 64, 65, 97, 1000, 8191, 300_001):
            m = min(m, n)
            sums, g = call(m, mode)
            assert g.shape == (m,)
            assert np.array_equal(g.view(np.int64), g_full[:m].view(np.int64)), (mode, m)
            if mode == pv.RT_GATED and 0 < m <= 8191:
                ah = [c[k][:m] for k in names[:5]]
                rqh = dict(r=c["r"][:m], q=c["q"][:m]) if bsm else {}
                ref = po.loss_roundtrip(*ah, sig_hat[:m], sstar_h[:m], floor, **rqh)
                assert abs(sums[2] - ref[2]) <= 1
                if sums[2] == ref[2]:
                    assert sums[1] == pytest.approx(ref[1], rel=1e-9, abs=1e-300)
                    assert sums[0] == pytest.approx(ref[0], rel=1e-8, abs=1e-300)
            if m == 0:
                assert (sums == 0).all()


def test_roundtrip_matches_the_composition_of_the_public_calls_at_scale():
    """4,194,304 mixed rows (more than the oracle does in seconds): the fused round-trip kernel against the same objective
    composed from the separately tested calls -- pivot_iv_black_price (price node, V_hat), pivot_iv_forward on P~ (the tile
    kernel; the fused kernel solves from its per-warp stack) and plain torch fp64 for the weights: same rows used, sums to
    1e-11, every gradient entry to 1e-9 of its own size (+ 1e-12 of the largest), nothing but +0 on the rows the sum skips."""
    n = 1 << 22
    cfg = wl.config4(n, seed=81, device="cuda")
    a = [cfg[k] for k in ("SorF", "K", "tau", "P", "flag")]
    F, K, tau, Pstar, flag = a
    sstar, _, st0 = pv.pivot_iv_forward(*a)
    g0 = torch.Generator(device="cuda").manual_seed(3)
    base = torch.where((st0 == 0) & (sstar > 0), sstar, torch.full_like(sstar, 0.3))
    sh = base * (1 + 0.05 * torch.randn(n, generator=g0, device="cuda", dtype=torch.float64))
    sh[::1009] = float("nan")
    ss = torch.where(torch.isfinite(sstar), sstar, torch.full_like(sstar, 0.25))
    floor, scale = 1e-6, 0.5
    sums, g = pv.pivot_iv_loss_roundtrip(*a, sh, ss, floor, mode=pv.RT_GATED, grad_scale=scale)
    pm, vh = pv.pivot_iv_black_price(F, K, tau, sh, flag)
    usable = torch.isfinite(pm) & torch.isfinite(vh) & torch.isfinite(ss)
    on = vh.abs() > floor
    Pt = torch.where(usable & on, pm, Pstar)
    srt, vrt, st = pv.pivot_iv_forward(F, K, tau, Pt, flag)
    ok = usable & (st == 0)
    f2 = floor * floor
    v2 = vh * vh
    den = v2 + f2
    w = v2 / den
    d = srt - ss
    z = torch.zeros_like(d)
    ref_sums = torch.stack([torch.where(ok, w * d * d, z).sum(), torch.where(ok, w, z).sum(), ok.double().sum()])
    assert sums[2].item() == ref_sums[2].item() and 0.3 * n < ref_sums[2].item() < n
    assert sums[0].item() == pytest.approx(ref_sums[0].item(), rel=1e-11)
    assert sums[1].item() == pytest.approx(ref_sums[1].item(), rel=1e-11)
    s_hat = sh * tau.sqrt()
    d1d2 = (torch.log(F / K) / s_hat) ** 2 - 0.25 * s_hat * s_hat
    vomma = torch.where(sh > 0, vh * d1d2 / sh, z)
    wp = torch.where(den > 0, 2.0 * vh * f2 / (den * den), z)
    gi = wp * d * d * vomma + torch.where(on & (vrt.abs() > floor), w * (2.0 * d / vrt) * vh, z)
    ref = torch.where(ok, scale * gi, z)
    assert torch.isfinite(g).all()
    assert (g[~ok] == 0).all() and not torch.signbit(g[~ok]).any()
    err = (g - ref).abs()
    assert (err <= 1e-9 * ref.abs() + 1e-12 * ref.abs().max()).all(), float((err / (ref.abs() + 1e-300)).max())


def test_nan_poisoning_diagnostic():
    """PAPER.md:404-428 (App. B.2, Fig.6): on the low_vega_tail chain (N = 65,536, seed 31, ~91 % of rows |V| <= 1e-14) the
    naive composition poisons every row of the singular set within one Adam step and never recovers; the gated objective
    keeps every row finite for 200 steps and its loss goes down.  The step-0 gradients are checked against the oracle."""
    from paper_2606_17065_b200.diagnostic import run_nan_poisoning_diagnostic
    cfg = wl.low_vega_tail()
    d, c = to_device(cfg), to_numpy(cfg)
    n = c["K"].size
    a = [d[k] for k in ("SorF", "K", "tau", "P", "flag")]
    ah = [c[k] for k in ("SorF", "K", "tau", "P", "flag")]
    sigma_star = d["sigma_true"]
    vstar = pv.pivot_iv_black_price(d["SorF"], d["K"], d["tau"], sigma_star, d["flag"])[1]
    dead = float((vstar <= 1e-14).double().mean().item())
    assert 0.89 <= dead <= 0.94, dead                      # the paper: 0.911
    g0 = torch.Generator(device="cuda").manual_seed(7)
    sigma_init = (sigma_star * (1 + 0.2 * torch.randn(n, generator=g0, device="cuda", dtype=torch.float64))).clamp_min(0.02)
    # step-0 gradients against the oracle
    si_h, ss_h = sigma_init.cpu().numpy(), c["sigma_true"]
    _, gn = pv.pivot_iv_loss_roundtrip(*a, sigma_init, sigma_star, 1e-14, mode=pv.RT_NAIVE, grad_scale=1.0)
    rn, _ = po.loss_roundtrip_grad(*ah, si_h, ss_h, 1e-14, naive=True)
    gn = gn.cpu().numpy()
    assert np.mean(np.isnan(gn) != np.isnan(rn)) < 1e-3 and np.isnan(rn).mean() > 0.8
    f = np.isfinite(rn) & np.isfinite(gn) & (np.abs(rn) > 1e-9)
    assert np.max(np.abs(gn[f] / rn[f] - 1)) < 1e-7
    _, gg = pv.pivot_iv_loss_roundtrip(*a, sigma_init, sigma_star, 1e-6, mode=pv.RT_GATED, grad_scale=1.0)
    rg, _ = po.loss_roundtrip_grad(*ah, si_h, ss_h, 1e-6, naive=False)
    gg = gg.cpu().numpy()
    assert np.isfinite(gg).all() and np.max(np.abs(gg - rg)) <= 1e-7 * np.max(np.abs(rg))
    naive = run_nan_poisoning_diagnostic(d, sigma_star, sigma_init, gated=False, steps=200)
    gated = run_nan_poisoning_diagnostic(d, sigma_star, sigma_init, gated=True, steps=200)
    # naive: NaN gradients at step 0, the poisoned rows are gone after one step and stay gone, the loss is NaN from step 1 on
    assert naive["nan_grads"][0] > 0.8 * n
    assert naive["finite_frac"][0] == 1.0 and naive["finite_frac"][1] < 0.2 and naive["finite_frac"][-1] <= naive["finite_frac"][1]
    assert all(np.isnan(x) for x in naive["loss"][1:])
    # gated: every row finite at every step, no NaN gradient, loss goes down
    assert all(f == 1.0 for f in gated["finite_frac"]) and all(k == 0 for k in gated["nan_grads"])
    assert all(np.isfinite(x) for x in gated["loss"]) and gated["loss"][-1] < 0.5 * gated["loss"][0]
    up = sum(1 for i in range(1, 200) if gated["loss"][i] > gated["loss"][i - 1])
    print(f"dead fraction {dead:.3f}; naive finite after 1 step {naive['finite_frac'][1]:.3f}; gated loss "
          f"{gated['loss'][0]:.3e} -> {gated['loss'][-1]:.3e} ({up} increasing steps of 199)")
