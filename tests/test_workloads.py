"""-m "not gpu": the seeded workload generators are deterministic, have the stated shapes and
class mix, and hold no method arithmetic that the oracle would inherit (they are checked against the oracle)."""
import numpy as np
import torch

from oracle import pyoracle as po
import workloads as wl

KEYS = ("SorF", "K", "tau", "P", "flag")


def _np(cfg):
    return {k: (v.numpy() if isinstance(v, torch.Tensor) else None) for k, v in cfg.items()}


def test_deterministic_and_shapes():
    a, b = wl.config0(4096), wl.config0(4096)
    for k in KEYS:
        assert torch.equal(a[k], b[k]) and a[k].dtype == torch.float64 and a[k].shape == (4096,)
    assert not torch.equal(wl.config0(4096, seed=1)["K"], a["K"])
    c2 = wl.config2(days=2, expiries=3, strikes=5)
    assert c2["SorF"].numel() == 30 and c2["r"] is not None and c2["q"] is not None
    k = c2["K"].view(2, 3, 5); s = c2["SorF"].view(2, 3, 5)
    assert torch.allclose(k[:, :, 0] / s[:, :, 0], torch.full((2, 3), 0.5, dtype=torch.float64))   # strike fastest
    assert torch.all(s[:, :, 0] == s[:, :, 4])


def test_config0_class_mix_under_the_oracle():
    c = _np(wl.config0())
    sig, vega, st = po.forward(*[c[k] for k in KEYS])
    pert = c["perturbed"]
    assert 0.01 < pert.mean() < 0.03
    assert np.all(np.isin(st[pert], (1, 2)))            # perturbed rows are NaN rows, with a margin >> 1 ulp
    assert np.all(np.isin(st[~pert], (0, 4)))
    otm = ((c["flag"] > 0) & (c["K"] >= c["SorF"])) | ((c["flag"] < 0) & (c["K"] <= c["SorF"]))
    m = (st == 0) & otm & (vega > 1.0)
    assert np.max(np.abs(sig[m] / c["sigma_true"][m] - 1)) < 1e-8   # the textbook pricer really prices sigma_true


def test_config1_covers_all_four_zones_and_solve_only_variant():
    c = _np(wl.config1(1 << 17))
    out = po.forward(*[c[k] for k in KEYS], debug=True)
    ok = out[2] == 0
    assert all((out[3][ok] == z).sum() > 500 for z in range(4))
    c = _np(wl.config1(1 << 17, solve_only=True))
    st = po.forward(*[c[k] for k in KEYS])[2]
    assert (st == 0).mean() > 0.6


def test_config3_low_vega_slice_is_valid_but_below_floor():
    c = _np(wl.config3(1 << 16))
    sig, vega, st = po.forward(*[c[k] for k in KEYS])
    low = c["low_vega"]
    assert 0.08 < low.mean() < 0.12
    okl = low & (st == 0)
    assert okl.sum() > 0.3 * low.sum()
    assert (vega[okl] < 1e-8).mean() > 0.9 and (vega[okl] > 0).mean() > 0.5
    assert c["grad_sigma"].shape == sig.shape


def test_config2_bsm_rows_solve():
    c = _np(wl.config2(days=3, expiries=8, strikes=100))
    sig, vega, st = po.forward(*[c[k] for k in KEYS], r=c["r"], q=c["q"])
    assert np.all(np.isin(st, (0, 4))) and (st == 0).mean() > 0.6
    m = (st == 0) & (vega > 10)
    assert np.median(np.abs(sig[m] / c["sigma_true"][m] - 1)) < 5e-3    # 1e-4 relative price noise moves sigma a little
