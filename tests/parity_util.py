"""Shared helpers of the GPU parity tests: run both sides on the same seeded arrays and compare element by element.

Tolerances:
  sigma   : max relative error <= 1e-12 on rows both sides call OK (north_star)
  status  : bit-exact; sigma of non-OK rows bit-exact (canonical NaN / +0); vega of non-OK rows exactly 0
  vega    : relative error <= 1e-12 + 16 eps (h^2+t^2): vega = C exp(-(h^2+t^2)/2) amplifies the (<= few eps) relative
            difference in s by h^2+t^2 and the exponent's own rounding by (h^2+t^2)/2
  grad_P  : relative error <= 1e-12 where the gate is on (north_star); exactly +0.0 elsewhere; rows whose vega is within
            1e-12 relative of the floor are exempt from the gate comparison (north_star)
"""
import numpy as np
import torch

from oracle import pyoracle as po
import paper_2606_17065_b200 as pv

EPS = np.finfo(np.float64).eps
KEYS = ("SorF", "K", "tau", "P", "flag")


def to_device(cfg, device="cuda"):
    return {k: (v.to(device) if isinstance(v, torch.Tensor) else v) for k, v in cfg.items()}


def to_numpy(cfg, idx=None):
    out = {}
    for k, v in cfg.items():
        if isinstance(v, torch.Tensor):
            v = v if idx is None else v[idx]
            out[k] = v.detach().cpu().numpy()
        else:
            out[k] = None
    return out


def gpu_forward(d):
    return pv.pivot_iv_forward(*[d[k] for k in KEYS], r=d.get("r"), q=d.get("q"))


def oracle_forward(c):
    return po.forward(c["SorF"], c["K"], c["tau"], c["P"], c["flag"], r=c.get("r"), q=c.get("q"))


def compare_forward(g, o, c, sigma_tol=1e-12):
    """g = (sigma, vega, status) numpy from the GPU, o = same from the oracle, c = numpy inputs. Returns stats."""
    gs, gv, gst = g
    os_, ov, ost = o
    assert np.array_equal(gst, ost), f"status mismatch on {(gst != ost).sum()} rows"
    bad = ost != 0
    assert np.array_equal(gs[bad].view(np.uint64), os_[bad].view(np.uint64)), "sigma bit pattern of non-OK rows"
    assert np.array_equal(gv[bad].view(np.uint64), ov[bad].view(np.uint64)), "vega of non-OK rows"
    ok = ~bad
    stats = {"n": int(gst.size), "ok": int(ok.sum())}
    if not ok.any():
        return stats
    assert np.isfinite(gs[ok]).all() and (gs[ok] > 0).all()
    rel = np.abs(gs[ok] - os_[ok]) / os_[ok]
    stats["sigma_max_rel"] = float(rel.max())
    assert rel.max() <= sigma_tol, f"sigma max rel err {rel.max():.3e}"
    # vega
    if c.get("r") is not None:
        F = c["SorF"] * np.exp((c["r"] - c["q"]) * c["tau"])
    else:
        F = c["SorF"]
    s = os_[ok] * np.sqrt(c["tau"][ok])
    h = np.log(np.minimum(F, c["K"]) / np.maximum(F, c["K"]))[ok] / s
    expo = h * h + 0.25 * s * s
    tol = 1e-12 + 16 * EPS * expo
    verr = np.abs(gv[ok] - ov[ok])
    assert np.all(verr <= tol * ov[ok] + 1e-322), f"vega rel err {np.max(verr / np.maximum(ov[ok], 1e-300)):.3e}"
    big = ov[ok] > 1e-8
    if big.any():
        stats["vega_max_rel_gate_on"] = float((verr[big] / ov[ok][big]).max())
        assert stats["vega_max_rel_gate_on"] <= 1e-12
    return stats


def compare_backward(gP_gpu, gs, vega_gpu, status, vega_or, floor, mode):
    """gP_gpu computed by the GPU from ITS OWN forward outputs (vega_gpu); reference = oracle backward on the
    oracle's forward outputs (vega_or).  Rows with vega within 1e-12 relative of the floor are exempt."""
    ref = po.backward(gs, vega_or, status, floor, mode)
    near = np.abs(vega_or / floor - 1.0) <= 1e-12 if floor > 0 else np.zeros_like(vega_or, bool)
    if mode == 0:
        on = (status == 0) & (np.abs(vega_or) > floor) & ~near
        off = ~((status == 0) & (np.abs(vega_or) > floor)) & ~near
    else:
        on = (status == 0) & (vega_or * vega_or + floor * floor > 0)
        off = ~on
    assert np.array_equal(gP_gpu[off].view(np.uint64), np.zeros(off.sum(), np.float64).view(np.uint64)), "off-gate rows must be +0.0"
    fin = on & np.isfinite(ref) & (ref != 0)
    rel = np.abs(gP_gpu[fin] - ref[fin]) / np.abs(ref[fin])
    if mode == 0:
        assert rel.max() <= 1e-12, f"grad_P max rel err {rel.max():.3e}"
    else:
        # attenuate also runs on rows far below the floor, where grad_P ~ gs V / floor^2 inherits vega's own tolerance
        well = np.abs(vega_or[fin]) > floor
        assert rel[well].max() <= 1e-12, f"grad_P max rel err (|V|>floor) {rel[well].max():.3e}"
        assert rel.max() <= 1e-10, f"grad_P max rel err (all) {rel.max():.3e}"
    z = on & (ref == 0)
    assert np.all(gP_gpu[z] == 0)
    return {"grad_max_rel": float(rel.max()) if rel.size else 0.0, "gate_on": int(on.sum()), "exempt": int(near.sum())}
