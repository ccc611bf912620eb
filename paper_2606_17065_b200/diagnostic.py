"""The paper's NaN-poisoning diagnostic (App. B.2, Fig.6) on top of the C-ABI loss entry points.

Per-row parameters sigma_hat_i are trained with Adam on the hybrid objective of eq.(16),
    L = L_price (eq.(11))  +  lambda * L_rt (eq.(12)),
once with the NAIVE composition sigma_imp o P_BS (no gate, no sentinel, no gradient sanitisation: the inverse channel
follows the layer's strict backward contract and returns NaN where |V| <= 1e-14) and once GATED (sentinel replace below
the floor, residual weighted by w_tau).  Every loss value and every gradient comes from pivot_iv_loss_price /
pivot_iv_loss_roundtrip (one fused kernel each); torch is used for the Adam update of the parameter vector only.
"""
from __future__ import annotations

from typing import Dict, List

import torch

from . import binding as pv


def run_nan_poisoning_diagnostic(chain: Dict[str, torch.Tensor], sigma_star: torch.Tensor, sigma_init: torch.Tensor,
                                 gated: bool, steps: int = 200, lr: float = 1e-2, lam: float = 1.0,
                                 gate_floor: float = 1e-6, strict_floor: float = 1e-14) -> Dict[str, List[float]]:
    """Runs `steps` Adam steps on sigma_hat (CUDA fp64, one parameter per row).  Returns per-step lists:
    `finite_frac` (fraction of sigma_hat rows that are finite BEFORE the step), `loss`, `nan_grads` (NaN gradient entries)."""
    a = [chain[k] for k in ("SorF", "K", "tau", "P", "flag")]
    rq = dict(r=chain.get("r"), q=chain.get("q"))
    n = a[0].numel()
    sig = sigma_init.clone()
    m = torch.zeros_like(sig)
    v = torch.zeros_like(sig)
    b1, b2, eps = 0.9, 0.999, 1e-8
    mean_abs_p = float(a[3].abs().mean().item())
    out = {"finite_frac": [], "loss": [], "nan_grads": []}
    for t in range(1, steps + 1):
        out["finite_frac"].append(float(torch.isfinite(sig).double().mean().item()))
        sp, gp = pv.pivot_iv_loss_price(*a, sig, grad_scale=1.0 / (n * mean_abs_p ** 2), **rq)
        if gated:
            sr, gr = pv.pivot_iv_loss_roundtrip(*a, sig, sigma_star, gate_floor, mode=pv.RT_GATED, grad_scale=lam / n, **rq)
        else:
            sr, gr = pv.pivot_iv_loss_roundtrip(*a, sig, sigma_star, strict_floor, mode=pv.RT_NAIVE, grad_scale=lam / n, **rq)
        sp, sr = sp.tolist(), sr.tolist()
        loss = (sp[0] / max(sp[2], 1.0)) / mean_abs_p ** 2 + lam * sr[0] / n
        g = gp + gr
        out["loss"].append(loss)
        out["nan_grads"].append(int(torch.isnan(g).sum().item()))
        # Adam on the parameter vector (no sanitisation of g: a NaN gradient poisons its row, as in the paper's naive run)
        m = b1 * m + (1 - b1) * g
        v = b2 * v + (1 - b2) * g * g
        sig = sig - lr * (m / (1 - b1 ** t)) / ((v / (1 - b2 ** t)).sqrt() + eps)
    out["finite_frac"].append(float(torch.isfinite(sig).double().mean().item()))
    out["sigma_hat"] = sig
    return out
