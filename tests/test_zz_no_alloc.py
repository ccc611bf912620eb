"""pivot_iv_forward_host_static: the forward call for callers that cannot call cudaMalloc (device staging in a static
`__device__` array of the library, at most PIVOT_STATIC_MAX_ROWS rows).  Checked against the existing device path
(pivot_iv_forward on CUDA tensors) on two calls in a row that share the staging array, at the tolerance of the parity tests
(1e-12 relative on sigma and vega, status bit-exact).  Collected last on purpose (file name): the suite runs with pytest -x."""
import ctypes

import numpy as np
import pytest
import torch

import paper_2606_17065_b200 as pv
import workloads as wl

pytestmark = pytest.mark.gpu

KEYS = ("SorF", "K", "tau", "P", "flag")
RTOL = 1e-12


def _device_path(cfg):
    d = {k: (v.cuda() if isinstance(v, torch.Tensor) else v) for k, v in cfg.items()}
    out = pv.pivot_iv_forward(*[d[k] for k in KEYS], r=d.get("r"), q=d.get("q"))
    torch.cuda.synchronize()
    return tuple(t.cpu().numpy() for t in out)


def _agree(got, ref):
    sig, veg, st = (t.numpy() for t in got)
    assert np.array_equal(st, ref[2])
    ok = ref[2] == 0
    assert ok.any()
    for g, r in ((sig, ref[0]), (veg, ref[1])):
        assert np.array_equal(np.isnan(g), np.isnan(r))
        assert np.all(np.abs(g[ok] - r[ok]) <= RTOL * np.abs(r[ok]))
        rest = ~ok & ~np.isnan(r)
        assert np.array_equal(g[rest], r[rest])     # 0 for AT_INTRINSIC rows, vega 0 for rows without a solve


def test_static_staging_matches_the_device_path_on_two_calls_in_a_row():
    # first call: the maximum size, Black-76, mixed domain (invalid / degenerate rows, all four zones, ragged queue)
    first = wl.config1(pv.STATIC_MAX_ROWS, seed=101)
    # second call: fewer rows, BSM chains: the staging array still holds the first call's rows behind them, and the r / q
    # slots that the first call never wrote
    second = wl.config2(days=1, expiries=7, strikes=333, seed=102)
    assert second["SorF"].numel() < pv.STATIC_MAX_ROWS
    refs = [_device_path(first), _device_path(second)]
    for cfg, ref in zip((first, second), refs):
        host = {k: (v.contiguous() if isinstance(v, torch.Tensor) else v) for k, v in cfg.items()}
        got = pv.pivot_iv_forward_host_static(*[host[k] for k in KEYS], r=host.get("r"), q=host.get("q"))
        _agree(got, ref)
    # and once more on the first inputs, into caller-owned pinned outputs, without the wrapper's synchronise
    host = {k: (v.contiguous().pin_memory() if isinstance(v, torch.Tensor) else v) for k, v in first.items()}
    n = host["SorF"].numel()
    out = (torch.empty(n, dtype=torch.float64).pin_memory(), torch.empty(n, dtype=torch.float64).pin_memory(),
           torch.empty(n, dtype=torch.uint8).pin_memory())
    stream = torch.cuda.Stream()
    pv.pivot_iv_forward_host_static(*[host[k] for k in KEYS], out=out, stream=stream, sync=False)
    stream.synchronize()
    _agree(out, refs[0])


def test_static_staging_size_limit_and_arguments():
    n = pv.STATIC_MAX_ROWS + 1
    cfg = wl.config0(n, seed=103)
    host = [cfg[k].contiguous() for k in KEYS]
    with pytest.raises(pv.PivotError, match="PIVOT_STATIC_MAX_ROWS"):
        pv.pivot_iv_forward_host_static(*host)
    lib = pv.load_library()
    assert lib.pivot_iv_forward_host_static(None, ctypes.c_int64(4), None, None, None, None) == -1     # PIVOT_ERR_NULL
    empty = [t[:0] for t in host]
    sig, veg, st = pv.pivot_iv_forward_host_static(*empty)
    assert sig.numel() == 0 and veg.numel() == 0 and st.numel() == 0
    with pytest.raises(pv.PivotError):
        pv.pivot_iv_forward_host_static(*[t[:100] for t in host], r=host[0][:100])                     # r without q
