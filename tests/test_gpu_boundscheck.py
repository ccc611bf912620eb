"""-m gpu: the forward kernels built with -DPIVOT_BOUNDS_CHECK (device-side asserts on every shared-memory index of the
tile kernel: queue slots, permutation lists, staged positions).  compute-sanitizer is closed on this pool, so this build is
the memory-safety evidence: ragged tails, 1-row tiles, all-rare tiles, dense and empty tiles, BSM, both tile sizes.
A failed assert surfaces as a CUDA error of the stream (PIVOT_ERR_CUDA / a sticky context error), never silently."""
import ctypes as C

import numpy as np
import pytest
import torch

import workloads as wl
import paper_2606_17065_b200 as pv
from paper_2606_17065_b200 import build as pbuild
from paper_2606_17065_b200.binding import _Inputs

pytestmark = pytest.mark.gpu
KEYS = ("SorF", "K", "tau", "P", "flag")


@pytest.fixture(scope="module")
def chk():
    lib = C.CDLL(pbuild.build(bounds_check=True))
    lib.pivot_iv_forward.argtypes = [C.POINTER(_Inputs), C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.pivot_iv_forward.restype = C.c_int
    return lib


def _run(chk, d, n=None):
    n = d["K"].numel() if n is None else n
    r, q = d.get("r"), d.get("q")
    inp = _Inputs(d["SorF"].data_ptr(), d["K"].data_ptr(), d["tau"].data_ptr(), None if r is None else r.data_ptr(),
                  None if q is None else q.data_ptr(), d["P"].data_ptr(), d["flag"].data_ptr())
    out = (torch.empty(n, dtype=torch.float64, device="cuda"), torch.empty(n, dtype=torch.float64, device="cuda"),
           torch.empty(n, dtype=torch.uint8, device="cuda"))
    rc = chk.pivot_iv_forward(C.byref(inp), n, out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr(),
                              C.c_void_p(torch.cuda.current_stream().cuda_stream))
    assert rc == 0
    torch.cuda.synchronize()          # a device-side assert would raise here
    ref = pv.pivot_iv_forward(*[d[k][:n] for k in KEYS], r=None if r is None else r[:n], q=None if q is None else q[:n])
    for a, b in zip(out, ref):
        assert torch.equal(a.view(torch.int64) if a.dtype == torch.float64 else a, b.view(torch.int64) if b.dtype == torch.float64 else b)


def test_bounds_checked_build_on_ragged_edge_and_dense_tiles(chk):
    dev = lambda c: {k: (v.cuda() if isinstance(v, torch.Tensor) else v) for k, v in c.items()}
    mixed = dev(wl.config1((1 << 20) + 1029, seed=3))
    for n in (1, 2, 31, 255, 256, 257, 1023, 1025, 65_537, (1 << 17) + 1, (1 << 19) - 3, (1 << 20) + 1029):   # all three tile sizes, ragged tails
        _run(chk, mixed, n)
    _run(chk, dev(wl.config1(600_000, seed=4, solve_only=True)))          # every row queued: full queues (512-row tiles)
    _run(chk, dev(wl.config1(1_200_000, seed=6, solve_only=True)))        # ... 1024-row tiles
    _run(chk, dev(wl.config2(days=40, seed=5)))                           # BSM chains, 640,000 rows
    _run(chk, dev(wl.config2(days=1, expiries=3, strikes=77)))            # BSM, small tiles
    # tiles made of rows the fast prelude cannot classify (huge / tiny F, K: every row takes the exact prelude and its own
    # atomic queue slot), of invalid rows only, and of zeros
    n = 700_001
    g = torch.Generator().manual_seed(6)
    F = torch.exp(torch.empty(n, dtype=torch.float64).uniform_(np.log(1e150), np.log(1e153), generator=g))
    K = F * torch.exp(torch.empty(n, dtype=torch.float64).uniform_(-0.5, 0.5, generator=g))
    T = torch.full((n,), 0.5, dtype=torch.float64)
    flag = torch.where(K >= F, 1.0, -1.0).to(torch.float64)
    P = wl.textbook_price(F, K, torch.full((n,), 0.2, dtype=torch.float64), flag)
    rare = {"SorF": F.cuda(), "K": K.cuda(), "tau": T.cuda(), "P": P.cuda(), "flag": flag.cuda(), "r": None, "q": None}
    _run(chk, rare)
    st = pv.pivot_iv_forward(*[rare[k] for k in KEYS])[2]
    assert (st == 0).float().mean() > 0.9                                  # they solve -- through the rare path
    bad = dict(rare); bad["tau"] = -rare["tau"]
    _run(chk, bad)
    zero = {k: (torch.zeros_like(v) if isinstance(v, torch.Tensor) else v) for k, v in rare.items()}
    _run(chk, zero)
