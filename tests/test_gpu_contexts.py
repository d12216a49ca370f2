"""Two contexts on one GPU (`-m gpu`).  The channel-walking kernels read their component blocks from ONE
constant bank per device (predict_walk.cu), which every walking call refills as it goes; the library orders
walking calls on a device one after another across contexts and streams, so contexts stay independent as
include/woden_b200.h promises.  Eq 9 against the oracle for both contexts' interleaved calls."""
import numpy as np
import pytest

import oracle
from paper_2005_09316_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = 1.0e-4


def test_two_contexts_on_two_streams_interleaving_walking_calls_match_the_oracle():
    import torch
    from paper_2005_09316_b200 import binding
    dev = torch.device("cuda", 0)
    rng = np.random.default_rng(77)
    T, B, F = 2, 1500, 64                      # 24 CTAs per launch: launches of the two streams would overlap
    u = rng.normal(0, 800.0, (T, B)); v = rng.normal(0, 800.0, (T, B)); w = rng.normal(0, 60.0, (T, B))
    fr = 150e6 + 80e3 * np.arange(F)
    d = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64, device=dev)
    uvw = binding.Uvw(d(u), d(v), d(w), fr)
    sets = []
    for n, seed in ((450, 1), (610, 2)):       # 3 constant blocks each (204 points per block)
        r = np.random.default_rng(seed)
        l, m = inputs.disk_lm(r, n, 12.0)
        s0 = r.lognormal(0.0, 1.0, n) * (1.0 + seed); al = r.normal(-0.8, 0.2, n)
        sets.append((l, m, s0, al))
    ctxs = [binding.Woden(0), binding.Woden(0)]
    streams = [torch.cuda.Stream(dev), torch.cuda.Stream(dev)]
    dsets = [[d(a) for a in s] for s in sets]
    outs = [[ctxs[i].new_vis(uvw) for _ in range(4)] for i in range(2)]
    torch.cuda.synchronize()
    for rep in range(4):                       # A, B, A, B, ... with nothing ordering the two streams
        for i in range(2):
            ctxs[i].predict_points(uvw, *dsets[i], 150e6, outs[i][rep], False, stream=streams[i])
            assert ctxs[i].last_path() == binding.WODEN_PATH_WALKING
    torch.cuda.synchronize()
    for i in range(2):
        ctxs[i].check()
        l, m, s0, al = sets[i]
        ref = oracle.predict_points(u, v, w, fr, l, m, s0, al, 150e6)
        scale = oracle.tolerance_scale(fr, s0, al, 150e6)
        for rep in range(4):
            err = np.abs(outs[i][rep].cpu().numpy() - ref) / scale[None, :, None]
            assert err.max() <= TOL, (i, rep, float(err.max()))
    for c in ctxs:
        c.close()
