"""World-size-2 `gloo` test of the multi-GPU host logic: the path shards
by time step with no data-path collective, so two ranks predicting their shards and one
all-gather must reproduce the unsharded prediction exactly, and the timed region is the max
over ranks.  No GPU here: the per-rank compute stand-in is the CPU oracle (test infrastructure);
what is under test is paper_2005_09316_b200.parallel + inputs.time_shard."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, scaling, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      OMP_NUM_THREADS="1")
    import torch
    import torch.distributed as dist
    import oracle
    from paper_2005_09316_b200 import parallel
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = parallel.rank_workload(2, rank, world, scaling=scaling)
        # a thin slice of the sky keeps the oracle at a fraction of a second per rank
        l, m = wl.points.l[:7], wl.points.m[:7]
        s0, al = wl.points.s0_jy[:7], wl.points.alpha[:7]
        fr = wl.freqs_hz[:3]
        u, v, w = (a[:, :50] for a in (wl.u_m, wl.v_m, wl.w_m))
        vis = torch.from_numpy(oracle.predict_points(u, v, w, fr, l, m, s0, al, wl.ref_freq_hz))
        parts = parallel.gather_time_shards(vis, dist)
        whole = torch.cat(parts).numpy()
        slowest = parallel.max_over_ranks(10.0 + rank, dist)
        q.put((rank, wl.n_times, whole, slowest, wl.meta["t_index0"]))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("scaling", ["weak", "strong"])
def test_two_rank_time_sharding_reproduces_the_unsharded_prediction(scaling):
    import torch.multiprocessing as mp
    import oracle
    from paper_2005_09316_b200 import inputs

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, scaling, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted((q.get(timeout=240) for _ in procs), key=lambda x: x[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0

    T_cfg = inputs.make_config_shape(2)[1]
    T_total = 2 * T_cfg if scaling == "weak" else T_cfg
    full = inputs.make_config(2, n_times=T_total, n_times_total=T_total)
    ref = oracle.predict_points(full.u_m[:, :50], full.v_m[:, :50], full.w_m[:, :50], full.freqs_hz[:3],
                                full.points.l[:7], full.points.m[:7], full.points.s0_jy[:7],
                                full.points.alpha[:7], full.ref_freq_hz)
    assert sum(g[1] for g in got) == T_total
    assert got[0][4] == 0 and got[1][4] == got[0][1]            # shards are contiguous in time
    for rank, _, whole, slowest, _ in got:
        assert whole.shape == ref.shape
        # same inputs, same oracle, disjoint outputs: the gathered buffer IS the unsharded one
        assert np.abs(whole - ref).max() <= 1e-9 * np.abs(ref).max()
        assert slowest == 11.0                                   # max over ranks, on every rank


def test_single_process_fallbacks_need_no_process_group():
    import torch
    from paper_2005_09316_b200 import parallel
    v = torch.zeros((2, 3, 4), dtype=torch.complex64)
    assert parallel.gather_time_shards(v)[0] is v
    assert parallel.max_over_ranks(3.5) == 3.5
    wl = parallel.rank_workload(1, 0, 1)
    assert wl.n_times == 1
    with pytest.raises(ValueError):
        parallel.rank_workload(1, 1, 2, scaling="strong")       # config 1 has one time step
