"""GPU-vs-oracle parity through the C ABI (libwoden_b200.so), `-m gpu`.

Criterion (BASELINE.json north_star): for every evaluated visibility
|V_gpu - V_oracle| <= 1e-4 * sum_k |S_k(nu_f)| (x sum|coeff| for shapelets, reading G12).
Configs 1-3 compare element by element where the oracle finishes in seconds (config 1 in
full; 2-3 on every baseline of first/last time step at first/middle/last channel plus a seeded
random sample); configs 4-5 run at full size in bench.py's launch configuration and are
compared on the declared seeded subset.
"""
import numpy as np
import pytest

import oracle
from paper_2005_09316_b200 import inputs

pytestmark = pytest.mark.gpu

TOL = 1.0e-4


@pytest.fixture(scope="module")
def torch_mod():
    import torch
    return torch


@pytest.fixture(scope="module")
def ctx():
    from paper_2005_09316_b200 import binding
    c = binding.Woden(0)
    yield c
    c.close()


def _gpu_total(ctx, wl, path):
    from paper_2005_09316_b200 import binding
    import torch
    ctx.set_path(path)
    dw = binding.DeviceWorkload(wl, ctx=ctx)          # M_j from woden_shapelet_uv_basis, not from the generator
    vis = dw.predict(ctx)
    torch.cuda.synchronize()
    ctx.check()
    return vis.cpu().numpy()


def _assert_parity(V_gpu_flat, V_ref, scale_f, idx, wl, what):
    B, F = wl.n_baselines, wl.n_freqs
    f_of = (idx // B) % F
    err = np.abs(V_gpu_flat.astype(np.complex128) - V_ref) / scale_f[f_of]
    worst = int(np.argmax(err))
    assert err[worst] <= TOL, f"{what}: max |dV|/scale = {err[worst]:.3e} at flat index {idx[worst]}"
    return float(err[worst])


@pytest.mark.parametrize("path", [0, 1], ids=["auto", "general"])
def test_config1_tiny_full_parity(ctx, path):
    wl = inputs.make_config(1)
    V = _gpu_total(ctx, wl, path)
    ref = oracle.predict_workload(wl)
    scale = oracle.workload_tolerance_scale(wl)
    idx = np.arange(wl.n_vis, dtype=np.int64)
    _assert_parity(V.reshape(-1), ref.reshape(-1), scale, idx, wl, "config 1")
    assert np.max(np.abs(ref)) > 1.0      # a non-trivial comparison


_ORACLE_CACHE = {}


def _oracle_on_declared_subset(cfg, n_random):
    """The declared seeded subset of SURVEY.md 8(d) / BASELINE.md (inputs.subset_indices): every baseline
    of the first and last time step at the first, middle and last channel, plus n_random uniformly drawn
    visibilities.  The oracle's values are computed once per config and shared by the two GPU paths."""
    if cfg not in _ORACLE_CACHE:
        wl = inputs.make_config(cfg)
        idx = inputs.subset_indices(wl, n_random=n_random)
        _ORACLE_CACHE[cfg] = (wl, idx, oracle.predict_workload(wl, vis_index=idx), oracle.workload_tolerance_scale(wl))
    return _ORACLE_CACHE[cfg]


@pytest.mark.parametrize("path", [0, 1], ids=["auto", "general"])
@pytest.mark.parametrize("cfg,n_random", [(2, 200_000), (3, 20_000), (4, 150_000), (5, 250_000), (6, 100_000),
                                          (7, 150_000)])
def test_configs_2_to_7_full_size_parity_on_the_declared_subset(ctx, cfg, n_random, path):
    wl, idx, ref, scale = _oracle_on_declared_subset(cfg, n_random)
    assert idx.size > n_random // 2 + 3 * wl.n_baselines        # the full rows are in
    V = _gpu_total(ctx, wl, path)
    from paper_2005_09316_b200 import binding
    if wl.points.n or wl.gaussians.n:
        assert ctx.last_path() == (binding.WODEN_PATH_WALKING if path == 0 else binding.WODEN_PATH_GENERAL)
    _assert_parity(V.reshape(-1)[idx], ref, scale, idx, wl, f"config {cfg}")
    assert np.all(np.isfinite(V.view(np.float32)))


def _small_case(seed=0, T=3, B=300, F=21, uniform=True):
    """A ragged case: B, F and component counts are not multiples of any tile."""
    rng = np.random.default_rng(seed)
    east, north = inputs.disk_antennas(rng, 25, 1500.0)
    u, v, w = inputs.uvw_metres(east, north, T, 8.0)
    u, v, w = (np.ascontiguousarray(a[:, :B]) for a in (u, v, w))
    if uniform:
        fr = 170e6 + 40e3 * np.arange(F)
    else:
        fr = np.sort(rng.uniform(80e6, 300e6, F))
    return u, v, w, fr


def _dev(torch, a, dtype=None):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=dtype or torch.float64, device="cuda:0")


@pytest.mark.parametrize("uniform", [True, False], ids=["uniform", "irregular"])
@pytest.mark.parametrize("n", [1, 63, 64, 65, 200])
def test_points_ragged_sizes_and_channel_lists(ctx, torch_mod, n, uniform):
    from paper_2005_09316_b200 import binding
    torch = torch_mod
    ctx.set_path(0)
    u, v, w, fr = _small_case(seed=n, uniform=uniform)
    rng = np.random.default_rng(100 + n)
    l, m = inputs.disk_lm(rng, n, 30.0)
    s0 = inputs.log_uniform(rng, n, 0.1, 10.0) * rng.choice([-1.0, 1.0], n)
    al = rng.normal(-0.8, 0.3, n)
    uvw = binding.Uvw(_dev(torch, u), _dev(torch, v), _dev(torch, w), fr)
    vis = ctx.new_vis(uvw)
    ctx.predict_points(uvw, _dev(torch, l), _dev(torch, m), _dev(torch, s0), _dev(torch, al), 150e6, vis)
    torch.cuda.synchronize(); ctx.check()
    ref = oracle.predict_points(u, v, w, fr, l, m, s0, al, 150e6)
    scale = oracle.tolerance_scale(fr, s0, al, 150e6)
    err = np.abs(vis.cpu().numpy() - ref) / scale[None, :, None]
    assert err.max() <= TOL


@pytest.mark.parametrize("F", [2, 7, 8, 9, 16, 17, 18, 31, 33, 40, 65])
def test_walking_path_channel_counts_around_the_tile_edges(ctx, torch_mod, F):
    # equally spaced channels take the channel-walking kernel (32-channel tiles, chains seeded at
    # tile positions 7 and 23): every F that leaves a seed position past the last channel, and
    # negative channel steps, must still meet parity for points and Gaussians
    from paper_2005_09316_b200 import binding
    torch = torch_mod
    ctx.set_path(0)
    n = 70
    for step in (40e3, -125e3):
        u, v, w, _ = _small_case(seed=F, T=2, B=130, F=F)
        fr = 180e6 + step * np.arange(F)
        rng = np.random.default_rng(500 + F)
        l, m = inputs.disk_lm(rng, n, 25.0)
        s0 = inputs.log_uniform(rng, n, 0.1, 10.0) * rng.choice([-1.0, 1.0], n)
        al = rng.normal(-0.8, 0.3, n)
        maj = inputs.log_uniform(rng, n, 0.5, 30.0) * inputs.ARCMIN
        mnr = maj * rng.uniform(0.1, 1.0, n)
        pa = rng.uniform(0, np.pi, n)
        uvw = binding.Uvw(_dev(torch, u), _dev(torch, v), _dev(torch, w), fr)
        vis = ctx.new_vis(uvw)
        args = [_dev(torch, a) for a in (l, m, s0, al)]
        ctx.predict_points(uvw, *args, 150e6, vis)
        ctx.predict_gaussians(uvw, *args, 150e6, _dev(torch, maj), _dev(torch, mnr), _dev(torch, pa), vis, True)
        torch.cuda.synchronize(); ctx.check()
        ref = oracle.predict_points(u, v, w, fr, l, m, s0, al, 150e6)
        oracle.predict_gaussians(u, v, w, fr, l, m, s0, al, 150e6, maj, mnr, pa, out=ref, accumulate=True)
        scale = 2.0 * oracle.tolerance_scale(fr, s0, al, 150e6)
        err = np.abs(vis.cpu().numpy() - ref) / scale[None, :, None]
        assert err.max() <= TOL, (F, step, err.max())


@pytest.mark.parametrize("uniform", [True, False], ids=["uniform", "irregular"])
def test_gaussians_ragged_including_zero_width(ctx, torch_mod, uniform):
    from paper_2005_09316_b200 import binding
    torch = torch_mod
    ctx.set_path(0)
    n = 131
    u, v, w, fr = _small_case(seed=7, uniform=uniform)
    rng = np.random.default_rng(77)
    l, m = inputs.disk_lm(rng, n, 20.0)
    s0 = inputs.log_uniform(rng, n, 0.01, 5.0)
    al = rng.normal(-0.8, 0.2, n)
    maj = inputs.log_uniform(rng, n, 0.2, 30.0) * inputs.ARCMIN
    mnr = maj * rng.uniform(0.0, 1.0, n)
    maj[:5] = 0.0; mnr[:5] = 0.0                         # zero-width Gaussians are points (G13)
    pa = rng.uniform(0, np.pi, n)
    uvw = binding.Uvw(_dev(torch, u), _dev(torch, v), _dev(torch, w), fr)
    vis = ctx.new_vis(uvw)
    args = [_dev(torch, a) for a in (l, m, s0, al)]
    ctx.predict_gaussians(uvw, *args, 150e6, _dev(torch, maj), _dev(torch, mnr), _dev(torch, pa), vis)
    torch.cuda.synchronize(); ctx.check()
    ref = oracle.predict_gaussians(u, v, w, fr, l, m, s0, al, 150e6, maj, mnr, pa)
    scale = oracle.tolerance_scale(fr, s0, al, 150e6)
    err = np.abs(vis.cpu().numpy() - ref) / scale[None, :, None]
    assert err.max() <= TOL


def _run_shapelets(ctx, torch, u, v, w, fr, l, m, s0, al, b1, b2, pa, M, off, n1, n2, cf, p_max):
    from paper_2005_09316_b200 import binding
    uvw = binding.Uvw(_dev(torch, u), _dev(torch, v), _dev(torch, w), fr)
    vis = ctx.new_vis(uvw)
    d = lambda a: None if a is None else _dev(torch, a)
    di = lambda a: _dev(torch, a, torch.int32)
    ctx.predict_shapelets(uvw, d(l), d(m), d(s0), d(al), 150e6, d(b1), d(b2), d(pa), d(M), di(off),
                          len(cf), p_max, di(n1), di(n2), d(cf), vis)
    torch.cuda.synchronize(); ctx.check()
    return vis.cpu().numpy()


ORDER_BUCKETS = (4, 8, 12, 16, 20, 24, 32, 40, 48, 60, 72, 86, 100)     # the kernels' compile-time orders
TENSOR_FROM = 24                                                          # AUTO's switch (api.cu)
# every bucket edge and the order just above it (which must take the next bucket), plus 0 and 1
BUCKET_EDGE_ORDERS = [0, 1] + sorted(set(ORDER_BUCKETS) | {b + 1 for b in ORDER_BUCKETS[:-1]})


def _bucket_of(p_max):
    return next(b for b in ORDER_BUCKETS if p_max <= b)


def _is_sparse(n_coeff, n, bucket):
    return n_coeff < 0.75 * n * ((bucket + 1) * (bucket + 2) // 2)      # api.cu: chunk-skipping variant below 3/4


def _expected_engine(engine, bucket, sparse):
    from paper_2005_09316_b200 import binding
    if engine == 2 or (engine == 0 and bucket >= TENSOR_FROM):
        return binding.WODEN_SHAPELET_TENSOR
    return binding.WODEN_SHAPELET_REGISTER_SPARSE if sparse else binding.WODEN_SHAPELET_REGISTER


@pytest.mark.parametrize("engine", [1, 2, 0], ids=["register", "tensor", "auto"])
@pytest.mark.parametrize("p_max", BUCKET_EDGE_ORDERS)
def test_shapelets_orders_up_to_the_limit(ctx, torch_mod, p_max, engine):
    # full triangles at EVERY order bucket's edge and the order above it, on both engines and under AUTO
    # (each bucket is its own template instantiation with its own tiling and descriptor table), incl. the
    # paper's p_max = 86 and the library limit; beta up to 20 arcmin on a 3 km array reaches
    # Hermite arguments ~30 (H4).  Eq 15-17.
    ctx.set_path(0)
    ctx.set_shapelet_path(engine)
    u, v, w, fr = _small_case(seed=p_max, T=2, B=333, F=5)
    rng = np.random.default_rng(1000 + p_max)
    n = 3
    l, m = inputs.disk_lm(rng, n, 10.0)
    s0 = np.array([1.0, 2.5, 0.7]); al = np.array([-0.8, -0.5, -1.1])
    b1 = np.array([5.0, 20.0, 1.0]) * inputs.ARCMIN
    b2 = np.array([7.0, 12.0, 0.5]) * inputs.ARCMIN
    pa = rng.uniform(0, np.pi, n)
    M = inputs.local_uv_basis(l, m)
    t1, t2 = inputs.full_triangle(p_max)
    P = len(t1)
    n1 = np.tile(t1, n); n2 = np.tile(t2, n)
    cf = rng.normal(0, 1, n * P) * np.exp(-(n1 + n2) / 10.0)
    off = np.arange(n + 1) * P
    V = _run_shapelets(ctx, torch_mod, u, v, w, fr, l, m, s0, al, b1, b2, pa, M, off, n1, n2, cf, p_max)
    ran = ctx.last_shapelet_path()
    ref = oracle.predict_shapelets(u, v, w, fr, l, m, s0, al, 150e6, b1, b2, pa, M, off, n1, n2, cf)
    scale = oracle.tolerance_scale(fr, s0, al, 150e6, off, cf)
    ctx.set_shapelet_path(0)
    bucket = _bucket_of(p_max)
    sparse = _is_sparse(n * P, n, bucket)
    assert ran == (_expected_engine(engine, bucket, sparse), bucket)
    err = np.abs(V - ref) / scale[None, :, None]
    assert err.max() <= TOL
    assert np.abs(ref).max() > 1e-3


@pytest.mark.parametrize("engine", [0, 2, 1], ids=["auto", "tensor", "register"])
@pytest.mark.parametrize("f_keep", [0.6, 0.2])
@pytest.mark.parametrize("p_max", [b for b in ORDER_BUCKETS if b >= TENSOR_FROM] + [23, 29, 42])
def test_truncated_triangles_on_every_tensor_bucket(ctx, torch_mod, p_max, f_keep, engine):
    # PAPER.md:267-288 (Eq 23-25): a model truncated to a fraction of its ranked absolute weight is a SPARSE
    # coefficient list whose highest surviving order decides the bucket.  Every bucket AUTO gives to the tensor
    # engine (and the p_max = 42 / 29 / 23 of config 4's truncated models, profiles/truncation_r2.md) is run
    # under AUTO, forced TENSOR and forced REGISTER against the oracle on the same ragged, unsorted lists.
    from oracle import truncate as otrunc
    ctx.set_path(0)
    ctx.set_shapelet_path(engine)
    u, v, w, fr = _small_case(seed=500 + p_max, T=2, B=257, F=3)
    rng = np.random.default_rng(7000 + 10 * p_max + int(10 * f_keep))
    n = 2
    l, m = inputs.disk_lm(rng, n, 10.0)
    s0 = np.array([1.3, 0.6]); al = np.array([-0.7, -1.0])
    b1 = np.array([4.0, 9.0]) * inputs.ARCMIN; b2 = np.array([6.0, 3.0]) * inputs.ARCMIN
    pa = rng.uniform(0, np.pi, n)
    M = inputs.local_uv_basis(l, m)
    t1, t2 = inputs.full_triangle(p_max)
    n1l, n2l, cfl, off = [], [], [], [0]
    for j in range(n):
        cf = rng.normal(0, 1, len(t1)) * np.exp(-(t1 + t2) / 8.0)
        keep = otrunc.keep_mask(cf, f_keep)                       # Eq 23-24 on |C| (Eq 25 with unit basis sums)
        keep[np.flatnonzero(t1 + t2 == p_max)[j]] = True           # one term of the highest order survives
        idx = rng.permutation(np.flatnonzero(keep))                # the list order is free
        n1l.append(t1[idx]); n2l.append(t2[idx]); cfl.append(cf[idx]); off.append(off[-1] + idx.size)
    n1, n2, cf = np.concatenate(n1l), np.concatenate(n2l), np.concatenate(cfl)
    bucket = _bucket_of(p_max)
    sparse = _is_sparse(cf.size, n, bucket)
    assert sparse and cf.size < 0.5 * n * len(t1)
    V = _run_shapelets(ctx, torch_mod, u, v, w, fr, l, m, s0, al, b1, b2, pa, M, off, n1, n2, cf, p_max)
    ran = ctx.last_shapelet_path()
    ctx.set_shapelet_path(0)
    assert ran == (_expected_engine(engine, bucket, sparse), bucket)
    ref = oracle.predict_shapelets(u, v, w, fr, l, m, s0, al, 150e6, b1, b2, pa, M, off, n1, n2, cf)
    scale = oracle.tolerance_scale(fr, s0, al, 150e6, off, cf)
    assert (np.abs(V - ref) / scale[None, :, None]).max() <= TOL
    assert np.abs(ref).max() > 1e-3


@pytest.mark.parametrize("engine", [0, 2, 1], ids=["auto", "tensor", "register"])
@pytest.mark.parametrize("f_comp", [0.8, 0.6, 0.4, 0.2])
def test_config4_models_truncated_by_eq25_weights_as_bench_times_them(ctx, torch_mod, f_comp, engine):
    # the exact models `bench.py --truncation` times (config 4's two lobes ranked by Eq 25 with the restoring
    # beam): p_max 42 / 29 / 23 / 17 -> buckets 48 / 32 / 24 / 20, here checked against the oracle
    from paper_2005_09316_b200 import truncate
    wl = inputs.make_config(4)
    w_sh = truncate.shapelet_basis_weights(ctx, wl.shapelets)
    s = truncate.truncate_shapelets(ctx, wl.shapelets, f_comp, w_sh)
    ctx.set_path(0)
    ctx.set_shapelet_path(engine)
    u, v, w = (a[:2, :1200] for a in (wl.u_m, wl.v_m, wl.w_m))
    fr = wl.freqs_hz[::64]
    pmax = int((s.n1 + s.n2).max())
    V = _run_shapelets(ctx, torch_mod, u, v, w, fr, s.l, s.m, s.s0_jy, s.alpha, s.beta1_rad, s.beta2_rad, s.pa_rad,
                       s.uv_basis, s.coeff_offset, s.n1, s.n2, s.coeff, pmax)
    ran = ctx.last_shapelet_path()
    ctx.set_shapelet_path(0)
    bucket = _bucket_of(pmax)
    sparse = _is_sparse(s.coeff.size, s.n, bucket)
    assert ran == (_expected_engine(engine, bucket, sparse), bucket)
    ref = oracle.predict_shapelets(u, v, w, fr, s.l, s.m, s.s0_jy, s.alpha, 150e6, s.beta1_rad, s.beta2_rad,
                                   s.pa_rad, s.uv_basis, s.coeff_offset, s.n1, s.n2, s.coeff)
    scale = oracle.tolerance_scale(fr, s.s0_jy, s.alpha, 150e6, s.coeff_offset, s.coeff)
    assert (np.abs(V - ref) / scale[None, :, None]).max() <= TOL
    assert np.abs(ref).max() > 1e-3


@pytest.mark.parametrize("engine", [1, 2], ids=["register", "tensor"])
def test_shapelets_single_high_order_terms_and_sparse_lists(ctx, torch_mod, engine):
    # one isolated coefficient at a time: no cancellation hides a wrong sign / index / scale;
    # truncated (sparse, unsorted, duplicated) lists: duplicates add, missing entries are zero.
    ctx.set_path(0)
    ctx.set_shapelet_path(engine)
    u, v, w, fr = _small_case(seed=3, T=1, B=257, F=3)
    u *= 0.3; v *= 0.3; w *= 0.3
    l = np.array([0.01]); m = np.array([-0.02]); s0 = np.array([1.0]); al = np.array([0.0])
    b1 = np.array([6.0]) * inputs.ARCMIN; b2 = np.array([4.0]) * inputs.ARCMIN; pa = np.array([0.8])
    for (a, b) in [(0, 0), (1, 0), (0, 1), (2, 3), (7, 0), (0, 9), (30, 30), (59, 1), (3, 97), (100, 0)]:
        V = _run_shapelets(ctx, torch_mod, u, v, w, fr, l, m, s0, al, b1, b2, pa, None,
                           [0, 1], [a], [b], [1.0], a + b)
        ref = oracle.predict_shapelets(u, v, w, fr, l, m, s0, al, 150e6, b1, b2, pa, None, [0, 1], [a], [b], [1.0])
        assert np.abs(V - ref).max() <= TOL, (a, b)
    n1 = np.array([5, 0, 2, 2, 11, 2]); n2 = np.array([1, 0, 2, 7, 0, 2]); cf = np.array([0.5, 1.0, -0.3, 0.2, 0.1, 0.4])
    V = _run_shapelets(ctx, torch_mod, u, v, w, fr, l, m, s0, al, b1, b2, pa, None, [0, 6], n1, n2, cf, 11)
    ref = oracle.predict_shapelets(u, v, w, fr, l, m, s0, al, 150e6, b1, b2, pa, None, [0, 6], n1, n2, cf)
    assert np.abs(V - ref).max() <= TOL * np.abs(cf).sum()
    ctx.set_shapelet_path(0)


@pytest.mark.parametrize("cfg,f_comp", [(5, 0.5), (5, 0.1), (4, 0.3)])
def test_truncated_shapelet_models_take_the_sparse_kernel(ctx, torch_mod, cfg, f_comp):
    ctx.set_shapelet_path(1)        # register engine: its chunk-skipping variant is what this test is about
    # PAPER.md section 5.3 (Eq 23-24): basis functions ranked by absolute flux, a fraction kept; the
    # ragged coefficient lists go through the chunk-skipping kernel variant (PM = 40 NV = 2, PM = 60)
    from paper_2005_09316_b200 import truncate
    wl = inputs.make_config(cfg)
    s = truncate.truncate_shapelets(ctx, wl.shapelets, f_comp)
    assert s.coeff.size < 0.75 * wl.shapelets.coeff.size
    u, v, w = (a[:2, :1500] for a in (wl.u_m, wl.v_m, wl.w_m))
    fr = wl.freqs_hz[::48]
    pmax = int((s.n1 + s.n2).max())
    V = _run_shapelets(ctx, torch_mod, u, v, w, fr, s.l, s.m, s.s0_jy, s.alpha, s.beta1_rad, s.beta2_rad, s.pa_rad,
                       s.uv_basis, s.coeff_offset, s.n1, s.n2, s.coeff, pmax)
    ref = oracle.predict_shapelets(u, v, w, fr, s.l, s.m, s.s0_jy, s.alpha, 150e6, s.beta1_rad, s.beta2_rad,
                                   s.pa_rad, s.uv_basis, s.coeff_offset, s.n1, s.n2, s.coeff)
    scale = oracle.tolerance_scale(fr, s.s0_jy, s.alpha, 150e6, s.coeff_offset, s.coeff)
    ctx.set_shapelet_path(0)
    assert (np.abs(V - ref) / scale[None, :, None]).max() <= TOL
    assert np.abs(ref).max() > 1e-3
    # AUTO (tensor engine from order bucket 40) must agree as well
    V2 = _run_shapelets(ctx, torch_mod, u, v, w, fr, s.l, s.m, s.s0_jy, s.alpha, s.beta1_rad, s.beta2_rad, s.pa_rad,
                        s.uv_basis, s.coeff_offset, s.n1, s.n2, s.coeff, pmax)
    assert (np.abs(V2 - ref) / scale[None, :, None]).max() <= TOL


def test_tensor_engine_accumulates_and_handles_ragged_batches(ctx, torch_mod):
    # the tcgen05 engine owns 128 visibilities per CTA: T x B = 3 x 171 = 513 leaves a one-row tail;
    # accumulate = 1 must add into the buffer; two identical calls must be bit-identical
    from paper_2005_09316_b200 import binding
    torch = torch_mod
    ctx.set_path(0)
    u, v, w, fr = _small_case(seed=44, T=3, B=171, F=4)
    rng = np.random.default_rng(44)
    n, p_max = 2, 44
    l, m = inputs.disk_lm(rng, n, 8.0)
    s0 = np.array([1.5, -0.7]); al = np.array([-0.8, -0.3])
    b1 = np.array([6.0, 15.0]) * inputs.ARCMIN; b2 = np.array([9.0, 4.0]) * inputs.ARCMIN
    pa = rng.uniform(0, np.pi, n)
    t1, t2 = inputs.full_triangle(p_max)
    P = len(t1)
    n1 = np.tile(t1, n); n2 = np.tile(t2, n)
    cf = rng.normal(0, 1, n * P) * np.exp(-(n1 + n2) / 10.0) * 1e3        # large coefficients: exercises the scaling
    off = np.arange(n + 1) * P
    d = lambda a: _dev(torch, a)
    di = lambda a: _dev(torch, a, torch.int32)
    uvw = binding.Uvw(d(u), d(v), d(w), fr)
    args = (uvw, d(l), d(m), d(s0), d(al), 150e6, d(b1), d(b2), d(pa), None, di(off), len(cf), p_max, di(n1), di(n2), d(cf))
    ctx.set_shapelet_path(2)
    base = torch.full(uvw.vis_shape, 2 - 3j, dtype=torch.complex64, device="cuda:0")
    acc = base.clone()
    ctx.predict_shapelets(*args, acc, True)
    plain = ctx.new_vis(uvw)
    ctx.predict_shapelets(*args, plain, False)
    again = ctx.new_vis(uvw)
    ctx.predict_shapelets(*args, again, False)
    torch.cuda.synchronize(); ctx.check()
    ctx.set_shapelet_path(0)
    assert torch.equal(plain, again)
    assert torch.max(torch.abs(acc - (base + plain))).item() <= 1e-3 * float(torch.max(torch.abs(plain)).item()) * 1e-3
    ref = oracle.predict_shapelets(u, v, w, fr, l, m, s0, al, 150e6, b1, b2, pa, None, off, n1, n2, cf)
    scale = oracle.tolerance_scale(fr, s0, al, 150e6, off, cf)
    assert (np.abs(plain.cpu().numpy() - ref) / scale[None, :, None]).max() <= TOL


def test_accumulate_zero_components_and_additivity(ctx, torch_mod):
    from paper_2005_09316_b200 import binding
    torch = torch_mod
    ctx.set_path(0)
    wl = inputs.make_config(1)
    dw = binding.DeviceWorkload(wl)
    total = dw.predict(ctx).clone()
    # n == 0: overwrite zero-fills, accumulate leaves the buffer alone
    vis = torch.full(dw.uvw.vis_shape, 3 + 4j, dtype=torch.complex64, device="cuda:0")
    ctx.predict_points(dw.uvw, None, None, None, None, wl.ref_freq_hz, vis, accumulate=True)
    assert torch.all(vis == 3 + 4j)
    ctx.predict_gaussians(dw.uvw, None, None, None, None, wl.ref_freq_hz, None, None, None, vis, accumulate=False)
    assert torch.all(vis == 0)
    # the three types in a different order, all accumulating into zeros, give the same total
    l, m, s0, al, mj, mn, pa = dw.g
    ctx.predict_gaussians(dw.uvw, l, m, s0, al, wl.ref_freq_hz, mj, mn, pa, vis, accumulate=True)
    l, m, s0, al, b1, b2, pa, M, off, nc, pmax, n1, n2, cf = dw.s
    ctx.predict_shapelets(dw.uvw, l, m, s0, al, wl.ref_freq_hz, b1, b2, pa, M, off, nc, pmax, n1, n2, cf, vis, True)
    ctx.predict_points(dw.uvw, *dw.p, wl.ref_freq_hz, vis, accumulate=True)
    torch.cuda.synchronize()
    assert torch.max(torch.abs(vis - total)).item() < 2e-5
    # determinism: the register reduction has a fixed order
    again = dw.predict(ctx)
    assert torch.equal(again, total)


@pytest.mark.parametrize("keep", ["points", "gaussians", "shapelets", "gaussians+shapelets", "none"])
def test_first_non_empty_type_overwrites_a_dirty_buffer(ctx, torch_mod, keep):
    """DeviceWorkload.predict and woden_simulate_host let the first non-empty component type overwrite the buffer
    (no zero-fill pass): whatever the buffer held before, the result is the sum of the types present."""
    from paper_2005_09316_b200 import binding
    torch = torch_mod
    ctx.set_path(0)
    wl = inputs.make_config(1)
    full = binding.DeviceWorkload(wl, ctx=ctx)
    dw = binding.DeviceWorkload(wl, ctx=ctx)
    if "points" not in keep: dw.p = None
    if "gaussians" not in keep: dw.g = None
    if "shapelets" not in keep: dw.s = None
    # reference: each present type alone into zeros, summed
    ref = torch.zeros(full.uvw.vis_shape, dtype=torch.complex64, device="cuda:0")
    if dw.p is not None:
        ctx.predict_points(full.uvw, *full.p, wl.ref_freq_hz, ref, accumulate=True)
    if dw.g is not None:
        l, m, s0, al, mj, mn, pa = full.g
        ctx.predict_gaussians(full.uvw, l, m, s0, al, wl.ref_freq_hz, mj, mn, pa, ref, accumulate=True)
    if dw.s is not None:
        l, m, s0, al, b1, b2, pa, M, off, nc, pmax, n1, n2, cf = full.s
        ctx.predict_shapelets(full.uvw, l, m, s0, al, wl.ref_freq_hz, b1, b2, pa, M, off, nc, pmax, n1, n2, cf, ref, True)
    dirty = torch.full(full.uvw.vis_shape, float("nan"), dtype=torch.complex64, device="cuda:0")
    out = dw.predict(ctx, vis=dirty)
    torch.cuda.synchronize()
    assert torch.all(torch.isfinite(torch.view_as_real(out)))
    assert torch.max(torch.abs(out - ref)).item() < 2e-5
    if keep == "none":
        assert torch.all(out == 0)
    # the same through woden_simulate_host (its device buffer is whatever the previous call left there)
    if "points" not in keep: wl.points = inputs.empty_components()
    if "gaussians" not in keep: wl.gaussians = inputs.empty_components()
    if "shapelets" not in keep: wl.shapelets = inputs.empty_components()
    host = np.full((wl.n_times, wl.n_freqs, wl.n_baselines), np.nan, dtype=np.complex64)
    ctx.simulate_host(wl, host)
    assert np.array_equal(host, out.cpu().numpy())


def test_phase_centre_point_and_hermitian_symmetry_on_gpu(ctx, torch_mod):
    from paper_2005_09316_b200 import binding
    torch = torch_mod
    wl = inputs.make_config(1)
    for path in (0, 1):
        ctx.set_path(path)
        uvw = binding.Uvw(_dev(torch, wl.u_m), _dev(torch, wl.v_m), _dev(torch, wl.w_m), wl.freqs_hz)
        vis = ctx.new_vis(uvw)
        z = _dev(torch, [0.0])
        ctx.predict_points(uvw, z, z, _dev(torch, [2.0]), _dev(torch, [-0.8]), 150e6, vis)
        expect = 2.0 * (wl.freqs_hz / 150e6) ** -0.8
        got = vis.cpu().numpy()
        assert np.abs(got - expect[None, :, None]).max() < 2e-6 * 2.0      # P1: V = S everywhere
        a = _gpu_total(ctx, wl, path)
        wl2 = inputs.make_config(1)
        wl2.u_m, wl2.v_m, wl2.w_m = -wl.u_m, -wl.v_m, -wl.w_m
        b = _gpu_total(ctx, wl2, path)
        scale = oracle.workload_tolerance_scale(wl)[None, :, None]
        assert (np.abs(b - np.conj(a)) / scale).max() < TOL                  # P7


def test_simulate_host_matches_device_path(ctx):
    wl = inputs.make_config(1)
    ctx.set_path(0)
    out = np.empty((wl.n_times, wl.n_freqs, wl.n_baselines), dtype=np.complex64)
    ctx.simulate_host(wl, out)
    dev = _gpu_total(ctx, wl, 0)
    assert np.array_equal(out, dev)


def _host_vis(torch, wl, pinned):
    """NaN-filled complex64 host buffer [T][F][B]; page-locked (the tile-wise copy-back needs it) or pageable."""
    shape = (wl.n_times, wl.n_freqs, wl.n_baselines)
    if pinned:
        t = torch.empty(shape, dtype=torch.complex64, pin_memory=True)
        out = t.numpy()
        out[...] = np.nan
        return out, t
    return np.full(shape, np.nan, dtype=np.complex64), None


@pytest.mark.parametrize("pinned", [True, False], ids=["pinned", "pageable"])
@pytest.mark.parametrize("path", [0, 1], ids=["auto", "general"])
@pytest.mark.parametrize("last", ["shapelets", "gaussians", "points"])
def test_simulate_host_overlapped_copy_back_is_bit_identical(ctx, torch_mod, last, path, pinned):
    # woden_simulate_host hides the copy-back behind its LAST predictor (Gaussians, else points, else shapelets):
    # on the channel-walking path, into a page-locked buffer, tile by tile (12 channel tiles here, strided 2-D
    # copies); on the general path, for a shapelet-only sky and into pageable memory in chunks of time steps of
    # >= 64 MB of output (7 steps of config 5's grid are 175 MB -> 3 ragged chunks of 2, 2, 3 steps).  Either way the
    # result must equal the device path (the three calls in the same order) bit for bit, and the oracle on a
    # sampled subset.
    import dataclasses
    wl = inputs.make_config(5, n_times=7, n_times_total=7)
    keep = lambda c, n: type(c)(**{f.name: (None if getattr(c, f.name) is None else getattr(c, f.name)[:n])
                                   for f in dataclasses.fields(c)})
    wl.points = keep(wl.points, 300) if last != "shapelets" else inputs.empty_components()
    wl.gaussians = keep(wl.gaussians, 200) if last == "gaussians" else inputs.empty_components()
    ctx.set_path(path)
    out, _keep = _host_vis(torch_mod, wl, pinned)
    assert out.nbytes > 2 * (64 << 20)
    ctx.simulate_host(wl, out)
    dev = _gpu_total(ctx, wl, path)
    assert np.array_equal(out, dev)
    rng = np.random.default_rng(12)
    idx = np.unique(np.concatenate([rng.integers(0, wl.n_vis, 4000), [0, wl.n_vis - 1]])).astype(np.int64)
    ref = oracle.predict_workload(wl, vis_index=idx)
    scale = oracle.workload_tolerance_scale(wl)
    _assert_parity(out.reshape(-1)[idx], ref, scale, idx, wl, "simulate_host")


@pytest.mark.parametrize("pinned", [True, False], ids=["pinned", "pageable"])
def test_simulate_host_ragged_last_channel_tile(ctx, torch_mod, pinned):
    # tile-wise copy-back (page-locked buffer) with a ragged last tile: F = 75 -> tiles of 32, 32, 11 channels
    u, v, w, fr = _small_case(seed=5, T=3, B=300, F=75, uniform=True)
    wl = inputs.make_config(1)
    wl.u_m, wl.v_m, wl.w_m, wl.freqs_hz = u, v, w, fr
    wl.shapelets = inputs.empty_components()
    ctx.set_path(0)
    out, _keep = _host_vis(torch_mod, wl, pinned)
    ctx.simulate_host(wl, out)
    dev = _gpu_total(ctx, wl, 0)
    assert np.array_equal(out, dev)


def test_uvw_and_uv_basis_on_device_match_the_oracle(ctx, torch_mod):
    # antenna XYZ -> (u,v,w) once per time step and M_j (G4)
    from paper_2005_09316_b200 import binding
    torch = torch_mod
    X, Y, Z, H, d0 = inputs.make_antennas(5)
    u, v, w = ctx.uvw_from_antennas(_dev(torch, X), _dev(torch, Y), _dev(torch, Z), H, d0)
    torch.cuda.synchronize()
    ru, rv, rw = oracle.uvw_from_antennas(X, Y, Z, H, d0)
    assert u.shape == (56, 8128)
    for got, ref in ((u, ru), (v, rv), (w, rw)):
        assert np.abs(got.cpu().numpy() - ref).max() <= 1e-9          # metres, FP64 both sides
    wl = inputs.make_config(5)
    assert np.abs(ru - wl.u_m).max() <= 1e-9 and np.abs(rw - wl.w_m).max() <= 1e-9   # the configs' own uvw
    for n_ant in (2, 3, 5):                                            # pair indexing at tiny sizes
        g = ctx.uvw_from_antennas(_dev(torch, X[:n_ant]), _dev(torch, Y[:n_ant]), _dev(torch, Z[:n_ant]), H[:3], d0)
        r = oracle.uvw_from_antennas(X[:n_ant], Y[:n_ant], Z[:n_ant], H[:3], d0)
        assert all(np.abs(a.cpu().numpy() - b).max() <= 1e-9 for a, b in zip(g, r))
    s = wl.shapelets
    M = ctx.shapelet_uv_basis(_dev(torch, s.l), _dev(torch, s.m), d0)
    torch.cuda.synchronize(); ctx.check()
    assert np.abs(M.cpu().numpy() - oracle.shapelet_uv_basis(s.l, s.m, d0)).max() <= 1e-14
    # end to end: device-made uvw and M_j through the shapelet predictor, against the oracle chain
    wl1 = inputs.make_config(1)
    X, Y, Z, H, d0 = inputs.make_antennas(1)
    u, v, w = ctx.uvw_from_antennas(_dev(torch, X), _dev(torch, Y), _dev(torch, Z), H, d0)
    s = wl1.shapelets
    Md = ctx.shapelet_uv_basis(_dev(torch, s.l), _dev(torch, s.m), d0)
    uvw = binding.Uvw(u, v, w, wl1.freqs_hz)
    vis = ctx.new_vis(uvw)
    d = lambda a: _dev(torch, a)
    di = lambda a: _dev(torch, a, torch.int32)
    ctx.predict_shapelets(uvw, d(s.l), d(s.m), d(s.s0_jy), d(s.alpha), 150e6, d(s.beta1_rad), d(s.beta2_rad),
                          d(s.pa_rad), Md, di(s.coeff_offset), len(s.coeff), 5, di(s.n1), di(s.n2), d(s.coeff), vis)
    torch.cuda.synchronize(); ctx.check()
    ou, ov, ow = oracle.uvw_from_antennas(X, Y, Z, H, d0)
    ref = oracle.predict_shapelets(ou, ov, ow, wl1.freqs_hz, s.l, s.m, s.s0_jy, s.alpha, 150e6, s.beta1_rad,
                                   s.beta2_rad, s.pa_rad, oracle.shapelet_uv_basis(s.l, s.m, d0),
                                   s.coeff_offset, s.n1, s.n2, s.coeff)
    scale = oracle.tolerance_scale(wl1.freqs_hz, s.s0_jy, s.alpha, 150e6, s.coeff_offset, s.coeff)
    assert (np.abs(vis.cpu().numpy() - ref) / scale[None, :, None]).max() <= TOL
    # a direction outside the unit disk gets identity rows and is counted for woden_check
    Mb = ctx.shapelet_uv_basis(_dev(torch, [0.9]), _dev(torch, [0.9]), d0)
    assert np.array_equal(Mb.cpu().numpy(), [[1.0, 0, 0, 0, 1.0, 0]])
    with pytest.raises(binding.WodenError):
        ctx.check()


def test_error_codes_and_device_side_checks(ctx, torch_mod):
    from paper_2005_09316_b200 import binding
    torch = torch_mod
    wl = inputs.make_config(1)
    dw = binding.DeviceWorkload(wl)
    vis = ctx.new_vis(dw.uvw)
    l, m, s0, al = dw.p
    with pytest.raises(binding.WodenError) as e:
        ctx.predict_points(dw.uvw, l, None, s0, al, wl.ref_freq_hz, vis)
    assert e.value.status == binding.WODEN_ERR_NULL
    with pytest.raises(binding.WodenError) as e:
        ctx.predict_points(dw.uvw, l, m, s0, al, -1.0, vis)
    assert e.value.status == binding.WODEN_ERR_DIM
    sl, sm, ss0, sal, b1, b2, pa, M, off, nc, pmax, n1, n2, cf = dw.s
    with pytest.raises(binding.WodenError) as e:
        ctx.predict_shapelets(dw.uvw, sl, sm, ss0, sal, wl.ref_freq_hz, b1, b2, pa, M, off, nc, 101, n1, n2, cf, vis)
    assert e.value.status == binding.WODEN_ERR_ORDER
    bad = binding.Uvw(*dw.uvw.tensors, np.array([150e6, -1.0]))
    with pytest.raises(binding.WodenError) as e:
        ctx.predict_points(bad, l, m, s0, al, wl.ref_freq_hz, ctx.new_vis(bad))
    assert e.value.status == binding.WODEN_ERR_DIM
    # device-side preconditions: a component below the horizon is flagged by woden_check()
    ctx.check()
    lbad = l.clone(); lbad[0] = 0.9; mbad = m.clone(); mbad[0] = 0.9
    ctx.predict_points(dw.uvw, lbad, mbad, s0, al, wl.ref_freq_hz, vis)
    with pytest.raises(binding.WodenError) as e:
        ctx.check()
    assert e.value.status == binding.WODEN_ERR_DATA
    ctx.check()                                            # counter was reset
    # an order above the declared p_max is flagged too
    ctx.predict_shapelets(dw.uvw, sl, sm, ss0, sal, wl.ref_freq_hz, b1, b2, pa, M, off, nc, 3, n1, n2, cf, vis)
    with pytest.raises(binding.WodenError):
        ctx.check()


# ---------------------------------------------------------------------------------------------
# Round-2 edge cases of the point / Gaussian kernels: strongly resolved Gaussians, long baselines,
# and the channel lists that may (not) take the channel-walking path.

def _array_case(radius_m, T, B, F, f0_hz, step_hz, seed):
    rng = np.random.default_rng(seed)
    east, north = inputs.disk_antennas(rng, 40, radius_m)
    u, v, w = inputs.uvw_metres(east, north, T, 8.0)
    order = np.argsort(-(u[0] ** 2 + v[0] ** 2))            # keep the LONGEST baselines and a few short ones
    keep = np.concatenate([order[: B - 20], order[-20:]])
    u, v, w = (np.ascontiguousarray(a[:, keep]) for a in (u, v, w))
    return u, v, w, f0_hz + step_hz * np.arange(F)


@pytest.mark.parametrize("path", [0, 1], ids=["auto", "general"])
@pytest.mark.parametrize("radius_m", [1500.0, 2750.0], ids=["3km", "5.5km"])
@pytest.mark.parametrize("step_hz", [80e3, -80e3, 1.28e6, -1.28e6])
def test_wide_gaussians_on_long_baselines_are_finite_and_match(ctx, torch_mod, path, radius_m, step_hz):
    # Eq 12-14 with maj >= 0 as the header allows: FWHM from 0.5 to 20 degrees on
    # 3 km / 5.5 km arrays.  The envelope underflows to an exact 0 on the long baselines (the oracle's
    # exp() does the same); the channel-walking envelope recurrence must give 0 there, not 0 x inf.
    from paper_2005_09316_b200 import binding
    torch = torch_mod
    ctx.set_path(path)
    F = 40
    f0 = 167e6 if step_hz > 0 else 200e6
    u, v, w, fr = _array_case(radius_m, 2, 150, F, f0, step_hz, seed=int(radius_m))
    rng = np.random.default_rng(99)
    fwhm_deg = np.repeat([0.5, 1.5, 3.0, 6.0, 20.0], 4)
    n = len(fwhm_deg)
    maj = np.deg2rad(fwhm_deg)
    mnr = maj * np.tile([1.0, 0.5, 0.05, 0.0], 5)
    pa = rng.uniform(0, np.pi, n)
    l, m = inputs.disk_lm(rng, n, 10.0)
    s0 = inputs.log_uniform(rng, n, 0.5, 5.0) * rng.choice([-1.0, 1.0], n)
    al = rng.normal(-0.8, 0.2, n)
    uvw = binding.Uvw(_dev(torch, u), _dev(torch, v), _dev(torch, w), fr)
    d = lambda a: _dev(torch, a)
    worst = 0.0
    # each width class alone (a NaN or a wrong zero cannot hide behind other components), then all
    for sel in [np.arange(4 * i, 4 * i + 4) for i in range(5)] + [np.arange(n)]:
        vis = ctx.new_vis(uvw)
        ctx.predict_gaussians(uvw, d(l[sel]), d(m[sel]), d(s0[sel]), d(al[sel]), 150e6, d(maj[sel]), d(mnr[sel]),
                              d(pa[sel]), vis)
        torch.cuda.synchronize(); ctx.check()
        assert ctx.last_path() == (binding.WODEN_PATH_WALKING if path == 0 else binding.WODEN_PATH_GENERAL)
        V = vis.cpu().numpy()
        assert np.all(np.isfinite(V.view(np.float32)))
        ref = oracle.predict_gaussians(u, v, w, fr, l[sel], m[sel], s0[sel], al[sel], 150e6, maj[sel], mnr[sel], pa[sel])
        scale = oracle.tolerance_scale(fr, s0[sel], al[sel], 150e6)
        worst = max(worst, float((np.abs(V - ref) / scale[None, :, None]).max()))
    assert worst <= TOL
    # the case is what it claims: some envelopes are an exact zero, some visibilities are not
    assert np.abs(ref).min() < 1e-3 * np.abs(ref).max() and np.abs(ref).max() > 0.1


@pytest.mark.parametrize("path", [0, 1], ids=["auto", "general"])
def test_envelope_near_the_underflow_threshold(ctx, torch_mod, path):
    # exponents Q s^2 swept through the FP32 flush threshold (2^-126) along the baseline axis: the
    # walking envelope's seed flushes while neighbouring channels are still (barely) normal
    from paper_2005_09316_b200 import binding
    torch = torch_mod
    ctx.set_path(path)
    B, F = 400, 64
    fr = 150e6 + 1.0e6 * np.arange(F)
    u = np.linspace(50.0, 4000.0, B)[None, :].copy()
    v = np.zeros((1, B)); w = np.zeros((1, B))
    z = np.array([0.0])
    maj = np.array([np.deg2rad(0.25)])
    uvw = binding.Uvw(_dev(torch, u), _dev(torch, v), _dev(torch, w), fr)
    vis = ctx.new_vis(uvw)
    ctx.predict_gaussians(uvw, _dev(torch, z), _dev(torch, z), _dev(torch, [1.0]), _dev(torch, z), 150e6,
                          _dev(torch, maj), _dev(torch, maj), _dev(torch, z), vis)
    torch.cuda.synchronize(); ctx.check()
    V = vis.cpu().numpy()
    ref = oracle.predict_gaussians(u, v, w, fr, z, z, [1.0], z, 150e6, maj, maj, z)
    assert np.all(np.isfinite(V.view(np.float32)))
    assert np.abs(V - ref).max() <= TOL
    assert ref.real.min() < 1e-40 and ref.real.max() > 0.9          # spans the whole dynamic range


@pytest.mark.parametrize("path", [0, 1], ids=["auto", "general"])
@pytest.mark.parametrize("scale,f0", [(1.0e3, 180e6), (30.0, 10.0e9), (1.2e4, 1.4e9)],
                         ids=["3000km@180MHz", "90km@10GHz", "36000km@1.4GHz"])
def test_phase_hand_off_on_very_long_baselines(ctx, torch_mod, path, scale, f0):
    # up to ~2^28 wavelengths: 5e5 ... 2e8 turns of phase.  The Q0.32 hand-off of the walking path
    # shifts its fixed point per thread (phase.cuh); MAGIC23 of the general path holds to 2^28.
    from paper_2005_09316_b200 import binding
    torch = torch_mod
    ctx.set_path(path)
    u, v, w, fr = _array_case(1500.0, 2, 140, 37, f0, 80e3, seed=5)
    u, v, w = u * scale, v * scale, w * scale
    rng = np.random.default_rng(6)
    n = 30
    l, m = inputs.disk_lm(rng, n, 30.0)
    s0 = inputs.log_uniform(rng, n, 0.1, 10.0)
    al = rng.normal(-0.8, 0.2, n)
    uvw = binding.Uvw(_dev(torch, u), _dev(torch, v), _dev(torch, w), fr)
    vis = ctx.new_vis(uvw)
    ctx.predict_points(uvw, _dev(torch, l), _dev(torch, m), _dev(torch, s0), _dev(torch, al), 150e6, vis)
    torch.cuda.synchronize(); ctx.check()
    assert ctx.last_path() == (binding.WODEN_PATH_WALKING if path == 0 else binding.WODEN_PATH_GENERAL)
    wavelengths = np.sqrt(u * u + v * v + w * w).max() * fr.max() / inputs.C_LIGHT
    assert 2.0 ** 19 < wavelengths * 0.5 and np.sqrt(2.0) * wavelengths < 2.0 ** 28
    ref = oracle.predict_points(u, v, w, fr, l, m, s0, al, 150e6)
    sc = oracle.tolerance_scale(fr, s0, al, 150e6)
    assert (np.abs(vis.cpu().numpy() - ref) / sc[None, :, None]).max() <= TOL


@pytest.mark.parametrize("path", [0, 1], ids=["auto", "general"])
def test_baselines_beyond_the_phase_range_are_reported(ctx, torch_mod, path):
    from paper_2005_09316_b200 import binding
    torch = torch_mod
    ctx.set_path(path)
    u, v, w, fr = _array_case(1500.0, 1, 64, 16, 180e6, 80e3, seed=5)
    u = u * 4.0e5                                          # ~1e9 m at 180 MHz: > 2^28 wavelengths
    uvw = binding.Uvw(_dev(torch, u), _dev(torch, v), _dev(torch, w), fr)
    vis = ctx.new_vis(uvw)
    ctx.check()
    ctx.predict_points(uvw, _dev(torch, [0.01]), _dev(torch, [0.02]), _dev(torch, [1.0]), _dev(torch, [0.0]), 150e6, vis)
    with pytest.raises(binding.WodenError) as e:
        ctx.check()
    assert e.value.status == binding.WODEN_ERR_DATA
    ctx.check()


def test_which_channel_lists_take_the_walking_path(ctx, torch_mod):
    # woden_b200.h, woden_set_path: an arithmetic progression of >= 8 channels with step <= 1/64 of
    # the lowest (padded) frequency walks; everything else is the general path.  The advisor's case:
    # [100, 150, 200] MHz and a Gaussian whose envelope is 2^-7 at 100 MHz must not come out as 0.
    from paper_2005_09316_b200 import binding
    torch = torch_mod
    ctx.set_path(0)
    z = np.array([0.0])
    cases = [
        (167e6 + 80e3 * np.arange(16), True),
        (167e6 + 80e3 * np.arange(8), True),
        (167e6 + 80e3 * np.arange(7), False),                    # too short
        (np.array([100e6, 150e6, 200e6]), False),
        (100e6 + 50e6 * np.arange(9), False),                    # uniform but far too wide
        (200e6 - 1.28e6 * np.arange(40), True),
        (200e6 - 3.0e6 * np.arange(40), False),                  # continuation to 64 channels is too low
        (167e6 + 80e3 * np.arange(16) ** 1.01, False),           # not equally spaced
    ]
    cg = np.pi / (2.0 * np.log(2.0))
    for fr, walks in cases:
        s_lo = fr.min() / inputs.C_LIGHT
        ub = np.array([[30.0, 400.0, 2500.0]])
        # circular Gaussian with envelope exactly 2^-7 on the 400 m baseline at the lowest frequency
        maj = np.array([np.sqrt(7.0) / (cg * 400.0 * s_lo)])
        uvw = binding.Uvw(_dev(torch, ub), _dev(torch, 0 * ub), _dev(torch, 0 * ub), fr)
        vis = ctx.new_vis(uvw)
        ctx.predict_gaussians(uvw, _dev(torch, z), _dev(torch, z), _dev(torch, [1.0]), _dev(torch, z), 150e6,
                              _dev(torch, maj), _dev(torch, maj), _dev(torch, z), vis)
        torch.cuda.synchronize(); ctx.check()
        assert (ctx.last_path() == binding.WODEN_PATH_WALKING) == walks, fr[:3]
        ref = oracle.predict_gaussians(ub, 0 * ub, 0 * ub, fr, z, z, [1.0], z, 150e6, maj, maj, z)
        V = vis.cpu().numpy()
        assert np.abs(V - ref).max() <= TOL
        f_lo = int(np.argmin(fr))
        assert abs(ref[0, f_lo, 1].real - 2.0 ** -7) < 1e-9 and abs(V[0, f_lo, 1].real - 2.0 ** -7) < 1e-6


def test_non_finite_flux_at_any_channel_is_reported(ctx, torch_mod):
    # s0 (nu/ref)^alpha overflows FP32 only at the upper channels: still counted (woden_check)
    from paper_2005_09316_b200 import binding
    torch = torch_mod
    ctx.set_path(0)
    u, v, w, _ = _small_case(seed=1, T=1, B=64, F=16)
    fr = 150e6 * (1.0 + 0.01 * np.arange(1, 17))
    uvw = binding.Uvw(_dev(torch, u), _dev(torch, v), _dev(torch, w), fr)
    vis = ctx.new_vis(uvw)
    al = np.array([np.log(3.0e38) / np.log(fr[8] / 150e6)])       # S(nu_8) ~ 3e38, S(nu_9 ...) > FLT_MAX
    ctx.check()
    ctx.predict_points(uvw, _dev(torch, [0.0]), _dev(torch, [0.0]), _dev(torch, [1.0]), _dev(torch, al), 150e6, vis)
    with pytest.raises(binding.WodenError) as e:
        ctx.check()
    assert e.value.status == binding.WODEN_ERR_DATA
