"""Seeded synthetic inputs for the five BASELINE.json configs.

This module holds NONE of the method's arithmetic (no phase, envelope, flux law or
Hermite evaluation).  It only draws array layouts, observation geometry and sky-model
parameters, and returns plain float64 numpy arrays.  It is the one module that both the
CUDA path (via the binding) and the oracle (via the tests) are fed from, so RNG details
never affect parity.

The paper's own workloads (MWA phase I/II layouts, the VLA Fornax A image, WSClean and
SHAMFI model files: PAPER.md:169-183, :269-271) are not available; these inputs stand in
for them with the same shapes (~3 km array :171; 8 s x 80 kHz cadence :201; 30.72 MHz
band :171; 56 time steps :179; two shapelet lobes :189; point:Gaussian = 4540:1791 :269).

Recipe (also stated in DESIGN.md):
  rng      = numpy.random.Generator(numpy.random.PCG64(200509316 + config))
  antennas : (E, N) = r (sin psi, cos psi), r = R sqrt(U), psi = 2 pi U, Up = 0
  uvw      : textbook XYZ -> uvw rotation (Thompson, Moran & Swenson; cited PAPER.md:110),
             sidereal rate 2 pi / 86164.0905 rad/s, latitude -26.7 deg, Dec0 = -37 deg,
             hour angles centred on 0
  channels : 167 MHz + f * 80 kHz, reference frequency 150 MHz
  (l, m)   : uniform on a disk of radius sin(rho) in the l-m plane
  fluxes   : log-uniform, alpha ~ N(-0.8, 0.2)
Draw order inside each config is exactly the order of the code below.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, Optional

import numpy as np

SEED_BASE = 200509316
C_LIGHT = 299792458.0
SIDEREAL_DAY_S = 86164.0905
LATITUDE_DEG = -26.7
DEC0_DEG = -37.0
FREQ0_HZ = 167.0e6
CHAN_WIDTH_HZ = 80.0e3
REF_FREQ_HZ = 150.0e6
ARCMIN = np.pi / (180.0 * 60.0)

CONFIG_NAMES = {
    1: "Tiny",
    2: "Point-source sky",
    3: "Gaussian-heavy sky",
    4: "Fornax-A-like shapelet model",
    5: "Full-band mixed sky",
    6: "Phase-II-like shapelet model (extra: SURVEY.md 8(f) NEXT-2)",
    7: "Phase-II-like point / Gaussian sky (extra: parity case on 5.5 km baselines)",
}


@dataclass
class Components:
    """One component type, struct-of-arrays, float64.  Empty arrays mean 'none'."""
    l: np.ndarray
    m: np.ndarray
    s0_jy: np.ndarray
    alpha: np.ndarray
    # Gaussians only
    maj_fwhm_rad: Optional[np.ndarray] = None
    min_fwhm_rad: Optional[np.ndarray] = None
    # Gaussians and shapelets
    pa_rad: Optional[np.ndarray] = None
    # shapelets only
    beta1_rad: Optional[np.ndarray] = None
    beta2_rad: Optional[np.ndarray] = None
    uv_basis: Optional[np.ndarray] = None      # [n, 6] row-major 2x3 (reading G4)
    coeff_offset: Optional[np.ndarray] = None  # [n + 1] int32 CSR offsets
    n1: Optional[np.ndarray] = None            # int32
    n2: Optional[np.ndarray] = None            # int32
    coeff: Optional[np.ndarray] = None         # float64

    @property
    def n(self) -> int:
        return int(self.l.shape[0])


@dataclass
class Workload:
    config: int
    name: str
    u_m: np.ndarray          # [T, B] metres
    v_m: np.ndarray
    w_m: np.ndarray
    freqs_hz: np.ndarray     # [F]
    ref_freq_hz: float
    points: Components
    gaussians: Components
    shapelets: Components
    meta: Dict = field(default_factory=dict)

    @property
    def n_times(self) -> int:
        return int(self.u_m.shape[0])

    @property
    def n_baselines(self) -> int:
        return int(self.u_m.shape[1])

    @property
    def n_freqs(self) -> int:
        return int(self.freqs_hz.shape[0])

    @property
    def n_vis(self) -> int:
        return self.n_times * self.n_baselines * self.n_freqs

    @property
    def n_coeff(self) -> int:
        return 0 if self.shapelets.n == 0 else int(self.shapelets.coeff_offset[-1])


def empty_components() -> Components:
    z = np.zeros(0, dtype=np.float64)
    return Components(l=z, m=z.copy(), s0_jy=z.copy(), alpha=z.copy())


# --------------------------------------------------------------------------- geometry

def disk_antennas(rng: np.random.Generator, n: int, radius_m: float):
    r = radius_m * np.sqrt(rng.random(n))
    psi = 2.0 * np.pi * rng.random(n)
    return r * np.sin(psi), r * np.cos(psi)          # East, North


def baseline_pairs(n_ant: int):
    p, q = np.triu_indices(n_ant, k=1)               # all p < q, p-major
    return p, q


def uvw_metres(east, north, n_times: int, dt_s: float, t_index0: int = 0,
               n_times_total: Optional[int] = None):
    """[T, B] u, v, w in metres for all pairs p<q (baseline = antenna p - antenna q).

    `t_index0` / `n_times_total` let a rank of a sharded run generate
    its own slice of one longer observation: hour angles are centred on the whole
    observation, H_t = (t_index0 + t - (n_times_total - 1)/2) dt * 2 pi / sidereal day.
    """
    if n_times_total is None:
        n_times_total = n_times
    lat = np.deg2rad(LATITUDE_DEG)
    dec0 = np.deg2rad(DEC0_DEG)
    p, q = baseline_pairs(len(east))
    be = east[p] - east[q]
    bn = north[p] - north[q]
    X = -bn * np.sin(lat)
    Y = be
    Z = bn * np.cos(lat)
    t = np.arange(n_times, dtype=np.float64) + t_index0
    H = (t - (n_times_total - 1) / 2.0) * dt_s * 2.0 * np.pi / SIDEREAL_DAY_S
    sH, cH = np.sin(H)[:, None], np.cos(H)[:, None]
    sd, cd = np.sin(dec0), np.cos(dec0)
    u = sH * X + cH * Y
    v = -sd * cH * X + sd * sH * Y + cd * Z
    w = cd * cH * X - cd * sH * Y + sd * Z
    return (np.ascontiguousarray(u), np.ascontiguousarray(v), np.ascontiguousarray(w))


def channel_freqs(n_freqs: int) -> np.ndarray:
    return FREQ0_HZ + CHAN_WIDTH_HZ * np.arange(n_freqs, dtype=np.float64)


def disk_lm(rng: np.random.Generator, n: int, radius_deg: float):
    r = np.sin(np.deg2rad(radius_deg)) * np.sqrt(rng.random(n))
    psi = 2.0 * np.pi * rng.random(n)
    return r * np.sin(psi), r * np.cos(psi)


def log_uniform(rng: np.random.Generator, n: int, lo: float, hi: float):
    return 10.0 ** rng.uniform(np.log10(lo), np.log10(hi), n)


def local_uv_basis(l, m, dec0_rad: float = np.deg2rad(DEC0_DEG)) -> np.ndarray:
    """[n, 6] rows (e_x, e_y, e_z, n_x, n_y, n_z): local East and North unit vectors at
    direction s = (l, m, n) expressed in the phase-centre (u, v, w) frame (reading G4,
    SURVEY.md §8(c); PAPER.md:157 'visibility co-ordinates ... calculated with a
    phase-centre ... which corresponds to the central position').  e = (p x s)/|p x s|,
    n = s x e, with p = (0, cos dec0, sin dec0) the celestial pole."""
    l = np.atleast_1d(np.asarray(l, dtype=np.float64))
    m = np.atleast_1d(np.asarray(m, dtype=np.float64))
    s = np.stack([l, m, np.sqrt(1.0 - l * l - m * m)], axis=1)
    p = np.array([0.0, np.cos(dec0_rad), np.sin(dec0_rad)])
    e = np.cross(np.broadcast_to(p, s.shape), s)
    e /= np.linalg.norm(e, axis=1, keepdims=True)
    nn = np.cross(s, e)
    return np.ascontiguousarray(np.concatenate([e, nn], axis=1))


def full_triangle(p_max: int):
    """All (n1, n2) with n1 + n2 <= p_max in n1-major order (Eq 6 count)."""
    n1 = [a for a in range(p_max + 1) for _ in range(p_max + 1 - a)]
    n2 = [b for a in range(p_max + 1) for b in range(p_max + 1 - a)]
    return np.asarray(n1, dtype=np.int32), np.asarray(n2, dtype=np.int32)


def basis_count(p_max: int) -> int:
    return (p_max + 2) * (p_max + 1) // 2


# --------------------------------------------------------------------------- components

def _points(rng, n, radius_deg, flux_lo, flux_hi) -> Components:
    l, m = disk_lm(rng, n, radius_deg)
    s0 = log_uniform(rng, n, flux_lo, flux_hi)
    alpha = rng.normal(-0.8, 0.2, n)
    return Components(l=l, m=m, s0_jy=s0, alpha=alpha)


def _gaussians(rng, n, radius_deg, flux_lo, flux_hi, maj_lo_arcmin, maj_hi_arcmin) -> Components:
    c = _points(rng, n, radius_deg, flux_lo, flux_hi)
    c.maj_fwhm_rad = log_uniform(rng, n, maj_lo_arcmin, maj_hi_arcmin) * ARCMIN
    c.min_fwhm_rad = c.maj_fwhm_rad * rng.uniform(0.2, 1.0, n)
    c.pa_rad = rng.uniform(0.0, np.pi, n)
    return c


def _shapelets(rng, l, m, p_max, beta_lo_arcmin, beta_hi_arcmin, beta_fixed_arcmin=None) -> Components:
    n = len(l)
    if beta_fixed_arcmin is not None:
        b1 = np.full(n, beta_fixed_arcmin * ARCMIN)
        b2 = b1.copy()
    else:
        b1 = rng.uniform(beta_lo_arcmin, beta_hi_arcmin, n) * ARCMIN
        b2 = rng.uniform(beta_lo_arcmin, beta_hi_arcmin, n) * ARCMIN
    pa = rng.uniform(0.0, np.pi, n)
    t1, t2 = full_triangle(p_max)
    P = len(t1)
    n1 = np.tile(t1, n)
    n2 = np.tile(t2, n)
    coeff = rng.normal(0.0, 1.0, n * P) * np.exp(-(n1 + n2) / 10.0)
    off = (np.arange(n + 1, dtype=np.int64) * P).astype(np.int32)
    return Components(l=np.asarray(l, dtype=np.float64), m=np.asarray(m, dtype=np.float64),
                      s0_jy=np.ones(n), alpha=np.full(n, -0.8),
                      beta1_rad=b1, beta2_rad=b2, pa_rad=pa,
                      uv_basis=local_uv_basis(l, m), coeff_offset=off,
                      n1=n1.astype(np.int32), n2=n2.astype(np.int32), coeff=coeff)


def _array(rng, which: str):
    if which == "A32":
        return disk_antennas(rng, 32, 500.0)
    e1, n1 = disk_antennas(rng, 64, 100.0)
    e2, n2 = disk_antennas(rng, 64, 2750.0 if which == "A128L" else 1500.0)
    return np.concatenate([e1, e2]), np.concatenate([n1, n2])


_OBS = {  # config: (array, T, dt_s, F)
    1: ("A32", 1, 8.0, 16),
    2: ("A128", 14, 8.0, 32),
    3: ("A128", 14, 8.0, 32),
    4: ("A128", 14, 8.0, 384),
    5: ("A128", 56, 2.0, 384),
    # not a BASELINE.json config: the 5.5 km phase II-like array with the paper's p_max = 86 lobes
    # (PAPER.md:171, :183), the sixth case SURVEY.md 8(f) NEXT-2 suggests
    6: ("A128L", 14, 8.0, 384),
    # not a BASELINE.json config: points and Gaussians on the same 5.5 km array, where the phase budget
    # of the channel-walking path is tightest; a parity case only
    7: ("A128L", 4, 8.0, 96),
}


def make_antennas(config: int, *, t_index0: int = 0, n_times_total: Optional[int] = None,
                  n_times: Optional[int] = None):
    """Antenna positions and hour angles behind config 1..5's u_m, v_m, w_m: local equatorial
    (X, Y, Z) in metres [n_ant], hour angles [T] in radians, and the phase-centre declination --
    the inputs of woden_uvw_from_antennas.  Same draws as make_config."""
    if config not in _OBS:
        raise ValueError(f"config must be 1..7, got {config}")
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + config))
    arr, T, dt, _ = _OBS[config]
    if n_times is None:
        n_times = T
    if n_times_total is None:
        n_times_total = max(T, n_times)
    east, north = _array(rng, arr)
    lat = np.deg2rad(LATITUDE_DEG)
    t = np.arange(n_times, dtype=np.float64) + t_index0
    H = (t - (n_times_total - 1) / 2.0) * dt * 2.0 * np.pi / SIDEREAL_DAY_S
    return -north * np.sin(lat), east.copy(), north * np.cos(lat), H, np.deg2rad(DEC0_DEG)


def make_config_shape(config: int):
    """(array name, T, dt_s, F) of config 1..5 without generating it."""
    if config not in _OBS:
        raise ValueError(f"config must be 1..7, got {config}")
    return _OBS[config]


def make_config(config: int, *, t_index0: int = 0, n_times_total: Optional[int] = None,
                n_times: Optional[int] = None) -> Workload:
    """Build config 1..5.  `n_times`/`t_index0`/`n_times_total` select a time shard of a
    longer observation with the same sky and array (weak-scaling ranks);
    the defaults give the config exactly as BASELINE.json words it."""
    if config not in _OBS:
        raise ValueError(f"config must be 1..7, got {config}")
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + config))
    arr, T, dt, F = _OBS[config]
    if n_times is None:
        n_times = T
    east, north = _array(rng, arr)
    u, v, w = uvw_metres(east, north, n_times, dt, t_index0,
                         n_times_total if n_times_total is not None else max(T, n_times))
    freqs = channel_freqs(F)

    pts, gau, shp = empty_components(), empty_components(), empty_components()
    if config == 1:
        pts = _points(rng, 10, 5.0, 0.1, 10.0)
        gau = _gaussians(rng, 2, 5.0, 0.1, 10.0, 2.0, 10.0)
        sl, sm = disk_lm(rng, 1, 5.0)
        shp = _shapelets(rng, sl, sm, 5, None, None, beta_fixed_arcmin=5.0)
    elif config == 2:
        pts = _points(rng, 1000, 20.0, 0.1, 10.0)
    elif config == 3:
        gau = _gaussians(rng, 10000, 20.0, 0.01, 5.0, 1.0, 30.0)
    elif config == 4:
        cl = np.array([-np.sin(np.deg2rad(0.25)), np.sin(np.deg2rad(0.25))])
        cm = np.zeros(2)
        shp = _shapelets(rng, cl, cm, 60, 5.0, 20.0)
        n_tot, n_pt = 20000, 14340            # 4540 : 1791 ratio
        which = rng.integers(0, 2, n_tot)
        dl, dm = disk_lm(rng, n_tot, 1.0)
        l = cl[which] + dl
        m = cm[which] + dm
        s0 = log_uniform(rng, n_tot, 0.01, 5.0)
        s0 = np.where(rng.random(n_tot) < 0.25, -s0, s0)   # MS CLEAN components may be negative, :277
        alpha = rng.normal(-0.8, 0.2, n_tot)
        maj = rng.uniform(0.0, 10.0, n_tot - n_pt) * ARCMIN
        mnr = maj * rng.uniform(0.2, 1.0, n_tot - n_pt)
        pa = rng.uniform(0.0, np.pi, n_tot - n_pt)
        pts = Components(l=l[:n_pt].copy(), m=m[:n_pt].copy(), s0_jy=s0[:n_pt].copy(),
                         alpha=alpha[:n_pt].copy())
        gau = Components(l=l[n_pt:].copy(), m=m[n_pt:].copy(), s0_jy=s0[n_pt:].copy(),
                         alpha=alpha[n_pt:].copy(), maj_fwhm_rad=maj, min_fwhm_rad=mnr, pa_rad=pa)
    elif config == 6:
        cl = np.array([-np.sin(np.deg2rad(0.25)), np.sin(np.deg2rad(0.25))])
        shp = _shapelets(rng, cl, np.zeros(2), 86, 5.0, 20.0)
    elif config == 7:
        pts = _points(rng, 1500, 25.0, 0.01, 10.0)
        gau = _gaussians(rng, 700, 25.0, 0.01, 10.0, 0.5, 30.0)
    elif config == 5:
        pts = _points(rng, 8000, 25.0, 0.01, 10.0)
        gau = _gaussians(rng, 2000, 25.0, 0.01, 10.0, 1.0, 30.0)
        sl, sm = disk_lm(rng, 4, 25.0)
        shp = _shapelets(rng, sl, sm, 40, 5.0, 20.0)

    return Workload(config=config, name=CONFIG_NAMES[config], u_m=u, v_m=v, w_m=w,
                    freqs_hz=freqs, ref_freq_hz=REF_FREQ_HZ, points=pts, gaussians=gau,
                    shapelets=shp,
                    meta={"array": arr, "dt_s": dt, "t_index0": t_index0, "dec0_rad": float(np.deg2rad(DEC0_DEG)),
                          "seed": SEED_BASE + config})


def subset_indices(wl: Workload, n_random: int = 1 << 20) -> np.ndarray:
    """Declared seeded visibility subset for configs too large for the oracle (SURVEY.md
    §8(d)): every baseline of the first and last time step at the first, middle and last
    channel, plus `n_random` flat indices drawn uniformly (seed = config seed + 1000).
    Flat index = (t * F + f) * B + b.  Returned sorted and unique, int64."""
    T, F, B = wl.n_times, wl.n_freqs, wl.n_baselines
    idx = []
    for t in sorted({0, T - 1}):
        for f in sorted({0, F // 2, F - 1}):
            idx.append((t * F + f) * B + np.arange(B, dtype=np.int64))
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + wl.config + 1000))
    idx.append(rng.integers(0, T * F * B, size=min(n_random, T * F * B), dtype=np.int64))
    return np.unique(np.concatenate(idx))


def time_shard(n_times_total: int, rank: int, world: int):
    """Contiguous split of time steps over ranks (shard the OUTPUT by time
    step, replicate components; no collective).  Returns (t_index0, n_times_local)."""
    base, rem = divmod(n_times_total, world)
    n_local = base + (1 if rank < rem else 0)
    t0 = rank * base + min(rank, rem)
    return t0, n_local
