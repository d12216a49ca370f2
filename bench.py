#!/usr/bin/env python
"""bench.py -- throughput of the WODEN hot path (points + Gaussians + shapelets) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 5]

One "step" = one pass of the whole hot path over one workload: woden_predict_shapelets,
woden_predict_points and woden_predict_gaussians (the first non-empty type overwrites the
buffer, the others accumulate) on config 5
("Full-band mixed sky", the largest BASELINE.json config; 1.75e8 visibilities, 8000 points,
2000 Gaussians, 4 shapelets of 861 coefficients), inputs resident in HBM.  Prints ONE JSON
line (rank 0).  See DESIGN.md "Measurement" for the definitions of every field.

--impl reference times the CPU oracle (oracle/, plain FP64 C, as it stands) on a bounded
seeded sample of the same workload per step; it is a deliberately slow program, reported as a
baseline, not a target.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2005_09316_b200 import inputs  # noqa: E402

METRIC = "component_x_visibility_evals_per_s"
UNIT = "evals/s"
SM_COUNT = 148
MUFU_LANES_PER_SM = 16          # measured: profiles/pipes_r1.md
FP32_LANES_PER_SM = 128
SM_MAX_HZ = 1965e6
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel on config 5, recorded
# from the ncu --set full captures summarised in profiles/ncu_r3_kernels.md (not measured in this run):
# (component type, path) -> (kernel, bytes, commit the capture was taken at)
NCU_DRAM_BYTES = {
    ("points", "walk"): ("predict_walk_kernel<false>", 11120384 + 66082048, "13aa7d5"),
    ("gaussians", "walk"): ("predict_walk_kernel<true>", 10993408 + 70302464, "13aa7d5"),
}
KERNEL_NAMES = {("points", "walk"): "predict_walk_kernel<false>", ("gaussians", "walk"): "predict_walk_kernel<true>",
                ("points", "general"): "predict_pg_kernel<16, false>", ("gaussians", "general"): "predict_pg_kernel<16, true>",
                ("shapelets", "walk"): "predict_shapelets_mma_kernel", ("shapelets", "general"): "predict_shapelets_mma_kernel"}


def _env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


def workload_counts(wl):
    nv = wl.n_vis
    return {
        "n_vis": nv,
        "points": nv * wl.points.n,
        "gaussians": nv * wl.gaussians.n,
        "shapelets": nv * wl.shapelets.n,
        "shapelet_coeffs": nv * wl.n_coeff,
    }


def config_dict(wl, extra=None):
    d = {
        "workload": f"config {wl.config}: {wl.name}",
        "n_baselines": wl.n_baselines, "n_times": wl.n_times, "n_freqs": wl.n_freqs,
        "n_vis": wl.n_vis, "n_points": wl.points.n, "n_gaussians": wl.gaussians.n,
        "n_shapelets": wl.shapelets.n, "n_shapelet_coeffs": wl.n_coeff,
        "eval_unit": "one sky component (point, Gaussian or whole shapelet) at one visibility",
    }
    if extra:
        d.update(extra)
    return d


# ------------------------------------------------------------------------------ clocks
class ClockSampler:
    """nvidia-smi clock / throttle-reason sampler running during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx = gpu_index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.idx}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        try:
            self.proc.terminate()
            self.proc.wait(timeout=5)
        except Exception:
            pass
        try:
            rows = [r.strip().split(",") for r in open(self.path) if r.strip()]
            os.unlink(self.path)
        except Exception:
            return out
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); power.append(float(r[2]))
                for n, v in zip(names, r[3:7]):
                    if v.strip().lower().startswith("active"):
                        reasons.add(n)
            except (ValueError, IndexError):
                continue
        if sm:
            busy = sorted(sm)[len(sm) // 2:]          # upper half = samples under load
            out.update(sm_mhz=float(np.median(busy)), sm_max_mhz=max(mx), reasons=sorted(reasons),
                       samples=len(sm), power_w_max=max(power))
        return out


# ------------------------------------------------------------------------------ reference arm
def oracle_sample_indices(wl, n, seed_off):
    rng = np.random.Generator(np.random.PCG64(inputs.SEED_BASE + wl.config + seed_off))
    return np.sort(rng.integers(0, wl.n_vis, size=n, dtype=np.int64))


def time_oracle(wl, n_vis_sample, seed_off):
    import oracle
    idx = oracle_sample_indices(wl, n_vis_sample, seed_off)
    t0 = time.perf_counter()
    oracle.predict_workload(wl, vis_index=idx)
    dt = time.perf_counter() - t0
    comps = wl.points.n + wl.gaussians.n + wl.shapelets.n
    return n_vis_sample * comps / dt, dt


def run_reference(args):
    rank = _env_int("RANK", 0)
    if rank != 0:
        return 0
    wl = inputs.make_config(args.config)
    cores = len(os.sched_getaffinity(0))
    # torchrun exports OMP_NUM_THREADS=1 to its ranks; the oracle's protocol is all cores of the
    # affinity mask (libgomp reads the variable when the oracle library is loaded, below)
    os.environ["OMP_NUM_THREADS"] = str(cores)
    n_sample = 1 << 14
    for i in range(args.warmup):
        time_oracle(wl, max(256, n_sample // 16), 5000 + i)
    t_tot, evals = 0.0, 0.0
    for i in range(args.steps):
        v, dt = time_oracle(wl, n_sample, 6000 + i)
        t_tot += dt
        evals += v * dt
    value = evals / t_tot
    sample = (f"{n_sample} seeded random visibilities of config {wl.config} per step, all "
              f"{wl.points.n + wl.gaussians.n + wl.shapelets.n} components each")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_tot / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": config_dict(wl, {"sample": sample}),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------ multi-GPU launch
def spawn_ranks_if_needed(args):
    """`python bench.py --gpus N` with no torchrun environment: start N ranks ourselves (one per GPU,
    NCCL rendezvous on 127.0.0.1) by re-executing this script under torch.distributed.run.  Under
    torchrun (WORLD_SIZE set) this is a no-op and the ranks read RANK / LOCAL_RANK / WORLD_SIZE."""
    if args.gpus <= 1 or "WORLD_SIZE" in os.environ:
        return
    import socket
    with socket.socket() as sock:
        sock.bind(("127.0.0.1", 0))
        port = sock.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    os.execv(sys.executable, cmd)


def run_dry(args):
    """Rendezvous only (gloo, no GPU): every rank joins, the world size is all-reduced, rank 0 prints it.
    Used by the CPU test of the --gpus N launch path."""
    import torch
    import torch.distributed as dist
    rank, world = _env_int("RANK", 0), _env_int("WORLD_SIZE", 1)
    if world > 1:
        dist.init_process_group("gloo")
        t = torch.ones(1)
        dist.all_reduce(t)
        seen = int(t.item())
        dist.destroy_process_group()
    else:
        seen = 1
    if rank == 0:
        print(json.dumps({"dry": True, "n_gpus": seen, "requested": args.gpus}))
    return 0


# order in which step() runs the three predictors between its four event marks (the first non-empty type
# overwrites the buffer; the channel-walking calls come last so that copy-back can hide under them)
STEP_ORDER = (("shapelets", 0, 1), ("points", 1, 2), ("gaussians", 2, 3))


def split_marks(recs):
    """Per-type call durations (ms) of every recorded step: {type: [ms, ...]} from the four marks of each
    step, labelled by STEP_ORDER (the ONE place that maps marks to predictor names)."""
    out = {name: [] for name, _, _ in STEP_ORDER}
    for marks in recs:
        for name, a, b in STEP_ORDER:
            out[name].append(float(marks[a].elapsed_time(marks[b])))
    return out


def general_path_record(general_ms, counts, mufu_rate, t_roof, world, evals_per_step, steps):
    """The SURVEY.md 8(d) rule (ii) block of the JSON line from the general path's per-type times."""
    rec = {"ms_per_step": general_ms["step"], "value": world * evals_per_step / (general_ms["step"] * 1e-3),
           "per_type": {}, "steps": steps, "warmup": 3}
    mufu_ops = {"points": 2, "gaussians": 3}
    for k in ("points", "gaussians", "shapelets"):
        if counts[k] and general_ms.get(k):
            r = {"ms_per_call": general_ms[k], "min_ms_per_call": general_ms.get(k + "_min"),
                 "evals_per_s": counts[k] / (general_ms[k] * 1e-3)}
            if k in mufu_ops:
                r["frac_of_mufu_roofline"] = r["evals_per_s"] / (mufu_rate / mufu_ops[k])
            rec["per_type"][k] = r
    rec["composite_frac"] = 1e3 * t_roof / general_ms["step"]
    # a kernel that issues 2 (3) MUFU per eval cannot beat the MUFU pipe: a fraction far above 1 means the
    # marks were mapped to the wrong predictor
    rec["labels_consistent"] = all(r.get("frac_of_mufu_roofline", 0.0) <= 1.10 for r in rec["per_type"].values())
    rec["note"] = ("woden_set_path(GENERAL): 2 MUFU per point eval, 3 per Gaussian eval; fractions are of the "
                   "MUFU-pipe roofline at the pipe rate measured in this run")
    return rec


def time_steps(step, n_warm, n_steps, barrier):
    """n_warm untimed + n_steps timed calls of step(record) between barriers; returns (ms_total, records)."""
    import torch
    for _ in range(n_warm):
        step(None)
    barrier()
    recs = []
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(n_steps):
        step(recs)
    e1.record()
    barrier()
    return e0.elapsed_time(e1), recs


# ------------------------------------------------------------------------------ our arm
def run_ours(args):
    import torch
    from paper_2005_09316_b200 import binding, parallel

    rank, world = _env_int("RANK", 0), _env_int("WORLD_SIZE", 1)
    local = _env_int("LOCAL_RANK", 0)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference "
                         "for the oracle baseline)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    # weak scaling: every rank predicts the config's T time steps of one
    # longer observation with the same sky; shards are disjoint in time, no data-path collective
    wl = parallel.rank_workload(args.config, rank, world, scaling="weak")
    ctx = binding.Woden(local)
    ctx.set_path(binding.WODEN_PATH_GENERAL if args.path == "general" else binding.WODEN_PATH_AUTO)
    dw = binding.DeviceWorkload(wl, device=f"cuda:{local}", ctx=ctx)
    vis = ctx.new_vis(dw.uvw)
    counts = workload_counts(wl)
    comps = wl.points.n + wl.gaussians.n + wl.shapelets.n
    evals_per_step = counts["n_vis"] * comps

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    ev = lambda: torch.cuda.Event(enable_timing=True)
    per_type_ms = {"points": [], "gaussians": [], "shapelets": []}

    def step(record):
        marks = [ev() for _ in range(4)]
        marks[0].record()
        # shapelets, points, Gaussians (the order of DeviceWorkload.predict and woden_simulate_host); the first
        # non-empty component type overwrites vis, the others accumulate
        written = False
        if dw.s is not None:
            l, m, s0, al, b1, b2, pa, M, off, nc, pmax, n1, n2, cf = dw.s
            ctx.predict_shapelets(dw.uvw, l, m, s0, al, dw.ref, b1, b2, pa, M, off, nc, pmax, n1, n2, cf, vis, False)
            written = True
        marks[1].record()
        if dw.p is not None:
            ctx.predict_points(dw.uvw, *dw.p, dw.ref, vis, written)
            written = True
        marks[2].record()
        if dw.g is not None:
            l, m, s0, al, mj, mn, pa = dw.g
            ctx.predict_gaussians(dw.uvw, l, m, s0, al, dw.ref, mj, mn, pa, vis, written)
            written = True
        if not written:
            ctx.predict_points(dw.uvw, None, None, None, None, dw.ref, vis, False)
        marks[3].record()
        if record is not None:
            record.append(marks)

    for _ in range(args.warmup):
        step(None)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    recs = []
    e0, e1 = ev(), ev()
    barrier()
    launches0 = binding.kernel_launches()
    e0.record()
    for _ in range(args.steps):
        step(recs)
    e1.record()
    launches = binding.kernel_launches() - launches0       # counted by the library at every <<< >>>
    barrier()
    clocks = sampler.stop() if rank == 0 else {}
    ms_total = e0.elapsed_time(e1)
    per_type_ms = split_marks(recs)
    ctx.check()
    ms_total = parallel.max_over_ranks(ms_total, dist, f"cuda:{local}")
    ms_per_step = ms_total / args.steps
    value = world * evals_per_step / (ms_per_step * 1e-3)

    # ---- end to end through the host-buffer C-ABI call (H2D + kernels + D2H inside the timing)
    vis_host_t = torch.empty(dw.uvw.vis_shape, dtype=torch.complex64, pin_memory=True)
    vis_host = vis_host_t.numpy()
    h2d = (3 * wl.u_m.nbytes + 8 * (4 * wl.points.n + 7 * wl.gaussians.n + 13 * wl.shapelets.n)
           + 16 * wl.n_coeff + 4 * (wl.shapelets.n + 1))
    d2h = vis_host.nbytes
    ctx.simulate_host(wl, vis_host)                       # warm-up (allocations)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        ctx.simulate_host(wl, vis_host)
    torch.cuda.synchronize()
    e2e_s = (time.perf_counter() - t0) / args.steps
    e2e_s = parallel.max_over_ranks(e2e_s, dist, f"cuda:{local}")
    e2e_value = world * evals_per_step / e2e_s

    # ---- SURVEY.md 8(d) rule (ii): the general path (one sin/cos, one exp2 per eval) in the same run
    general_ms = None
    if args.path != "general" and not args.no_general:
        ctx.set_path(binding.WODEN_PATH_GENERAL)
        g_total, g_recs = time_steps(step, 3, max(3, min(5, args.steps)), barrier)
        ctx.set_path(binding.WODEN_PATH_AUTO)
        g_split = split_marks(g_recs)
        general_ms = {k: float(np.median(v)) for k, v in g_split.items()}
        general_ms.update({k + "_min": float(np.min(v)) for k, v in g_split.items()})
        general_ms["step"] = parallel.max_over_ranks(g_total / len(g_recs), dist, f"cuda:{local}")

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    # ---- per-type rates and the roofline of the dominant kernel (rank 0)
    med = {k: float(np.median(v)) if v else None for k, v in per_type_ms.items()}
    per_type = {}
    for name, key in (("points", "points"), ("gaussians", "gaussians"), ("shapelets", "shapelets")):
        if med[name] and counts[key]:
            per_type[name] = {"evals_per_s": counts[key] / (med[name] * 1e-3), "ms_per_call": med[name],
                              "min_ms_per_call": float(np.min(per_type_ms[name]))}
    if "shapelets" in per_type:
        per_type["shapelets"]["coeff_evals_per_s"] = counts["shapelet_coeffs"] / (med["shapelets"] * 1e-3)

    walk = args.path != "general"        # all configs have uniformly spaced channels
    mufu_rate, mufu_clk = ctx.pipe_rate("MUFU")
    fma_rate, _ = ctx.pipe_rate("FFMA")
    ffma2_rate, _ = ctx.pipe_rate("FFMA2")          # the instruction the walking kernels issue
    dominant = max((k for k in per_type), key=lambda k: med[k])
    if dominant == "points":
        ops = {"walk": ("FP32 FMA pipe: 4 FP32 lane-ops per eval (2 three-term recurrence + 2 accumulate)",
                        ffma2_rate / 4.0),
               "general": ("MUFU pipe: 2 MUFU (sin, cos) per eval", mufu_rate / 2.0)}
    elif dominant == "gaussians":
        ops = {"walk": ("FP32 FMA pipe: 7 FP32 lane-ops per eval (2 recurrence + 2 envelope walk + 1 flux*envelope "
                        "+ 2 accumulate)", ffma2_rate / 7.0),
               "general": ("MUFU pipe: 3 MUFU (sin, cos, ex2) per eval", mufu_rate / 3.0)}
    else:
        ops = {"walk": ("FP32 FMA pipe: 1 FFMA per coefficient", fma_rate),
               "general": ("FP32 FMA pipe: 1 FFMA per coefficient", fma_rate)}
    basis, peak = ops["walk" if walk else "general"]
    ach = (per_type[dominant]["coeff_evals_per_s"] if dominant == "shapelets"
           else per_type[dominant]["evals_per_s"])
    # DRAM bytes of the dominant kernel per launch (ncu --set full, profiles/ncu_r3_kernels.md):
    # the visibility buffer once, plus the component blocks that miss L2
    key = (dominant, "walk" if walk else "general")
    rec_traffic = NCU_DRAM_BYTES.get(key) if args.config == 5 else None
    ffma2_3reg, _ = ctx.pipe_rate("FFMA2_3REG")
    walk_rate, _ = ctx.pipe_rate("WALK")
    roofline = {
        "bound": "alu", "kernel": KERNEL_NAMES.get(key, f"predict_{dominant}"), "achieved": ach / 1e9, "peak": peak / 1e9,
        "unit": "Gevals/s", "frac": ach / peak,
        "traffic": rec_traffic[1] if rec_traffic else None,
        "traffic_source": (f"ncu --set full capture of one launch of {rec_traffic[0]} at commit {rec_traffic[2]} "
                           "(profiles/ncu_r3_kernels.md): a recorded constant, not measured in this run")
        if rec_traffic else None,
        "achieved_basis": "evals of the whole woden_predict_* call / its CUDA-event duration (the call is a sequence "
                          "of launches of this kernel plus three O(K) staging kernels)",
        "operand_delivery": {"ffma2_three_fresh_pairs_fma_per_s": ffma2_3reg, "ffma_reused_operands_fma_per_s": fma_rate,
                             "walk_pattern_fma_per_s": walk_rate,
                             "frac_of_walk_pattern": (ach * 4.0 / walk_rate) if (walk and dominant == "points") else None,
                             "note": "each register bank (even / odd) feeds one operand per lane per clock: an FMA with "
                                     "three fresh register operands runs at 2/3 of the pipe rate (the read-cycle count of "
                                     "the shipped SASS is prose in profiles/walk_rf_r2.md, not part of this record); "
                                     "the kernel's own 4-FFMA2 pattern in isolation sustains walk_pattern_fma_per_s "
                                     "(DESIGN.md section 7)"},
        "peak_basis": basis + ("; packed FFMA2 rate (the instruction the kernel issues)" if walk and dominant != "shapelets"
                               else "") + f" measured live by woden_pipe_rate at {mufu_clk / 1e6:.0f} MHz",
        "pipe_rates_fma_per_s": {"FFMA2": ffma2_rate, "FFMA": fma_rate,
                                 "nominal_fp32": SM_COUNT * FP32_LANES_PER_SM * SM_MAX_HZ},
        "nominal_mufu_roofline_gevals": SM_COUNT * MUFU_LANES_PER_SM * SM_MAX_HZ / (2 if dominant == "points" else 3) / 1e9,
    }
    roofline["frac_of_mufu_roofline"] = ach / 1e9 / roofline["nominal_mufu_roofline_gevals"]
    if walk and dominant in ("points", "gaussians"):
        lane_ops = 4.0 if dominant == "points" else 7.0
        roofline["frac_of_nominal_fp32"] = ach * lane_ops / (SM_COUNT * FP32_LANES_PER_SM * SM_MAX_HZ)
    # SURVEY.md §8(d) composite roofline time for the whole step at the measured pipe rates
    t_roof = (counts["points"] / (mufu_rate / 2) + counts["gaussians"] / (mufu_rate / 3)
              + counts["shapelet_coeffs"] / fma_rate)
    composite = {"t_roof_ms": 1e3 * t_roof, "t_measured_ms": ms_per_step, "frac": 1e3 * t_roof / ms_per_step,
                 "definition": "sum_type evals/R_type with R from 2 / 3 MUFU per point / Gaussian eval and "
                               "1 FFMA per shapelet coefficient (SURVEY.md 8(d)); >1 means the channel-walking "
                               "path removed MUFU work"}

    cpu_baseline = None
    if world == 1 and not args.no_cpu_baseline:
        cores = len(os.sched_getaffinity(0))
        os.environ.setdefault("OMP_NUM_THREADS", str(cores))
        time_oracle(wl, 2048, 4000)                       # load + build the oracle library
        n_sample = 1 << 17
        v, dt = time_oracle(wl, n_sample, 7000)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": f"{n_sample} seeded random visibilities of config {wl.config}, all {comps} "
                                  f"components each ({dt:.1f} s)"}

    general_path = None
    if general_ms is not None:
        general_path = general_path_record(general_ms, counts, mufu_rate, t_roof, world, evals_per_step,
                                           max(3, min(5, args.steps)))
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": config_dict(wl, {
            "path": "auto (channel walking: uniform 80 kHz channels)" if walk else "general",
            "arithmetic": "FP32 sums and phasors, FP64 phase before reduction to its fraction; complex64 output",
            "l2": "no flush: each step writes 1.4 GB of visibilities, 11x the 126 MB L2; component blocks "
                  "are meant to be L2 resident",
            "parallelism": "1 GPU" if world == 1 else f"time-sharded x{world}, no collective"}),
        "per_type": per_type, "roofline": roofline, "composite_roofline": composite, "general_path": general_path,
        "cpu_baseline": cpu_baseline,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                "ms_per_step": 1e3 * e2e_s, "call": "woden_simulate_host (pinned host vis buffer)"},
        "gpu_launches": launches, "clocks": clocks,
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


# ---- register-file read-cycle model of a kernel's main loop (profiles/walk_rf_r3.md) -------------------
_UNIFORM_OPS = ("LDCU", "UIADD", "UIMAD", "UISETP", "USEL", "UMOV", "ULDC", "UMOV", "BRA", "ULEA", "USHF", "ULOP")
_WIDE_OPS = ("FFMA2", "FMUL2", "FADD2", "DFMA", "DMUL", "DADD")


def read_cycle_model(sass_text, kernel_tag):
    """Sum of register-file read cycles over the largest loop of the kernel whose mangled name contains
    `kernel_tag`, from `cuobjdump -sass` text.  Rule (measured on the B200, profiles/walk_rf_r2.md and
    walk_rf_r3.md): an instruction holds the read stage for max(#distinct even, #distinct odd) source registers;
    a 64-bit / .F32x2 operand is an even + odd pair, a `.F32` scalar-broadcast operand one register; uniform
    registers, constants and immediates are free; an operand is free when the PREVIOUS instruction of the
    listing had the same register in the same source slot flagged `.reuse` -- ANY instruction in between,
    uniform-datapath ones (LDCU) included, drops it.  Returns a dict with the loop's instruction count, its
    packed-FP32 instruction count, the read-cycle sum and the sum per opcode."""
    import re
    fn = [f for f in sass_text.split("Function :")[1:] if kernel_tag in f.split("\n")[0]]
    if not fn:
        raise ValueError(f"no function matching {kernel_tag!r}")
    ins = []
    for line in fn[0].split("\n"):
        m = re.search(r"/\*([0-9a-f]{4,5})\*/\s+(.*?);", line)
        if m:
            ins.append((int(m.group(1), 16), m.group(2).strip()))
    loops = []
    for addr, text in ins:
        m = re.search(r"\bBRA\S*\s.*0x([0-9a-f]+)", text)
        if m and int(m.group(1), 16) < addr:
            loops.append((int(m.group(1), 16), addr))
    if not loops:
        raise ValueError("no backward branch found")
    lo, hi = max(loops, key=lambda x: x[1] - x[0])
    body = [t for a, t in ins if lo <= a <= hi]
    total, per_op, prev = 0, {}, {}
    for text in body:
        if text.startswith("@"):
            text = text.split(None, 1)[1]
        opc = text.split()[0]
        srcs = [o.strip() for o in (text.split(None, 1)[1] if " " in text else "").split(",")][1:]
        wide = opc.startswith(_WIDE_OPS) or opc.startswith("F2F.F32.F64")
        even, odd, cur = set(), set(), {}
        for slot, op in enumerate(srcs):
            m = re.match(r"[-|~]*R(\d+)(\.reuse)?(\.F32x2|\.F32|\.64)?", op)
            if not m:
                continue
            r = int(m.group(1))
            cur[slot] = (r, bool(m.group(2)))
            if prev.get(slot) == (r, True):
                continue
            for x in ([r] if (m.group(3) == ".F32" or not wide) else [r, r + 1]):
                (odd if x % 2 else even).add(x)
        c = max(len(even), len(odd))
        total += c
        per_op[opc] = per_op.get(opc, 0) + c
        prev = cur
    return {"instructions": len(body), "packed_fp32": sum(1 for t in body if "FFMA2" in t or "FMUL2" in t),
            "read_cycles": total, "per_opcode": dict(sorted(per_op.items(), key=lambda kv: -kv[1]))}


def run_rf_model(args):
    """`bench.py --rf-model`: the read-cycle model of both channel-walking kernels from the SASS of the committed
    build (cuobjdump on paper_2005_09316_b200/build/predict_walk.o; no GPU needed)."""
    import subprocess
    from paper_2005_09316_b200 import build
    build.build()
    obj = os.path.join(build.OBJ, "predict_walk.o")
    if not os.path.exists(obj):
        build.build(force=True)
    sass = subprocess.run(["cuobjdump", "-sass", obj], check=True, capture_output=True, text=True).stdout
    out = {}
    for name, tag, unroll in (("points", "predict_walk_kernelILb0", 2), ("gaussians", "predict_walk_kernelILb1", 4)):
        m = read_cycle_model(sass, tag)
        m["components_per_pass"] = unroll
        m["read_cycles_per_component"] = m["read_cycles"] / unroll
        m["fma_pipe_cycles_per_component"] = 2.0 * m["packed_fp32"] / unroll
        out[name] = m
    print(json.dumps({"rf_model": out, "source": "cuobjdump -sass paper_2005_09316_b200/build/predict_walk.o"}))
    return 0



def run_pipes(args):
    """Pipe-rate microbenchmarks (woden_pipe_rate): the measured ALU roofline denominators."""
    import torch
    from paper_2005_09316_b200 import binding
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --pipes: no CUDA device")
    ctx = binding.Woden(0)
    out = {}
    for name in binding.PIPES:
        ctx.pipe_rate(name, 2000)
        best = max((ctx.pipe_rate(name, 20000) for _ in range(3)), key=lambda r: r[0])
        out[name] = {"thread_ops_per_s": best[0], "sm_clock_hz": best[1],
                     "per_sm_per_clk": best[0] / SM_COUNT / best[1] if best[1] else None}
    print(json.dumps({"pipes": out, "sm_count": SM_COUNT}))
    return 0


def run_truncation(args):
    """GPU time against the kept fraction f_comp (section 5.3, Eq 23-24; the shape of Fig 7's
    timing panels): config 4's MS-CLEAN-like point/Gaussian model and its two-lobe shapelet model."""
    import torch
    from paper_2005_09316_b200 import binding, truncate
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --truncation: no CUDA device")
    wl = inputs.make_config(4)
    ctx = binding.Woden(0)
    uvw = binding.Uvw(*(torch.as_tensor(a, device="cuda:0") for a in (wl.u_m, wl.v_m, wl.w_m)), wl.freqs_hz)
    vis = ctx.new_vis(uvw)
    dev = lambda a, dt=torch.float64: torch.as_tensor(np.ascontiguousarray(a), dtype=dt, device="cuda:0")
    w_sh = truncate.shapelet_basis_weights(ctx, wl.shapelets)

    def timed(fn):
        for _ in range(2):
            fn()
        torch.cuda.synchronize()
        ts = []
        for _ in range(max(3, args.steps)):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); fn(); e1.record(); torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        return float(np.median(ts))

    rows = []
    for f in (1.0, 0.8, 0.6, 0.4, 0.2, 0.1):
        p, g = truncate.truncate_components(ctx, wl.points, f), truncate.truncate_components(ctx, wl.gaussians, f)
        s = truncate.truncate_shapelets(ctx, wl.shapelets, f, w_sh)
        dp = [dev(a) for a in (p.l, p.m, p.s0_jy, p.alpha)]
        dg = [dev(a) for a in (g.l, g.m, g.s0_jy, g.alpha, g.maj_fwhm_rad, g.min_fwhm_rad, g.pa_rad)]
        ds_ = [dev(a) for a in (s.l, s.m, s.s0_jy, s.alpha, s.beta1_rad, s.beta2_rad, s.pa_rad, s.uv_basis)]
        di = [dev(a, torch.int32) for a in (s.coeff_offset, s.n1, s.n2)]
        dc = dev(s.coeff)
        pmax = int((s.n1 + s.n2).max())

        def clean():
            ctx.predict_points(uvw, *dp, wl.ref_freq_hz, vis, False)
            ctx.predict_gaussians(uvw, *dg[:4], wl.ref_freq_hz, *dg[4:], vis, True)

        def shp():
            ctx.predict_shapelets(uvw, *ds_[:4], wl.ref_freq_hz, *ds_[4:], di[0], int(s.coeff.size), pmax,
                                  di[1], di[2], dc, vis, False)

        row = {"f_comp": f, "msclean_components": p.n + g.n, "msclean_ms": timed(clean),
               "shapelet_basis_functions": int(s.coeff.size), "shapelet_p_max": pmax, "shapelet_ms": timed(shp)}
        eng, bucket = ctx.last_shapelet_path()
        row["shapelet_engine_auto"] = {1: "register", 2: "tensor", 3: "register-sparse"}.get(eng, str(eng))
        row["shapelet_order_bucket"] = bucket
        for name, code in (("register", 1), ("tensor", 2)):          # the two engines forced, for AUTO's policy table
            ctx.set_shapelet_path(code)
            row[f"shapelet_ms_{name}"] = timed(shp)
        ctx.set_shapelet_path(0)
        rows.append(row)
    ctx.check()
    print(json.dumps({"truncation": rows, "workload": "config 4 (8128 baselines x 14 steps x 384 channels)",
                      "note": "one launch set per model; medians of CUDA-event times"}))
    return 0


def run_only(args):
    """One C-ABI predict call of one component type on the config's grid (what the per-kernel ncu
    captures under profiles/ run): `--only points|gaussians|shapelets`, optionally the first
    `--max-components` components, for shapelets optionally full triangles of `--shapelet-order`
    (the config's decay law, seed 1) and a forced `--shapelet-engine`.  Prints one JSON line."""
    import torch
    from paper_2005_09316_b200 import binding
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --only: no CUDA device")
    wl = inputs.make_config(args.config)
    ctx = binding.Woden(0)
    ctx.set_path(binding.WODEN_PATH_GENERAL if args.path == "general" else binding.WODEN_PATH_AUTO)
    ctx.set_shapelet_path({"auto": 0, "register": 1, "tensor": 2}[args.shapelet_engine])
    dev = lambda a, dt=torch.float64: torch.as_tensor(np.ascontiguousarray(a), dtype=dt, device="cuda:0")
    uvw = binding.Uvw(dev(wl.u_m), dev(wl.v_m), dev(wl.w_m), wl.freqs_hz)
    vis = ctx.new_vis(uvw)
    n_max = args.max_components if args.max_components > 0 else None
    if args.only == "points":
        p = wl.points
        a = [dev(x[:n_max]) for x in (p.l, p.m, p.s0_jy, p.alpha)]
        call = lambda: ctx.predict_points(uvw, *a, wl.ref_freq_hz, vis, False)
        units, unit_name = int(a[0].numel()), "components"
    elif args.only == "gaussians":
        g = wl.gaussians
        a = [dev(x[:n_max]) for x in (g.l, g.m, g.s0_jy, g.alpha, g.maj_fwhm_rad, g.min_fwhm_rad, g.pa_rad)]
        call = lambda: ctx.predict_gaussians(uvw, *a[:4], wl.ref_freq_hz, *a[4:], vis, False)
        units, unit_name = int(a[0].numel()), "components"
    else:
        sh = wl.shapelets
        n1, n2, cf, off = sh.n1, sh.n2, sh.coeff, sh.coeff_offset
        if args.shapelet_order >= 0:
            rng = np.random.default_rng(1)
            t1, t2 = inputs.full_triangle(args.shapelet_order)
            n1, n2 = np.tile(t1, sh.n), np.tile(t2, sh.n)
            cf = rng.normal(0, 1, n1.size) * np.exp(-(n1 + n2) / 10.0)
            off = np.arange(sh.n + 1) * len(t1)
        a = [dev(x) for x in (sh.l, sh.m, sh.s0_jy, sh.alpha)]
        b = [dev(x) for x in (sh.beta1_rad, sh.beta2_rad, sh.pa_rad, sh.uv_basis)]
        i = [dev(x, torch.int32) for x in (off, n1, n2)]
        c = dev(cf)
        pmax = int((n1 + n2).max())
        call = lambda: ctx.predict_shapelets(uvw, *a, wl.ref_freq_hz, *b, i[0], int(cf.size), pmax, i[1], i[2], c, vis,
                                             False)
        units, unit_name = int(cf.size), "coefficients"
    for _ in range(max(1, args.warmup)):
        call()
    torch.cuda.synchronize()
    ts = []
    for _ in range(max(1, args.steps)):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); call(); e1.record(); torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1))
    ctx.check()
    ms = float(np.median(ts))
    print(json.dumps({"only": args.only, "config": args.config, unit_name: units, "n_vis": wl.n_vis, "path": args.path,
                      "shapelet_engine": args.shapelet_engine, "ms": ms, "min_ms": float(min(ts)),
                      f"{unit_name}_x_visibility_per_s": units * wl.n_vis / (ms * 1e-3)}))
    return 0


def run_basis(args):
    """NEXT-5 experiment: evaluate the 1-D shapelet series sum_p c_p h_p(x) for 2^26 arguments by the
    recurrence of the predict kernels and by the paper's look-up tables; time and
    maximum error against the oracle's long-double Hermite routine on a 4096-point sample."""
    import torch
    import oracle
    from paper_2005_09316_b200 import binding
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --basis: no CUDA device")
    ctx = binding.Woden(0)
    rng = np.random.default_rng(7)
    n = 1 << 26
    x = torch.empty(n, dtype=torch.float32, device="cuda:0").uniform_(-12.0, 12.0, generator=torch.Generator("cuda:0").manual_seed(7))
    out = torch.empty_like(x)
    rows = []
    for pm in (40, 86):
        c = (rng.normal(0, 1, pm + 1) * np.exp(-np.arange(pm + 1) / 10.0)).astype(np.float32)
        cd = torch.as_tensor(c, device="cuda:0")
        xs = x[:4096].cpu().numpy()
        ref = np.array([np.dot(c.astype(np.float64), oracle.hermite_functions(pm, float(v))) for v in xs])
        for name, method, dx in (("recurrence", 0, 0.0), ("lut dx=2^-7", 1, 2.0 ** -7), ("lut dx=2^-10", 1, 2.0 ** -10)):
            call = lambda: ctx.shapelet_series(method, x, cd, lut_dx=dx or 1.0, lut_x_max=32.0, out=out)
            call(); torch.cuda.synchronize()
            ts = []
            for _ in range(max(3, args.steps)):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(); call(); e1.record(); torch.cuda.synchronize()
                ts.append(e0.elapsed_time(e1))
            err = float(np.abs(out[:4096].cpu().numpy() - ref).max() / np.abs(c).sum())
            table_mb = 0.0 if method == 0 else np.ceil(32.0 / dx) * (pm + 1) * 8 / 1e6
            rows.append({"p_max": pm, "method": name, "ms": float(np.median(ts)), "basis_values_per_s": n * (pm + 1) / (np.median(ts) * 1e-3),
                         "max_err_over_sum_abs_coeff": err, "table_MB": table_mb})
    print(json.dumps({"basis": rows, "n_arguments": n}))
    return 0


def run_peel(args):
    """The paper's consumer of the predicted visibilities (section 5.1): fit one complex gain
    per antenna and (time, frequency) cell by 10 passes of Eq 22, then subtract the calibrated model.
    "Observed" = config 5's sky through the predictors, model = its truncated version (Eq 23-24,
    f_comp = 0.8) through the predictors."""
    import torch
    from paper_2005_09316_b200 import binding, truncate
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --peel: no CUDA device")
    wl = inputs.make_config(args.config)
    n_ant = int(round((1 + (1 + 8 * wl.n_baselines) ** 0.5) / 2))
    ctx = binding.Woden(0)
    dw = binding.DeviceWorkload(wl)
    full = dw.predict(ctx)
    wl_t = inputs.make_config(args.config)
    wl_t.points = truncate.truncate_components(ctx, wl.points, 0.8)
    wl_t.gaussians = truncate.truncate_components(ctx, wl.gaussians, 0.8)
    wl_t.shapelets = truncate.truncate_shapelets(ctx, wl.shapelets, 0.8)
    model = binding.DeviceWorkload(wl_t).predict(ctx)
    out = torch.empty_like(full)
    torch.cuda.synchronize()

    def timed(fn, reps):
        fn(); torch.cuda.synchronize()
        ts = []
        for _ in range(reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); fn(); e1.record(); torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        return float(np.median(ts))

    g = [None]
    ms_cal = timed(lambda: g.__setitem__(0, ctx.calibrate_gains(n_ant, full, model, 10)), max(3, args.steps))
    ms_peel = timed(lambda: ctx.peel(n_ant, full, model, g[0], out=out), max(3, args.steps))
    ctx.check()
    cells = wl.n_times * wl.n_freqs
    before = float(torch.sum(torch.abs(full - model) ** 2).item())
    after = float(torch.sum(torch.abs(out) ** 2).item())
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm = peaks.get("hbm_gbs", 6650.0)
    gbs = 3 * full.numel() * 8 / (ms_peel * 1e-3) / 1e9
    print(json.dumps({
        "peel": {"workload": f"config {wl.config}: {cells} cells x {n_ant} antennas ({wl.n_baselines} baselines)",
                 "calibrate_ms": ms_cal, "cell_fits_per_s": cells / (ms_cal * 1e-3), "iterations": 10,
                 "peel_ms": ms_peel,
                 "peel_roofline": {"bound": "hbm", "achieved": gbs, "peak": hbm, "unit": "GB/s", "frac": gbs / hbm,
                                   "peak_source": "measured" if peaks else "fallback",
                                   "algorithmic_bytes_per_visibility": 24},
                 "residual_power_raw_model": before, "residual_power_after_peel": after}}))
    return 0


def run_fit(args):
    """NEXT-4: the image-space shapelet fit on a synthetic restored image: a planted
    p_max = 40 model (861 basis functions, the order of config 5's shapelets) rendered through
    woden_fit_shapelets' own inverse is not available, so the image is a sum of seeded Gaussian blobs
    (device-made, no oracle); 256 x 256 pixels, restoring beam of 3 pixels FWHM, 3 x 3 grid of (beta1, beta2).
    Reports the whole call and the roofline of its dense contraction, the Gram-matrix kernel."""
    import torch
    from paper_2005_09316_b200 import binding
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --fit: no CUDA device")
    ctx = binding.Woden(0)
    n, pix, p_max = args.fit_pixels, 0.3 * inputs.ARCMIN, args.fit_order
    P = (p_max + 1) * (p_max + 2) // 2
    gen = torch.Generator("cuda:0").manual_seed(inputs.SEED_BASE + 40)
    ax = (torch.arange(n, device="cuda:0", dtype=torch.float64) - (n - 1) / 2) * pix
    L, M = -ax[None, :], ax[:, None]
    img = torch.zeros((n, n), dtype=torch.float64, device="cuda:0")
    cen = (torch.rand((40, 2), generator=gen, device="cuda:0", dtype=torch.float64) - 0.5) * 0.5 * n * pix
    wid = (0.02 + 0.08 * torch.rand(40, generator=gen, device="cuda:0", dtype=torch.float64)) * n * pix
    amp = torch.randn(40, generator=gen, device="cuda:0", dtype=torch.float64)
    for k in range(40):
        img += amp[k] * torch.exp(-((L - cen[k, 0]) ** 2 + (M - cen[k, 1]) ** 2) / (2 * wid[k] ** 2))
    beta = 0.9 * n * pix * 2.3548 / (2.0 * 2.6 * (2 * p_max + 1.0) ** 0.5)
    f1, f2 = np.meshgrid([0.9, 1.0, 1.1], [0.9, 1.0, 1.1], indexing="ij")
    B1, B2 = (beta * f1).ravel(), (beta * f2).ravel()
    beam = (3.0 * pix, 2.0 * pix, 0.5, 6)
    call = lambda: ctx.fit_shapelets(img, -pix, pix, 0.0, 0.0, 0.0, 0.0, 0.3, p_max, B1, B2, beam=beam, want_weights=True)
    for _ in range(max(1, args.warmup)):
        out = call()
    torch.cuda.synchronize()
    ts, gs = [], []
    l0 = binding.kernel_launches()
    for _ in range(max(3, args.steps)):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); out = call(); e1.record(); torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1)); gs.append(ctx.fit_gram_ms())
    launches = binding.kernel_launches() - l0
    ctx.check()
    coeff, resid, weights, best = out
    ms, gram_ms = float(np.median(ts)), float(np.median(gs))
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    peak = peaks.get("bf16_tflops", 1650.0)
    n_pix = n * n
    alg_flops = float(n_pix) * P * (P + 1)                      # A^T A, symmetric half, 2 flops per MAC
    n_rt = (P + 127) // 128
    exe_flops = 3.0 * 2.0 * (n_rt * (n_rt + 1) // 2) * 128 * 128 * ((n_pix + 63) // 64 * 64)
    print(json.dumps({"fit": {
        "workload": f"{n} x {n} pixel synthetic image, p_max {p_max} ({P} basis functions), 3 x 3 (beta1, beta2) grid, "
                    f"beam stencil {2 * beam[3] + 1}^2, 6 refinement passes",
        "ms_per_call": ms, "fits_per_s": 9.0 / (ms * 1e-3), "gpu_launches": launches, "best_index": int(best[0]),
        "residual_best_over_image_power": float(resid[int(best[0])] / (img ** 2).sum()),
        "roofline": {"bound": "tensor", "kernel": "fit_gram_kernel (tcgen05 kind::f16, FP16 hi+lo split, 3 products)",
                     "achieved": alg_flops / (gram_ms * 1e-3) / 1e12, "peak": peak, "unit": "TFLOP/s",
                     "frac": alg_flops / (gram_ms * 1e-3) / 1e12 / peak,
                     "executed_tensor_tflops": exe_flops / (gram_ms * 1e-3) / 1e12,
                     "ms_per_launch": gram_ms,
                     "peak_source": ("MEASURED_PEAKS.json bf16_tflops (fp16 dense peak = bf16 dense peak nominally)"
                                     if peaks else "fallback 1650 TFLOP/s"),
                     "algorithmic_flops_per_launch": alg_flops,
                     "note": "algorithmic = n_pix P (P + 1): the symmetric half of A^T A once; the kernel executes 3 "
                             "split-precision products on 128-padded tiles (executed_tensor_tflops)", "traffic": None}}}))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--path", choices=["auto", "general"], default="auto")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-general", action="store_true", help="skip the general-path record of the line")
    ap.add_argument("--dry", action="store_true",
                    help="rendezvous only (gloo, no GPU work): checks that --gpus N starts N ranks")
    ap.add_argument("--pipes", action="store_true", help="print the measured pipe rates and exit")
    ap.add_argument("--rf-model", action="store_true",
                    help="register-file read-cycle model of the walking kernels from the build's SASS (no GPU) and exit")
    ap.add_argument("--only", choices=["points", "gaussians", "shapelets"], default=None,
                    help="time ONE predict call of one component type (used for the per-kernel ncu captures) and exit")
    ap.add_argument("--max-components", type=int, default=0, help="--only: use the first N components")
    ap.add_argument("--shapelet-order", type=int, default=-1, help="--only shapelets: full triangles of this order")
    ap.add_argument("--shapelet-engine", choices=["auto", "register", "tensor"], default="auto")
    ap.add_argument("--basis", action="store_true",
                    help="look-up-table vs recurrence evaluation of the shapelet basis (PAPER.md:159) and exit")
    ap.add_argument("--peel", action="store_true",
                    help="time the gain fit and peel of PAPER.md section 5.1 on the config and exit")
    ap.add_argument("--fit", action="store_true",
                    help="time the image-space shapelet fit (PAPER.md section 2.1) on a synthetic image and exit")
    ap.add_argument("--fit-pixels", type=int, default=256)
    ap.add_argument("--fit-order", type=int, default=40)
    ap.add_argument("--truncation", action="store_true",
                    help="GPU time vs kept fraction of components (PAPER.md section 5.3) and exit")
    args = ap.parse_args()
    spawn_ranks_if_needed(args)
    if args.dry:
        return run_dry(args)
    if args.rf_model:
        return run_rf_model(args)
    if args.pipes:
        return run_pipes(args)
    if args.truncation:
        return run_truncation(args)
    if args.only:
        return run_only(args)
    if args.basis:
        return run_basis(args)
    if args.peel:
        return run_peel(args)
    if args.fit:
        return run_fit(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
