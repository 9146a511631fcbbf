#!/usr/bin/env python
"""bench.py -- exact-exchange apply throughput on B200 (contract: see DESIGN.md "Measurement").

A step = one pass of the whole hot path (pair scheduling, pass A, pass B, pass C, energy reduction) over one
synthetic workload, i.e. one exx_apply of all N(N+1)/2 orbital pairs.  `value` = pair-solves/s with the orbitals
resident in HBM; `e2e` = the same metric through exx_apply_host (pinned host buffers, H2D of psi and D2H of K psi
inside the timed region).  Default workload: C5 (periodic 192^3, 1024 orbitals, ~58 GB of orbitals), the largest
single-GPU configuration of BASELINE.json; the other two configurations the north_star target is quoted on (C3, C4)
are measured in the same run and reported under `per_config`.  N > 1 GPUs: replicas, one
process per GPU (under torchrun, or spawned here when WORLD_SIZE is unset), barrier + max-over-ranks timing,
value = pairs of all ranks / that time; `--parallel rr` distributes the orbitals of ONE workload round-robin instead
(paper_1712_07973_b200.distributed, strong scaling).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C1..C5] [--impl ours|reference]
"""
from __future__ import annotations

import argparse
import json
import os
import socket
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "pair_solves_per_s"
UNIT = "pair-solves/s"
HBM_SPEC_GBS = 8000.0            # north_star: "bytes over 8 TB/s HBM"
# A C5 step takes the better part of a minute: the driver's --steps / --warmup are honoured up to these caps and the
# counts actually run are printed as steps / warmup (the requested ones as steps_requested / warmup_requested).
STEP_CAP = {"C1": 1000, "C2": 200, "C3": 50, "C4": 5, "C5": 2}
WARMUP_CAP = {"C1": 20, "C2": 10, "C3": 5, "C4": 3, "C5": 3}
DEFAULT_STEPS = {"C1": 20, "C2": 10, "C3": 10, "C4": 3, "C5": 2}


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def _ncu_traffic(config: str, pass_name: str, xforms_per_launch: float):
    """dram__bytes_read+write per launch of the dominant kernel from the committed `ncu --set full` captures
    (profiles/r02_traffic.csv: config,pass,transforms_in_launch,dram_bytes), scaled to this run's mean launch size."""
    path = os.path.join(ROOT, "profiles", "r02_traffic.csv")
    if not os.path.exists(path):
        return None
    try:
        with open(path) as fh:
            for line in fh:
                f = line.strip().split(",")
                if len(f) == 4 and f[0] == config and f[1] == pass_name:
                    return float(f[3]) / float(f[2]) * xforms_per_launch
    except Exception:
        return None
    return None


def aggregate_over_ranks(step_ms_local: float, pairs_per_rank: int, world: int, all_reduce_max=None):
    """Replicas-only scaling: every rank applies the whole operator to its own copy; the job's
    time is the MAX over ranks (all_reduce_max: callable float -> float, identity for one rank) and the job's
    throughput is the pairs of all ranks over that time."""
    step_ms = all_reduce_max(step_ms_local) if (all_reduce_max is not None and world > 1) else step_ms_local
    return step_ms, pairs_per_rank * world / (step_ms * 1e-3)


def effective_counts(config: str, steps, warmup, quick=False):
    """(steps, warmup) actually run for a config given the requested ones (None = default).  quick: one warm-up step and
    one timed step -- for runs under a profiler, whose printed numbers are never bench values."""
    if quick:
        return 1, 1
    k = DEFAULT_STEPS[config] if steps is None else max(1, min(int(steps), STEP_CAP[config]))
    w = max(3, min(int(warmup), WARMUP_CAP[config]))                      # timing rule: at least three warm-up steps
    return k, w


def rank_env(gpus: int):
    """(rank, local_rank, world, spawn) from the torchrun environment; spawn = this process must start the ranks itself
    (plain `python bench.py --gpus N` with N > 1 and no WORLD_SIZE)."""
    if "WORLD_SIZE" in os.environ:
        return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ["WORLD_SIZE"]), False
    return 0, 0, 1, gpus > 1


class ClockSampler(threading.Thread):
    """Samples nvidia-smi clocks and throttle reasons during the timed region."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index = index
        self.samples = []
        self.reasons = set()
        self.max_mhz = None
        self._stop_evt = threading.Event()

    def run(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        while not self._stop_evt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-i", str(self.index)],
                                     capture_output=True, text=True, timeout=5).stdout.strip().split(",")
                self.samples.append(float(out[0]))
                self.max_mhz = float(out[1])
                for name, val in zip(names, out[2:]):
                    if val.strip().lower() == "active":
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop_evt.wait(0.2)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=10)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def alg_bytes_per_transform(spec):
    """HBM bytes per packed transform and per pass as the kernels move them.

    periodic: complex intermediate I = 16 B/point written by A, read+written by B, read by C; the streamed psi_i read by
    A and again by C; K psi_i read-modify-written by C.  free: the intermediate has 4M points (n x 2n x 2n).  The two
    resident orbitals psi_j, psi_l / K psi_j, K psi_l of a batch and K^ (L2-resident) are amortised to zero.
    """
    M = spec.n_points
    inter = 16 * M * (4 if spec.bc == "free" else 1)
    return {"A": 8 * M + inter, "B": 2 * inter, "C": inter + 8 * M + 16 * M}


def nominal_flops_per_transform(spec):
    """Nominal FFT flops (5 T log2 T per complex line of T points, pruned lines not counted) per packed transform and
    pass: A = forward c axis + first stage of the forward b axis; B = second b stage + a axis, forward and inverse, +
    the K^ multiply; C = mirror of A + the Kernel-3 epilogue (12 flop/point).  Shares of the b axis by log2 of the stage
    lengths.  Sums to SURVEY.md 8(d)'s 2 x 5 M log2 M (periodic) per transform up to the pointwise terms."""
    n = spec.dims
    free = spec.bc == "free"
    t = [2 * d for d in n] if free else list(n)
    r2 = {16: 4, 24: 12, 32: 4, 48: 12, 64: 8, 72: 12, 96: 12, 128: 8, 144: 12, 192: 16, 256: 16}.get(t[1], 16)
    r1 = t[1] // r2
    lg = np.log2
    lines_c = n[0] * n[1]                       # non-zero lines along c
    cols_b = n[0] * t[2]                        # lines along b (all c frequencies, non-zero a planes)
    lines_a = t[1] * t[2]                       # lines along a
    f_c = lines_c * 5 * t[2] * lg(t[2])
    f_b1 = cols_b * 5 * t[1] * lg(r1)
    f_b2 = cols_b * 5 * t[1] * lg(r2)
    f_a = lines_a * 5 * t[0] * lg(t[0])
    M = spec.n_points
    return {"A": f_c + f_b1 + 2 * M, "B": 2 * (f_b2 + f_a) + 2 * t[0] * t[1] * t[2], "C": f_c + f_b1 + 12 * M}


def survey_b_alg_per_pair(spec):
    """SURVEY.md 8(d) B_alg per pair-solve: 64 M bytes (periodic), 160 M bytes (free)."""
    return (160 if spec.bc == "free" else 64) * spec.n_points


def cpu_baseline(spec, kernel, psi_np, seconds_target=15.0):
    """The oracle, as it stands, timed on this host's cores on a bounded sample of the same workload."""
    from oracle import Oracle, threads_used
    o = Oracle(spec.dims, spec.spacing, spec.bc, kernel)
    n_orb = spec.n_orb
    rng = np.random.default_rng(12345)
    cores = os.cpu_count() or 1
    first = [(int(a), int(b)) for a, b in rng.integers(0, n_orb, size=(cores, 2))]
    t0 = time.perf_counter()
    o.pair_energies(psi_np, first)
    t1 = time.perf_counter() - t0
    n_more = int(max(0, min(64 * cores, (seconds_target - t1) / max(t1, 1e-3) * cores)))
    n_more -= n_more % cores
    total_solves, total_time = len(first), t1
    if n_more > 0:
        more = [(int(a), int(b)) for a, b in rng.integers(0, n_orb, size=(n_more, 2))]
        t0 = time.perf_counter()
        o.pair_energies(psi_np, more)
        total_time += time.perf_counter() - t0
        total_solves += n_more
    return {"value": total_solves / total_time, "unit": UNIT, "cores": threads_used(), "kind": "oracle",
            "sample": f"{total_solves} seeded random pair solves (co-density, padded 3-D FFT Poisson solve, energy) of {spec.name}, "
                      f"{total_time:.1f} s wall"}


def cufft_comparison(spec, psi, occ, kernel_table, plan_pair_energies, seconds_target=2.0):
    """GPU comparison baseline ("the cuFFT path ... same inputs, same metric"; reported, never the
    product): an UNTUNED library pipeline -- co-densities as a torch product, torch.fft.rfftn / irfftn (cuFFT D2Z / Z2D,
    zero-padded to 2n for free BC), pointwise multiply by K^, pointwise epilogue -- timed on a bounded sample of rows i
    (all j >= i of a row, batched).  Returns pair-solves/s and a sanity check against the library."""
    import torch
    n = spec.dims
    free = spec.bc == "free"
    t = tuple(2 * d for d in n) if free else tuple(n)
    dev = psi.device
    if free:
        g = torch.as_tensor(kernel_table, dtype=torch.float64, device=dev)
        idx = [torch.minimum(torch.arange(tt, device=dev), tt - torch.arange(tt, device=dev)) for tt in t]
        mask = [(i != tt // 2) for i, tt in zip(idx, t)]
        ext = g[idx[0].clamp(max=n[0] - 1)][:, idx[1].clamp(max=n[1] - 1)][:, :, idx[2].clamp(max=n[2] - 1)]
        ext = ext * (mask[0][:, None, None] & mask[1][None, :, None] & mask[2][None, None, :])
        khat = torch.fft.rfftn(ext).real * spec.dV
    else:
        freq = [2.0 * np.pi * torch.fft.fftfreq(tt, d=h, device=dev, dtype=torch.float64) for tt, h in zip(t, spec.spacing)]
        g2 = freq[0][:, None, None] ** 2 + freq[1][None, :, None] ** 2 + (freq[2][None, None, : t[2] // 2 + 1]) ** 2
        khat = torch.where(g2 > 0, 4.0 * np.pi / g2.clamp(min=1e-300), torch.zeros_like(g2))
    n_orb = psi.shape[0]
    kpsi = torch.zeros_like(psi)
    bmax = max(1, int(2e9 // (8 * t[0] * t[1] * t[2])))              # about 2 GB of padded real co-densities per batch
    sl = tuple(slice(0, d) for d in n)

    def row(i):
        e_row = torch.zeros(n_orb, dtype=torch.float64, device=dev)
        for j0 in range(i, n_orb, bmax):
            js = slice(j0, min(n_orb, j0 + bmax))
            rho = psi[i][None] * psi[js]
            v = torch.fft.irfftn(torch.fft.rfftn(rho, s=t, dim=(1, 2, 3)) * khat, s=t, dim=(1, 2, 3))[(slice(None),) + sl]
            kpsi[i] -= torch.einsum("j,jabc->abc", torch.as_tensor(occ[js], device=dev), v * psi[js])
            off = torch.as_tensor(occ[i] * (np.arange(js.start, js.stop) != i), device=dev)
            kpsi[js] -= off[:, None, None, None] * v * psi[i][None]
            e_row[js] = spec.dV * (rho * v).sum(dim=(1, 2, 3))
        return e_row

    rows = [0]
    e0 = row(0)                                                     # warm-up (cuFFT plans) and the sanity row
    torch.cuda.synchronize()
    ref = torch.as_tensor(plan_pair_energies[0], device=dev)
    err = float((e0 - ref).abs().max() / ref.abs().max())
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    pairs, ms = 0, 0.0
    rng = np.random.default_rng(7)
    while ms < seconds_target * 1e3 and len(rows) < 64:
        i = int(rng.integers(0, n_orb))
        ev0.record()
        row(i)
        ev1.record()
        torch.cuda.synchronize()
        ms += ev0.elapsed_time(ev1)
        pairs += n_orb - i
        rows.append(i)
    return {"value": pairs / (ms * 1e-3), "unit": UNIT,
            "kind": "untuned library pipeline: torch.fft (cuFFT D2Z/Z2D) + pointwise torch ops, one real co-density per transform",
            "sample": f"{pairs} pair solves ({len(rows) - 1} seeded rows i, all j >= i), {ms * 1e-3:.2f} s device time",
            "max_rel_err_pair_energies_row0_vs_library": err}


def _workload_name(spec, note=""):
    t = "x".join(str(d) for d in spec.dims)
    return f"{spec.name}: {spec.bc} {t} grid, h={spec.spacing[0]} bohr, {spec.n_orb} orbitals, {spec.n_pairs} pairs{note}"


def _config_dict(spec, world, parallel, note=""):
    """The `config` object: the SAME keys for the product arm and the reference arm."""
    return {"workload": _workload_name(spec, note),
            "pairs": spec.n_pairs,
            "l2_policy": "inputs larger than L2 (orbitals %.2f GB)" % (spec.n_orb * spec.n_points * 8 / 1e9),
            "parallelism": ("round-robin orbital blocks" if parallel == "rr" else "replicas") if world > 1 else "single GPU"}


def choose_default_config():
    """C5 (the largest single-GPU configuration) when the device and the host can hold it, else C4."""
    try:
        import torch
        if not torch.cuda.is_available():
            return "C5", ""
        dev_gb = torch.cuda.get_device_properties(torch.cuda.current_device()).total_memory / 1e9
    except Exception:
        return "C5", ""
    try:
        host_gb = os.sysconf("SC_PAGE_SIZE") * os.sysconf("SC_PHYS_PAGES") / 1e9
    except (ValueError, OSError):
        host_gb = 0.0
    if dev_gb >= 150 and host_gb >= 130:
        return "C5", ""
    return "C4", f" [fallback: C5 needs >= 150 GB of HBM and >= 130 GB of host memory; this box has {dev_gb:.0f} / {host_gb:.0f} GB]"


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle on the same config/metric; each step a bounded sample of the workload."""
    if rank != 0:
        return
    import torch
    from oracle import Oracle, threads_used
    from workloads import CONFIGS, make_workload
    note = ""
    if args.config is None:
        args.config, note = choose_default_config()
    spec = CONFIGS[args.config]
    steps, warmup = effective_counts(args.config, args.steps, args.warmup)
    # the seeded input generator (plain torch, none of this repo's kernels) runs on the GPU when there is one: generating
    # 58 GB of orbitals on the host cores would take longer than the whole measurement
    gen_dev = "cuda" if (torch.cuda.is_available() and spec.n_orb * spec.n_points * 8 > 2e9) else "cpu"
    w = make_workload(spec, device=gen_dev)
    psi = w["psi"].cpu().numpy()
    del w["psi"]
    if gen_dev == "cuda":
        torch.cuda.empty_cache()
    o = Oracle(spec.dims, spec.spacing, spec.bc, w["kernel"])
    cores = os.cpu_count() or 1
    rng = np.random.default_rng(999)
    n_solves = 2 * cores if spec.n_points <= 96 ** 3 else cores

    def step():
        pairs = [(int(a), int(b)) for a, b in rng.integers(0, spec.n_orb, size=(n_solves, 2))]
        o.pair_energies(psi, pairs)
    steps = min(steps if args.steps is None else int(args.steps), 20)
    for _ in range(min(warmup, 3)):
        step()
    t0 = time.perf_counter()
    for _ in range(steps):
        step()
    dt = (time.perf_counter() - t0) / steps
    value = n_solves / dt
    sample = f"{n_solves} seeded random pair solves of {spec.name} per step"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": min(warmup, 3), "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": _config_dict(spec, 1, "replicas", note),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads_used(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------ the product arm
def measure_resident(name, steps, warmup, local_rank, barrier, batch=0, n_orb=0):
    """Device-resident measurement of one configuration.  Returns (result dict, state) where state keeps the workload,
    the plan and the device tensors alive for the caller (e2e, cpu_baseline, cuFFT comparison)."""
    import torch

    import paper_1712_07973_b200 as exx
    from workloads import CONFIGS, make_workload
    spec = CONFIGS[name]
    if n_orb > 0:                                                   # development runs only: same grid, fewer orbitals
        from workloads import small_spec
        spec = small_spec(name, n_orb=n_orb, name=f"{name}-dev{n_orb}", orthonormalize=False)
    w = make_workload(spec, device="cuda")
    psi, occ = w["psi"], w["occ"]
    kpsi = torch.empty_like(psi)
    stream = torch.cuda.current_stream().cuda_stream
    plan = exx.ExxPlan(spec.dims, spec.spacing, spec.bc, w["kernel"], max_orbitals=spec.n_orb, stream=stream)
    if batch > 0:
        plan.set_batch(batch)
    n_pairs, n_xforms = exx.exx_schedule_pairs(occ)
    ex_dev = torch.zeros(1, dtype=torch.float64, device="cuda")
    for _ in range(warmup):
        plan.apply_async(psi, occ, kpsi, ex_dev)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    launches0 = plan.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(steps):                                          # profiling events are OFF in the timed region
        plan.apply_async(psi, occ, kpsi, ex_dev)
    ev1.record()
    barrier()
    elapsed_ms = ev0.elapsed_time(ev1)
    launches = plan.launch_count() - launches0
    clocks = sampler.stop()
    ex_value = float(ex_dev[0])
    # per-pass device times: one extra step with CUDA events around every pass launch (outside the timed region)
    plan.set_profiling(True)
    plan.apply_async(psi, occ, kpsi, ex_dev)
    pass_ms, pass_n = plan.get_profile()
    plan.set_profiling(False)
    pass_ms, pass_n = np.array(pass_ms), np.array(pass_n)
    res = {"spec": spec, "n_pairs": n_pairs, "n_xforms": n_xforms, "step_ms_local": elapsed_ms / steps, "launches": int(launches),
           "clocks": clocks, "E_x": ex_value, "pass_ms": pass_ms, "pass_n": pass_n, "steps": steps, "warmup": warmup,
           "workspace_bytes": plan.workspace_bytes(), "kernels": [plan.kernel_name(k) for k in range(3)]}
    return res, {"w": w, "plan": plan, "psi": psi, "kpsi": kpsi, "occ": occ, "ex_dev": ex_dev}


def roofline_objects(res, step_ms, fp64):
    """`roofline` (dominant kernel) and `roofline_path` (whole path against north_star's definition)."""
    spec, n_pairs, n_xforms = res["spec"], res["n_pairs"], res["n_xforms"]
    pass_ms, pass_n = res["pass_ms"], res["pass_n"]
    peak, peak_src = _peaks()
    per_x = alg_bytes_per_transform(spec)
    flops_x = nominal_flops_per_transform(spec)
    names = ["A", "B", "C"]
    dom = int(np.argmax(pass_ms[:3]))
    dom_name = names[dom]
    n_launch = max(1, int(pass_n[dom]))
    dom_ms = pass_ms[dom] / n_launch
    dom_bytes = per_x[dom_name] * n_xforms / n_launch
    dom_flops = flops_x[dom_name] * n_xforms / n_launch
    achieved_gbs = dom_bytes / (dom_ms * 1e-3) / 1e9
    achieved_tf = dom_flops / (dom_ms * 1e-3) / 1e12
    t_hbm = dom_bytes / (peak * 1e9)
    fp_peak = fp64["dfma_tflops"] if fp64 else 37.2
    t_fp = dom_flops / (fp_peak * 1e12)
    bound = "hbm" if t_hbm >= t_fp else "alu"
    roofline = {"bound": bound, "kernel": res["kernels"][dom],
                "achieved": achieved_gbs if bound == "hbm" else achieved_tf,
                "peak": peak if bound == "hbm" else fp_peak,
                "unit": "GB/s" if bound == "hbm" else "TFLOP/s",
                "frac": (achieved_gbs / peak) if bound == "hbm" else (achieved_tf / fp_peak),
                "traffic": _ncu_traffic(spec.name, dom_name, n_xforms / n_launch),
                "peak_source": peak_src if bound == "hbm" else "measured DFMA rate (exx_diag_fp64, this run)",
                "alg_bytes_per_launch": dom_bytes, "nominal_flops_per_launch": dom_flops, "ms_per_launch": dom_ms,
                "t_hbm_ms": t_hbm * 1e3, "t_fp64_ms": t_fp * 1e3, "hbm_frac": achieved_gbs / peak, "fp64_frac": achieved_tf / fp_peak,
                "pass_ms_per_step": {k: float(v) for k, v in zip(["A", "B", "C", "reduce"], pass_ms)},
                "pass_GBps": {k: float(per_x[k] * n_xforms / (pass_ms[i] * 1e-3) / 1e9) for i, k in enumerate(names)},
                "pass_nominal_TFLOPs": {k: float(flops_x[k] * n_xforms / (pass_ms[i] * 1e-3) / 1e12) for i, k in enumerate(names)}}
    # whole path: two fractions side by side -- SURVEY's B_alg (the north_star numerator, a two-streamed-orbital model) and
    # the bytes the row-pair kernels really move (smaller: one streamed orbital per transform)
    b_alg_pair = survey_b_alg_per_pair(spec)
    path_gbs = b_alg_pair * n_pairs / (step_ms * 1e-3) / 1e9
    moved_gbs = sum(per_x.values()) * n_xforms / (step_ms * 1e-3) / 1e9
    flops_pair = sum(flops_x.values()) * n_xforms / max(1, n_pairs)
    t_hbm_pair, t_fp_pair = b_alg_pair / (HBM_SPEC_GBS * 1e9), flops_pair / (fp_peak * 1e12)
    roofline_path = {"definition": "north_star: per pair, the slower of B_alg / 8 TB/s and nominal flops / FP64 peak",
                     "alg_bytes_per_pair": b_alg_pair, "nominal_flops_per_pair": flops_pair,
                     "t_hbm_us_per_pair": t_hbm_pair * 1e6, "t_fp64_us_per_pair": t_fp_pair * 1e6,
                     "bound": "hbm" if t_hbm_pair >= t_fp_pair else "alu",
                     "frac_of_roofline": max(t_hbm_pair, t_fp_pair) / (step_ms * 1e-3 / n_pairs),
                     "achieved_GBps": path_gbs, "frac_of_8TBps_spec": path_gbs / HBM_SPEC_GBS, "frac_of_measured_copy": path_gbs / peak,
                     "target_frac_of_spec": 0.60,
                     "bytes_moved_per_pair_model": sum(per_x.values()) * n_xforms / max(1, n_pairs), "moved_GBps": moved_gbs,
                     "moved_frac_of_8TBps_spec": moved_gbs / HBM_SPEC_GBS, "moved_frac_of_measured_copy": moved_gbs / peak}
    return roofline, roofline_path


def run_ours(args, rank, local_rank, world):
    import torch
    import torch.distributed as dist

    import paper_1712_07973_b200 as exx

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    distributed = world > 1
    if distributed:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if distributed:
            dist.barrier()
        torch.cuda.synchronize()

    def all_reduce_max(x: float) -> float:
        t = torch.tensor([x], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t[0])

    note = ""
    if args.config is None:
        args.config, note = choose_default_config()
    if args.parallel == "rr" and distributed:
        run_round_robin(args, rank, local_rank, world, dist, barrier, all_reduce_max, note)
        dist.destroy_process_group()
        return
    fp64 = exx.exx_diag_fp64(torch.cuda.current_stream().cuda_stream)
    fp64.update(exx.exx_diag_shfl(torch.cuda.current_stream().cuda_stream))

    # ---- the other target configurations, same run, device-resident only
    per_config = {}
    others = [] if (args.no_per_config or args.config not in ("C4", "C5")) else [c for c in ("C3", "C4") if c != args.config]
    for name in others:
        k, wu = effective_counts(name, None, 3)
        res, st = measure_resident(name, k, wu, local_rank, barrier)
        step_ms, value = aggregate_over_ranks(res["step_ms_local"], res["n_pairs"], world, all_reduce_max if distributed else None)
        rl, rp = roofline_objects(res, step_ms, fp64)
        per_config[name] = {"workload": _workload_name(res["spec"]), "value": value, "unit": UNIT, "ms_per_step": step_ms, "steps": k, "warmup": wu,
                            "frac_of_8TBps_spec": rp["frac_of_8TBps_spec"], "frac_of_measured_copy": rp["frac_of_measured_copy"],
                            "moved_frac_of_measured_copy": rp["moved_frac_of_measured_copy"], "frac_of_roofline": rp["frac_of_roofline"],
                            "bound": rp["bound"], "clocks": res["clocks"], "dominant_kernel": rl["kernel"], "dominant_hbm_frac": rl["hbm_frac"],
                            "dominant_fp64_frac": rl["fp64_frac"], "pass_ms_per_step": rl["pass_ms_per_step"], "E_x": res["E_x"]}
        st["plan"].destroy()
        del st, res
        torch.cuda.empty_cache()

    # ---- the headline configuration
    steps, warmup = effective_counts(args.config, args.steps, args.warmup, args.quick)
    res, st = measure_resident(args.config, steps, warmup, local_rank, barrier, args.batch, args.dev_orbitals)
    spec = res["spec"]
    step_ms, value = aggregate_over_ranks(res["step_ms_local"], res["n_pairs"], world, all_reduce_max if distributed else None)
    roofline, roofline_path = roofline_objects(res, step_ms, fp64)
    plan, psi, kpsi, occ = st["plan"], st["psi"], st["kpsi"], st["occ"]
    n_pairs = res["n_pairs"]

    cufft = None
    if rank == 0 and world == 1 and args.compare_cufft and psi.numel() * 8 <= 24e9:
        plan.apply_async(psi, occ, kpsi, st["ex_dev"])
        cufft = cufft_comparison(spec, psi, occ, st["w"]["kernel"], plan.pair_energies(spec.n_orb))

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region.  The library stages
    # psi and K psi in device memory of its own, so the bench's device copies are released first (C5: 2 x 58 GB).
    nbytes = psi.numel() * 8
    host_budget = 0.0
    try:
        host_budget = os.sysconf("SC_PAGE_SIZE") * os.sysconf("SC_AVPHYS_PAGES") * 0.8
    except (ValueError, OSError):
        pass
    psi_h = None
    pinned = True
    need_host = not args.no_e2e or (rank == 0 and world == 1 and not args.no_cpu_baseline)
    if need_host and 2 * nbytes * (world if distributed else 1) <= max(host_budget, 8e9):
        try:
            psi_h = torch.empty(psi.shape, dtype=torch.float64, pin_memory=True)
        except RuntimeError:
            pinned = False
            psi_h = torch.empty(psi.shape, dtype=torch.float64)
        psi_h.copy_(psi)
    e2e = None
    if not args.no_e2e:
        if psi_h is None:
            e2e = {"value": None, "unit": UNIT, "note": "host memory cannot hold psi and K psi for every rank of this run"}
        else:
            del psi, kpsi
            st["psi"] = st["kpsi"] = None
            torch.cuda.empty_cache()
            try:
                kpsi_h = torch.empty(psi_h.shape, dtype=torch.float64, pin_memory=pinned)
            except RuntimeError:
                pinned = False
                kpsi_h = torch.empty(psi_h.shape, dtype=torch.float64)
            psi_np, kpsi_np = psi_h.numpy(), kpsi_h.numpy()
            e2e_steps = 1 if args.config == "C5" else max(1, min(steps, 3))
            plan.apply_host(psi_np, occ, kpsi_np)                   # untimed: grows the library's device staging
            barrier()
            t0 = time.perf_counter()
            for _ in range(e2e_steps):
                _, ex_h = plan.apply_host(psi_np, occ, kpsi_np)
            barrier()
            dt = torch.tensor([(time.perf_counter() - t0) / e2e_steps], dtype=torch.float64, device="cuda")
            if distributed:
                dist.all_reduce(dt, op=dist.ReduceOp.MAX)
            e2e = {"value": n_pairs * world / float(dt[0]), "unit": UNIT, "h2d_bytes_per_step": int(nbytes + occ.nbytes),
                   "d2h_bytes_per_step": int(nbytes + 8), "ms_per_step": float(dt[0]) * 1e3, "steps": e2e_steps,
                   "api": "exx_apply_host (%s host buffers; the library stages psi and K psi in its own device memory)" % ("pinned" if pinned else "pageable")}
            assert abs(ex_h - res["E_x"]) <= 1e-12 * abs(res["E_x"])
            plan.release_staging()
            del kpsi_h, kpsi_np

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline and psi_h is not None:
        cpu = cpu_baseline(spec, st["w"]["kernel"], psi_h.numpy())

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
                "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
                "data": "synthetic", "config": _config_dict(spec, world, args.parallel, note),
                "steps_requested": args.steps, "warmup_requested": args.warmup,
                "details": {"packed_transforms": res["n_xforms"], "workspace_bytes": res["workspace_bytes"], "kernels": res["kernels"]},
                "apply_seconds": step_ms * 1e-3, "E_x": res["E_x"], "clocks": res["clocks"], "gpu_launches": res["launches"],
                "e2e": e2e, "roofline": roofline, "roofline_path": roofline_path, "fp64_peak_measured": fp64,
                "per_config": per_config, "cpu_baseline": cpu, "cufft_comparison": cufft}
        if args.dev_orbitals:
            line["dev"] = f"development run with {args.dev_orbitals} orbitals instead of the configuration's: not a bench value"
        if args.quick:
            line["quick"] = "profiling run (1 warm-up step, 1 timed step): not a bench value"
        print(json.dumps(line))
    plan.destroy()
    if distributed:
        dist.destroy_process_group()


def run_round_robin(args, rank, local_rank, world, dist, barrier, all_reduce_max, note):
    """--parallel rr: ONE workload, its orbitals distributed round-robin over the ranks (strong
    scaling).  Every rank generates the seeded workload and keeps its own block."""
    import torch

    import paper_1712_07973_b200 as exx
    from paper_1712_07973_b200.distributed import CudaBlockBackend, block_range, round_robin_apply
    from workloads import CONFIGS, make_workload
    spec = CONFIGS[args.config]
    steps, warmup = effective_counts(args.config, args.steps, args.warmup)
    w = make_workload(spec, device="cuda")
    lo, hi = block_range(spec.n_orb, world, rank)
    psi_own = w["psi"][lo:hi].clone()
    del w["psi"]
    torch.cuda.empty_cache()
    n_max = max(block_range(spec.n_orb, world, r)[1] - block_range(spec.n_orb, world, r)[0] for r in range(world))
    plan = exx.ExxPlan(spec.dims, spec.spacing, spec.bc, w["kernel"], max_orbitals=n_max, stream=torch.cuda.current_stream().cuda_stream)
    backend = CudaBlockBackend(plan)
    for _ in range(warmup):
        round_robin_apply(backend, psi_own, w["occ"], rank, world, dist)
    sampler = ClockSampler(local_rank)
    sampler.start()
    launches0 = plan.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(steps):
        _, ex = round_robin_apply(backend, psi_own, w["occ"], rank, world, dist)
    ev1.record()
    barrier()
    step_ms = all_reduce_max(ev0.elapsed_time(ev1) / steps)
    clocks = sampler.stop()
    if rank == 0:
        line = {"metric": METRIC, "value": spec.n_pairs / (step_ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
                "ms_per_step": step_ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64",
                "data": "synthetic", "config": _config_dict(spec, world, "rr", note), "E_x": ex, "clocks": clocks,
                "gpu_launches": int(plan.launch_count() - launches0), "e2e": None, "roofline": None, "cpu_baseline": None}
        print(json.dumps(line))
    plan.destroy()


def _spawn_entry(local_rank, world, port, argv):
    os.environ.update({"RANK": str(local_rank), "LOCAL_RANK": str(local_rank), "WORLD_SIZE": str(world),
                       "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    sys.argv = argv
    main()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default=None, choices=["C1", "C2", "C3", "C4", "C5"],
                    help="default: C5 when the box can hold it (>= 150 GB HBM, >= 130 GB host memory), else C4")
    ap.add_argument("--parallel", default="replicas", choices=["replicas", "rr"], help="N > 1: independent replicas, or round-robin orbital blocks")
    ap.add_argument("--batch", type=int, default=0, help="max packed transforms per batch (0 = library default)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the C3 / C4 lines of per_config")
    ap.add_argument("--quick", action="store_true", help="profiling runs: 1 warm-up + 1 timed step, no per_config / e2e / cpu_baseline")
    ap.add_argument("--dev-orbitals", type=int, default=0, help="development runs: the configuration's grid with this many orbitals (not a bench value)")
    ap.add_argument("--compare-cufft", action="store_true", help="also time a torch.fft (cuFFT) pipeline on a sample, as a comparison")
    args = ap.parse_args()

    if args.quick or args.dev_orbitals:
        args.no_per_config = args.no_e2e = args.no_cpu_baseline = True
    rank, local_rank, world, spawn = rank_env(args.gpus)
    if spawn and args.impl == "ours":
        # plain `python bench.py --gpus N`: start the N ranks here (what torchrun would do), one process per GPU
        import torch.multiprocessing as mp
        with socket.socket() as s:
            s.bind(("127.0.0.1", 0))
            port = s.getsockname()[1]
        mp.spawn(_spawn_entry, args=(args.gpus, port, list(sys.argv)), nprocs=args.gpus, join=True)
        return
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    run_ours(args, rank, local_rank, world)


if __name__ == "__main__":
    main()
