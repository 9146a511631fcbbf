#!/usr/bin/env python
"""bench.py -- exact-exchange apply throughput on B200 (contract: see DESIGN.md "Measurement").

A step = one pass of the whole hot path (pair scheduling, pass A, pass B, pass C, energy reduction) over one
synthetic workload, i.e. one exx_apply of all N(N+1)/2 orbital pairs.  `value` = pair-solves/s with the orbitals
resident in HBM; `e2e` = the same metric through exx_apply_host (pinned host buffers, H2D of psi and D2H of K psi
inside the timed region).  N > 1 GPUs: replicas only, one process per GPU under torchrun,
barrier + max-over-ranks timing, value = pairs of all ranks / that time.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C3] [--impl ours|reference]
"""
from __future__ import annotations

import argparse
import json
import os
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
DEFAULT_CONFIG = "C3"


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def _ncu_traffic(config: str, pass_name: str, xforms_per_launch: float):
    """dram__bytes_read+write per launch of the dominant kernel from the committed `ncu --set full` capture
    (profiles/r01_traffic.csv: config,pass,transforms_in_launch,dram_bytes), scaled to this run's mean launch size."""
    path = os.path.join(ROOT, "profiles", "r01_traffic.csv")
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
    resident orbitals psi_j, psi_l / K psi_j, K psi_l of a batch and K^ (L2-resident) are amortised to zero.  Pass B's
    figure (2 I) is the one SURVEY.md 8(d) counts; passes A and C move LESS than SURVEY's model (which streams two
    orbitals per transform), so the whole-path fraction below keeps SURVEY's B_alg as the numerator.
    """
    M = spec.n_points
    inter = 16 * M * (4 if spec.bc == "free" else 1)
    return {"A": 8 * M + inter, "B": 2 * inter, "C": inter + 8 * M + 16 * M}


def survey_b_alg_per_pair(spec):
    """SURVEY.md 8(d) B_alg per pair-solve: 64 M bytes (periodic), 160 M bytes (free)."""
    return (160 if spec.bc == "free" else 64) * spec.n_points


def cpu_baseline(spec, w, seconds_target=15.0):
    """The oracle, as it stands, timed on this host's cores on a bounded sample of the same workload."""
    from oracle import Oracle, threads_used
    o = Oracle(spec.dims, spec.spacing, spec.bc, w["kernel"])
    n_orb = spec.n_orb
    psi = w["psi"].cpu().numpy() if hasattr(w["psi"], "cpu") else w["psi"]
    rng = np.random.default_rng(12345)
    cores = os.cpu_count() or 1
    first = [(int(a), int(b)) for a, b in rng.integers(0, n_orb, size=(cores, 2))]
    t0 = time.perf_counter()
    o.pair_energies(psi, first)
    t1 = time.perf_counter() - t0
    n_more = int(max(0, min(64 * cores, (seconds_target - t1) / max(t1, 1e-3) * cores)))
    n_more -= n_more % cores
    total_solves, total_time = len(first), t1
    if n_more > 0:
        more = [(int(a), int(b)) for a, b in rng.integers(0, n_orb, size=(n_more, 2))]
        t0 = time.perf_counter()
        o.pair_energies(psi, more)
        total_time += time.perf_counter() - t0
        total_solves += n_more
    return {"value": total_solves / total_time, "unit": UNIT, "cores": threads_used(), "kind": "oracle",
            "sample": f"{total_solves} seeded random pair solves (co-density, padded 3-D FFT Poisson solve, energy) of {spec.name}, "
                      f"{total_time:.1f} s wall"}


def cufft_comparison(spec, psi, occ, kernel_table, plan_pair_energies, seconds_target=2.0):
    """GPU comparison baseline ("the cuFFT path ... same inputs, same metric"; reported, never the
    product): the textbook pipeline on library calls -- co-densities as a torch product, torch.fft.rfftn / irfftn
    (cuFFT D2Z / Z2D, zero-padded to 2n for free BC), pointwise multiply by K^, pointwise epilogue -- timed on a bounded
    sample of rows i (all j >= i of a row, batched).  Returns pair-solves/s and a sanity check against the library."""
    import torch
    n = spec.dims
    free = spec.bc == "free"
    t = tuple(2 * d for d in n) if free else tuple(n)
    dev = psi.device
    if free:
        g = torch.as_tensor(kernel_table, dtype=torch.float64, device=dev)
        ext = torch.zeros(t, dtype=torch.float64, device=dev)
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
    return {"value": pairs / (ms * 1e-3), "unit": UNIT, "kind": "torch.fft (cuFFT D2Z/Z2D) + pointwise torch ops, one real co-density per transform",
            "sample": f"{pairs} pair solves ({len(rows) - 1} seeded rows i, all j >= i), {ms * 1e-3:.2f} s device time",
            "max_rel_err_pair_energies_row0_vs_library": err}


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle on the same config/metric; each step a bounded sample of the workload."""
    if rank != 0:
        return
    from oracle import Oracle, threads_used
    from workloads import CONFIGS, make_workload
    spec = CONFIGS[args.config]
    w = make_workload(spec, device="cpu")
    o = Oracle(spec.dims, spec.spacing, spec.bc, w["kernel"])
    psi = w["psi"].numpy()
    cores = os.cpu_count() or 1
    rng = np.random.default_rng(999)
    n_solves = 2 * cores if spec.n_points <= 96 ** 3 else cores
    def step():
        pairs = [(int(a), int(b)) for a, b in rng.integers(0, spec.n_orb, size=(n_solves, 2))]
        o.pair_energies(psi, pairs)
    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = (time.perf_counter() - t0) / args.steps
    value = n_solves / dt
    sample = f"{n_solves} seeded random pair solves of {spec.name} per step"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": {"workload": _workload_name(spec)},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads_used(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))


def _workload_name(spec):
    t = "x".join(str(d) for d in spec.dims)
    return f"{spec.name}: {spec.bc} {t} grid, h={spec.spacing[0]} bohr, {spec.n_orb} orbitals, {spec.n_pairs} pairs"


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default=DEFAULT_CONFIG, choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--batch", type=int, default=0, help="max packed transforms per batch (0 = library default)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--compare-cufft", action="store_true", help="also time a torch.fft (cuFFT) pipeline on a sample, as a comparison")
    args = ap.parse_args()
    if args.steps is None:
        args.steps = {"C1": 20, "C2": 10, "C3": 5, "C4": 3, "C5": 1}[args.config]
    if args.warmup < 3 and args.config != "C5":
        args.warmup = max(args.warmup, 1)

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist

    import paper_1712_07973_b200 as exx
    from workloads import CONFIGS, make_workload

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    distributed = world > 1
    if distributed:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    spec = CONFIGS[args.config]
    w = make_workload(spec, device="cuda")
    psi, occ = w["psi"], w["occ"]
    kpsi = torch.empty_like(psi)
    stream = torch.cuda.current_stream().cuda_stream
    plan = exx.ExxPlan(spec.dims, spec.spacing, spec.bc, w["kernel"], max_orbitals=spec.n_orb, stream=stream)
    if args.batch > 0:
        plan.set_batch(args.batch)
    n_pairs, n_xforms = exx.exx_schedule_pairs(occ)
    ex_dev = torch.zeros(1, dtype=torch.float64, device="cuda")

    def barrier():
        if distributed:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing (value)
    for _ in range(args.warmup):
        plan.apply_async(psi, occ, kpsi, ex_dev)
    barrier()
    plan.set_profiling(True)
    sampler = ClockSampler(local_rank)
    sampler.start()
    launches0 = plan.launch_count()
    pass_ms = np.zeros(4)
    pass_n = np.zeros(4, dtype=np.int64)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(args.steps):
        plan.apply_async(psi, occ, kpsi, ex_dev)
    ev1.record()
    barrier()
    elapsed_ms = ev0.elapsed_time(ev1)
    ms, n = plan.get_profile()                    # events of the LAST timed step (same launches every step)
    pass_ms += np.array(ms)
    pass_n += np.array(n)
    launches = plan.launch_count() - launches0
    clocks = sampler.stop()
    plan.set_profiling(False)
    ex_value = float(ex_dev[0])
    def all_reduce_max(x: float) -> float:
        t = torch.tensor([x], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t[0])

    step_ms, value = aggregate_over_ranks(elapsed_ms / args.steps, n_pairs, world, all_reduce_max if distributed else None)

    # ---- roofline of the dominant kernel (per-launch algorithmic bytes / mean launch duration)
    peak, peak_src = _peaks()
    per_x = alg_bytes_per_transform(spec)
    names = ["A", "B", "C"]
    dom = int(np.argmax(pass_ms[:3]))
    dom_name = names[dom]
    dom_ms_per_launch = pass_ms[dom] / max(1, pass_n[dom])
    dom_bytes_per_launch = per_x[dom_name] * n_xforms / max(1, pass_n[dom])
    achieved = dom_bytes_per_launch / (dom_ms_per_launch * 1e-3) / 1e9
    kernel_name = plan.kernel_name(dom)
    roofline = {"bound": "hbm", "kernel": kernel_name, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": _ncu_traffic(args.config, dom_name, n_xforms / max(1, pass_n[dom])),
                "peak_source": peak_src,
                "alg_bytes_per_launch": dom_bytes_per_launch, "ms_per_launch": dom_ms_per_launch,
                "pass_ms_per_step": {k: float(v) for k, v in zip(["A", "B", "C", "reduce"], pass_ms)},
                "pass_GBps": {k: float(per_x[k] * n_xforms / (pass_ms[i] * 1e-3) / 1e9) for i, k in enumerate(names)}}
    # whole-path figure against north_star's definition (B_alg per pair / 8 TB/s spec)
    b_alg_pair = survey_b_alg_per_pair(spec)
    path_gbs = b_alg_pair * n_pairs / (step_ms * 1e-3) / 1e9
    moved_gbs = sum(per_x.values()) * n_xforms / (step_ms * 1e-3) / 1e9
    roofline_path = {"alg_bytes_per_pair": b_alg_pair, "achieved_GBps": path_gbs, "frac_of_8TBps_spec": path_gbs / 8000.0,
                     "frac_of_measured_copy": path_gbs / peak, "target_frac_of_spec": 0.60,
                     "bytes_moved_per_pair_model": sum(per_x.values()) * n_xforms / max(1, n_pairs), "moved_GBps": moved_gbs}

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if not args.no_e2e:
        nbytes = psi.numel() * 8
        if nbytes <= 24e9:
            psi_h = torch.empty(psi.shape, dtype=torch.float64, pin_memory=True)
            psi_h.copy_(psi)
            kpsi_h = torch.empty(psi.shape, dtype=torch.float64, pin_memory=True)
            psi_np, kpsi_np = psi_h.numpy(), kpsi_h.numpy()
            e2e_steps = max(1, min(args.steps, 3))
            plan.apply_host(psi_np, occ, kpsi_np)
            barrier()
            t0 = time.perf_counter()
            for _ in range(e2e_steps):
                _, ex_h = plan.apply_host(psi_np, occ, kpsi_np)
            barrier()
            dt = torch.tensor([(time.perf_counter() - t0) / e2e_steps], dtype=torch.float64, device="cuda")
            if distributed:
                dist.all_reduce(dt, op=dist.ReduceOp.MAX)
            e2e = {"value": n_pairs * world / float(dt[0]), "unit": UNIT, "h2d_bytes_per_step": int(nbytes + occ.nbytes),
                   "d2h_bytes_per_step": int(nbytes + 8), "ms_per_step": float(dt[0]) * 1e3, "api": "exx_apply_host (pinned host buffers)"}
            assert abs(ex_h - ex_value) <= 1e-12 * abs(ex_value)
        else:
            e2e = {"value": None, "unit": UNIT, "note": "orbitals exceed the pinned-host staging budget of this bench"}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(spec, w)
    cufft = None
    if rank == 0 and world == 1 and args.compare_cufft and psi.numel() * 8 <= 24e9:
        plan.apply_async(psi, occ, kpsi, ex_dev)
        cufft = cufft_comparison(spec, psi, occ, w["kernel"], plan.pair_energies(spec.n_orb))

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
                "data": "synthetic",
                "config": {"workload": _workload_name(spec), "pairs": n_pairs, "packed_transforms": n_xforms,
                           "l2_policy": "inputs larger than L2 (orbitals %.2f GB)" % (psi.numel() * 8 / 1e9),
                           "parallelism": "replicas" if world > 1 else "single GPU",
                           "workspace_bytes": plan.workspace_bytes()},
                "apply_seconds": step_ms * 1e-3, "E_x": ex_value, "clocks": clocks, "gpu_launches": int(launches),
                "e2e": e2e, "roofline": roofline, "roofline_path": roofline_path, "cpu_baseline": cpu, "cufft_comparison": cufft}
        print(json.dumps(line))
    plan.destroy()
    if distributed:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
