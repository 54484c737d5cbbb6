#!/usr/bin/env python
"""Benchmark of the POLFED hot path on B200 (contract: see the task statement / DESIGN.md).

One "step" = one pass of the whole hot path over one block: polfed_filter_apply with a filter
of order K_filter on BASELINE.json config 5 (spinless fermions L=26, N=13, D=10 400 600,
nnz=275 407 888, s=32), i.e. one scaled copy + K_filter fused SpMM+Clenshaw launches.
metric = algorithmic GB/s of that pass, bytes per fused launch = nnz*12 + 4(N+1) + 32*s*N
(the first launch of a pass has no b_{k+2} read and is counted without it).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--order K_filter]
  python bench.py --impl reference ...      # the CPU oracle on a bounded sample of the workload
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

import workloads  # noqa: E402  (seeded parameters only; no arithmetic of the method)

METRIC = "fused_spmm_clenshaw_algorithmic_bandwidth"
UNIT = "GB/s"
NOMINAL_HBM_GBS = 8000.0          # BASELINE.json north_star: "B200's ~8 TB/s peak"
FALLBACK_HBM_GBS = 6650.0         # B200_PROFILING.md fallback
WORKLOAD_NAMES = {1: "config1_xxz_L12_s1", 2: "config2_xxz_L16_s8", 3: "config3_xxz_L20_s16",
                  4: "config4_quantum_sun_2^20_s16", 5: "config5_fermions_L26_N13_s32"}


def step_bytes(n: int, nnz: int, s: int, with_z: bool = True, with_v: bool = True) -> int:
    """Algorithmic bytes of one fused launch: CSR once, X read, Y written, Z and V read
    (nnz*12 + 4(N+1) + 8*s*N*4 for the full recurrence step)."""
    return nnz * 12 + 4 * (n + 1) + 8 * s * n * (2 + int(with_z) + int(with_v))


def pass_bytes(n: int, nnz: int, s: int, coeffs) -> int:
    """One filter application of order K >= 1: the scaled copy b_K = c_K V, then K fused launches.
    The first launch has no b_{k+2}; a launch whose coefficient is exactly zero (every odd k
    when lambda~ = 0) has no V term, and the library does not read V for it."""
    K = len(coeffs) - 1
    total = 16 * s * n
    for k in range(K - 1, -1, -1):
        total += step_bytes(n, nnz, s, with_z=(k != K - 1), with_v=(coeffs[k] != 0.0))
    return total


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def recorded_traffic(workload: str):
    """DRAM bytes per launch of the dominant kernel from the committed ncu capture, or None."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as fh:
            return json.load(fh).get(workload)
    except Exception:
        return None


def replica_seed(config: int, rank: int) -> int:
    """Weak scaling over replicas: rank r filters its own disorder realisation."""
    return 1000 + config + 100 * rank


def reduce_max(value: float, device="cpu") -> float:
    """MAX over ranks of a per-rank time (identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_gbs(bytes_per_rank: int, world: int, seconds_max: float) -> float:
    """Aggregate throughput: what all ranks processed / the slowest rank's time."""
    return bytes_per_rank * world / seconds_max / 1e9


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""

    QUERY = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.lines, self.proc = index, [], None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.QUERY}",
                 "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None
        return self

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def __exit__(self, *exc):
        if self.proc is not None:
            time.sleep(0.25)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.lines:
            parts = [p.strip() for p in line.split(",")]
            if len(parts) < 6:
                continue
            try:
                sm.append(float(parts[0]))
                mx.append(float(parts[1]))
            except ValueError:
                continue
            for name, flag in zip(names, parts[2:6]):
                if flag.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)),
                "reasons": sorted(reasons), "samples": len(sm)}


# ---- CPU oracle legs (the only places bench.py executes oracle/) -------------------------------

def oracle_sample(config: int, rows_target: int, seed: int):
    """First `rows_target` rows of the workload's matrix and full-size random blocks."""
    from oracle import core
    w = workloads.make_workload(config)
    states = core.basis_states(w.n_sites, w.n_up)
    n = int(states.shape[0])
    m = min(n, rows_target)
    mini = core.build_csr_rows(states, np.arange(m, dtype=np.int64), w.terms, w.dot_bits, w.dot_dense)
    rng = np.random.Generator(np.random.PCG64(seed))
    B1 = rng.standard_normal((n, w.s))
    V = rng.standard_normal((m, w.s))
    B2 = rng.standard_normal((m, w.s))
    T = np.empty((m, w.s))
    return w, n, mini, B1, B2, V, T


def oracle_time_steps(mini, w, B1, B2, V, T, n_steps: int):
    from oracle import core
    t0 = time.perf_counter()
    for k in range(n_steps):
        core.clenshaw_step(mini, 0.3, 17.0, 1e-3 * (k + 1), V, B1, B2, T)
    return time.perf_counter() - t0


def cpu_baseline(config: int, budget_s: float = 12.0):
    """Oracle recurrence steps (orc_clenshaw_step, as it stands) on the first rows of the workload,
    on all host cores and (the same library, OpenMP told to use one thread) on a single core."""
    import ctypes
    from oracle import core
    rows = {1: 924, 2: 12870, 3: 184756, 4: 262144, 5: 262144}[config]
    w, n, mini, B1, B2, V, T = oracle_sample(config, rows, seed=7000 + config)
    by = step_bytes(mini.n, mini.nnz, w.s)

    def timed(budget):
        oracle_time_steps(mini, w, B1, B2, V, T, 1)
        t1 = oracle_time_steps(mini, w, B1, B2, V, T, 2) / 2
        n_steps = int(max(3, min(200, budget / max(t1, 1e-6))))
        return oracle_time_steps(mini, w, B1, B2, V, T, n_steps) / n_steps, n_steps

    cores = core.num_threads()
    t, n_steps = timed(budget_s)
    single = None
    try:
        gomp = ctypes.CDLL("libgomp.so.1")
        gomp.omp_set_num_threads(1)
        t_single, n_single = timed(budget_s / 2)
        gomp.omp_set_num_threads(cores)
        single = {"value": by / t_single / 1e9, "unit": UNIT, "cores": 1, "steps": n_single,
                  "ms_per_recurrence_step": t_single * 1e3}
    except OSError:
        pass
    return {"value": by / t / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{n_steps} recurrence steps (orc_clenshaw_step) on rows [0,{mini.n}) of "
                      f"{WORKLOAD_NAMES[config]} (nnz {mini.nnz}), full-size X block, "
                      f"{t * 1e3:.2f} ms/step",
            "ms_per_recurrence_step": t * 1e3, "single_thread": single}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle import core
    rows = {1: 924, 2: 12870, 3: 184756, 4: 131072, 5: 131072}[args.config]
    w, n, mini, B1, B2, V, T = oracle_sample(args.config, rows, seed=7000 + args.config)
    order = max(1, min(args.order, 4))
    for _ in range(args.warmup):
        oracle_time_steps(mini, w, B1, B2, V, T, order)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_time_steps(mini, w, B1, B2, V, T, order)
    dt = time.perf_counter() - t0
    by = step_bytes(mini.n, mini.nnz, w.s) * order * args.steps
    value = by / dt / 1e9
    sample = (f"each step = {order} oracle recurrence steps on rows [0,{mini.n}) of "
              f"{WORKLOAD_NAMES[args.config]} (nnz {mini.nnz}), full-size X block")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT,
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD_NAMES[args.config], "N": n, "s": w.s, "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": core.num_threads(),
                             "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ---- the CUDA arm -----------------------------------------------------------------------------

def run_cuda(args):
    import torch
    import torch.distributed as dist

    import paper_2605_10191_b200 as P

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    P.lib()

    # weak scaling: every rank filters its own block of its own disorder realisation (8(e))
    w = workloads.make_workload(args.config, seed=replica_seed(args.config, rank))
    t0 = time.perf_counter()
    basis = P.polfed_build_basis(w.n_sites, w.n_up)
    # auto: the tiled format where the library supports it and the tiles are large enough to pay
    # (measured: config 5 4.8 vs 6.9 ms per step; config 3, tiles of <= 252 rows, 52 vs 35 us)
    tiled = args.format == "tiled" or (args.format == "auto" and w.n_up >= 0 and w.s in (16, 32)
                                       and not w.dot_bits and w.n_sites >= 24)
    # auto: the flip format (matrix-free rows) for full-space models it supports (config 4)
    flip = args.format == "flip" or (args.format == "auto" and w.n_up < 0 and w.s in (8, 16, 32)
                                     and all(t[0] in ("XX", "Z", "ZZ") for t in w.terms))
    fmt_name = "tiled" if tiled else ("flip" if flip else
                                      ("sector" if args.format == "sector" else "csr"))
    ham = P.polfed_build_hamiltonian(basis, w.terms, w.dot_bits, w.dot_dense,
                                     fmt={"tiled": P.FORMAT_TILED, "flip": P.FORMAT_FLIP,
                                          "csr": P.FORMAT_CSR,
                                          "sector": P.FORMAT_SECTOR}[fmt_name])
    tiled = tiled or fmt_name == "sector"     # same launch structure and timing method
    torch.cuda.synchronize()
    build_s = time.perf_counter() - t0
    n, nnz, s, K = ham.n, ham.nnz, w.s, args.order

    # a, b: the middle of the spectrum with a Gershgorin-safe half-width (the bench measures
    # throughput; parameter selection is not on the timed path).  lambda~ = 0.
    a, b = 0.0, 80.0
    coeffs = P.polfed_filter_coeffs(a, b, a, K_in=K)
    gen = torch.Generator(device="cuda").manual_seed(2000 + args.config + 100 * rank)
    V = torch.randn(n, s, dtype=torch.float64, device="cuda", generator=gen)
    V /= V.norm(dim=0, keepdim=True)
    W = torch.empty_like(V)
    work = torch.empty(P.polfed_filter_workspace_bytes_ham(ham, s) // 8, dtype=torch.float64,
                       device="cuda")

    def one_pass():
        P.polfed_filter_apply(ham, a, b, coeffs, s, V, W, work)

    def sync_all():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        one_pass()
    sync_all()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clocks:
        e0.record()
        for _ in range(args.steps):
            one_pass()
        e1.record()
        sync_all()
        ms = e0.elapsed_time(e1)
        # dominant kernel alone: back-to-back recurrence launches, events on the launching stream
        n_l = max(10, min(200, int(0.5e12 / max(step_bytes(n, nnz, s), 1))))
        k0, k1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        if tiled:
            # one sweep launch per recurrence step; the library has no single-sweep entry point,
            # so time two filter orders and divide the difference by the extra launches (the
            # pack kernel and the special first/last sweeps cancel).  All coefficients non-zero
            # so that every sweep reads V (the full-step byte count).
            c_short = np.full(9, 1e-3)
            c_long = np.full(9 + n_l, 1e-3)
            t_pair = []
            for cc in (c_short, c_long):
                P.polfed_filter_apply(ham, a, b, cc, s, V, W, work)
                k0.record()
                P.polfed_filter_apply(ham, a, b, cc, s, V, W, work)
                k1.record()
                torch.cuda.synchronize()
                t_pair.append(k0.elapsed_time(k1))
            kernel_ms = (t_pair[1] - t_pair[0]) / n_l
        else:
            B1, B2 = work[: n * s].view(n, s), work[n * s: 2 * n * s].view(n, s)
            B1.copy_(V)
            B2.copy_(V)
            for _ in range(3):
                P.polfed_fused_step(ham, s, 2.0 / b, -2.0 * a / b, -1.0, 1e-3, B1, B2, V, B2)
                B1, B2 = B2, B1
            k0.record()
            for _ in range(n_l):
                P.polfed_fused_step(ham, s, 2.0 / b, -2.0 * a / b, -1.0, 1e-3, B1, B2, V, B2)
                B1, B2 = B2, B1
            k1.record()
            torch.cuda.synchronize()
            kernel_ms = k0.elapsed_time(k1) / n_l
    ms = reduce_max(ms, "cuda")
    value = whole_job_gbs(pass_bytes(n, nnz, s, coeffs) * args.steps, world, ms * 1e-3)

    # end to end through the host-buffer entry point: H2D of V and D2H of W inside the region
    Vh = torch.empty(n, s, dtype=torch.float64).pin_memory()
    Wh = torch.empty(n, s, dtype=torch.float64).pin_memory()
    Vh.copy_(V)
    del W, work
    torch.cuda.empty_cache()
    e2e_steps = max(1, min(args.steps, 3))
    P.polfed_filter_apply_host(ham, a, b, coeffs, s, Vh, Wh)
    sync_all()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        P.polfed_filter_apply_host(ham, a, b, coeffs, s, Vh, Wh)
    sync_all()
    e2e_s = time.perf_counter() - t0
    e2e_value = whole_job_gbs(pass_bytes(n, nnz, s, coeffs) * e2e_steps, world,
                              reduce_max(e2e_s, "cuda"))
    checksum = float(Wh.double().abs().sum())

    if rank == 0:
        peak, peak_src = measured_peak()
        achieved = step_bytes(n, nnz, s) / (kernel_ms * 1e-3) / 1e9
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD_NAMES[args.config], "N": n, "nnz": nnz, "s": s,
                       "filter_order_per_step": K, "format": fmt_name,
                       # R22: launches of one pass whose coefficient is exactly 0 skip the V read
                       "launches_without_v_read": int(np.count_nonzero(coeffs[:K] == 0.0)),
                       "bytes_per_fused_launch": step_bytes(n, nnz, s),
                       "l2": "inputs exceed L2 (no flush)" if step_bytes(n, nnz, s) > 4 * 126e6
                             else "working set fits L2; not flushed (the filter re-reads it by design)",
                       "parallelism": f"replicas x{world}" if world > 1 else "single gpu",
                       "build_seconds": build_s},
            "filter_steps_per_s": K * args.steps * world / (ms * 1e-3),
            "frac_of_nominal_8TBps": value / world / NOMINAL_HBM_GBS,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 8 * s * n,
                    "d2h_bytes_per_step": 8 * s * n, "steps": e2e_steps, "checksum": checksum},
            "gpu_launches": args.steps * (K + 2 if tiled else K + 1),
            "clocks": clocks.summary(),
            "roofline": {"bound": "hbm",
                         "kernel": {"tiled": "tiled_sweep_kernel", "flip": "flip_step_kernel",
                                    "sector": "sector_sweep_kernel",
                                    "csr": "fused_step_kernel"}[fmt_name], "achieved": achieved,
                         "peak": peak, "peak_source": peak_src, "unit": UNIT,
                         "frac": achieved / peak, "frac_of_nominal_8TBps": achieved / NOMINAL_HBM_GBS,
                         "launch_ms": kernel_ms, "launches_timed": n_l,
                         "traffic": recorded_traffic(WORKLOAD_NAMES[args.config]
                                                    + "/" + fmt_name)},
        }
        if world == 1 and args.per_config:
            del Vh, Wh, V
            torch.cuda.empty_cache()
            todo = [(int(c), "") for c in args.per_config.split(",") if c and int(c) != args.config]
            line["per_config"] = [hot_path_on_config(P, c, peak, f) for c, f in todo]
            if args.config == 5 and fmt_name == "tiled":   # the evaluated alternative (DESIGN 5d)
                line["per_config"].append(hot_path_on_config(P, 5, peak, "sector"))
            torch.cuda.empty_cache()
        if world == 1 and not args.no_reorth:
            line["reorth"] = reorth_timing(P, n, s, peak)
            torch.cuda.empty_cache()
        if world == 1 and args.eigs:
            torch.cuda.empty_cache()
            warm_up_solver(P)
            line["seconds_to_nev"] = [time_to_nev(P, int(c)) for c in args.eigs.split(",") if c]
            # the library's option for a wider filter window (include/polfed.h):
            # the solve again with the window sized for 2 nev levels, reported beside the
            # paper's rule, not instead of it
            wide = [int(c) for c in args.eigs_wide.split(",") if c and c in args.eigs.split(",")]
            if wide:
                line["seconds_to_nev_wide_window"] = [
                    time_to_nev(P, c, window_levels=2 * workloads.make_workload(c).nev) for c in wide]
            line["seconds_to_nev_warmup"] = "one untimed solve of config 1 shrunk to L = 10 (loads cuSOLVER and the solver's kernels)"
            # solved only with the 2 nev window (labelled: NOT the paper's rule for K), because the
            # paper-rule solve takes twice as long (config 4: 540 s against 290 s)
            for c in [int(c) for c in args.eigs_wide_only.split(",") if c]:
                line.setdefault("seconds_to_nev_wide_window", []).append(
                    time_to_nev(P, c, window_levels=2 * workloads.make_workload(c).nev))
        if world == 1 and args.eigs_partial and args.config == 5 and tiled:
            torch.cuda.empty_cache()
            ratios = [r["krylov_dim"] / r["nev"] for r in line.get("seconds_to_nev", []) if r["converged"]]
            line["partial_solve"] = partial_solve(P, ham, w, kernel_ms, max(ratios) if ratios else 5.0)
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(args.config)
        if world == 1:
            # compact copies as the LAST keys of the line (a reader that keeps only the tail of a long
            # line still gets every config): short keys, rounded values
            line["per_config_summary"] = [
                {"w": r["workload"].split("_")[0], "fmt": r["format"], "launch_ms": round(r["launch_ms"], 5),
                 "frac": round(r["frac_of_measured"], 4),
                 "us_in_filter": round(r["us_per_product_in_filter"], 3),
                 "frac_in_filter": round(r["frac_of_measured_in_filter"], 4)}
                for r in line.get("per_config", [])]
            line["seconds_to_nev_summary"] = [
                {"w": r["workload"].split("_")[0], "window": r["window_levels"], "s": round(r["seconds"], 3),
                 "K": r["K"], "steps": r["block_steps"], "ok": r["converged"],
                 "res": float(f"{r['max_residual_over_normH']:.2e}")}
                for r in line.get("seconds_to_nev", []) + line.get("seconds_to_nev_wide_window", [])]
            if "partial_solve" in line:
                ps = line["partial_solve"]
                line["seconds_to_nev_summary"].append(
                    {"w": ps["workload"].split("_")[0], "partial": True, "s": round(ps["seconds"], 2),
                     "K": ps["K"], "steps": ps["block_steps"],
                     "full_solve_hours_extrapolated": round(ps["extrapolated_full_solve_hours"], 2)})
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def hot_path_on_config(P, config: int, peak: float, fmt_name: str = ""):
    """The fused launch alone on another BASELINE config: format, ms per
    launch (CUDA events over back-to-back launches on the launching stream), algorithmic GB/s and
    the fraction of the measured and of the nominal HBM rate, and filter steps/s of one filter
    application.  Configs 1-3 fit L2 (noted: the filter re-reads its working set by design)."""
    import torch
    w = workloads.make_workload(config)
    basis = P.polfed_build_basis(w.n_sites, w.n_up)
    flip = w.n_up < 0 and w.s in (8, 16, 32) and all(t[0] in ("XX", "Z", "ZZ") for t in w.terms)
    fmt_name = fmt_name or ("flip" if flip else "csr")
    ham = P.polfed_build_hamiltonian(basis, w.terms, w.dot_bits, w.dot_dense,
                                     fmt=getattr(P, "FORMAT_" + fmt_name.upper()))
    n, nnz, s = ham.n, ham.nnz, w.s
    a, b = 0.0, 80.0
    gen = torch.Generator(device="cuda").manual_seed(2000 + config)
    V = torch.randn(n, s, dtype=torch.float64, device="cuda", generator=gen)
    W = torch.empty_like(V)
    work = torch.empty(P.polfed_filter_workspace_bytes_ham(ham, s) // 8, dtype=torch.float64,
                       device="cuda")
    by = step_bytes(n, nnz, s)
    n_l = max(20, min(2000, int(0.25e12 / max(by, 1))))
    k0, k1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if fmt_name in ("tiled", "sector"):
        t_pair = []
        for cc in (np.full(9, 1e-3), np.full(9 + n_l, 1e-3)):
            P.polfed_filter_apply(ham, a, b, cc, s, V, W, work)
            k0.record()
            P.polfed_filter_apply(ham, a, b, cc, s, V, W, work)
            k1.record()
            torch.cuda.synchronize()
            t_pair.append(k0.elapsed_time(k1))
        launch_ms = (t_pair[1] - t_pair[0]) / n_l
    else:
        B1, B2 = work[: n * s].view(n, s), work[n * s: 2 * n * s].view(n, s)
        B1.copy_(V)
        B2.copy_(V)
        for _ in range(5):
            P.polfed_fused_step(ham, s, 2.0 / b, -2.0 * a / b, -1.0, 1e-3, B1, B2, V, B2)
            B1, B2 = B2, B1
        k0.record()
        for _ in range(n_l):
            P.polfed_fused_step(ham, s, 2.0 / b, -2.0 * a / b, -1.0, 1e-3, B1, B2, V, B2)
            B1, B2 = B2, B1
        k1.record()
        torch.cuda.synchronize()
        launch_ms = k0.elapsed_time(k1) / n_l
    # one whole filter application (the library call): filter steps per second
    K = w.K_fixed or 1000
    coeffs = np.full(K + 1, 1e-3)
    P.polfed_filter_apply(ham, a, b, coeffs, s, V, W, work)
    k0.record()
    P.polfed_filter_apply(ham, a, b, coeffs, s, V, W, work)
    k1.record()
    torch.cuda.synchronize()
    apply_ms = k0.elapsed_time(k1)
    gbs = by / (launch_ms * 1e-3) / 1e9
    return {"workload": WORKLOAD_NAMES[config], "format": fmt_name, "N": n, "nnz": nnz, "s": s,
            "bytes_per_fused_launch": by, "launch_ms": launch_ms, "launches_timed": n_l,
            "algorithmic_gbs": gbs, "frac_of_measured": gbs / peak,
            "frac_of_nominal_8TBps": gbs / NOMINAL_HBM_GBS,
            "filter_order": K, "filter_apply_ms": apply_ms,
            "filter_steps_per_s": K / (apply_ms * 1e-3),
            "us_per_product_in_filter": apply_ms * 1e3 / K,
            # the same byte count over the time of one product inside polfed_filter_apply (for the
            # small configs the single launches above are bound by the Python call, not the GPU)
            "frac_of_measured_in_filter": by / (apply_ms * 1e-3 / K) / 1e9 / peak,
            "traffic": recorded_traffic(WORKLOAD_NAMES[config] + "/" + fmt_name),
            "l2": "inputs exceed L2" if by > 4 * 126e6 else "working set fits L2 (not flushed)"}


def reorth_timing(P, n: int, s: int, peak: float, k: int = 8):
    """The two tall-skinny products of the full reorthogonalisation (Eq. 9, 11 PAPER.md:147-153) at
    this workload's size against k basis panels: C_j = Q_j^T W and W -= sum_j Q_j C_j, CUDA events,
    best of 5.  Bytes: Q once plus W (read; the update also writes it)."""
    import torch
    Q = torch.randn(k, n, s, dtype=torch.float64, device="cuda")
    B = torch.randn(n, s, dtype=torch.float64, device="cuda")

    def timed(f):
        f()
        torch.cuda.synchronize()
        best = float("inf")
        for _ in range(5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            f()
            e1.record()
            torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1))
        return best

    out = {"n": n, "s": s, "panels": k}
    for name, variant in (("gram_fma", 1), ("gram_tensor", 2)):
        ms = timed(lambda: P.polfed_block_gram(Q, B, variant=variant))
        by = 8 * n * s * (k + 1)
        out[name] = {"ms": ms, "gbs": by / ms / 1e6, "frac_of_measured": by / ms / 1e6 / peak,
                     "fp64_tflops": 2.0 * n * s * s * k / ms / 1e9}
    C = P.polfed_block_gram(Q, B)
    ms = timed(lambda: P.polfed_block_update(Q, C, B, -1.0, 1.0))
    by = 8 * n * s * (k + 2)
    out["update_tensor"] = {"ms": ms, "gbs": by / ms / 1e6, "frac_of_measured": by / ms / 1e6 / peak,
                            "fp64_tflops": 2.0 * n * s * s * k / ms / 1e9}
    return out


def warm_up_solver(P):
    """One untimed eigen-solve of a 252-state chain: the first call in a process pays for loading
    cuSOLVER and every kernel of the solver (CUDA loads modules lazily), which is not the metric."""
    import torch
    w = workloads.make_workload(1, L_override=10)
    basis = P.polfed_build_basis(w.n_sites, w.n_up)
    ham = P.polfed_build_hamiltonian(basis, w.terms, w.dot_bits, w.dot_dense, fmt=P.FORMAT_CSR)
    for s in (1, 8, 16):
        V0 = torch.from_numpy(workloads.start_block(ham.n, s, seed=7)).cuda()
        P.polfed_block_lanczos_eigs(ham, w.target, 8, s, V0, sigma_is_rescaled=(w.target_kind == "rescaled"),
                                    K_override=40, allow_unconverged=True)
    torch.cuda.synchronize()


def time_to_nev(P, config: int, window_levels: int = 0):
    """Second half of BASELINE.json's metric: wall seconds of polfed_block_lanczos_eigs (bounds,
    order rule, block Lanczos on P(H~), Rayleigh-Ritz, residuals) for the workload's nev pairs.
    window_levels = 0: the paper's rule for K (window for nev levels)."""
    import torch
    w = workloads.make_workload(config)
    basis = P.polfed_build_basis(w.n_sites, w.n_up)
    # the flip format (matrix-free rows) where the model allows it, else CSR (the tiled format
    # only pays on tiles larger than configs 1-3 have)
    flip = w.n_up < 0 and w.s in (8, 16, 32) and all(t[0] in ("XX", "Z", "ZZ") for t in w.terms)
    ham = P.polfed_build_hamiltonian(basis, w.terms, w.dot_bits, w.dot_dense,
                                     fmt=P.FORMAT_FLIP if flip else P.FORMAT_CSR)
    V0 = torch.from_numpy(workloads.start_block(ham.n, w.s, seed=2000 + config)).cuda()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    evals, evecs, resid, rep = P.polfed_block_lanczos_eigs(
        ham, w.target, w.nev, w.s, V0, sigma_is_rescaled=(w.target_kind == "rescaled"),
        K_override=(w.K_fixed or 0), allow_unconverged=True, window_levels=window_levels)
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    hnorm = max(abs(rep["e_min"]), abs(rep["e_max"]))
    return {"workload": WORKLOAD_NAMES[config], "format": "flip" if flip else "csr", "nev": w.nev,
            "seconds": wall, "seconds_inside_library": rep["seconds_total"], "window_levels": rep["nev_window"],
            "converged": rep["status"] == 0, "K": rep["K"], "block_steps": rep["block_steps"],
            "krylov_dim": rep["krylov_dim"], "sparse_products": rep["sparse_products"],
            "fraction_of_products_without_v_read": rep["products_without_v"] / max(rep["sparse_products"], 1),
            "max_residual_over_normH": float(resid.max()) / hnorm,
            "seconds_filter": rep["seconds_filter"], "seconds_reorth": rep["seconds_reorth"],
            "seconds_qr": rep["seconds_qr"], "seconds_projected_eig": rep["seconds_projected_eig"],
            "seconds_extraction": rep["seconds_extraction"], "seconds_bounds": rep["seconds_bounds"]}


def partial_solve(P, ham, w, launch_ms: float, krylov_per_nev: float, K: int = 512):
    """Config 5's whole solve is hours: run a STATED part of it -- the solver itself
    with K_override = 512 and the smallest Krylov space it accepts (nev + s rounded up: 8 block steps
    at nev = 200, s = 32), unconverged by design -- and extrapolate the full solve as
    K_rule x expected block steps x the measured sweep time.  K_rule: Eq. (40)-(42) with the KPM
    density of states (75 moments, 8 random vectors) on the bounds of polfed_spectrum_bounds;
    expected block steps: the Krylov dimension per wanted pair of the largest config solved to the
    end in this run."""
    import torch
    n, s, nev = ham.n, w.s, w.nev
    gen = torch.Generator(device="cuda").manual_seed(2005)
    V0 = torch.randn(n, s, dtype=torch.float64, device="cuda", generator=gen)
    e_min, e_max, a, b = P.polfed_spectrum_bounds(ham, V0[:, 0].contiguous())
    lam = w.target if w.target_kind == "rescaled" else (w.target - a) / b
    R = torch.randn(n, 8, dtype=torch.float64, device="cuda", generator=gen)
    mu = P.polfed_kpm_moments(ham, a, b, 75, R)      # already averaged over the 8 vectors
    rho = float(P.polfed_kpm_dos(mu, lam)[0])
    nev_window = nev + max(2, (nev + 9) // 10)
    K_rule = int(P.polfed_filter_coeffs(a, b, a + b * lam, nev=nev_window, rho_rescaled=rho).shape[0] - 1)
    del R
    m_min = -(-(nev + s) // s) * s
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    evals, evecs, resid, rep = P.polfed_block_lanczos_eigs(
        ham, w.target, nev, s, V0, sigma_is_rescaled=(w.target_kind == "rescaled"), a=a, b=b,
        K_override=K, max_krylov_dim=m_min, allow_unconverged=True)
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    steps_full = int(np.ceil(krylov_per_nev * nev / s))
    return {"workload": WORKLOAD_NAMES[5], "format": "tiled", "nev": nev, "K": rep["K"],
            "block_steps": rep["block_steps"], "krylov_dim": rep["krylov_dim"], "converged": rep["status"] == 0,
            "seconds": wall, "seconds_filter": rep["seconds_filter"], "seconds_reorth": rep["seconds_reorth"],
            "seconds_qr": rep["seconds_qr"], "seconds_extraction": rep["seconds_extraction"],
            "sparse_products": rep["sparse_products"], "rho_kpm_rescaled": rho, "K_rule": K_rule,
            "expected_block_steps": steps_full, "krylov_dim_per_nev_assumed": krylov_per_nev,
            "launch_ms": launch_ms,
            "extrapolated_full_solve_hours": K_rule * steps_full * launch_ms * 1e-3 / 3600.0}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--order", type=int, default=64, help="filter order K per step")
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--per-config", default="1,2,3,4",
                    help="other configs whose fused launch is timed at N=1 ('' to skip)")
    ap.add_argument("--format", default="auto", choices=["auto", "csr", "tiled", "flip", "sector"],
                    help="auto: tiled where supported and n_sites >= 24, flip for full-space XX models, "
                         "else CSR")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-reorth", action="store_true",
                    help="skip the timing of the reorthogonalisation products")
    ap.add_argument("--eigs-wide", default="3",
                    help="configs of --eigs that are solved a second time with window_levels = 2 nev")
    ap.add_argument("--eigs-wide-only", default="4",
                    help="configs solved ONLY with window_levels = 2 nev (config 4: about 5 minutes)")
    ap.add_argument("--eigs-partial", default="5",
                    help="'5': when the main line is config 5 (tiled), run 8 block steps of its solve at "
                         "K = 512 and extrapolate the full solve ('' to skip)")
    ap.add_argument("--eigs", default="1,2,3",
                    help="configs whose full eigen-solve is timed at N=1 ('' to skip; 4 takes minutes)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    if args.impl == "reference":
        return run_reference(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
