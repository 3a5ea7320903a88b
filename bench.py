#!/usr/bin/env python
"""bench.py -- one JSON line for BASELINE.json's metric: FP64 cell-pair interactions/s per Fx,Fy evaluation.

A "step" is one pass of the whole hot path over one density field: sg_set_density (S2: vertex weights +
line tables) then sg_force (S3 interaction kernel, S4/S5 finalise).  Workload at N = 1 GPU: BASELINE.json
config 5 (uniform 1024 x 1024, 1,048,576 leaves, 1.1e12 pairs per evaluation), the >= 1 M-cell case the
north_star bar is quoted on.  With N > 1 GPUs the targets are sharded across ranks (targets are
independent; :265: "12 cards"), every rank sums over all sources, no data-path collective: strong scaling.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

With --gpus N > 1 and no torchrun environment the script re-executes itself under `python -m torch.distributed.run
--standalone --nproc-per-node N` (one rank per GPU); under torchrun it uses the ranks it is given.

--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "FP64 cell-pair interactions/s per Fx,Fy evaluation"
UNIT = "pairs/s"
# Nominal FP64 peak used as the roofline denominator: 148 SMs x 64 FP64 FMA lanes x 2 flop x 1.965 GHz
# (SM count and max SM clock from /opt/skills/guides/B200_PROFILING.md; 64 lanes/SM = 4 sub-partitions x 16,
# consistent with the DFMA micro-benchmark measured live below).  DESIGN.md "Roofline".
FP64_LANES_PER_SM = 64
DIRECT_LEG_STEPS = 3          # timed steps of the direct-kernel leg (after 3 warm-ups; SURVEY.md 8(d) protocol)


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.rows, self._halt = index, [], threading.Event()

    def run(self):
        while not self._halt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                      "-i", str(self.index)], capture_output=True, text=True, timeout=5).stdout
                self.rows.append([c.strip() for c in out.strip().split(",")])
            except Exception:
                pass
            self._halt.wait(0.2)

    def stop(self) -> dict:
        self._halt.set()
        self.join(timeout=6)
        sm, smax, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); smax.append(float(r[1]))
            except ValueError:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json config 1..5 (default 5)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-baseline-seconds", type=float, default=15.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config list (all five configs)")
    ap.add_argument("--mode", default="auto", choices=["auto", "direct", "lattice"],
                    help="S3 algorithm: direct pair sum, lattice-offset reuse, or auto (lattice when the layout allows)")
    ap.add_argument("--paper-layout", default=None, metavar="RULE:DISK:L:NK",
                    help="instead of a BASELINE.json config: one of the paper's own zone-wise quadtrees, e.g. ILR:D2:3:1024 "
                         "(PAPER.md:164, Tables 3-9; 1 x 1 patches, regrouped into 16 x 16 blocks in lattice mode) with the "
                         "paper's D2 / D22 disk; add --slopes for the full second-order method the paper times")
    ap.add_argument("--slopes", action="store_true",
                    help="time the first-order path (sg_set_density_linear); default is the zeroth-order hot path")
    return ap.parse_args()


KERNEL_SOURCE = {"interaction_kernel": "sg_kernels.cu", "interaction_lin_kernel": "sg_kernels_lin.cu",
                 "patch_offset_kernel": "sg_kernels_patch.cu", "lattice_corr_kernel": "sg_kernels_lattice.cu"}


def kernel_source_sha256(kernel: str):
    """sha256 of the .cu file that holds `kernel` (the captured traffic figure is tied to it)."""
    import hashlib
    for name, fn in KERNEL_SOURCE.items():
        if kernel.startswith(name):
            path = os.path.join(ROOT, "paper_2001_02765_b200", "csrc", fn)
            if os.path.exists(path):
                return hashlib.sha256(open(path, "rb").read()).hexdigest()
    return None


def measured_traffic(workload: str, kernel: str):
    """(dram__bytes_read.sum + dram__bytes_write.sum per launch, capture id) of `kernel` from the committed ncu
    capture of this workload (profiles/traffic.csv), or (None, why): ncu cannot run inside the bench, so the figure
    is a recorded one, and it is dropped when the kernel's source file has changed since the capture."""
    import csv
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(path):
        with open(path) as f:
            for row in csv.DictReader(f):
                if row["workload"] == workload and kernel.startswith(row["kernel"]):
                    if row.get("source_sha256") and row["source_sha256"] != kernel_source_sha256(kernel):
                        return None, f"stale: kernel source changed since capture {row.get('capture')}"
                    return int(row["dram_bytes_per_launch"]), row.get("capture")
    return None, "no ncu capture of this kernel on this workload"


def per_config_measurement(torch, device, flush, cfg, nominal_tflops, steps=5, warmup=3):
    """One BASELINE.json config through the same calls as the headline: `steps` steps of sg_set_density + sg_force
    between CUDA events after `warmup` warm-up steps, L2 flushed between steps; lattice mode where the layout allows
    (P = 8 or 16), else the direct kernel.  Roofline fraction on algorithmic units (count x N_v pairs)."""
    from paper_2001_02765_b200 import SgDisk
    from workloads import make_config
    lay, sigma = make_config(cfg)
    t0 = time.perf_counter()
    d = SgDisk.from_layout(lay, device=device)
    create_ms = (time.perf_counter() - t0) * 1e3
    try:
        mode = "lattice" if lay.P in (8, 16) else "direct"
        t0 = time.perf_counter()
        d.set_interaction_mode(mode)
        mode_ms = (time.perf_counter() - t0) * 1e3
        s = torch.as_tensor(sigma).to(torch.device("cuda", device))
        Fx = torch.empty(lay.n_cells, dtype=torch.float64, device=s.device)
        Fy = torch.empty_like(Fx)

        def step():
            flush.zero_()
            d.set_density(s)
            d.force(Fx, Fy)
        for _ in range(warmup):
            step()
        mdl = d.kernel_model()
        d.set_kernel_timing(True)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(steps):
            step()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / steps
        kms = d.kernel_times_ms()
        k = sum(kms) / max(1, len(kms))
        sd, fl = d.launch_counts()
    finally:
        d.close()
    achieved = mdl["pair_evaluations"] * mdl["flops_per_pair"] / (k * 1e-3) / 1e12
    return {"config": cfg, "workload": workload_name(cfg), "n_cells": lay.n_cells, "n_levels": lay.n_levels,
            "patch_cells": lay.P, "interaction_mode": mode, "value": float(lay.n_cells) ** 2 / (ms * 1e-3),
            "unit": UNIT, "ms_per_step": ms, "interaction_ms": k, "steps": steps, "warmup": warmup,
            "gpu_launches_per_step": sd + fl, "create_ms": create_ms, "set_mode_ms": mode_ms,
            "roofline": {"bound": "alu", "achieved": achieved, "peak": nominal_tflops, "unit": "TFLOP/s",
                         "frac": achieved / nominal_tflops, "flops_per_pair": mdl["flops_per_pair"],
                         "pair_evaluations_per_launch": mdl["pair_evaluations"],
                         "executed_over_algorithmic": mdl["executed_evaluations"] / max(1.0, mdl["pair_evaluations"])}}


def workload_name(cfg) -> str:
    from workloads import CONFIG_NAMES
    return CONFIG_NAMES[cfg] if isinstance(cfg, int) else str(cfg)


def load_workload(args):
    """(workload key, layout, sigma, slopes or None): a BASELINE.json config, or one of the paper's quadtrees."""
    from workloads import make_config, expected_counts
    if args.paper_layout:
        from workloads import paper_ilr_layout, paper_vlr_layout, d2_sigma, d2_slopes, d22_sigma, d22_slopes
        from workloads.configs import cell_centres
        rule, disk, L, Nk = args.paper_layout.split(":")
        lay = (paper_ilr_layout if rule.upper() == "ILR" else paper_vlr_layout)(int(Nk), int(L), disk)
        x, y, _ = cell_centres(lay)
        if disk == "D2":
            return f"paper_{rule}_{disk}_L{L}_Nk{Nk}", lay, d2_sigma(x, y, 0.5), d2_slopes(x, y, 0.5)
        return f"paper_{rule}_{disk}_L{L}_Nk{Nk}", lay, d22_sigma(x, y), d22_slopes(x, y)
    lay, sigma = make_config(args.config)
    exp = expected_counts(args.config)
    assert lay.n_cells == exp["n_cells"] and lay.n_patches == exp["n_patches"], "frozen layout changed"
    return args.config, lay, sigma, None


# --------------------------------------------------------------------------------------------------
# CPU legs: the oracle as it stands (oracle/sg_oracle.c, double build, OpenMP over targets)
# --------------------------------------------------------------------------------------------------
def oracle_sample_rate(lay, sigma, seconds: float, seed: int = 99, slopes=None):
    """Time the oracle on a bounded, seeded sample of targets of this workload (every sampled target is
    summed over ALL N leaves, so pairs/s does not depend on the sample size).  Returns
    (pairs_per_s, threads, n_targets, elapsed_s)."""
    import numpy as np
    import oracle
    from workloads import cell_rects, sample_targets
    r = cell_rects(lay)
    cores = os.cpu_count() or 1
    n_cal = min(lay.n_cells, max(2 * cores, 8))
    idx = sample_targets(lay, n_cal, seed)
    t0 = time.perf_counter()
    kw = {} if slopes is None else {"dx": slopes[0], "dy": slopes[1]}
    _, _, threads = oracle.force(r, sigma, r["kxc"][idx], r["kyc"][idx], lay.unit, precision="f64", **kw)
    dt = max(time.perf_counter() - t0, 1e-6)
    rate = idx.size * lay.n_cells / dt
    n = int(min(lay.n_cells, max(n_cal, seconds * rate / lay.n_cells)))
    n = max(threads, (n // threads) * threads)
    idx = sample_targets(lay, min(n, lay.n_cells), seed + 1)
    t0 = time.perf_counter()
    oracle.force(r, sigma, r["kxc"][idx], r["kyc"][idx], lay.unit, precision="f64", **kw)
    dt = time.perf_counter() - t0
    return idx.size * lay.n_cells / dt, threads, int(idx.size), dt


def run_reference(args):
    """--impl reference: the oracle on the box's host cores, same config / metric / unit."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wkey, lay, sigma, _ = load_workload(args)
    per_step = max(1.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    rates, threads, n_t = [], 1, 0
    for i in range(args.warmup + args.steps):
        rate, threads, n_t, dt = oracle_sample_rate(lay, sigma, per_step, seed=100 + i)
        if i >= args.warmup:
            rates.append((rate, dt))
    total_pairs = sum(r * d for r, d in rates)
    total_t = sum(d for _, d in rates)
    value = total_pairs / total_t
    sample = (f"{n_t} seeded targets per step (stratified by level), each summed over all "
              f"{lay.n_cells} leaves, double-precision build of oracle/sg_oracle.c")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total_t / max(1, args.steps),
        "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(wkey), "n_cells": lay.n_cells,
                   "pairs_per_evaluation": lay.n_cells ** 2},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------------
# the GPU path
# --------------------------------------------------------------------------------------------------
def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2001_02765_b200 import SgDisk, measure_fp64_peak, measure_fp64_mma_peak, shard_range
    from paper_2001_02765_b200.sharding import lattice_patch_costs, regrouped_patch_costs, shard_range_by_cost
    from workloads import make_config, expected_counts

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    wkey, lay, sigma, paper_slopes = load_workload(args)
    N = lay.n_cells
    lattice = args.mode != "direct" and (lay.P in (1, 2, 4, 16) or (lay.P == 8 and not args.slopes))
    if args.mode == "lattice" and not lattice:
        raise SystemExit("--mode lattice needs patches of 1, 2, 4 or 16 cells (8x8 for the zeroth-order path only)")
    if lattice and lay.P in (1, 2, 4, 16):
        # lattice mode works on whole patches and a target's cost depends on its level: split by estimated cost
        # (small patches are regrouped into 16 x 16 blocks inside the library, which evaluates the blocks that hold
        # the slice: the same per-level estimate applies)
        costs = (lattice_patch_costs(lay.patches[:, 0]) if lay.P == 16 else regrouped_patch_costs(lay.patches, lay.P))
        first, count = shard_range_by_cost(costs, lay.P * lay.P, rank, world)
    else:
        first, count = shard_range(N, rank, world)

    t_create = time.perf_counter()
    d = SgDisk.from_layout(lay, device=local)
    create_ms = (time.perf_counter() - t_create) * 1e3
    d.set_target_range(first, count)
    info = d.layout_info()

    fields = [sigma]
    if args.slopes and paper_slopes is not None:
        fields += list(paper_slopes)                # exact Taylor coefficients of the paper's disks (R10)
    elif args.slopes:
        # first-order Taylor coefficients of the smooth Kuzmin profile every bench config is
        # built on (cfg 3/4: centred differences of the cell samples along the library's own rows would need the
        # neighbour links; analytic slopes of the base profile are the paper's choice, R10)
        from workloads.configs import cell_centres
        xc, yc, _ = cell_centres(lay)
        g = -3.0 * sigma / (xc * xc + yc * yc + 0.04)
        fields += [g * xc, g * yc]
    hosts = [torch.from_numpy(np.ascontiguousarray(f)).pin_memory() for f in fields]
    devs = [h.to(dev) for h in hosts]

    def set_density():
        if args.slopes:
            d.set_density_linear(*devs)
        else:
            d.set_density(devs[0])
    Fx = torch.empty(count, dtype=torch.float64, device=dev)
    Fy = torch.empty(count, dtype=torch.float64, device=dev)
    Fx_host = torch.empty(count, dtype=torch.float64).pin_memory()
    Fy_host = torch.empty(count, dtype=torch.float64).pin_memory()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2

    def step_resident():
        flush.zero_()                       # L2 flush between steps (the vertex tiles are L2-sized)
        set_density()
        d.force(Fx, Fy)

    def step_e2e():
        flush.zero_()
        for dv, h in zip(devs, hosts):
            dv.copy_(h, non_blocking=True)
        set_density()
        d.force(Fx, Fy)
        Fx_host.copy_(Fx, non_blocking=True)
        Fy_host.copy_(Fy, non_blocking=True)
        torch.cuda.current_stream().synchronize()      # the caller holds the result on the host

    peak_tflops, peak_winstr = measure_fp64_peak(local)
    dmma_tflops, dmma_mixed_tflops = measure_fp64_mma_peak(local)

    # ---- device-resident timing -------------------------------------------------------------------
    def timed_resident(steps, warmup):
        """W warm-up steps, then `steps` steps between CUDA events with a barrier + synchronize on both sides; the
        interaction kernel(s) of every step are timed by the library's own event ring on the same stream."""
        for _ in range(warmup):
            step_resident()
        mdl = d.kernel_model()              # of the path the warm-up just selected
        d.set_kernel_timing(True)
        smp = ClockSampler(local)
        barrier()
        smp.start()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            step_resident()
        e1.record()
        barrier()
        clk = smp.stop()
        total = e0.elapsed_time(e1)
        kms = d.kernel_times_ms()
        d.set_kernel_timing(False)
        return total, kms, clk, mdl

    t_mode = time.perf_counter()
    d.set_interaction_mode("lattice" if lattice else "direct")
    set_mode_ms = (time.perf_counter() - t_mode) * 1e3
    set_density()                                   # (a regrouped layout wants its density after the mode is chosen)
    sd_launches, f_launches = d.launch_counts()
    ms_total, k_ms, clocks, model = timed_resident(args.steps, max(3, args.warmup))
    direct_run = None
    if lattice and world == 1 and N <= 2200000:
        # the north_star kernel (every pair: sqrt + 2 ln) on the same workload, same run, for its roofline line
        # (skipped above 2.2 M cells, where six direct steps would take minutes)
        d.set_interaction_mode("direct")
        direct_run = timed_resident(DIRECT_LEG_STEPS, 3)
        d.set_interaction_mode("lattice")
        step_resident()

    # ---- end-to-end timing (host buffers, copies inside the timed region) --------------------------
    for _ in range(2):
        step_e2e()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step_e2e()
    barrier()
    e2e_s = time.perf_counter() - t0

    t = torch.tensor([ms_total, e2e_s * 1e3, sum(k_ms) / max(1, len(k_ms))], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_total, e2e_ms, k_ms_avg = [float(v) for v in t.tolist()]

    if rank == 0:
        pairs = float(N) * float(N)
        value = pairs * args.steps / (ms_total * 1e-3)
        e2e_value = pairs * args.steps / (e2e_ms * 1e-3)
        sm_count = torch.cuda.get_device_properties(local).multi_processor_count
        sm_max = clocks.get("sm_max_mhz") or 1965.0
        nominal_tflops = sm_count * FP64_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
        def roofline_of(mdl, kms, step_ms, kernel, traffic):
            # achieved: ALGORITHMIC units (count x N_v deduplicated (target, vertex) pairs) x flops
            # per unit / kernel time.  fp64_pipe_util: the hardware number, from the pairs the kernels EXECUTE
            # (per-patch vertices in lattice mode, padding slots in direct mode), i.e. what ncu's
            # sm__pipe_fp64_cycles_active sees (tables and far pairs excluded).
            evals = mdl["pair_evaluations"]
            executed = mdl["executed_evaluations"]
            achieved = evals * mdl["flops_per_pair"] / (kms * 1e-3) / 1e12
            winstr = executed * mdl["fp64_instr_per_pair"] / 32.0 / (kms * 1e-3)      # warp instructions / s
            traffic_bytes, traffic_note = traffic if traffic is not None else (None, "not looked up (multi-GPU run)")
            return {
                "bound": "alu", "achieved": achieved, "peak": nominal_tflops, "unit": "TFLOP/s",
                "frac": achieved / nominal_tflops, "traffic": traffic_bytes, "traffic_capture": traffic_note,
                "kernel": kernel, "executed_over_algorithmic": executed / max(1.0, evals),
                "kernel_ms": kms, "kernel_share_of_step": kms / step_ms,
                "peak_kind": f"nominal {sm_count} SM x {FP64_LANES_PER_SM} FP64 lanes x 2 x {sm_max:.0f} MHz",
                "peak_measured_dfma_tflops": peak_tflops, "frac_of_measured_dfma": achieved / peak_tflops,
                "fp64_pipe_util": winstr / (sm_count * FP64_LANES_PER_SM / 32.0 * sm_max * 1e6),
                "fp64_pipe_util_of_measured_dfma": winstr / peak_winstr,
                "flops_per_pair": mdl["flops_per_pair"], "fp64_instr_per_pair": mdl["fp64_instr_per_pair"],
                "pair_evaluations_per_launch": evals,
            }

        if args.slopes:
            direct_name = "interaction_lin_kernel<4>"
        else:
            direct_name = "interaction_kernel<4>" if count > 16384 else "interaction_kernel<1>"
        direct_traffic = measured_traffic(workload_name(wkey), direct_name) if world == 1 else None
        if lattice:
            lattice_name = ("lattice_corr_kernel<0> (same-level pairs; <1>..<4> for pairs one and two levels apart"
                            + ("; three planes per offset: slope terms)" if args.slopes else ")"))
            if lay.P == 8:
                lattice_name = "patch_interaction_kernel<8>"
            roofline = roofline_of(model, k_ms_avg, ms_total / args.steps, lattice_name,
                                   measured_traffic(workload_name(wkey) + ("+slopes" if args.slopes else ""),
                                                    lattice_name) if world == 1 else None)
        else:
            roofline = roofline_of(model, k_ms_avg, ms_total / args.steps, direct_name, direct_traffic)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(3, args.warmup), "ms_per_step": ms_total / args.steps, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(wkey), "n_cells": N, "n_vertices": info["n_vertices"],
                       "pairs_per_evaluation": pairs,
                       "order": "sigma0 + slope terms (Eq. 6)" if args.slopes else "sigma0 (north_star hot path)",
                       "interaction_mode": ("lattice-offset reuse (SG_MODE_LATTICE): precomputed function lattices "
                                            "streamed by TMA, 2 DFMA per pair" + (" and plane (6 with slopes)" if args.slopes else ""))
                                           if lattice else "direct",
                       "parallelism": f"targets sharded over {world} GPU(s)" + (" by estimated cost, whole patches" if lattice else " by count"),
                       "create_ms": create_ms, "set_mode_ms": set_mode_ms,
                       "l2": "256 MiB memset between steps (inside the timed region)"},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 8 * N * len(fields), "d2h_bytes_per_step": 16 * count,
                    "ms_per_step": e2e_ms / args.steps},
            "gpu_launches": args.steps * (sd_launches + f_launches),
            "clocks": clocks, "roofline": roofline,
            "fp64_probes": {"dfma_tflops": peak_tflops, "mma_m8n8k4_f64_tflops": dmma_tflops,
                            "mma_interleaved_with_dfma_total_tflops": dmma_mixed_tflops,
                            "what": "micro-benchmarks outside the timed region (sg_measure_fp64_peak, "
                                    "sg_measure_fp64_mma_peak): FP64 tensor-core MMA does not add to the DFMA rate"},
        }
        if direct_run is not None:
            d_total, d_kms, _, d_model = direct_run
            d_k = sum(d_kms) / max(1, len(d_kms))
            line["direct_kernel"] = {
                "what": "same workload, same run, SG_MODE_DIRECT: every (target, vertex) pair = 1 sqrt + 2 ln "
                        f"(the north_star interaction kernel{'; with slope terms' if args.slopes else ''}); "
                        f"{DIRECT_LEG_STEPS} timed steps after 3 warm-ups",
                "value": pairs * DIRECT_LEG_STEPS / (d_total * 1e-3), "unit": UNIT, "ms_per_step": d_total / DIRECT_LEG_STEPS,
                "steps": DIRECT_LEG_STEPS, "warmup": 3,
                "roofline": roofline_of(d_model, d_k, d_total / DIRECT_LEG_STEPS, direct_name, direct_traffic)}
        if world == 1 and not args.slopes and not args.no_per_config and not args.paper_layout:
            # north_star: "report throughput on synthetic disks shaped like the paper's workloads": all five configs,
            # same calls, same run (the headline workload's own entry repeats the numbers above)
            line["per_config"] = []
            for cfg in (1, 2, 3, 4, 5):
                if cfg == args.config:
                    line["per_config"].append({
                        "config": cfg, "workload": workload_name(cfg), "n_cells": N, "n_levels": lay.n_levels,
                        "patch_cells": lay.P, "interaction_mode": "lattice" if lattice else "direct", "value": value,
                        "unit": UNIT, "ms_per_step": ms_total / args.steps, "interaction_ms": k_ms_avg,
                        "steps": args.steps, "warmup": max(3, args.warmup),
                        "gpu_launches_per_step": sd_launches + f_launches, "create_ms": create_ms,
                        "roofline": {k: roofline[k] for k in ("bound", "achieved", "peak", "unit", "frac",
                                                               "flops_per_pair", "pair_evaluations_per_launch",
                                                               "executed_over_algorithmic")}})
                else:
                    line["per_config"].append(per_config_measurement(torch, local, flush, cfg, nominal_tflops))
        # The record the driver keeps is `roofline` (top-level extras survive only as names): the north_star kernel's
        # own fraction and the five per-config fractions are repeated inside it, compactly.
        if "direct_kernel" in line:
            dr = line["direct_kernel"]["roofline"]
            roofline["north_star_kernel"] = {
                "kernel": dr["kernel"], "mode": "direct (every pair: 1 sqrt + 2 ln)", "kernel_ms": dr["kernel_ms"],
                "achieved": dr["achieved"], "peak": dr["peak"], "unit": dr["unit"], "frac": dr["frac"],
                "fp64_pipe_util": dr["fp64_pipe_util"], "flops_per_pair": dr["flops_per_pair"],
                "fp64_instr_per_pair": dr["fp64_instr_per_pair"], "traffic": dr["traffic"],
                "value": line["direct_kernel"]["value"], "ms_per_step": line["direct_kernel"]["ms_per_step"]}
        if "per_config" in line:
            roofline["per_config"] = [
                {"config": e["config"], "workload": e["workload"], "mode": e["interaction_mode"], "value": e["value"],
                 "ms_per_step": e["ms_per_step"], "frac": e["roofline"]["frac"],
                 "flops_per_pair": e["roofline"]["flops_per_pair"]} for e in line["per_config"]]
        if not args.no_cpu_baseline and world == 1:
            rate, threads, n_t, dt = oracle_sample_rate(lay, sigma, args.cpu_baseline_seconds,
                                                        slopes=fields[1:] if args.slopes else None)
            line["cpu_baseline"] = {
                "value": rate, "unit": UNIT, "cores": threads, "kind": "oracle",
                "sample": f"{n_t} seeded targets (stratified by level), each summed over all {N} leaves; "
                          f"{dt:.1f} s; double-precision build of oracle/sg_oracle.c, OpenMP over targets"}
        print(json.dumps(line), flush=True)
    d.close()
    if world > 1:
        dist.destroy_process_group()


def spawn_command(args, argv):
    """`python bench.py --gpus N` without a torchrun environment starts the N ranks itself: the command that re-runs
    this script under torch.distributed.run (one process per GPU, rendezvous on 127.0.0.1), or None when no spawn
    is needed (N = 1, the reference arm, or already inside a torchrun launch)."""
    if args.impl != "ours" or args.gpus <= 1 or "WORLD_SIZE" in os.environ:
        return None
    return [sys.executable, "-m", "torch.distributed.run", "--standalone", "--nnodes=1",
            f"--nproc-per-node={args.gpus}", "--local-addr", "127.0.0.1", os.path.abspath(__file__), *argv]


def main():
    args = parse_args()
    cmd = spawn_command(args, sys.argv[1:])
    if cmd is not None:
        env = dict(os.environ)
        # NCCL's own log (one "Init COMPLETE" line per rank) goes to stderr; stdout stays the one JSON line
        env.setdefault("NCCL_DEBUG", "INFO")
        env.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")
        env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        if os.environ.get("SG_BENCH_PRINT_SPAWN"):             # tests: show the launch instead of running it
            print(json.dumps({"spawn": cmd}))
            return
        sys.stdout.flush()
        os.execvpe(cmd[0], cmd, env)
    if args.impl == "reference":
        run_reference(args)
    else:
        world = int(os.environ.get("WORLD_SIZE", "1"))
        if args.gpus != world:
            raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={world}: launch with torchrun --nproc-per-node "
                             f"{args.gpus}, or run `python bench.py --gpus {args.gpus}` and let it spawn the ranks")
        run_ours(args)


if __name__ == "__main__":
    main()
