#!/usr/bin/env python
"""Benchmark of the hot path (BASELINE.json metric): grind time, ns per (cell x equation x RHS evaluation), fp64.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg3] [--n 256]

One "step" is one pass of the whole path over the workload (mfc_step_cfl): the CFL reduction (mfc_cfl_dt) and one 3-stage
TVD-RK step (mfc_rk3_step = 3 launches of the fused kernel: ghost fill + cons->prim, WENO5+HLLC in x, y, z, flux
difference, stage combine).  The workload is BASELINE.json configs[3] (256^3 two-fluid bubble cloud), seeded and synthetic.
N > 1 (torchrun): independent replicas, one per GPU, no data-path collective ("replicas only");
time is the max over ranks and the value counts the cells of all ranks.

--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "grind_time_ns_per_cell_eqn_rhs"
UNIT = "ns/(cell*eqn*RHS)"
RHS_PER_STEP = 3
FP64_NOMINAL_TFLOPS = 2 * 64 * 148 * 1.965e9 / 1e12   # 64 DFMA/clk/SM x 148 SMs x 1.965 GHz


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured"
    return 6650.0, "fallback"


TRAFFIC_CSV = os.path.join("profiles", "r03_dram_traffic.csv")


def ncu_traffic(workload: str, kernel: str):
    """(dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` on `workload`, provenance) from the committed
    ncu capture (profiles/r03_dram_traffic.csv: one `ncu --set full` run, its command and the commit it profiled are in
    the file).  It is RECORDED, not measured in this run: the provenance string says which commit it belongs to.
    (None, None) when no capture is recorded for the workload."""
    path = os.path.join(ROOT, TRAFFIC_CSV)
    if not os.path.exists(path):
        return None, None
    import csv
    with open(path) as f:
        rows = [r for r in csv.DictReader(l for l in f if not l.startswith("#"))]
    for row in rows:
        if row["workload"] == workload and row["kernel"] == kernel:
            return (float(row["dram_read_bytes"]) + float(row["dram_write_bytes"]),
                    f"recorded: {TRAFFIC_CSV} (ncu --set full of commit {row.get('commit', '?')}), not measured in this run")
    return None, None


class ClockSampler:
    """SM clock, power and throttle reasons sampled through NVML every few ms WHILE the timed region runs
    (the quantities of the B200_PROFILING.md clocks line; a polling thread sees a 100 ms region, an
    nvidia-smi -lms loop does not)."""

    REASONS = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
               "hw_power_brake_slowdown": 0x80}

    def __init__(self, index: int, period_s: float = 0.004):
        self.index, self.period = index, period_s
        self.sm, self.pw, self.mask = [], [], 0
        self.smax = None
        self.stop_flag = threading.Event()
        self.thread = None
        self.err = None

    def start(self):
        try:
            import pynvml as N
            N.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            idx = self.index
            if vis:
                ids = [v.strip() for v in vis.split(",") if v.strip()]
                if self.index < len(ids) and ids[self.index].isdigit():
                    idx = int(ids[self.index])
            h = N.nvmlDeviceGetHandleByIndex(idx)
            self.smax = float(N.nvmlDeviceGetMaxClockInfo(h, N.NVML_CLOCK_SM))
        except Exception as exc:  # NVML missing: the record says so, the run is not hidden
            self.err = f"nvml unavailable: {exc}"
            return

        def pump():
            while not self.stop_flag.is_set():
                try:
                    self.sm.append(float(N.nvmlDeviceGetClockInfo(h, N.NVML_CLOCK_SM)))
                    self.pw.append(N.nvmlDeviceGetPowerUsage(h) / 1000.0)
                    self.mask |= int(N.nvmlDeviceGetCurrentClocksEventReasons(h))
                except Exception as exc:
                    self.err = str(exc)
                    return
                time.sleep(self.period)

        self.thread = threading.Thread(target=pump, daemon=True)
        self.thread.start()

    def stop(self):
        self.stop_flag.set()
        if self.thread:
            self.thread.join(timeout=2)
        reasons = sorted(k for k, bit in self.REASONS.items() if self.mask & bit)
        if self.err:
            reasons.append(self.err)
        return {"sm_mhz": statistics.median(self.sm) if self.sm else None, "sm_max_mhz": self.smax,
                "sm_min_mhz": min(self.sm) if self.sm else None, "power_w_max": max(self.pw) if self.pw else None,
                "samples": len(self.sm), "reasons": reasons}


def get_workload(name: str, n: int | None):
    from paper_2305_09163_b200 import workloads as wl
    idx = int(name.replace("cfg", ""))
    fn = wl.CONFIGS[idx]
    return fn(n=n) if n else fn()


# --------------------------------------------------------------------------------------------------------
# algorithmic work of one launch of the fused right-hand side, per cell
# --------------------------------------------------------------------------------------------------------
def rhs_algorithmic(prob):
    neq, nf, D = prob.neq, prob.nf, prob.ndim
    # WENO5 in the common-denominator form (80 flops per variable and direction), HLLC (102 / 116 per face),
    # flux difference (3 per equation and direction), cons->prim (25) and RK combine (4 per equation)
    flops = D * (neq * 80 + (102 if nf <= 2 else 116) + 3 * neq) + 25 + 4 * neq
    # compulsory bytes of an RK stage: q_s read once, result written once, q_n read in two of the three stages
    doubles = neq * (1 + 1 + 2.0 / 3.0)
    return flops, 8.0 * doubles


def reduce_over_ranks(ms_total, e2e_ms, state_ok, dist, device):
    """Replicas-only multi-GPU rule: the job takes as long as its slowest rank (max over ranks of the
    device-timed region and of the end-to-end time) and is valid only if every rank's state is finite."""
    if dist is None:
        return ms_total, e2e_ms, state_ok
    import torch
    t = torch.tensor([ms_total, e2e_ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ok = torch.tensor([1.0 if state_ok else 0.0], device=device, dtype=torch.float64)
    dist.all_reduce(ok, op=dist.ReduceOp.MIN)
    return float(t[0]), float(t[1]), bool(ok.item() > 0.5)


def whole_job_grind(ms_step, cells_per_rank, world, neq):
    """ns per (cell x equation x RHS evaluation) of the whole job: every rank advances its own replica."""
    return ms_step * 1e6 / (cells_per_rank * world * neq * RHS_PER_STEP)


def time_workload(B, torch, prob, q, local, steps, warmup, segment=0):
    """K device-timed steps (CFL + RK3) of one workload with inputs resident in HBM; kernel times from the library's event
    brackets.  Returns (ms per step, per-kernel profile, launches, state finite, ctx-free)."""
    ctx = B.init_from_problem(prob, device=local, march_segment=segment)
    try:
        stream = torch.cuda.current_stream().cuda_stream
        qd = torch.from_numpy(q).cuda()
        for _ in range(max(3, warmup)):
            B.mfc_step_cfl(ctx, qd.data_ptr(), stream)
        torch.cuda.synchronize()
        for kid in range(B.MFC_K_COUNT):
            B.mfc_profile_get(ctx, kid, reset=True)
        B.mfc_profile_enable(ctx, True)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            B.mfc_step_cfl(ctx, qd.data_ptr(), stream)
        e1.record()
        torch.cuda.synchronize()
        prof = {}
        for kid in range(B.MFC_K_COUNT):
            n, ms = B.mfc_profile_get(ctx, kid, reset=True)
            prof[B.KERNEL_NAMES[kid]] = {"launches": n, "ms_total": ms, "ms_avg": (ms / n if n else 0.0)}
        B.mfc_profile_enable(ctx, False)
        return e0.elapsed_time(e1) / steps, prof, bool(torch.isfinite(qd).all().item())
    finally:
        B.mfc_destroy(ctx)


def extra_config_line(B, torch, name, prob, q, local, steps, fp64_tf, hbm_peak, note=None):
    """One entry of `extra_configs`: the same step, event-timed, on a non-headline workload, with its roofline fractions."""
    ms_step, prof, ok = time_workload(B, torch, prob, q, local, steps, 3)
    flops_cell, bytes_cell = rhs_algorithmic(prob)
    t_avg = prof["rhs_fused"]["ms_avg"] * 1e-3
    return {"workload": f"{prob.name} {prob.n[0]}x{prob.n[1]}x{prob.n[2]} nf={prob.nf} neq={prob.neq} ({name})", "steps": steps,
            **({"note": note} if note else {}),
            "ms_per_step": ms_step, "value": ms_step * 1e6 / (prob.cells * prob.neq * RHS_PER_STEP), "unit": UNIT,
            "cells_steps_per_s": prob.cells / (ms_step * 1e-3),
            "kernels_ms_avg": {k: v["ms_avg"] for k, v in prof.items() if v["launches"]},
            "roofline": {"kernel": "rhs_fused", "bound": "alu", "achieved": flops_cell * prob.cells / t_avg / 1e12, "peak": fp64_tf,
                         "unit": "TFLOP/s", "frac": flops_cell * prob.cells / t_avg / 1e12 / fp64_tf,
                         "hbm_frac": bytes_cell * prob.cells / t_avg / 1e9 / hbm_peak,
                         "algorithmic_flops_per_cell": flops_cell, "algorithmic_bytes_per_cell": bytes_cell},
            "state_finite": ok}


def run_ours(args):
    import torch

    from paper_2305_09163_b200 import binding as B
    from paper_2305_09163_b200 import build as mfc_build

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        mfc_build.build()
    if dist:
        dist.barrier()
    B.lib()

    prob, q = get_workload(args.workload, args.n)
    if args.kapila:
        import dataclasses
        prob = dataclasses.replace(prob, name=prob.name + "+kapila", kapila=True)
    if args.stretched:
        from paper_2305_09163_b200 import workloads as wl
        prob = wl.with_stretched_grid(prob)
    ctx = B.init_from_problem(prob, device=local, march_segment=args.segment)
    neq, ng, padded, elems = B.mfc_layout(ctx)
    stream = torch.cuda.current_stream().cuda_stream
    q_host = torch.from_numpy(q).pin_memory()
    qd = q_host.cuda(non_blocking=True)
    torch.cuda.synchronize()

    def step():
        return B.mfc_step_cfl(ctx, qd.data_ptr(), stream)    # CFL reduction, then the three stages at that dt

    for _ in range(max(3, args.warmup)):
        step()
    torch.cuda.synchronize()

    def barrier():
        if dist:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- timed region: exactly K steps, inputs resident in HBM ----
    for kid in range(B.MFC_K_COUNT):
        B.mfc_profile_get(ctx, kid, reset=True)
    B.mfc_profile_enable(ctx, True)
    sampler = ClockSampler(local) if rank == 0 else None
    barrier()
    if sampler:
        sampler.start()
    n0 = B.mfc_launch_count(ctx)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    clocks = sampler.stop() if sampler else None
    ms_total = e0.elapsed_time(e1)
    launches = B.mfc_launch_count(ctx) - n0
    prof = {}
    for kid in range(B.MFC_K_COUNT):
        n, ms = B.mfc_profile_get(ctx, kid, reset=True)
        prof[B.KERNEL_NAMES[kid]] = {"launches": n, "ms_total": ms, "ms_avg": (ms / n if n else 0.0)}
    B.mfc_profile_enable(ctx, False)
    state_ok = bool(torch.isfinite(qd).all().item())

    # ---- e2e: same step through the C ABI from HOST buffers (H2D + D2H inside the timed region) ----
    q_host.copy_(torch.from_numpy(q))
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    B.mfc_advance_host(ctx, q_host.data_ptr(), 1, 0.0, stream)       # warm-up (allocates the library's device copy)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        B.mfc_advance_host(ctx, q_host.data_ptr(), 1, 0.0, stream)   # synchronous: returns after the D2H copy
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3 / e2e_steps

    ms_total, e2e_ms, state_ok = reduce_over_ranks(ms_total, e2e_ms, state_ok, dist, "cuda")

    if rank == 0:
        ms_step = ms_total / args.steps
        work = prob.cells * world * neq * RHS_PER_STEP
        grind = whole_job_grind(ms_step, prob.cells, world, neq)
        hbm_peak, hbm_src = measured_peaks()
        fp64_tf, fp64_ms = B.mfc_probe_dfma(local)
        # dominant kernel: the fused right-hand side (one launch per RK stage)
        dom = "rhs_fused"
        flops_cell, bytes_cell = rhs_algorithmic(prob)
        t_avg = prof[dom]["ms_avg"] * 1e-3
        ach_gbs = bytes_cell * prob.cells / t_avg / 1e9
        ach_tf = flops_cell * prob.cells / t_avg / 1e12
        t_hbm = bytes_cell * prob.cells / (hbm_peak * 1e9)
        t_alu = flops_cell * prob.cells / (fp64_tf * 1e12)
        plain = not (args.n or args.kapila or args.stretched or args.segment)
        traffic, traffic_src = ncu_traffic(args.workload if plain else "", dom)
        if t_hbm >= t_alu:
            roof = {"kernel": dom, "bound": "hbm", "achieved": ach_gbs, "peak": hbm_peak, "unit": "GB/s",
                    "frac": ach_gbs / hbm_peak, "traffic": traffic, "peak_source": f"MEASURED_PEAKS.json ({hbm_src})"}
        else:
            roof = {"kernel": dom, "bound": "alu", "achieved": ach_tf, "peak": fp64_tf, "unit": "TFLOP/s",
                    "frac": ach_tf / fp64_tf, "traffic": traffic,
                    "peak_source": "mfc_probe_dfma (register-resident DFMA chains, faster of two operand shapes: 99.95 % of the FP64 pipe under ncu, profiles/r03_probe.md), measured in this run; DESIGN.md 6.1"}
        roof.update({"algorithmic_flops_per_cell": flops_cell, "algorithmic_bytes_per_cell": bytes_cell,
                     "avg_launch_ms": prof[dom]["ms_avg"], "hbm_frac": ach_gbs / hbm_peak, "fp64_frac": ach_tf / fp64_tf,
                     "hbm_peak_gbs": hbm_peak, "hbm_peak_source": f"MEASURED_PEAKS.json ({hbm_src})",
                     "traffic_source": traffic_src,
                     "fp64_pipe_busy_recorded": "profiles/r03_ncu_full.md (sm__inst_executed_pipe_fp64 68 %, executed-flop fraction)",
                     "fp64_peak_measured_tflops": fp64_tf, "fp64_peak_nominal_tflops": FP64_NOMINAL_TFLOPS,
                     "kernel_ms_sum_over_step_ms": sum(v["ms_total"] for v in prof.values()) / ms_total})
        out = {
            "metric": METRIC, "value": grind, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(3, args.warmup),
            "ms_per_step": ms_step, "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "impl": "ours",
            "config": {"workload": f"{prob.name} {prob.n[0]}x{prob.n[1]}x{prob.n[2]} nf={prob.nf} neq={neq} (BASELINE.json configs[{args.workload[3:]}])",
                       "cells_per_gpu": prob.cells, "rhs_per_step": RHS_PER_STEP, "parallelism": f"replicas x{world}",
                       "l2": "inputs larger than L2 (each state array >= 1 GB at 256^3)", "march_segment": args.segment,
                       "step": "mfc_step_cfl (= mfc_cfl_dt + mfc_rk3_step, the first ghost fill enqueued before the wait for dt)"},
            "cells_steps_per_s": prob.cells * world / (ms_step * 1e-3),
            "gpu_launches": launches,
            "kernels": prof,
            "roofline": roof,
            "e2e": {"value": e2e_ms * 1e6 / work, "unit": UNIT, "ms_per_step": e2e_ms, "steps": e2e_steps,
                    "h2d_bytes_per_step": elems * 8, "d2h_bytes_per_step": elems * 8,
                    "call": "mfc_advance_host(q_host pinned, nsteps=1, CFL dt)"},
            "clocks": clocks, "state_finite": state_ok,
        }
        if world == 1 and not args.no_cpu:
            out["cpu_baseline"] = cpu_baseline(args)
    B.mfc_destroy(ctx)
    del qd
    torch.cuda.empty_cache()
    if rank == 0:
        if world == 1 and not args.no_extra and plain:
            # non-headline workloads, event-timed the same way: the paper's ~2 M cells per device
            # regime (cfg2), the three-fluid 384^3 case (cfg4) and the headline data on the Eq. 15 stretched grid
            from paper_2305_09163_b200 import workloads as wl
            extra = []
            small = ("the 1D / 2D kernel (rhs_fused_plane_kernel) at the parity-test size: the state fits L2 and a step is a "
                     "handful of microsecond launches plus the host round trip of mfc_cfl_dt -- launch- and latency-bound, "
                     "not a roofline figure")
            for name, make, nsteps, note in (
                    ("BASELINE.json configs[0], 1D shock tube", lambda: wl.cfg0(), 50, small),
                    ("BASELINE.json configs[1], 2D advected interface", lambda: wl.cfg1(), 50, small),
                    ("BASELINE.json configs[2]", lambda: wl.cfg2(), 5, None), ("BASELINE.json configs[4]", lambda: wl.cfg4(), 5, None),
                    ("configs[3] on the Eq. 15 stretched grid", lambda: (lambda pq: (wl.with_stretched_grid(pq[0]), pq[1]))(wl.cfg3()), 5, None)):
                p2, q2 = make()
                extra.append(extra_config_line(B, torch, name, p2, q2, local, nsteps, fp64_tf, hbm_peak, note))
                del q2
                torch.cuda.empty_cache()
            out["extra_configs"] = extra
        print(json.dumps(out))
    if dist:
        dist.barrier()
        dist.destroy_process_group()


# --------------------------------------------------------------------------------------------------------
# CPU oracle legs (the only places bench.py may execute oracle/)
# --------------------------------------------------------------------------------------------------------
def oracle_step_time(args, n_sample: int, steps: int, warmup: int):
    import oracle
    prob, q = get_workload(args.workload, n_sample)
    orc = oracle.Oracle(prob)
    times = []
    for i in range(warmup + steps):
        t0 = time.perf_counter()
        dt = orc.cfl_dt(q, prob.cfl)
        orc.rk3_step(q, dt)
        if i >= warmup:
            times.append(time.perf_counter() - t0)
    return prob, times, oracle.threads()


def cpu_model() -> str:
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def cpu_baseline(args):
    """The oracle as it stands on the box's host cores: all cores (OpenMP on the outer loops) and ONE thread
    (BASELINE.md section 3), on bounded samples of the headline workload; grind time is size-normalised."""
    import oracle
    n_sample = args.cpu_n
    prob, times, cores = oracle_step_time(args, n_sample, 2, 0)
    sec = sum(times) / len(times)
    oracle.set_threads(1)
    try:
        n1 = args.cpu_n1
        prob1, times1, _ = oracle_step_time(args, n1, 1, 0)
    finally:
        oracle.set_threads(cores)
    sec1 = times1[0]
    full = {"cfg0": 1000, "cfg1": 512, "cfg2": 128, "cfg3": 256, "cfg4": 384}[args.workload]   # default sizes of workloads.py
    size = f"at its full size, {n_sample}^3 cells" if n_sample == full else f"shrunk to {n_sample}^3 cells"
    return {"value": sec * 1e9 / (prob.cells * prob.neq * RHS_PER_STEP), "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{prob.name} {size}, 2 steps of (CFL + RK3) with the OpenMP oracle, {sec:.2f} s/step",
            "cpu_model": cpu_model(),
            "one_thread": {"value": sec1 * 1e9 / (prob1.cells * prob1.neq * RHS_PER_STEP), "unit": UNIT, "cores": 1,
                           "sample": f"{prob1.name} shrunk to {n1}^3 cells, 1 step of (CFL + RK3), {sec1:.2f} s/step"}}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n_sample = args.ref_n
    prob, times, cores = oracle_step_time(args, n_sample, args.steps, min(args.warmup, 1))
    sec = sum(times) / len(times)
    grind = sec * 1e9 / (prob.cells * prob.neq * RHS_PER_STEP)
    sample = f"{prob.name} shrunk to {n_sample}^3 cells per step (CPU oracle, OpenMP, {cores} threads)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": grind, "unit": UNIT, "n_gpus": int(os.environ.get("WORLD_SIZE", "1")),
        "steps": args.steps, "warmup": min(args.warmup, 1), "ms_per_step": sec * 1e3, "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{prob.name} (BASELINE.json configs[{args.workload[3:]}]), bounded sample {n_sample}^3", "rhs_per_step": RHS_PER_STEP},
        "cpu_baseline": {"value": grind, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": grind, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3", choices=["cfg0", "cfg1", "cfg2", "cfg3", "cfg4"])
    ap.add_argument("--n", type=int, default=None, help="override cells per dimension (default: the config's size)")
    ap.add_argument("--segment", type=int, default=0, help="z planes each block of the fused kernel marches (0 = heuristic)")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--cpu-n", type=int, default=256, help="cells per dimension of the all-cores cpu_baseline sample (256 = the headline workload at full size: about 4 s per step on 16 cores)")
    ap.add_argument("--cpu-n1", type=int, default=64, help="cells per dimension of the one-thread cpu_baseline sample")
    ap.add_argument("--ref-n", type=int, default=96, help="cells per dimension of the --impl reference sample")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-extra", action="store_true", help="skip the extra_configs leg (cfg2, cfg4, stretched cfg3)")
    ap.add_argument("--kapila", action="store_true", help="switch the K div(u) source of PAPER.md Eq. 2 on (not the headline config)")
    ap.add_argument("--stretched", action="store_true", help="same per-cell data on the Eq. 15 stretched grid (non-uniform spacing; not the headline config)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
