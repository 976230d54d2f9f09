#!/usr/bin/env python
"""bench.py -- Poisson solves/s (fp64, 256^3 mesh) on B200, with roofline and CPU-oracle baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
        --master-port P bench.py --gpus N --steps K --warmup W

A "step" is one pass of the whole hot path: one dks_poisson_solve (P1..P5) on the config's mesh
(default: BASELINE.json configs[3], the 256^3 mesh the metric is quoted on).  Multi-GPU = replicas
only: every rank solves its own bunch, no data-path collective; value =
solves of all ranks / max-over-ranks device time.

Prints ONE JSON line on rank 0.
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

METRIC = "poisson_solves_per_s_fp64"
UNIT = "solves/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config index 1..5 (default 4 = 256^3)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=20)
    ap.add_argument("--slab", type=int, default=None, help="planes per P2-P4 slab (default: the plan's automatic choice)")
    ap.add_argument("--prof-steps", type=int, default=50, help="extra solves with per-launch events, for the per-pass split")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--ref-full", action="store_true", help="--impl reference: time full-size oracle solves")
    return ap.parse_args()


def workload_name(w):
    return f"{w.name}: {w.n[0]}x{w.n[1]}x{w.n[2]} mesh (padded {2*w.n[0]}x{2*w.n[1]}x{2*w.n[2]}), {w.description}"


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def max_over_ranks(ms_local: float, device="cpu") -> float:
    """Device time of the slowest rank (replicas only: there is no data-path collective; this all-reduce of one
    scalar is the measurement's own).  Works on NCCL (device="cuda") and on gloo (device="cpu")."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, steps: int, ms_max: float) -> float:
    """Solves/s of the whole job: every rank did `steps` solves of its own bunch in at most ms_max."""
    return world * steps / (ms_max * 1e-3)


class ClockSampler:
    """Samples nvidia-smi SM clocks and throttle reasons while the timed region runs."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.rows, self._stop, self._t = index, [], threading.Event(), None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                      "-i", str(self.index)], capture_output=True, text=True, timeout=5).stdout
                self.rows.append([c.strip() for c in out.strip().split(",")])
            except Exception:
                pass
            self._stop.wait(0.1)

    def __enter__(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=10)

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except ValueError:
                continue
            for name, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------------------------
# CPU oracle legs (the only places bench.py executes oracle/)
# ------------------------------------------------------------------------------------------------
def _work(n):
    import math
    N = 8.0 * n[0] * n[1] * n[2]
    return N * math.log2(N)


def oracle_full_solve(w, rho, repeats=1):
    """Times `repeats` full oracle solves (double build, FT{G} precomputed as for the GPU timer)."""
    from oracle import oracle as O
    plan = O.Plan(w.n, w.h, precision="d")
    try:
        t0 = time.perf_counter()
        for _ in range(repeats):
            plan.solve(rho)
        dt = (time.perf_counter() - t0) / repeats
    finally:
        plan.close()
    return dt, O.num_threads("d")


def oracle_sample_plan(w, rho):
    """Bounded sample of the workload: the central half-extent sub-mesh (1/8 of the nodes) of the same
    rho, same spacings.  Returns (plan, sub_rho, n_sub)."""
    from oracle import oracle as O
    import numpy as np
    nx, ny, nz = w.n
    sx, sy, sz = max(nx // 2, 8), max(ny // 2, 8), max(nz // 2, 8)
    x0, y0, z0 = (nx - sx) // 2, (ny - sy) // 2, (nz - sz) // 2
    sub = np.ascontiguousarray(rho[z0:z0 + sz, y0:y0 + sy, x0:x0 + sx])
    return O.Plan((sx, sy, sz), w.h, precision="d"), sub, (sx, sy, sz)


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, on the host cores, rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1509_07685_b200 import workloads as W
    from oracle import oracle as O
    w = W.config(args.config)
    rho = W.make_rho(w)
    if args.ref_full:
        plan, sub, n_sub, scale = O.Plan(w.n, w.h, precision="d"), rho, w.n, 1.0
        sample = f"each step = one full oracle solve of {w.name} (double build, FT{{G}} precomputed)"
    else:
        plan, sub, n_sub = oracle_sample_plan(w, rho)
        scale = _work(n_sub) / _work(w.n)
        sample = (f"each step = one oracle solve (double build, FT{{G}} precomputed) of the central "
                  f"{n_sub[0]}x{n_sub[1]}x{n_sub[2]} sub-mesh of {w.name}; solves/s scaled by the N*log2(N) "
                  f"work ratio {scale:.4f} (N = padded points)")
    try:
        for _ in range(args.warmup):
            plan.solve(sub)
        t0 = time.perf_counter()
        for _ in range(args.steps):
            plan.solve(sub)
        dt = time.perf_counter() - t0
    finally:
        plan.close()
    value = args.steps / dt * scale
    cores = O.num_threads("d")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 / value, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(w), "timing": "host wall clock around the oracle's solve"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1509_07685_b200 import dks, workloads as W

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    distributed = world > 1
    if distributed:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if distributed:
            dist.barrier()
        torch.cuda.synchronize()

    w = W.config(args.config)
    # replicas only: every rank gets the same bunch shape from its own seed offset is not needed --
    # run time is data independent; all ranks use the config's rho.
    rho = W.make_rho(w)
    nbytes = rho.nbytes
    d_rho = torch.from_numpy(rho).cuda()
    d_phi = torch.empty_like(d_rho)
    plan = dks.PoissonPlan(w.n, w.h, slab_planes=args.slab)
    stream = torch.cuda.current_stream()
    launches = dks.dks_poisson_launches_per_solve(plan.handle)
    ws_bytes = dks.dks_poisson_workspace_bytes(plan.handle)

    # ---- device-resident timing ------------------------------------------------------------------
    for _ in range(args.warmup):
        plan.solve(d_rho, d_phi)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    with ClockSampler(local) as clocks:
        e0.record(stream)
        for _ in range(args.steps):
            plan.solve(d_rho, d_phi)
        e1.record(stream)
        barrier()
    ms_total = e0.elapsed_time(e1)
    # per-pass split: a second, untimed-for-the-headline run with events around every launch
    dks.dks_poisson_set_profiling(plan.handle, min(args.prof_steps, 256))
    for _ in range(min(args.prof_steps, 256)):
        plan.solve(d_rho, d_phi)
    pass_ms = dks.dks_poisson_pass_times(plan.handle)
    dks.dks_poisson_set_profiling(plan.handle, 0)
    ms_total = max_over_ranks(ms_total, "cuda")
    ms_per_step = ms_total / args.steps
    value = whole_job_value(world, args.steps, ms_total)

    # ---- secondary: the Green's-function rebuild (dks_greens_setup), which OPAL needs whenever h changes ----
    e0.record(stream)
    for _ in range(5):
        plan.set_spacing(w.h)
    e1.record(stream)
    torch.cuda.synchronize()
    greens_ms = e0.elapsed_time(e1) / 5

    # ---- secondary: batched solves (dks_poisson_solve_batch, 8 meshes per call) on the small meshes, which are
    # launch-latency bound one at a time
    batched = None
    if w.n[0] * w.n[1] * w.n[2] <= 128 ** 3:
        nb = 8
        bplan = dks.PoissonPlan(w.n, w.h, max_batch=nb)
        b_rho = d_rho.unsqueeze(0).repeat(nb, 1, 1, 1).contiguous()
        b_phi = torch.empty_like(b_rho)
        for _ in range(3):
            bplan.solve_batch(b_rho, b_phi)
        reps = max(10, args.steps // nb)
        e0.record(stream)
        for _ in range(reps):
            bplan.solve_batch(b_rho, b_phi)
        e1.record(stream)
        torch.cuda.synchronize()
        batched = {"nbatch": nb, "value": nb * reps / (e0.elapsed_time(e1) * 1e-3), "unit": UNIT}
        bplan.close()
        del b_rho, b_phi

    # ---- end to end through the public API with HOST buffers (H2D + solve + D2H per step) --------
    h_rho = torch.from_numpy(rho).pin_memory()
    h_phi = torch.empty_like(h_rho).pin_memory()
    for _ in range(3):
        plan.solve_host(h_rho, h_phi)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.e2e_steps):
        plan.solve_host(h_rho, h_phi)                  # one blocking call per step: copy in, solve, copy out
    barrier()
    e2e_sync_ms = (time.perf_counter() - t0) * 1e3
    # pipelined: every step still copies its own rho in and its own phi out, consecutive steps overlap
    # (copy streams beside the solve stream); timed on the host clock up to the last copy-out, since the
    # copies run on plan-owned streams that an event on torch's stream would not see
    h_phi2 = torch.empty_like(h_rho).pin_memory()
    outs = [h_phi, h_phi2]
    for i in range(3):
        plan.solve_host_async(h_rho, outs[i & 1])
    plan.host_sync()
    barrier()
    t0 = time.perf_counter()
    for i in range(args.e2e_steps):
        plan.solve_host_async(h_rho, outs[i & 1])
    plan.host_sync()
    barrier()
    e2e_ms = (time.perf_counter() - t0) * 1e3
    e2e_value = whole_job_value(world, args.e2e_steps, max_over_ranks(e2e_ms, "cuda"))
    e2e_sync_value = whole_job_value(world, args.e2e_steps, max_over_ranks(e2e_sync_ms, "cuda"))

    if rank != 0:
        plan.close()
        if distributed:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel -----------------------------------------------------------
    peak, peak_src = measured_peaks()
    top = max(range(len(pass_ms)), key=lambda i: pass_ms[i])
    top_bytes = plan.model_bytes(top + 1)
    achieved = top_bytes / (pass_ms[top] * 1e-3) / 1e9
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    top_name = dks.dks_poisson_pass_name(plan.handle, top + 1)
    if os.path.exists(tpath):
        try:
            traffic = json.load(open(tpath)).get(w.name, {}).get(top_name)
        except Exception:
            traffic = None
    m3 = plan.model_bytes(0)
    roofline = {
        "bound": "hbm", "kernel": top_name, "achieved": achieved, "peak": peak, "unit": "GB/s",
        "frac": achieved / peak, "traffic": traffic, "peak_source": peak_src,
        "algorithmic_bytes_per_launch": top_bytes, "kernel_ms": pass_ms[top],
        "passes": {dks.dks_poisson_pass_name(plan.handle, i + 1): {
            "ms": pass_ms[i], "model_bytes": plan.model_bytes(i + 1),
            "gbs": plan.model_bytes(i + 1) / (pass_ms[i] * 1e-3) / 1e9} for i in range(len(pass_ms))},
        "whole_solve": {"model_bytes_M3": m3, "gbs": m3 / (ms_per_step * 1e-3) / 1e9,
                        "frac": m3 / (ms_per_step * 1e-3) / 1e9 / peak,
                        "frac_of_8TBs": m3 / (ms_per_step * 1e-3) / 8e12},
    }
    plan.close()

    # ---- CPU oracle timed beside it (rank 0, N = 1 only) ---------------------------------------------
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        dt, cores = oracle_full_solve(w, rho)
        cpu = {"value": 1.0 / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"1 full solve of {w.name} by oracle/poisson_oracle.c (double build, OpenMP, "
                         f"FT{{G}} precomputed and not timed), {dt:.2f} s"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(w), "parallelism": "replicas only" if world > 1 else "1 gpu",
                   "l2": ("inputs larger than L2 (rho + phi + workspace >> 126 MB); no explicit flush"
                          if ws_bytes + 2 * nbytes > 126e6 else
                          "working set fits the 126 MB L2 (L2-resident workload); no flush"),
                   "greens_setup": "precomputed, outside the timed region (DESIGN.md reading A11)",
                   "greens_setup_ms": greens_ms, "batched": batched},
        "clocks": clocks.summary(),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
                "steps": args.e2e_steps, "timing": "host clock around the loop, device idle before and after",
                "api": "dks_poisson_solve_host_async per step + one dks_poisson_host_sync (pinned host rho -> H2D -> P1..P5 -> "
                       "D2H -> host phi every step; copies of neighbouring steps overlap the solve)",
                "blocking_api_value": e2e_sync_value},
        "gpu_launches": launches * args.steps,
        "roofline": roofline,
    }
    if cpu is not None:
        line["cpu_baseline"] = cpu
    print(json.dumps(line), flush=True)
    if distributed:
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
