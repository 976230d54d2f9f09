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
    ap.add_argument("--mesh", type=int, nargs=3, metavar=("NX", "NY", "NZ"), default=None,
                    help="context workload instead of a BASELINE config (never the headline): e.g. 512 512 256, the largest mesh of "
                         "the paper's Table 1 (PAPER.md:157-158); uniform random rho, no CPU / cuFFT / particle legs")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=60, help="host-path steps per e2e loop (pipeline fill and drain are inside the timed region)")
    ap.add_argument("--slab", type=int, default=None, help="planes per P2-P4 slab (default: the plan's automatic choice)")
    ap.add_argument("--prof-steps", type=int, default=50, help="extra solves with per-launch events, for the per-pass split")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-cufft", action="store_true", help="skip the torch.fft (cuFFT) side reference")
    ap.add_argument("--ref-sample", action="store_true",
                    help="--impl reference: time the central half-extent sub-mesh instead of the full mesh (reported unscaled, under its own workload name)")
    ap.add_argument("--field-reps", type=int, default=10, help="timed repetitions of each particle-kernel measurement (1 for ncu captures)")
    ap.add_argument("--repeats", type=int, default=5, help="timed windows of --steps solves each; the median is reported")
    ap.add_argument("--sustained-s", type=float, default=2.0, help="length of the additional back-to-back run (0 = skip)")
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
    """One long-running `nvidia-smi -lms 20` whose rows are stamped on arrival; summary(t0, t1) looks at the rows that
    arrived inside a window of host time (time.perf_counter()).  Windows shorter than the period see few or no rows:
    `samples` says how many, and the summary then falls back to the rows nearest to the window."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    PERIOD_MS = 20

    def __init__(self, index=0):
        self.index, self.rows, self._t, self._p = index, [], None, None

    def _run(self):
        for line in self._p.stdout:
            self.rows.append((time.perf_counter(), [c.strip() for c in line.strip().split(",")]))

    def __enter__(self):
        try:
            self._p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                        "-i", str(self.index), "-lms", str(self.PERIOD_MS)],
                                       stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self._t = threading.Thread(target=self._run, daemon=True)
            self._t.start()
        except Exception:
            self._p = None
        return self

    def __exit__(self, *a):
        if self._p is not None:
            self._p.terminate()
            try:
                self._p.wait(timeout=5)
            except Exception:
                self._p.kill()
            self._t.join(timeout=5)

    def summary(self, t0=None, t1=None):
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for (t, r) in self.rows if (t0 is None or t >= t0) and (t1 is None or t <= t1)]
        inside = len(rows)
        if not rows and self.rows and t0 is not None:      # window shorter than the sampling period: nearest rows
            mid = 0.5 * (t0 + (t1 if t1 is not None else t0))
            rows = [r for (_, r) in sorted(self.rows, key=lambda tr: abs(tr[0] - mid))[:2]]
        sm, mx, pw, reasons = [], [], [], set()
        for r in rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except ValueError:
                continue
            for name, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_min_mhz": sm[0], "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "reasons": sorted(reasons), "samples": inside, "period_ms": self.PERIOD_MS}


# ------------------------------------------------------------------------------------------------
# CPU oracle legs (the only places bench.py executes oracle/)
# ------------------------------------------------------------------------------------------------
def _refuse_sanitized_oracle():
    from oracle import build as OB
    if OB.SANITIZE:
        raise SystemExit("ORACLE_SANITIZE=1 selects the ASan/UBSan oracle build: not a CPU baseline to time; unset it")


def oracle_full_solve(w, rho, budget_s=20.0):
    """One untimed full oracle solve (first touch of its 2 x 2 GB work arrays at 256^3), then timed full solves until
    about `budget_s` of CPU time is spent, at least one (double build, FT{G} precomputed as for the GPU timer)."""
    from oracle import oracle as O
    _refuse_sanitized_oracle()
    plan = O.Plan(w.n, w.h, precision="d")
    try:
        t0 = time.perf_counter()
        plan.solve(rho)
        first = time.perf_counter() - t0
        reps = max(1, min(20, int((budget_s - first) / max(first, 1e-3))))
        t0 = time.perf_counter()
        for _ in range(reps):
            plan.solve(rho)
        dt = (time.perf_counter() - t0) / reps
    finally:
        plan.close()
    return dt, reps, first, O.num_threads("d")


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, on the host cores, rank 0 only.  Every step is one FULL oracle
    solve of the benchmarked mesh (2-3 s at 256^3), ms_per_step the wall time a step took.  --ref-sample times the
    central half-extent sub-mesh instead and says so in config.workload; nothing is extrapolated."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1509_07685_b200 import workloads as W
    from oracle import oracle as O
    import numpy as np
    _refuse_sanitized_oracle()
    w = W.config(args.config)
    rho = W.make_rho(w)
    name = workload_name(w)
    n = w.n
    sample = f"each step = one full oracle solve of {w.name} (double build, OpenMP, FT{{G}} precomputed and not timed)"
    if args.ref_sample:
        nx, ny, nz = w.n
        n = (max(nx // 2, 8), max(ny // 2, 8), max(nz // 2, 8))
        x0, y0, z0 = (nx - n[0]) // 2, (ny - n[1]) // 2, (nz - n[2]) // 2
        rho = np.ascontiguousarray(rho[z0:z0 + n[2], y0:y0 + n[1], x0:x0 + n[0]])
        name = f"central {n[0]}x{n[1]}x{n[2]} sub-mesh of {name} (NOT the benchmarked mesh; --ref-sample)"
        sample = f"each step = one oracle solve of the central {n[0]}x{n[1]}x{n[2]} sub-mesh of {w.name} (double build, FT{{G}} precomputed)"
    plan = O.Plan(n, w.h, precision="d")
    try:
        for _ in range(args.warmup):
            plan.solve(rho)
        t0 = time.perf_counter()
        for _ in range(args.steps):
            plan.solve(rho)
        dt = time.perf_counter() - t0
    finally:
        plan.close()
    value = args.steps / dt
    cores = O.num_threads("d")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        # the same keys as the product arm's config (the driver compares the two); what that arm measures is None here
        "config": {"workload": name, "parallelism": "cpu oracle on rank 0's host cores", "l2": None,
                   "greens_setup": "precomputed, outside the timed region (DESIGN.md reading A11)", "greens_setup_ms": None,
                   "batched": None, "sustained_solves_per_s": None, "sustained_ms_per_step": None, "sustained_sm_mhz": None,
                   "timing": "host wall clock around the oracle's solves"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def cufft_side_reference(torch, w, d_rho, d_phi, stream, reps=10):
    """Padded rfftn -> multiply by the complex half-spectrum of G -> irfftn -> crop with torch.fft (cuFFT), Green's transform
    precomputed; d_phi (the product's result for d_rho) is only used to check that the side reference computes the same thing."""
    import math
    nx, ny, nz = w.n
    hx, hy, hz = w.h
    k = 1.0 / (4.0 * math.pi * 8.8541878128e-12)

    def mirrored(n, h):
        i = torch.arange(2 * n, device="cuda", dtype=torch.float64)
        return torch.minimum(i, 2 * n - i) * h

    r = torch.sqrt(mirrored(nz, hz)[:, None, None] ** 2 + mirrored(ny, hy)[None, :, None] ** 2 + mirrored(nx, hx)[None, None, :] ** 2)
    r[0, 0, 0] = 0.5 * min(hx, hy, hz)
    ghat = torch.fft.rfftn(k / r) * (hx * hy * hz)
    del r
    shape = (2 * nz, 2 * ny, 2 * nx)

    def solve():
        return torch.fft.irfftn(torch.fft.rfftn(d_rho, s=shape) * ghat, s=shape)[:nz, :ny, :nx]

    out = solve()
    rel = float(torch.linalg.norm((out - d_phi).flatten()) / torch.linalg.norm(d_phi.flatten()))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(reps):
        out = solve()
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    return {"value": 1e3 / ms, "unit": UNIT, "ms_per_step": ms, "rel_l2_vs_product": rel,
            "what": "torch.fft.rfftn(rho, s = doubled grid) * FT{G} -> irfftn -> crop (cuFFT, fp64), FT{G} precomputed; "
                    "the pipeline of PAPER.md:132 on this GPU, context only"}


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

    if args.mesh:
        nx_, ny_, nz_ = args.mesh
        w = W.Workload(f"mesh_{nx_}x{ny_}x{nz_}", (nx_, ny_, nz_), (1e-4, 1e-4, 2e-4), 0, 7,
                       "context workload (--mesh): uniform random rho, seed 7; run time is data independent")
        rho = W.random_rho(w.n, seed=w.seed, signed=False)
        args.no_cpu_baseline = args.no_cufft = True
        args.e2e_steps = min(args.e2e_steps, 6)
    else:
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
    windows, sustained = [], None
    with ClockSampler(local) as clocks:
        barrier()
        t_first = time.perf_counter()
        for _ in range(max(1, args.repeats)):            # each window: exactly --steps solves between two events
            barrier()
            e0.record(stream)
            for _ in range(args.steps):
                plan.solve(d_rho, d_phi)
            e1.record(stream)
            barrier()
            windows.append(max_over_ranks(e0.elapsed_time(e1), "cuda"))
        t_last = time.perf_counter()
        clocks_timed = clocks.summary(t_first, t_last)
        if args.sustained_s > 0:                         # a per-time-step solver runs for minutes: the same loop for >= 2 s
            n_sus = max(args.steps, int(args.sustained_s * 1e3 / (sorted(windows)[len(windows) // 2] / args.steps)) + 1)
            barrier()
            ts0 = time.perf_counter()
            e0.record(stream)
            for _ in range(n_sus):
                plan.solve(d_rho, d_phi)
            e1.record(stream)
            barrier()
            ts1 = time.perf_counter()
            ms_sus = max_over_ranks(e0.elapsed_time(e1), "cuda")
            sustained = {"steps": n_sus, "ms_per_step": ms_sus / n_sus, "value": whole_job_value(world, n_sus, ms_sus),
                         "unit": UNIT, "clocks": clocks.summary(ts0 + 0.5 * (ts1 - ts0), ts1)}   # clocks of the second half
    ms_total = sorted(windows)[len(windows) // 2]        # median window
    # per-pass split: a second, untimed-for-the-headline run with events around every launch
    dks.dks_poisson_set_profiling(plan.handle, min(args.prof_steps, 256))
    for _ in range(min(args.prof_steps, 256)):
        plan.solve(d_rho, d_phi)
    pass_ms = dks.dks_poisson_pass_times(plan.handle)
    dks.dks_poisson_set_profiling(plan.handle, 0)
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
    # the step the paper runs: new spacings every step, Green's rebuild beside the rho copy
    for i in range(3):
        plan.step_host_async(w.h, h_rho, outs[i & 1])
    plan.host_sync()
    barrier()
    t0 = time.perf_counter()
    for i in range(args.e2e_steps):
        hh = tuple(v * (1.0 + 1e-3 * (i + 1)) for v in w.h)
        plan.step_host_async(hh, h_rho, outs[i & 1])
    plan.host_sync()
    barrier()
    e2e_rebuild_value = whole_job_value(world, args.e2e_steps, max_over_ranks((time.perf_counter() - t0) * 1e3, "cuda"))
    plan.set_spacing(w.h)
    # yardstick: what the host link gives for the same buffers (pinned, one mesh per copy), one direction at a time
    # and both at once on two streams -- the pipelined e2e cannot beat the bidirectional figure
    s_a, s_b = torch.cuda.Stream(), torch.cuda.Stream()
    d_tmp = torch.empty_like(d_rho)

    def _copy_rate(h2d, d2h, reps=5):
        torch.cuda.synchronize()
        t = time.perf_counter()
        for _ in range(reps):
            if h2d:
                with torch.cuda.stream(s_a):
                    d_tmp.copy_(h_rho, non_blocking=True)
            if d2h:
                with torch.cuda.stream(s_b):
                    h_phi2.copy_(d_phi, non_blocking=True)
        torch.cuda.synchronize()
        return reps * nbytes / (time.perf_counter() - t) / 1e9

    link = {"h2d_gbs": _copy_rate(True, False), "d2h_gbs": _copy_rate(False, True),
            "bidirectional_gbs_per_direction": _copy_rate(True, True)}
    link["steps_per_s_at_link_limit"] = link["bidirectional_gbs_per_direction"] * 1e9 / nbytes
    del d_tmp

    # ---- f4: the whole space-charge step with the particles resident on the device (deposit -> solve -> E -> gather):
    # nothing but a scalar crosses the host link (PAPER.md:160 names that link as the limiter)
    field_ops = None
    if world == 1 and not args.mesh:
        px, py, pz, pq, origin = W.particles(w)
        dpx, dpy, dpz, dpq = (torch.from_numpy(a).cuda() for a in (px, py, pz, pq))
        n_p = dpx.numel()
        f_rho = torch.empty_like(d_rho)

        def space_charge_step():
            plan.deposit(dpx, dpy, dpz, dpq, origin, f_rho)
            plan.solve(f_rho, d_phi)
            return plan.field_at_particles(d_phi, dpx, dpy, dpz, origin)

        def timed(fn, reps=args.field_reps):
            for _ in range(2):
                fn()
            e0.record(stream)
            for _ in range(reps):
                fn()
            e1.record(stream)
            torch.cuda.synchronize()
            return e0.elapsed_time(e1) / reps

        ex, ey, ez = plan.gradient(d_phi)
        field_ops = {
            "particles": n_p,
            "deposit_ms": timed(lambda: plan.deposit(dpx, dpy, dpz, dpq, origin, f_rho)),
            "gradient_ms": timed(lambda: plan.gradient(d_phi)),
            "gather_ms": timed(lambda: plan.gather(ex, ey, ez, dpx, dpy, dpz, origin)),
            "field_at_particles_ms": timed(lambda: plan.field_at_particles(d_phi, dpx, dpy, dpz, origin)),
        }
        step_ms = timed(space_charge_step)
        field_ops["device_resident_step"] = {"ms_per_step": step_ms, "value": 1e3 / step_ms, "unit": "steps/s",
                                             "api": "dks_deposit_cic + dks_poisson_solve + dks_field_at_particles (= gradient + gather), "
                                                    "particles and meshes resident on the device; no host traffic"}
        # the step as the paper runs it: the mesh follows the bunch, so the spacings change and the Green's
        # transform is rebuilt every step (dks_poisson_set_spacing + dks_greens_setup on the same stream, inside the timed region)
        calls = [0]

        def space_charge_step_with_rebuild():
            calls[0] += 1
            plan.set_spacing(tuple(v * (1.0 + 1e-3 * (calls[0] % 7)) for v in w.h))
            return space_charge_step()

        step2_ms = timed(space_charge_step_with_rebuild)
        plan.set_spacing(w.h)
        field_ops["device_resident_step_with_greens_rebuild"] = {
            "ms_per_step": step2_ms, "value": 1e3 / step2_ms, "unit": "steps/s",
            "api": "dks_poisson_set_spacing + dks_greens_setup + dks_deposit_cic + dks_poisson_solve + dks_field_at_particles"}
        # algorithmic bytes of the f4 kernels against the measured copy bandwidth; the particle kernels
        # touch the mesh at random in generator order, so their floors assume every node is moved once
        nodes = w.n[0] * w.n[1] * w.n[2]
        peak_gbs = measured_peaks()[0]

        def roof(ms, nbytes_alg):
            gbs = nbytes_alg / (ms * 1e-3) / 1e9
            return {"bound": "hbm", "ms": ms, "algorithmic_bytes": nbytes_alg, "achieved": gbs, "peak": peak_gbs, "unit": "GB/s",
                    "frac": gbs / peak_gbs}

        field_ops["roofline"] = {
            "cic_deposit_kernel (+ memset of rho)": roof(field_ops["deposit_ms"], 32.0 * n_p + 16.0 * nodes),
            "gradient_kernel": roof(field_ops["gradient_ms"], 32.0 * nodes),
            "gather_field_kernel": roof(field_ops["gather_ms"], 48.0 * n_p + 24.0 * nodes),
            "gradient_aos_kernel + gather_aos_kernel": roof(field_ops["field_at_particles_ms"], 48.0 * n_p + 72.0 * nodes),
            "bytes": "deposit: 32 B/particle (x, y, z, q) + 8 B/node memset + 8 B/node of sums; gradient: 8 B/node read + 24 written; "
                     "gather: 24 B/particle read + 24 written + 24 B/node; fused: 48 B/particle + 8 B/node phi + 32 B/node record "
                     "written + 32 read",
        }
        del dpx, dpy, dpz, dpq, f_rho, ex, ey, ez

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
        "kernel_ms_source": (f"a second loop of {min(args.prof_steps, 256)} solves with CUDA events around every launch "
                             f"(dks_poisson_set_profiling); its passes sum to {sum(pass_ms):.4f} ms against ms_per_step "
                             f"{ms_per_step:.4f} of the uninstrumented windows: frac is on the "
                             + ("low side" if sum(pass_ms) >= ms_per_step else
                                "high side (the event gaps let a power-capped board clock higher; sustained_frac is the one to read)")),
        # the dominant kernel's fraction at the sustained (power-capped) clocks, assuming its share of the step is unchanged
        "sustained_frac": (achieved / peak) * ms_per_step / sustained["ms_per_step"] if sustained else None,
        "passes": {dks.dks_poisson_pass_name(plan.handle, i + 1): {
            "ms": pass_ms[i], "model_bytes": plan.model_bytes(i + 1),
            "gbs": plan.model_bytes(i + 1) / (pass_ms[i] * 1e-3) / 1e9} for i in range(len(pass_ms))},
        "whole_solve": {"model_bytes_M3": m3, "gbs": m3 / (ms_per_step * 1e-3) / 1e9,
                        "frac": m3 / (ms_per_step * 1e-3) / 1e9 / peak,
                        "frac_of_8TBs": m3 / (ms_per_step * 1e-3) / 8e12,
                        "sustained_frac": m3 / (sustained["ms_per_step"] * 1e-3) / 1e9 / peak if sustained else None,
                        "sustained_frac_of_8TBs": m3 / (sustained["ms_per_step"] * 1e-3) / 8e12 if sustained else None},
    }
    # a0 (dks_greens_setup: three kernels): the octant is written once by the x kernel and transformed in place along y and z
    g_bytes = 8.0 * (w.n[0] + 1) * (w.n[1] + 1) * (w.n[2] + 1)
    roofline["greens_setup"] = {"bound": "hbm", "ms": greens_ms, "algorithmic_bytes": 5 * g_bytes,
                                "achieved": 5 * g_bytes / (greens_ms * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                                "frac": 5 * g_bytes / (greens_ms * 1e-3) / 1e9 / peak,
                                "bytes": "octant written once (x kernel, G evaluated on the fly) + read and written by the y and the z kernel"}
    plan.close()

    # ---- side reference (north_star: "cuFFT may be timed as a side reference"): the paper-style pipeline
    # of PAPER.md:132 -- library FFT of the zero-padded mesh, separate multiplication, library inverse FFT, crop -- through
    # torch.fft (cuFFT) on the same GPU, Green's transform precomputed as for the product.  Context only: no product code.
    cufft = None
    if world == 1 and not args.no_cufft:
        try:
            cufft = cufft_side_reference(torch, w, d_rho, d_phi, stream)
        except Exception as e:                          # e.g. out of memory on a smaller device: the side reference is optional
            cufft = {"unavailable": repr(e)[:200]}

    # ---- CPU oracle timed beside it (rank 0, N = 1 only) ---------------------------------------------
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        dt, reps, first, cores = oracle_full_solve(w, rho)
        cpu = {"value": 1.0 / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{reps} full solves of {w.name} by oracle/poisson_oracle.c (double build, OpenMP, FT{{G}} precomputed "
                         f"and not timed) after one untimed solve ({first:.2f} s, first touch): {dt:.2f} s each"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(w), "parallelism": "replicas only" if world > 1 else "1 gpu",
                   "l2": ("inputs larger than L2 (rho + phi + workspace >> 126 MB); no explicit flush"
                          if ws_bytes + 2 * nbytes > 126e6 else
                          "working set fits the 126 MB L2 (L2-resident workload); no flush"),
                   "greens_setup": "precomputed, outside the timed region (DESIGN.md reading A11)",
                   "greens_setup_ms": greens_ms, "batched": batched,
                   # the >= --sustained-s run of the same loop (power-capped clocks): the rate a per-time-step solver sees
                   "sustained_solves_per_s": sustained["value"] if sustained else None,
                   "sustained_ms_per_step": sustained["ms_per_step"] if sustained else None,
                   "sustained_sm_mhz": sustained["clocks"].get("sm_mhz") if sustained else None,
                   "timing": "CUDA events on the launching stream, median of the windows; max over ranks"},
        "clocks": clocks_timed,
        "timing": {"windows": len(windows), "ms_per_step_each": [t / args.steps for t in windows],
                   "reported": "median window", "clock_sampling": f"nvidia-smi -lms {ClockSampler.PERIOD_MS} over all windows"},
        "sustained": sustained,
        "field_ops": field_ops,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
                "steps": args.e2e_steps, "timing": "host clock around the loop, device idle before and after",
                "api": "dks_poisson_solve_host_async per step + one dks_poisson_host_sync (pinned host rho -> H2D -> P1..P5 -> "
                       "D2H -> host phi every step; copies of neighbouring steps overlap the solve)",
                "blocking_api_value": e2e_sync_value,
                "with_greens_rebuild_per_step": {"value": e2e_rebuild_value, "unit": UNIT,
                                                 "api": "dks_poisson_step_host_async (new spacings every step: Green's rebuild on its own "
                                                        "stream beside the rho copy, PAPER.md:132) + one dks_poisson_host_sync"},
                "host_link": link},
        "gpu_launches": launches * args.steps,
        "roofline": roofline,
    }
    if cufft is not None:
        line["cufft_side_reference"] = cufft
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
