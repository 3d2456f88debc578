#!/usr/bin/env python
"""bench.py — whole-path throughput of libwri on BASELINE.json's headline workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

One "step" = one complete batched LSQR solve (Golub-Kahan start + maxit iterations + final x
update) of the workload's 64 sources through the C ABI.  Metric: LSQR iterations x sources per
second (sum of per-column iteration counts / time).  `value` is timed with the inputs resident
in HBM; `e2e` is the same solve through wri_lsqr_batch_host with pinned HOST buffers (H2D of q, d
and D2H of u, resnorms, iters inside the timed region).  N > 1 (torchrun): batch columns are
independent systems, so every rank solves its own 64-source group with no
collective on the data path (weak scaling); time = max over ranks.

--impl reference times the complex128 CPU oracle (oracle/) on a bounded sample of the same
workload; it is a deliberately plain program, reported as context.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import workloads  # noqa: E402

METRIC = "lsqr_iterations_x_sources_per_s"
UNIT = "iter*src/s"

WORKLOADS = {
    # BASELINE.json metric: "LSQR iterations.sources/s at 128^3 x 64 src" = configs[2], one
    # frequency group (f = 6 Hz), 200 iterations
    "config2_128cubed_x64src": dict(name="config2", freqs=(6.0,)),
    "config2_128cubed_x192col": dict(name="config2"),
    "config1_64cubed_x16src": dict(name="config1"),
    "config3_vsp_200x200x160_x48src": dict(name="config3"),
    "config4_256cubed_x32src": dict(name="config4"),
}
DEFAULT_WORKLOAD = "config2_128cubed_x64src"

BYTES_PASS_F = 56   # per cell per source: reads v,u,w,x + writes u,w,x (complex64)  [DESIGN.md]
BYTES_PASS_A = 24   # reads u,v + writes v
BYTES_ITER = BYTES_PASS_F + BYTES_PASS_A


def measured_hbm_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic_bytes():
    """dram bytes (read + write) per pass-F launch from the committed ncu capture, or None."""
    path = os.path.join(ROOT, "profiles", "traffic_pass_f.csv")
    try:
        with open(path) as f:
            for line in f:
                if line.startswith("#") or not line.strip():
                    continue
                k, v = line.strip().split(",")[:2]
                if k == "dram_bytes_per_launch":
                    return float(v)
    except Exception:
        pass
    return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            parts = [p.strip() for p in ln.split(",")]
            if len(parts) < 6:
                continue
            try:
                sm.append(float(parts[0]))
                mx.append(float(parts[1]))
            except ValueError:
                continue
            for n, p in zip(names, parts[2:6]):
                if p.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None,
                "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def reduce_over_ranks(times, counts, dist=None, device=None):
    """Whole-job aggregation for N ranks: times -> MAX over ranks, counts -> SUM over ranks.
    (Columns are independent systems, so this is the only cross-rank traffic of the bench.)"""
    if dist is None:
        return list(times), list(counts)
    import torch
    t = torch.tensor(list(times), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor(list(counts), dtype=torch.float64, device=device)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return [float(x) for x in t], [float(x) for x in c]


def e2e_entry(iters_all, serial_steps, serial_s, pipe_steps, pipe_s, h2d, d2h):
    """e2e = host buffers in, host buffers out, copies inside the timed region.  The headline value is
    the pipelined entry (wri_lsqr_batch_host_async: successive steps overlap their copies with the
    neighbouring solves, as an inversion looping over source groups would); the strictly serial
    entry (wri_lsqr_batch_host: upload, solve, download, one after the other) is reported beside it."""
    serial = iters_all * serial_steps / serial_s
    e = {"unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "serial_value": serial,
         "serial_steps": serial_steps}
    if pipe_s is not None and pipe_s != float("inf"):
        e.update(value=iters_all * pipe_steps / pipe_s, steps=pipe_steps,
                 mode="pipelined over the steps (wri_lsqr_batch_host_async + wri_host_wait)")
    else:
        e.update(value=serial, steps=serial_steps, mode="serial (wri_lsqr_batch_host)")
    return e


def oracle_sample(w, cores, iters):
    """Time the CPU oracle as it stands on min(nb, cores) columns x `iters` iterations
    (one column per thread; cores = 1 gives the single-thread figure)."""
    from oracle import oracle as O
    ncols = max(1, min(w.nb, cores))
    cols = list(range(ncols))
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    ops = [O.Operator(w.nx, w.ny, w.nz, w.h, w.omegas[j], w.sponge_width, w.gamma_max, w.power, w.faces)
           for j in w.omega_idx]
    O.build()
    t0 = time.perf_counter()
    out = O.lsqr_batch(ops, w.m, w.lam, rec, w.Q, w.D, None, maxit=iters, threads=ncols, columns=cols)
    dt = time.perf_counter() - t0
    done = int(out["iters"].sum())
    return done / dt, ncols, dt, "%d columns x %d LSQR iterations of %s (incl. Golub-Kahan start)" % (
        ncols, iters, w.name)


def oracle_iters_for(w):
    # ~60 ns per cell per operator application, 2 applications per iteration -> ~10-20 s
    per_iter = 2.6e-7 * w.ng
    return int(max(4, min(64, round(12.0 / per_iter))))


def run_reference(args, wl_name, w):
    rank, world, _ = dist_env()
    if rank != 0:
        return
    cores = os.cpu_count() or 1
    iters = oracle_iters_for(w)
    times, rate, ncols, sample = [], 0.0, 0, ""
    for i in range(args.warmup + args.steps):
        r, ncols, dt, sample = oracle_sample(w, cores, iters)
        if i >= args.warmup:
            times.append(dt)
    total = ncols * iters * len(times)
    value = total / sum(times)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / len(times),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "c128",
            "data": "synthetic",
            "config": {"workload": wl_name, "grid": [w.nx, w.ny, w.nz], "nb": w.nb, "n_rec": w.n_rec,
                       "maxit": w.maxit, "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": ncols, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_width_sweep(args, wl_name, w):
    """Per-pass fraction of the copy bandwidth of the persistent pass kernel at each working width
    a shrinking batch passes through (fixed-K solves of the first nb columns of the workload, per-launch
    CUDA events of wri_profile_*): one JSON line per width.  The tables under profiles/ come from this."""
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    dev = torch.device("cuda", 0)
    from paper_2410_18429_b200 import Wri
    ctx = Wri.from_workload(w, device=dev)
    if args.stencil:
        ctx.set_stencil(args.stencil)
    if args.debug_opts:
        ctx.set_debug_opts(**{k: int(v) for k, v in (kv.split("=") for kv in args.debug_opts.split(","))})
    peak, _ = measured_hbm_peak()
    K = args.maxit or 20
    for nbw in [int(x) for x in args.width_sweep.split(",")]:
        if nbw > w.nb:
            continue
        q = torch.from_numpy(np.ascontiguousarray(w.Q[:, :nbw])).to(dev)
        d = torch.from_numpy(np.ascontiguousarray(w.D[:, :nbw])).to(dev)
        oi = w.omega_idx[:nbw]
        out = ctx._outputs(nbw, K, dev)
        for _ in range(2):
            ctx.lsqr_batch(q, d, w.lam, None, maxit=K, omega_idx=oi, out=out)
        torch.cuda.synchronize()
        ctx.profile_enable(True)
        ctx.profile_read()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            ctx.lsqr_batch(q, d, w.lam, None, maxit=K, omega_idx=oi, out=out)
        e1.record()
        torch.cuda.synchronize()
        ms_f, n_f, cols_f, ms_a, n_a, cols_a = ctx.profile_read()
        ctx.profile_enable(False)
        # the same solves without the per-launch events (they widen the gaps between the kernels)
        e2, e3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e2.record()
        for _ in range(args.steps):
            ctx.lsqr_batch(q, d, w.lam, None, maxit=K, omega_idx=oi, out=out)
        e3.record()
        torch.cuda.synchronize()
        bf = (BYTES_PASS_F * nbw + 4) * w.ng
        ba = (BYTES_PASS_A * nbw + 4) * w.ng
        ach_f = bf / (ms_f / n_f * 1e-3) / 1e9
        ach_a = ba / (ms_a / n_a * 1e-3) / 1e9
        whole = BYTES_ITER * w.ng * nbw * K * args.steps / (e2.elapsed_time(e3) * 1e-3) / 1e9
        print(json.dumps({"workload": wl_name, "nb": nbw, "maxit": K, "plan": ctx.plan_info(nbw + (nbw & 1)),
                          "pass_f": {"ms": ms_f / n_f, "GBps": ach_f, "frac": ach_f / peak},
                          "pass_a": {"ms": ms_a / n_a, "GBps": ach_a, "frac": ach_a / peak},
                          "whole_solve_frac": whole / peak, "ms_per_iteration": e2.elapsed_time(e3) / (K * args.steps)}),
              flush=True)
        del q, d, out


def run_ours(args, wl_name, w):
    import torch
    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    use_dist = world > 1
    if use_dist:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    from paper_2410_18429_b200 import Wri
    ctx = Wri.from_workload(w, device=dev)
    if args.stencil:
        ctx.set_stencil(args.stencil)
    if args.debug_opts:
        ctx.set_debug_opts(**{k: int(v) for k, v in (kv.split("=") for kv in args.debug_opts.split(","))})
    nb, maxit = w.nb, w.maxit
    q = torch.from_numpy(w.Q).to(dev)
    d = torch.from_numpy(w.D).to(dev)
    tol = torch.from_numpy(w.tol).to(dev) if ((w.tol > 0).any() and not args.fixed_k) else None
    ctx.ensure_workspace(nb, host_staging=True, compaction=tol is not None)
    out = ctx._outputs(nb, maxit, dev)

    def barrier():
        if use_dist:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        return ctx.lsqr_batch(q, d, w.lam, tol, maxit=maxit, omega_idx=w.omega_idx, out=out)

    for _ in range(args.warmup):
        step()
    barrier()
    iters_per_step = int(out[2].sum().item())

    # ---- device-resident timing (value) and clock sampling: K steps as a user runs them, no
    #      instrumentation inside (events between the launches would serialise them and undo the
    #      programmatic dependent launch of the passes)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    l0 = ctx.launch_count()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    launches = ctx.launch_count() - l0
    # ---- the same K steps once more with a pair of CUDA events around every pass launch on the
    #      library's stream (wri_profile_*): per-kernel durations for the roofline
    ctx.profile_enable(True)
    ctx.profile_read()
    barrier()
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record()
    for _ in range(args.steps):
        step()
    p1.record()
    barrier()
    ms_profiled = p0.elapsed_time(p1)
    ms_f, n_f, cols_f, ms_a, n_a, cols_a = ctx.profile_read()
    ctx.profile_enable(False)
    clocks = sampler.stop() if rank == 0 else None
    time.sleep(0.3)          # let nvidia-smi go: its start-up and exit stall launches for tens of ms on a short run

    # ---- end-to-end timing through the host-buffer entry
    qh = torch.from_numpy(w.Q).pin_memory()
    dh = torch.from_numpy(w.D).pin_memory()
    tolh = torch.from_numpy(w.tol).pin_memory() if tol is not None else None
    outh = (torch.empty((w.ng, nb), dtype=torch.complex64).pin_memory(),
            torch.empty((maxit + 1, nb), dtype=torch.float32).pin_memory(),
            torch.empty(nb, dtype=torch.int32).pin_memory())
    e2e_steps = max(1, args.steps)
    ctx.lsqr_batch_host(qh, dh, w.lam, tolh, maxit=maxit, omega_idx=w.omega_idx, out=outh)   # warm-up
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        ctx.lsqr_batch_host(qh, dh, w.lam, tolh, maxit=maxit, omega_idx=w.omega_idx, out=outh)
    barrier()
    e2e_s = time.perf_counter() - t0
    # the same steps through the pipelined host entry: step i+1's upload and step i-1's download ride
    # under step i's solve on the library's copy streams; every step's copies are inside the timed region
    e2e_pipe_s, e2e_pipe_steps = None, max(e2e_steps, args.steps)
    try:
        ctx.lsqr_batch_host_async(qh, dh, w.lam, tolh, maxit=maxit, omega_idx=w.omega_idx, out=outh)   # warm-up
        ctx.host_wait()
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_pipe_steps):
            ctx.lsqr_batch_host_async(qh, dh, w.lam, tolh, maxit=maxit, omega_idx=w.omega_idx, out=outh)
        ctx.host_wait()
        barrier()
        e2e_pipe_s = time.perf_counter() - t0
    except Exception as e:                                       # keep the serial number if the pipeline fails
        sys.stderr.write("bench.py: pipelined host entry failed: %r\n" % (e,))
    h2d = qh.numel() * 8 + dh.numel() * 8 + (tolh.numel() * 4 if tolh is not None else 0)
    d2h = outh[0].numel() * 8 + outh[1].numel() * 4 + outh[2].numel() * 4
    iters_e2e = int(outh[2].sum().item())

    # ---- the same workload through the paper's own source-free system (unknown source weight per
    #      column, eq. 4-6) and one objective + gradient evaluation (eq. 8-9); context lines, N = 1 only
    extras = None
    if world == 1 and not args.no_extras and w.src_ijk is not None:
        extras = {}
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
        ctx.lsqr_sf_batch(d, w.lam, w.src_ijk, tol, maxit=maxit, omega_idx=w.omega_idx)      # warm-up
        torch.cuda.synchronize()
        ev[0].record()
        n_sf = 2
        for _ in range(n_sf):
            u_sf, a_sf, _, it_sf = ctx.lsqr_sf_batch(d, w.lam, w.src_ijk, tol, maxit=maxit, omega_idx=w.omega_idx)
        ev[1].record()
        torch.cuda.synchronize()
        ms_sf = ev[0].elapsed_time(ev[1]) / n_sf
        extras["sourcefree_lsqr"] = {"value": int(it_sf.sum().item()) / (ms_sf * 1e-3), "unit": UNIT,
                                     "ms_per_step": ms_sf, "system": "S = [lam A, -lam e; P, 0], b = [0; d]"}
        g = torch.zeros(w.ng, dtype=torch.float32, device=dev)
        ctx.objective_gradient(u_sf, d, w.lam, omega_idx=w.omega_idx, src_ijk=w.src_ijk, alpha=a_sf, g=g)
        torch.cuda.synchronize()
        n_g = 5
        ev[2].record()
        for _ in range(n_g):
            ctx.objective_gradient(u_sf, d, w.lam, omega_idx=w.omega_idx, src_ijk=w.src_ijk, alpha=a_sf, g=g)
        ev[3].record()
        torch.cuda.synchronize()
        ms_g = ev[2].elapsed_time(ev[3]) / n_g
        bytes_g = (8 * nb + 4 + 8) * w.ng          # u read once, m read, g read + written
        peak_g, _ = measured_hbm_peak()
        # this pass is bound by its instruction stream: 2.22 executed warp-instructions per
        # cell-column (ncu, profiles/r02_gradient.md) against 148 SMs x 4 schedulers x the maximum SM clock
        alu_peak = 148 * 4 * 1.965e9
        extras["objective_gradient"] = {"ms": ms_g, "algorithmic_bytes": bytes_g,
                                        "achieved": bytes_g / (ms_g * 1e-3) / 1e9, "unit": "GB/s",
                                        "frac": bytes_g / (ms_g * 1e-3) / 1e9 / peak_g,
                                        "bound": "alu", "warp_instructions_per_cell_column": 2.22,
                                        "frac_alu": 2.22 * w.ng * nb / (ms_g * 1e-3) / alu_peak,
                                        "clock_state": "timed right after the K steps, at the sustained "
                                                       "(power-capped) SM clock of `clocks`, not at the burst clock",
                                        "kernel": "k_pass_rt<MODE_G> + k_add_f32 + k_objective (eq. 9 fused with "
                                                  "the stencil residual); k_grad at widths the pass kernel "
                                                  "does not take"}
        # the operator entries on their own (wri_apply_M / wri_apply_MH): read x, write y = 16 B per cell-column
        ev2 = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
        yb = torch.empty((w.n_rec, nb), dtype=torch.complex64, device=dev)
        yt = torch.empty_like(u_sf)
        ctx.apply_M(u_sf, w.lam, w.omega_idx, out=(yt, yb)); ctx.apply_MH(u_sf, yb, w.lam, w.omega_idx, out=yt)
        torch.cuda.synchronize()
        n_ap = 20
        ev2[0].record()
        for _ in range(n_ap):
            ctx.apply_M(u_sf, w.lam, w.omega_idx, out=(yt, yb))
        ev2[1].record()
        ev2[2].record()
        for _ in range(n_ap):
            ctx.apply_MH(u_sf, yb, w.lam, w.omega_idx, out=yt)
        ev2[3].record()
        torch.cuda.synchronize()
        bytes_ap = (16 * nb + 4) * w.ng
        for nm, a, b in (("apply_M", 0, 1), ("apply_MH", 2, 3)):
            ms_ap = ev2[a].elapsed_time(ev2[b]) / n_ap
            extras[nm] = {"ms": ms_ap, "algorithmic_bytes": bytes_ap, "achieved": bytes_ap / (ms_ap * 1e-3) / 1e9,
                          "unit": "GB/s", "frac": bytes_ap / (ms_ap * 1e-3) / 1e9 / peak_g,
                          "note": "the C call into caller-allocated outputs (pass kernel + receiver rows)"}
        del yb, yt
        # one misfit evaluation (Algorithm 2 lines 4-5; the unit the paper times in Table 1):
        # source-free solve of every column to a tolerance + objective + gradient, one C-ABI call
        eps_m = 1e-2
        ctx.misfit_sf(d, w.lam, w.src_ijk, eps_m, maxit, omega_idx=w.omega_idx, g=g)           # warm-up
        t0 = time.perf_counter()
        mf = ctx.misfit_sf(d, w.lam, w.src_ijk, eps_m, maxit, omega_idx=w.omega_idx, g=g)       # synchronises (f)
        s_m = time.perf_counter() - t0
        it_m = int(mf["iters"].sum().item())
        extras["misfit_evaluation"] = {"ms": s_m * 1e3, "eps": eps_m, "lsqr_iterations_x_sources": it_m,
                                       "value": it_m / s_m, "unit": UNIT, "f": mf["f"],
                                       "timing": "host wall clock around wri_misfit_sf (it ends with a stream sync)"}
        del u_sf, g, mf

    # ---- N > 1: the misfit of all ranks' columns with its one collective, the all-reduce of the
    #      gradient and the objective (eq. 8-9 are sums over sources and frequencies); context line
    if use_dist and not args.no_extras and w.src_ijk is not None:
        try:
            from paper_2410_18429_b200.sharded import ShardedMisfit

            def evaluate(lo, hi, eps, mit, g, warm):          # every rank owns one nb-column group
                o = ctx.misfit_sf(d, w.lam, w.src_ijk, eps, mit, omega_idx=w.omega_idx, g=g)
                return o["f"], int(o["iters"].sum().item()), None

            sm = ShardedMisfit(nb * world, evaluate, w.ng, dev, dist)
            sm.misfit(1e-2, maxit)                               # warm-up (NCCL communicator, workspace)
            barrier()
            t0 = time.perf_counter()
            f_all, g_all, it_all, _ = sm.misfit(1e-2, maxit)
            barrier()
            s_sm = time.perf_counter() - t0
            extras = extras or {}
            extras["sharded_misfit"] = {"ms": s_sm * 1e3, "eps": 1e-2, "columns": nb * world,
                                        "lsqr_iterations_x_sources": it_all, "value": it_all / s_sm, "unit": UNIT,
                                        "f": f_all, "collective": "all-reduce of g (float32 [n_g]) and f over NCCL",
                                        "g_norm": float(g_all.double().norm().item())}
        except Exception as e:                                   # a context line must never cost the bench line
            extras = extras or {}
            extras["sharded_misfit"] = {"error": repr(e)}

    (ms, e2e_s, e2e_pipe_s), (iters_all, iters_e2e_all, launches_all) = reduce_over_ranks(
        [ms, e2e_s, e2e_pipe_s if e2e_pipe_s is not None else float("inf")],
        [iters_per_step, iters_e2e, launches], dist if use_dist else None, dev)
    launches_all = int(launches_all)

    if rank == 0:
        value = iters_all * args.steps / (ms * 1e-3)
        peak, peak_src = measured_hbm_peak()
        cells = w.ng * nb
        # bytes per launch from the widths the launches really had (compaction narrows the batch)
        bytes_f = (BYTES_PASS_F * w.ng * cols_f + 4 * w.ng * n_f) / max(n_f, 1)
        bytes_a = (BYTES_PASS_A * w.ng * cols_a + 4 * w.ng * n_a) / max(n_a, 1)
        ach_f = bytes_f / (ms_f / max(n_f, 1) * 1e-3) / 1e9 if n_f else None
        ach_a = bytes_a / (ms_a / max(n_a, 1) * 1e-3) / 1e9 if n_a else None
        # whole-iteration algorithmic bandwidth over the full step (includes start/end kernels)
        ach_iter = BYTES_ITER * w.ng * iters_per_step * args.steps / (ms * 1e-3) / 1e9
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "c64", "data": "synthetic",
            "config": {"workload": wl_name, "grid": [w.nx, w.ny, w.nz], "h": w.h, "nb": nb,
                       "n_rec": w.n_rec, "freqs_hz": list(w.freqs), "lambda": w.lam, "maxit": maxit,
                       "iters_per_step": iters_per_step, "sharding": "columns per rank, no collective",
                       "stencil": "27-point" if args.stencil else "7-point", "tile_plan": ctx.plan_info(nb + (nb & 1)),
                       "l2": "working set %.1f GB per rank exceeds the 126 MB L2" % (4 * cells * 8 / 1e9)},
            "clocks": clocks,
            "e2e": e2e_entry(iters_e2e_all, e2e_steps, e2e_s, e2e_pipe_steps, e2e_pipe_s, h2d, d2h),
            "gpu_launches": launches_all,
            "roofline": {"bound": "hbm", "kernel": "k_pass_rt<MODE_F> (forward stencil + u axpy + x,w update + ||u||^2)",
                         "achieved": ach_f, "peak": peak, "peak_source": peak_src, "unit": "GB/s",
                         "frac": (ach_f / peak) if ach_f else None,
                         "traffic": ncu_traffic_bytes() if wl_name == DEFAULT_WORKLOAD else None,
                         "traffic_source": ("profiles/traffic_pass_f.csv (static: one ncu --set full capture of this "
                                            "kernel at this workload, committed; not re-measured per run)"
                                            if wl_name == DEFAULT_WORKLOAD else None),
                         "algorithmic_bytes_per_launch": bytes_f,
                         "avg_launch_ms": ms_f / max(n_f, 1), "launches_timed": n_f,
                         "avg_columns_per_launch": cols_f / max(n_f, 1),
                         "pass_a": {"achieved": ach_a, "frac": (ach_a / peak) if ach_a else None,
                                    "avg_launch_ms": ms_a / max(n_a, 1)},
                         "whole_step": {"achieved": ach_iter, "frac": ach_iter / peak,
                                        "frac_of_8000": ach_iter / 8000.0},
                         "timing": "per-kernel CUDA events over a second run of the same K steps (ms_per_step_profiled); "
                                   "value and whole_step from the K steps timed without events inside",
                         "ms_per_step_profiled": ms_profiled / args.steps},
        }
        if extras:
            line["extras"] = extras
            for key, src in (("pass_g", "objective_gradient"), ("apply_M", "apply_M"), ("apply_MH", "apply_MH")):
                if src in extras and "frac" in extras[src]:
                    line["roofline"][key] = {"achieved": extras[src]["achieved"], "frac": extras[src]["frac"],
                                             "ms": extras[src]["ms"]}
                    if "frac_alu" in extras[src]:
                        line["roofline"][key]["frac_alu"] = extras[src]["frac_alu"]
        if world == 1 and not args.no_cpu_baseline:
            cores = os.cpu_count() or 1
            r, ncols, dt, sample = oracle_sample(w, cores, oracle_iters_for(w))
            line["cpu_baseline"] = {"value": r, "unit": UNIT, "cores": ncols, "kind": "oracle",
                                    "sample": sample, "seconds": dt}
            it1 = max(2, oracle_iters_for(w) // 2)
            r1, _, dt1, sample1 = oracle_sample(w, 1, it1)
            line["cpu_baseline"]["one_thread"] = {"value": r1, "unit": UNIT, "cores": 1, "sample": sample1,
                                                  "seconds": dt1}
        print(json.dumps(line), flush=True)
    if use_dist:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=sorted(WORKLOADS))
    ap.add_argument("--maxit", type=int, default=None, help="override the workload's iteration count")
    ap.add_argument("--nb", type=int, default=None,
                    help="sub-sample the workload's columns to this batch width (per-width kernel tables)")
    ap.add_argument("--fixed-k", action="store_true",
                    help="ignore the workload's tolerances: every column runs maxit iterations")
    ap.add_argument("--stencil", type=int, default=0, choices=[0, 1],
                    help="0: 7-point (north_star), 1: 27-point box discretisation of the Laplacian")
    ap.add_argument("--debug-opts", default=None,
                    help="tuning switches of wri_debug_opts, e.g. txc=4,tyc=4,nstage_a=8 (sweeps under profiles/)")
    ap.add_argument("--width-sweep", default=None,
                    help="comma-separated batch widths: per-pass roofline fractions of fixed-K solves at each "
                         "width, one JSON line per width (instead of the bench line)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true",
                    help="skip the source-free solve and the objective/gradient context lines")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference" and dist_env()[0] != 0:
        return                                   # the oracle arm runs on rank 0 alone
    spec = dict(WORKLOADS[args.workload])
    if args.nb:
        spec["nb"] = args.nb
    w = workloads.make(spec.pop("name"), **spec)
    if args.maxit:
        w.maxit = args.maxit
    if args.impl == "reference":
        run_reference(args, args.workload, w)
    elif args.width_sweep:
        run_width_sweep(args, args.workload, w)
    else:
        run_ours(args, args.workload, w)


if __name__ == "__main__":
    main()
