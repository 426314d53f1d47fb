#!/usr/bin/env python
"""bench.py — projected samples/s to ||h||_inf < 1e-10 (fp64) and achieved fraction of the HBM roofline.

Headline workload (BASELINE.json configs[4], "cfg5"): 1D Burgers at scale — batch 1024, 256x256,
Lax-Friedrichs finite-volume rows + IC rows + per-level mass border rows, projected at 50 interleaved
flow-matching times tau_j = j/50 with the multiplier warm start carried from tau to tau.
One "step" = that whole 50-call sequence = 51 200 projections.  All 50 inputs (25.6 GB) are resident in
HBM before the timed region, so the working set is far larger than L2 and no L2 flush is needed.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg5|cfg1..cfg4|cfg6|cfg7|cfg8] [--impl reference]

Multi-GPU (torchrun): samples are independent blocks, so each rank projects its own
batch of the same size with no data-path collective ("scaling": "weak"); NCCL carries only the barrier
and the max-over-ranks of the device time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import workloads as W  # noqa: E402

METRIC = "projected samples/sec to ||h||inf<1e-10 (fp64, 1 B200); % of HBM roofline"
UNIT = "projections/s"
N_TAU = 50
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "traffic.json")   # written next to the ncu summaries it quotes


def profiled_traffic(cfg: int):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the latest
    `ncu --set full` capture summarised under profiles/ (profiles/traffic.json names the summary it comes from).
    None if no capture of this workload is recorded."""
    try:
        with open(TRAFFIC_FILE) as f:
            return json.load(f).get(f"cfg{cfg}")
    except Exception:
        return None


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            pk = json.load(f)
        return float(pk["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def algorithmic_bytes(run):
    """Bytes one snap_project launch must move, from the kernel's own per-sample work counters
    (snap_project_stats): (rows read + rows written) x doubles per row x 8.  A "row" is one time level of one
    field; the counters describe the traffic of the variant that actually ran, e.g. 88 n bytes for
    a typical cfg-5 projection on the fused path -- not the 64 n per iteration model of SURVEY.md §8(d)."""
    st = run.stats.cpu()
    S = run.S
    rows = (st[:, S.STAT_ROWS_READ] + st[:, S.STAT_ROWS_WRITTEN]).to(torch.float64)
    return float((rows * st[:, S.STAT_ROW_DOUBLES].to(torch.float64)).sum() * 8.0)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "25"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            parts = [x.strip() for x in r.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0]))
                smax.append(float(parts[1]))
            except ValueError:
                continue
            for nm, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------------------------------
# reference arm = the oracle, as it stands, on the host cores (bounded sample)
# ------------------------------------------------------------------------------------------------------
def oracle_sample(cfg: int, n_samples: int, workers: int, taus=(25,)):
    """Time the CPU oracle, as it stands, on `n_samples` problems of workload `cfg` (for cfg 5: at each flow time
    tau_j, j in `taus`).  Returns (projections/s, seconds, description, workers used)."""
    import oracle as O
    total_t, total_n, ok = 0.0, 0, True
    used = workers
    if cfg == 5:
        wl = W.make_workload(5, batch=n_samples, with_u_hat=False)
        for j in taus:
            uh = W.burgers_tau_input(wl, j)
            t0 = time.perf_counter()
            out = O.project_batch(wl.kind, uh.numpy(), wl.cdata.numpy(), wl.params, workers=workers)
            total_t += time.perf_counter() - t0
            total_n += n_samples
            ok = ok and bool((out["iters"] > 0).all())
            used = out["workers"]
        desc = (f"{n_samples} samples of cfg5 (256x256, Burgers-LF + mass rows) at each of tau in "
                f"{{{', '.join(f'{j}/{N_TAU}' for j in taus)}}}")
    else:
        wl = W.make_workload(cfg, batch=n_samples)
        t0 = time.perf_counter()
        out = O.project_batch(wl.kind, wl.u_hat.numpy(), wl.cdata.numpy(), wl.params, workers=workers)
        total_t = time.perf_counter() - t0
        total_n = n_samples
        ok = bool((out["iters"] > 0).all())
        used = out["workers"]
        desc = f"{n_samples} samples of cfg{cfg}"
    return total_n / total_t, total_t, desc + ("" if ok else " [oracle reported non-convergence]"), used


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = int(args.workload[3:])
    cores = os.cpu_count() or 1
    workers = min(cores, 16)
    n_samples = workers if cfg in (4, 5, 6, 7, 8, 9) else max(workers, 16)
    times = []
    desc = ""
    for s in range(args.warmup + args.steps):
        v, dt, desc, used = oracle_sample(cfg, n_samples, workers, taus=(25,))
        if s >= args.warmup:
            times.append(dt)
    total = sum(times)
    value = n_samples * len(times) / total
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / len(times), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "reference": "CPU oracle (oracle/, numpy/scipy), one step = a bounded sample"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": used, "host_cpu_count": cores, "kind": "oracle",
                         "sample": desc + " per step"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_name(cfg: int) -> str:
    return {
        1: "cfg1: 1D heat IC+mass projection, batch 4, 64x64 (linear)",
        2: "cfg2: 1D viscous Burgers LF projection, batch 32, 128x128",
        3: "cfg3: 1D Fisher-KPP implicit projection, batch 256, 128x128",
        4: "cfg4: 2D Allen-Cahn implicit projection, batch 64, 64x64x32 (product-form sweeps, level solves in shared memory)",
        5: "cfg5: 1D Burgers LF + mass rows at scale, batch 1024, 256x256, 50 flow times tau=j/50, warm-started",
        6: "cfg6 (SURVEY 8(f) NEXT-1): Burgers IC + Flux(k=5, Lax-Friedrichs) + mass + energy rows, batch 1024, 256x256 (wide J, banded border solve)",
        7: "cfg7 (SURVEY 8(f) NEXT-1/4): inviscid Burgers IC + Flux(k=5, Godunov) + mass rows, batch 1024, 256x256",
        8: "cfg8 (SURVEY 8(f) NEXT-2): cfg6 with the exact Lagrangian Hessian (Newton-KKT, quadratic rate)",
        9: "cfg9 (paper Eq. 20): 2D Navier-Stokes vorticity rows IC + total vorticity + enstrophy, batch 256, 16x16x50 (closed form per level)",
    }[cfg]


# ------------------------------------------------------------------------------------------------------
# GPU arm
# ------------------------------------------------------------------------------------------------------
class GpuRun:
    """One workload resident on the device, ready to be stepped."""

    def __init__(self, S, cfg: int, dev, seed_offset: int = 0):
        self.S, self.cfg, self.dev = S, cfg, dev
        kind, B, nx, ny, nt, seed = W.CONFIG_SHAPES[cfg]
        self.wl = W.make_workload(cfg, device=dev, with_u_hat=(cfg != 5), seed=seed + 1000 * seed_offset)
        wl = self.wl
        self.p = S.snap_problem_create(wl.kind, wl.nx, wl.ny, wl.nt, wl.params)
        self.B = wl.batch
        if cfg == 5:
            self.inputs = [W.burgers_tau_input(wl, j) for j in range(1, N_TAU + 1)]
        else:
            self.inputs = [wl.u_hat]
        self.calls = len(self.inputs)
        self.cdata = wl.cdata.contiguous()
        self.u_star = torch.empty(self.B, wl.n, dtype=torch.float64, device=dev)
        self.lam = torch.zeros(self.B, self.p.m, dtype=torch.float64, device=dev)
        self.iters = torch.zeros(self.calls, self.B, dtype=torch.int32, device=dev)
        self.ws = torch.empty(S.snap_workspace_bytes(self.p, self.B), dtype=torch.uint8, device=dev)
        self.norms = torch.empty(self.B, 5, dtype=torch.float64, device=dev)
        self.stats = torch.zeros(self.B, S.STAT_COUNT, dtype=torch.int64, device=dev)

    lam_free = False     # True: multiplier-free calls (lambda = NULL), the sampler-facing variant (Eq. 3)

    def step(self, events=None):
        """The whole hot path over one batch of input: `calls` back-to-back snap_project launches."""
        for c, uh in enumerate(self.inputs):
            if events is not None:
                events[c][0].record()
            self.S.snap_project(self.p, self.B, uh, self.cdata, self.u_star, None if self.lam_free else self.lam, self.iters[c],
                                warm=(self.cfg == 5 and c > 0 and not self.lam_free), workspace=self.ws)
            if events is not None:
                events[c][1].record()

    def traffic_model(self):
        """Untimed replay of one step that reads the kernel's own per-sample row counters after every call
        (deterministic: same inputs, same counts as the timed steps).  Returns algorithmic bytes per call."""
        out = []
        for c, uh in enumerate(self.inputs):
            self.S.snap_project(self.p, self.B, uh, self.cdata, self.u_star, None if self.lam_free else self.lam, self.iters[c],
                                warm=(self.cfg == 5 and c > 0 and not self.lam_free), workspace=self.ws)
            self.S.snap_project_stats(self.p, self.B, self.ws, self.stats)
            torch.cuda.synchronize()
            out.append(algorithmic_bytes(self))
        self.variants = sorted(set(self.stats[:, self.S.STAT_VARIANT].cpu().tolist()))
        return out

    def check(self):
        """Every sample converged and the last call's output is feasible."""
        it = self.iters.cpu()
        self.S.snap_residual(self.p, self.B, self.u_star, self.cdata, None, self.norms)
        hmax = float(self.norms[:, 0].max())
        return bool((it > 0).all()), hmax, it

    def projections_per_step(self):
        return self.B * self.calls


def time_steps(run: GpuRun, steps: int, warmup: int, dist):
    for _ in range(warmup):
        run.step()
    ev = [[(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(run.calls)]
          for _ in range(steps)]
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    l0 = run.p.launch_count()
    t0 = torch.cuda.Event(enable_timing=True)
    t1 = torch.cuda.Event(enable_timing=True)
    torch.cuda.profiler.start()       # cudaProfilerStart: `ncu --profile-from-start off` sees the timed region only
    t0.record()
    for s in range(steps):
        run.step(ev[s])
    t1.record()
    torch.cuda.synchronize()
    torch.cuda.profiler.stop()
    if dist is not None:
        dist.barrier()
    total_ms = t0.elapsed_time(t1)
    launches = run.p.launch_count() - l0
    kern_ms = [[a.elapsed_time(b) for a, b in evs] for evs in ev]
    return total_ms, kern_ms, launches


def e2e_steps(run: GpuRun, steps: int, warmup: int):
    """Same metric through the host-buffer C-ABI entry: every call copies its input from pinned host memory
    and reads u*, lam, iters back, inside the timed region."""
    S, wl, p, B = run.S, run.wl, run.p, run.B
    host_in = [x.cpu().pin_memory() for x in run.inputs]
    cd = run.cdata.cpu().pin_memory()
    us = torch.empty(B, wl.n, dtype=torch.float64).pin_memory()
    lam = torch.zeros(B, p.m, dtype=torch.float64).pin_memory()
    it = torch.empty(B, dtype=torch.int32).pin_memory()

    def one():
        for c, uh in enumerate(host_in):
            S.snap_project_host(p, B, uh, cd, us, lam, it, warm=(run.cfg == 5 and c > 0))

    for _ in range(warmup):
        one()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(steps):
        one()
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    warm_calls = (run.calls - 1) if run.cfg == 5 else 0
    h2d = run.calls * (B * wl.n * 8 + B * wl.nx * wl.ny * 8) + warm_calls * B * p.m * 8
    d2h = run.calls * (B * wl.n * 8 + B * p.m * 8 + B * 4)
    ok = bool((it > 0).all())
    return run.projections_per_step() * steps / dt, h2d, d2h, ok


def flow_step_lines(run, steps, warmup):
    """PCFM step around the projection (Eq. 1-3): the fused snap_flow_step (one launch per
    flow step, multiplier-free) against the same three operations as separate launches (torch elementwise shoot, snap_project,
    torch elementwise pull-back).  Stub velocity = 0, so u_hat_j is the headline workload's input j and the projections are
    the headline's; the velocity, prior and u_next fields are still read / written."""
    S, p, B, dev = run.S, run.p, run.B, run.dev
    n = run.wl.n
    vel = torch.zeros(B, n, dtype=torch.float64, device=dev)
    g = torch.Generator(device=dev).manual_seed(99)
    prior = torch.randn(B, n, generator=g, dtype=torch.float64, device=dev)
    u1 = torch.empty(B, n, dtype=torch.float64, device=dev)
    un = torch.empty(B, n, dtype=torch.float64, device=dev)
    uh_tmp = torch.empty(B, n, dtype=torch.float64, device=dev)
    taus = [(c + 1) / N_TAU for c in range(run.calls)]

    def fused():
        for c, ut in enumerate(run.inputs):
            S.snap_flow_step(p, B, ut.view(B, n), vel, prior, taus[c], min(1.0, taus[c] + 1.0 / N_TAU), run.cdata, u1, un, None,
                             run.iters[c], workspace=run.ws)

    def unfused():
        for c, ut in enumerate(run.inputs):
            torch.add(ut.view(B, n), vel, alpha=1.0 - taus[c], out=uh_tmp)                      # Eq. 1
            S.snap_project(p, B, uh_tmp, run.cdata, u1, None, run.iters[c], workspace=run.ws)   # Eq. 2
            torch.lerp(prior, u1, min(1.0, taus[c] + 1.0 / N_TAU), out=un)                      # Eq. 3

    out = {}
    for name, fn in (("fused", fused), ("separate_launches", unfused)):
        for _ in range(warmup):
            fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / steps
        out[name] = {"ms_per_step": ms, "flow_steps_per_s": B * run.calls / (ms * 1e-3), "converged_all": bool((run.iters > 0).all())}
    S.snap_project_stats(p, B, run.ws, run.stats)
    torch.cuda.synchronize()
    out["note"] = ("50 flow steps x 1024 samples, multiplier-free; fused = snap_flow_step (Eq. 1 in the first forward pass, Eq. 3 in "
                   "the final stream), separate = torch.add + snap_project + torch.lerp")
    return out


def float32_lines(run, steps, warmup, peak):
    """The paper's arithmetic setting (Float32, solver tolerance 1e-5) on the headline
    workload: the same 50 inputs cast to fp32, multiplier-free snap_project_f32.  Bytes: the kernel reads the iterate and
    writes the next one per pass (4 n bytes each) -- counted from the evaluations it reports."""
    S, p, B, dev = run.S, run.p, run.B, run.dev
    n = run.wl.n
    inputs = [x.to(torch.float32).reshape(B, n).contiguous() for x in run.inputs]
    cd = run.cdata.to(torch.float32).contiguous()
    us = torch.empty(B, n, dtype=torch.float32, device=dev)
    iters = torch.zeros(run.calls, B, dtype=torch.int32, device=dev)

    def step():
        for c, uh in enumerate(inputs):
            S.snap_project_f32(p, B, uh, cd, us, iters[c], tol=1e-5, workspace=run.ws)

    for _ in range(warmup):
        step()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    it = iters.cpu()
    ok = bool((it > 0).all())
    norms = torch.empty(B, 5, dtype=torch.float64, device=dev)
    S.snap_residual(p, B, us.double(), cd.double(), None, norms)
    torch.cuda.synchronize()
    # passes: an evaluation count e means ceil((e - 1) / 3) passes of up to 3 updates, read + write 4 n bytes each (the
    # iterates alternate between a work buffer and u_star: the usual two passes end in u_star, no copy)
    passes = torch.ceil((it.clamp(min=1).double() - 1.0) / 3.0).clamp(min=1.0)
    alg = float(passes.sum()) * 8.0 * n
    return {"value": B * run.calls / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms, "dtype": "f32", "tol": 1e-5,
            "converged_all": ok, "max_hinf_last_call_fp64": float(norms[:, 0].max()),
            "mean_evaluations_per_projection": float(it.clamp(min=0).double().mean()),
            "alg_bytes_per_projection": alg / (B * run.calls), "achieved_GBs": alg / (ms * 1e-3) / 1e9,
            "frac_of_measured_hbm": alg / (ms * 1e-3) / 1e9 / peak,
            "note": "snap_project_f32: the paper's Float32 / 1e-5 setting, multiplier-free, same inputs cast to fp32"}


KERNEL_NAMES = {5: "project1d_fused_kernel<KB,1,8,3> (Burgers family, nx=256)", 2: "project1d_fused_kernel<KB,1,4,4> (nx=128)",
                3: "project1d_fused_kernel<KF,1,4,3> (Fisher, nx=128)",
                4: "project2d_direct_kernel<4,256> (variant 6; variant 5 = project2d_kernel, PCG)",
                1: "heat_project_kernel", 6: "project1d_fluxk_kernel<8,LF>", 7: "project1d_fluxk_kernel<8,Godunov>",
                8: "project1d_fluxk_kernel<8,LF> (hessian = 1)", 9: "ns_project_kernel"}


def roofline_of(run, cfg, kern_s, alg_bytes_call, steps, peak, peak_src):
    """HBM roofline of the workload's (single) kernel: algorithmic bytes per launch / live CUDA-event duration."""
    alg_total = sum(alg_bytes_call) * steps
    achieved = alg_total / kern_s / 1e9
    prof = profiled_traffic(cfg)
    out = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
           "traffic": None, "kernel": KERNEL_NAMES[cfg], "variants": getattr(run, "variants", None),
           "peak_source": peak_src, "alg_bytes_per_launch_mean": alg_total / (steps * run.calls),
           "launch_ms_mean": 1e3 * kern_s / (steps * run.calls), "frac_of_8TBs_spec": achieved / 8000.0,
           "achieved_is": "model-based: the kernel's own row counters x row bytes / CUDA-event time"}
    if prof is not None:
        out["traffic"] = prof["dram_bytes_per_launch"]
        out["traffic_note"] = prof.get("note")
        # the same fraction on measured DRAM bytes: scale by the profiled launch's DRAM / algorithmic ratio
        ratio = prof["dram_bytes_per_launch"] / prof["alg_bytes_per_launch"]
        out["frac_dram"] = achieved * ratio / peak
        out["dram_over_alg"] = ratio
    return out


def run_gpu(args):
    from paper_2607_00095_b200 import sharding as SH
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        os.environ.setdefault("NCCL_DEBUG", "WARN")
        dist_mod.init_process_group(backend=args.backend)
        dist = dist_mod
    if args.selftest_dist:
        # launcher / reduction plumbing only (CPU, gloo): every rank reports fake device times
        ms, units, ok = SH.reduce_timing(dist, torch.device("cpu"), 10.0 + rank, 100, True)
        if rank == 0:
            print(json.dumps({"selftest": "dist", "n_gpus": world, "max_ms": ms, "units": units, "ok": ok,
                              "value": SH.throughput(units, 1, ms)}), flush=True)
        if dist is not None:
            dist.destroy_process_group()
        return
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    import paper_2607_00095_b200 as S
    S.load_library()          # fails loudly if libsnap.so is missing: there is no fallback path

    cfg = int(args.workload[3:])
    run = GpuRun(S, cfg, dev, seed_offset=rank)
    wl, p = run.wl, run.p
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    total_ms, kern_ms, launches = time_steps(run, args.steps, args.warmup, dist)
    clocks = sampler.stop() if rank == 0 else None
    ok, hmax, iters = run.check()

    # max over ranks of the device time, sum of the units, AND of the converged flags (sharding.reduce_timing)
    total_ms, units, ok = SH.reduce_timing(dist, dev, total_ms, run.projections_per_step(), ok)
    value = SH.throughput(units, args.steps, total_ms)

    # roofline of the dominant kernel (the persistent projection kernel), live CUDA-event durations
    peak, peak_src = load_peaks()
    solves = iters.clamp(min=0).sum(dim=1).to(torch.float64)        # per call, over the batch
    alg_bytes_call = run.traffic_model()
    kern_s = sum(sum(k) for k in kern_ms) * 1e-3
    roof = roofline_of(run, cfg, kern_s, alg_bytes_call, args.steps, peak, peak_src)
    if args.traffic is not None:
        roof["traffic"] = args.traffic
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "batch_per_gpu": run.B, "nx": wl.nx, "ny": wl.ny, "nt": wl.nt,
                   "calls_per_step": run.calls, "projections_per_step": units,
                   "l2": "inputs (25.6 GB resident) exceed L2; no flush" if cfg == 5 else
                         ("iterate / multiplier vectors (0.4 GB) exceed L2; no flush" if cfg == 4 else
                          ("input + iterates (1.5 GB) exceed L2; no flush" if cfg in (6, 7, 8) else
                           "working set smaller than L2 (latency-bound config; see DESIGN.md)")),
                   "tol": wl.params["tol"], "converged_all": ok, "max_hinf_last_call": hmax,
                   "mean_linearisations_per_projection": float(solves.sum() / (run.B * run.calls)),
                   "alg_bytes_per_projection": sum(alg_bytes_call) / (run.B * run.calls)},
        "roofline": roof,
        "gpu_launches": launches,
        "clocks": clocks,
    }
    if rank == 0 and not args.no_e2e:
        e_val, h2d, d2h, e_ok = e2e_steps(run, max(1, min(args.steps, 2)), 1)
        line["e2e"] = {"value": e_val * world, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                       "converged_all": e_ok, "note": "snap_project_host: pinned host buffers, copies inside the timed region"}
    if rank == 0 and world == 1 and not args.no_cpu:
        cores = os.cpu_count() or 1
        workers = min(cores, 16)
        taus = (1, 25, 49) if cfg == 5 else (25,)
        v, dt, desc, used = oracle_sample(cfg, workers if cfg in (4, 5, 6, 7, 8, 9) else max(workers, 16), workers, taus=taus)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": used, "host_cpu_count": cores, "kind": "oracle",
                                "sample": desc, "seconds": dt}
    if rank == 0 and world == 1 and args.others:
        # second line of the same workload: multiplier-free calls (lambda = NULL): no y row, no multiplier sweep, no
        # min-norm correction; its fraction is quoted against ITS OWN algorithmic bytes
        run.lam_free = True
        ms_f, km_f, _ = time_steps(run, args.steps, args.warmup, None)
        ok_f, hm_f, _ = run.check()
        ab_f = run.traffic_model()
        ks_f = sum(sum(k) for k in km_f) * 1e-3
        rf = roofline_of(run, cfg, ks_f, ab_f, args.steps, peak, peak_src)
        rf.pop("traffic", None); rf.pop("traffic_note", None); rf.pop("frac_dram", None); rf.pop("dram_over_alg", None)
        line["lambda_free"] = {"value": run.projections_per_step() * args.steps / (ms_f * 1e-3), "unit": UNIT,
                               "ms_per_step": ms_f / args.steps, "converged_all": ok_f, "max_hinf_last_call": hm_f,
                               "alg_bytes_per_projection": sum(ab_f) / (run.B * run.calls), "roofline": rf,
                               "note": "snap_project(lambda = NULL): u* only, as PCFM's pull-back needs (PAPER.md Eq. 3 L54)"}
        run.lam_free = False
    if rank == 0 and world == 1 and args.others and cfg == 5:
        line["flow_step"] = flow_step_lines(run, args.steps, args.warmup)
        line["float32_mode"] = float32_lines(run, args.steps, args.warmup, peak)
    if rank == 0 and world == 1 and args.others and cfg == 5:
        others = {}
        for c in (1, 2, 3, 4, 6, 7, 8, 9):
            r = GpuRun(S, c, dev)
            ms, km, _ = time_steps(r, 5, 3, None)
            okc, hm, itc = r.check()
            ab = r.traffic_model()
            ks = sum(sum(k) for k in km) * 1e-3
            others[f"cfg{c}"] = {"projections_per_s": r.B * 5 / (ms * 1e-3), "ms_per_call": ms / 5, "converged_all": okc,
                                 "max_hinf": hm, "roofline": roofline_of(r, c, ks, ab, 5, peak, peak_src),
                                 "note": {1: "4 samples x 32 KiB: latency-bound, fits L2", 2: "32 samples, 4 MiB per field: fits L2, latency-bound",
                                          3: "256 samples, 32 MiB per field: L2-borderline",
                                          4: "64 samples, 64 MiB per field; 64 CTAs on 148 SMs: level solves bound by shared-memory latency (DESIGN.md 6.2)",
                                          6: "not a BASELINE.json config: the paper's IC + Mass + Flux(k=5) row set with energy rows at cfg-5 scale",
                                          7: "not a BASELINE.json config: Godunov flux variant",
                                          8: "cfg6's inputs and row set, exact Lagrangian Hessian on the free levels (circulant tridiagonal solves per level)",
                                          9: "the paper's Navier-Stokes row set at its own grid; 25 MiB per field: fits L2, latency-bound"}[c]}
            del r
        line["other_workloads"] = others
    if rank == 0:
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def self_launch(args) -> int:
    """`python bench.py --gpus N` with N > 1 and no torchrun environment: re-exec under torch.distributed.run
    with one rank per GPU (the launch line the driver itself uses)."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg5", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5", "cfg6", "cfg7", "cfg8", "cfg9"])
    ap.add_argument("--impl", default="snap", choices=["snap", "reference"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-others", dest="others", action="store_false")
    ap.add_argument("--traffic", type=float, default=None,
                    help="override: dram bytes per launch of the dominant kernel (default: profiles/traffic.json)")
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"], help="torch.distributed backend (N > 1)")
    ap.add_argument("--selftest-dist", action="store_true",
                    help="exercise only the multi-rank launch + reduction plumbing (no GPU work; use with --backend gloo)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(self_launch(args))
    run_gpu(args)


if __name__ == "__main__":
    main()
