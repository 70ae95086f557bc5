"""bench.py -- node-step updates/s of the full P(t,x) evolution (BASELINE.json's metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl cuda|reference]

One "step" = one pass of the whole hot path over one workload: fk_reset (P = repmat(chi)),
fk_set_coeffs_range (all N coefficient slices) and fk_evolve(N -> 0), i.e. Algorithm 1
 start to end: J*N(N+1)/2 node-step updates.  Default workload: BASELINE.json
config 3 (2-D cellular flow, 257x129, Q=8x8, N=2000) -- the first configuration whose state
leaves L2, so that "HBM GB/s vs peak" means something.

  value     device-timed (CUDA events on the library's stream), coefficients resident in HBM
  e2e       same metric through the C ABI with pinned HOST buffers: per step the H2D copy of
            the coefficient table and the D2H read-out of all N+1 columns are inside the timing
  roofline  the dominant kernel class, timed live with per-launch CUDA events in one extra pass
            (fk_profile), 16 B per node-step update of algorithmic traffic
  cpu_baseline  the oracle as it stands on the host cores, on a bounded prefix of the workload

N > 1: replicas only (north_star: one GPU, no sharding, no collectives) -- every rank runs the
same workload independently; value = N*U / max-over-ranks time.  --impl reference times the
oracle (rank 0 only).
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

from paper_2104_14561_b200 import workloads as W  # noqa: E402  (inputs only)

METRIC = "fp64 node-step updates/s, full P(t,x) evolution (Algorithm 1)"
UNIT = "updates/s"
BYTES_PER_UPDATE = 16          # read P_old + write P_new, fp64


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def max_over_ranks(x, device=None):
    """MAX over the ranks of the default process group (replicas: the job is as slow as its
    slowest rank); identity when torch.distributed is not initialised."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(updates_per_replica, secs_per_step, world):
    """Replicas only: every rank evolves the same workload; the job did world x U updates."""
    return world * updates_per_replica / secs_per_step


def load_traffic(wl_name):
    """DRAM bytes of the dominant kernel from the committed ncu --set full capture (one launch),
    with the algorithmic bytes of that same launch; None if there is no capture for the workload."""
    path = os.path.join(ROOT, "profiles", "r1_traffic_cfg3.json.txt")
    if os.path.exists(path):
        with open(path) as f:
            t = json.load(f)
        if t.get("workload") == wl_name:
            return t
    return None


def coeff_table(wl):
    """(b, sigma) for all N steps as numpy [N][d][J] (autonomous: [1][d][J])."""
    if wl.autonomous:
        b, s = wl.coeffs(0)
        return np.ascontiguousarray(b[None]), np.ascontiguousarray(s[None])
    return wl.coeff_table(0, wl.N)


class ClockSampler:
    """nvidia-smi SM clock / throttle reasons sampled DURING the timed region."""

    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.stop_flag, self.th = index, [], False, None

    def _run(self):
        while not self.stop_flag:
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                      "--format=csv,noheader,nounits"], capture_output=True,
                                     text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([c.strip() for c in out.split(",")])
            except Exception:
                pass
            time.sleep(0.1)

    def start(self):
        self.th = threading.Thread(target=self._run, daemon=True)
        self.th.start()

    def stop(self):
        self.stop_flag = True
        if self.th:
            self.th.join(timeout=10)
        sm, mx, reasons = [], 0.0, set()
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = max(mx, float(r[1]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(self.NAMES, r[2:]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx or None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------------------
# the oracle leg (cpu_baseline, and --impl reference): oracle/ as it stands, never tuned
# ------------------------------------------------------------------------------------------
def oracle_sample(wl, budget_s=15.0):
    """Time the oracle's Algorithm 1 on a prefix N' of the workload (columns 0..N' of the full
    run are exactly this prefix problem).  -> (updates/s, cores, sample text, seconds)."""
    from oracle import fk_oracle
    orc = fk_oracle.Oracle(wl)
    cores = fk_oracle.num_threads()
    n0 = min(wl.N, max(4, 2 * cores))          # calibration: enough columns for every thread
    t0 = time.perf_counter()
    orc.algorithm1(n0)
    t_cal = time.perf_counter() - t0
    apps0 = n0 * (n0 + 1) // 2
    per_app = t_cal / apps0
    apps = max(apps0, int(budget_s / per_app))
    n1 = min(wl.N, int((np.sqrt(8.0 * apps + 1.0) - 1.0) / 2.0))
    if n1 <= n0:
        n1, secs = n0, t_cal
    else:
        t0 = time.perf_counter()
        orc.algorithm1(n1)
        secs = time.perf_counter() - t0
    upd = wl.J * n1 * (n1 + 1) // 2
    sample = (f"{wl.name}: Algorithm 1 on the prefix N'={n1} of N={wl.N} "
              f"({n1 * (n1 + 1) // 2} column applications, {upd:.3e} updates, {secs:.1f} s)")
    return upd / secs, cores, sample, secs


def run_reference(args, wl, rank):
    if rank != 0:
        return None
    vals = []
    info = None
    for i in range(args.warmup + args.steps):
        v, cores, sample, secs = oracle_sample(wl, budget_s=args.ref_budget)
        if i >= args.warmup:
            vals.append((v, secs))
        info = (cores, sample)
    value = float(np.mean([v for v, _ in vals]))
    ms = float(np.mean([s for _, s in vals])) * 1e3
    return {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "grid": list(wl.n), "N": wl.N, "Q": list(wl.Q),
                   "note": "each step = a bounded prefix sample of the workload on the host cores"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": info[0], "kind": "oracle",
                         "sample": info[1]},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }


# ------------------------------------------------------------------------------------------
# the CUDA arm
# ------------------------------------------------------------------------------------------
def run_cuda(args, wl, rank, world):
    import torch
    import torch.distributed as dist
    from paper_2104_14561_b200 import binding as B

    B.lib()                                     # raises if the CUDA library is missing
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    stream = torch.cuda.Stream(device=dev)
    N, J, d = wl.N, wl.J, wl.d
    U = wl.updates

    b_np, s_np = coeff_table(wl)
    steps_loaded = b_np.shape[0]
    hb = torch.from_numpy(b_np).pin_memory()
    hs = torch.from_numpy(s_np).pin_memory()
    db = hb.to(dev)
    ds = hs.to(dev)
    h_out = torch.empty((N + 1, J), dtype=torch.float64).pin_memory()
    slots = 1 if wl.autonomous else N
    ctx = B.fk_create(wl.x, wl.dt, N, wl.Q, wl.face_kind, wl.face_value, coeff_slots=slots,
                      device=local, stream=stream.cuda_stream)

    def set_coeffs(b, s):
        if wl.autonomous:
            B.fk_set_coeffs(ctx, B.FK_ALL_STEPS, b[0], s[0])
        else:
            B.fk_set_coeffs_range(ctx, 0, steps_loaded, b, s)

    def step_device():
        B.fk_reset(ctx)
        set_coeffs(db, ds)
        B.fk_evolve(ctx, N, 0)

    def step_e2e():
        B.fk_reset(ctx)
        set_coeffs(hb, hs)                      # pinned host -> device inside the call
        B.fk_evolve(ctx, N, 0)
        B.fk_read(ctx, 0, N + 1, h_out)         # device -> pinned host, synchronises

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    def timed(fn, steps):
        """-> (seconds for `steps` calls by CUDA events on the library's stream, launches)."""
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        barrier()
        l0 = B.fk_launch_count(ctx)
        with torch.cuda.stream(stream):
            e0.record(stream)
            for _ in range(steps):
                fn()
            e1.record(stream)
        barrier()
        secs = max_over_ranks(e0.elapsed_time(e1) * 1e-3, dev)
        return secs, B.fk_launch_count(ctx) - l0

    try:
        for _ in range(args.warmup):
            step_device()
        sampler = ClockSampler(local)
        if rank == 0:
            sampler.start()
        secs, launches = timed(step_device, args.steps)
        clocks = sampler.stop() if rank == 0 else None

        # end to end through the public API with host buffers
        step_e2e()
        e2e_secs, _ = timed(step_e2e, max(1, min(args.steps, 3)))
        e2e_steps = max(1, min(args.steps, 3))

        # per-class kernel time, one extra pass with per-launch events (not the timed region)
        prof = None
        if rank == 0:
            B.fk_profile(ctx, True)
            pe0 = torch.cuda.Event(enable_timing=True)
            pe1 = torch.cuda.Event(enable_timing=True)
            with torch.cuda.stream(stream):
                pe0.record(stream)
                step_device()
                pe1.record(stream)
            prof = B.fk_profile_read(ctx)                   # synchronises the stream
            prof_step_ms = pe0.elapsed_time(pe1)
            B.fk_profile(ctx, False)
            B.fk_reset(ctx)
        barrier()
    finally:
        B.fk_destroy(ctx)

    if rank != 0:
        return None
    peak, peak_src = load_peaks()
    ms_step = secs / args.steps * 1e3
    value = whole_job_value(U, secs / args.steps, world)
    # fk_assemble runs on the library's side stream, overlapped with the previous step's
    # kernels, so the classes do not add up to the step: shares are taken against the step time
    dom = max(prof, key=lambda k: prof[k][0])
    dom_ms, dom_launches = prof[dom]
    achieved = BYTES_PER_UPDATE * U / (dom_ms * 1e-3) / 1e9
    tr = load_traffic(wl.name)
    h2d = int(hb.numel() * 8 + hs.numel() * 8)
    d2h = int(h_out.numel() * 8)
    return {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "grid": list(wl.n), "N": N, "Q": list(wl.Q), "dt": wl.dt,
                   "updates_per_step": U, "parallelism": "replicas only" if world > 1 else "1 gpu",
                   "l2": "inputs larger than L2 (state + coefficient table in HBM)"
                   if (N + 1) * J * 16 > 126e6 else "state fits in L2: HBM roofline not meaningful"},
        "algorithmic_gbs": BYTES_PER_UPDATE * U / (secs / args.steps) / 1e9,
        "roofline": {"bound": "hbm", "kernel": f"fk_{dom}", "achieved": achieved, "peak": peak,
                     "unit": "GB/s", "frac": achieved / peak,
                     "traffic": tr["dram_bytes"] if tr else None,
                     "traffic_note": (f"ncu dram bytes of the launch {tr['launch']}; algorithmic bytes "
                                      f"of that launch: {tr['algorithmic_bytes']}") if tr else None,
                     "peak_source": peak_src, "launches": dom_launches,
                     "avg_launch_ms": dom_ms / max(1, dom_launches),
                     "share_of_step": dom_ms / prof_step_ms, "profiled_step_ms": prof_step_ms,
                     "class_ms": {k: v[0] for k, v in prof.items()}},
        "e2e": {"value": whole_job_value(U, e2e_secs / e2e_steps, world), "unit": UNIT,
                "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e2e_secs / e2e_steps * 1e3},
        "gpu_launches": int(launches),
        "clocks": clocks,
    }


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config 1..5")
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-budget", type=float, default=15.0, help="seconds of oracle work")
    ap.add_argument("--ref-budget", type=float, default=8.0, help="seconds per reference step")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "cuda" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    wl = W.config(args.config)

    if args.impl == "reference":
        line = run_reference(args, wl, rank)
        if line is not None:
            print(json.dumps(line), flush=True)
        return

    if world > 1:
        import torch
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
        dist.init_process_group("nccl")
    try:
        line = run_cuda(args, wl, rank, world)
        if rank == 0:
            if not args.no_cpu_baseline:
                v, cores, sample, _ = oracle_sample(wl, budget_s=args.cpu_budget)
                line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores,
                                        "kind": "oracle", "sample": sample}
            print(json.dumps(line), flush=True)
    finally:
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
            dist.destroy_process_group()


if __name__ == "__main__":
    main()
