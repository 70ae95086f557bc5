"""bench.py -- node-step updates/s of the full P(t,x) evolution (BASELINE.json's metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..7] [--impl cuda|reference]

One "step" = one pass of the whole hot path over one workload: fk_reset (P = repmat(chi)),
fk_set_coeffs_range (the coefficient slices) and fk_evolve(N -> 0), i.e. Algorithm 1
 start to end: J*N(N+1)/2 node-step updates.

Workload.  BASELINE.json quotes its metric on no particular config, so the headline is the largest
configuration the driver's command (25 or more evolutions) can finish: config 4 (2-D runaway
electrons, 401x201, N=5000, 1.0e12 updates, state + coefficient table = 19 GB in HBM).  Config 5
(3-D, 1.7e12 updates, ~2 minutes per evolution, 81 GB coefficient table streamed through the
slot ring) and the other configs are measured once each in the same run under `per_config`
(DESIGN.md "Measurement"); `--config k` makes any of them the headline.

  value     device-timed (CUDA events on the library's stream), coefficients resident in HBM
  e2e       same metric through the C ABI with HOST buffers: per step the H2D copy of the
            coefficient table and the D2H read-out of all N+1 columns are inside the timing
  roofline  the dominant kernel class, timed live with per-launch CUDA events in one extra pass
            (fk_profile); its algorithmic bytes (16 B per node-step update) against the measured
            HBM copy rate AND its algorithmic flops (counted on the device, fk_work) against the
            fp64 rate measured in-process (fk_peak_fp64); `bound` names the larger time floor
  cpu_baseline  the oracle as it stands (an untuned checker, not a tuned CPU code) on the host
            cores, on a bounded prefix of the workload

N > 1: replicas only (north_star: one GPU, no sharding, no collectives) -- every rank runs the
same workload independently; value = N*U / max-over-ranks time.  (`--multi shard` instead splits
the output-time columns over the ranks with fk_params.shard_*: no exchange, strong scaling.)
--impl reference times the oracle (rank 0 only).
"""
from __future__ import annotations

import argparse
import hashlib
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
SLOPE_FLOPS_PER_DIM = 14       # Eq. 15 per update and dimension
DEFAULT_CONFIG = 4
RING_SLOTS = 32                # coefficient ring for tables that are streamed (config 5)
SM_CLOCK_HZ = 1.965e9          # clocks.max.sm of the B200 (the run's own clock record is in `clocks`)

# DRAM traffic of the dominant kernel from this round's `ncu --set full` captures (profiles/*.md
# name the commands).  An entry counts only while the kernel's source file is byte-identical to
# the one profiled (sha1 below); otherwise `traffic` is null rather than stale.
TRAFFIC = {
    ("cfg4_runaway_2d", "far2d"): {
        "source": "fk_far2d.cu", "source_sha1": "45e1659936146f32bc7e8d238ca631e4ee91c23f",
        "dram_bytes": 455071488, "algorithmic_bytes": 193100000,
        "launch": "step n = 424 of config 4's grid (601 active columns, 20 chunks, about 20.1e3 rows: 17.8e3 far rows "
                  "and the near rows of the lines handed over whole); this path also "
                  "reads the two slope fields: 32 B per update",
        "profile": "profiles/r3_cfg4_cfg5_kernels_ncu_full.md"},
    ("cfg4_runaway_2d", "fused"): {
        "source": "fk_fused2d.cu", "source_sha1": "a69b7c46b8f12346ea4808a2f39802e3470c1529",
        "dram_bytes": 650159104, "algorithmic_bytes": 578100000,
        "launch": "step n = 424 of config 4's grid (601 active columns, 20 chunks, about 60.1e3 near rows on the "
                  "output lines ~95..399; 39 idle lanes in the first chunk)",
        "profile": "profiles/r2_cfg4_kernels_ncu_full.md"},
    ("cfg3_cellular_2d", "fused"): {
        "source": "fk_fused2d.cu", "source_sha1": "a69b7c46b8f12346ea4808a2f39802e3470c1529",
        "dram_bytes": 308636928, "algorithmic_bytes": 311414160,
        "launch": "step n = 424 of config 3's grid (601 active columns, 20 chunks)",
        "profile": "profiles/r2_fused2d_ncu_full.md"},
    ("cfg5_runaway_3d", "rowblock"): {
        "source": "fk_rowblock3d.cu", "source_sha1": "e37193f408aa37f583ca81e12153df066f980be5",
        "dram_bytes": 12413479000, "algorithmic_bytes": 2954133504,
        "launch": "step n = 32 of config 5's grid evolved for 255 steps (224 active columns = 7 FULL chunks, every lane "
                  "busy: 16 B x 824256 updated nodes x 224 columns); this path also reads three slope fields "
                  "(40 B per update) and the factored rows once per group of two chunks",
        "profile": "profiles/r3_cfg4_cfg5_kernels_ncu_full.md"},
}


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def max_over_ranks(x, device=None):
    """MAX over the ranks of the default process group (the job is as slow as its slowest
    rank); identity when torch.distributed is not initialised."""
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


def traffic_for(wl_name, kernel):
    t = TRAFFIC.get((wl_name, kernel))
    if not t:
        return None
    path = os.path.join(ROOT, "paper_2104_14561_b200", "csrc", t["source"])
    try:
        with open(path, "rb") as f:
            if hashlib.sha1(f.read()).hexdigest() != t["source_sha1"]:
                return None
    except OSError:
        return None
    return t


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
            time.sleep(0.2)

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
    sample = (f"{wl.name}: the oracle (untuned checker: one quadrature point at a time, long-double "
              f"sums) on Algorithm 1's prefix N'={n1} of N={wl.N} "
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
def pinned_table(wl, torch):
    """(b, sigma) for all N steps in pinned host memory, [N][d][J] (autonomous: [1][d][J]);
    falls back to pageable memory when the host cannot pin that much."""
    steps = 1 if wl.autonomous else wl.N
    shape = (steps, wl.d, wl.J)
    try:
        hb = torch.empty(shape, dtype=torch.float64, pin_memory=True)
        hs = torch.empty(shape, dtype=torch.float64, pin_memory=True)
        kind = "pinned"
    except RuntimeError:
        hb = torch.empty(shape, dtype=torch.float64)
        hs = torch.empty(shape, dtype=torch.float64)
        kind = "pageable (pinning failed)"
    nb, ns = hb.numpy(), hs.numpy()
    for n in range(steps):
        b, s = wl.coeffs(n)
        nb[n] = b
        ns[n] = s
    return hb, hs, kind


class Runner:
    """One context on one workload; coefficients either resident (full table on the device) or
    streamed through a slot ring (tables that do not fit: config 5)."""

    def __init__(self, B, torch, wl, dev, stream, resident, shard=(0, 1)):
        self.B, self.torch, self.wl, self.dev, self.stream = B, torch, wl, dev, stream
        self.resident = resident
        self.slots = 1 if wl.autonomous else (wl.N if resident else min(wl.N, RING_SLOTS))
        flags = B.FK_FLAG_WEIGHTED_SLOPES if getattr(wl, "slope_rule", 0) else 0
        self.ctx = B.fk_create(wl.x, wl.dt, wl.N, wl.Q, wl.face_kind, wl.face_value,
                               coeff_slots=self.slots, device=dev.index, stream=stream.cuda_stream,
                               flags=flags, shard_index=shard[0], shard_count=shard[1])
        self.hb = self.hs = self.db = self.ds = None
        self.host_kind = None

    def load_tables(self, host=True, device=True):
        if host and self.hb is None:
            self.hb, self.hs, self.host_kind = pinned_table(self.wl, self.torch)
        if device and self.db is None:
            self.db, self.ds = self.hb.to(self.dev), self.hs.to(self.dev)

    def _set(self, b, s):
        B = self.B
        if self.wl.autonomous:
            B.fk_set_coeffs(self.ctx, B.FK_ALL_STEPS, b[0], s[0])
        else:
            B.fk_set_coeffs_range(self.ctx, 0, self.wl.N, b, s)

    def step_device(self):
        self.B.fk_reset(self.ctx)
        self._set(self.db, self.ds)
        self.B.fk_evolve(self.ctx, self.wl.N, 0)

    def step_e2e(self, h_out):
        self.B.fk_reset(self.ctx)
        self._set(self.hb, self.hs)                   # host -> device inside the call
        self.B.fk_evolve(self.ctx, self.wl.N, 0)
        self.B.fk_read(self.ctx, 0, self.wl.N + 1, h_out)   # device -> host, synchronises

    def evolve_streamed(self, n_stop=0):
        """Ring-buffered evolution; only the fk_evolve pieces are timed (the coefficient slices of
        the next piece are generated on the host and uploaded between them).  -> device ms."""
        B, torch, wl = self.B, self.torch, self.wl
        B.fk_reset(self.ctx)
        total = 0.0
        n = wl.N
        while n > n_stop:
            lo = max(n_stop, n - self.slots)
            b, s = wl.coeff_table(lo, n)
            B.fk_set_coeffs_range(self.ctx, lo, n - lo, b, s)
            e0 = torch.cuda.Event(enable_timing=True)
            e1 = torch.cuda.Event(enable_timing=True)
            with torch.cuda.stream(self.stream):
                e0.record(self.stream)
                B.fk_evolve(self.ctx, n, lo)
                e1.record(self.stream)
            e1.synchronize()
            total += e0.elapsed_time(e1)
            n = lo
        return total

    def evolve_streamed_e2e(self, read_batch=64):
        """End to end for a workload whose coefficient table does not fit memory: ONE timed region
        (CUDA events on the library's stream) around the whole ring loop -- every piece's slices are
        generated on the host by a producer thread into two page-locked buffers, uploaded with
        FK_MEM_HOST_PINNED (queued, not waited for: the host goes on generating while the kernels
        run), evolved, and at the end every column is read back to page-locked host memory in batches.
        -> (ms, h2d_bytes, d2h_bytes)."""
        import queue
        import threading
        B, torch, wl = self.B, self.torch, self.wl
        d, J, N = wl.d, wl.J, wl.N
        piece = max(1, self.slots // 2)
        pieces = []
        n = N
        while n > 0:
            pieces.append((max(0, n - piece), n))
            n = pieces[-1][0]
        bufs = [tuple(torch.empty((piece, d, J), dtype=torch.float64).pin_memory() for _ in range(2)) for _ in range(2)]
        h_out = torch.empty((read_batch, J), dtype=torch.float64).pin_memory()
        free = [queue.Queue(), queue.Queue()]         # main -> producer: the event behind the buffer's last upload
        ready = queue.Queue()                         # producer -> main: piece index, or the exception
        for f in free:
            f.put(None)

        def producer():
            try:
                for k, (lo, hi) in enumerate(pieces):
                    ev = free[k % 2].get(timeout=900)
                    if ev is not None:
                        ev.synchronize()              # the copies out of this buffer have been done
                    b, s_ = wl.coeff_table(lo, hi)
                    bufs[k % 2][0][:hi - lo].copy_(torch.from_numpy(b))
                    bufs[k % 2][1][:hi - lo].copy_(torch.from_numpy(s_))
                    ready.put(k)
            except BaseException as exc:              # noqa: BLE001 -- handed to the main thread
                ready.put(exc)

        th = threading.Thread(target=producer, daemon=True)
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        h2d = 0
        torch.cuda.synchronize(self.dev)
        with torch.cuda.stream(self.stream):
            e0.record(self.stream)
            th.start()
            B.fk_reset(self.ctx)
            for k, (lo, hi) in enumerate(pieces):
                got = ready.get(timeout=900)
                if isinstance(got, BaseException):
                    raise got
                cnt = hi - lo
                hb, hs = bufs[k % 2]
                B.fk_set_coeffs_range(self.ctx, lo, cnt, hb[:cnt], hs[:cnt], pinned_async=True)
                ev = torch.cuda.Event()
                ev.record(self.stream)
                free[k % 2].put(ev)
                B.fk_evolve(self.ctx, hi, lo)
                h2d += 2 * cnt * d * J * 8
            for m0 in range(0, N + 1, read_batch):    # device -> host, synchronises per batch
                m1 = min(N + 1, m0 + read_batch)
                B.fk_read(self.ctx, m0, m1, h_out[:m1 - m0])
            e1.record(self.stream)
        e1.synchronize()
        th.join(timeout=60)
        return e0.elapsed_time(e1), h2d, (N + 1) * J * 8

    def close(self):
        self.B.fk_destroy(self.ctx)
        self.db = self.ds = self.hb = self.hs = None


def roofline_of(B, runner, prof, prof_step_ms, upd, work, peak_hbm, peak_src, fp64_tf, fp64_ms, fp64_iters, sm_count):
    """The dominant kernel class against both roofs."""
    wl = runner.wl
    d = wl.d
    classes = {k: v for k, v in prof.items() if k != "assemble" and v[1] > 0}
    dom = max(classes, key=lambda k: classes[k][0])
    dom_ms, dom_launches = classes[dom]
    u_dom = upd[dom]
    if dom == "fused":
        flops = 2.0 * work["fma_near"] + SLOPE_FLOPS_PER_DIM * d * work["updates_near"]
    elif dom == "line1d":                             # 1-D rows are counted as "other" by fk_assemble
        flops = 2.0 * work["fma_other"] + SLOPE_FLOPS_PER_DIM * d * work["updates_other"]
    elif dom == "slopes":
        flops = SLOPE_FLOPS_PER_DIM * d * u_dom
    else:                                             # apply / rowblock / far2d: the rows outside the fused kernel
        flops = 2.0 * work["fma_other"]
    secs = dom_ms * 1e-3
    hbm_gbs = BYTES_PER_UPDATE * u_dom / secs / 1e9
    fp64_tfs = flops / secs / 1e12
    t_hbm = BYTES_PER_UPDATE * u_dom / (peak_hbm * 1e9)
    t_fp64 = flops / (fp64_tf * 1e12)
    alu_bound = t_fp64 > t_hbm
    # the operand roof of a contraction without register reuse: every
    # multiply-add takes one 8-byte u / dP operand per lane through the 128 B/clk L1 / shared-memory
    # data stage = 16 multiply-adds per clock and SM; context for the kernels whose rows share no nodes
    operand = None
    if dom in ("apply", "far2d", "rowblock", "line1d"):
        contraction = 2.0 * work["fma_other"]
        roof = 16.0 * sm_count * SM_CLOCK_HZ
        operand = {"achieved_fma_per_s": contraction / 2.0 / secs, "roof_fma_per_s": roof,
                   "frac": contraction / 2.0 / secs / roof,
                   "note": "1 operand per multiply-add: 16 FMA/clk/SM x SMs x 1.965 GHz (128 B/clk data stage, "
                           "B300_MICROARCH guide); row-blocked paths (banded far rows, 3-D groups) may exceed it"}
    tr = traffic_for(wl.name, dom)
    total_upd = work["updates_near"] + work["updates_other"]
    total_flops = 2.0 * (work["fma_near"] + work["fma_other"]) + SLOPE_FLOPS_PER_DIM * d * total_upd
    return {
        "bound": "alu" if alu_bound else "hbm",
        "kernel": {"fused": "fk_fused2d", "apply": f"fk_apply<{d}>", "rowblock": "fk_rowblock3d", "far2d": "fk_far2d", "line1d": "fk_line1d",
                   "slopes": f"fk_slopes<{d}>"}[dom],
        "achieved": fp64_tfs if alu_bound else hbm_gbs,
        "peak": fp64_tf if alu_bound else peak_hbm,
        "unit": "TFLOP/s" if alu_bound else "GB/s",
        "frac": (fp64_tfs / fp64_tf) if alu_bound else (hbm_gbs / peak_hbm),
        "hbm": {"achieved_gbs": hbm_gbs, "peak_gbs": peak_hbm, "frac": hbm_gbs / peak_hbm,
                "peak_source": peak_src, "bytes_per_update": BYTES_PER_UPDATE},
        "fp64": {"achieved_tflops": fp64_tfs, "peak_tflops": fp64_tf, "frac": fp64_tfs / fp64_tf,
                 "flops_per_update": flops / max(u_dom, 1.0),
                 "peak_source": (f"fk_peak_fp64 in this process: {4 * sm_count} blocks x 512 threads x 8 chains x "
                                 f"{fp64_iters} dependent fma x 2 flops in {fp64_ms:.3f} ms (second launch, CUDA events)")},
        "floor_ms": {"hbm": t_hbm * 1e3, "fp64": t_fp64 * 1e3},
        "operand_roof": operand,
        "traffic": tr["dram_bytes"] if tr else None,
        "traffic_note": (f"ncu dram bytes of the launch {tr['launch']}; algorithmic bytes of that launch: "
                         f"{tr['algorithmic_bytes']}; {tr['profile']}") if tr else
                        "null: no ncu capture of this kernel's current source (profiles/ holds the captures)",
        "units": u_dom, "launches": dom_launches, "avg_launch_ms": dom_ms / max(1, dom_launches),
        "share_of_step": dom_ms / prof_step_ms, "profiled_step_ms": prof_step_ms,
        "class_ms": {k: v[0] for k, v in classes.items()},
        "assemble_note": "fk_assemble runs on the library's side stream under the previous step's kernels and "
                         "is left out of class_ms (its events measure wall time while sharing the SMs)",
        "whole_step": {"updates": total_upd, "flops_per_update": total_flops / max(total_upd, 1.0),
                       "hbm_frac": BYTES_PER_UPDATE * total_upd / (prof_step_ms * 1e-3) / 1e9 / peak_hbm,
                       "fp64_frac": total_flops / (prof_step_ms * 1e-3) / 1e12 / fp64_tf},
    }


def profile_pass(B, torch, runner, streamed):
    """One extra evolution with per-launch events -> (class times, step ms, class updates, work)."""
    B.fk_profile(runner.ctx, True)
    if streamed:
        step_ms = runner.evolve_streamed()
    else:
        pe0 = torch.cuda.Event(enable_timing=True)
        pe1 = torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(runner.stream):
            pe0.record(runner.stream)
            runner.step_device()
            pe1.record(runner.stream)
        pe1.synchronize()
        step_ms = pe0.elapsed_time(pe1)
    prof = B.fk_profile_read(runner.ctx)                 # synchronises the stream
    upd = B.fk_profile_updates(runner.ctx)
    work = B.fk_work(runner.ctx)
    B.fk_profile(runner.ctx, False)
    return prof, step_ms, upd, work


def compact(x, digits=5):
    """Floats rounded to `digits` significant digits, recursively: keeps the per_config block (one
    entry per configuration) short enough that a record which keeps only the tail of the line still
    holds every configuration."""
    if isinstance(x, float):
        return float(f"{x:.{digits}g}")
    if isinstance(x, dict):
        return {k: compact(v, digits) for k, v in x.items()}
    if isinstance(x, (list, tuple)):
        return [compact(v, digits) for v in x]
    return x


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
    shard = (rank, world) if (args.multi == "shard" and world > 1) else (0, 1)
    U = wl.updates
    table_bytes = (1 if wl.autonomous else N) * 2 * d * J * 8
    resident = table_bytes < 40e9               # config 5's 81 GB table goes through the ring

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    peak, peak_src = load_peaks()
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    fp64_iters = 1 << 15
    fp64_tf, fp64_ms = B.fk_peak_fp64(local, stream.cuda_stream, fp64_iters)

    runner = Runner(B, torch, wl, dev, stream, resident, shard)
    e2e = None
    try:
        if resident:
            runner.load_tables()

            def timed(fn, steps):
                e0 = torch.cuda.Event(enable_timing=True)
                e1 = torch.cuda.Event(enable_timing=True)
                barrier()
                l0 = B.fk_launch_count(runner.ctx)
                with torch.cuda.stream(stream):
                    e0.record(stream)
                    for _ in range(steps):
                        fn()
                    e1.record(stream)
                barrier()
                return max_over_ranks(e0.elapsed_time(e1) * 1e-3, dev), B.fk_launch_count(runner.ctx) - l0

            for _ in range(args.warmup):
                runner.step_device()
            sampler = ClockSampler(local)
            if rank == 0:
                sampler.start()
            secs, launches = timed(runner.step_device, args.steps)
            clocks = sampler.stop() if rank == 0 else None
            # end to end through the public API with host buffers
            h_out = torch.empty((N + 1, J), dtype=torch.float64)
            try:
                h_out = h_out.pin_memory()
            except RuntimeError:
                pass
            e2e_steps = max(1, min(args.steps, 3))
            runner.step_e2e(h_out)
            e2e_secs, _ = timed(lambda: runner.step_e2e(h_out), e2e_steps)
            e2e = {"value": whole_job_value(U, e2e_secs / e2e_steps, 1 if shard[1] > 1 else world), "unit": UNIT,
                   "h2d_bytes_per_step": int(runner.hb.numel() * 8 + runner.hs.numel() * 8),
                   "d2h_bytes_per_step": int(h_out.numel() * 8),
                   "ms_per_step": e2e_secs / e2e_steps * 1e3, "host_buffers": runner.host_kind}
            del h_out
        else:
            # streamed workload: every step regenerates and uploads the ring pieces between the
            # timed fk_evolve calls; the e2e leg would need the 81 GB table in host memory
            for _ in range(min(args.warmup, 1)):
                runner.evolve_streamed(n_stop=N - 8)
            sampler = ClockSampler(local)
            if rank == 0:
                sampler.start()
            l0 = B.fk_launch_count(runner.ctx)
            ms = [runner.evolve_streamed() for _ in range(args.steps)]
            launches = B.fk_launch_count(runner.ctx) - l0
            clocks = sampler.stop() if rank == 0 else None
            secs = max_over_ranks(sum(ms) * 1e-3, dev)
            e2e_ms, h2d, d2h = runner.evolve_streamed_e2e()
            e2e_secs = max_over_ranks(e2e_ms * 1e-3, dev)
            e2e = {"value": whole_job_value(U, e2e_secs, 1 if shard[1] > 1 else world), "unit": UNIT,
                   "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h), "ms_per_step": e2e_secs * 1e3,
                   "host_buffers": "pinned ring halves, slices generated on a host producer thread inside the timed region"}
        prof = None
        if rank == 0:
            prof, prof_step_ms, upd, work = profile_pass(B, torch, runner, not resident)
        barrier()
    finally:
        runner.close()
    torch.cuda.empty_cache()

    # one evolution of each other configuration, same process (per_config)
    per_config = {}
    if rank == 0 and not args.no_per_config:
        # BASELINE.json's configs 1-5 in full; the section 8(f) workloads 6 (the paper's periodic cellular
        # flow, in full) and 7 (config 5 on the paper's radial grid with weighted slopes: its first 96
        # steps, i.e. columns 0..96 of the full run -- a full evolution is 3.3e12 updates)
        for idx in (1, 2, 3, 4, 5, 6, 7):
            if idx == args.config:
                continue
            w2 = W.config(idx) if idx != 7 else W.config(7, N=96, dt=W.config(7).dt)
            tb = (1 if w2.autonomous else w2.N) * 2 * w2.d * w2.J * 8
            res2 = tb < 40e9
            r2 = Runner(B, torch, w2, dev, stream, res2)
            try:
                if res2:
                    r2.load_tables(host=True, device=True)
                    r2.step_device()                                  # warm-up
                    torch.cuda.synchronize(dev)
                    e0 = torch.cuda.Event(enable_timing=True)
                    e1 = torch.cuda.Event(enable_timing=True)
                    reps = 3 if w2.updates < 1e11 else 1
                    with torch.cuda.stream(stream):
                        e0.record(stream)
                        for _ in range(reps):
                            r2.step_device()
                        e1.record(stream)
                    e1.synchronize()
                    ms2 = e0.elapsed_time(e1) / reps
                else:
                    r2.evolve_streamed(n_stop=w2.N - 8)               # short warm-up
                    ms2 = r2.evolve_streamed()
                    e2e_ms2, h2d2, d2h2 = r2.evolve_streamed_e2e()
                p2, pms2, u2, wk2 = profile_pass(B, torch, r2, not res2)
                rl2 = roofline_of(B, r2, p2, pms2, u2, wk2, peak, peak_src, fp64_tf, fp64_ms, fp64_iters, sm_count)
                per_config[w2.name] = {
                    "grid": list(w2.n), "N": w2.N, "prefix_of_N": W.config(7).N if idx == 7 else None, "updates": w2.updates, "ms_per_evolution": ms2,
                    "updates_per_s": w2.updates / (ms2 * 1e-3),
                    # "ring": generated on the host and uploaded between the timed fk_evolve pieces
                    "coefficients": "resident" if res2 else f"ring{RING_SLOTS}",
                    "dominant": {k: rl2[k] for k in ("kernel", "bound", "frac", "share_of_step")},
                    "hbm_frac": rl2["hbm"]["frac"], "fp64_frac": rl2["fp64"]["frac"],
                    "whole_step": rl2["whole_step"], "class_ms": rl2["class_ms"]}
                if not res2:                                          # the whole ring loop in one timed region
                    per_config[w2.name]["e2e"] = {
                        "value": w2.updates / (e2e_ms2 * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms2,
                        "h2d_bytes_per_step": int(h2d2), "d2h_bytes_per_step": int(d2h2),
                        "note": "slices generated on a host producer thread, uploaded from pinned memory "
                                "(FK_MEM_HOST_PINNED) inside the timed region; all columns read back"}
            finally:
                r2.close()
            torch.cuda.empty_cache()

    if rank != 0:
        return None
    ms_step = secs / args.steps * 1e3
    value = whole_job_value(U, secs / args.steps, 1 if shard[1] > 1 else world)
    rl = roofline_of(B, runner, prof, prof_step_ms, upd, work, peak, peak_src, fp64_tf, fp64_ms, fp64_iters, sm_count)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
        "scaling": "strong" if shard[1] > 1 else "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "grid": list(wl.n), "N": N, "Q": list(wl.Q), "dt": wl.dt,
                   "updates_per_step": U,
                   "parallelism": ("column shards, no exchange" if shard[1] > 1 else
                                   "replicas only" if world > 1 else "1 gpu"),
                   "coefficients": "resident in HBM" if resident else f"streamed through a ring of {RING_SLOTS} slots",
                   "l2": "inputs larger than L2 (state + coefficient table in HBM)"
                   if (N + 1) * J * 16 > 126e6 else "state fits in L2: HBM roofline not meaningful"},
        "algorithmic_gbs": BYTES_PER_UPDATE * U / (secs / args.steps) / 1e9,
        "roofline": rl,
        "gpu_launches": int(launches),
        "clocks": clocks,
        "per_config": compact(per_config),
    }
    if e2e is not None:
        line["e2e"] = e2e
    else:
        line["e2e"] = {"value": None, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                       "note": "streamed workload: no end-to-end leg (the coefficient table does not fit host memory)"}
    return line


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=DEFAULT_CONFIG, help="BASELINE.json config 1..5 (6, 7: section 8(f) workloads)")
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--multi", default="replicas", choices=["replicas", "shard"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true")
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
