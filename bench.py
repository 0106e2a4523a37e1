#!/usr/bin/env python
"""bench.py -- regular-force throughput (G pair-interactions/s: acc + jerk + neighbour list in one pass).

One "step" = one pass of the whole hot path over one synthetic workload: nb_set_j (GPUNB_SEND),
nb_predict_j (S1, all N particles) and nb_regular_force (S2-S5, N_i x N pairs).  Default workload:
BASELINE.json config 5 (N = N_i = 1048576 equal-mass Plummer, k ~ 100, cap 512), the largest single-GPU
configuration and the one SURVEY.md 8(d) names as the headline row.  Inputs are seeded and synthetic
(paper_1205_1222_b200/inputs.py); r_s is calibrated on the unpredicted positions.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--n-i M] [--impl reference]

N > 1 (torchrun): independent replicas, one per GPU, no collective on the data path ("replicas only").
--impl reference times the fp64 CPU oracle (oracle/, test infrastructure) on a bounded row sample.
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

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

FLOPS_PER_PAIR = 60.0  # convention of BASELINE.json ("e.g. 60 for force+jerk"), SURVEY.md R13
# FP32-pipe work the force kernel actually issues: 25 packed f32x2 instructions per TWO pairs on the common (far)
# path = 25 of the SM's 128 FP32 lane-slots per pair.
LANE_SLOTS_PER_PAIR = 25.0
# dram__bytes_read.sum + dram__bytes_write.sum of ONE force_kernel launch of the default workload, from the
# committed capture profiles/r2_force_kernel_c5_ncu_full.md (ncu --set full); None for other workloads.
FORCE_DRAM_BYTES_C5 = 1450.77e6 + 945.16e6
# algorithmic bytes of the predictor per particle on the regular-force path: 112 B of fp64 state read, 40 B of
# pair-interleaved record written (the 48 B particle-major copy is written only for gathering consumers)
PRED_BYTES_PER_J = 152
# dram__bytes_read.sum + dram__bytes_write.sum of one predict_kernel launch of the default workload (ncu --set full,
# profiles/r2_force_kernel_c5_ncu_full.md): 117.45 MB read + 16.15 MB written -- less than the 159 MB the kernel moves,
# because most of the 42 MB of records it writes are still in the 126 MB L2 when the capture ends
PRED_DRAM_BYTES_C5 = 117.45e6 + 16.15e6
METRIC = "regular-force Ginteractions/s (acc+jerk+nbr list)"
UNIT = "Gpairs/s"


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), src="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, src="fallback")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        sm, mx, pw, reasons = [], [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


def max_over_ranks(seconds: float, dist, device) -> float:
    """Replicas only: every rank runs the same workload on its own GPU, no data-path
    collective.  The job's time is the slowest rank's; this MAX all-reduce is the only communication."""
    import torch
    t = torch.tensor([seconds], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(pairs_per_rank_step: int, steps: int, world: int, t_max_seconds: float) -> float:
    """G pairs/s of the whole job: all ranks' pairs over the slowest rank's time."""
    return world * pairs_per_rank_step * steps / t_max_seconds / 1e9


def shard_job(wl, rank: int, world: int, mode: str):
    """What one rank runs and how the job is counted.  mode "none": every rank runs the whole workload (N independent
    replicas: the job is `world` times the workload's pairs).  mode "rows": ONE job, its rows split over
    the ranks on CTA boundaries, no data-path collective (strong scaling: the job is the workload's pairs once).
    Returns (this rank's workload, pairs of ONE replica or of the whole job, replicas, this rank's rows or None)."""
    if mode != "rows":
        return wl, wl.pairs, world, None
    import dataclasses
    from paper_1205_1222_b200 import sharding
    lo, hi = sharding.row_shard(wl.n_i, rank, world)
    local = dataclasses.replace(wl, i_idx=np.ascontiguousarray(wl.i_idx[lo:hi]), r_s=np.ascontiguousarray(wl.r_s[lo:hi]))
    return local, wl.pairs, 1, (lo, hi)


def build_workload(config: int, n_i: int | None):
    from paper_1205_1222_b200 import inputs
    wl = inputs.make_workload(config, n_i=n_i)
    return wl


def cpu_description() -> dict:
    """CPU model, logical CPUs, physical cores and whether SMT siblings are counted."""
    model = "unknown"
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    logical = os.cpu_count() or 0
    physical = None
    try:
        import psutil
        physical = psutil.cpu_count(logical=False)
    except Exception:
        pass
    try:
        affinity = len(os.sched_getaffinity(0))
    except Exception:
        affinity = logical
    smt = None if not physical else (logical > physical)
    return {"cpu_model": model, "logical_cpus": logical, "physical_cores": physical, "usable_cpus": affinity,
            "smt": ("on: OpenMP threads land on SMT siblings too" if smt else "off or not visible") if smt is not None
                   else "unknown"}


def cpu_baseline(wl, target_seconds: float = 12.0, steps: int = 1, min_rows: int = 0, single_thread: bool = True):
    """The oracle as it stands, on this host's cores, on a bounded sample of rows of the same workload (the first
    `rows` active rows against all j).  Returns (report, seconds per pass, rows, oracle results of those rows): the
    results double as the reference of the in-run parity check, so the oracle runs once."""
    from oracle import oracle
    s = wl.state
    xp, vp = oracle.predict_state(s)
    cores = oracle.num_threads()
    # size the sample: probe with 32 rows per thread (the oracle hands out rows 16 at a time), grow the probe until it
    # runs for a quarter of a second, then take the rows that make target_seconds of work
    rows = min(wl.n_i, 32 * cores)
    while True:
        t0 = time.perf_counter()
        oracle.regular_force(xp, vp, s.m, wl.i_idx[:rows], wl.r_s[:rows], list_stride=2 * wl.cap)
        dt = time.perf_counter() - t0
        if dt >= 0.25 or rows >= wl.n_i or dt >= target_seconds / 4:
            break
        rows = min(wl.n_i, rows * 4)
    rate = rows * s.n / dt
    rows = int(min(wl.n_i, max(min_rows, rate * target_seconds / s.n)))
    rows = max(cores, rows // cores * cores)
    rows = min(rows, wl.n_i)
    times, res = [], None
    for _ in range(steps):
        t0 = time.perf_counter()
        res = oracle.regular_force(xp, vp, s.m, wl.i_idx[:rows], wl.r_s[:rows], list_stride=2 * wl.cap)
        times.append(time.perf_counter() - t0)
    dt = float(np.mean(times))
    rep = dict(value=rows * s.n / dt / 1e9, unit=UNIT, cores=cores, kind="oracle",
               sample=f"first {rows} active rows x all {s.n} j (fp64, OpenMP, gcc -O2), {dt:.2f} s per pass")
    rep.update(cpu_description())
    if single_thread:  # one thread, fewer rows (about a second of work)
        r1 = int(max(4, min(rows, rate / max(cores, 1) * 1.5 / s.n)))
        oracle.set_num_threads(1)
        t0 = time.perf_counter()
        oracle.regular_force(xp, vp, s.m, wl.i_idx[:r1], wl.r_s[:r1], list_stride=2 * wl.cap)
        t1 = time.perf_counter() - t0
        oracle.set_num_threads(cores)
        rep["single_thread"] = {"value": r1 * s.n / t1 / 1e9, "unit": UNIT, "sample": f"first {r1} rows, {t1:.2f} s"}
    return rep, dt, rows, (res, xp, vp)


def parity_in_run(wl, out, rows, oracle_results) -> dict:
    """parity checked in the same run, on the outputs of the last timed repetition, against the oracle
    results the cpu_baseline leg has just computed for the first `rows` rows (north_star's tolerances, tests/parity.py)."""
    tests_dir = os.path.join(ROOT, "tests")
    if tests_dir not in sys.path:
        sys.path.insert(0, tests_dir)
    import parity
    from oracle import oracle
    (acc_o, jerk_o, cnt_o, lists_o), xp, vp = oracle_results
    gpu = {k: v[:rows].cpu().numpy() if k != "n_overflow" else v.cpu().numpy() for k, v in out.items()}
    s = wl.state
    try:
        rep = parity.compare(oracle, xp, vp, s.m, wl.i_idx[:rows], wl.r_s[:rows], wl.cap, gpu,
                             precomputed=(acc_o, jerk_o, cnt_o, lists_o))
        return {"ok": True, "rows": rep["rows"], "max_acc": rep["max_acc_err"], "max_jerk": rep["max_jerk_err"],
                "band_pairs": rep["band_pairs"], "overflow_rows": rep["overflow_rows"],
                "tolerance": {"acc": parity.TOL_ACC, "jerk": parity.TOL_JERK, "band": parity.BAND}}
    except AssertionError as e:
        return {"ok": False, "rows": int(rows), "error": str(e)[:300]}


def run_reference(args):
    """--impl reference: the oracle (fp64 CPU) on a bounded sample, same metric/config keys."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    wl = build_workload(args.config, args.n_i)
    base, _, rows, _ = cpu_baseline(wl, target_seconds=4.0, steps=1, single_thread=False)  # sizes the sample
    from oracle import oracle
    s = wl.state
    xp, vp = oracle.predict_state(s)
    for _ in range(args.warmup):
        oracle.regular_force(xp, vp, s.m, wl.i_idx[:rows], wl.r_s[:rows], list_stride=2 * wl.cap)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        xp, vp = oracle.predict_state(s)
        oracle.regular_force(xp, vp, s.m, wl.i_idx[:rows], wl.r_s[:rows], list_stride=2 * wl.cap)
    dt = (time.perf_counter() - t0) / args.steps
    val = rows * s.n / dt / 1e9
    cb = dict(value=val, unit=UNIT, cores=base["cores"], kind="oracle",
              sample=f"each step: predictor on all {s.n} + first {rows} active rows x all j")
    cb.update(cpu_description())
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(wl, args.config), "cpu_baseline": cb,
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))
    return 0


def workload_config(wl, config):
    return {"workload": f"BASELINE.json configs[{config - 1}]: N={wl.state.n} Plummer, N_i={wl.n_i}, "
                        f"k~{wl.k}, nbr cap {wl.cap}", "n": wl.state.n, "n_i": wl.n_i, "nbr_cap": wl.cap,
            "pairs_per_step": wl.pairs, "flops_per_pair_convention": FLOPS_PER_PAIR,
            "r_s_calibrated_on": wl.rs_positions,
            "l2": "a 256 MiB device fill (> the 126 MB L2) flushes L2 before every timed step, outside the per-step "
                  "events (--sweep rows: back-to-back calls, no flush)"}


def run_sweep(args):
    """SURVEY 8(d) protocol for config 3: one row per active-block size 32 ... 65536 (us per call and Gpairs/s),
    for nb_regular_force alone and for the fused call (predictor + force).  Prints one JSON line."""
    import torch
    from paper_1205_1222_b200 import binding, inputs

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the regular-force path has no CPU fallback)")
    full = inputs.make_workload(3)
    s = full.state
    ctx = binding.Context(s.n, full.n_i, full.cap)
    state_dev = ctx.set_state(s)
    dev = ctx.workspace.device
    rows = []
    blocks = inputs.CONFIG3_BLOCKS
    if args.sweep_large:       # the same sweep on the N = 2^20 state of config 5 (predict-all costs 38 us there)
        full = inputs.make_workload(5)
        s = full.state
        ctx.close()
        ctx = binding.Context(s.n, full.n_i, full.cap)
        state_dev = ctx.set_state(s)
        blocks = [b for b in inputs.CONFIG3_BLOCKS if b <= 16384]
    for n_i in blocks:
        i_idx = torch.from_numpy(full.i_idx[:n_i].copy()).to(dev)
        r_s = torch.from_numpy(full.r_s[:n_i].copy()).to(dev)
        out = ctx.alloc_outputs(n_i)
        ctx.nb_predict_j(s.t)
        for _ in range(3):
            ctx.nb_regular_force(i_idx, r_s, s.t, out=out)
        reps = 20 if n_i >= 8192 else 200
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
        torch.cuda.synchronize()
        ev[0].record()
        for _ in range(reps):
            ctx.nb_regular_force(i_idx, r_s, s.t, out=out)
        ev[1].record()
        torch.cuda.synchronize()
        ev[2].record()
        for _ in range(reps):
            ctx.nb_set_j(*state_dev)                       # invalidates the prediction: the next call is fused
            ctx.nb_regular_force(i_idx, r_s, s.t, out=out)
        ev[3].record()
        torch.cuda.synchronize()
        us = ev[0].elapsed_time(ev[1]) / reps * 1e3
        us_fused = ev[2].elapsed_time(ev[3]) / reps * 1e3
        # the same fused step (predictor + force + gather) captured once in a CUDA graph and replayed: the calls only
        # enqueue kernels, so the enqueue cost of Python/ctypes and of three launches drops out
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            ctx.nb_predict_j(s.t)
            ctx.nb_regular_force(i_idx, r_s, s.t, out=out)
        graph.replay()
        gv = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        torch.cuda.synchronize()
        gv[0].record()
        for _ in range(reps):
            graph.replay()
        gv[1].record()
        torch.cuda.synchronize()
        us_graph = gv[0].elapsed_time(gv[1]) / reps * 1e3
        del graph
        info = ctx.nb_last_launch_info()
        # irregular force of the same block over the lists just made: predict-all + gather (PRED_ALL) against the
        # prediction fused into the gather (PRED_ACT), each with a fresh prediction per call
        irr = None
        iv = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
        for _ in range(3):
            irr = ctx.nb_irregular_force(i_idx, out["nbr_count"], out["nbr_list"], s.t, out=irr)
            ctx.nb_irregular_force_act(i_idx, out["nbr_count"], out["nbr_list"], s.t, out=irr)
        torch.cuda.synchronize()
        iv[0].record()
        ctx.nb_set_option("irr_pred", 1)
        for _ in range(reps):
            ctx.nb_set_j(*state_dev)
            ctx.nb_irregular_force(i_idx, out["nbr_count"], out["nbr_list"], s.t, out=irr)
        ctx.nb_set_option("irr_pred", 0)
        iv[1].record()
        torch.cuda.synchronize()
        iv[2].record()
        for _ in range(reps):
            ctx.nb_set_j(*state_dev)
            ctx.nb_irregular_force_act(i_idx, out["nbr_count"], out["nbr_list"], s.t, out=irr)
        iv[3].record()
        torch.cuda.synchronize()
        rows.append({"n_i": n_i, "us_per_call": us, "gpairs": n_i * s.n / us / 1e3, "us_fused": us_fused, "us_fused_graph": us_graph,
                     "rows_per_cta": info["rows_per_cta"], "j_chunks": info["j_chunks"], "ctas": info["ctas"],
                     "us_irr_pred_all": iv[0].elapsed_time(iv[1]) / reps * 1e3,
                     "us_irr_pred_act": iv[2].elapsed_time(iv[3]) / reps * 1e3})
    print(json.dumps({"metric": METRIC, "unit": UNIT, "config": {"workload": "BASELINE.json configs[2] block sweep",
                                                                 "n": s.n, "timing": "back-to-back calls between two events"},
                      "sweep": rows}))
    return 0


class Bench:
    """One workload resident on one GPU: context, device inputs, outputs, and the timed step."""

    def __init__(self, wl, local: int):
        import torch
        from paper_1205_1222_b200 import binding
        self.torch, self.wl, self.s = torch, wl, wl.state
        self.dev = torch.device(f"cuda:{local}")
        self.ctx = binding.Context(self.s.n, wl.n_i, wl.cap, device=local)
        self.state_dev = self.ctx.set_state(self.s)
        self.i_idx = torch.from_numpy(wl.i_idx).to(self.dev)
        self.r_s = torch.from_numpy(wl.r_s).to(self.dev)
        self.out = self.ctx.alloc_outputs(wl.n_i)

    def step(self, ev=None):
        """One pass of the whole hot path: nb_set_j -> nb_predict_j (S1) -> nb_regular_force (S2-S6 + fix-up)."""
        self.ctx.nb_set_j(*self.state_dev)     # GPUNB_SEND: new block-step, prediction invalid
        if ev: ev[0].record()
        self.ctx.nb_predict_j(self.s.t)        # S1
        if ev: ev[1].record()
        self.ctx.nb_regular_force(self.i_idx, self.r_s, self.s.t, out=self.out)  # prediction already at t
        if ev: ev[2].record()

    def timed(self, steps: int, warmup: int, flush, dist=None):
        """W warm-up steps, then K steps, each bracketed by CUDA events on the launching stream; the L2 flush between
        steps sits outside the events.  Returns per-step seconds (step, predictor, force) and the launch info."""
        torch = self.torch
        for _ in range(max(warmup, 3)):
            self.step()
        torch.cuda.synchronize()
        info = self.ctx.nb_last_launch_info()
        evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(steps)]
        if dist: dist.barrier()
        torch.cuda.synchronize()
        for k in range(steps):
            flush.fill_(k & 0xff)              # L2 flush between timed iterations (outside the per-step events)
            self.step(evs[k])
        torch.cuda.synchronize()
        if dist: dist.barrier()
        t_step = np.array([e[0].elapsed_time(e[2]) for e in evs]) / 1e3
        t_pred = np.array([e[0].elapsed_time(e[1]) for e in evs]) / 1e3
        t_force = np.array([e[1].elapsed_time(e[2]) for e in evs]) / 1e3
        info["fixup_rows"] = self.ctx.nb_fixup_stats()["last"]
        return t_step, t_pred, t_force, info

    def close(self):
        self.ctx.close()


def fp32_peak_tflops(torch, local, peaks):
    nsm = torch.cuda.get_device_properties(local).multi_processor_count
    return nsm, nsm * 128 * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12


def run_also(config: int, local: int, flush, peaks, steps: int) -> dict:
    """The other configs of BASELINE.json beside the headline: the same step, the same event protocol, clocks sampled
    during the timed region, and parity of the last timed repetition against the oracle on >= 1024 seeded rows."""
    import torch
    wl = build_workload(config, None)
    b = Bench(wl, local)
    sampler = ClockSampler(local)
    sampler.start()
    t_step, t_pred, t_force, info = b.timed(steps, 3, flush)
    clocks = sampler.stop()
    nsm, peak_tf = fp32_peak_tflops(torch, local, peaks)
    cb, _, rows, ores = cpu_baseline(wl, target_seconds=1.0, min_rows=min(wl.n_i, 1024), single_thread=False)
    par = parity_in_run(wl, b.out, rows, ores)
    med = float(np.median(t_step))
    res = {"config": config, "workload": f"N={wl.state.n}, N_i={wl.n_i}, k~{wl.k}, cap {wl.cap}",
           "value": wl.pairs / float(np.mean(t_step)) / 1e9, "unit": UNIT,
           "value_median": wl.pairs / med / 1e9, "value_best": wl.pairs / float(t_step.min()) / 1e9,
           "us_per_step": float(np.mean(t_step)) * 1e6, "us_force_call": float(np.mean(t_force)) * 1e6,
           "us_predictor": float(np.mean(t_pred)) * 1e6, "steps": steps,
           "frac": wl.pairs * FLOPS_PER_PAIR / float(np.mean(t_force)) / 1e12 / peak_tf,
           "frac_whole_step": wl.pairs * FLOPS_PER_PAIR / float(np.mean(t_step)) / 1e12 / peak_tf,
           "launch": info, "clocks": clocks, "parity": par,
           "cpu_baseline": {"value": cb["value"], "unit": UNIT, "cores": cb["cores"], "sample": cb["sample"]}}
    b.close()
    return res


def run_gpu_arm(args):
    import torch

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the regular-force path has no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    dev = torch.device(f"cuda:{local}")
    peaks = _peaks()
    wl = build_workload(args.config, args.n_i)  # every rank: the same seeded workload (independent replicas)
    wl, job_pairs, job_replicas, shard_rows = shard_job(wl, rank, world, args.shard)
    s = wl.state
    b = Bench(wl, local)
    ctx, i_idx, r_s, out, state_dev = b.ctx, b.i_idx, b.r_s, b.out, b.state_dev
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ts, tp, tf, info = b.timed(args.steps, args.warmup, flush, dist)
    clocks = sampler.stop() if rank == 0 else None
    t_step = float(ts.sum())                                            # s, all K steps, device time
    t_pred, t_force = float(tp.mean()), float(tf.mean())
    t_max = max_over_ranks(t_step, dist, dev)
    value = whole_job_rate(job_pairs, args.steps, job_replicas, t_max)
    n_over = int(out["n_overflow"].item())
    mean_cnt = float(out["nbr_count"].double().mean().item())
    # the predictor alone: ten launches back to back between two events (one launch inside the step is 25 us of kernel
    # behind ~15 us of event-to-kernel latency, which says nothing about the kernel).  State + records = 159 MB > L2.
    # Replayed from a CUDA graph, so that the host's enqueue rate (two ctypes calls per launch) is not what is timed.
    pgraph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(pgraph):
        for _ in range(10):
            ctx.nb_predict_j(s.t)
    pgraph.replay()
    pe = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    flush.fill_(1)
    torch.cuda.synchronize()
    pe[0].record()
    pgraph.replay()
    pe[1].record()
    torch.cuda.synchronize()
    t_pred_b2b = pe[0].elapsed_time(pe[1]) / 10 / 1e3
    del pgraph
    ctx.nb_set_j(*state_dev)

    # ---- the step on the other side of the neighbour list: irregular force eq. (7), (8) over the
    # lists the last step produced.  Reported beside the headline, not part of it.
    irr = None
    if not args.no_irregular:
        irr_out = None
        for _ in range(3):
            irr_out = ctx.nb_irregular_force(i_idx, out["nbr_count"], out["nbr_list"], s.t, out=irr_out)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        torch.cuda.synchronize()
        ev[0].record()
        for _ in range(5):
            ctx.nb_irregular_force(i_idx, out["nbr_count"], out["nbr_list"], s.t, out=irr_out)
        ev[1].record()
        torch.cuda.synchronize()
        t_irr = ev[0].elapsed_time(ev[1]) / 5 / 1e3
        irr_pairs = int(torch.clamp(out["nbr_count"], max=wl.cap).sum().item())
        rec_bytes = irr_pairs * 48
        irr = {"kernel": "irregular_kernel", "pairs": irr_pairs, "ms": t_irr * 1e3,
               "value": irr_pairs / t_irr / 1e9, "unit": UNIT, "bound": "l2-gather",
               "gathered_gb_per_s": rec_bytes / t_irr / 1e9,
               "hbm_frac_if_all_gathers_missed_l2": rec_bytes / t_irr / 1e9 / peaks["hbm_gbs"],
               "note": "eq. (7), (8) over the neighbour lists of the last step; one 48 B particle-major record gathered per pair "
                       "(L2-resident at this N); bound by the L1/TEX sector rate for scattered accesses (profiles/): the "
                       "fractions of the HBM and L2 peaks the kernel reaches are in profiles/r2_irregular_kernel_ncu_full.md"}

    # ---- step (vii) and eq. (1): the regular corrector on the lists of two regular-force calls
    # (radii of the second scaled by a seeded factor in [0.9, 1.1]).  Reported beside the headline, not part of it.
    cor = None
    if not args.no_irregular:
        rng = np.random.default_rng(12345)
        fac = torch.from_numpy(rng.uniform(0.9, 1.1, size=wl.n_i)).to(dev)
        old = ctx.nb_regular_force(i_idx, r_s * fac, s.t)
        f64 = dict(dtype=torch.float64, device=dev)
        dt_r = torch.from_numpy(2.0 ** -rng.integers(3, 9, size=wl.n_i).astype(np.float64)).to(dev)
        fr0, frd0 = torch.randn((wl.n_i, 3), **f64), torch.randn((wl.n_i, 3), **f64)
        n_p = torch.full((wl.n_i,), float(wl.k), **f64)
        cargs = (i_idx, dt_r, fr0, frd0, out["acc"], out["jerk"], out["nbr_count"], out["nbr_list"],
                 old["nbr_count"], old["nbr_list"], s.t)
        c_out = None
        for _ in range(3):
            c_out = ctx.nb_regular_correct(*cargs, r_s=r_s, n_p=n_p, out=c_out)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        torch.cuda.synchronize()
        ev[0].record()
        for _ in range(5):
            ctx.nb_regular_correct(*cargs, r_s=r_s, n_p=n_p, out=c_out)
        ev[1].record()
        torch.cuda.synchronize()
        t_cor = ev[0].elapsed_time(ev[1]) / 5 / 1e3
        n_old = int(torch.clamp(old["nbr_count"], max=wl.cap).sum().item())
        n_new = int(torch.clamp(out["nbr_count"], max=wl.cap).sum().item())
        cor_bytes = (n_old + n_new) * 4 + wl.n_i * (4 * 24 + 8 * 3 + 4 * 3 + 6 * 24 + 8)
        cor = {"kernel": "corrector_kernel", "rows": wl.n_i, "ms": t_cor * 1e3, "rows_per_s": wl.n_i / t_cor,
               "list_entries_compared": n_old + n_new, "stream_gb_per_s": cor_bytes / t_cor / 1e9,
               "hbm_frac": cor_bytes / t_cor / 1e9 / peaks["hbm_gbs"],
               "note": "step (vii) + eq. (1): symmetric difference of the old and new list, pair terms of the members that "
                       "changed, fp64 Hermite arithmetic; stream_gb_per_s counts both lists and the per-row arrays once "
                       "(the gathers of the changed members come on top)"}
        del old

    # ---- e2e: C-ABI call with HOST (pinned) buffers, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        h_in = [pin(a) for a in (s.x0, s.v0, s.a0, s.j0, s.m, s.t0)]
        h_idx, h_rs = pin(wl.i_idx), pin(wl.r_s)
        # the lists come back in CSR form (nb_regular_force_host_csr): the stored entries packed back to back
        stored = int(torch.clamp(out["nbr_count"], max=wl.cap).sum().item())
        h_out = dict(acc=torch.empty((wl.n_i, 3), dtype=torch.float64).pin_memory(),
                     jerk=torch.empty((wl.n_i, 3), dtype=torch.float64).pin_memory(),
                     nbr_count=torch.empty(wl.n_i, dtype=torch.int32).pin_memory(),
                     nbr_offset=torch.empty(wl.n_i + 1, dtype=torch.int64).pin_memory(),
                     nbr_packed=torch.empty(stored + stored // 16 + 1024, dtype=torch.int32).pin_memory(),
                     n_overflow=torch.zeros(1, dtype=torch.int32).pin_memory())
        h2d = sum(t.numel() * t.element_size() for t in h_in + [h_idx, h_rs])
        # device -> host: acc, jerk, counts, row offsets, n_overflow in full, and the stored list entries
        d2h = wl.n_i * (24 + 24 + 4 + 8) + 8 + 4 + 4 * stored
        ksteps = max(1, min(args.steps, 3))
        ctx.nb_regular_force_host_csr(*h_in, h_idx, h_rs, s.t, h_out)  # warm-up (allocates the mirrors)
        if dist: dist.barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(ksteps):
            ctx.nb_regular_force_host_csr(*h_in, h_idx, h_rs, s.t, h_out)  # synchronises internally
        te = time.perf_counter() - t0
        te_max = max_over_ranks(te, dist, dev)
        e2e = {"value": whole_job_rate(job_pairs, ksteps, job_replicas, te_max), "unit": UNIT,
               "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h), "steps": ksteps,
               "ms_per_step": te_max / ksteps * 1e3,
               "api": "nb_regular_force_host_csr (pinned host buffers; neighbour lists returned in CSR form)",
               "lists_match_device_run": bool(int(h_out["nbr_offset"][-1]) == stored)}
        ctx.nb_set_j(*state_dev)

    if rank != 0:
        if dist: dist.destroy_process_group()
        return 0
    nsm, peak_tf = fp32_peak_tflops(torch, local, peaks)
    ach_tf = wl.pairs * FLOPS_PER_PAIR / t_force / 1e12
    pred_bytes = s.n * PRED_BYTES_PER_J
    headline = args.config == 5 and args.n_i is None
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": t_max / args.steps * 1e3,
        "ms_per_step_median": float(np.median(ts)) * 1e3, "ms_per_step_best": float(ts.min()) * 1e3,
        "value_best": whole_job_rate(job_pairs, 1, job_replicas, float(ts.min())) if world == 1 else None,
        "higher_is_better": True,
        "scaling": "strong" if shard_rows else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": workload_config(wl, args.config),
        "fp32_peak_fraction": value / world * 1e9 * FLOPS_PER_PAIR / (peak_tf * 1e12),
        "roofline": {"bound": "alu", "kernel": "force_kernel", "achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s",
                     "frac": ach_tf / peak_tf,
                     "traffic": FORCE_DRAM_BYTES_C5 if headline else None,
                     "fma_pipe_busy": wl.pairs * LANE_SLOTS_PER_PAIR / t_force / (nsm * 128 * peaks["sm_max_mhz"] * 1e6),
                     "note": f"achieved = N_i*N pairs x {FLOPS_PER_PAIR:.0f} flop (convention) / time of "
                             f"nb_regular_force on its stream (CUDA events; force_kernel plus the small gather and "
                             f"fp64 fix-up kernels); peak = {nsm} SMs x 128 FP32 lanes x 2 x "
                             f"{peaks['sm_max_mhz']:.0f} MHz (MEASURED_PEAKS.json sm_max_mhz, {peaks['src']}; the "
                             f"file holds no FP32 figure, DESIGN.md section 7 derives this one); fma_pipe_busy = "
                             f"{LANE_SLOTS_PER_PAIR:.0f} issued FP32 lane-slots per pair / 128 per clock per SM",
                     "ms": t_force * 1e3},
        "roofline_predictor": {"bound": "hbm", "kernel": "predict_kernel", "achieved": pred_bytes / t_pred_b2b / 1e9,
                               "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": pred_bytes / t_pred_b2b / 1e9 / peaks["hbm_gbs"],
                               "frac_at_survey_160_bytes": s.n * 160 / t_pred_b2b / 1e9 / peaks["hbm_gbs"],
                               "traffic": PRED_DRAM_BYTES_C5 if headline else None, "ms": t_pred_b2b * 1e3,
                               "ms_inside_step": t_pred * 1e3,
                               "note": f"{PRED_BYTES_PER_J} B/j algorithmic (112 B of fp64 state read, 40 B pair record written; SURVEY "
                                       f"8(a) S1 budgets 112 + 48 = 160 B/j for a padded record: frac_at_survey_160_bytes), peak "
                                       f"{peaks['src']} copy bandwidth; ms = average of ten launches back to back (one CUDA-graph replay) between two "
                                       f"CUDA events (L2 flushed before; state + records exceed the L2); ms_inside_step = the interval between "
                                       f"two events around the ONE launch of a timed step, which includes the event-to-kernel "
                                       f"latency (the kernel alone under ncu, cold: 24.8 us = 6.4 TB/s, "
                                       f"profiles/r2_bench_c5_launches.md)"},
        "launch": info, "gpu_launches": int(info["launches"] + 1) * args.steps,
        "fixup_rows_per_step": info["fixup_rows"],
        "mean_neighbours": mean_cnt, "overflow_rows": n_over, "clocks": clocks, "e2e": e2e,
        "next_irregular": irr,
        "next_corrector": cor,
    }
    if shard_rows:
        line["config"]["parallelism"] = f"rows sharded over {world} ranks (rank 0 owns rows {shard_rows[0]}..{shard_rows[1]}); " \
                                        "every rank predicts all j; no data-path collective"
        line["config"]["job_pairs_per_step"] = job_pairs
    if not args.no_cpu and world >= 1:
        cb, _, rows, ores = cpu_baseline(wl, target_seconds=args.cpu_seconds, min_rows=min(wl.n_i, 1024))
        line["cpu_baseline"] = cb
        # parity of the last timed repetition (out has not been written since) against those oracle rows
        line["parity"] = parity_in_run(wl, out, rows, ores)
    b.close()
    if headline and not args.no_also and world == 1:
        # the other configs, incl. the N = 65536 full block the ">= 50 % for N >= 65536" target names
        line["also"] = [run_also(c, local, flush, peaks, steps=(10 if c == 3 else 20)) for c in (3, 4, 2, 1)]
    print(json.dumps(line))
    if dist: dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--n-i", type=int, default=None, help="active-block size (configs 1, 3, 5 only)")
    ap.add_argument("--sweep-large", action="store_true", help="with --sweep: blocks 32 ... 16384 of the config 5 state")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-irregular", action="store_true")
    ap.add_argument("--no-also", action="store_true", help="skip the other configs beside the headline (configs 3, 4, 2, 1)")
    ap.add_argument("--sweep", action="store_true", help="config 3 active-block sweep 32 ... 65536 (one JSON line)")
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--shard", default="none", choices=["none", "rows"],
                    help="none: N independent replicas (default, weak); rows: one job, rows split over the ranks (strong)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.sweep:
        return run_sweep(args)
    return run_gpu_arm(args)


if __name__ == "__main__":
    sys.exit(main())
