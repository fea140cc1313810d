#!/usr/bin/env python
"""bench.py — throughput of the lrmd hot path on B200, one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload KEY] [--only] [--f32-pairs] [--ordered-pairs]
                    [--sharded] [--fp64-peak] [--impl reference]

A bench "step" is one complete integrator time step of the workload (three force
evaluations + the kick/drift updates — what the paper's Tables 1-3 time).  The primary workload is
BASELINE.json configs[4], the largest single-GPU configuration (2D self-gravitating, N = 1,048,576,
eps = 1e-3, dt = 0.005, fp64).  The LAST stdout line is that headline alone, trimmed to under 4 KB (the
driver keeps only the tail of stdout).  With one GPU and without --only / --no-others the other configs are
measured too, together with the ordered-pair kernels (the paper's own scheme, LRMD_OPT_PAIR_SYMMETRIC = 0)
on the pair configs, config 5's fp32-pair variant and the sizes of the paper's Tables 1-3: their full
objects go to gpurun_out/bench_others.json (with the untrimmed headline) and one short line each to stderr.

Numbers reported (all measured in this process, never under a profiler):
  value      whole-job throughput, state resident in HBM, CUDA events on the launching stream
  e2e        the same metric through lrmd_step_host: pinned HOST buffers, H2D + (3K+1) force
             evaluations + D2H inside the timed region
  roofline   the dominant kernel (pair-force kernel / HMF fused substage): work per force evaluation (pair
             models) or per launch (HMF) / its device time from event pairs around every launch (second pass).
             Pair models (fp64): `frac` = EXECUTED FP64 instructions / s over 148 x 64 x f_max (the
             acceptance number), `flop_frac` = executed flops (FMA = 2) over 148 x 64 x 2 x f_max beside it; the
             symmetric kernels evaluate every unordered pair once, so their executed work per delivered pair is about
             half the ordered kernels' (`flop_frac_ordered_convention` gives that reading).  HMF: 32 B per
             particle-substage against the measured HBM copy bandwidth.
  energy     lrmd_energy timed apart from the steps
  cpu_baseline  the oracle (oracle/lrmd_ref.cpp), as it stands, on this box's host cores, bounded sample

Multi-GPU (torchrun, --gpus N): the path does not shard under BASELINE.json's north_star ("no sharding
or collectives between GPUs"): N independent replicas, one per rank, weak scaling; value = units all
ranks processed / max-over-ranks device time.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

L2_BYTES = 126 * 1024 * 1024
SM_COUNT = 148
FP64_LANES_PER_SM = 64          # DFMA lanes per SM (guide: 148 SMs; FP64 issue = 64/clk/SM on B200)

# flops per ordered pair with FMA = 2: Ring 7 DFMA + 4 DMUL = 18; 2D 7 DFMA + 2 DADD = 16
PAIR_FLOP = {1: 18.0, 2: 16.0}
PAIR_FP64_INSTR = {1: 11.0, 2: 9.0}
# symmetric kernel (row N4): per UNORDERED pair Ring 8 DFMA + 4 DMUL, 2D 9 DFMA + 2 DADD = 20 flop; the figures below are
# per ordered pair delivered (half), i.e. the work the kernel EXECUTES, not the ordered-pair convention
SYM_PAIR_FLOP = {1: 10.0, 2: 10.0}
SYM_PAIR_FP64_INSTR = {1: 6.0, 2: 5.5}
HMF_BYTES_PER_PARTICLE_SUBSTAGE = 32.0

# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel come from the committed
# `ncu --set full` captures: profiles/r03_traffic.csv names, per bench entry, the kernel, the two byte counts and
# the capture they were read from (profiles/r03_ncu.md and profiles/r02_ncu_full.md give the commands).
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r03_traffic.csv")


def ncu_traffic(entry, kernel):
    """(bytes per launch, source) of `kernel` in bench entry `entry` from profiles/r03_traffic.csv, or (None, why)."""
    import csv
    if not os.path.exists(TRAFFIC_CSV):
        return None, "profiles/r03_traffic.csv missing"
    with open(TRAFFIC_CSV) as fh:
        for row in csv.DictReader(fh):
            if row["entry"] == entry:
                if row["kernel"] != kernel:
                    return None, "capture is of %s, this run launched %s" % (row["kernel"], kernel)
                return float(row["dram_read_bytes"]) + float(row["dram_write_bytes"]), "profiles/" + row["capture"]
    return None, "no capture of this entry"


DEFAULT_STEPS = {"hmf_1e4": 1000, "ring_16k": 100, "grav2d_64k": 50, "hmf_5e7": 100, "grav2d_1m": 5,
                 "hmf_1e5": 1000, "hmf_1e6": 500, "hmf_1e7": 200, "ring_102k": 10, "ring_512k": 3, "grav2d_102k": 10}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            d = json.load(fh)
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)), "source": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback"}


# ---- clocks sampler (nvidia-smi's numbers through NVML) ---------------------------------------------------

class ClockSampler:
    REASONS = {
        0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
        0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x100: "display_clock_setting",
    }

    def __init__(self, index: int):
        self.index = index
        self.samples, self.bits = [], 0
        self.max_mhz = None
        self._stop = threading.Event()
        self._thr = None
        self._nvml = None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nvml = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nvml = None
            return self
        self._thr = threading.Thread(target=self._run, daemon=True)
        self._thr.start()
        return self

    def _run(self):
        nv = self._nvml
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                get = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or nv.nvmlDeviceGetCurrentClocksThrottleReasons
                self.bits |= int(get(self._h))
            except Exception:
                pass
            self._stop.wait(0.02)

    def stop(self):
        self._stop.set()
        if self._thr:
            self._thr.join(timeout=2)
        reasons = [name for bit, name in self.REASONS.items() if self.bits & bit]
        return {
            "sm_mhz": statistics.median(self.samples) if self.samples else None,
            "sm_max_mhz": self.max_mhz,
            "reasons": reasons,
            "samples": len(self.samples),
        }


# ---- replicas over ranks (the path does not shard; no data-path collective) -----------

def max_over_ranks(x: float, dist_mod, device) -> float:
    """MAX of a per-rank scalar over all ranks (the only collective bench.py uses: timing, not data)."""
    if dist_mod is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist_mod.all_reduce(t, op=dist_mod.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(units_per_rank_step: float, steps: int, ms_max: float, world: int) -> float:
    """Aggregate throughput of `world` independent replicas: all units processed / slowest rank's device time."""
    return world * units_per_rank_step * steps / (ms_max * 1e-3)


# ---- one workload on this rank's GPU ------------------------------------------------------------------------

def units_per_force(w):
    """(metric, unit, units per force evaluation)."""
    if w.model == 0:
        return "particle-steps/s", "particle-steps/s", None
    return "pair-interactions/s", "pair-interactions/s", float(w.N) * float(w.N)


def run_workload(w, K, W, dist_ctx, with_e2e=True, with_roofline=True, f32_pairs=False, ordered_pairs=False,
                 force_symmetric=False, roofline_steps=2000, e2e_steps=20, fp64_peak=None, with_energy=True):
    import torch
    from paper_1212_0262_b200 import lrmd

    dev = torch.device("cuda", torch.cuda.current_device())
    peaks = measured_peaks()
    st = w.state()
    opts = {}
    if f32_pairs:
        opts[lrmd.OPT_PAIR_PRECISION] = 1
    if w.model != 0 and (ordered_pairs or force_symmetric):
        opts[lrmd.OPT_PAIR_SYMMETRIC] = 0 if ordered_pairs else 1
    ctx = lrmd.Context(w.model, w.N, w.eps, device=dev, options=opts or None)
    ctx.set_state(*st)
    stream = torch.cuda.current_stream(dev)
    state_bytes = ctx.narrays * w.N * 8
    larger_than_l2 = state_bytes > L2_BYTES
    resident_by_design = w.model == 0 and ctx.get_option(lrmd.OPT_HMF_VARIANT) in (3, 4)
    flush = None
    if not larger_than_l2 and not resident_by_design:
        flush = torch.empty(2 * L2_BYTES, dtype=torch.uint8, device=dev)

    def barrier():
        if dist_ctx is not None:
            dist_ctx.barrier()
        torch.cuda.synchronize(dev)

    def timed_pass(K):
        """K steps; returns device ms (sum of the event pairs) on this rank."""
        if flush is None:
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            ctx.step(K, w.dt)
            b.record(stream)
            b.synchronize()
            return a.elapsed_time(b)
        evs = []
        for _ in range(K):
            flush.fill_(1)                                   # untimed: outside the event pair
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            ctx.step(1, w.dt)
            b.record(stream)
            evs.append((a, b))
        torch.cuda.synchronize(dev)
        return sum(a.elapsed_time(b) for a, b in evs)

    # warm-up (also caches the force at the current positions)
    timed_pass(W)
    if resident_by_design and ctx.get_option(lrmd.OPT_HMF_VARIANT) not in (3, 4):
        # the device refused the cooperative launch and the library fell back to the streaming kernels: flush after all
        resident_by_design = False
        if not larger_than_l2:
            flush = torch.empty(2 * L2_BYTES, dtype=torch.uint8, device=dev)
        timed_pass(W)
    barrier()
    sampler = ClockSampler(torch.cuda.current_device()).start()
    l0 = ctx.launch_count()
    ms = timed_pass(K)
    launches = ctx.launch_count() - l0
    barrier()
    clocks = sampler.stop()
    ms_max = max_over_ranks(ms, dist_ctx, dev)
    world = dist_ctx.get_world_size() if dist_ctx is not None else 1

    metric, unit, upf = units_per_force(w)
    if w.model == 0:
        units_per_step = float(w.N)
    else:
        units_per_step = 3.0 * upf
    value = whole_job_value(units_per_step, K, ms_max, world)

    out = {
        "metric": metric, "value": value, "unit": unit, "ms_per_step": ms_max / K,
        "gpu_launches": int(launches), "clocks": clocks,
        "l2": l2_statement(w, hmf_resident=resident_by_design),
        "options": {"pair_ctas": ctx.get_option(lrmd.OPT_PAIR_CTAS), "pair_variant": ctx.get_option(lrmd.OPT_PAIR_VARIANT),
                    "pair_slots": ctx.get_option(lrmd.OPT_PAIR_SLOTS), "graph": ctx.get_option(lrmd.OPT_GRAPH),
                    "hmf_grid": ctx.get_option(lrmd.OPT_HMF_GRID), "hmf_variant": ctx.get_option(lrmd.OPT_HMF_VARIANT),
                    "pair_precision": ctx.get_option(lrmd.OPT_PAIR_PRECISION),
                    "pair_symmetric": ctx.get_option(lrmd.OPT_PAIR_SYMMETRIC)},
    }

    # ---- roofline of the dominant kernel: second pass with an event pair around each of its launches
    if with_roofline:
        ctx.set_option(lrmd.OPT_KERNEL_TIMING, 1)
        Kr = min(K, roofline_steps)
        ctx.kernel_time()
        ms_r = timed_pass(Kr)
        kms, kn = ctx.kernel_time()
        ctx.set_option(lrmd.OPT_KERNEL_TIMING, 0)
        avg_s = (kms / max(kn, 1)) * 1e-3
        if w.model != 0:
            # pair models: per FORCE EVALUATION (3 per step; the warp-level symmetric kernel may take several launches, one
            # per batch of i-tiles, for one evaluation)
            avg_s = (kms / (3.0 * Kr)) * 1e-3
        clk = (clocks.get("sm_mhz") or peaks["sm_max_mhz"])
        symk = ctx.get_option(lrmd.OPT_PAIR_SYMMETRIC) if w.model != 0 else 0     # 0 ordered, 1 warp-level, 2 band
        if w.model == 0:
            kernel = {0: "hmf_substage_kernel", 3: "hmf_cluster_kernel", 4: "hmf_grid_kernel"}.get(
                ctx.get_option(lrmd.OPT_HMF_VARIANT), "hmf_substage_tma_kernel")
            bytes_per_launch = HMF_BYTES_PER_PARTICLE_SUBSTAGE * w.N
            if ctx.get_option(lrmd.OPT_HMF_VARIANT) in (3, 4):
                # cluster- / grid-resident kernels: one launch runs all Kr steps with the state on chip; the figure is
                # what the same substages would stream through HBM (context only: the working set is on chip)
                bytes_per_launch *= 3.0 * Kr
            achieved = bytes_per_launch / avg_s / 1e9
            roof = {"bound": "hbm", "achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                    "frac": achieved / peaks["hbm_gbs"], "peak_source": peaks["source"] + " (MEASURED_PEAKS.json hbm_gbs)",
                    "algorithmic_bytes_per_launch": bytes_per_launch}
            if ctx.get_option(lrmd.OPT_HMF_VARIANT) == 4:
                roof["note"] = ("grid-resident kernel: the state (%.1f MB) stays in shared memory for the whole call; the step is bound by "
                                "the grid barrier between substages, the HBM figure is context only" % (state_bytes / 1e6))
            elif 2.0 * state_bytes <= L2_BYTES:
                roof["note"] = ("state (%.1f MB) fits the 126 MB L2: the substages stream it through L2, not HBM; the HBM figure "
                                "is context only" % (state_bytes / 1e6))
        elif f32_pairs:
            # fp32 pair arithmetic: one MUFU.RCP per pair on the special-function unit, 16 lanes per SM per clock
            kernel = "ring_force_f32_kernel" if w.model == 1 else {0: "grav_force_f32_kernel", 1: "grav_force_sym_f32_kernel", 2: "grav_force_band_f32_kernel"}[symk]
            mufu = float(w.N) * float(w.N) * (0.5 if symk else 1.0)      # executed: one per (un)ordered pair evaluated
            peak = SM_COUNT * 16 * peaks["sm_max_mhz"] * 1e6 / 1e12
            achieved = mufu / avg_s / 1e12
            roof = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "T MUFU.RCP/s",
                    "frac": achieved / peak,
                    "peak_source": "derived: 148 SM x 16 SFU lanes x sm_max_mhz (DESIGN.md); FP32 pipe second: %d FADD/FMUL/FFMA per pair"
                                   % (12 if w.model == 1 else 6),
                    "algorithmic_mufu_per_launch": mufu}
            if w.model == 1:
                # Ring, half-angle form: 12 FADD/FMUL/FFMA per pair bind before the one MUFU.RSQ (128 FP32 lanes per SM per
                # clock: 12 / 128 clock per pair against 1 / 16 for the SFU)
                fp32 = 12.0 * float(w.N) * float(w.N)
                peak32 = SM_COUNT * 128 * peaks["sm_max_mhz"] * 1e6 / 1e12
                roof.update({"achieved": fp32 / avg_s / 1e12, "peak": peak32, "unit": "T FP32 instr/s (thread level)",
                             "frac": fp32 / avg_s / 1e12 / peak32,
                             "peak_source": "derived: 148 SM x 128 FP32 lanes x sm_max_mhz (DESIGN.md); SFU second: one MUFU.RSQ per pair",
                             "algorithmic_fp32_instr_per_launch": fp32,
                             "mufu_frac": mufu / avg_s / 1e12 / peak})
            if symk:
                roof["note"] = ("symmetric fp32 kernel: one MUFU.RCP and 8 FADD/FFMA per UNORDERED pair (N^2/2 evaluations deliver "
                                "N^2 pair interactions), ~10.5 issued instructions per evaluation: instruction issue binds before "
                                "the SFU; by the ordered-pair convention (one MUFU per delivered pair) the launch reads %.3f"
                                % (float(w.N) * float(w.N) / avg_s / 1e12 / peak))
        else:
            kernel = {0: "pair_force_kernel", 1: "pair_force_sym_kernel", 2: "pair_force_band_kernel"}[symk]
            # (i) pipe utilisation = EXECUTED FP64 instructions / s over 148 x 64 x f_max — the acceptance
            # number, reported as `frac`; (ii) the flop fraction (FMA = 2) beside it.  The symmetric kernels evaluate every
            # unordered pair once: their executed work per delivered pair is about half the ordered kernels'.
            flop = (SYM_PAIR_FLOP if symk else PAIR_FLOP)[w.model] * w.N * w.N
            instr = (SYM_PAIR_FP64_INSTR if symk else PAIR_FP64_INSTR)[w.model] * w.N * w.N
            instr_rate = instr / avg_s
            peak_instr = SM_COUNT * FP64_LANES_PER_SM * peaks["sm_max_mhz"] * 1e6
            roof = {"bound": "alu", "achieved": instr_rate / 1e12, "peak": peak_instr / 1e12, "unit": "T FP64 instr/s",
                    "frac": instr_rate / peak_instr,
                    "peak_source": "derived: 148 SM x 64 FP64 lanes x sm_max_mhz (DESIGN.md 6)",
                    "algorithmic_fp64_instr_per_launch": instr,
                    "tflops": flop / avg_s / 1e12, "peak_tflops": 2.0 * peak_instr / 1e12,
                    "flop_frac": flop / avg_s / (2.0 * peak_instr),
                    "frac_at_held_clock": instr_rate / (SM_COUNT * FP64_LANES_PER_SM * clk * 1e6)}
            if fp64_peak is not None:
                # the committed microbenchmark (lrmd_fp64_peak): what the FP64 pipe sustains on this box
                roof["frac_of_measured_issue_rate"] = instr_rate / fp64_peak["dmul_instr_per_s"]
                roof["flop_frac_of_measured_dfma"] = flop / avg_s / 1e12 / fp64_peak["dfma_tflops"]
            if symk:
                # by the ordered-pair convention (16 / 18 flop per delivered pair) the same launch would read:
                roof["flop_frac_ordered_convention"] = PAIR_FLOP[w.model] * w.N * w.N / avg_s / (2.0 * peak_instr)
        entry = w.key + ("_f32pairs" if f32_pairs else "") + ("_ordered_pairs" if (w.model != 0 and not symk) else "")
        traffic, tsrc = ncu_traffic(entry, kernel)
        if w.model == 0:
            alg_bytes = roof["algorithmic_bytes_per_launch"]
        else:
            # the j-stream read once (16 N, fp32 stream 8 N) + the force written once (8 N per component)
            alg_bytes = (8.0 if f32_pairs else 16.0) * w.N + 8.0 * w.N * (2 if w.model == 2 else 1)
        launches_per_eval = (kn / (3.0 * Kr)) if w.model != 0 else None
        roof.update({"kernel": kernel, "kernel_avg_ms": avg_s * 1e3, "kernel_launches_timed": kn,
                     "kernel_launches_per_force_evaluation": launches_per_eval,
                     "kernel_share_of_step": kms / ms_r if ms_r > 0 else None,
                     "traffic": traffic, "traffic_source": tsrc,
                     "traffic_what": "dram__bytes_read.sum + dram__bytes_write.sum per launch (ncu --set full)",
                     "algorithmic_dram_bytes_per_force_evaluation" if w.model != 0 else "algorithmic_dram_bytes_per_launch": alg_bytes,
                     "traffic_ratio": (traffic * (launches_per_eval or 1.0) / alg_bytes) if traffic is not None else None,
                     "workspace_bytes": ctx.workspace_bytes()})
        out["roofline"] = roof

    # ---- energy sums (rows a-E1..a-E3), timed apart from the steps
    if with_energy:
        ctx.energy()
        torch.cuda.synchronize(dev)
        ts = []
        for _ in range(2 if w.N >= 500_000 and w.model != 0 else 5):    # config 5: about half a second per O(N^2) sweep
            if flush is not None:
                flush.fill_(1)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            ctx.energy()
            b.record(stream)
            b.synchronize()
            ts.append(a.elapsed_time(b))
        ems = statistics.median(ts)
        out["energy"] = {"ms_per_call": ems, "what": "lrmd_energy: K, V and momentum / magnetisation (3 launches)"}
        if w.model != 0:
            out["energy"]["pair_interactions_per_s"] = float(w.N) * float(w.N) / (ems * 1e-3)

    # ---- end to end through lrmd_step_host: pinned host buffers, copies inside the timed region
    if with_e2e:
        host = [torch.from_numpy(a.copy()).pin_memory() for a in st]
        Ke = max(1, min(K, e2e_steps if w.model != 0 else K))
        ctx.step_host(host, 1, w.dt)                          # warm-up of the copy path
        for h, a in zip(host, st):
            h.copy_(torch.from_numpy(a))
        barrier()
        t0 = time.perf_counter()
        ctx.step_host(host, Ke, w.dt)                         # synchronises the stream before returning
        t1 = time.perf_counter()
        dt_s = t1 - t0
        dt_s = max_over_ranks(dt_s, dist_ctx, dev)
        if w.model == 0:
            e_units = float(w.N) * Ke
        else:
            e_units = (3.0 * Ke + 1.0) * upf
        out["e2e"] = {"value": world * e_units / dt_s, "unit": unit, "h2d_bytes_per_step": state_bytes / Ke,
                      "d2h_bytes_per_step": state_bytes / Ke, "steps_per_call": Ke,
                      "note": "lrmd_step_host: H2D state + force evaluation + %d steps + D2H state, host wall clock "
                              "around the synchronous call; bytes are per step of the %d-step call" % (Ke, Ke)}
    ctx.close()
    del flush
    torch.cuda.empty_cache()
    return out


# ---- the oracle on the host cores --------------------------------------------------------------------------

def oracle_sample_rate(w, seconds, nthreads=0):
    """Times the oracle, as it stands, on a bounded sample of workload w for about `seconds`.
    Returns (units_per_second, description, threads)."""
    import numpy as np
    from oracle import ref
    threads = ref.max_threads() if nthreads <= 0 else nthreads
    st = w.state()
    if w.model == 0:
        n_s = min(w.N, 2_000_000)
        th, p = st[0][:n_s].copy(), st[1][:n_s].copy()
        t0 = time.perf_counter()
        f0, _ = ref.step(0, 0.0, th, None, p, None, 1, w.dt)
        per_step = time.perf_counter() - t0
        n = max(1, int(seconds / max(per_step, 1e-6)))
        t0 = time.perf_counter()
        ref.step(0, 0.0, th, None, p, None, n, w.dt, f0, None, force_valid=True)
        el = time.perf_counter() - t0
        return n_s * n / el, f"{n} serial steps of the first {n_s} particles (eqs.(6)-(7) path)", 1
    q0, q1 = (st[0], st[1]) if w.model == 2 else (st[0], None)
    rng = np.random.default_rng(1)
    form = 1
    r0 = max(threads * 8, 64)
    rows = rng.choice(w.N, min(r0, w.N), replace=False)
    t0 = time.perf_counter()
    ref.forces_rows(w.model, w.eps, q0, q1, rows, form=form, nthreads=nthreads)
    el = time.perf_counter() - t0
    rate = len(rows) * w.N / el
    R = int(min(w.N, max(len(rows), seconds * rate / w.N)))
    rows = rng.choice(w.N, R, replace=False)
    t0 = time.perf_counter()
    ref.forces_rows(w.model, w.eps, q0, q1, rows, form=form, nthreads=nthreads)
    el = time.perf_counter() - t0
    what = "eq.(9) precomputed sin/cos form" if w.model == 1 else "eq.(3) force, true division"
    return R * w.N / el, f"forces on {R} sampled rows x all {w.N} j ({what}), OpenMP over rows", threads


HMF_RESIDENT_MAX_N = 1_070_336      # up to here the default HMF kernel keeps the state on chip (lrmd.h, LRMD_OPT_HMF_VARIANT)


def l2_statement(w, hmf_resident=None):
    """How the timed iterations keep L2 from flattering the number.  Decided by the SAME two predicates that switch the
    flush in run_workload: the state is larger than L2, or the HMF kernel in use keeps the state on chip for the whole call
    (`hmf_resident`; None = what the library chooses by default for this N, which is all the reference arm can know)."""
    narr = 4 if w.model == 2 else 2
    state_bytes = narr * w.N * 8
    if hmf_resident is None:
        hmf_resident = w.model == 0 and w.N <= HMF_RESIDENT_MAX_N
    if state_bytes > L2_BYTES:
        return "inputs larger than L2 (%.0f MB state)" % (state_bytes / 1e6)
    if hmf_resident:
        return "not flushed: %.2f MB state kept on chip by the resident kernel for all steps of one launch" % (state_bytes / 1e6)
    return "L2 flushed (256 MiB write) before every timed step"


def workload_config(w, world, l2=None):
    """The `config` object of the JSON line: the workload, identical for the b200 and the reference arm (`l2` = the
    statement of the run that was timed; None = the default choice for this N)."""
    return {"workload": w.key, "model": ["hmf", "ring", "grav2d"][w.model], "N": w.N, "eps": w.eps, "dt": w.dt,
            "step": "one 4th-order time step = 3 force evaluations + kick/drift updates (PAPER.md:54-63)",
            "parallelism": "replicas only (no sharding, no collectives)" if world > 1 else "1 GPU",
            "l2": l2 or l2_statement(w)}


def run_reference(args, w):
    """--impl reference: the oracle timed on the host cores; each step is a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    metric, unit, _ = units_per_force(w)
    per_step_s = 2.0
    rates = []
    desc, threads = "", 1
    for k in range(args.warmup + args.steps):
        r, desc, threads = oracle_sample_rate(w, per_step_s)
        if k >= args.warmup:
            rates.append(r)
    value = len(rates) / sum(1.0 / r for r in rates)
    line = {
        "impl": "reference", "metric": metric, "value": value, "unit": unit, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": None, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": workload_config(w, int(os.environ.get("WORLD_SIZE", "1"))),
        "cpu_baseline": {"value": value, "unit": unit, "cores": threads, "kind": "oracle", "sample": "per step: " + desc},
        "e2e": {"value": value, "unit": unit, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(headline(line)))      # trimmed like the b200 arm's line, so that both print the same `config`
    return 0


def fp64_peak_table(device=None, iters=20000, full=True):
    """bench.py --fp64-peak: the committed FP64 issue-rate microbenchmark (lrmd_fp64_peak), one JSON object.
    `peak` = the best sustained DFMA rate over the resident-warp sweep; `mixes` = FP64 lanes busy per clock per SM
    when each group of 16 DFMA carries k instructions of another class (what a non-FP64 instruction costs)."""
    import torch
    from paper_1212_0262_b200 import lrmd
    dev = device or torch.device("cuda", torch.cuda.current_device())
    scratch = torch.empty(148 * 64 * 32 * 8 + 148 * 64 * 4 + 4096 + 256, dtype=torch.uint8, device=dev)
    ptr = (scratch.data_ptr() + 255) // 256 * 256
    stream = int(torch.cuda.current_stream(dev).cuda_stream)

    def run(op, mix, xn, warps):
        rc, out = lrmd.lrmd_fp64_peak(op, mix, xn, warps, iters, ptr, scratch.numel() - 256, stream)
        if rc != lrmd.OK:
            raise lrmd.LrmdError(rc, "lrmd_fp64_peak")
        return {"instr_per_s": out[0], "sm_mhz": out[1], "lanes_per_clk_per_sm": out[2], "ms": out[3]}

    res = {"what": "lrmd_fp64_peak: 16 independent FP64 chains per thread, 148 x warps_per_sm warps, CUDA events around one launch; "
                   "sm_mhz = clock64 / globaltimer inside the kernel", "iters": iters, "ops": {}, "mixes": {}}
    best = None
    for name, op in (("dfma", 0), ("dmul", 1), ("dadd", 2), ("dfma_3_private_regs", 3), ("dfma_1_shared_reg", 4),
                     ("dfma_square", 5), ("dfma_imm_addend", 6)):
        res["ops"][name] = {}
        for warps in ((4, 8, 16, 32, 64) if full else (32,)):
            r = run(op, 0, 0, warps)
            res["ops"][name][str(warps)] = r
            if op == 0 and (best is None or r["instr_per_s"] > best["instr_per_s"]):
                best = dict(r, warps_per_sm=warps)
    res["peak"] = best
    if full:
        for name, mix in (("int_lop3", 1), ("mufu_rcp64h", 2), ("shfl", 3), ("lds64", 4), ("mufu_seed_plus_dfma", 5),
                          ("mov", 6), ("sts64", 7)):
            res["mixes"][name] = {}
            for warps in (8, 16, 32):
                res["mixes"][name][str(warps)] = {str(xn): run(0, mix, xn, warps)["lanes_per_clk_per_sm"] for xn in (2, 4, 8, 16)}
    del scratch
    return res


# ---- strong scaling through the sharded path — opt-in, never the default ------

def sharded_plan(w, world, rank):
    """Host logic of --sharded: which particles rank `rank` owns and what one substage exchanges.
    HMF: one all-reduce of 2 doubles; Ring / 2D: one all-gather of the packed positions, 16 bytes per
    particle.  Pure host code (tested with gloo, world 2)."""
    from paper_1212_0262_b200 import sharded
    i0, n = sharded.shard_bounds(w.N, world)[rank]
    if w.model == 0:
        exchange = {"collective": "all_reduce", "bytes_per_substage": 16}
        units_per_step = float(w.N)
    else:
        exchange = {"collective": "all_gather", "bytes_per_substage": 16 * w.N}
        units_per_step = 3.0 * float(w.N) * float(w.N)
    return {"i0": i0, "n_local": n, "exchange": exchange, "units_per_step": units_per_step,
            "rows_x_columns": [n, w.N] if w.model != 0 else None}


def strong_scaling_value(units_per_step, steps, ms_max):
    """Whole-job throughput of ONE problem split over the ranks: its units / the slowest rank's device time."""
    return units_per_step * steps / (ms_max * 1e-3)


def run_sharded(w, K, W, dist_ctx, world, rank):
    import torch
    from paper_1212_0262_b200 import sharded
    dev = torch.device("cuda", torch.cuda.current_device())
    plan = sharded_plan(w, world, rank)
    coll = sharded.TorchDistCollectives(dist_ctx, rank, world) if dist_ctx is not None else sharded.SingleRankCollectives()
    ctx = sharded.ShardedContext(w.model, w.N, w.eps, coll, device=dev)
    ctx.set_state_global(*w.state())
    stream = torch.cuda.current_stream(dev)

    def barrier():
        if dist_ctx is not None:
            dist_ctx.barrier()
        torch.cuda.synchronize(dev)

    ctx.step(W, w.dt)
    barrier()
    sampler = ClockSampler(torch.cuda.current_device()).start()
    l0 = ctx.launch_count()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(stream)
    ctx.step(K, w.dt)
    b.record(stream)
    b.synchronize()
    ms = a.elapsed_time(b)
    launches = ctx.launch_count() - l0
    barrier()
    clocks = sampler.stop()
    ms_max = max_over_ranks(ms, dist_ctx, dev)
    metric, unit, _ = units_per_force(w)
    ctx.close()
    return {"metric": metric, "value": strong_scaling_value(plan["units_per_step"], K, ms_max), "unit": unit, "n_gpus": world,
            "steps": K, "warmup": W, "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": dict(workload_config(w, world), parallelism="sharded: %d ranks, rows split, %s of %d bytes per substage"
                           % (world, plan["exchange"]["collective"], plan["exchange"]["bytes_per_substage"])),
            "clocks": clocks, "e2e": None, "gpu_launches": int(launches),
            "note": "opt-in strong-scaling line (lrmd_set_shard + torch.distributed collectives between the kernels); "
                    "BASELINE.json's north_star fixes one GPU, so the default bench line runs replicas"}


def fp64_peak_summary():
    """The numbers bench.py quotes beside the derived FP64 peak: sustained DFMA rate (two operands shared, the best
    case the register file allows), DMUL rate (two register operands: the pipe's issue rate) and the rate of a DFMA
    that reads three private registers (what an accumulate fma(dx, y, f) of the pair kernels is), 32 warps per SM."""
    t = fp64_peak_table(full=False)
    ops = t["ops"]
    dfma, dmul, dfma3 = ops["dfma"]["32"], ops["dmul"]["32"], ops["dfma_3_private_regs"]["32"]
    return {"dfma_tflops": 2.0 * dfma["instr_per_s"] / 1e12, "dfma_instr_per_s": dfma["instr_per_s"],
            "dmul_instr_per_s": dmul["instr_per_s"], "dfma_3_private_regs_instr_per_s": dfma3["instr_per_s"],
            "sm_mhz": dfma["sm_mhz"],
            "what": "lrmd_fp64_peak (bench.py --fp64-peak), 32 warps per SM: DFMA a*m+c %.3e instr/s = %.2f TFLOP/s, DMUL %.3e "
                    "instr/s, DFMA on three private registers %.3e instr/s, SM clock held %.0f MHz"
                    % (dfma["instr_per_s"], 2.0 * dfma["instr_per_s"] / 1e12, dmul["instr_per_s"], dfma3["instr_per_s"],
                       dfma["sm_mhz"])}


# ---- the one stdout line --------------------------------------------------------------------------------------
# The driver keeps only the tail of stdout, so the LAST line must be small: the headline object alone, trimmed to the keys
# below and bounded by HEADLINE_MAX_BYTES.  Everything else (the other configs, the paper's table sizes, the ordered-pair
# and fp32 variants, the long explanations) goes to OTHERS_FILE and, one compact line per entry, to stderr.  What the
# roofline keys mean is written once, instead of in every line.
HEADLINE_MAX_BYTES = 4000
OTHERS_FILE = os.path.join("gpurun_out", "bench_others.json")

HEADLINE_KEYS = ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                 "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline", "energy",
                 "options", "others_file")
ROOFLINE_KEYS = ("bound", "achieved", "peak", "unit", "frac", "traffic", "kernel", "kernel_avg_ms", "kernel_share_of_step",
                 "peak_source", "flop_frac", "tflops", "peak_tflops", "frac_at_held_clock", "frac_of_measured_issue_rate",
                 "flop_frac_of_measured_dfma", "flop_frac_ordered_convention", "mufu_frac", "traffic_ratio", "traffic_source",
                 "workspace_bytes")
SUB_KEYS = {
    "config": ("workload", "model", "N", "eps", "dt", "parallelism", "l2"),
    "clocks": ("sm_mhz", "sm_max_mhz", "reasons", "samples"),
    "e2e": ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "steps_per_call"),
    "roofline": ROOFLINE_KEYS,
    "cpu_baseline": ("value", "unit", "cores", "kind", "sample"),
    "energy": ("ms_per_call", "pair_interactions_per_s"),
}


def _short(v, limit=160):
    if isinstance(v, float):
        return float("%.6g" % v)
    if isinstance(v, str) and len(v) > limit:
        return v[: limit - 3] + "..."
    return v


def headline(line: dict) -> dict:
    """The object printed as the last stdout line: `line` cut down to HEADLINE_KEYS / SUB_KEYS, floats to 6 digits, long
    strings clipped; if it is still over HEADLINE_MAX_BYTES the optional keys go, last first (never the contract's)."""
    out = {}
    for k in HEADLINE_KEYS:
        if k not in line:
            continue
        v = line[k]
        if isinstance(v, dict) and k in SUB_KEYS:
            v = {kk: _short(v[kk]) for kk in SUB_KEYS[k] if kk in v and v[kk] is not None or kk == "traffic" and kk in v}
        elif isinstance(v, dict):
            v = {kk: _short(vv) for kk, vv in v.items()}
        else:
            v = _short(v)
        out[k] = v
    optional = [("options", None), ("energy", None)] + [("roofline", kk) for kk in reversed(ROOFLINE_KEYS[6:])]
    while len(json.dumps(out)) > HEADLINE_MAX_BYTES and optional:
        k, kk = optional.pop(0)
        if kk is None:
            out.pop(k, None)
        elif isinstance(out.get(k), dict):
            out[k].pop(kk, None)
    return out


def write_others(others: dict, line: dict):
    """Side file with the full objects (headline untrimmed + the other entries); returns its path or None."""
    try:
        os.makedirs(os.path.dirname(os.path.join(ROOT, OTHERS_FILE)), exist_ok=True)
        with open(os.path.join(ROOT, OTHERS_FILE), "w") as fh:
            json.dump({"headline": line, "others": others}, fh, indent=1)
        return OTHERS_FILE
    except OSError:
        return None


def run_others(w, inputs, peak):
    """The entries beside the headline (1 GPU, default run): the other BASELINE.json configs, the paper's Table 1-3 sizes,
    the ordered-pair kernels (the paper's own scheme) and the fp32-pair variants.  An entry that fails is recorded, not
    raised: the headline line must still be printed."""
    keep = ("metric", "value", "unit", "ms_per_step", "gpu_launches", "l2", "options", "clocks", "roofline", "e2e", "energy")
    others = {}

    def add(name, ow, steps, **kw):
        try:
            r = run_workload(ow, steps, 3, None, fp64_peak=peak, **kw)
            others[name] = {k: r[k] for k in keep if k in r}
            others[name]["steps"] = steps
            roof = r.get("roofline") or {}
            print(json.dumps({"other": name, "value": _short(r["value"]), "unit": r["unit"], "ms_per_step": _short(r["ms_per_step"]),
                              "kernel": roof.get("kernel"), "frac": _short(roof.get("frac"))}), file=sys.stderr)
        except Exception as exc:      # noqa: BLE001 — recorded in the side file
            others[name] = {"error": "%s: %s" % (type(exc).__name__, exc)}
            print(json.dumps({"other": name, "error": others[name]["error"]}), file=sys.stderr)

    for key in ("ring_16k", "grav2d_64k", "hmf_5e7", "grav2d_1m", "hmf_1e4"):
        if key == w.key:
            continue
        add(key, inputs.WORKLOADS[key], DEFAULT_STEPS[key], with_e2e=(key != "grav2d_1m"), roofline_steps=(3 if key == "grav2d_1m" else 2000))
    # HMF at the sizes of the paper's Table 1 that lie between configs 1 and 4
    for key, ow in inputs.TABLE1_WORKLOADS.items():
        if key != w.key:
            add(key, ow, DEFAULT_STEPS[key], with_e2e=False)
    # pair-model sizes of the paper's Tables 2 and 3 beyond the configs
    for key, ow in inputs.TABLE23_WORKLOADS.items():
        if key != w.key:
            add(key, ow, DEFAULT_STEPS[key], with_e2e=False, roofline_steps=3)
    for key, sec in inputs.PAPER_SECONDS_PER_STEP.items():
        if key in others:
            others[key]["paper_seconds_per_step_one_gk104"] = sec      # PAPER.md Tables 1-3: context, other hardware
    # the paper's own scheme, every ORDERED pair, on the configs where a symmetric kernel is the default
    for key in ("ring_16k", "grav2d_64k", "grav2d_1m"):
        steps = 3 if key == "grav2d_1m" else DEFAULT_STEPS[key]
        add(key + "_ordered_pairs", inputs.WORKLOADS[key], steps, with_e2e=False, ordered_pairs=True, with_energy=(key != "grav2d_1m"),
            roofline_steps=3 if key == "grav2d_1m" else 2000)
    # config 5's optional variant: fp32 pair arithmetic, fp64 accumulation across chunks
    add("grav2d_1m_f32pairs", inputs.WORKLOADS["grav2d_1m"], DEFAULT_STEPS["grav2d_1m"], with_e2e=False, f32_pairs=True, roofline_steps=3,
        with_energy=False)
    add("grav2d_1m_f32pairs_ordered_pairs", inputs.WORKLOADS["grav2d_1m"], 3, with_e2e=False, f32_pairs=True, ordered_pairs=True,
        roofline_steps=3, with_energy=False)
    add("ring_16k_f32pairs", inputs.WORKLOADS["ring_16k"], DEFAULT_STEPS["ring_16k"], with_e2e=False, f32_pairs=True)
    for key, what in (("grav2d_1m_f32pairs", "f32 pair terms, f64 state and accumulation"),
                      ("ring_16k_f32pairs", "f32 pair terms (half-angle form), f64 state and accumulation")):
        if "error" not in others.get(key, {"error": 1}):
            others[key]["dtype"] = what
    return others


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--workload", default="grav2d_1m")
    ap.add_argument("--only", action="store_true", help="primary workload only (no 'others', no cpu_baseline)")
    ap.add_argument("--no-others", action="store_true", help="headline with cpu_baseline, without the other entries")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--f32-pairs", action="store_true", help="pair workloads: fp32 pair arithmetic (PAPER.md:110, 136)")
    ap.add_argument("--fp64-peak", action="store_true", help="run only the FP64 issue-rate microbenchmark and print its table")
    ap.add_argument("--ordered-pairs", action="store_true", help="pair workloads: the paper's scheme, every ordered pair (PAPER.md:108)")
    ap.add_argument("--sharded", action="store_true",
                    help="strong scaling through ShardedContext (lrmd_set_shard + NCCL collectives) instead of replicas")
    args = ap.parse_args()

    if args.fp64_peak:
        import torch
        from paper_1212_0262_b200 import lrmd
        if not torch.cuda.is_available():
            raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
        lrmd.load()
        print(json.dumps(fp64_peak_table()))
        return 0

    from paper_1212_0262_b200 import inputs
    all_workloads = dict(inputs.WORKLOADS, **inputs.TABLE1_WORKLOADS, **inputs.TABLE23_WORKLOADS)
    w = all_workloads[args.workload]
    if args.impl == "reference":
        args.steps = args.steps or 3
        args.warmup = 1 if args.warmup is None else args.warmup
        return run_reference(args, w)

    K = args.steps or DEFAULT_STEPS[w.key]
    W = max(3, args.warmup if args.warmup is not None else 3)

    import torch
    from paper_1212_0262_b200 import lrmd
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    lrmd.load()

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local_rank)
    dist_ctx = None
    if world > 1:
        import torch.distributed as dist
        if args.sharded:
            os.environ.setdefault("NCCL_DEBUG", "INFO")     # the communicator's rank count shows in the log
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        dist_ctx = dist

    if args.sharded:
        line = run_sharded(w, K, W, dist_ctx, world, rank)
        if rank == 0:
            print(json.dumps(line))
        if dist_ctx is not None:
            dist_ctx.barrier()
            dist_ctx.destroy_process_group()
        return 0

    f32 = bool(args.f32_pairs and w.model != 0)
    peak = fp64_peak_summary() if (w.model != 0 and not f32) else None
    # the roofline pass and the end-to-end call repeat the steps: bounded for the seconds-long steps of config 5
    heavy = w.key == "grav2d_1m"
    res = run_workload(w, K, W, dist_ctx, f32_pairs=f32, ordered_pairs=bool(args.ordered_pairs and w.model != 0),
                       roofline_steps=(3 if heavy else 2000), e2e_steps=(2 if heavy else 20), fp64_peak=peak)
    line = {
        "metric": res["metric"], "value": res["value"], "unit": res["unit"], "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": res["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if f32 else "f64", "data": "synthetic",
        "config": workload_config(w, world, l2=res["l2"]), "options": res["options"],
        "clocks": res["clocks"], "e2e": res.get("e2e"), "gpu_launches": res["gpu_launches"],
        "roofline": res.get("roofline"), "energy": res.get("energy"),
    }

    others = None
    if world == 1 and not args.only:
        rate, desc, threads = oracle_sample_rate(w, args.cpu_seconds)
        line["cpu_baseline"] = {"value": rate, "unit": res["unit"], "cores": threads, "kind": "oracle", "sample": desc}
        if not args.no_others:
            others = run_others(w, inputs, peak)

    if rank == 0:
        if others is not None:
            line["others_file"] = write_others(others, line)
        print(json.dumps(headline(line)))
    if dist_ctx is not None:
        dist_ctx.barrier()
        dist_ctx.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
