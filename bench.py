#!/usr/bin/env python
"""bench.py -- clone-spin updates/ns of the quasi-greedy sweep on BASELINE.json configs[1].

A step = one pass of the hot path over the workload: xs_run_sweeps(10^4 sweeps) on N=256,
2^16 clones (a-3..a-10 + termination of a-11), then xs_energy (a-11) and xs_tts (a-12).
`value`: inputs resident in HBM, device time of the step (CUDA events).  `e2e`: the same step
through the C ABI with HOST buffers: initial spin words uploaded from pinned host memory
(xs_set_spins), results (energies, spin words, TTS records) read back, copies inside the timed
region.  `roofline`: integer-pipe (LOP3) roofline of the sweep kernel, the dominant kernel.
`cpu_baseline` / `--impl reference`: the CPU oracle (oracle/) on a bounded sample of the same
workload on this box's host cores.

The default run appends to the headline line a `workloads` map (short measurements of the other
BASELINE.json configs: value / e2e / roofline.frac / clocks each) and a `tts` block (the second
half of BASELINE.json's metric: N=128 percentiles and the censored N=512 bound); `--no-extras`
skips both, `--workload NAME` makes another workload the headline.

Multi-GPU (`torchrun ... bench.py --gpus N`): replicas only -- every rank runs the same
workload with its own run seed ("multiple GPUs ... executing the same code with
different random seeds"); no data-path collective; value = sum of updates / max time.
"""
from __future__ import annotations

import argparse
import csv
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

# BASELINE.json configs[1]
WORKLOADS = {
    # balanced independent sets of 64 = the slot count of the clause-word kernel's CTA (DESIGN.md R-balance)
    "config2": dict(N=256, W=1024, I=1, sweeps=10_000, graph_seed=2, run_seed=2, balanced=True, set_cap=64,
                    desc="configs[1]: N=256, 1 instance (graph seed 2), 2^16 clones, 10^4 sweeps, no early stop; "
                         "update order = 4 balanced independent sets of 64"),
    "config2_greedy": dict(N=256, W=1024, I=1, sweeps=10_000, graph_seed=2, run_seed=2,
                           desc="configs[1] with the uncapped greedy sets (61,62,59,50,23,1): N=256, 1 instance "
                                "(graph seed 2), 2^16 clones, 10^4 sweeps, no early stop"),
    # the paper's own order: greedy sets capped at 32 spins
    "config2_cap32": dict(N=256, W=1024, I=1, sweeps=2_000, graph_seed=2, run_seed=2, set_cap=32,
                          desc="configs[1] with the paper's cap-32 greedy sets (L279): N=256, 1 instance (graph seed 2), "
                               "2^16 clones, 2000 sweeps per step"),
    # Metropolis table w0 = w1^3 at T_run on the config-2 workload
    "config2_metropolis": dict(N=256, W=1024, I=1, sweeps=1_000, graph_seed=2, run_seed=2, balanced=True, set_cap=64,
                               metropolis=True,
                               desc="configs[1] with the Metropolis table w0 = w1^3, w2 = w3 = 1 (L69) at w1 = 0.055: N=256, "
                                    "2^16 clones, 1000 sweeps per step, first hits looked for after every sweep (clause-word kernel, W0 form)"),
    # SURVEY.md 8(f) NEXT-2 on chip: per-clone noise on the config-2 workload (clause-word kernel, PCN form)
    "config2_clone_noise": dict(N=256, W=1024, I=1, sweeps=500, graph_seed=2, run_seed=2, balanced=True, set_cap=64,
                                clone_noise=True,
                                desc="configs[1] with per-clone noise (XS_FLAG_CLONE_NOISE, w1 = 7/128): N=256, 2^16 clones, "
                                     "500 sweeps per step (clause-word kernel, 16 x the Philox work)"),
    "config1": dict(N=64, W=1, I=1, sweeps=10_000, graph_seed=1, run_seed=1,
                    desc="configs[0] shape: N=64, 1 instance (graph seed 1), 64 clones, 10^4 sweeps per step, no early stop "
                         "(latency: one warp of work)"),
    "config5": dict(N=1 << 20, W=16, I=1, sweeps=100, graph_seed=5, run_seed=5,
                    desc="configs[4]: N=2^20, 1 instance (graph seed 5), 2^10 clones, 100 sweeps (streaming)"),
    "config3": dict(N=512, W=64, I=256, sweeps=2_000, graph_seed=100, run_seed=100, balanced=True,
                    desc="configs[2] shape: N=512, 256 instances (seeds 100..355), 2^12 clones each, 2000 sweeps per step; "
                         "update order = 4 balanced independent sets of 128"),
    "config3_greedy": dict(N=512, W=64, I=256, sweeps=2_000, graph_seed=100, run_seed=100,
                           desc="configs[2] shape with the uncapped greedy sets: N=512, 256 instances (seeds 100..355), "
                                "2^12 clones each, 2000 sweeps per step"),
    # SURVEY.md F3 / 8(d) "5b": as config 5 with 2^14 clones = 2 GiB of state, DRAM resident
    "config5b": dict(N=1 << 20, W=256, I=1, sweeps=10, graph_seed=5, run_seed=5,
                     desc="config 5b: N=2^20, 1 instance (graph seed 5), 2^14 clones (2 GiB state), 10 sweeps (streaming)"),
    # config 5 with an independent random number per clone (16 x the Philox work)
    "config5_clone_noise": dict(N=1 << 20, W=16, I=1, sweeps=20, graph_seed=5, run_seed=5, clone_noise=True,
                                desc="configs[4] with per-clone noise (XS_FLAG_CLONE_NOISE, w1 = 7/128): N=2^20, 1 instance "
                                     "(graph seed 5), 2^10 clones, 20 sweeps (streaming)"),
}
# configs[3] shapes: 128 instances (graph seeds 1000 N + i), 2^14 clones each
for _n, _s in ((128, 2000), (192, 1500), (256, 1000), (384, 700), (512, 500), (768, 350), (1024, 250)):
    WORKLOADS[f"config4_{_n}"] = dict(N=_n, W=256, I=128, sweeps=_s, graph_seed=1000 * _n, run_seed=1000 * _n,
                                      balanced=True,
                                      desc=f"configs[3] shape: N={_n}, 128 instances, 2^14 clones each, {_s} sweeps "
                                           f"per step; update order = balanced independent sets (DESIGN.md R-balance)")
# what the default run measures after the headline (short runs)
EXTRAS = ["config1", "config2_greedy", "config2_cap32", "config2_metropolis", "config2_clone_noise", "config3", "config3_greedy"] + \
         [f"config4_{n}" for n in (128, 192, 256, 384, 512, 768, 1024)] + ["config5", "config5b"]

# Integer-pipe work per update.
#  - SURVEY.md 8(d) contract: 14 LOP3/IADD lane-ops per 32 clone-spin updates (3 + 2 + 2 update, 2
#    detection per sweep, 5 Philox share) -- the figure `roofline.frac` is quoted on;
#  - the clause-word kernel's own count: 7 update + 2.5 Philox XORs + 1 compare / mask per 32
#    updates, detection amortised over the 256-sweep batch: what the method needs in this form.
ALU_OPS_PER_UPDATE = 14.0 / 32.0
ALU_OPS_PER_UPDATE_OWN = (28.0 + 10.0 + 4.0) / 128.0 + 12.0 / (256.0 * 128.0)


def ncu_counters(workload: str) -> dict:
    """Counters of the dominant kernel copied from the committed ncu captures (profiles/): rows
    `workload,metric,value,source`.  Absent file or workload: {}."""
    path = os.path.join(ROOT, "profiles", "r02_ncu_counters.csv")
    out = {}
    try:
        with open(path, newline="") as f:
            for row in csv.DictReader(f):
                if row.get("workload") == workload:
                    try:
                        out[row["metric"]] = float(row["value"])
                    except ValueError:
                        out[row["metric"]] = row["value"]
    except OSError:
        pass
    return out


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
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
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "50",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [c.strip() for c in line.split(",")]))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.06)
        self.proc.terminate()
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 + 0.06] or [r for (_, r) in self.rows]
        sm, mx, reasons = [], [], set()
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"], r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def energy_histogram(e):
    """Final energy histogram over all clones (north_star: configs[1] reports it): [[E, count], ...]
    over the distinct values, or 32 equal-width bins [[E_lo, E_hi, count], ...] if there are many."""
    vals, cnt = np.unique(e, return_counts=True)
    if vals.size <= 96:
        return [[int(v), int(c)] for v, c in zip(vals, cnt)]
    h, edges = np.histogram(e, bins=32)
    return [[int(edges[i]), int(edges[i + 1]), int(h[i])] for i in range(32)]


def metropolis_table(w1: float = 0.055):
    """w0 = w1^3, w2 = w3 = 1 (detailed balance at T = -2 / ln w1), as thresholds."""
    two32 = 1 << 32
    return [int(w1 ** 3 * two32), int(w1 * two32), two32, two32]


def cpu_oracle_rate(wl, target_s: float = 20.0):
    """The oracle as it stands, OpenMP over words, on a bounded sample of the workload."""
    from oracle.xs_oracle import NO_HIT, Instance, omp_threads
    cores = omp_threads()
    N = wl["N"]
    inst = Instance(N, wl["graph_seed"], True, wl.get("set_cap", 0), balanced=bool(wl.get("balanced")))
    clone_m = 7 if wl.get("clone_noise") else None          # the variant's oracle is single threaded
    thr4 = metropolis_table() if wl.get("metropolis") else None
    if clone_m is not None or thr4 is not None:
        cores = 1
    W = max(1, min(wl["W"], 4 * cores))      # enough words for ~target_s of work on all cores
    s = inst.init_spins(W, wl["run_seed"])
    fh = np.full(64 * W, NO_HIT, np.uint32)
    t0 = time.perf_counter()
    inst.run(s, fh, wl["run_seed"], 0, 1, omp=True, clone_m=clone_m, thr4=thr4)         # calibration sweep
    dt1 = max(time.perf_counter() - t0, 1e-6)
    sweeps = int(max(1, min(wl["sweeps"], target_s / dt1)))
    t0 = time.perf_counter()
    inst.run(s, fh, wl["run_seed"], 1, sweeps, omp=True, clone_m=clone_m, thr4=thr4)
    dt = time.perf_counter() - t0
    rate = N * 64.0 * W * sweeps / (dt * 1e9)
    return {"value": rate, "unit": "clone-spin updates/ns", "cores": cores, "kind": "oracle",
            "sample": f"N={N}, {W} of {wl['W']} words (64 clones each), {sweeps} sweeps, "
                      f"{dt:.1f} s wall, OpenMP over words"}, dt


def run_reference(args, wl, rank):
    """--impl reference: the oracle arm (tier rule: the reference arm is the oracle, rank 0 only)."""
    if rank != 0:
        return
    per_step = []
    cb = None
    target = max(2.0, min(20.0, 150.0 / max(1, args.steps + args.warmup)))
    for it in range(args.warmup + args.steps):
        cb, dt = cpu_oracle_rate(wl, target_s=target)
        if it >= args.warmup:
            per_step.append((cb["value"], dt))
    val = float(np.mean([v for v, _ in per_step]))
    ms = float(np.mean([d for _, d in per_step])) * 1e3
    cb["value"] = val
    print(json.dumps({
        "impl": "reference", "metric": "clone-spin updates/ns", "value": val, "unit": "clone-spin updates/ns",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int8 (one spin per byte)",
        "data": "synthetic", "config": {"workload": wl["desc"], "sample": cb["sample"]},
        "cpu_baseline": cb,
        "e2e": {"value": val, "unit": "clone-spin updates/ns", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}), flush=True)


def measure(name, wl, steps, warmup, ctx, with_e2e=True):
    """One workload on this rank's GPU: `warmup` untimed steps, then `steps` timed device-resident
    steps (L2 flushed between them) and, with_e2e, the same number of end-to-end steps.
    Returns a dict of raw results; rank 0 turns it into JSON."""
    import torch
    import paper_2102_09510_b200 as xs
    from paper_2102_09510_b200 import replicas
    dev, dist, rank, world = ctx["dev"], ctx["dist"], ctx["rank"], ctx["world"]
    N, W, I, sweeps = wl["N"], wl["W"], wl["I"], wl["sweeps"]
    gseeds = [wl["graph_seed"] + i for i in range(I)]
    rseeds = replicas.replica_run_seeds([wl["run_seed"] + i for i in range(I)], rank)   # replicas (L87)
    flags = xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP | (xs.XS_FLAG_BALANCED if wl.get("balanced") else 0) | \
        (xs.XS_FLAG_CLONE_NOISE if wl.get("clone_noise") else 0)
    b = xs.Batch(N, W, gseeds, rseeds, set_cap=wl.get("set_cap", 0), flags=flags, device=dev)
    if wl.get("metropolis"):
        b.set_flip_table(metropolis_table())
    lay = b.layout()
    updates_per_step = float(N) * 64.0 * W * I * sweeps
    flush = ctx["flush"]

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def mk():
        return [torch.cuda.Event(enable_timing=True) for _ in range(3)]

    def dev_step(ev):
        """device-resident step; ev = (start, after_sweeps, end) events"""
        ev[0].record()
        b.run_sweeps(sweeps)
        ev[1].record()
        e = b.energy()
        recs = b.tts()              # synchronises the stream
        ev[2].record()
        return e, recs

    for _ in range(max(warmup, 3)):
        flush.fill_(1)
        dev_step(mk())
    launches0 = xs.xs_kernel_launches()
    sampler = ClockSampler(ctx["local_rank"])
    sampler.start()
    time.sleep(0.12)
    barrier()
    t_wall0 = time.time()
    evs = []
    for _ in range(steps):
        flush.fill_(1)                  # L2 flush between timed iterations (outside the event pairs)
        ev = mk()
        e_last, recs = dev_step(ev)
        evs.append(ev)
    barrier()
    t_wall1 = time.time()
    clocks = sampler.stop(t_wall0, t_wall1)
    launches = xs.xs_kernel_launches() - launches0
    step_ms = [ev[0].elapsed_time(ev[2]) for ev in evs]
    sweep_ms = [ev[0].elapsed_time(ev[1]) for ev in evs]
    total_ms = float(sum(step_ms))
    e_np = e_last.cpu().numpy()
    del e_last

    # e2e: host buffers, copies inside the timed region
    e2e_ms, h2d, d2h = None, 0, 0
    if with_e2e:
        x0_host = torch.from_numpy(b.spins_numpy().view(np.int64).copy()).pin_memory()
        x_dev = torch.empty_like(x0_host, device=dev)
        e_host = torch.empty((I, 64 * W), dtype=torch.int32).pin_memory()
        x_host = torch.empty_like(x0_host).pin_memory()
        h2d = x0_host.numel() * 8
        d2h = e_host.numel() * 4 + x_host.numel() * 8 + I * 24

        def e2e_step(ev):
            ev[0].record()
            x_dev.copy_(x0_host, non_blocking=True)
            b.set_spins(x_dev)
            b.run_sweeps(sweeps)
            e = b.energy()
            e_host.copy_(e, non_blocking=True)
            x_host.copy_(b.get_spins(), non_blocking=True)
            r = b.tts()
            ev[2].record()
            return r

        for _ in range(2):
            e2e_step(mk())
        barrier()
        evs2 = []
        for _ in range(steps):
            flush.fill_(1)
            ev = mk()
            e2e_step(ev)
            evs2.append(ev)
        barrier()
        e2e_ms = float(sum(ev[0].elapsed_time(ev[2]) for ev in evs2))
        del x0_host, x_dev, e_host, x_host
    tot = replicas.max_over_ranks([total_ms, e2e_ms if e2e_ms is not None else 0.0], dist, dev)   # max over ranks
    out = dict(name=name, wl=wl, lay=lay, steps=steps, warmup=max(warmup, 3), updates_per_step=updates_per_step,
               total_ms=tot[0], e2e_ms=tot[1] if with_e2e else None, kernel_ms=float(np.mean(sweep_ms)),
               clocks=clocks, launches=int(launches), e_np=e_np, recs=list(recs), h2d=h2d, d2h=d2h,
               value=replicas.job_rate(updates_per_step, steps, world, tot[0]),
               e2e_value=replicas.job_rate(updates_per_step, steps, world, tot[1]) if with_e2e else None)
    b.close()
    del b
    torch.cuda.empty_cache()
    return out


def roofline_of(m, alu_peak, peaks, sms=148):
    """The `roofline` object of a measured workload (dominant kernel = the sweep kernel)."""
    wl, lay, k_ms, ups, clocks = m["wl"], m["lay"], m["kernel_ms"], m["updates_per_step"], m["clocks"]
    N, W = wl["N"], wl["W"]
    ncu = ncu_counters(m["name"])
    if lay.regime == 0:
        achieved = ALU_OPS_PER_UPDATE * ups / (k_ms * 1e6) / 1e3      # Tlop/s
        kname = {1: "k_sweep_static", 2: "k_sweep_clause", 3: "k_sweep_warp"}.get(lay.variant, "k_sweep_tile")
        roof = {"bound": "alu", "achieved": achieved, "peak": alu_peak / 1e3, "unit": "Tlop/s (32-bit LOP3/IADD lane-ops)",
                "frac": achieved / (alu_peak / 1e3), "traffic": ncu.get("dram_bytes_per_launch"),
                "peak_source": "xs_alu_peak LOP3 micro-kernel measured in this run",
                "peak_nominal_at_sampled_clock": (sms * 64 * clocks["sm_mhz"] / 1e6) if clocks.get("sm_mhz") else None,
                "alg_ops_per_update": ALU_OPS_PER_UPDATE,
                "alg_ops_model": "SURVEY.md 8(d): 14 lane-ops per 32 updates (algorithmic model, not pipe occupancy)",
                "kernel": kname, "kernel_ms": k_ms}
        if lay.variant == 2:
            # the kernel's own count: what this form of the method must execute
            own = ALU_OPS_PER_UPDATE_OWN * ups / (k_ms * 1e6) / 1e3
            roof["alg_ops_per_update_own"] = ALU_OPS_PER_UPDATE_OWN
            roof["frac_own"] = own / (alu_peak / 1e3)
        # measured pipe use of the same command under ncu (profiles/r02_ncu_counters.csv)
        for key in ("alu_pipe_pct", "fma_pipe_pct", "smem_wavefront_pct", "issue_active_pct",
                    "executed_alu_ops_per_update", "inst_per_warp_task"):
            if key in ncu:
                roof[key] = ncu[key]
        if "executed_alu_ops_per_update" in ncu and lay.variant == 2:
            roof["alu_overhead_ratio"] = ncu["executed_alu_ops_per_update"] / ALU_OPS_PER_UPDATE_OWN
        # co-limiter: shared-memory pipe, 128 B/clk/SM.  Bytes the kernel's layout
        # moves per update: clause-word kernel 3 loads + 3 stores of 16 B per 128 updates; static
        # kernel 6 loads + NC stores (T = 8: two row copies, T = 4: four); generic kernel 11 accesses.
        n_copies = 16 // lay.tile_words if lay.tile_words <= 16 else 1
        sm_bpu = {1: (6 + n_copies) * 16 / 128.0, 2: 6 * 16 / 128.0}.get(lay.variant, 11 * 16 / 128.0)
        if clocks.get("sm_mhz") and lay.variant != 3:
            sm_peak = sms * 128 * clocks["sm_mhz"] / 1e3                          # GB/s
            roof["shared_memory"] = {"bytes_per_update": sm_bpu,
                                     "achieved_gbs": sm_bpu * ups / (k_ms * 1e6),
                                     "peak_gbs": sm_peak,
                                     "frac": sm_bpu * ups / (k_ms * 1e6) / sm_peak}
    else:
        hbm = peaks.get("hbm_gbs", 6650.0)
        bpu = (8 * 8 * W + 28) / (64.0 * W)      # 6 partner rows + own row read + write + record
        achieved = bpu * ups / (k_ms * 1e6)                                           # GB/s
        roof = {"bound": "hbm", "achieved": achieved, "peak": hbm, "unit": "GB/s", "frac": achieved / hbm,
                "traffic": ncu.get("dram_bytes_per_launch"),
                "peak_source": "MEASURED_PEAKS.json hbm_gbs (of measured)" if peaks else "fallback 6650 GB/s",
                "alg_bytes_per_update": bpu, "kernel": "k_stream_set", "kernel_ms": k_ms}
        for key in ("dram_gbs", "dram_pct_of_peak", "l2_hit_rate_pct", "alg_bytes_per_launch"):
            if key in ncu:
                roof[key] = ncu[key]
    return roof


def tts_block():
    """The second half of BASELINE.json's metric ("median & p99 TTS at N=512"), as SURVEY.md 8(d)
    restates it (F2: N = 512 cannot be solved): the censored lower bound at N = 512 and genuine
    percentiles "as the paper defines" (L103-L149) at the solvable size N = 128 (config 3')."""
    from paper_2102_09510_b200 import tts_run
    import paper_2102_09510_b200 as xs
    keep = ("n_spins", "clones", "instances", "runs_per_instance", "cap_sweeps", "solved_runs", "total_runs",
            "instances_with_a_solved_run", "median_tau_sweeps", "median_tts50_sweeps", "median_tts90_sweeps",
            "median_tts99_sweeps", "tau_lower_bound_95_if_unsolved_sweeps", "sec_per_sweep_per_run",
            "median_tts99_seconds", "updates_per_ns", "gpu_ms")
    r128 = tts_run.run_size(128, 64, 256, 16, 200_000, 500, 100, flags_extra=xs.XS_FLAG_BALANCED)
    r512 = tts_run.run_size(512, 64, 256, 1, 100_000, 10_000, 100, flags_extra=xs.XS_FLAG_BALANCED)
    out = {"n128_config3prime": {k: r128[k] for k in keep}, "n512_config3_capped": {k: r512[k] for k in keep}}
    lb = r512["tau_lower_bound_95_if_unsolved_sweeps"]
    if lb:
        # P[TTS > t] = exp(-t / tau) (Eq. (2)): percentile bounds from the 95 % bound on tau
        out["n512_config3_capped"]["median_tts_lower_bound_sweeps"] = float(np.log(2.0) * lb)
        out["n512_config3_capped"]["tts99_lower_bound_sweeps"] = float(-np.log(0.01) * lb)
    out["note"] = ("N=512 with 2^12 clones needs ~1e20 clone-sweeps (SURVEY.md F2): no run solves, so median / p99 TTS "
                   "at N=512 are lower bounds from the censored posterior (L139-L147); DESIGN.md section 7 has the "
                   "10^6-sweep cap run and the 128-instance size sweep")
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config2", choices=sorted(WORKLOADS))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true",
                    help="skip the `workloads` map and the `tts` block (headline workload only)")
    ap.add_argument("--extras", nargs="*", default=None, help="workloads of the `workloads` map (default: all)")
    args = ap.parse_args()
    wl = WORKLOADS[args.workload]
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, wl, rank)
        return

    import torch
    import paper_2102_09510_b200 as xs
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    ctx = dict(dev=dev, dist=dist, rank=rank, local_rank=local_rank, world=world,
               flush=torch.empty(256 << 20, dtype=torch.uint8, device=dev))     # > 126 MB L2
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except OSError:
        pass

    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    m = measure(args.workload, wl, args.steps, args.warmup, ctx)
    alu_peak, _ = xs.xs_alu_peak()
    out = None
    if rank == 0:
        lay, e_np, recs, N = m["lay"], m["e_np"], m["recs"], wl["N"]
        out = {
            "metric": "clone-spin updates/ns", "value": m["value"], "unit": "clone-spin updates/ns", "n_gpus": world,
            "steps": args.steps, "warmup": m["warmup"], "ms_per_step": m["total_ms"] / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u64 bit-sliced (LOP3 on u32)",
            "data": "synthetic",
            "config": {"workload": wl["desc"], "l2": "flushed between timed iterations (256 MiB write)",
                       "regime": "on-chip" if lay.regime == 0 else "streaming", "tile_words": lay.tile_words,
                       "threads": lay.threads, "ctas": lay.ctas, "smem_bytes": lay.smem_bytes, "kernel_variant": lay.variant,
                       "batch_sweeps": lay.batch_sweeps, "n_sets": lay.n_sets_max, "multi_gpu": "replicas only"},
            "clocks": m["clocks"],
            "e2e": {"value": m["e2e_value"], "unit": "clone-spin updates/ns", "h2d_bytes_per_step": m["h2d"],
                    "d2h_bytes_per_step": m["d2h"]},
            "gpu_launches": m["launches"],
            "roofline": roofline_of(m, alu_peak, peaks, sms),
            "energy": {"mean_per_spin": float(e_np.mean() / N), "min": int(e_np.min()), "max": int(e_np.max()),
                       "histogram": energy_histogram(e_np)},
        }
    # ---- the other configs, short runs (every rank runs them: replicas; rank 0 reports) ----------
    extras = not args.no_extras and world == 1      # the scaling runs time the headline workload only
    if extras:
        names = [n for n in (EXTRAS if args.extras is None else args.extras) if n != args.workload]
        wmap = {}
        for name in names:
            w2 = WORKLOADS[name]
            try:
                m2 = measure(name, w2, 3, 3, ctx)
            except Exception as ex:      # a workload that cannot run must not take the headline down
                wmap[name] = {"error": f"{type(ex).__name__}: {ex}"}
                continue
            if rank == 0:
                r2 = roofline_of(m2, alu_peak, peaks, sms)
                l2 = m2["lay"]
                ent = {"value": m2["value"], "e2e": m2["e2e_value"], "ms_per_step": m2["total_ms"] / m2["steps"],
                       "roofline": {k: r2[k] for k in ("bound", "frac", "frac_own", "achieved", "peak", "unit", "kernel",
                                                       "alu_pipe_pct", "smem_wavefront_pct", "dram_gbs", "traffic")
                                    if k in r2},
                       "clocks": m2["clocks"], "gpu_launches": m2["launches"],
                       "geometry": {"regime": l2.regime, "variant": l2.variant, "tile_words": l2.tile_words,
                                    "threads": l2.threads, "ctas": l2.ctas, "n_sets": l2.n_sets_max},
                       "workload": w2["desc"]}
                if name == "config1":
                    ent["sweeps_per_us"] = w2["sweeps"] / (m2["kernel_ms"] * 1e3)
                wmap[name] = ent
        if rank == 0:
            out["workloads"] = wmap
    if rank == 0:
        if extras:
            try:
                out["tts"] = tts_block()
            except Exception as ex:
                out["tts"] = {"error": f"{type(ex).__name__}: {ex}"}
        else:
            recs = m["recs"]
            out["tts"] = {"solved_instances": int(sum(r.solved for r in recs)), "sweeps_done": int(recs[0].sweeps_done)}
        if not args.no_cpu_baseline:
            out["cpu_baseline"], _ = cpu_oracle_rate(wl)
        print(json.dumps(out), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
