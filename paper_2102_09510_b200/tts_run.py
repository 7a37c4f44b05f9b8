"""TTS accounting runs (SURVEY.md 8(a) a-12, 8(d) "TTS percentiles as the paper defines").

    python -m paper_2102_09510_b200.tts_run --n 128 --words 64 --instances 256 --runs 16 --cap 200000

For every instance (graph seed) R independent runs (different run seeds: "running
the QG algorithm 1008 times") are put into one batch of instances x runs entries; the batch is
advanced K sweeps per call (L293: ~100) until every entry is solved or the cap (timeout t_max,
L129) is reached; entries that already have a solved clone are skipped by the library.  Per
instance: tau_hat, model and empirical TTS_50/90/99, posterior quantiles (xs_tts_stats).  Over
instances: the median of TTS_99 (the competition's figure) and the median tau.  Times are
reported in sweeps (hardware free) and in seconds = sweeps x measured seconds per sweep of a run
of this batch shape.  Only marshals calls into the C ABI; prints one JSON line per size.
"""
from __future__ import annotations

import argparse
import json
import math
import time

import numpy as np


def run_size(n, words, instances, runs, cap, chunk, seed0, flags_extra=0, w1=None):
    import torch
    import paper_2102_09510_b200 as xs
    gseeds = [seed0 + i for i in range(instances) for _ in range(runs)]
    rseeds = [seed0 + i + 7919 * (r + 1) for i in range(instances) for r in range(runs)]
    thr = xs.XS_W1_THRESHOLD_DEFAULT if w1 is None else int(math.floor(w1 * 2.0 ** 32))
    b = xs.Batch(n, words, gseeds, rseeds, flags=xs.XS_FLAG_GAUGE | flags_extra, w1_threshold=thr)
    lay = b.layout()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    done = 0
    gpu_ms = 0.0
    t0 = time.time()
    unsolved_sweeps = 0.0
    while done < cap:
        k = min(chunk, cap - done)
        recs_before = b.tts()
        active = sum(1 for r in recs_before if not r.solved)
        if active == 0:
            break
        ev0.record()
        b.run_sweeps(k)
        ev1.record()
        torch.cuda.synchronize()
        gpu_ms += ev0.elapsed_time(ev1)
        unsolved_sweeps += active * k
        done += k
    recs = b.tts()
    tts = np.array([r.tts_sweeps for r in recs], dtype=np.uint32).reshape(instances, runs)
    clones = 64 * words
    sec_per_sweep = (gpu_ms * 1e-3) / max(unsolved_sweeps, 1.0)      # per batch entry
    per_inst = [xs.xs_tts_stats(tts[i], cap) for i in range(instances)]
    taus = np.array([s["tau_hat"] for s in per_inst])
    tts99 = np.array([s["tts99_model"] for s in per_inst])
    n_solved_runs = int((tts != xs.XS_NO_HIT).sum())
    # PAPER.md Eq. (2), Fig. 2: P[TTS > t] = exp(-t / tau).  Per instance with all runs solved:
    # Kolmogorov-Smirnov distance between the empirical distribution of the R TTS values and
    # 1 - exp(-t / tau_hat), and the empirical / model ratios of TTS_50 and TTS_99 (Fig. 3).
    ks, r50, r99, ks_shift, t_min_over_tau = [], [], [], [], []
    for i in range(instances):
        if per_inst[i]["n_solved"] < runs or runs < 8:
            continue
        v = np.sort(tts[i].astype(np.float64))
        cdf = 1.0 - np.exp(-v / per_inst[i]["tau_hat"])
        k = np.arange(1, runs + 1) / runs
        ks.append(float(max(np.max(k - cdf), np.max(cdf - (k - 1.0 / runs)))))
        # same with an onset time: no clone can hit before the initial relaxation, so at finite
        # tau the law is exp(-(t - t_on) / (tau - t_on)); t_on estimated by the smallest TTS
        t_on = v[0] - (v.mean() - v[0]) / runs
        cdf_s = 1.0 - np.exp(-np.maximum(v - t_on, 0.0) / (v.mean() - t_on))
        ks_shift.append(float(max(np.max(k - cdf_s), np.max(cdf_s - (k - 1.0 / runs)))))
        t_min_over_tau.append(float(t_on / v.mean()))
        r50.append(per_inst[i]["tts50_emp"] / per_inst[i]["tts50_model"])
        r99.append(per_inst[i]["tts99_emp"] / per_inst[i]["tts99_model"])
    # KS critical value at 1 % for a fully specified law is 1.63 / sqrt(R); with tau estimated
    # from the same data (Lilliefors, exponential) it is about 1.25 / sqrt(R)
    ks_crit = 1.25 / math.sqrt(runs) if runs else None
    solved_inst = int(sum(1 for s in per_inst if s["n_solved"] > 0))
    med = lambda a: float(np.median(a)) if np.isfinite(np.median(a)) else None   # noqa: E731
    lower = [s["tau_q16"] for s in per_inst if s["n_solved"] == 0]
    out = {
        "n_spins": n, "w1": (thr / 2.0 ** 32), "clones": clones, "instances": instances, "runs_per_instance": runs,
        "cap_sweeps": cap, "chunk": chunk, "regime": lay.regime, "tile_words": lay.tile_words,
        "solved_runs": n_solved_runs, "total_runs": instances * runs, "instances_with_a_solved_run": solved_inst,
        "median_tau_sweeps": med(taus), "median_tts99_sweeps": med(tts99),
        "median_tts50_sweeps": med(np.array([s["tts50_model"] for s in per_inst])),
        "median_tts90_sweeps": med(np.array([s["tts90_model"] for s in per_inst])),
        "p90_over_instances_tau_sweeps": float(np.percentile(taus, 90)) if np.isfinite(np.percentile(taus, 90)) else None,
        "hardest_decile_median_tts_sweeps": (float(np.median(np.sort(taus)[-max(1, instances // 10):]) * math.log(2))
                                             if np.isfinite(taus).all() else None),
        "tau_lower_bound_95_if_unsolved_sweeps": float(np.median(lower)) if lower else None,
        "single_clone_t0_clone_sweeps": (med(taus) * clones) if med(taus) else None,
        "sec_per_sweep_per_run": sec_per_sweep,
        "median_tts99_seconds": (med(tts99) * sec_per_sweep) if med(tts99) else None,
        "updates_per_ns": n * clones * unsolved_sweeps / max(gpu_ms * 1e6, 1e-9),
        "survival_ks_median": float(np.median(ks)) if ks else None,
        "survival_ks_max": float(np.max(ks)) if ks else None,
        "survival_ks_crit_1pct": ks_crit,
        "survival_ks_fraction_below_crit": float(np.mean(np.array(ks) < ks_crit)) if ks else None,
        "survival_ks_with_onset_median": float(np.median(ks_shift)) if ks_shift else None,
        "survival_ks_with_onset_fraction_below_crit": float(np.mean(np.array(ks_shift) < ks_crit)) if ks_shift else None,
        "onset_over_tau_median": float(np.median(t_min_over_tau)) if t_min_over_tau else None,
        "tts50_emp_over_model_median": float(np.median(r50)) if r50 else None,
        "tts99_emp_over_model_median": float(np.median(r99)) if r99 else None,
        "gpu_ms": gpu_ms, "wall_s": time.time() - t0,
    }
    b.close()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, nargs="+", default=[128])
    ap.add_argument("--words", type=int, default=64)
    ap.add_argument("--instances", type=int, default=256)
    ap.add_argument("--runs", type=int, default=16)
    ap.add_argument("--cap", type=int, default=200000)
    ap.add_argument("--chunk", type=int, default=100)
    ap.add_argument("--seed0", type=int, default=100)
    ap.add_argument("--balanced", action="store_true",
                    help="update order = 4 balanced independent sets (XS_FLAG_BALANCED) instead of the greedy sets")
    ap.add_argument("--clone-noise", action="store_true",
                    help="SURVEY.md 8(f) NEXT-2: an independent random number per clone (w1 = m/128, m = round(128 w1)) "
                         "instead of one per word (PAPER.md L87)")
    ap.add_argument("--w1", type=float, nargs="*", default=None,
                    help="scan of w1 (PAPER.md Fig. 1, L91/L101: optimum 0.054(1)); default 0.055")
    args = ap.parse_args()
    rows = []
    for n in args.n:
        for w1 in (args.w1 or [None]):
            import paper_2102_09510_b200 as xs
            fx = (xs.XS_FLAG_BALANCED if args.balanced else 0) | (xs.XS_FLAG_CLONE_NOISE if args.clone_noise else 0)
            r = run_size(n, args.words, args.instances, args.runs, args.cap, args.chunk, args.seed0,
                         flags_extra=fx, w1=w1)
            r["update_order"] = "balanced" if args.balanced else "greedy"
            r["noise"] = "per clone" if args.clone_noise else "per word"

            rows.append(r)
            print(json.dumps(r), flush=True)
    if args.w1:
        best = min((r for r in rows if r["median_tau_sweeps"]), key=lambda r: r["median_tau_sweeps"])
        print(json.dumps({"w1_scan": [[round(r["w1"], 4), r["median_tau_sweeps"]] for r in rows],
                          "best_w1": best["w1"], "paper_optimum": "0.054(1), instance #38, N=256"}), flush=True)
        return
    # exponential growth of the typical time with N (L151: TTS_99 ~ exp(a N), a = 0.0786(4))
    pts = [(r["n_spins"], math.log(r["median_tau_sweeps"] * r["clones"])) for r in rows
           if r["median_tau_sweeps"]]
    if len(pts) >= 2:
        xs_, ys_ = np.array([p[0] for p in pts], float), np.array([p[1] for p in pts], float)
        a, c = np.polyfit(xs_, ys_, 1)
        print(json.dumps({"fit": "ln(t0) = a N + c over solved sizes", "a": float(a), "c": float(c),
                          "sizes": [p[0] for p in pts], "paper_a": 0.0786}), flush=True)


if __name__ == "__main__":
    main()
