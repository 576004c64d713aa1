"""Search-quality experiment in the spirit of the paper's Fig. 5: how much of
the exhaustive search's bandwidth do the heuristics reach when only the best-ranked 1, 10 or
100 candidates are timed?

The paper's own 57-case benchmark is referenced only by URL and is not
reproduced; this sweep draws 57 seeded random cases of the same shape: rank 2..6, about 200 MB
per tensor, a random non-identity permutation, beta != 0 (Eq. 2's factor 3), fp32 and fp64.

    python -m paper_1607_01249_b200.search_quality [--cases 57] [--out report.md]

Needs a B200 (or any CUDA device); everything timed runs in libttc.so.
"""
from __future__ import annotations

import argparse
import os
import statistics
import sys

import numpy as np

os.environ.setdefault("TTC_TUNE", "0")          # plans are tuned explicitly below

from . import ttc                                # noqa: E402


def draw_case(rng: np.random.Generator, target_bytes: int = 200 << 20):
    n = int(rng.integers(2, 7))
    dtype = ttc.TTC_F32 if rng.integers(0, 2) == 0 else ttc.TTC_F64
    es = 4 if dtype == ttc.TTC_F32 else 8
    total = target_bytes // es
    while True:
        w = rng.uniform(0.5, 1.5, n)
        logs = w / w.sum() * np.log(total)
        sizes = [max(2, int(round(float(np.exp(x))))) for x in logs]
        if all(s >= 4 for s in sizes):
            break
    while True:
        perm = [int(p) for p in rng.permutation(n)]
        if perm != list(range(n)):
            break
    return dtype, sizes, perm


def time_selected(torch, plan, dtype, a_dev, b_dev, flush, reps=5) -> float:
    """Median device time (us) of the plan's current beta != 0 choice, L2 evicted before each run by a READ
    sweep of a 256 MB buffer (clean lines; a memset would leave dirty lines whose write-back the timed kernel pays)."""
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ts = []
    for _ in range(reps + 1):
        flush.max()
        e0.record()
        ttc.ttc_execute(plan, 1.5, a_dev, 0.5, b_dev)
        e1.record()
        e1.synchronize()
        ts.append(e0.elapsed_time(e1) * 1e3)
    return statistics.median(ts[1:])


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--cases", type=int, default=57)
    ap.add_argument("--seed", type=int, default=160701249)
    ap.add_argument("--out", default=None)
    args = ap.parse_args()
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("search_quality: needs a CUDA device")
    rng = np.random.default_rng(args.seed)
    flush = torch.zeros(64 << 20, dtype=torch.int32, device="cuda")
    levels = [1, 10, 32, 0]                      # 0 = every candidate; 32 = the library's default search depth
    rows = []
    for c in range(args.cases):
        dtype, sizes, perm = draw_case(rng)
        es = 4 if dtype == ttc.TTC_F32 else 8
        numel = int(np.prod(sizes, dtype=np.int64))
        tdt = torch.float32 if dtype == ttc.TTC_F32 else torch.float64
        a_dev = torch.rand(numel, dtype=tdt, device="cuda")
        b_dev = torch.rand(numel, dtype=tdt, device="cuda")
        plan = ttc.ttc_plan(dtype, len(sizes), sizes, perm)
        info = ttc.ttc_plan_info(plan)
        gbs = []
        for k in levels:
            if k == 1:
                ttc.ttc_plan_select(plan, 1, 0)  # heuristic top-1, nothing timed
            else:
                ttc.ttc_plan_select(plan, 1, -1)
                ttc.ttc_plan_tune(plan, k, 3)
            us = time_selected(torch, plan, dtype, a_dev, b_dev, flush)
            gbs.append(3 * numel * es / us / 1e3)
        # the exhaustive search's winner re-compiled for this size (ttc_plan_specialize)
        ttc.ttc_plan_specialize(plan)
        us = time_selected(torch, plan, dtype, a_dev, b_dev, flush)
        gbs.append(max(gbs[-1], 3 * numel * es / us / 1e3) if ttc.ttc_plan_info(plan).specialized[1] != 2 else 3 * numel * es / us / 1e3)
        rows.append((sizes, perm, "f32" if es == 4 else "f64", info.canon_rank, info.n_candidates[1], gbs))
        ttc.ttc_destroy(plan)
        del a_dev, b_dev
        print("case %2d %s %-28s perm=%s rank=%d cands=%d  GB/s top1=%.0f top10=%.0f top32=%.0f all=%.0f" % (
            c, rows[-1][2], "x".join(map(str, sizes)), "".join(map(str, perm)), info.canon_rank,
            info.n_candidates[1], *gbs[:4]), file=sys.stderr, flush=True)
    out = ["# Search quality on B200: bandwidth reached when only the k best-ranked candidates are timed", "",
           "`python -m paper_1607_01249_b200.search_quality --cases %d --seed %d`; %d seeded random cases, ~200 MB per tensor, "
           "beta != 0, GB/s = 3*|A|*sizeof / time (L2 evicted by a 256 MB read sweep before every run, median of 5); top-32 is the "
           "library's default search depth." % (args.cases, args.seed, args.cases), "",
           "| # | dtype | sizes | perm | canon. rank | candidates | top-1 | top-10 | top-32 | all | all, size-specialised | top-1 / all | top-10 / all |",
           "|---|---|---|---|---|---|---|---|---|---|---|---|---|"]
    for i, (sizes, perm, dt, cr, nc, g) in enumerate(rows):
        best = max(g[:4])
        out.append("| %d | %s | %s | %s | %d | %d | %.0f | %.0f | %.0f | %.0f | %.0f | %.3f | %.3f |" % (
            i, dt, "x".join(map(str, sizes)), "".join(map(str, perm)), cr, nc, g[0], g[1], g[2], g[3], g[4], g[0] / best, g[1] / best))
    def col(j):
        return [r[5][j] for r in rows]
    out += ["", "| | top-1 | top-10 | top-32 | all | all, size-specialised |", "|---|---|---|---|---|---|",
            "| mean GB/s | %.0f | %.0f | %.0f | %.0f | %.0f |" % tuple(statistics.mean(col(j)) for j in range(5)),
            "| min GB/s | %.0f | %.0f | %.0f | %.0f | %.0f |" % tuple(min(col(j)) for j in range(5)),
            "| mean fraction of the case's best generic | %.3f | %.3f | %.3f | %.3f | %.3f |" % tuple(
                statistics.mean(r[5][j] / max(r[5][:4]) for r in rows) for j in range(5))]
    text = "\n".join(out) + "\n"
    if args.out:
        with open(args.out, "w") as fh:
            fh.write(text)
    print(text)


if __name__ == "__main__":
    main()
