"""Re-fit the ranking heuristic of the plan generator (candidates are ranked by a cost
model so that only a few need to be timed) against measured kernel times on the current device.

    python -m paper_1607_01249_b200.fit_cost collect --out samples.jsonl [--cases 40]   # needs a GPU
    python -m paper_1607_01249_b200.fit_cost fit samples.jsonl                          # CPU only

``collect`` times EVERY candidate (the paper's exhaustive mode) of seeded random transpositions shaped like
the paper's benchmark (2-D..6-D, ~200 MB) plus BASELINE.json's configs and writes one JSON
line per case with each candidate's raw features (``ttc_plan_candidate_features``) and time.  ``fit`` runs a
least-squares fit of log(time / ideal time) on a handful of terms built from those features and prints the
C array that ``fitted_tile_cost`` in csrc/plan.cpp holds, together with the ranking quality (how close the
best of the top-k ranked candidates comes to the best of all).  No arithmetic of the method lives here.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys

import numpy as np

TERMS = ["bias", "runA_256", "runB_64", "runA_2048", "runB_512", "log_waste", "log_conflicts", "small_tile", "tile_over_32k",
         "tile_over_16k", "tiles_under_1184", "tiles_under_4736", "ring", "ring4", "cpasync_rows", "shifted_rows", "peel",
         "staggered", "narrow_a", "narrow_b", "narrow_a_4", "narrow_b_4", "beta", "cpasync_short_row", "beta_runB_64",
         "beta_narrow_b", "tile_conflicts", "staggered_conflicts", "gather", "wide"]


def terms(F):
    """Regression terms from the 16 raw features (mirrors fitted_tile_cost in csrc/plan.cpp, same order)."""
    runA, runB, waste, conf, tile_b, n_tiles, ring, rowmode, peel, xp, vab, vbb, beta, kern, row_b, items_b = F
    lc = math.log(max(conf, 1.0))
    na, nb = (1.0 if vab < 16 else 0.0), (1.0 if vbb < 16 else 0.0)
    return np.array([
        1.0,
        math.log1p(256.0 / max(runA, 1.0)), math.log1p(64.0 / max(runB, 1.0)),
        math.log1p(2048.0 / max(runA, 1.0)), math.log1p(512.0 / max(runB, 1.0)),
        math.log(max(waste, 1.0)), lc,
        4096.0 / max(tile_b, 256.0), max(0.0, tile_b - 32768.0) / 65536.0, max(0.0, tile_b - 16384.0) / 65536.0,
        max(0.0, 1.0 - n_tiles / 1184.0), max(0.0, 1.0 - n_tiles / 4736.0),
        1.0 if ring > 0 else 0.0, 1.0 if ring >= 4 else 0.0,
        1.0 if rowmode == 1 else 0.0, 1.0 if rowmode == 2 else 0.0, 1.0 if peel else 0.0, 1.0 if xp else 0.0,
        na, nb, na * (1.0 if vab <= 4 else 0.0), nb * (1.0 if vbb <= 4 else 0.0),
        beta, (1.0 if rowmode == 1 else 0.0) * 128.0 / max(row_b, 16.0), beta * math.log1p(64.0 / max(runB, 1.0)),
        beta * nb, (1.0 if ring == 0 else 0.0) * lc, lc * (1.0 if xp else 0.0),
        1.0 if kern == 3 else 0.0, 1.0 if kern == 4 else 0.0])


def collect(args) -> None:
    os.environ["TTC_TUNE"] = "0"
    import torch
    from . import ttc
    from . import workloads as wl
    from .search_quality import draw_case
    rng = np.random.default_rng(args.seed)
    cases = []
    for w in wl.baseline_configs():
        cases.append((w.dtype, list(w.sizes), list(w.perm), w.lda, w.ldb, 1 if w.beta_nonzero else 0))
    for _ in range(args.cases):
        dtype, sizes, perm = draw_case(rng)
        cases.append((dtype, sizes, perm, None, None, 1))
    with open(args.out, "w") as fh:
        for ci, (dtype, sizes, perm, lda, ldb, which) in enumerate(cases):
            plan = ttc.ttc_plan(dtype, len(sizes), sizes, perm, lda, ldb)
            ttc.ttc_plan_tune(plan, 0, 3)
            info = ttc.ttc_plan_info(plan)
            es = wl.ELEM_SIZE[dtype]
            nbytes = (3 if which else 2) * info.numel * es
            rows = []
            for i in range(info.n_candidates[which]):
                c = ttc.ttc_plan_candidate(plan, which, i)
                if c.tuned_us > 0:
                    rows.append({"i": i, "us": c.tuned_us, "F": ttc.ttc_plan_candidate_features(plan, which, i),
                                 "kernel": c.kernel, "cost": c.est_cost})
            fh.write(json.dumps({"dtype": dtype, "sizes": sizes, "perm": perm, "which": which, "bytes": nbytes,
                                 "cands": rows}) + "\n")
            fh.flush()
            ttc.ttc_destroy(plan)
            print("case %d/%d: %d candidates timed" % (ci + 1, len(cases), len(rows)), file=sys.stderr, flush=True)


def quality(cases, score):
    """Mean over cases of best(top-k by score) / best(all), for k = 1, 10, 32."""
    out = {1: [], 10: [], 32: []}
    for case in cases:
        cands = [c for c in case["cands"] if c["kernel"] != 1]
        if not cands:
            continue
        best = min(c["us"] for c in case["cands"])
        order = sorted(case["cands"], key=score)
        for k in out:
            out[k].append(best / min(c["us"] for c in order[:k]))
    return {k: (float(np.mean(v)), float(np.min(v))) for k, v in out.items()}


def fit(args) -> None:
    cases = [json.loads(ln) for ln in open(args.samples)]
    X, y, wts = [], [], []
    for case in cases:
        ideal = case["bytes"] / 6.5e6                    # us at 6.5 TB/s
        best = min(c["us"] for c in case["cands"])
        for c in case["cands"]:
            if c["kernel"] == 1:
                continue                                   # direct kernels keep their own formula
            X.append(terms(c["F"]))
            y.append(math.log(c["us"] / ideal))
            # the ranking matters near the top: weight candidates by closeness to the case's best
            wts.append((1.0 / (0.10 + c["us"] / best - 1.0)) ** 2)
    X, y, wts = np.array(X), np.array(y), np.sqrt(np.array(wts))
    coef, *_ = np.linalg.lstsq(X * wts[:, None], y * wts, rcond=None)
    res = y - X @ coef
    print("samples %d, rms log error %.3f" % (len(y), float(np.sqrt(np.mean(res ** 2)))))
    for n, c in zip(TERMS, coef):
        print("  %-18s %+.4f" % (n, c))
    print("static const double kCostW[%d] = {%s};" % (len(coef), ", ".join("%.5f" % c for c in coef)))

    # direct candidates are ranked by their own cost; put both on one scale with the median ratio
    print("ranking quality, best(top-k)/best(all): mean (min)")
    print("  shipped est_cost :", {k: "%.3f (%.3f)" % v for k, v in quality(cases, lambda c: c["cost"]).items()})
    # scale of direct costs relative to fitted tile costs: fitted is time/ideal, est_cost of direct is ~2 at its best
    print("  fitted, tile/ring:", {k: "%.3f (%.3f)" % v for k, v in quality(
        cases, lambda c: math.exp(float(terms(c["F"]) @ coef)) if c["kernel"] != 1 else args.direct_scale * c["cost"]).items()})


def main() -> None:
    ap = argparse.ArgumentParser()
    sub = ap.add_subparsers(dest="cmd", required=True)
    a = sub.add_parser("collect")
    a.add_argument("--out", required=True)
    a.add_argument("--cases", type=int, default=40)
    a.add_argument("--seed", type=int, default=20260701)
    b = sub.add_parser("fit")
    b.add_argument("samples")
    b.add_argument("--direct-scale", type=float, default=0.5,
                   help="factor that puts the direct kernels' own cost (about 2.0 at its best) on the fitted scale")
    args = ap.parse_args()
    (collect if args.cmd == "collect" else fit)(args)


if __name__ == "__main__":
    main()
