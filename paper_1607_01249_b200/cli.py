"""Command line in the spirit of the paper's ``ttc`` tool (Table 1: ``--perm``, ``--size``,
``--dataType``, ``--alpha``, ``--beta``, ``--lda``, ``--ldb``, ``--maxImplementations``): plan one
transposition with libttc.so, report what the plan chose, time it on the device and (optionally) list
the best candidates.  Argument marshalling and reporting only; everything timed runs in the library.

    python -m paper_1607_01249_b200.cli --perm=1,0 --size=9379,5590 --dataType=s --beta=0.5
    python -m paper_1607_01249_b200.cli --perm=2,1,0 --size=8,16,16 --lda=32,32,32 --dataType=d --list 5

``--dataType`` takes s, d, c, z and the mixed pairs sd, ds, cz, zc.  ``--profile`` puts ONE
launch of the chosen candidate inside a cudaProfilerStart/Stop range (for ``ncu --profile-from-start off``).
"""
from __future__ import annotations

import argparse
import json
import statistics

DT = {"s": 0, "d": 1, "c": 2, "z": 3}
ES = {0: 4, 1: 8, 2: 8, 3: 16}


def ints(s):
    return tuple(int(x) for x in s.split(",")) if s else None


def main(argv=None) -> dict:
    ap = argparse.ArgumentParser(description=__doc__.split("\n\n")[0])
    ap.add_argument("--perm", required=True)
    ap.add_argument("--size", required=True)
    ap.add_argument("--dataType", default="s")
    ap.add_argument("--alpha", type=float, default=1.0)
    ap.add_argument("--beta", type=float, default=0.0)
    ap.add_argument("--lda", default=None)
    ap.add_argument("--ldb", default=None)
    ap.add_argument("--maxImplementations", type=int, default=None,
                    help="time only this many best-ranked candidates (PAPER.md:79; sets TTC_TUNE_TOPK)")
    ap.add_argument("--reps", type=int, default=21)
    ap.add_argument("--list", type=int, default=0, help="also print the N fastest timed candidates")
    ap.add_argument("--select", type=int, default=None, help="force candidate index (of the list beta selects)")
    ap.add_argument("--profile", action="store_true")
    ap.add_argument("--specialize", action="store_true",
                    help="also re-compile the winner for this size (ttc_plan_specialize, NVRTC) and time it")
    args = ap.parse_args(argv)
    if args.maxImplementations is not None:
        import os
        os.environ["TTC_TUNE_TOPK"] = str(args.maxImplementations)

    import torch
    from . import ttc
    from . import workloads as wl

    perm, sizes, lda, ldb = ints(args.perm), ints(args.size), ints(args.lda), ints(args.ldb)
    t = args.dataType
    da, db = (DT[t[0]], DT[t[1]]) if len(t) == 2 else (DT[t], DT[t])
    plan = ttc.ttc_plan_mixed(da, db, len(sizes), sizes, perm, lda, ldb)
    info = ttc.ttc_plan_info(plan)
    which = 1 if args.beta != 0 else 0
    if args.select is not None:
        ttc.ttc_plan_select(plan, which, args.select)
    chosen = args.select if args.select is not None else info.chosen[which]
    numel = info.numel
    a = torch.from_numpy(wl.uniform_values(wl.SEED_A, info.span_a, da)).cuda()      # padding holds values too: never read
    b = torch.from_numpy(wl.uniform_values(wl.SEED_B, info.span_b, db)).cuda()
    evict = torch.zeros(64 << 20, dtype=torch.int32, device="cuda")
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for _ in range(3):
        ttc.ttc_execute(plan, args.alpha, a, args.beta, b)
    ts = []
    for _ in range(args.reps):
        evict.max()                      # read sweep: L2 full of clean lines
        e0.record()
        ttc.ttc_execute(plan, args.alpha, a, args.beta, b)
        e1.record()
        e1.synchronize()
        ts.append(e0.elapsed_time(e1) * 1e3)
    if args.profile:
        torch.cuda.synchronize()
        torch.cuda.cudart().cudaProfilerStart()
        ttc.ttc_execute(plan, args.alpha, a, args.beta, b)
        torch.cuda.synchronize()
        torch.cuda.cudart().cudaProfilerStop()
    nbytes = numel * (ES[da] + (2 if which else 1) * ES[db])
    us = statistics.median(ts)
    spec = None
    if args.specialize:
        st = ttc.ttc_plan_specialize(plan)
        i2 = ttc.ttc_plan_info(plan)
        spec = {"status": ttc.STATUS_NAMES[st], "used": i2.specialized[which], "generic_us": i2.generic_us[which],
                "specialized_us": i2.spec_us[which]}
        if i2.specialized[which] == 2:
            t2 = []
            for _ in range(args.reps):
                evict.max()
                e0.record()
                ttc.ttc_execute(plan, args.alpha, a, args.beta, b)
                e1.record()
                e1.synchronize()
                t2.append(e0.elapsed_time(e1) * 1e3)
            spec["us_median"] = statistics.median(t2)
            spec["GB/s"] = nbytes / spec["us_median"] / 1e3
            if args.profile:             # second profiled launch: the specialised twin
                torch.cuda.synchronize()
                torch.cuda.cudart().cudaProfilerStart()
                ttc.ttc_execute(plan, args.alpha, a, args.beta, b)
                torch.cuda.synchronize()
                torch.cuda.cudart().cudaProfilerStop()
    out = {"perm": perm, "size": sizes, "dataType": t, "alpha": args.alpha, "beta": args.beta, "lda": lda, "ldb": ldb,
           "canonical": [(info.canon_extent[i], info.canon_stride_a[i], info.canon_stride_b[i]) for i in range(info.canon_rank)],
           "candidates": info.n_candidates[which], "plan_ms": info.plan_ms, "tune_ms": info.tune_ms,
           "chosen_index": chosen, "chosen": ttc.describe_candidate(ttc.ttc_plan_candidate(plan, which, chosen), info.canon_rank),
           "us_min_of_3": min(ts[:3]), "us_median": us, "bytes": nbytes, "GB/s": nbytes / us / 1e3,
           "GiB/s": nbytes / us / 1e3 * 1e9 / 2 ** 30, "specialize": spec}
    print(json.dumps(out))
    if args.list:
        rows = []
        for i in range(info.n_candidates[which]):
            c = ttc.ttc_plan_candidate(plan, which, i)
            if c.tuned_us > 0:
                rows.append((c.tuned_us, i, ttc.describe_candidate(c, info.canon_rank)))
        for us_i, i, d in sorted(rows)[:args.list]:
            print("%4d  %8.1f us  %s" % (i, us_i, d))
    ttc.ttc_destroy(plan)
    return out


if __name__ == "__main__":
    main()
