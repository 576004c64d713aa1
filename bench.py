#!/usr/bin/env python
"""bench.py -- effective transpose bandwidth of libttc.so on B200 (BASELINE.json `metric`).

Workload at N=1 (and per rank at N>1, "replicas only"): BASELINE.json configs[1],
fp64 4-D tensor 96x72x64x56 (198 MB), all 23 non-identity permutations, alpha=1, beta=0.
One STEP = the whole hot path over that batch: 23 ttc_execute launches, one per permutation
(plans are built and autotuned once, before the timed region, as the paper generates code
once per transposition).  value = (2 * |A| * 8 bytes * 23 * ranks) / step time.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--detail PATH]

stdout carries exactly ONE JSON line.  --detail additionally writes per-config results of all
five BASELINE.json configs (cold L2, min of 3 and median) to PATH as JSON.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "effective transpose GB/s ((2|3)\u00b7|A| bytes / device time) and % of B200 HBM peak"
UNIT = "GB/s"
WORKLOAD = "configs[1]: fp64 96x72x64x56 (198 MB), all 23 non-identity permutations, alpha=1, beta=0"
NOMINAL_HBM_GBS = 8000.0      # north_star's "~8 TB/s"
FALLBACK_HBM_GBS = 6650.0     # B200_PROFILING.md fallback


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (measured)"
    except Exception:
        return FALLBACK_HBM_GBS, "B200_PROFILING.md fallback"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (profiling recipe)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "100"],
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
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for name, v in zip(self.NAMES, r[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "reasons": sorted(reasons),
                "samples": len(sm)}


# ------------------------------------------------------------------------------ CPU legs
REF_SAMPLE_PERMS = [(2, 3, 0, 1), (3, 1, 2, 0), (1, 3, 0, 2)]   # canonical rank 2, 3, 4


def time_oracle(perms, A, B) -> float:
    """Seconds the oracle (as it stands, 1 thread) needs for the given c2 permutations."""
    import oracle
    from paper_1607_01249_b200 import workloads as wl
    t0 = time.perf_counter()
    for perm in perms:
        w = wl.config2(perm)
        oracle.transpose(w.dtype, w.sizes, w.perm, None, None, 1.0, A, 0.0, B)
    return time.perf_counter() - t0


def time_ref_omp(works, A_host) -> dict:
    """The paper's OpenMP reference loop nest -- BASELINE.md section 3's timed CPU baseline --
    built with -O3 -march=native -fopenmp on this box, all host cores, arrays first-touched in parallel
    (PAPER.md:147, 183), minimum of 3 runs per permutation; its result is compared with the oracle's."""
    import oracle
    A = oracle.first_touch_copy(A_host)
    B = oracle.first_touch_zeros(A_host)
    secs = 0.0
    for w in works:
        best = None
        for _ in range(3):
            t0 = time.perf_counter()
            oracle.ref_omp_native_transpose(w.dtype, w.sizes, w.perm, None, None, 1.0, A, 0.0, B)
            dt = time.perf_counter() - t0
            best = dt if best is None or dt < best else best
        secs += best
    last = works[-1]
    B_or = np.zeros_like(A_host)
    oracle.transpose(last.dtype, last.sizes, last.perm, None, None, 1.0, A_host, 0.0, B_or)
    if not np.array_equal(B_or.view(np.uint8), B.view(np.uint8)):
        raise SystemExit("bench.py: the OpenMP reference loop differs from the oracle")
    step_bytes = sum(w.algorithmic_bytes for w in works)
    try:
        affinity = len(os.sched_getaffinity(0))
    except Exception:
        affinity = None
    return {"value": step_bytes / secs / 1e9, "unit": UNIT, "cores": oracle.ref_omp_native_threads(),
            "nproc": os.cpu_count(), "affinity_cores": affinity, "kind": "paper's OpenMP reference loop nest (PAPER.md:167)",
            "flags": oracle.NATIVE_FLAGS, "seconds": secs,
            "sample": "one whole step: all %d permutations, min of 3 runs each, whole 198 MB tensors" % len(works),
            "checked": "bit-identical to the oracle on the last permutation"}


def run_reference(args) -> None:
    """--impl reference: the oracle on the host cores, same metric/config; a step is a bounded
    sample (3 of the 23 permutations: canonical rank 2, 3 and 4)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1607_01249_b200 import workloads as wl
    steps = args.steps if args.steps is not None else 3
    warmup = args.warmup if args.warmup is not None else 1
    w0 = wl.config2(REF_SAMPLE_PERMS[0])
    A, B = w0.make_a(), w0.make_b()
    for _ in range(warmup):
        time_oracle(REF_SAMPLE_PERMS, A, B)
    t = 0.0
    for _ in range(steps):
        t += time_oracle(REF_SAMPLE_PERMS, A, B)
    bytes_per_step = sum(wl.config2(p).algorithmic_bytes for p in REF_SAMPLE_PERMS)
    value = bytes_per_step * steps / t / 1e9
    sample = "%d of the 23 permutations per step: %s, whole 198 MB tensor each" % (
        len(REF_SAMPLE_PERMS), REF_SAMPLE_PERMS)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": warmup, "ms_per_step": t / steps * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic (seeded SplitMix64)",
        "config": {"workload": WORKLOAD, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ------------------------------------------------------------------------------ GPU arm
class Evictor:
    """Puts the 126 MB L2 into a known state before a timed launch (the paper clears the
    caches before every run).  Two ways, reported side by side so that their difference is attributed:
      read   -- a reduction READS a 256 MB buffer: L2 ends up full of CLEAN lines of that buffer, the timed
                kernel pays nothing for the eviction (the clean-cold figure);
      memset -- the buffer is WRITTEN: L2 ends up full of DIRTY lines whose write-back to HBM is
                charged to the timed kernel (what round 1 reported as "cold")."""
    METHODS = ("read", "memset")

    def __init__(self, torch, nbytes: int = 256 << 20):
        self.torch = torch
        self.buf = torch.zeros(nbytes // 4, dtype=torch.int32, device="cuda")

    def __call__(self, method: str) -> None:
        if method == "read":
            self.buf.max()
        elif method == "memset":
            self.buf.zero_()
        else:
            raise ValueError(method)


def cold_times(torch, ttc, plan, alpha, beta, a_dev, b_dev, evict, method: str, reps: int):
    """Per-launch device times (us), L2 evicted before every run."""
    out = []
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for _ in range(reps):
        evict(method)
        e0.record()
        ttc.ttc_execute(plan, alpha, a_dev, beta, b_dev)
        e1.record()
        e1.synchronize()
        out.append(e0.elapsed_time(e1) * 1e3)
    return out


def cold_row(torch, ttc, plan, w, nbytes, alpha, beta, a_dev, b_dev, evict, peak, reps: int = 21) -> dict:
    """min of 3 (the paper's statistic) and median of `reps`, for both eviction methods."""
    for _ in range(3):
        ttc.ttc_execute(plan, alpha, a_dev, beta, b_dev)
    row = {"config": w.name, "perm": "".join(map(str, w.perm)), "bytes": nbytes}
    for m in Evictor.METHODS:
        ts = cold_times(torch, ttc, plan, alpha, beta, a_dev, b_dev, evict, m, reps)
        t3, tm = min(ts[:3]), statistics.median(ts)
        row[m] = {"us_min_of_3": t3, "us_median": tm, "gbs_min_of_3": nbytes / t3 / 1e3, "gbs_median": nbytes / tm / 1e3,
                  "frac_of_measured_copy": nbytes / tm / 1e3 / peak, "frac_of_8TBs": nbytes / tm / 1e3 / NOMINAL_HBM_GBS}
    return row


def cold_block(torch, ttc, wl, peak, works, plans, a_dev, b_dev) -> dict:
    """SURVEY.md 8(d) protocol inside the driver-run line: every permutation of configs[1] and
    configs[0], [2], [3], [4], L2 evicted before EVERY timed launch, min of 3 and median of 21."""
    evict = Evictor(torch)
    rows = []
    for p, w in zip(plans, works):
        rows.append(cold_row(torch, ttc, p, w, w.algorithmic_bytes, w.alpha, w.beta, a_dev, b_dev, evict, peak))
    others = {}
    for w in (wl.config1(), wl.config3(), wl.config4(), wl.config5()):
        plan = ttc.ttc_plan(w.dtype, w.n, w.sizes, w.perm, w.lda, w.ldb)
        info = ttc.ttc_plan_info(plan)
        xa = torch.from_numpy(w.make_a()).cuda()
        xb = torch.from_numpy(w.make_b()).cuda()
        row = cold_row(torch, ttc, plan, w, w.algorithmic_bytes, w.alpha, w.beta, xa, xb, evict, peak)
        which = 1 if w.beta_nonzero else 0
        row["chosen"] = ttc.describe_candidate(ttc.ttc_plan_candidate(plan, which, info.chosen[which]), info.canon_rank)
        row["plan_ms"] = info.plan_ms
        # the NVRTC size-specialised twin of the winner against the generic instance
        t_sp = time.perf_counter()
        st = ttc.ttc_plan_specialize(plan)
        i2 = ttc.ttc_plan_info(plan)
        row["specialize"] = {"status": ttc.STATUS_NAMES[st], "seconds": time.perf_counter() - t_sp,
                             "generic_us": i2.generic_us[which], "specialized_us": i2.spec_us[which],
                             "used": {0: "generic (no twin)", 1: "generic (twin slower)", 2: "specialised"}[i2.specialized[which]]}
        if i2.specialized[which] == 2:
            r2 = cold_row(torch, ttc, plan, w, w.algorithmic_bytes, w.alpha, w.beta, xa, xb, evict, peak)
            row["specialize"]["gbs_median_cold"] = r2["read"]["gbs_median"]
        if w.name.startswith("c1"):      # small tensor (23.6 MB): also the warm, L2-resident figure
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ts = []
            for _ in range(21):
                torch.cuda._sleep(40000)        # ~20 us of device spin: the launch below is queued before e0 is reached
                e0.record()
                ttc.ttc_execute(plan, w.alpha, xa, w.beta, xb)
                e1.record()
                e1.synchronize()
                ts.append(e0.elapsed_time(e1) * 1e3)
            row["warm_l2_resident"] = {"us_median": statistics.median(ts),
                                       "gbs_median": w.algorithmic_bytes / statistics.median(ts) / 1e3}
        rows.append(row)
        others[w.name.split("_")[0]] = row
        ttc.ttc_destroy(plan)
        del xa, xb
    c2 = rows[:len(works)]

    def summary(method):
        g = [r[method]["gbs_median"] for r in c2]
        return {"min": min(g), "median": statistics.median(g), "max": max(g),
                "min_frac_of_measured_copy": min(g) / peak, "median_frac_of_measured_copy": statistics.median(g) / peak,
                "median_frac_of_8TBs": statistics.median(g) / NOMINAL_HBM_GBS}
    per_config = {"c2": {"gbs_median_over_perms": summary("read")["median"], "gbs_min_over_perms": summary("read")["min"],
                         "frac_of_measured_copy": summary("read")["median_frac_of_measured_copy"],
                         "frac_of_8TBs": summary("read")["median_frac_of_8TBs"]}}
    for k, r in others.items():
        # as for c2 (whose plans were specialised before this block): the figure of the kernel the plan launches after
        # ttc_plan_specialize -- the NVRTC twin where it measured faster -- with the generic instance's beside it
        spec = r.get("specialize", {}).get("gbs_median_cold")
        used = spec if spec else r["read"]["gbs_median"]          # spec is only there when the plan launches the twin
        per_config[k] = {"gbs_median": used, "gbs_median_generic": r["read"]["gbs_median"], "gbs_min_of_3": r["read"]["gbs_min_of_3"],
                         "kernel_used": "size-specialised (NVRTC)" if spec else "generic",
                         "frac_of_measured_copy": used / peak, "frac_of_8TBs": used / NOMINAL_HBM_GBS}
    return {"protocol": "L2 evicted before every timed launch (PAPER.md:147); min of 3 and median of 21 per case; "
                        "read = 256 MB read sweep (clean lines), memset = 256 MB write (dirty lines, their write-back "
                        "is charged to the timed kernel); per_config quotes the read-evicted medians",
            "c2_read": summary("read"), "c2_memset": summary("memset"), "per_config": per_config, "rows": rows}


def _legacy_fields(row: dict, peak: float) -> dict:
    """Flat keys of the round-1 detail table, taken from the read-evicted (clean-cold) measurement."""
    r = row["read"]
    row.update({"us_min_of_3": r["us_min_of_3"], "us_median_21": r["us_median"], "gbs_min_of_3": r["gbs_min_of_3"],
                "gbs_median": r["gbs_median"], "gibs_median": r["gbs_median"] * 1e9 / 2 ** 30,
                "frac_of_8TBs": r["frac_of_8TBs"], "frac_of_measured_copy": r["frac_of_measured_copy"],
                "gbs_median_memset_evicted": row["memset"]["gbs_median"]})
    return row


def profiled_launch(torch, ttc, plan, alpha, beta, a_dev, b_dev) -> None:
    """One launch inside a cudaProfilerStart/Stop range (for ncu --profile-from-start off)."""
    torch.cuda.synchronize()
    torch.cuda.cudart().cudaProfilerStart()
    ttc.ttc_execute(plan, alpha, a_dev, beta, b_dev)
    torch.cuda.synchronize()
    torch.cuda.cudart().cudaProfilerStop()


def detail_all_configs(torch, ttc, wl, path: str, peak: float, profile: bool = False) -> None:
    """Per-config report of all five BASELINE.json configs (north_star: 'reported per config')."""
    evict = Evictor(torch)
    rows = []
    for w in wl.baseline_configs():
        plan = ttc.ttc_plan(w.dtype, w.n, w.sizes, w.perm, w.lda, w.ldb)
        info = ttc.ttc_plan_info(plan)
        a_dev = torch.from_numpy(w.make_a()).cuda()
        b_dev = torch.from_numpy(w.make_b()).cuda()
        row = cold_row(torch, ttc, plan, w, w.algorithmic_bytes, w.alpha, w.beta, a_dev, b_dev, evict, peak)
        if profile and not w.name.startswith("c2"):
            profiled_launch(torch, ttc, plan, w.alpha, w.beta, a_dev, b_dev)
        which = 1 if w.beta_nonzero else 0
        cand = ttc.ttc_plan_candidate(plan, which, info.chosen[which])
        row.update({"chosen": ttc.describe_candidate(cand, info.canon_rank), "n_candidates": info.n_candidates[which],
                    "plan_ms": info.plan_ms, "tune_ms": info.tune_ms})
        rows.append(_legacy_fields(row, peak))
        ttc.ttc_destroy(plan)
        del a_dev, b_dev
    rows.extend(detail_misaligned(torch, ttc, wl, evict, peak))
    rows.extend(detail_mixed(torch, ttc, wl, evict, peak, profile))
    with open(path, "w") as fh:
        json.dump(rows, fh, indent=1)


def batched_block(torch, ttc, wl, peak: float) -> dict:
    """ttc_execute_batched: many small transpositions that share a plan in one launch.
    (a) 256 BLAS A-panel packs of 8 x 32 x 1024 fp64 blocks (2 MB each) cut out of one padded
    operand; (b) 24 copies of configs[0] (the 23.6 MB, launch-bound case).  Each against the same work issued
    as one ttc_execute per block; L2 evicted (read sweep) before every timed run, median of 11."""
    evict = Evictor(torch)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    out = {}
    c1 = wl.config1()
    cases = (("a_panel_packs_256x2MB", wl.F64, (8, 32, 1024), (0, 2, 1), (8, 40, 1024), 256),
             ("configs0_x24", c1.dtype, c1.sizes, c1.perm, None, 24))
    for name, dtype, sizes, perm, lda, batch in cases:
        plan = ttc.ttc_plan(dtype, len(sizes), sizes, perm, lda, None)
        info = ttc.ttc_plan_info(plan)
        tdt = torch.float64 if dtype == wl.F64 else torch.float32
        la, lb = info.span_a + 8, info.numel + 8
        big_a = torch.rand(batch * la, dtype=tdt, device="cuda")
        big_b = torch.zeros(batch * lb, dtype=tdt, device="cuda")
        As = [big_a[i * la:i * la + info.span_a] for i in range(batch)]
        Bs = [big_b[i * lb:i * lb + info.numel] for i in range(batch)]
        nbytes = 2 * info.numel * wl.ELEM_SIZE[dtype] * batch

        def looped():
            for a, b in zip(As, Bs):
                ttc.ttc_execute(plan, 1.0, a, 0.0, b)

        def batched():
            ttc.ttc_execute_batched(plan, 1.0, As, 0.0, Bs)
        res = {}
        for label, fn in (("batched", batched), ("one_launch_per_block", looped)):
            fn()
            ts = []
            for _ in range(11):
                evict("read")
                torch.cuda._sleep(200000)       # the (slow, Python-issued) launches are queued before the timer starts
                e0.record()
                fn()
                e1.record()
                e1.synchronize()
                ts.append(e0.elapsed_time(e1) * 1e3)
            us = statistics.median(ts)
            res[label] = {"us_median": us, "gbs": nbytes / us / 1e3, "frac_of_measured_copy": nbytes / us / 1e3 / peak}
        res["blocks"] = batch
        res["bytes"] = nbytes
        res["launches_batched"] = (batch + 63) // 64
        out[name] = res
        ttc.ttc_destroy(plan)
        del big_a, big_b, As, Bs
    return out


def detail_misaligned(torch, ttc, wl, evict, peak: float) -> list:
    """Element-aligned but not 16-byte aligned pointers: the alignment-aware fallback
    candidate of the same plan, timed on three permutations of configs[1]'s tensor."""
    rows = []
    for perm in ((0, 2, 1, 3), (2, 3, 0, 1), (3, 1, 0, 2)):
        w = wl.config2(perm)
        plan = ttc.ttc_plan(w.dtype, w.n, w.sizes, w.perm)
        a_all = torch.zeros(w.numel + 2, dtype=torch.float64, device="cuda")
        b_all = torch.zeros(w.numel + 2, dtype=torch.float64, device="cuda")
        a_all[1:1 + w.numel] = torch.from_numpy(w.make_a()).cuda()
        for ma, mb in ((1, 0), (0, 1), (1, 1)):
            name = "misaligned A+%d B+%d elements, %s" % (ma, mb, w.name)
            row = cold_row(torch, ttc, plan, wl.Workload(name, w.dtype, w.sizes, w.perm), w.algorithmic_bytes, 1.0, 0.0,
                           a_all[ma:ma + w.numel], b_all[mb:mb + w.numel], evict, peak)
            rows.append(_legacy_fields(row, peak))
        ttc.ttc_destroy(plan)
        del a_all, b_all
    return rows


def detail_mixed(torch, ttc, wl, evict, peak: float, profile: bool = False) -> list:
    """Mixed-precision transpositions on configs[1]'s tensor:
    A of one type, B of the other.  Algorithmic bytes = |A| * (sizeof(A) + (1 | 2) * sizeof(B))."""
    rows = []
    pairs = (("sd", wl.F32, wl.F64), ("ds", wl.F64, wl.F32), ("cz", wl.C64, wl.C128), ("zc", wl.C128, wl.C64))
    cases = [(p, perm, 0.0) for p in pairs[:2] for perm in ((0, 2, 1, 3), (2, 3, 0, 1), (3, 1, 0, 2))]
    cases += [(pairs[0], (2, 3, 0, 1), 0.5), (pairs[1], (2, 3, 0, 1), 0.5), (pairs[2], (3, 1, 0, 2), 0.0),
              (pairs[3], (3, 1, 0, 2), 0.0)]
    # the paper's mixed-precision use case is packing for GEMM: configs[3]'s shape and lda
    cases += [(pairs[0], "c4", 0.0), (pairs[1], "c4", 0.0)]
    for (name, da, db), perm, beta in cases:
        w = wl.config4() if perm == "c4" else wl.config2(perm)
        perm = w.perm
        numel = w.numel
        plan = ttc.ttc_plan_mixed(da, db, w.n, w.sizes, perm, w.lda, w.ldb)
        info = ttc.ttc_plan_info(plan)
        szb = tuple(w.sizes[q] for q in perm)
        a_dev = torch.from_numpy(wl.embed(wl.uniform_values(wl.SEED_A, numel, da), w.sizes, w.lda)).cuda()
        b_dev = torch.from_numpy(wl.embed(wl.uniform_values(wl.SEED_B, numel, db), szb, w.ldb)).cuda()
        alpha = 1.5
        which = 1 if beta != 0 else 0
        nbytes = numel * (wl.ELEM_SIZE[da] + (2 if which else 1) * wl.ELEM_SIZE[db])
        label = "mixed-%s %s on configs[%d]'s tensor, beta=%g" % (name, wl.DTYPE_NAME[da] + "->" + wl.DTYPE_NAME[db],
                                                                   3 if w.name.startswith("c4") else 1, beta)
        row = cold_row(torch, ttc, plan, wl.Workload(label, db, w.sizes, perm), nbytes, alpha, beta, a_dev, b_dev, evict, peak)
        if profile and beta == 0 and name in ("sd", "ds") and perm != (3, 1, 0, 2) and w.name.startswith("c2"):   # 4 launches for ncu
            profiled_launch(torch, ttc, plan, alpha, beta, a_dev, b_dev)
        cand = ttc.ttc_plan_candidate(plan, which, info.chosen[which])
        row.update({"chosen": ttc.describe_candidate(cand, info.canon_rank), "n_candidates": info.n_candidates[which],
                    "plan_ms": info.plan_ms})
        rows.append(_legacy_fields(row, peak))
        ttc.ttc_destroy(plan)
        del a_dev, b_dev
    return rows


def whole_job_value(step_bytes: int, steps: int, world: int, ms_local: float, dist, device) -> tuple:
    """(value in GB/s, ms) of the whole job: bytes of ALL ranks over the MAX of the ranks' device times."""
    import torch
    ms = torch.tensor([ms_local], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    ms_total = float(ms.item())
    return step_bytes * steps * world / (ms_total * 1e-3) / 1e9, ms_total


def run_ours(args) -> None:
    import torch
    from paper_1607_01249_b200 import ttc            # raises if libttc.so cannot be built/loaded
    from paper_1607_01249_b200 import workloads as wl
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU path")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    steps = args.steps if args.steps is not None else 200
    warmup = max(3, args.warmup if args.warmup is not None else 5)
    peak, peak_src = measured_peak()

    works = list(wl.config2_all())
    if args.perms:     # profiling aid (ncu captures of single permutations); not the headline workload
        keep = {tuple(int(ch) for ch in x) for x in args.perms.split(",")}
        works = [w for w in works if w.perm in keep]
    t_plan0 = time.perf_counter()
    plans = [ttc.ttc_plan(w.dtype, w.n, w.sizes, w.perm) for w in works]      # tuned here, untimed
    plan_wall_s = time.perf_counter() - t_plan0
    # TTC compiles code for the specific size.  The tuned winners are re-compiled by NVRTC with
    # their parameter blocks as compile-time constants (untimed, once per transposition, like the tuning) and
    # used where they measure faster than the generic instances.
    t_sp0 = time.perf_counter()
    spec_status = [ttc.ttc_plan_specialize(p) for p in plans] if not args.no_specialize else []
    specialize_wall_s = time.perf_counter() - t_sp0
    A_host = works[0].make_a()
    a_dev = torch.from_numpy(A_host).cuda()
    b_dev = torch.zeros_like(a_dev)
    step_bytes = sum(w.algorithmic_bytes for w in works)
    stream = torch.cuda.current_stream()

    def one_step(events=None, st=None):
        # one event between consecutive launches: events[i] .. events[i + 1] brackets launch i
        st = st or stream
        for i, (p, w) in enumerate(zip(plans, works)):
            if events is not None:
                events[i].record(st)
            ttc.ttc_execute(p, 1.0, a_dev, 0.0, b_dev, st)
        if events is not None:
            events[len(plans)].record(st)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # A step is launched as ONE CUDA graph replay: the 23 ttc_execute calls are captured once
    # (untimed) and replayed -- ttc_execute is a single asynchronous kernel launch with no library
    # state, so it captures as one kernel node.  Kernel-to-kernel edges of a graph cost ~2.5 us less
    # than stream launches on this machine and let programmatic dependent launch overlap a kernel's
    # prologue with its predecessor's tail.  --no-graph: plain stream launches.
    use_graph = not args.no_graph
    n_ev = 0 if args.no_launch_events else min(8, max(1, steps // 10))
    ev_steps = list(range(0, steps, 10))[:n_ev]
    ev = {s: [torch.cuda.Event(enable_timing=True, external=use_graph) for _ in range(len(works) + 1)]
          for s in ev_steps} if n_ev else None
    side = torch.cuda.Stream()

    def capture(events=None):
        g = torch.cuda.CUDAGraph()
        side.wait_stream(stream)
        with torch.cuda.stream(side):
            with torch.cuda.graph(g, stream=side):
                one_step(events, side)
        return g

    for _ in range(warmup if not use_graph else 1):
        one_step()
    graph_plain = graph_ev = None
    if use_graph:
        graph_plain = capture()
        # per-launch events for the roofline of the dominant kernel, live in the timed region: every
        # 10th of the first steps replays a twin graph with an (external) event node between the launches
        graph_ev = {s: capture(ev[s]) for s in ev_steps} if ev else {}
        for _ in range(warmup):
            graph_plain.replay()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    barrier()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.cudart().cudaProfilerStart()     # ncu --profile-from-start off sees only the timed region
    t0.record(stream)
    for s in range(steps):
        if use_graph:
            (graph_ev.get(s) or graph_plain).replay()
        else:
            one_step(ev.get(s) if ev else None)
    t1.record(stream)
    barrier()
    torch.cuda.cudart().cudaProfilerStop()
    launches = steps * len(plans)               # kernels of libttc.so launched inside the timed region
    clocks = sampler.stop()
    value, ms_total = whole_job_value(step_bytes, steps, world, t0.elapsed_time(t1), dist, "cuda")

    # the same step as plain stream launches (what round 1 timed), for comparison
    stream_launch = None
    if use_graph:
        k = min(steps, 20)
        for _ in range(3):
            one_step()
        barrier()
        t0.record(stream)
        for _ in range(k):
            one_step()
        t1.record(stream)
        barrier()
        v2, ms2 = whole_job_value(step_bytes, k, world, t0.elapsed_time(t1), dist, "cuda")
        stream_launch = {"value": v2, "unit": UNIT, "ms_per_step": ms2 / k, "steps": k,
                         "note": "23 ttc_execute calls per step issued on the stream, no graph"}

    # per-permutation launch durations (median over steps) and the roofline of the tile kernel
    per_perm, infos = [], []
    for i, (p, w) in enumerate(zip(plans, works)):
        info = ttc.ttc_plan_info(p)
        cand = ttc.ttc_plan_candidate(p, 0, info.chosen[0])
        us = statistics.median(ev[s][i].elapsed_time(ev[s][i + 1]) for s in ev_steps) * 1e3 if ev else None
        infos.append((w, cand, info))
        per_perm.append({"perm": "".join(map(str, w.perm)), "kernel": ttc.KERNEL_NAMES[cand.kernel],
                         "us": us, "gbs": (w.algorithmic_bytes / us / 1e3) if us else None,
                         "frac_of_measured_copy": (w.algorithmic_bytes / us / 1e3 / peak) if us else None,
                         "plan_ms": info.plan_ms, "tune_ms": info.tune_ms, "tune_errors": info.tune_errors,
                         "n_candidates": info.n_candidates[0],
                         "kernel_used": {0: "generic", 1: "generic (specialised twin slower)", 2: "size-specialised (NVRTC)"}[info.specialized[0]],
                         "generic_us": info.generic_us[0], "specialized_us": info.spec_us[0],
                         "chosen": ttc.describe_candidate(cand, info.canon_rank)})
    roofline = None
    if ev:
        dom = [r for r in per_perm if r["kernel"] != "copy"] or per_perm      # a copy-only --perms subset
        dom_us = sum(r["us"] for r in dom)
        achieved = works[0].algorithmic_bytes * len(dom) / dom_us / 1e3
        n_ring = sum(1 for r in dom if r["kernel"] == "tma")
        n_tmap = sum(1 for r in dom if r["kernel"] == "tensormap")
        roofline = {"bound": "hbm",
                    "kernel": "K2/K3 transposing kernels (ring_kernel: %d, tmap_kernel: %d, tile_kernel: %d) of %d launches per step" % (
                        n_ring, n_tmap, len(dom) - n_ring - n_tmap, len(per_perm)),
                    "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                    "peak_source": peak_src, "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS,
                    "avg_launch_us": dom_us / len(dom), "algorithmic_bytes_per_launch": works[0].algorithmic_bytes,
                    "share_of_step": dom_us / sum(r["us"] for r in per_perm),
                    "per_launch_gbs": {"min": min(r["gbs"] for r in dom), "median": statistics.median(r["gbs"] for r in dom),
                                       "max": max(r["gbs"] for r in dom)},
                    "traffic": None, "traffic_source": None}
        # dram__bytes_read.sum + dram__bytes_write.sum per launch of that kernel, from the committed
        # ncu --set full capture of this round (a run under ncu cannot be the timed run)
        import glob
        for tr in sorted(glob.glob(os.path.join(ROOT, "profiles", "traffic_r*.csv")), reverse=True):
            for ln in open(tr):
                if ln.startswith("transpose_kernel_dram_bytes_per_launch,"):
                    roofline["traffic"] = int(ln.split(",")[1])
                    roofline["traffic_source"] = "profiles/" + os.path.basename(tr)
            if roofline["traffic"] is not None:
                break

    # ---- end to end through the public host-buffer call: pinned host A -> device, kernel,
    # device -> pinned host B, every permutation, inside the timed region
    e2e_steps = max(1, min(steps, args.e2e_steps))
    a_pin = torch.from_numpy(A_host).pin_memory()
    b_pin = torch.zeros_like(a_pin).pin_memory()
    a_np, b_np = a_pin.numpy(), b_pin.numpy()

    def e2e_step():
        for p in plans:
            ttc.ttc_execute_host(p, 1.0, a_np, 0.0, b_np, stream)

    e2e_step()
    barrier()
    w0 = time.perf_counter()
    t0.record(stream)
    for _ in range(e2e_steps):
        e2e_step()
    t1.record(stream)
    barrier()
    wall = time.perf_counter() - w0
    ms = torch.tensor([max(t0.elapsed_time(t1), wall * 1e3)], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    e2e_value = step_bytes * e2e_steps * world / (float(ms.item()) * 1e-3) / 1e9
    nbytes = a_pin.numel() * a_pin.element_size()
    e2e = {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": nbytes * len(plans),
           "d2h_bytes_per_step": nbytes * len(plans), "steps": e2e_steps,
           "api": "ttc_execute_host (pinned host A and B)"}
    # last e2e result doubles as a live parity spot check of the timed configuration
    last = works[-1]
    idx = np.random.default_rng(0).integers(0, last.numel, 4096)

    if args.detail and rank == 0:
        detail_all_configs(torch, ttc, wl, args.detail, peak, args.profile_detail)

    cold = None
    if rank == 0 and world == 1 and not args.no_cold:
        cold = cold_block(torch, ttc, wl, peak, works, plans, a_dev, b_dev)

    batched = None
    if rank == 0 and world == 1 and not args.no_cold:
        batched = batched_block(torch, ttc, wl, peak)

    cpu = cpu_omp = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu_omp = time_ref_omp(works, A_host)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        B_or = np.zeros_like(A_host)
        perms = [w.perm for w in works]
        secs = time_oracle(perms, A_host, B_or)
        # the oracle's last permutation is the e2e leg's last permutation: compare samples
        if not np.array_equal(B_or[idx], b_np[idx]):
            raise SystemExit("bench.py: GPU result differs from the oracle on sampled outputs")
        cpu = {"value": step_bytes / secs / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle",
               "seconds": secs, "sample": "one whole step: all 23 permutations once, single thread"}

    for p in plans:
        ttc.ttc_destroy(p)
    if rank == 0:
        gbs = [r["gbs"] for r in per_perm if r["gbs"]]
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps,
                "warmup": warmup, "ms_per_step": ms_total / steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64",
                "data": "synthetic (seeded SplitMix64 uniform [-1,1))",
                "config": {"workload": WORKLOAD if not args.perms else WORKLOAD + " -- SUBSET " + args.perms,
                           "parallelism": "replicas only (no collective)",
                           "l2": "inputs larger than L2: A and B are 198 MB each, L2 is 126 MB; no explicit flush "
                                 "between the 23 back-to-back launches of a step (the `cold` block holds the "
                                 "flush-before-every-launch figures of SURVEY.md 8(d))",
                           "launches_per_step": len(plans),
                           "launch_mode": "one CUDA graph replay per step (23 kernel nodes, captured once before "
                                          "the timed region)" if use_graph else "stream launches"},
                "stream_launch": stream_launch,
                "frac_of_measured_copy": value / world / peak, "frac_of_nominal_8TBs": value / world / NOMINAL_HBM_GBS,
                "per_perm_gbs": {"min": min(gbs), "median": statistics.median(gbs), "max": max(gbs)} if gbs else None,
                "per_perm": per_perm, "roofline": roofline, "cold": cold,
                "per_config": cold["per_config"] if cold else None, "batched": batched,
                "plan_ms": {"median": statistics.median(r["plan_ms"] for r in per_perm),
                            "max": max(r["plan_ms"] for r in per_perm), "total_wall_s": plan_wall_s,
                            "specialize_total_wall_s": specialize_wall_s,
                            "specialized_plans": sum(1 for r in per_perm if r["kernel_used"].startswith("size-")),
                            "note": "ttc_plan incl. on-device tuning of the beta=0 and beta!=0 lists; untimed, once per transposition"},
                "cpu_baseline": cpu, "cpu_baseline_omp": cpu_omp, "e2e": e2e,
                "gpu_launches": launches, "clocks": clocks}
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--detail", default=None, help="write per-config results of all 5 configs here")
    ap.add_argument("--perms", default=None, help="comma-separated subset of the 23 permutations, e.g. 1023,3021 "
                    "(profiling aid; the step is then NOT the headline workload)")
    ap.add_argument("--profile-detail", action="store_true", help="with --detail: one extra launch of c1, c3, c4, c5 "
                    "inside a cudaProfilerStart/Stop range (for ncu --profile-from-start off)")
    ap.add_argument("--no-launch-events", action="store_true")
    ap.add_argument("--no-specialize", action="store_true", help="keep the generic kernel instances (no NVRTC)")
    ap.add_argument("--no-graph", action="store_true", help="issue the 23 launches of a step on the stream instead of replaying a CUDA graph")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-cold", action="store_true", help="skip the cold-L2 block (profiling runs)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
