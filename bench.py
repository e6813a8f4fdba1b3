#!/usr/bin/env python
"""bench.py -- throughput of the Omega(Delta; q, h, T) hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--mode coop_eo|coop|...]
                    [--scaling strong|weak] [--workload omega|chi|paper]

Workload (config.workload): BASELINE.json configs[3] "cfg4_fflo_N1024": two-band s+- model, N = 1024 x 1024 k-grid,
32 q along (1,1), 64 h, 512 Delta -- the configuration north_star quotes its FP64-roofline target on.
One STEP = one pass of the whole hot path over one batch: fe_omega_grid (K0 trig, KS constant sum, K1 k-sum,
K2 finish) + fe_argmin over the batch's full (q, h, Delta) grid at one temperature; successive steps alternate
T = 0.001 / 0.01 (config 4 names both).  The batch is `--q-per-step` q-values of the config (default: all 32),
so a default step is the whole 1.1e12-evaluation scan.

Output: ONE JSON line (rank 0).  value = k-point x parameter evaluations per second, whole job, inputs resident
(device timing with CUDA events per step, L2 flushed between steps, max over ranks).  e2e = same metric through
fe_scan_host with HOST buffers (lists H2D, Omega + minima D2H inside the timed region).
roofline: bound "alu" (plain FP64 pipe; no contraction, HBM negligible), see DESIGN.md "Roofline".  The FP64
instruction counts behind `roofline.achieved` are NOT constants of this file: they are parsed at run time from the
committed ncu captures listed in profiles/COUNTS.md, and used only if the kernel-source hash recorded beside the capture
equals the hash of the sources in the tree and of the sources libfe.so was built from; otherwise frac is null and
`stale_counts` says why.
cpu_baseline: the oracle (oracle/fe_oracle.c) as it stands, timed on this host's cores (1 thread and all cores) on a
bounded sample.  `--impl reference` times the oracle instead (the reference arm of this tier).
N > 1 GPUs: one process per GPU (torchrun), the q list is sharded by paper_1412_8754_b200.sharding (the code the
world-size-2 gloo tests run); no collective on the data path, NCCL only for the barrier, the max-over-ranks time and
the final gather of the minima.
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1412_8754_b200 import sharding, workloads as W  # noqa: E402

METRIC = "Omega evaluations/s (k-points x grid points, fp64)"
UNIT = "k-point x (q,h,Delta) evaluations/s"
PROFILES = os.path.join(ROOT, "profiles")

# FP64 roofline denominator, derived from unit counts and clocks (MEASURED_PEAKS.json has no fp64
# entry): 148 SMs x 64 FP64 lanes x 1.965 GHz thread-level FP64-pipe instructions per second; a DFMA counts 2 flop.
SM_COUNT, FP64_LANES_PER_SM, SM_MAX_GHZ = 148, 64, 1.965
PEAK_DFMA_PER_S = SM_COUNT * FP64_LANES_PER_SM * SM_MAX_GHZ * 1e9
PEAK_TFLOPS = 2 * PEAK_DFMA_PER_S / 1e12
FP64_OPS = ("dadd", "dmul", "dfma")


# ----------------------------------------------------------------------------------------------------
# profiler counts: parsed from the committed ncu CSVs, never typed in
# ----------------------------------------------------------------------------------------------------
def parse_ncu_metrics_csv(path):
    """`ncu --metrics ... --csv --log-file` output (long format: one row per launch and metric) -> one dict per
    launch, in launch order: {kernel, grid, block, metrics: {name: float}}."""
    launches = {}
    with open(path, newline="") as f:
        rows = [r for r in csv.reader(f) if len(r) >= 15]
    head = rows[0]
    col = {n: head.index(n) for n in ("ID", "Kernel Name", "Block Size", "Grid Size", "Metric Name", "Metric Value")}
    for r in rows[1:]:
        if r[0] == "ID":
            continue
        d = launches.setdefault(int(r[col["ID"]]), dict(kernel=r[col["Kernel Name"]], grid=r[col["Grid Size"]],
                                                        block=r[col["Block Size"]], metrics={}))
        try:
            d["metrics"][r[col["Metric Name"]]] = float(r[col["Metric Value"]].replace(",", ""))
        except ValueError:
            pass
    return [launches[k] for k in sorted(launches)]


def load_counts_index(path=None):
    """profiles/COUNTS.md: a markdown table | key | file | launches | source_hash | -> {key: row dict}."""
    path = path or os.path.join(PROFILES, "COUNTS.md")
    out = {}
    if not os.path.exists(path):
        return out
    for line in open(path):
        cells = [c.strip().strip("`") for c in line.strip().strip("|").split("|")]
        if len(cells) < 4 or cells[0] in ("key", "") or set(cells[0]) <= set("-: "):
            continue
        out[cells[0]] = dict(file=cells[1], labels=[x.strip() for x in cells[2].split(",")], source_hash=cells[3])
    return out


def kernel_counts(key, kernel_regex, hashes):
    """Instruction counts of the launches recorded under `key`: {label: {inst, flop, dadd, dmul, dfma, pipe_pct,
    dram_bytes, ncu_ms}} plus a status string (None = usable).  `hashes` = (tree hash, hash built into libfe.so)."""
    import re
    idx = load_counts_index()
    row = idx.get(key)
    if row is None:
        return None, f"no capture recorded for '{key}' in profiles/COUNTS.md"
    path = os.path.join(PROFILES, row["file"])
    if not os.path.exists(path):
        return None, f"profiles/{row['file']} is missing"
    launches = [l for l in parse_ncu_metrics_csv(path) if re.search(kernel_regex, l["kernel"])]
    if len(launches) != len(row["labels"]):
        return None, f"profiles/{row['file']} has {len(launches)} matching launches, COUNTS.md names {len(row['labels'])}"
    out = {}
    for lab, l in zip(row["labels"], launches):
        m = l["metrics"]
        ops = {o: m.get(f"smsp__sass_thread_inst_executed_op_{o}_pred_on.sum") for o in FP64_OPS}
        if any(v is None for v in ops.values()):
            return None, f"profiles/{row['file']} lacks the smsp__sass_thread_inst_executed_op_d* counters"
        out[lab] = dict(ops, inst=sum(ops.values()), flop=ops["dadd"] + ops["dmul"] + 2 * ops["dfma"],
                        pipe_pct=m.get("sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_elapsed"),
                        dram_bytes=(m.get("dram__bytes_read.sum", 0.0) + m.get("dram__bytes_write.sum", 0.0)) or None,
                        ncu_ms=m.get("gpu__time_duration.sum", 0.0) * 1e-6, kernel=l["kernel"], grid=l["grid"],
                        file=f"profiles/{row['file']}")
    tree, built = hashes
    if row["source_hash"] != tree or tree != built:
        return out, (f"stale: capture profiles/{row['file']} was taken at kernel-source hash {row['source_hash']}, the tree is at "
                     f"{tree}, libfe.so was built from {built}; re-profile (profiles/COUNTS.md says how)")
    return out, None


# ----------------------------------------------------------------------------------------------------
class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        hot = [s for s in sm if s > 0.5 * (max(mx) if mx else 1)] or sm
        return {"sm_mhz": statistics.median(hot) if hot else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ----------------------------------------------------------------------------------------------------
# the oracle as CPU baseline / reference arm
# ----------------------------------------------------------------------------------------------------
def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.lower().startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_sample(w, T, n_delta, nthreads=None, columns=1):
    """Time the oracle on `columns` (q, h) columns of the workload with n_delta evenly spaced Delta values each."""
    from oracle import fe_oracle as O
    O.set_num_threads(nthreads if nthreads else (os.cpu_count() or 1))
    ids = np.unique(np.linspace(0, w.nd - 1, n_delta).round().astype(int))
    cols = [(w.nq // 2, w.nh // 2), (w.nq // 4, (3 * w.nh) // 4), ((3 * w.nq) // 4, w.nh // 4)][:columns]
    t0 = time.perf_counter()
    vals = [O.omega_column(w.params, w.N, T, w.q[iq], w.h[ih], w.delta[ids]) for iq, ih in cols]
    dt = time.perf_counter() - t0
    evals = w.N * w.N * len(ids) * len(cols)
    oracle_sample.last = dict(T=T, cols=cols, ids=ids, values=vals)       # bench.py's parity figure reuses these columns
    return evals / dt, dt, len(ids), O.num_threads(), cols


def parity_vs_oracle_columns(om_gpu, col_idx, cols):
    """Parity figure of the Omega bench line: the oracle columns cpu_baseline computed anyway (cols = oracle_sample.last)
    against ONE untimed fe_omega_grid launch of exactly the shape the timed loop runs (om_gpu[row, ih, id], row r = q number
    col_idx[r] of the workload).  Elementwise max relative error; argmin compared when the whole Delta list was sampled."""
    ids, errs, arg_eq, ncmp = cols["ids"], [], [], 0
    pos = {int(g): r for r, g in enumerate(col_idx)}
    for (iq, ih), ref in zip(cols["cols"], cols["values"]):
        if iq not in pos or pos[iq] >= om_gpu.shape[0]:
            continue                                     # a q-value another rank owns
        got = om_gpu[pos[iq], ih]
        errs.append(float(np.max(np.abs(got[ids] - ref) / np.abs(ref))))
        ncmp += 1
        if len(ids) == om_gpu.shape[2]:
            arg_eq.append(int(np.argmin(got)) == int(np.argmin(ref)))
    return {"max_rel_err": max(errs) if errs else None, "columns": ncmp, "delta_values_per_column": int(len(ids)), "T": cols["T"],
            "argmin_equal": (all(arg_eq) if arg_eq else None), "tolerance": 1e-12,
            "what": "oracle columns of cpu_baseline vs one untimed fe_omega_grid launch of the timed shape (all q of the step, same eval mode)"}


def cpu_baseline(w, T, n_delta_all, n_delta_one):
    """the oracle on 1 thread and on all host cores (the paper's serial / OpenMP pair)."""
    ncores = os.cpu_count() or 1
    v1, dt1, nd1, th1, cols1 = oracle_sample(w, T, n_delta_one, nthreads=1)
    va, dta, nda, tha, colsa = oracle_sample(w, T, n_delta_all, nthreads=ncores, columns=2)
    cpu_baseline.columns = oracle_sample.last
    return {"value": va, "unit": UNIT, "cores": tha, "kind": "oracle", "seconds": dta, "cpu_model": cpu_model(),
            "sample": (f"{len(colsa)} of {w.nq * w.nh} (q,h) columns of {w.name} {colsa} x {nda} of {w.nd} Delta, "
                       f"full {w.N}x{w.N} k-sum, T={T}, OpenMP over Delta"),
            "one_thread": {"value": v1, "cores": th1, "seconds": dt1,
                           "sample": f"1 column {cols1} x {nd1} of {w.nd} Delta, full k-sum, T={T}"},
            "all_cores_over_one_thread": va / v1}


def run_reference(args, w):
    """Reference arm of this tier: the oracle on the host cores, same metric/config; rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    T = w.T[0]
    n_delta = args.ref_deltas
    for _ in range(args.warmup):
        oracle_sample(w, T, max(2, n_delta // 8))
    times, evals = [], 0
    for _ in range(args.steps):
        v, dt, nd_used, cores, col = oracle_sample(w, T, n_delta)
        times.append(dt)
        evals += w.N * w.N * nd_used
    value = evals / sum(times)
    sample = (f"per step: 1 of {w.nq * w.nh} (q,h) columns {col} x {nd_used} of {w.nd} Delta, "
              f"full {w.N}x{w.N} k-sum, T={T}")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / len(times),
            "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "N": w.N, "nq": w.nq, "nh": w.nh, "nd": w.nd, "T": list(w.T)},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                             "cpu_model": cpu_model()},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------------------
# N > 1: the rank -> q mapping and the gather of the minima (driven on CPU by tests/test_bench_host_logic.py)
# ----------------------------------------------------------------------------------------------------
def rank_q(w_q, rank, world, scaling):
    """q-values of this rank.  strong: the workload's own q list, round-robin (sharding.shard_q).  weak: every rank
    scans the whole q list (fixed work per GPU, equal on every rank; global column index = rank * nq + i).
    Returns (global column indices, q array, total number of columns of the job)."""
    q = np.ascontiguousarray(w_q, dtype=np.float64).reshape(-1, 2)
    if scaling == "strong":
        idx, qs = sharding.shard_q(q, rank, world)
        return idx, qs, q.shape[0]
    if scaling == "weak":
        return np.arange(rank * q.shape[0], (rank + 1) * q.shape[0], dtype=np.int64), q, q.shape[0] * world
    raise ValueError(scaling)


def job_reduce(x, op, world, device="cuda", group=None):
    """One number per rank -> the job's number on every rank: op = "sum" (units all ranks processed in a step) or "max"
    (the slowest rank's time: what the whole job takes).  The only collectives bench.py issues besides the gather of the
    minima; world == 1 returns x unchanged.  `device` is "cuda" under NCCL, "cpu" in the gloo test of this function."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op={"sum": dist.ReduceOp.SUM, "max": dist.ReduceOp.MAX}[op], group=group)
    return float(t.item())


def sharded_scan(evaluate, w_q, h, delta, rank, world, scaling, group=None):
    """One multi-GPU pass: this rank evaluates its q-values with `evaluate(q, h, delta) -> (idx, delta*, omega*)`
    (FreeEnergy.scan_host on a GPU; a stub in the CPU test) and the minima of all ranks are gathered in column order."""
    idx, qs, ntotal = rank_q(w_q, rank, world, scaling)
    nh = int(np.asarray(h).reshape(-1).shape[0])
    if len(idx):
        i, ds, os_ = evaluate(qs, h, delta)
    else:
        i, ds, os_ = np.empty((0, nh), np.int32), np.empty((0, nh)), np.empty((0, nh))
    return sharding.gather_columns(idx, dict(idx=i, delta_star=ds, omega_star=os_), ntotal, rank, world, group)


# ----------------------------------------------------------------------------------------------------
def roofline_base(kernel_desc, dfma_rate):
    return {"bound": "alu", "kernel": kernel_desc,
            "unit": "Tinst/s (FP64-pipe thread-instructions: DFMA, DADD, DMUL each count 1)",
            "peak": PEAK_DFMA_PER_S / 1e12,
            "peak_source": "nominal: 148 SM x 64 FP64 lanes x 1.965 GHz (DESIGN.md section 6); MEASURED_PEAKS.json has no fp64 entry",
            "peak_measured_dfma_probe": dfma_rate / 1e12, "peak_tflops": PEAK_TFLOPS,
            "achieved": None, "frac": None, "traffic": None}


def apply_counts(roof, counts, status, labels, k_ms, units_per_launch, unit_name):
    """Fill achieved / frac from the parsed ncu counts of the launches `labels` (one per timed step) and the CUDA-event
    durations k_ms of the same steps."""
    if counts is None or status is not None:
        roof["stale_counts"] = status
        if counts is None:
            return
    missing = [l for l in labels if l not in counts]
    if missing:
        roof["stale_counts"] = f"no recorded launch for {sorted(set(missing))}"
        return
    inst = sum(counts[l]["inst"] for l in labels)
    flop = sum(counts[l]["flop"] for l in labels)
    secs = sum(k_ms) * 1e-3
    per_label = {l: {"fp64_inst_per_" + unit_name: counts[l]["inst"] / units_per_launch,
                     "dadd_dmul_dfma_per_" + unit_name: [counts[l][o] / units_per_launch for o in FP64_OPS],
                     "ncu_fp64_pipe_active_pct": counts[l]["pipe_pct"], "ncu_launch_ms": counts[l]["ncu_ms"],
                     "dram_bytes": counts[l]["dram_bytes"], "kernel": counts[l]["kernel"], "grid": counts[l]["grid"]}
                 for l in sorted(set(labels))}
    roof["counts"] = {"source": counts[labels[0]]["file"], "per_launch": per_label}
    tr = [counts[l]["dram_bytes"] for l in labels if counts[l]["dram_bytes"]]
    roof["traffic"] = sum(tr) / len(tr) if tr else None
    if status is not None:
        return                                   # stale: show what the capture said, claim nothing
    ach = inst / secs / 1e12
    tfl = flop / secs / 1e12
    roof.update({"achieved": ach, "frac": ach / (PEAK_DFMA_PER_S / 1e12),
                 "frac_of_measured_dfma_peak": ach / roof["peak_measured_dfma_probe"],
                 "fp64_inst_per_" + unit_name: inst / (units_per_launch * len(labels)),
                 "achieved_tflops": tfl, "frac_tflops": tfl / PEAK_TFLOPS})


def run_chi(args):
    """q map of the static Cooper-pair susceptibility (Appendix C).  One step = fe_pair_susceptibility
    over the whole q list (K0 trig, [KB bands], K-chi k-sum, finish).  value = (k, q) points per second."""
    import torch
    from paper_1412_8754_b200 import fe
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a B200: no CUDA device visible (there is no CPU fallback)")
    torch.cuda.set_device(0)
    w = W.chi_map(model=args.chi_model, N=args.chi_N, nside=args.chi_nside, T=0.001, h=0.025)
    F = fe.FreeEnergy(w.params, w.N, w.T[0])
    F.enable_timing(True)
    stream = torch.cuda.current_stream()
    nb = w.nbands
    chi = torch.empty((w.nq, nb, nb), dtype=torch.float64, device="cuda")
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device="cuda")
    hz = float(w.h[0])
    for _ in range(args.warmup):
        F.pair_susceptibility(w.q, hz, out=chi, stream=stream)
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    sampler.start()
    l0 = F.launch_count()
    step_ms, k_ms = [], []
    for _ in range(args.steps):
        flush.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        F.pair_susceptibility(w.q, hz, out=chi, stream=stream)
        e1.record(stream)
        e1.synchronize()
        step_ms.append(e0.elapsed_time(e1))
        k_ms.append(F.last_ksum()[0])
    torch.cuda.synchronize()
    launches = F.launch_count() - l0
    clocks = sampler.stop()
    points = w.N * w.N * w.nq
    value = points * args.steps / (sum(step_ms) * 1e-3)
    host = torch.empty((w.nq, nb, nb), dtype=torch.float64).pin_memory()
    hq = torch.from_numpy(w.q.copy()).pin_memory().numpy()
    e2e_steps = max(5, min(args.steps, 10))
    e2e_steps += (-e2e_steps) % len(temps)           # whole cycles of the alternating temperatures: the same mix as an even K
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        F.pair_susceptibility(hq, hz, out=chi, stream=stream)
        host.copy_(chi, non_blocking=True)
        torch.cuda.synchronize()
    e2e = points * e2e_steps / (time.perf_counter() - t0)
    dfma_rate, _ = fe.fp64_peak_probe()
    roofline = roofline_base(f"fe_chi_kernel<{nb}, {w.params['form_factor']}>", dfma_rate)
    roofline.update({"avg_launch_ms": sum(k_ms) / len(k_ms), "kernel_share_of_step": sum(k_ms) / sum(step_ms)})
    counts, status = kernel_counts(f"chi/{w.name}", "fe_chi_kernel", (fe.source_hash(), fe.built_source_hash()))
    apply_counts(roofline, counts, status, ["map"] * len(k_ms), k_ms, points, "kq_point")
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import fe_oracle as O
        O.set_num_threads(os.cpu_count() or 1)
        nsamp = max(1, min(w.nq, O.num_threads()))
        t0 = time.perf_counter()
        ref = O.pair_susceptibility(w.params, w.N, w.T[0], w.q[:nsamp], hz)
        dt = time.perf_counter() - t0
        err = float(np.max(np.abs(chi[:nsamp].cpu().numpy() - ref) / np.abs(ref).max()))
        cpu = {"value": w.N * w.N * nsamp / dt, "unit": "(k, q) points/s", "cores": O.num_threads(), "kind": "oracle",
               "cpu_model": cpu_model(), "seconds": dt,
               "sample": f"first {nsamp} of {w.nq} q-points, full {w.N}x{w.N} k-sum", "max_rel_err_vs_gpu": err}
    line = {"metric": "pair-susceptibility (k, q) point evaluations/s (all band pairs, fp64)", "value": value,
            "unit": "(k, q) points/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": sum(step_ms) / len(step_ms), "ms_per_step_median": statistics.median(step_ms),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "N": w.N, "nq": w.nq, "bands": nb, "T": w.T[0], "h": hz,
                       "pair_terms_per_step": points * nb * nb, "l2": "flushed between timed steps (256 MB memset)"},
            "e2e": {"value": e2e, "unit": "(k, q) points/s", "steps": e2e_steps, "h2d_bytes_per_step": 16 * w.nq,
                    "d2h_bytes_per_step": 8 * w.nq * nb * nb},
            "gpu_launches": launches, "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)


def run_paper(args):
    """Context run in the shape of the paper's own benchmark (Fig. 4): one q, one h, 200 Delta,
    N = 2000 (two-band model), timed per evaluation mode: library default, the direct Eq. 4 / Eq. 5 form, and the paper's
    SP / SPFM builds.  Prints the numbers BASELINE.md section 3 quotes (another machine and decade than the paper's K40:
    context, not a target)."""
    import torch
    from paper_1412_8754_b200 import fe
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a B200: no CUDA device visible (there is no CPU fallback)")
    torch.cuda.set_device(0)
    w = W.paper_shaped(args.paper_N)
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device="cuda")
    omega = torch.empty((w.nq, w.nh, w.nd), dtype=torch.float64, device="cuda")
    modes, launches = {}, 0
    with fe.FreeEnergy(w.params, w.N, w.T[0]) as F:
        for name in ("default", "direct", "sp", "spfm"):
            F.set_eval_mode(fe.EVAL_DIRECT if name == "direct" else fe.EVAL_COOP_EO)

            def step():
                if name in ("sp", "spfm"):
                    F.omega_grid_sp(w.q, w.h, w.delta, fast_math=name == "spfm", out=omega, stream=stream)
                else:
                    F.omega_grid(w.q, w.h, w.delta, out=omega, stream=stream)
                return F.argmin(omega, w.delta, stream=stream)
            for _ in range(args.warmup):
                step()
            torch.cuda.synchronize()
            ms = []
            l0 = F.launch_count()
            for _ in range(args.steps):
                flush.zero_()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                res = step()
                e1.record(stream)
                e1.synchronize()
                ms.append(e0.elapsed_time(e1))
            launches += F.launch_count() - l0
            modes[name] = {"ms_median": statistics.median(ms), "ms_mean": sum(ms) / len(ms),
                           "kernel_mode_run": F.last_launch_info()["mode"], "delta_star": float(res[1].reshape(-1)[0].item())}
    evals = w.N * w.N * w.nq * w.nh * w.nd
    cpu = None
    if not args.no_cpu_baseline:
        v1, dt1, nd1, th1, _ = oracle_sample(w, w.T[0], 8, nthreads=1)
        va, dta, nda, tha, _ = oracle_sample(w, w.T[0], w.nd)
        cpu = {"value": va, "unit": UNIT, "cores": tha, "kind": "oracle", "seconds": dta, "cpu_model": cpu_model(),
               "sample": f"the whole workload ({nda} Delta), OpenMP over Delta (PAPER.md:161)",
               "one_thread": {"value": v1, "cores": th1, "seconds": dt1, "sample": f"{nd1} of {w.nd} Delta"}}
    line = {"metric": METRIC, "value": evals / (modes["default"]["ms_mean"] * 1e-3), "unit": UNIT, "n_gpus": 1,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": modes["default"]["ms_mean"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "N": w.N, "nq": w.nq, "nh": w.nh, "nd": w.nd, "T": w.T[0],
                       "shape": "PAPER.md:186 benchmark shape (1 q, 200 Delta, N x N); context only",
                       "l2": "flushed between timed steps (256 MB memset)"},
            "modes_ms": modes, "gpu_launches": launches, "cpu_baseline": cpu,
            "paper": {"K40_SPFM_vs_OpenMP": 19.2, "K40_SPFM_vs_one_core": 119.1, "K40_DP_vs_OpenMP": 7.0,
                      "source": "PAPER.md:194 (i7-3960X, Tesla K40 @ 875 MHz, N = 2000)"}}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=6)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--mode", default="coop_eo", choices=["coop_eo", "coop", "factored", "direct", "windowed", "sp", "spfm", "verified_sp", "verified_spfm"],
                    help="coop_eo = library default (early-out); coop = dense variant (every pair multiplied out)")
    ap.add_argument("--scaling", default="strong", choices=["strong", "weak"],
                    help="N > 1 GPUs: strong = the config's own q list split round-robin over the ranks; weak = every rank scans the whole q list")
    ap.add_argument("--shape", type=int, default=0, help="block shape of the cooperative kernel (0 = auto)")
    ap.add_argument("--config", type=int, default=4, help="4 = BASELINE.json headline config; 6 = same shape, three-band model")
    ap.add_argument("--q-per-step", type=int, default=0, help="q-values per step (0 = the rank's whole q list)")
    ap.add_argument("--tile", type=int, default=0)
    ap.add_argument("--ref-deltas", type=int, default=64)
    ap.add_argument("--cpu-baseline-deltas", type=int, default=512)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-dense", action="store_true", help="skip the extra timing of the dense variant")
    ap.add_argument("--workload", default="omega", choices=["omega", "chi", "paper"],
                    help="omega = the free-energy scan (BASELINE.json metric); chi = pair-susceptibility q map (SURVEY 8f-4); "
                         "paper = the paper's own benchmark shape (1 q, 200 Delta, N = 2000), context only")
    ap.add_argument("--chi-model", type=int, default=2)
    ap.add_argument("--chi-N", type=int, default=1024)
    ap.add_argument("--chi-nside", type=int, default=48)
    ap.add_argument("--paper-N", type=int, default=2000)
    args = ap.parse_args()
    if args.workload == "chi":
        return run_chi(args)
    if args.workload == "paper":
        return run_paper(args)

    w = W.config(args.config)
    if args.impl == "reference":
        return run_reference(args, w)

    import torch
    import torch.distributed as dist
    from paper_1412_8754_b200 import fe

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a B200: no CUDA device visible (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        os.environ.setdefault("NCCL_DEBUG", "INFO")      # keep NCCL's log on (transport, NVLS) for the scaling record
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    fe.lib()
    hashes = (fe.source_hash(), fe.built_source_hash())

    # ---- workload of this rank: the tested sharding code owns the mapping (sharding.shard_q via rank_q) ----
    col_idx, q_all, ncols_job = rank_q(w.q, rank, world, args.scaling)
    nq_rank = len(q_all)
    nq_step = min(args.q_per_step or nq_rank, max(nq_rank, 1))
    temps = list(w.T)
    sp_mode = args.mode in ("sp", "spfm", "verified_sp", "verified_spfm")   # the paper's SP / SPFM builds
    mode = {"coop": fe.EVAL_COOP, "factored": fe.EVAL_FACTORED, "direct": fe.EVAL_DIRECT,
            "windowed": fe.EVAL_WINDOWED}.get(args.mode, fe.EVAL_COOP_EO)

    F = fe.FreeEnergy(w.params, w.N, temps[0])
    F.set_eval_mode(mode)
    F.set_tuning(args.tile, 0)
    F.set_coop_shape(args.shape)
    F.enable_timing(True)
    stream = torch.cuda.current_stream()
    omega = torch.empty((max(nq_step, 1), w.nh, w.nd), dtype=torch.float64, device="cuda")
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device="cuda")    # 256 MB > 126 MB L2

    def q_of(step):
        s = (step * nq_step) % max(nq_rank, 1)
        return np.ascontiguousarray(np.take(q_all, range(s, s + nq_step), axis=0, mode="wrap"))

    verified = []

    def one_step(step):
        F.set_temperature(temps[step % len(temps)])
        if nq_rank == 0:                                # more ranks than q-values: this rank idles
            return None
        if args.mode in ("sp", "spfm"):
            F.omega_grid_sp(q_of(step), w.h, w.delta, fast_math=args.mode == "spfm", out=omega, stream=stream)
        elif sp_mode:
            r = F.scan_verified(q_of(step), w.h, w.delta, screen={"verified_sp": "sp", "verified_spfm": "spfm"}[args.mode],
                                stream=stream)
            verified.append({"delta_values_verified_in_fp64": r[3], "of": w.nd, "columns_whose_minimum_moved": r[4],
                             "columns": nq_step * w.nh})
            return r[:3]
        else:
            F.omega_grid(q_of(step), w.h, w.delta, out=omega, stream=stream)
        return F.argmin(omega, w.delta, stream=stream)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    evals_rank_step = w.N * w.N * nq_step * w.nh * w.nd
    # units all ranks process per step (strong: the job's q list once; weak: once per rank)
    evals_job_step = job_reduce(evals_rank_step, "sum", world)
    for s in range(args.warmup):
        one_step(s)
    barrier()

    sampler = ClockSampler(local_rank)
    sampler.start()
    launches0 = F.launch_count()
    step_ms, ksum_ms, step_T, band_evals = [], [], [], 0.0
    slot_kinds = {}                                     # per temperature: what the timed launches were made of (in-run counters)
    tiles_by_T = {}                                     # per temperature: block tile the library chose
    res = None
    barrier()
    t_wall0 = time.perf_counter()
    for s in range(args.steps):
        flush.zero_()                                   # L2 flush between timed iterations (outside the events)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        res = one_step(args.warmup + s)
        e1.record(stream)
        e1.synchronize()
        step_ms.append(e0.elapsed_time(e1))
        step_T.append(temps[(args.warmup + s) % len(temps)])
        if nq_rank:
            ms, be = F.last_ksum()
            ksum_ms.append(ms)
            band_evals = be
            li = F.last_launch_info()
            tiles_by_T[f"T={step_T[-1]:g}"] = f"{li['th']}x{li['td']}"
    barrier()
    t_wall = time.perf_counter() - t_wall0
    launches = F.launch_count() - launches0
    clocks = sampler.stop()
    if args.mode in ("coop", "coop_eo") and nq_rank:
        # what the launches were made of: the kernel counts its slot kinds with global atomics, so the counters are OFF in
        # every timed launch above and collected here in one extra, untimed step per temperature (same inputs: the
        # classification does not depend on timing)
        F.enable_slot_counts(True)
        for s in range(len(temps)):
            one_step(args.warmup + s)
            if F.last_launch_info()["mode"] not in (fe.EVAL_COOP, fe.EVAL_COOP_EO):
                break                                   # a grid far smaller than a block tile ran on the per-thread kernel: no slots
            c = F.slot_counts()                         # waits for the launch, reads five counters
            tot = c["dense"] + c["a_dominated"] + c["b_dominated"]
            slot_kinds[f"T={temps[(args.warmup + s) % len(temps)]:g}"] = {k: v / tot for k, v in c.items()}
        F.enable_slot_counts(False)
    idx_check = int(res[0].sum().item()) if res is not None else 0      # device->host read of the step's result

    total_ms = sum(step_ms)
    total_ms_max = job_reduce(total_ms, "max", world)
    value = evals_job_step * args.steps / (total_ms_max * 1e-3)

    # ---- the dense variant of the same kernel (every pair multiplied out), timed beside the early-out default:
    #      north_star's FP64-roofline target is read on it ----
    dense = None
    if args.mode == "coop_eo" and not args.no_dense and nq_rank:
        F.set_eval_mode(fe.EVAL_COOP)
        one_step(0); one_step(1)
        barrier()
        d_ms, dk_ms, d_T = [], [], []
        for s in range(2 * len(temps)):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            one_step(s)
            e1.record(stream)
            e1.synchronize()
            d_ms.append(e0.elapsed_time(e1))
            dk_ms.append(F.last_ksum()[0])
            d_T.append(temps[s % len(temps)])
        barrier()
        dinfo = F.last_launch_info()
        dense = {"eval_mode": "coop", "steps": len(d_ms), "value": evals_rank_step * len(d_ms) / (sum(d_ms) * 1e-3), "unit": UNIT,
                 "ms_per_step": sum(d_ms) / len(d_ms), "ms_per_step_median": statistics.median(d_ms), "ksum_ms": sum(dk_ms) / len(dk_ms),
                 "ksum_ms_steps": [[f"T={t:g}", round(x, 3)] for t, x in zip(d_T, dk_ms)],
                 "tile": [dinfo["th"], dinfo["td"]], "grid": dinfo["grid"]}
        droof = roofline_base("dense", 1.0)
        dcounts, dstatus = kernel_counts(f"omega/coop/{w.name}/q{nq_step}", "fe_ksum", hashes)
        apply_counts(droof, dcounts, dstatus, [f"T={x:g}" for x in d_T], dk_ms, band_evals, "band_eval")
        for k in ("achieved", "frac", "achieved_tflops", "frac_tflops", "fp64_inst_per_band_eval", "counts", "stale_counts"):
            if k in droof:
                dense["roofline_" + k] = droof[k]
        F.set_eval_mode(mode)

    # ---- the opt-in mirror-symmetry variant (fe_set_symmetry), timed beside the headline and NEVER folded
    #      into `value`: when every q of the step is invariant under a lattice mirror (config 4: q on the diagonal) the
    #      k-sum visits one k-point per orbit.  `value` counts the nominal N x N k-points, as the headline does. ----
    symv = None
    if args.mode == "coop_eo" and not args.no_dense and nq_rank and w.nbands < 3:
        F.set_symmetry(True)
        one_step(0); one_step(1)
        barrier()
        s_ms, s_sym = [], 0
        for s in range(2 * len(temps)):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            one_step(s)
            e1.record(stream)
            e1.synchronize()
            s_ms.append(e0.elapsed_time(e1))
            s_sym = F.last_symmetry()
        barrier()
        F.set_symmetry(False)
        if s_sym:
            symv = {"what": "fe_set_symmetry(1): k-sum over one k-point per mirror orbit (weights 2 / 1); same Omega to rounding, "
                            "parity-tested against the oracle; reported separately, not the headline",
                    "mirror": {1: "k_y -> -k_y", 2: "k_x -> -k_x", 3: "k_x <-> k_y"}[s_sym], "steps": len(s_ms),
                    "value": evals_rank_step * len(s_ms) / (sum(s_ms) * 1e-3), "unit": UNIT + " (nominal N x N k-points)",
                    "ms_per_step": sum(s_ms) / len(s_ms), "ms_per_step_median": statistics.median(s_ms)}

    # ---- e2e: host buffers through fe_scan_host (pinned), copies inside the timed region; N > 1: + gather of the minima ----
    pin = lambda shape, dt: torch.empty(shape, dtype=dt).pin_memory().numpy()    # noqa: E731
    nqe = max(nq_rank, 1)
    out = dict(omega=pin((nqe, w.nh, w.nd), torch.float64), idx=pin((nqe, w.nh), torch.int32),
               delta_star=pin((nqe, w.nh), torch.float64), omega_star=pin((nqe, w.nh), torch.float64))
    hq = [pin((nqe, 2), torch.float64) for _ in range(2)]
    hh, hd = pin((w.nh,), torch.float64), pin((w.nd,), torch.float64)
    hh[:] = w.h
    hd[:] = w.delta
    e2e_steps = max(5, min(args.steps, 10))
    if sp_mode:
        F.set_eval_mode(fe.EVAL_COOP_EO)       # e2e below is the fp64 host path; the SP numbers are the device-timed ones

    def scan_host_eval(qs, h, d):
        buf = hq[scan_host_eval.n % 2][:len(qs)]
        scan_host_eval.n += 1
        buf[:] = qs
        o = {k: v[:len(qs)] for k, v in out.items()}
        _, i, ds, os_ = F.scan_host(buf, h, d, out=o, stream=stream)      # synchronous: returns with results on the host
        return i, ds, os_
    scan_host_eval.n = 0

    F.set_temperature(temps[0])
    gathered = sharded_scan(scan_host_eval, w.q, hh, hd, rank, world, args.scaling)      # warm-up
    barrier()
    t0 = time.perf_counter()
    for s in range(e2e_steps):
        F.set_temperature(temps[s % len(temps)])
        gathered = sharded_scan(scan_host_eval, w.q, hh, hd, rank, world, args.scaling)
    torch.cuda.synchronize()
    e2e_seconds = job_reduce(time.perf_counter() - t0, "max", world)
    evals_job_scan = w.N * w.N * ncols_job * w.nh * w.nd
    e2e_value = evals_job_scan * e2e_steps / e2e_seconds
    assert gathered["idx"].shape == (ncols_job, w.nh)
    h2d = 8 * (2 * nq_rank + w.nh + 2 * w.nd)           # q, h, Delta^2 lists + Delta list for the argmin
    d2h = 8 * nq_rank * w.nh * w.nd + nq_rank * w.nh * (4 + 8 + 8)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (K1 k-sum): counts from the committed ncu capture of these launches ----
    info = F.last_launch_info()
    info["block"] = 256
    if info["mode"] in (fe.EVAL_COOP, fe.EVAL_COOP_EO):
        info["block"] = next((c[4] for c in fe.coop_shapes() if (c[2], c[3]) == (info["th"], info["td"])), 128)
    k_ms = sum(ksum_ms) / len(ksum_ms)
    dfma_rate, _ = fe.fp64_peak_probe()
    # Primary roofline = FP64-pipe lane-instructions/s: a DADD or DMUL occupies an FP64 lane for a cycle exactly like a
    # DFMA, and the kernel's pair update acc *= (A + B) has no fused form, so instructions (not flops, which count a
    # DFMA twice) measure how busy the bounding unit is; frac_tflops (DFMA = 2) is printed beside it.
    tile_desc = ", ".join(f"{k}: {v}" for k, v in sorted(tiles_by_T.items())) if len(set(tiles_by_T.values())) > 1 else f"{info['th']}x{info['td']}"
    roofline = roofline_base(f"k-sum kernel ({args.mode}, block tile {tile_desc}, grid {info['grid']} x {info['block']})", dfma_rate)
    roofline.update({"avg_launch_ms": k_ms, "median_launch_ms": statistics.median(ksum_ms), "band_evals_per_launch": band_evals,
                     "kernel_share_of_step": sum(ksum_ms) / total_ms})
    if slot_kinds:
        roofline["slot_kinds"] = {"what": "fractions of the (k, band, block tile) slots of one launch per temperature, counted by the kernel in an extra untimed step of this run (the counters are off in the timed launches): "
                                          "dense slots (and padding, relative to the same total) run through the pair products, "
                                          "dominated slots are summed without exponentials", **slot_kinds}
    if sp_mode:
        roofline["note"] = ("lower-precision builds (SURVEY 8f-2): see profiles/; avg_launch_ms is the last k-sum launch of a step "
                            "(verified_*: the fp64 pass on the candidate list); fp64-verified Delta values per step: " + str(verified[-4:]))
    else:
        counts, status = kernel_counts(f"omega/{args.mode}/{w.name}/q{nq_step}", "fe_ksum", hashes)
        apply_counts(roofline, counts, status, [f"T={x:g}" for x in step_T], ksum_ms, band_evals, "band_eval")

    cpu, parity = None, None
    if not args.no_cpu_baseline:
        cpu = cpu_baseline(w, temps[0], args.cpu_baseline_deltas, 32)
        if not sp_mode and nq_rank:
            F.set_temperature(temps[0])                 # one untimed launch of the timed shape at the oracle's temperature
            F.omega_grid(q_of(0), w.h, w.delta, out=omega, stream=stream)
            torch.cuda.synchronize()
            parity = parity_vs_oracle_columns(omega.cpu().numpy(), col_idx[:nq_step] % max(len(w.q), 1), cpu_baseline.columns)
            parity["launch"] = F.last_launch_info()

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms_max / args.steps, "ms_per_step_median": statistics.median(step_ms),
            "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "N": w.N, "nq_per_step": nq_step, "nq_job": ncols_job, "nh": w.nh, "nd": w.nd,
                       "T_alternating": temps, "eval_mode": args.mode, "band_evals_per_step": evals_rank_step * w.nbands,
                       "l2": "flushed between timed steps (256 MB memset); inputs are a few KB",
                       "parallelism": f"q-sharded x{world} ({args.scaling}; paper_1412_8754_b200.sharding), no collective on the data path"},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": e2e_steps, "api": "fe_scan_host (host buffers in/out, synchronous)" +
                    (" + all_gather of the minima" if world > 1 else "")},
            "gpu_launches": launches, "wall_s_timed_region": t_wall, "clocks": clocks, "source_hash": hashes[0],
            "roofline": roofline, "dense_variant": dense, "symmetric_variant": symv, "cpu_baseline": cpu, "parity": parity, "result_check": idx_check}
    if sp_mode:
        line["verified_per_step"] = verified[-args.steps:]
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
