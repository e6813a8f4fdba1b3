#!/usr/bin/env python
"""bench.py -- throughput of the Omega(Delta; q, h, T) hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--mode coop|factored|direct|windowed]

Workload (config.workload): BASELINE.json configs[3] "cfg4_fflo_N1024": two-band s+- model, N = 1024 x 1024 k-grid,
32 q along (1,1), 64 h, 512 Delta -- the configuration north_star quotes its FP64-roofline target on.
One STEP = one pass of the whole hot path over one batch: fe_omega_grid (K0 trig, KS constant sum, K1 k-sum,
K2 finish) + fe_argmin over the batch's full (q, h, Delta) grid at one temperature; successive steps alternate
T = 0.001 / 0.01 (config 4 names both).  The batch is `--q-per-step` q-values of the config (default: all 32),
so a default step is the whole 1.1e12-evaluation scan.

Output: ONE JSON line (rank 0).  value = k-point x parameter evaluations per second, whole job, inputs resident
(device timing with CUDA events per step, L2 flushed between steps, max over ranks).  e2e = same metric through
fe_scan_host with HOST buffers (lists H2D, Omega + minima D2H inside the timed region).
roofline: bound "alu" (plain FP64 pipe; no contraction, HBM negligible), see DESIGN.md "Roofline".
cpu_baseline: the oracle (oracle/fe_oracle.c) as it stands, timed on this host's cores on a bounded sample.
`--impl reference` times the oracle instead (the reference arm of this tier).
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

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1412_8754_b200 import workloads as W  # noqa: E402

METRIC = "Omega evaluations/s (k-points x grid points, fp64)"
UNIT = "k-point x (q,h,Delta) evaluations/s"

# FP64-pipe instructions and flops EXECUTED per (k, band, q, h, Delta) term by the k-sum kernel as built
# (DESIGN.md "Roofline").  coop / factored: ncu counters smsp__sass_thread_inst_executed_op_{dfma,dadd,dmul}_pred_on of the
# cfg4 launch (profiles/); direct: cuobjdump -sass count of the band-loop body (every term takes the same path).
KERNEL_COUNTS = {
    # (eval mode, (TH, TD)): (fp64 pipe instructions, flops [DFMA = 2, DADD/DMUL = 1]) per band-eval, source
    ("coop_eo", (64, 128)): (0.5391, 0.6683, "ncu on the benchmark's own launches (whole 32-q step), profiles/r1p_fullstep_eo.csv: mean of the "
                              "T = 0.01 launch (0.662 = 0.252 DADD + 0.269 DMUL + 0.141 DFMA) and the T = 0.001 launch (0.416 = 0.142 + 0.158 + 0.117)"),
    ("coop_eo", (64, 128), 3): (0.3307, 0.4419, "ncu, whole step, profiles/r1p_fullstep_b3_eo.csv (T = 0.001: 0.102 DADD + 0.118 DMUL + 0.111 DFMA)"),
    ("coop", (64, 128)): (2.368, 2.647, "ncu, whole step, profiles/r1p_fullstep_dense.csv (1.032 DADD + 1.057 DMUL + 0.279 DFMA)"),
    ("coop", (64, 128), 3): (2.375, 2.656, "ncu, profiles/r1e_ksum_coop_3band_raw.csv (1.036 DADD + 1.059 DMUL + 0.281 DFMA)"),
    ("factored", (8, 4)): (8.49, 13.31, "ncu, profiles/r1b_ksum_factored_8x4_raw.csv"),
    ("factored", (16, 4)): (4.20, 5.62, "ncu, profiles/r1c_ksum_factored_16x4_raw.csv"),
    ("direct", (4, 4)): (40.6, 61.3, "SASS count"),
    ("direct", (8, 4)): (39.4, 59.4, "SASS count"),
}
# DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) of ONE k-sum launch of the default whole-step benchmark
# (profiles/r1p_fullstep_*.csv: ~10 MB read, ~255 MB written = the partial sums [ksplit][nq*nh*nd]; three-band: + 1.1 GB
# of band tables read).  Against 6.5 TB/s this is < 1 % of the launch time: HBM is idle, the bound is the FP64 pipe.
KERNEL_TRAFFIC = {"coop_eo": 265.0e6, "coop": 280.0e6, ("coop", 3): 1.40e9, ("coop_eo", 3): 1.404e9}   # whole-step launches (r1p_fullstep_*)
SM_COUNT, FP64_LANES_PER_SM, SM_MAX_GHZ = 148, 64, 1.965
PEAK_DFMA_PER_S = SM_COUNT * FP64_LANES_PER_SM * SM_MAX_GHZ * 1e9        # 1.861e13 thread-level FP64 instr/s
PEAK_TFLOPS = 2 * PEAK_DFMA_PER_S / 1e12                                  # 37.2 TFLOP/s nominal


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


def oracle_sample(w, T, n_delta, nthreads=None):
    """Time the oracle on ONE (q, h) column of the workload with the first n_delta... evenly spaced Delta values."""
    from oracle import fe_oracle as O
    if nthreads:
        O.set_num_threads(nthreads)
    ids = np.unique(np.linspace(0, w.nd - 1, n_delta).round().astype(int))
    iq, ih = w.nq // 2, w.nh // 2
    t0 = time.perf_counter()
    O.omega_column(w.params, w.N, T, w.q[iq], w.h[ih], w.delta[ids])
    dt = time.perf_counter() - t0
    evals = w.N * w.N * len(ids)
    return evals / dt, dt, len(ids), O.num_threads(), (iq, ih)


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
    sample = (f"per step: 1 of {w.nq * w.nh} (q,h) columns (iq={col[0]}, ih={col[1]}) x {nd_used} of {w.nd} Delta, "
              f"full {w.N}x{w.N} k-sum, T={T}")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / len(times),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "N": w.N, "nq": w.nq, "nh": w.nh, "nd": w.nd, "T": list(w.T)},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# FP64-pipe instructions per (k, q) point of the susceptibility kernel (all nb^2 band pairs), ncu (profiles/r1f_*)
CHI_COUNTS = {(2,): (170.2, "ncu, profiles/r1m_chi_2band_raw.csv (89.2 DFMA + 36.5 DADD + 44.5 DMUL per (k, q) point, 4 band pairs)")}


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
    t0 = time.perf_counter()
    for _ in range(2):
        F.pair_susceptibility(hq, hz, out=chi, stream=stream)
        host.copy_(chi, non_blocking=True)
        torch.cuda.synchronize()
    e2e = points * 2 / (time.perf_counter() - t0)
    kms = sum(k_ms) / len(k_ms)
    dfma_rate, _ = fe.fp64_peak_probe()
    cnt = CHI_COUNTS.get((args.chi_model,))
    roofline = {"bound": "alu", "kernel": f"fe_chi_kernel<{nb}, {w.params['form_factor']}>", "unit": "Tinst/s (FP64-pipe thread-instructions)",
                "peak": PEAK_DFMA_PER_S / 1e12, "peak_measured_dfma_probe": dfma_rate / 1e12, "avg_launch_ms": kms,
                "kernel_share_of_step": kms * len(k_ms) / sum(step_ms), "traffic": None,
                "achieved": None, "frac": None}
    if cnt:
        ach = points * cnt[0] / (kms * 1e-3) / 1e12
        roofline.update({"achieved": ach, "frac": ach / (PEAK_DFMA_PER_S / 1e12), "fp64_inst_per_kq_point": cnt[0],
                         "counts_source": cnt[1]})
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import fe_oracle as O
        nsamp = max(1, min(w.nq, O.num_threads()))
        t0 = time.perf_counter()
        ref = O.pair_susceptibility(w.params, w.N, w.T[0], w.q[:nsamp], hz)
        dt = time.perf_counter() - t0
        err = float(np.max(np.abs(chi[:nsamp].cpu().numpy() - ref) / np.abs(ref).max()))
        cpu = {"value": w.N * w.N * nsamp / dt, "unit": "(k, q) points/s", "cores": O.num_threads(), "kind": "oracle",
               "seconds": dt, "sample": f"first {nsamp} of {w.nq} q-points, full {w.N}x{w.N} k-sum", "max_rel_err_vs_gpu": err}
    line = {"metric": "pair-susceptibility (k, q) point evaluations/s (all band pairs, fp64)", "value": value,
            "unit": "(k, q) points/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": sum(step_ms) / len(step_ms), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "N": w.N, "nq": w.nq, "bands": nb, "T": w.T[0], "h": hz,
                       "pair_terms_per_step": points * nb * nb, "l2": "flushed between timed steps (256 MB memset)"},
            "e2e": {"value": e2e, "unit": "(k, q) points/s", "h2d_bytes_per_step": 16 * w.nq, "d2h_bytes_per_step": 8 * w.nq * nb * nb},
            "gpu_launches": launches, "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=4)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--mode", default="coop_eo", choices=["coop_eo", "coop", "factored", "direct", "windowed", "sp", "spfm", "verified_sp", "verified_spfm"],
                    help="coop_eo = library default (early-out); coop = dense variant (every pair multiplied out)")
    ap.add_argument("--shape", type=int, default=0, help="block shape of the cooperative kernel (0 = auto)")
    ap.add_argument("--config", type=int, default=4, help="4 = BASELINE.json headline config; 6 = same shape, three-band model")
    ap.add_argument("--q-per-step", type=int, default=0, help="q-values per step (0 = the whole q list)")
    ap.add_argument("--tile", type=int, default=0)
    ap.add_argument("--ref-deltas", type=int, default=64)
    ap.add_argument("--cpu-baseline-deltas", type=int, default=256)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-dense", action="store_true", help="skip the extra timing of the dense variant")
    ap.add_argument("--workload", default="omega", choices=["omega", "chi"],
                    help="omega = the free-energy scan (BASELINE.json metric); chi = pair-susceptibility q map (SURVEY 8f-4)")
    ap.add_argument("--chi-model", type=int, default=2)
    ap.add_argument("--chi-N", type=int, default=1024)
    ap.add_argument("--chi-nside", type=int, default=48)
    args = ap.parse_args()
    if args.workload == "chi":
        return run_chi(args)

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
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    fe.lib()

    # ---- workload of this rank (weak scaling: every rank scans nq q-values of a `world`-times finer q grid) ----
    nq_step = args.q_per_step or w.nq
    if world > 1:
        qfine = np.linspace(w.q[0], w.q[-1], w.nq * world)
        q_all = qfine[rank::world]
    else:
        q_all = w.q
    temps = list(w.T)
    sp_mode = args.mode in ("sp", "spfm", "verified_sp", "verified_spfm")       # the paper's SP / SPFM builds
    mode = {"sp": fe.EVAL_COOP_EO, "spfm": fe.EVAL_COOP_EO, "verified_sp": fe.EVAL_COOP_EO, "verified_spfm": fe.EVAL_COOP_EO,
            "coop_eo": fe.EVAL_COOP_EO, "coop": fe.EVAL_COOP, "factored": fe.EVAL_FACTORED, "direct": fe.EVAL_DIRECT,
            "windowed": fe.EVAL_WINDOWED}[args.mode]

    F = fe.FreeEnergy(w.params, w.N, temps[0])
    F.set_eval_mode(mode)
    F.set_tuning(args.tile, 0)
    F.set_coop_shape(args.shape)
    F.enable_timing(True)
    stream = torch.cuda.current_stream()
    omega = torch.empty((nq_step, w.nh, w.nd), dtype=torch.float64, device="cuda")
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device="cuda")    # 256 MB > 126 MB L2

    def q_of(step):
        s = (step * nq_step) % len(q_all)
        return np.ascontiguousarray(np.take(q_all, range(s, s + nq_step), axis=0, mode="wrap"))

    verified_n = []

    def one_step(step):
        F.set_temperature(temps[step % len(temps)])
        if args.mode in ("sp", "spfm"):
            F.omega_grid_sp(q_of(step), w.h, w.delta, fast_math=args.mode == "spfm", out=omega, stream=stream)
        elif sp_mode:
            r = F.scan_verified(q_of(step), w.h, w.delta, fast_math=args.mode == "verified_spfm", stream=stream)
            verified_n.append(r[3])
            return r[:3]
        else:
            F.omega_grid(q_of(step), w.h, w.delta, out=omega, stream=stream)
        return F.argmin(omega, w.delta, stream=stream)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    evals_per_step = w.N * w.N * nq_step * w.nh * w.nd
    for s in range(args.warmup):
        one_step(s)
    barrier()

    sampler = ClockSampler(local_rank)
    sampler.start()
    launches0 = F.launch_count()
    step_ms, ksum_ms, band_evals = [], [], 0.0
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
        ms, be = F.last_ksum()
        ksum_ms.append(ms)
        band_evals = be
    barrier()
    t_wall = time.perf_counter() - t_wall0
    launches = F.launch_count() - launches0
    clocks = sampler.stop()
    idx_check = int(res[0].sum().item())               # device->host read of the step's result

    total_ms = sum(step_ms)
    t = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms_max = float(t.item())
    value = evals_per_step * args.steps * world / (total_ms_max * 1e-3)

    # ---- the dense variant of the same kernel (every pair multiplied out), timed beside the early-out default:
    #      north_star's FP64-roofline target is read on it ----
    dense = None
    if args.mode == "coop_eo" and not args.no_dense:
        F.set_eval_mode(fe.EVAL_COOP)
        one_step(0); one_step(1)
        barrier()
        d_ms, dk_ms = [], []
        for s in range(2):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            one_step(s)
            e1.record(stream)
            e1.synchronize()
            d_ms.append(e0.elapsed_time(e1))
            dk_ms.append(F.last_ksum()[0])
        barrier()
        dinfo = F.last_launch_info()
        dc = KERNEL_COUNTS.get(("coop", (dinfo["th"], dinfo["td"]), w.nbands), KERNEL_COUNTS.get(("coop", (dinfo["th"], dinfo["td"]))))
        dense = {"eval_mode": "coop", "steps": 2, "value": evals_per_step * 2 * world / (sum(d_ms) * 1e-3), "unit": UNIT,
                 "ms_per_step": sum(d_ms) / 2, "ksum_ms": sum(dk_ms) / 2}
        if dc:
            ach = evals_per_step * w.nbands * dc[0] / (dense["ksum_ms"] * 1e-3) / 1e12
            dense.update({"roofline_achieved": ach, "roofline_frac": ach / (PEAK_DFMA_PER_S / 1e12),
                          "fp64_inst_per_band_eval": dc[0], "counts_source": dc[2]})
        F.set_eval_mode(mode)

    # ---- e2e: host buffers through fe_scan_host (pinned), copies inside the timed region ----
    pin = lambda shape, dt: torch.empty(shape, dtype=dt).pin_memory().numpy()    # noqa: E731
    out = dict(omega=pin((nq_step, w.nh, w.nd), torch.float64), idx=pin((nq_step, w.nh), torch.int32),
               delta_star=pin((nq_step, w.nh), torch.float64), omega_star=pin((nq_step, w.nh), torch.float64))
    hq = [pin((nq_step, 2), torch.float64) for _ in range(2)]
    hh, hd = pin((w.nh,), torch.float64), pin((w.nd,), torch.float64)
    hh[:] = w.h
    hd[:] = w.delta
    e2e_steps = max(1, min(args.steps, 2))
    F.set_temperature(temps[0])
    hq[0][:] = q_of(0)
    if sp_mode:
        F.set_eval_mode(fe.EVAL_COOP_EO)       # e2e below is the fp64 host path; the SP numbers are the device-timed ones
    F.scan_host(hq[0], hh, hd, out=out, stream=stream)              # warm-up
    barrier()
    t0 = time.perf_counter()
    for s in range(e2e_steps):
        F.set_temperature(temps[s % len(temps)])
        hq[s % 2][:] = q_of(s)
        F.scan_host(hq[s % 2], hh, hd, out=out, stream=stream)      # synchronous: returns with results on the host
    torch.cuda.synchronize()
    te = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(te, op=dist.ReduceOp.MAX)
    e2e_value = evals_per_step * e2e_steps * world / float(te.item())
    h2d = 8 * (2 * nq_step + w.nh + 2 * w.nd)           # q, h, Delta^2 lists + Delta list for the argmin
    d2h = 8 * nq_step * w.nh * w.nd + nq_step * w.nh * (4 + 8 + 8)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (K1 k-sum) ----
    info = F.last_launch_info()
    info["block"] = 256
    if info["mode"] in (fe.EVAL_COOP, fe.EVAL_COOP_EO):
        info["block"] = next(c[4] for c in fe.coop_shapes() if (c[2], c[3]) == (info["th"], info["td"]))
    tile_key = (args.mode, (info["th"], info["td"]))
    counts = KERNEL_COUNTS.get(tile_key + (w.nbands,), KERNEL_COUNTS.get(tile_key, (None, None, None)))
    k_ms = sum(ksum_ms) / len(ksum_ms)
    dfma_rate, _ = fe.fp64_peak_probe()
    # Primary roofline = FP64-pipe lane-instructions/s: a DADD or DMUL occupies an FP64 lane for a cycle exactly like a
    # DFMA, and the kernel's pair update acc *= (A + B) has no fused form, so instructions (not flops, which count a
    # DFMA twice) measure how busy the bounding unit is; ncu sm__pipe_fp64_cycles_active agrees (profiles/README.md).
    roofline = {"bound": "alu", "kernel": f"k-sum kernel ({args.mode}, tile {info['th']}x{info['td']}, grid {info['grid']} x {info['block']})",
                "unit": "Tinst/s (FP64-pipe thread-instructions: DFMA, DADD, DMUL each count 1)",
                "peak": PEAK_DFMA_PER_S / 1e12,
                "peak_source": "nominal: 148 SM x 64 FP64 lanes x 1.965 GHz (DESIGN.md section 6); MEASURED_PEAKS.json has no fp64 entry",
                "peak_measured_dfma_probe": dfma_rate / 1e12, "avg_launch_ms": k_ms,
                "band_evals_per_launch": band_evals, "traffic": KERNEL_TRAFFIC.get((args.mode, w.nbands), KERNEL_TRAFFIC.get(args.mode)),
                "kernel_share_of_step": k_ms * len(ksum_ms) / total_ms}
    if sp_mode:
        counts = (None, None, None)
        roofline["note"] = ("single-precision builds (SURVEY 8f-2): FP32 / MUFU bound, see profiles/r1h_*; k_ms is the last k-sum launch "
                            "(verified_*: the fp64 pass on the candidate list); candidates verified per step: " + str(verified_n[-4:]))
    if counts[0]:
        achieved = band_evals * counts[0] / (k_ms * 1e-3) / 1e12
        tflops = band_evals * counts[1] / (k_ms * 1e-3) / 1e12
        roofline.update({"achieved": achieved, "frac": achieved / (PEAK_DFMA_PER_S / 1e12),
                         "fp64_inst_per_band_eval": counts[0], "flop_per_band_eval": counts[1], "counts_source": counts[2],
                         "frac_of_measured_dfma_peak": achieved / (dfma_rate / 1e12),
                         "achieved_tflops": tflops, "peak_tflops": PEAK_TFLOPS, "frac_tflops": tflops / PEAK_TFLOPS})
    else:
        roofline.update({"achieved": None, "frac": None})

    cpu = None
    if not args.no_cpu_baseline:
        v, dt, nd_used, cores, col = oracle_sample(w, temps[0], args.cpu_baseline_deltas)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": dt,
               "sample": (f"1 of {w.nq * w.nh} (q,h) columns of {w.name} (iq={col[0]}, ih={col[1]}) x {nd_used} of "
                          f"{w.nd} Delta, full {w.N}x{w.N} k-sum, T={temps[0]}")}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms_max / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "model": None, "N": w.N, "nq_per_step": nq_step, "nh": w.nh, "nd": w.nd,
                       "T_alternating": temps, "eval_mode": args.mode, "band_evals_per_step": evals_per_step * w.nbands,
                       "l2": "flushed between timed steps (256 MB memset); inputs are a few KB",
                       "parallelism": f"q-sharded x{world}, no collective on the data path"},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": e2e_steps, "api": "fe_scan_host (host buffers in/out, synchronous)"},
            "gpu_launches": launches, "wall_s_timed_region": t_wall, "clocks": clocks,
            "roofline": roofline, "dense_variant": dense, "cpu_baseline": cpu, "result_check": idx_check}
    del line["config"]["model"]
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
