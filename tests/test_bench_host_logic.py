"""CPU tests of bench.py's host logic: (1) the N > 1 path -- the rank -> q mapping and the gather of the minima that
`bench.py --gpus N` runs, driven at world_size 2 over gloo with the oracle standing in for the per-rank GPU handle;
(2) the roofline counts are parsed from ncu CSVs and refused when the kernel-source hash beside them is stale."""
import os
import socket
import sys

import numpy as np
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, ret):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import bench
    from oracle import fe_oracle as O
    from paper_1412_8754_b200 import workloads as W
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    O.set_num_threads(2)
    w = W.interior_minimum(N=12, U=5.0, T=0.01, nq=5, nh=3, nd=16)
    calls = []

    def evaluate(qs, h, delta):                       # stands in for FreeEnergy.scan_host of this rank's GPU
        calls.append(len(qs))
        return O.argmin(O.omega_grid(w.params, w.N, w.T[0], qs, h, delta), delta)

    for scaling in ("strong", "weak"):
        idx, qs, ntot = bench.rank_q(w.q, rank, world, scaling)
        g = bench.sharded_scan(evaluate, w.q, w.h, w.delta, rank, world, scaling)
        ret[(scaling, rank)] = (idx.tolist(), qs.tolist(), ntot, g["idx"], g["delta_star"], g["omega_star"])
    # more ranks than q-values: the empty shard still takes part in the gather
    g1 = bench.sharded_scan(evaluate, w.q[:1], w.h, w.delta, rank, world, "strong")
    ret[("one", rank)] = g1["idx"]
    ret[("calls", rank)] = calls
    # the two reductions of bench.py's N > 1 path (units per step summed, times maximised), on CPU tensors over gloo
    ret[("reduce", rank)] = (bench.job_reduce(3.0 + rank, "sum", world, device="cpu"),
                             bench.job_reduce(10.0 * (rank + 1), "max", world, device="cpu"),
                             bench.job_reduce(5.0, "max", 1, device="cpu"))
    dist.barrier()
    dist.destroy_process_group()


def test_bench_rank_mapping_and_gather_world2():
    import bench
    from oracle import fe_oracle as O
    from paper_1412_8754_b200 import sharding, workloads as W
    w = W.interior_minimum(N=12, U=5.0, T=0.01, nq=5, nh=3, nd=16)
    # the mapping bench.py uses IS sharding.shard_q (strong) / the whole list per rank (weak)
    for r in range(2):
        idx, qs, ntot = bench.rank_q(w.q, r, 2, "strong")
        sidx, sq = sharding.shard_q(w.q, r, 2)
        assert np.array_equal(idx, sidx) and np.array_equal(qs, sq) and ntot == 5
        idx, qs, ntot = bench.rank_q(w.q, r, 2, "weak")
        assert idx.tolist() == list(range(5 * r, 5 * r + 5)) and np.array_equal(qs, w.q) and ntot == 10
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(2, _free_port(), ret), nprocs=2, join=True)
    ref = O.argmin(O.omega_grid(w.params, w.N, w.T[0], w.q, w.h, w.delta), w.delta)
    for r in range(2):
        _, _, ntot, gi, gd, go = ret[("strong", r)]          # every rank ends with the job's minima in q order
        assert ntot == 5 and np.array_equal(gi, ref[0]) and np.array_equal(gd, ref[1]) and np.array_equal(go, ref[2])
        _, _, ntot, gi, gd, go = ret[("weak", r)]            # weak: the job is `world` copies of the scan, equal work
        assert ntot == 10 and np.array_equal(gi, np.vstack([ref[0]] * 2)) and np.array_equal(go, np.vstack([ref[2]] * 2))
        assert np.array_equal(ret[("one", r)], ref[0][:1])
    assert ret[("calls", 0)] == [3, 5, 1] and ret[("calls", 1)] == [2, 5]     # rank 1's shard of a 1-q list is empty
    assert ret[("reduce", 0)] == (7.0, 20.0, 5.0) and ret[("reduce", 1)] == (7.0, 20.0, 5.0)


def _worker8(rank, world, port, ret):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import bench
    from paper_1412_8754_b200 import workloads as W
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = W.config(4)                                    # the headline q list: 32 q over 8 ranks = 4 q per rank

    def evaluate(qs, h, delta):                        # a stub with a recognisable answer per (q, h): no Omega needed here
        qs = np.asarray(qs).reshape(-1, 2)
        v = qs[:, :1] * 1000.0 + np.asarray(h)[None, :]
        return (v * 7).astype(np.int32), v + 0.5, -v

    g = bench.sharded_scan(evaluate, w.q, w.h, w.delta, rank, world, "strong")
    idx, qs, ntot = bench.rank_q(w.q, rank, world, "strong")
    few = bench.sharded_scan(evaluate, w.q[:3], w.h, w.delta, rank, world, "strong")      # more ranks than q-values
    ret[rank] = (idx.tolist(), ntot, g["idx"], g["delta_star"], g["omega_star"], few["omega_star"])
    dist.barrier()
    dist.destroy_process_group()


def test_bench_rank_mapping_and_gather_world8_config4():
    """bench.py --gpus 8 on the headline config, host side: 32 q round-robin over 8 ranks (4 each), every rank ends with
    all 32 x 64 minima in q order; and a 3-q list on 8 ranks (5 empty shards that still take part in the gather)."""
    from paper_1412_8754_b200 import workloads as W
    w = W.config(4)
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker8, args=(8, _free_port(), ret), nprocs=8, join=True)
    v = w.q[:, :1] * 1000.0 + w.h[None, :]
    owned = []
    for r in range(8):
        idx, ntot, gi, gd, go, few = ret[r]
        assert idx == list(range(r, 32, 8)) and ntot == 32
        assert gi.shape == (32, 64) and np.array_equal(gi, (v * 7).astype(np.int32))
        assert np.array_equal(gd, v + 0.5) and np.array_equal(go, -v)
        assert few.shape == (3, 64) and np.array_equal(few, -v[:3])
        owned += idx
    assert sorted(owned) == list(range(32))             # every q-value has exactly one owner


CSV_HEAD = '"ID","Process ID","Process Name","Host Name","Kernel Name","Context","Stream","Block Size","Grid Size","Device","CC","Section Name","Metric Name","Metric Unit","Metric Value"\n'


def _row(i, kern, metric, unit, val):
    return f'"{i}","1","python","h","{kern}","1","7","(128, 1, 1)","(10, 1, 1)","0","10.0","Command line profiler metrics","{metric}","{unit}","{val}"\n'


def test_roofline_counts_come_from_csv_and_go_stale(tmp_path, monkeypatch):
    import bench
    p = tmp_path / "cap.csv"
    text = "==PROF== Connected to process 1\n" + CSV_HEAD
    for i, (a, m, f) in enumerate(((100, 200, 50), (10, 20, 5))):
        for op, v in (("dadd", a), ("dmul", m), ("dfma", f)):
            text += _row(i, "void fe_ksum_coop_kernel<2>(P)", f"smsp__sass_thread_inst_executed_op_{op}_pred_on.sum", "inst", v)
        text += _row(i, "void fe_ksum_coop_kernel<2>(P)", "gpu__time_duration.sum", "ns", "2,000,000")
        text += _row(i, "void fe_ksum_coop_kernel<2>(P)", "dram__bytes_read.sum", "byte", 64)
        text += _row(i, "void fe_ksum_coop_kernel<2>(P)", "dram__bytes_write.sum", "byte", 36)
    text += _row(2, "void other_kernel()", "gpu__time_duration.sum", "ns", 5)
    p.write_text(text)
    (tmp_path / "COUNTS.md").write_text("| key | file | launches | source_hash |\n|---|---|---|---|\n"
                                        "| `omega/coop_eo/wl/q2` | `cap.csv` | T=0.01, T=0.001 | abcd |\n")
    monkeypatch.setattr(bench, "PROFILES", str(tmp_path))
    monkeypatch.setattr(bench, "load_counts_index", lambda path=None, _f=bench.load_counts_index: _f(str(tmp_path / "COUNTS.md")))
    launches = bench.parse_ncu_metrics_csv(str(p))
    assert len(launches) == 3 and launches[0]["metrics"]["gpu__time_duration.sum"] == 2e6
    counts, status = bench.kernel_counts("omega/coop_eo/wl/q2", "fe_ksum", ("abcd", "abcd"))
    assert status is None and counts["T=0.01"]["inst"] == 350 and counts["T=0.001"]["flop"] == 40 and counts["T=0.01"]["dram_bytes"] == 100
    roof = bench.roofline_base("k", 1.8e13)
    bench.apply_counts(roof, counts, status, ["T=0.01", "T=0.001", "T=0.01"], [1.0, 1.0, 2.0], 10.0, "band_eval")
    assert abs(roof["achieved"] - (350 + 35 + 350) / 4e-3 / 1e12) < 1e-18 and roof["frac"] == roof["achieved"] / roof["peak"]
    assert roof["traffic"] == 100 and roof["counts"]["per_launch"]["T=0.001"]["fp64_inst_per_band_eval"] == 3.5
    # a kernel edit without re-profiling: the tree hash differs from the recorded one -> no fraction is claimed
    counts, status = bench.kernel_counts("omega/coop_eo/wl/q2", "fe_ksum", ("ffff", "ffff"))
    roof = bench.roofline_base("k", 1.8e13)
    bench.apply_counts(roof, counts, status, ["T=0.01"], [1.0], 10.0, "band_eval")
    assert roof["frac"] is None and roof["achieved"] is None and "stale" in roof["stale_counts"]
    # a library built from other sources than the tree's is refused as well; an unknown key says so
    assert "stale" in bench.kernel_counts("omega/coop_eo/wl/q2", "fe_ksum", ("abcd", "eeee"))[1]
    assert bench.kernel_counts("omega/coop/wl/q2", "fe_ksum", ("abcd", "abcd"))[0] is None


def test_committed_counts_index_is_consistent():
    """Every capture profiles/COUNTS.md names exists, parses, and has as many matching launches as labels."""
    import bench
    idx = bench.load_counts_index()
    for key, row in idx.items():
        path = os.path.join(bench.PROFILES, row["file"])
        assert os.path.exists(path), (key, path)
        regex = "fe_chi_kernel" if key.startswith("chi/") else "fe_ksum"
        import re
        n = sum(1 for l in bench.parse_ncu_metrics_csv(path) if re.search(regex, l["kernel"]))
        assert n == len(row["labels"]), (key, n, row["labels"])
        assert len(row["source_hash"]) == 16
