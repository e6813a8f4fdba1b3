"""N > 1 path on CPU: world_size-2 gloo processes shard the q list, each evaluates its shard (here with the
oracle standing in for the per-rank GPU handle: tests may call the oracle), and the gathered minima equal the
single-process result.  No data-path collective exists; only the final tiny gather is exercised."""
import os
import socket
import sys

import numpy as np
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, ret):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from oracle import fe_oracle as O
    from paper_1412_8754_b200 import sharding, workloads as W
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    O.set_num_threads(2)
    w = W.interior_minimum(N=16, U=5.0, T=0.01, nq=5, nh=3, nd=24)     # 5 q over 2 ranks: ragged shards (3 + 2)

    def evaluate(qs, h, delta):
        om = O.omega_grid(w.params, w.N, w.T[0], qs, h, delta)
        return O.argmin(om, delta)

    out = sharding.scan_sharded(evaluate, w.q, w.h, w.delta, rank, world)
    # a rank with an empty shard must still take part (world > nq)
    out1 = sharding.scan_sharded(evaluate, w.q[:1], w.h, w.delta, rank, world)
    # outer loop of Algorithm 1 across ranks: per-rank argmin over its q shard, then the tiny host-side combine
    idx_q, qs = sharding.shard_q(w.q, rank, world)
    om = O.omega_grid(w.params, w.N, w.T[0], qs, w.h, w.delta)
    liq, lid, lval = O.argmin_q(om, ref_id=0)
    giq, gid, gval = sharding.combine_argmin_q(idx_q, liq, lid, lval, rank, world)
    if rank == 0:
        ret["gq"] = (giq, gid, gval)
        ret["idx"], ret["ds"], ret["os"] = out["idx"], out["delta_star"], out["omega_star"]
        ret["idx1"] = out1["idx"]
    dist.barrier()
    dist.destroy_process_group()


def test_world2_sharded_scan_equals_single_process():
    sys.path.insert(0, ROOT)
    from oracle import fe_oracle as O
    from paper_1412_8754_b200 import sharding, workloads as W
    assert list(sharding.shard_indices(5, 0, 2)) == [0, 2, 4] and list(sharding.shard_indices(5, 1, 2)) == [1, 3]
    assert sorted(np.concatenate([sharding.shard_indices(7, r, 3) for r in range(3)]).tolist()) == list(range(7))
    port = _free_port()
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(2, port, ret), nprocs=2, join=True)
    w = W.interior_minimum(N=16, U=5.0, T=0.01, nq=5, nh=3, nd=24)
    om = O.omega_grid(w.params, w.N, w.T[0], w.q, w.h, w.delta)
    idx, ds, os_ = O.argmin(om, w.delta)
    assert np.array_equal(ret["idx"], idx) and np.array_equal(ret["ds"], ds) and np.array_equal(ret["os"], os_)
    assert np.array_equal(ret["idx1"], idx[:1])
    rq, rd, rv = O.argmin_q(om, ref_id=0)
    assert np.array_equal(ret["gq"][0], rq) and np.array_equal(ret["gq"][1], rd) and np.array_equal(ret["gq"][2], rv)


def test_world1_is_identity():
    sys.path.insert(0, ROOT)
    from paper_1412_8754_b200 import sharding
    out = sharding.scan_sharded(lambda q, h, d: (np.zeros((len(q), 2), np.int32), np.ones((len(q), 2)), np.ones((len(q), 2))),
                                np.zeros((3, 2)), [0.0, 0.1], [0.0], 0, 1)
    assert out["idx"].shape == (3, 2)
