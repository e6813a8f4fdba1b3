"""Multi-GPU: the path shards over (q, h) columns with NO data-path collective.

Every (q, h) column of Algorithm 1 is independent ("embarrassingly parallel ... for all combinations
of {q, k, Delta}"), so rank r of `world` evaluates the q-values q[r::world] with its own handle on its own GPU and
finds its own minima; the only communication is the final gather of the small per-column results
(idx, Delta*, Omega*), done with torch.distributed (NCCL on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

import numpy as np


def shard_indices(n: int, rank: int, world: int) -> np.ndarray:
    """Round-robin ownership: item i belongs to rank i % world (keeps neighbouring q on different GPUs)."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    return np.arange(rank, n, world, dtype=np.int64)


def shard_q(q, rank: int, world: int):
    q = np.ascontiguousarray(q, dtype=np.float64).reshape(-1, 2)
    idx = shard_indices(q.shape[0], rank, world)
    return idx, q[idx]


def gather_columns(local_idx, local_vals, nq: int, rank: int, world: int, group=None):
    """All-gather per-q results computed on each rank's shard back into q order.

    local_vals: dict name -> numpy array of shape (len(local_idx), nh).  Returns dict name -> (nq, nh) array.
    Uses torch.distributed.all_gather_object (tiny payloads: a few KB); no tensor collective on the data path."""
    import torch.distributed as dist
    if world == 1:
        return {k: np.asarray(v) for k, v in local_vals.items()}
    payload = (np.asarray(local_idx), {k: np.asarray(v) for k, v in local_vals.items()})
    got = [None] * world
    dist.all_gather_object(got, payload, group=group)
    out = {}
    for name, v in local_vals.items():
        v = np.asarray(v)
        full = np.empty((nq,) + v.shape[1:], dtype=v.dtype)
        for idx_r, vals_r in got:
            if len(idx_r):
                full[idx_r] = vals_r[name]
        out[name] = full
    return out


def scan_sharded(evaluate, q, h, delta, rank: int, world: int, group=None):
    """Run `evaluate(q_shard, h, delta) -> (idx, delta_star, omega_star)` (each (nq_local, nh)) on this rank's
    shard of q and gather the minima of all ranks in q order.  `evaluate` is FreeEnergy.scan_host-like."""
    q = np.ascontiguousarray(q, dtype=np.float64).reshape(-1, 2)
    idx, qs = shard_q(q, rank, world)
    nh = int(np.asarray(h).reshape(-1).shape[0])
    if len(idx):
        i, ds, os_ = evaluate(qs, h, delta)
    else:
        i = np.empty((0, nh), dtype=np.int32)
        ds = np.empty((0, nh))
        os_ = np.empty((0, nh))
    return gather_columns(idx, dict(idx=i, delta_star=ds, omega_star=os_), q.shape[0], rank, world, group)


def combine_argmin_q(local_idx, iq_local, id_local, val_local, rank: int, world: int, group=None):
    """Outer loop of Algorithm 1 (min over q) across ranks: every rank has run FreeEnergy.argmin_q on its own shard
    (iq_local indexes the shard); the per-h winners are gathered (3 small arrays per rank) and reduced on the host
    with the library's tie-break (lowest value, then lowest GLOBAL iq, then lowest Delta index).
    Returns (iq, id, value) arrays of length nh, identical on every rank."""
    import torch.distributed as dist
    local_idx = np.asarray(local_idx, dtype=np.int64)
    val = np.asarray(val_local, dtype=np.float64)
    if len(local_idx):
        giq = local_idx[np.asarray(iq_local, dtype=np.int64)]
        payload = (giq, np.asarray(id_local, dtype=np.int64), val)
    else:
        payload = None
    got = [payload]
    if world > 1:
        got = [None] * world
        dist.all_gather_object(got, payload, group=group)
    got = [g for g in got if g is not None]
    nh = got[0][2].shape[0]
    iq, idd, best = np.zeros(nh, np.int32), np.zeros(nh, np.int32), np.full(nh, np.inf)
    first = np.ones(nh, dtype=bool)
    for giq, gid, gval in got:
        for ih in range(nh):
            v = gval[ih]
            better = v < best[ih] or (v == best[ih] and (giq[ih], gid[ih]) < (iq[ih], idd[ih]))
            if (first[ih] and not np.isnan(v)) or better:
                if not np.isnan(v):
                    iq[ih], idd[ih], best[ih], first[ih] = giq[ih], gid[ih], v, False
    return iq, idd, best
