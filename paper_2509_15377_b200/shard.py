"""Multi-GPU plumbing of the avalanche path: shard, run, merge.

Avalanches are independent and every random number is keyed by (electron id, collision index), so a job of Np
primaries partitions over ranks by primary range with NO data-path collective: rank r runs primaries [p0, p1) with
`id_offset = job_id_offset + p0` and gets bit-identical avalanches to the ones the single-rank job computes for those
primaries.  What is exchanged is the result only: one all-reduce of the tallies (<= (L + 5) u64 + 5 f64) and a gather of
the endpoint columns and per-avalanche counts.  Works with any torch.distributed backend ("nccl" with device tensors
on the GPU box, "gloo" with CPU tensors in the tests); nothing here touches the transport arithmetic.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional

import numpy as np
import torch


def shard_range(n_primaries: int, rank: int, world: int) -> tuple:
    """Contiguous, balanced primary range [p0, p1) of `rank` (sizes differ by at most one; empty when n < world)."""
    if not (0 <= rank < world):
        raise ValueError(f"rank {rank} outside world {world}")
    return (n_primaries * rank) // world, (n_primaries * (rank + 1)) // world


@dataclass
class MergedRun:
    """Whole-job result assembled from the shards (rank order = primary order)."""
    n: int
    id: np.ndarray
    avalanche: np.ndarray        # job-wide avalanche index = shard-local index + p0
    status: np.ndarray
    n_steps: np.ndarray
    birth: np.ndarray            # [5, n]
    end: np.ndarray              # [8, n]
    per_avalanche: np.ndarray    # [Np, 3]
    tallies_u64: np.ndarray
    tallies_f64: np.ndarray
    n_per_rank: list


def _dev(dist, device: Optional[torch.device]):
    if device is not None:
        return device
    return torch.device("cuda", torch.cuda.current_device()) if dist.get_backend() == "nccl" else torch.device("cpu")


def merge_tallies(tallies_u64: np.ndarray, tallies_f64: np.ndarray, dist, device=None) -> tuple:
    """Sum of the shards' tallies over all ranks (every rank gets the result).  u64 counts travel as int64."""
    dev = _dev(dist, device)
    tu = torch.from_numpy(np.ascontiguousarray(tallies_u64, dtype=np.uint64).view(np.int64).copy()).to(dev)
    tf = torch.from_numpy(np.ascontiguousarray(tallies_f64, dtype=np.float64).copy()).to(dev)
    dist.all_reduce(tu, op=dist.ReduceOp.SUM)
    dist.all_reduce(tf, op=dist.ReduceOp.SUM)
    return tu.cpu().numpy().view(np.uint64), tf.cpu().numpy()


def merge_signal(signal: np.ndarray, dist, device=None) -> np.ndarray:
    """Sum of the shards' induced-signal histograms (NEXT-4; the signal is a plain sum over electrons, so the whole job's
    histogram is the all-reduce of the shards' — same bins on every rank)."""
    dev = _dev(dist, device)
    t = torch.from_numpy(np.ascontiguousarray(signal, dtype=np.float64).copy()).to(dev)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return t.cpu().numpy()


def _gather_rows(local: np.ndarray, counts: list, dist, dev) -> np.ndarray:
    """all_gather of arrays whose LAST axis has a per-rank length (padded to the maximum, trimmed after)."""
    world, rank = dist.get_world_size(), dist.get_rank()
    m = max(max(counts), 1)
    kind = local.dtype
    as_i64 = kind in (np.uint64, np.uint32)
    send = np.zeros(local.shape[:-1] + (m,), dtype=np.int64 if as_i64 else kind)
    send[..., :counts[rank]] = local[..., :counts[rank]].astype(np.int64) if kind == np.uint32 else (
        local[..., :counts[rank]].view(np.int64) if kind == np.uint64 else local[..., :counts[rank]])
    t = torch.from_numpy(send).to(dev)
    out = [torch.empty_like(t) for _ in range(world)]
    dist.all_gather(out, t)
    parts = [o.cpu().numpy()[..., :counts[r]] for r, o in enumerate(out)]
    cat = np.concatenate(parts, axis=-1)
    if kind == np.uint64:
        return cat.view(np.uint64)
    return cat.astype(kind) if kind == np.uint32 else cat


def merge_run(local, p0: int, n_primaries_job: int, dist, device=None) -> MergedRun:
    """Assemble the whole-job result from this rank's shard result `local` (an avm.RunResult-like object holding the
    shard's n endpoints, per_avalanche [p1 - p0, 3] and tallies).  Every rank returns the same MergedRun."""
    dev = _dev(dist, device)
    world = dist.get_world_size()
    cnt = torch.tensor([int(local.n), int(local.per_avalanche.shape[0])], dtype=torch.int64, device=dev)
    allc = [torch.empty_like(cnt) for _ in range(world)]
    dist.all_gather(allc, cnt)
    n_end = [int(c[0]) for c in allc]
    n_av = [int(c[1]) for c in allc]
    if sum(n_av) != n_primaries_job:
        raise ValueError(f"shards cover {sum(n_av)} primaries, job has {n_primaries_job}")
    n = local.n
    aval = (np.asarray(local.avalanche[:n], dtype=np.uint32).astype(np.int64) + int(p0)).astype(np.uint32)
    ident = _gather_rows(np.ascontiguousarray(local.id[:n], dtype=np.uint64), n_end, dist, dev)
    avalanche = _gather_rows(aval, n_end, dist, dev)
    status = _gather_rows(np.ascontiguousarray(local.status[:n], dtype=np.int32), n_end, dist, dev)
    n_steps = _gather_rows(np.ascontiguousarray(local.n_steps[:n], dtype=np.uint32), n_end, dist, dev)
    birth = _gather_rows(np.ascontiguousarray(local.birth[:, :n], dtype=np.float64), n_end, dist, dev)
    end = _gather_rows(np.ascontiguousarray(local.end[:, :n], dtype=np.float64), n_end, dist, dev)
    pa = _gather_rows(np.ascontiguousarray(local.per_avalanche, dtype=np.uint64).T.copy(), n_av, dist, dev).T
    tu, tf = merge_tallies(local.tallies_u64, local.tallies_f64, dist, dev)
    return MergedRun(sum(n_end), ident, avalanche, status, n_steps, birth, end, np.ascontiguousarray(pa), tu, tf, n_end)
