"""The N > 1 path on CPU: world_size-2 `gloo` job over disjoint primary ranges.

The host-side plumbing (paper_2509_15377_b200.shard: partition, id offsets, tally all-reduce, endpoint gather) is what
runs here; each rank's shard is computed by the oracle standing in for the GPU (tests may call oracle/), so the merged
result must be IDENTICAL to the whole job computed in one piece — the property the multi-GPU design rests on
(draws keyed by electron id, no data-path collective).  The shards run with banded rates and an induced signal: the
banded streams are keyed by electron id as well, and the job's histogram is the all-reduce of the shards'.
"""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2509_15377_b200 import shard  # noqa: E402


def test_shard_range_partitions_exactly():
    for n in (0, 1, 2, 7, 100, 1001):
        for world in (1, 2, 3, 8):
            r = [shard.shard_range(n, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.shard_range(10, 2, 2)


def _free_port() -> int:
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank: int, world: int, port: int, n_prim: int, out_dir: str):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import avmo
        from paper_2509_15377_b200.gen import fields, gas, primaries
        g0 = gas.gas_g0()
        fd = fields.uniform_gap((0.0, 0.0, -45000.0), 0.0, 60e-4)
        prim = primaries.isotropic_primaries(n_prim, 3)
        p0, p1 = shard.shard_range(n_prim, rank, world)
        wf = fields.uniform_gap((0.0, 0.0, 1.0 / 60e-4), 0.0, 60e-4)
        local = avmo.run(g0, fd, prim[p0:p1], seed=3, id_offset=p0, capacity=1 << 16, flags=avmo.BANDED, signal=(wf, 0.0, 0.01, 40))
        merged = shard.merge_run(local, p0, n_prim, dist)
        signal = shard.merge_signal(local.signal, dist)
        np.savez(os.path.join(out_dir, f"merged_{rank}.npz"), n=merged.n, id=merged.id, avalanche=merged.avalanche,
                 status=merged.status, n_steps=merged.n_steps, birth=merged.birth, end=merged.end,
                 per_avalanche=merged.per_avalanche, tallies_u64=merged.tallies_u64, tallies_f64=merged.tallies_f64,
                 n_per_rank=np.array(merged.n_per_rank), signal=signal)
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_rank_gloo_job_equals_single_rank_job(tmp_path):
    from oracle import avmo
    from paper_2509_15377_b200.gen import fields, gas, primaries
    n_prim, world = 48, 2
    avmo.build()
    mp.spawn(_worker, args=(world, _free_port(), n_prim, str(tmp_path)), nprocs=world, join=True)
    g0 = gas.gas_g0()
    fd = fields.uniform_gap((0.0, 0.0, -45000.0), 0.0, 60e-4)
    wf = fields.uniform_gap((0.0, 0.0, 1.0 / 60e-4), 0.0, 60e-4)
    whole = avmo.run(g0, fd, primaries.isotropic_primaries(n_prim, 3), seed=3, capacity=1 << 16, flags=avmo.BANDED, signal=(wf, 0.0, 0.01, 40))
    assert whole.n > 2 * n_prim                      # the avalanches multiply: secondaries cross the gather too
    m = [np.load(os.path.join(tmp_path, f"merged_{r}.npz")) for r in range(world)]
    for key in m[0].files:                           # every rank assembled the same job result
        assert np.array_equal(m[0][key], m[1][key]), key
    r = m[0]
    assert int(r["n"]) == whole.n and int(r["n_per_rank"].sum()) == whole.n and np.all(r["n_per_rank"] > 0)
    oc, om = np.argsort(whole.id, kind="stable"), np.argsort(r["id"], kind="stable")
    assert np.array_equal(whole.id[oc], r["id"][om])
    for key, ref in (("avalanche", whole.avalanche), ("status", whole.status), ("n_steps", whole.n_steps)):
        assert np.array_equal(ref[oc], r[key][om]), key
    assert np.array_equal(whole.birth[:, oc], r["birth"][:, om])     # bit-identical: same code, same streams
    assert np.array_equal(whole.end[:, oc], r["end"][:, om])
    assert np.array_equal(whole.per_avalanche, r["per_avalanche"])
    assert np.array_equal(whole.tallies_u64, r["tallies_u64"])
    assert np.allclose(whole.tallies_f64, r["tallies_f64"], rtol=1e-12, atol=1e-14)   # sums in a different order (dx, dy cancel to ~1e-5)
    assert np.abs(whole.signal).max() > 1.0 and np.allclose(whole.signal, r["signal"], rtol=1e-12, atol=1e-13)   # NEXT-4 histogram
