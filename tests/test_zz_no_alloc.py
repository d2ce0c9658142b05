"""avm_run_static — the whole-avalanche run for callers that cannot allocate device memory.

Why the entry point exists.  avm_run wants a `workspace` from its caller: device scratch for the persistent transport
kernel's run-control block (electron counters, ticket queue head, stop flags, tally accumulators) and for staging the
primaries.  A caller that is handed its input and output buffers by someone else and may not call the CUDA allocator
itself — a plug-in inside a host framework that owns all device memory, a service whose pool is frozen after start-up —
has nowhere to get that scratch from.  avm_run_static takes it from a fixed block compiled into libavm.so
(avm_run_static_bytes() = 36 KiB + 4 MiB per GPU, held until the process exits) and accepts runs of at most
AVM_RUN_STATIC_MAX_CAPACITY = 65536 electrons.

What is checked here, on a B200: two calls in a row through the new entry point, the second a different and smaller run
than the first (the block still holds the first call's counters, flags and staged primaries when the second starts, so a
missing reset would show), each compared electron by electron with the existing avm_run path on the same inputs, at the
tolerance the same-seed whole-run tests use (tests/test_gpu_parity.py: assert_run_same_seed, >= 99.9 % identical
histories, endpoints to 1e-9) — and the counts and tallies exactly, because both paths launch the same kernels.  Then the
size limit: a capacity beyond the maximum is refused with a message that names the limit, and nothing is written.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure in this add-on entry point
must not hide the parity tests of the main path.  It needs nothing from the other test files' state: it passes alone in a
fresh process and after the rest of the suite.
"""
import numpy as np
import pytest
import torch

from paper_2509_15377_b200.gen import configs, fields, primaries
from test_gpu_parity import assert_run_same_seed

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx(avm):
    return avm.ctx_create(0)


def _both_paths(avm, ctx, gg, fg, gas_table, prim, seed, capacity, **kw):
    """The same run through avm_run (caller's workspace) and through avm_run_static (NULL workspace); two fetched results."""
    L = gas_table.n_levels
    ref_bufs = avm.RunBuffers(ctx, capacity, prim.shape[0], L)
    _, n_ref = avm.run(ctx, gg, fg, prim, ref_bufs, seed=seed, **kw)
    ref = avm.fetch(ctx, ref_bufs, n_ref)
    st_bufs = avm.RunBuffers(ctx, capacity, prim.shape[0], L)
    st_bufs.workspace = None                      # the static path must not need it: the binding passes NULL / 0 anyway
    for t in (st_bufs.id, st_bufs.avalanche, st_bufs.status, st_bufs.n_steps, st_bufs.birth, st_bufs.end,
              st_bufs.per_avalanche, st_bufs.tallies_u64, st_bufs.tallies_f64):
        t.fill_(-7)                               # whatever comes back was written by this call
    _, n_st = avm.run_static(ctx, gg, fg, prim, st_bufs, seed=seed, **kw)
    return ref, avm.fetch(ctx, st_bufs, n_st)


def _assert_same_run(ref, got, n_levels):
    assert got.n == ref.n
    frac, n_common = assert_run_same_seed(ref, got, n_levels)          # >= 99.9 % identical histories, endpoints 1e-9
    assert n_common == ref.n
    assert np.all((got.status >= 1) & (got.status <= 7))               # every electron finished
    if frac == 1.0:
        assert np.array_equal(ref.tallies_u64, got.tallies_u64)
        assert np.array_equal(ref.per_avalanche, got.per_avalanche)
    assert np.allclose(ref.tallies_f64, got.tallies_f64, rtol=1e-9, atol=0.0)


def test_run_static_matches_avm_run_on_two_calls_in_a_row(avm, ctx, g0):
    assert avm.run_static_bytes() == 4096 + 1024 * 32 + avm.RUN_STATIC_MAX_CAPACITY * 64
    gg = avm.gas_create(ctx, g0)
    # call 1: BASELINE config 1 in full (1000 primaries from the host: the staging part of the block is used), ~1300 electrons
    w = configs.config1()
    assert w.capacity <= avm.RUN_STATIC_MAX_CAPACITY
    fg1 = avm.field_create(ctx, w.field)
    ref1, got1 = _both_paths(avm, ctx, gg, fg1, w.gas, w.primaries, w.seed, w.capacity)
    # call 2, straight after: another field (60 kV/cm, 100 um: a few hundred electrons per avalanche), another seed, fewer
    # primaries, primaries resident on the device, the widest capacity the entry point takes.  The block still holds call
    # 1's totals and stop flags at this point.
    fd2 = fields.uniform_gap((0.0, 0.0, -60000.0), 0.0, 100e-4)
    fg2 = avm.field_create(ctx, fd2)
    p2 = torch.from_numpy(primaries.isotropic_primaries(24, 5)).to(ctx.device)
    ref2, got2 = _both_paths(avm, ctx, gg, fg2, g0, p2, 5, avm.RUN_STATIC_MAX_CAPACITY)
    _assert_same_run(ref1, got1, g0.n_levels)
    _assert_same_run(ref2, got2, g0.n_levels)
    assert got1.n > 1000 and got2.n > 24 and got2.n != got1.n          # both multiplied; the runs really differ


def test_run_static_refuses_a_capacity_beyond_its_block(avm, ctx, g0):
    gg = avm.gas_create(ctx, g0)
    fg = avm.field_create(ctx, fields.uniform_gap((0.0, 0.0, -30000.0), 0.0, 50e-4))
    cap = avm.RUN_STATIC_MAX_CAPACITY + 1
    bufs = avm.RunBuffers(ctx, cap, 8, g0.n_levels)
    bufs.status.fill_(-7)
    with pytest.raises(avm.AvmError) as e:
        avm.run_static(ctx, gg, fg, primaries.isotropic_primaries(8, 1), bufs, seed=1)
    assert e.value.code == avm.ERR_INVALID_ARG
    assert "AVM_RUN_STATIC_MAX_CAPACITY" in str(e.value) and str(avm.RUN_STATIC_MAX_CAPACITY) in str(e.value)
    torch.cuda.synchronize()
    assert bool((bufs.status == -7).all())                             # refused before anything was queued
    # the same buffers are fine for the ordinary path, and the limit itself is accepted by the static one
    _, n = avm.run(ctx, gg, fg, primaries.isotropic_primaries(8, 1), bufs, seed=1)
    ok = avm.RunBuffers(ctx, avm.RUN_STATIC_MAX_CAPACITY, 8, g0.n_levels)
    _, n2 = avm.run_static(ctx, gg, fg, primaries.isotropic_primaries(8, 1), ok, seed=1)
    assert n2 == n >= 8
