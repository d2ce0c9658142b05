"""NEXT-4 on the device (DESIGN.md §3.7 readings W1-W4): the induced signal accumulated inside the
persistent kernel (every step form: time-parallel batches, serial batches, full warps; banded too) and the ion-drift kernel,
against the oracle on the same seeded runs — histograms bin by bin, ion endpoints ion by ion (matched through the electron
ids: slot order differs) — and against the Ramo identity on the device's own endpoints."""
import os

import numpy as np
import pytest
import torch

from paper_2509_15377_b200.gen import configs, fields, gas, primaries

pytestmark = pytest.mark.gpu
CORES = os.cpu_count() or 1
B30 = (0.0, 0.5, 0.8660254037844387)


@pytest.fixture(scope="module")
def ctx(avm):
    return avm.ctx_create(0)


def _plate(z_lo, z_hi):
    return fields.uniform_gap((0.0, 0.0, 1.0 / (z_hi - z_lo)), z_lo, z_hi)


def gpu_run_signal(avm, ctx, g, fd, wf, prim, seed, t0, dtb, nb, flags=0, t_max=float("inf"), capacity=1 << 18):
    gg, fg, wg = avm.gas_create(ctx, g), avm.field_create(ctx, fd), avm.field_create(ctx, wf)
    bufs = avm.RunBuffers(ctx, capacity, prim.shape[0], g.n_levels)
    sig = torch.zeros(nb, dtype=torch.float64, device=ctx.device)
    _, n = avm.run(ctx, gg, fg, prim, bufs, seed=seed, t_max=t_max, flags=flags, signal=(wg, t0, dtb, sig))
    return avm.fetch(ctx, bufs, n), sig.cpu().numpy(), (gg, fg, wg, bufs, n)


def assert_signal(cpu_sig, gpu_sig, what):
    scale = np.abs(cpu_sig).max()
    assert scale > 0
    assert np.all(np.abs(cpu_sig - gpu_sig) <= 1e-9 * scale + 1e-9 * np.abs(cpu_sig)), (what, np.abs(cpu_sig - gpu_sig).max() / scale)


@pytest.mark.parametrize("flags", [0, 4, 16], ids=["time-parallel", "serial", "banded"])
def test_signal_config1_all_forms(avm, ctx, oracle, g0, flags):
    """Config 1 (one electron per warp: batches) with a uniform weighting field over the gap: the device histogram equals
    the oracle's bin by bin and obeys the Ramo identity on the device's own endpoints."""
    w = configs.config1()
    d = 50e-4
    wf = _plate(0.0, d)
    cpu = oracle.run(w.gas, w.field, w.primaries, seed=0, n_threads=CORES, flags=1 if flags & 16 else 0, signal=(wf, 0.0, 0.008, 400))
    gpu, sig, _ = gpu_run_signal(avm, ctx, w.gas, w.field, wf, w.primaries, 0, 0.0, 0.008, 400, flags=flags)
    assert gpu.end[3].max() < 3.2
    assert gpu.n == cpu.n and (np.abs(cpu.signal) > 0).sum() > 30
    assert_signal(cpu.signal, sig, f"config1 flags {flags}")
    exact = -((gpu.end[2] - gpu.birth[2]) / d).sum()
    assert abs(sig.sum() - exact) < 1e-9 * abs(exact)


def test_signal_full_warps_with_b_and_grid_weighting(avm, ctx, oracle, g0):
    """Throughput regime (full-warp iterations) with B, and a NON-uniform weighting field from a grid map."""
    w = configs.config3(n_primaries=40000, t_max=1.0)
    h = 0.05
    z = np.arange(24) * h
    nodes = np.zeros((24, 6, 6, 4), dtype=np.float32)
    nodes[..., 2] = (1.0 + 0.5 * np.sin(8.0 * z))[:, None, None]
    nodes[..., 0] = 0.2; nodes[..., 3] = 1.0
    wf = fields.FieldDesc([fields.grid_slab(nodes, (-0.15, -0.15, -0.05), (h, h, h), -0.05, 1.1, fields.BC_PERIODIC, fields.BC_PERIODIC, 0.25, 0.25)])
    m = 4000
    cpu = oracle.run(w.gas, w.field, w.primaries[:m], seed=0, t_max=1.0, n_threads=CORES, signal=(wf, 0.0, 0.05, 24))
    gpu, sig, _ = gpu_run_signal(avm, ctx, w.gas, w.field, wf, w.primaries[:m], 0, 0.0, 0.05, 24, t_max=1.0, flags=avm.RUN_SHAPE_WIDE)
    assert_signal(cpu.signal, sig, "config3 first 4000, wide")
    # all 40000 at once: full warps
    cpu2 = oracle.run(w.gas, w.field, w.primaries, seed=0, t_max=1.0, n_threads=CORES, signal=(wf, 0.0, 0.05, 24))
    gpu2, sig2, _ = gpu_run_signal(avm, ctx, w.gas, w.field, wf, w.primaries, 0, 0.0, 0.05, 24, t_max=1.0)
    assert_signal(cpu2.signal, sig2, "config3 40000, full warps")
    # banded
    cb = oracle.run(w.gas, w.field, w.primaries[:m], seed=0, t_max=1.0, n_threads=CORES, flags=1, signal=(wf, 0.0, 0.05, 24))
    gb, sb, _ = gpu_run_signal(avm, ctx, w.gas, w.field, wf, w.primaries[:m], 0, 0.0, 0.05, 24, t_max=1.0, flags=avm.RUN_BANDED)
    assert_signal(cb.signal, sb, "config3 banded")


def test_signal_on_a_grid_map_run(avm, ctx, oracle, g0):
    """Serial batches on a map (drift field AND weighting field from grids), electrons leaving and hitting material."""
    rng = np.random.default_rng(3)
    nodes = (rng.normal(size=(40, 14, 12, 4)) * 8e3).astype(np.float32)
    nodes[..., 2] -= 3e4
    nodes[..., 3] = (rng.uniform(size=(40, 14, 12)) > 0.03).astype(np.float32)
    hh = (1e-4, 1e-4, 1e-4)
    fd = fields.FieldDesc([fields.grid_slab(nodes, (0, 0, 0), hh, 0.0, 39e-4, fields.BC_MIRROR, fields.BC_MIRROR, 10e-4, 12e-4)])
    wn = (rng.normal(size=(40, 14, 12, 4)) * 50.0).astype(np.float32); wn[..., 2] += 250.0
    wf = fields.FieldDesc([fields.grid_slab(wn, (0, 0, 0), hh, 0.0, 39e-4, fields.BC_MIRROR, fields.BC_MIRROR, 10e-4, 12e-4)])
    p = primaries.isotropic_primaries(300, 9, pos=(0, 0, 2e-4), xy_box=((0, 10e-4), (0, 12e-4)))
    cpu = oracle.run(g0, fd, p, seed=9, n_threads=CORES, signal=(wf, 0.0, 0.01, 40))
    gpu, sig, _ = gpu_run_signal(avm, ctx, g0, fd, wf, p, 9, 0.0, 0.01, 40)
    assert cpu.n == gpu.n and cpu.n > 320
    scale = np.abs(cpu.signal).max()
    assert np.all(np.abs(cpu.signal - sig) <= 1e-7 * scale), np.abs(cpu.signal - sig).max() / scale     # ~1e3-step histories through random gradients


def _match(cpu, gpu):
    oc, og = np.argsort(cpu.id, kind="stable"), np.argsort(gpu.id, kind="stable")
    assert np.array_equal(cpu.id[oc], gpu.id[og])
    return oc, og


def test_ion_drift_against_the_oracle(avm, ctx, oracle):
    """Ions of a multiplying AND attaching run in a uniform field and through a map: which ions exist, endpoints, times,
    statuses and step counts ion by ion; the ion signal bin by bin; one elementary charge per collected pair."""
    d = 50e-4
    g = gas.multi_level_constant([2000.0, 8.0, 4.0], [gas.ELASTIC, gas.IONISATION, gas.ATTACHMENT], recoil=[0.02, 0, 0], w=[0, 10.0, 0], n_bins=32, e_max=100.0)
    fd = fields.uniform_gap((0.0, 0.0, -30000.0), 0.0, d)
    wf = _plate(-1e-4, d + 1e-4)
    p = primaries.isotropic_primaries(500, 11)
    cpu = oracle.run(g, fd, p, seed=11, n_threads=CORES)
    gpu, _, (gg, fg, wg, bufs, n) = gpu_run_signal(avm, ctx, g, fd, wf, p, 11, 0.0, 1.0, 4)
    oc, og = _match(cpu, gpu)
    sig_def = (wf, 0.0, 5.0, 40)
    ic = oracle.ion_drift(fd, cpu, 500, 1.5e-9, 2.0e-9, 0.25e-4, signal=sig_def)
    sdev = torch.zeros(40, dtype=torch.float64, device=ctx.device)
    ig = avm.ion_drift(ctx, fg, bufs, n, 1.5e-9, 2.0e-9, 0.25e-4, signal=(wg, 0.0, 5.0, sdev))
    nn = cpu.n
    for off in (0, nn):
        assert np.array_equal(ic.status[off:off + nn][oc], ig.status[off:off + nn][og])
        assert np.array_equal(ic.n_steps[off:off + nn][oc], ig.n_steps[off:off + nn][og])
        assert np.allclose(ic.end[:, off:off + nn][:, oc], ig.end[:, off:off + nn][:, og], rtol=1e-10, atol=1e-14)
    assert (ig.status[:nn] == 1).sum() == nn - 500 and (ig.status[nn:] == 2).sum() == (gpu.status == 5).sum() > 10
    assert_signal(ic.signal, sdev.cpu().numpy(), "ion signal, uniform field")
    # electrons + ions: sum q (z_end - z_start) / d' on the device's own arrays
    dd = d + 2e-4
    have_p, have_n = ig.status[:nn] >= 0, ig.status[nn:] >= 0
    q_i = ((ig.end[2, :nn] - gpu.birth[2])[have_p] / dd).sum() - ((ig.end[2, nn:] - gpu.end[2])[have_n] / dd).sum()
    assert abs(sdev.cpu().numpy().sum() - q_i) < 1e-9 * abs(q_i)
    # through a map: curved paths, material, time limit
    rng = np.random.default_rng(4)
    nodes = (rng.normal(size=(40, 14, 12, 4)) * 6e3).astype(np.float32)
    nodes[..., 2] -= 3e4
    nodes[..., 3] = (rng.uniform(size=(40, 14, 12)) > 0.02).astype(np.float32)
    hh = (1e-4, 1e-4, 1e-4)
    fm = fields.FieldDesc([fields.grid_slab(nodes, (0, 0, 0), hh, 0.0, 39e-4, fields.BC_MIRROR, fields.BC_MIRROR, 10e-4, 12e-4)])
    p = primaries.isotropic_primaries(300, 12, pos=(0, 0, 2e-4), xy_box=((0, 10e-4), (0, 12e-4)))
    cpu = oracle.run(g, fm, p, seed=12, n_threads=CORES)
    gpu, _, (gg, fg, wg, bufs, n) = gpu_run_signal(avm, ctx, g, fm, wf, p, 12, 0.0, 1.0, 4)
    oc, og = _match(cpu, gpu)
    same = (cpu.n_steps[oc] == gpu.n_steps[og]) & (cpu.status[oc] == gpu.status[og])
    assert same.mean() > 0.99
    ic = oracle.ion_drift(fm, cpu, 300, 1.5e-9, 2.0e-9, 0.2e-4, t_max=60.0)
    ig = avm.ion_drift(ctx, fg, bufs, n, 1.5e-9, 2.0e-9, 0.2e-4, t_max=60.0)
    nn = cpu.n
    for off in (0, nn):
        sc, sg = ic.status[off:off + nn][oc][same], ig.status[off:off + nn][og][same]
        assert (sc == sg).mean() > 0.995                              # a rounding difference can move one step across a mask edge
        ok = sc == sg
        assert np.allclose(ic.end[:, off:off + nn][:, oc][:, same][:, ok], ig.end[:, off:off + nn][:, og][:, same][:, ok], rtol=1e-7, atol=1e-10)
    assert set(np.unique(ig.status)) >= {-1, 1, 4, 6}


def test_signal_and_ions_invalid_arguments(avm, ctx, g0):
    fd = fields.uniform_gap((0.0, 0.0, -30000.0), 0.0, 50e-4)
    gg, fg = avm.gas_create(ctx, g0), avm.field_create(ctx, fd)
    bufs = avm.RunBuffers(ctx, 1 << 12, 10, g0.n_levels)
    p = primaries.isotropic_primaries(10, 1)
    sig = torch.zeros(8, dtype=torch.float64, device=ctx.device)
    with pytest.raises(avm.AvmError):
        avm.run(ctx, gg, fg, p, bufs, signal=(fg, 0.0, 0.0, sig))           # dt_bin = 0
    _, n = avm.run(ctx, gg, fg, p, bufs)
    with pytest.raises(avm.AvmError):
        avm.ion_drift(ctx, fg, bufs, n, 1e-9, 1e-9, 0.0)                  # step = 0


def test_ion_drift_ignores_slots_that_hold_no_electron(avm, ctx, g0):
    """avm_ion_drift with n beyond the run's endpoint count (slots of status -1 with stale birth values) produces no ions
    there; n_primaries > n is refused."""
    from paper_2509_15377_b200.gen import tetmesh
    fd = fields.uniform_gap((0.0, 0.0, -30000.0), 0.0, 50e-4)
    gg, fg = avm.gas_create(ctx, g0), avm.field_create(ctx, fd)
    bufs = avm.RunBuffers(ctx, 1 << 12, 200, g0.n_levels)
    bufs.birth.fill_(10e-4)                                                  # stale slots would look like ions born mid-gap
    bufs.end.fill_(10e-4)
    p = primaries.isotropic_primaries(200, 2)
    _, n = avm.run(ctx, gg, fg, p, bufs, seed=2)
    assert 200 < n < (1 << 12) - 64
    a = avm.ion_drift(ctx, fg, bufs, n, 1.5e-9, 2.0e-9, 0.25e-4)
    b = avm.ion_drift(ctx, fg, bufs, n + 64, 1.5e-9, 2.0e-9, 0.25e-4)
    m = n + 64
    assert np.all(b.status[n:m] == -1) and np.all(b.status[m + n:] == -1) and np.all(b.n_steps[n:m] == 0)
    assert np.array_equal(a.status[:n], b.status[:n]) and np.array_equal(a.status[n:], b.status[m:m + n])
    assert np.array_equal(a.end[:, :n], b.end[:, :n]) and (a.status[:n] >= 1).sum() == n - 200
    with pytest.raises(avm.AvmError) as e:
        avm.ion_drift(ctx, fg, avm.RunBuffers(ctx, 1 << 12, n + 1, g0.n_levels), n, 1.5e-9, 2.0e-9, 0.25e-4)   # n_primaries = n + 1
    assert "n_primaries" in str(e.value)
    # a tetrahedral weighting field is refused (uniform slabs and grid maps only), for runs and for ion drift alike
    mesh = tetmesh.kuhn_mesh(4, 4, 4, (20e-4, 20e-4, 20e-4), lambda x, y, z: z, seed=1)
    wt = avm.field_create(ctx, fields.FieldDesc([fields.tet_slab(mesh, (0, 0, 0), 0.0, 60e-4)]))
    sig = torch.zeros(8, dtype=torch.float64, device=ctx.device)
    for call in (lambda: avm.run(ctx, gg, fg, p, bufs, seed=2, signal=(wt, 0.0, 1.0, sig)),
                 lambda: avm.ion_drift(ctx, fg, bufs, n, 1.5e-9, 2.0e-9, 0.25e-4, signal=(wt, 0.0, 1.0, sig))):
        with pytest.raises(avm.AvmError) as e:
            call()
        assert "weighting" in str(e.value)


def test_extras_on_a_table_too_large_for_shared_memory_are_refused_before_any_work(avm, ctx):
    """A signal (or a NEXT-3 gas) needs the kernel variant with the threshold table in shared memory (at most ~24000
    energy bins).  Beyond that avm_run refuses BEFORE it queues anything: the output arrays are untouched.  The same gas without
    a signal runs (the table is then read through L1)."""
    g = gas.gas_g0(n_bins=30000)
    fd = fields.uniform_gap((0.0, 0.0, -30000.0), 0.0, 50e-4)
    gg, fg = avm.gas_create(ctx, g), avm.field_create(ctx, fd)
    bufs = avm.RunBuffers(ctx, 1 << 12, 50, g.n_levels)
    bufs.status.fill_(-7)
    p = primaries.isotropic_primaries(50, 3)
    sig = torch.zeros(8, dtype=torch.float64, device=ctx.device)
    with pytest.raises(avm.AvmError) as e:
        avm.run(ctx, gg, fg, p, bufs, seed=3, signal=(fg, 0.0, 1.0, sig))
    assert "shared memory" in str(e.value)
    torch.cuda.synchronize()
    assert bool((bufs.status == -7).all()) and float(sig.abs().sum()) == 0.0
    _, n = avm.run(ctx, gg, fg, p, bufs, seed=3)
    assert n >= 50 and bool((bufs.status[:n] >= 1).all())
