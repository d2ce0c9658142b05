"""NEXT-3 on the device (DESIGN.md §3.6 readings X1-X3): table-driven anisotropic scattering, Penning
transfer and gas thermal motion in the CUDA path against the oracle — per-step tolerance T (1e-12) through every step form
(general, full-warp, time-parallel batch, serial batch; banded too), then same-seed whole runs with identical avalanches
and tallies (the Penning count included).  PAPER.md:121: Penning transfer is the feature the paper had to switch off."""
import copy
import os

import numpy as np
import pytest

from paper_2509_15377_b200.gen import configs, fields, gas, primaries
from test_gpu_parity import assert_step_parity, assert_run_same_seed, _states, _random_map
from test_gpu_step_forms import assert_form2_parity, oracle_sequence
from test_gpu_banded import oracle_sequence_banded

pytestmark = pytest.mark.gpu
B30 = (0.0, 0.5, 0.8660254037844387)
CORES = os.cpu_count() or 1


@pytest.fixture(scope="module")
def ctx(avm):
    return avm.ctx_create(0)


def extended_g0(g0, aniso=True, penning=True, thermal=True, seed=5):
    """Gas G0 with a smooth forward-scattering table (xi rising with energy, different per level, backward for one),
    Penning transfer on the three highest excitation levels and the gas at 293.15 K."""
    g = copy.copy(g0)
    rng = np.random.default_rng(seed)
    if aniso:
        e = (np.arange(g0.n_bins) + 0.5) * g0.e_max / g0.n_bins
        amp = rng.uniform(0.2, 0.95, g0.n_levels); amp[3] = -0.6
        g.scat_xi = amp[None, :] * (e[:, None] / (e[:, None] + rng.uniform(1.0, 10.0, g0.n_levels)[None, :]))
    if penning:
        pp = np.zeros(g0.n_levels); pe = np.zeros(g0.n_levels)
        exc = np.flatnonzero(g0.level_type == gas.EXCITATION)
        pp[exc[-3:]] = (0.4, 0.7, 1.0)
        pe[exc[-3:]] = np.maximum(g0.level_loss[exc[-3:]] - 13.8, 0.05)
        pp[exc[0]] = 0.2; pe[exc[0]] = 0.0                                   # zero available energy: the child sits at the floor
        g.level_penning_prob, g.level_penning_eV = pp, pe
    if thermal:
        g.kT_eV = 0.02526
    return g


CASES = [dict(aniso=True, penning=False, thermal=False), dict(aniso=False, penning=True, thermal=False),
         dict(aniso=False, penning=False, thermal=True), dict(aniso=True, penning=True, thermal=True)]


@pytest.mark.parametrize("case", CASES, ids=["aniso", "penning", "thermal", "all"])
@pytest.mark.parametrize("B", [(0.0, 0.0, 0.0), B30])
def test_next3_steps_forms_0_and_1(avm, ctx, oracle, g0, case, B):
    g = extended_g0(g0, **case)
    rng = np.random.default_rng(231)
    n = 1 << 16
    st = _states(n, rng, box=30e-4, center=(0, 0, 30e-4))
    st[4, : n // 4] = np.exp(rng.uniform(np.log(1e-3), np.log(0.2), n // 4))        # thermal energies too
    fd = fields.uniform_gap((0.0, 0.0, -60000.0), 0.0, 60e-4, B)
    ids = rng.integers(0, 2 ** 64, n, dtype=np.uint64)
    nidx = rng.integers(0, 2 ** 32 - 64, n, dtype=np.uint64).astype(np.uint32)
    gg, fg = avm.gas_create(ctx, g), avm.field_create(ctx, fd)
    cpu = oracle.step_batch(g, fd, 3, st, ids, nidx, t_max=4.9)
    for form in (0, 1):
        gpu = avm.step_batch_form(ctx, gg, fg, 3, st, ids, nidx, form=form, t_max=4.9)
        assert_step_parity(cpu, gpu, st, f"NEXT-3 {case} form {form} B={B}")
    assert all((cpu.event == l).sum() > 0 for l in range(0, 16))
    if case["penning"]:
        exc = cpu.event >= 0
        exc &= g.level_type[np.maximum(cpu.event, 0)] == gas.EXCITATION
        assert ((cpu.child_id != 0) & exc).sum() > 100 and ((cpu.child_id == 0) & exc).sum() > 100
    # banded rates with the extensions
    cb = oracle.step_batch(g, fd, 3, st, ids, nidx, t_max=4.9, flags=1)
    gb = avm.step_batch_form(ctx, gg, fg, 3, st, ids, nidx, form=1, t_max=4.9, flags=avm.RUN_BANDED)
    assert_step_parity(cb, gb, st, f"NEXT-3 {case} banded form 1 B={B}")


@pytest.mark.parametrize("form", [2, 3])
@pytest.mark.parametrize("k", [1, 4, 8])
def test_next3_batches(avm, ctx, oracle, g0, form, k):
    """Time-parallel batches (the speculative elastic collision is off: every real collision takes the general path) and
    serial batches with all three extensions."""
    g = extended_g0(g0)
    rng = np.random.default_rng(240 + k)
    gl = avm.step_form_lanes(k)
    n = k * 1200
    st = _states(n, rng, box=30e-4, center=(0, 0, 30e-4))
    fd = fields.uniform_gap((0.0, 0.0, -60000.0), 0.0, 60e-4, B30 if k == 4 else (0, 0, 0))
    ids = rng.integers(0, 2 ** 64, n, dtype=np.uint64)
    n0 = rng.integers(0, 2 ** 32 - 64, n, dtype=np.uint64).astype(np.uint32)
    cpu, st_in = oracle_sequence(oracle, g, fd, 3, st, ids, n0, gl, 5.0)
    gpu = avm.step_batch_form(ctx, avm.gas_create(ctx, g), avm.field_create(ctx, fd), 3, st, ids, n0, form=form, k=k, t_max=5.0)
    total = assert_form2_parity(avm, cpu, st_in, gpu, gl, f"NEXT-3 form {form} k={k}", composed=form == 2)
    assert total > n * min(gl, 3) * 0.5
    if form == 3:
        cb, sb = oracle_sequence_banded(oracle, g, fd, 3, st, ids, n0, gl, 5.0)
        gb = avm.step_batch_form(ctx, avm.gas_create(ctx, g), avm.field_create(ctx, fd), 3, st, ids, n0, form=3, k=k, t_max=5.0, flags=avm.RUN_BANDED)
        assert_form2_parity(avm, cb, sb, gb, gl, f"NEXT-3 banded form 3 k={k}")


def test_next3_steps_on_a_grid_map(avm, ctx, oracle, g0):
    g = extended_g0(g0)
    rng = np.random.default_rng(250)
    nodes = _random_map(rng, 12, 14, 20, e_scale=5e4)
    fd = fields.FieldDesc([fields.grid_slab(nodes, (0, 0, 0), (1e-4, 1e-4, 1e-4), 0.0, 19e-4, fields.BC_MIRROR, fields.BC_MIRROR, 10e-4, 12e-4),
                           fields.Slab(19e-4, 40e-4, fields.KIND_UNIFORM, (0.0, 0.0, 3000.0))], (0.3, -0.2, 0.9))
    n = 1 << 15
    st = _states(n, rng, box=20e-4, center=(3e-4, -7e-4, 20e-4))
    ids = rng.integers(0, 2 ** 64, n, dtype=np.uint64)
    nidx = rng.integers(0, 1 << 20, n, dtype=np.uint64).astype(np.uint32)
    cpu = oracle.step_batch(g, fd, 5, st, ids, nidx)
    gpu = avm.step_batch_form(ctx, avm.gas_create(ctx, g), avm.field_create(ctx, fd), 5, st, ids, nidx, form=1)
    assert_step_parity(cpu, gpu, st, "NEXT-3 form 1 grid")


def test_next3_textbook_gases(avm, ctx, oracle):
    """The pins' gases on the device: strong forward scattering, Penning-only multiplication, a hot heavy-recoil gas."""
    rng = np.random.default_rng(260)
    n = 30000
    st = _states(n, rng, e_hi=60.0)
    fd = fields.uniform_gap((1500.0, -700.0, 2500.0), -1.0, 1.0, (0.1, 0.2, -0.4))
    ids = np.arange(n, dtype=np.uint64); nidx = np.zeros(n, dtype=np.uint32)
    ga = gas.constant_elastic(100.0, 0.02); ga.scat_xi = np.full((ga.n_bins, 1), 0.97)
    gp = gas.multi_level_constant([100.0], [gas.EXCITATION], loss=[11.5], n_bins=16, e_max=100.0)
    gp.level_penning_prob = np.array([0.37]); gp.level_penning_eV = np.array([4.2])
    gt = gas.constant_elastic(100.0, 0.3); gt.kT_eV = 2.0
    for g in (ga, gp, gt):
        cpu = oracle.step_batch(g, fd, 9, st, ids, nidx)
        for form in (0, 1):
            gpu = avm.step_batch_form(ctx, avm.gas_create(ctx, g), avm.field_create(ctx, fd), 9, st, ids, nidx, form=form)
            assert_step_parity(cpu, gpu, st, f"NEXT-3 textbook form {form}")


def test_next3_invalid_tables_are_rejected(avm, ctx, g0):
    g = copy.copy(g0); g.scat_xi = np.ones((g0.n_bins, g0.n_levels))
    with pytest.raises(avm.AvmError):
        avm.gas_create(ctx, g)
    g = copy.copy(g0); g.level_penning_prob = np.full(g0.n_levels, 1.5); g.level_penning_eV = np.zeros(g0.n_levels)
    with pytest.raises(avm.AvmError):
        avm.gas_create(ctx, g)
    g = copy.copy(g0); g.kT_eV = -1.0
    with pytest.raises(avm.AvmError):
        avm.gas_create(ctx, g)


@pytest.mark.parametrize("flags", [0, 16, 4])
def test_next3_config1_same_seed(avm, ctx, oracle, g0, flags):
    """Config 1 in full with all three extensions: identical avalanches, identical tallies (level counts, Penning
    transfers, null count); un-banded (time-parallel batches), banded, wide shape (serial batches)."""
    w = configs.config1()
    g = extended_g0(g0)
    cpu = oracle.run(g, w.field, w.primaries, seed=0, n_threads=CORES, flags=1 if flags & 16 else 0, capacity=1 << 16)
    gpu = avm.simulate(ctx, avm.gas_create(ctx, g), avm.field_create(ctx, w.field), w.primaries, seed=0, flags=flags, capacity=1 << 16)
    frac, _ = assert_run_same_seed(cpu, gpu, g.n_levels, label=f"NEXT-3 config1 full (flags {flags})")
    L = g.n_levels
    assert int(cpu.tallies_u64[L + 4]) > 20
    ion = sum(int(cpu.tallies_u64[l]) for l in range(L) if g.level_type[l] == gas.IONISATION)
    assert cpu.n == 1000 + ion + int(cpu.tallies_u64[L + 4])
    if frac == 1.0 and cpu.n == gpu.n:
        assert np.array_equal(cpu.tallies_u64, gpu.tallies_u64), (cpu.tallies_u64, gpu.tallies_u64)


def test_next3_full_warps_and_config2_same_seed(avm, ctx, oracle, g0):
    g = extended_g0(g0)
    w = configs.config2(n_primaries=16)
    fd = fields.uniform_gap((0.0, 0.0, -60000.0), 0.0, 80e-4)                  # config 2's field; the Penning gain fills 128 um with > 1e6 electrons
    cpu = oracle.run(g, fd, w.primaries, seed=0, capacity=1 << 20, n_threads=CORES)
    gpu = avm.simulate(ctx, avm.gas_create(ctx, g), avm.field_create(ctx, fd), w.primaries, seed=0, capacity=1 << 20)
    assert cpu.n > 20000
    assert_run_same_seed(cpu, gpu, g.n_levels, min_identical=0.999, label="NEXT-3 config2 field, 80 um gap, 16 primaries")
    # thermalisation on the device: no field, constant collision frequency, 293 K — <eps> = thermal_mean (oracle pin X3)
    gt = gas.constant_elastic(400.0, 0.04, n_bins=64, e_max=10.0); gt.kT_eV = 0.02526
    p = primaries.isotropic_primaries(80000, 61, e_scale=1.0)
    fd = fields.uniform_gap((0, 0, 0), -1e6, 1e6)
    r = avm.simulate(ctx, avm.gas_create(ctx, gt), avm.field_create(ctx, fd), p, seed=61, t_max=1.2, capacity=80000)
    e = r.end[4]
    from test_oracle_pins_next3 import thermal_mean
    exact = thermal_mean(gt.kT_eV, 0.04)
    assert abs(e.mean() - exact) < 4 * e.std(ddof=1) / np.sqrt(len(e)), (e.mean(), exact)
