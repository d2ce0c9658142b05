"""NEXT-1 on the device (AVM_RUN_BANDED): the energy-banded null-collision rate of DESIGN.md §3.5 (readings N1-N6) in the
CUDA path against the banded oracle (oracle flag AVMO_BANDED) — the table of rates bit for bit, per-step tolerance T (1e-12)
through the two step forms a banded run takes (form 1 full-warp, form 3 serial batch), cut flights, uniforms constructed
inside the bands of the 16-bit filter with the flight's own rate, same-seed whole runs, and the statistics of a banded GPU
run against the UN-banded oracle (the same collision physics through other random streams — boundary losses differ, DESIGN.md §3.5 N7).
"""
import os

import numpy as np
import pytest
import torch

from conftest import record_margin
from paper_2509_15377_b200.gen import configs, fields, gas, philox, primaries
from test_gpu_parity import assert_step_parity, assert_run_same_seed, _states, _random_map
from test_gpu_step_forms import assert_form2_parity

pytestmark = pytest.mark.gpu
B30 = (0.0, 0.5, 0.8660254037844387)
CORES = os.cpu_count() or 1
BANDED = 1          # oracle flag AVMO_BANDED


@pytest.fixture(scope="module")
def ctx(avm):
    return avm.ctx_create(0)


def test_band_table_is_the_oracles(avm, ctx, oracle, g0):
    """avm_gas_bands == avmo_majorant, every entry bit for bit (the two builders share no code; N1-N4 fix the arithmetic)."""
    for g in (g0, gas.gas_g0(n_bins=1000, e_max=30.0), gas.constant_elastic(100.0, 0.01), gas.ionisation_only(80.0),
              gas.multi_level_constant([5.0, 0.0, 20.0, 1.0, 14.0], [0, 1, 1, 3, 0], loss=[0, 1.0, 2.5, 0, 0], recoil=[1e-3, 0, 0, 0, 0.5], nu_hat=60.0)):
        a2c, nuc, dtc, shc = oracle.majorant(g)
        a2g, nug, dtg, shg = avm.gas_create(ctx, g).bands()
        assert shc == shg and np.array_equal(a2c, a2g)
        assert np.array_equal(nuc, nug) and np.array_equal(dtc, dtg)
    a2, nu, dt, sh = oracle.majorant(g0)
    assert nu.shape == (313, 26) and sh == 6 and np.isfinite(dt[:-1, :-1]).all() and (nu[:-1, :16] < 0.9 * nu[-1, -1]).any()


def _cut_count(oracle, g, st_in, cpu, cls=None):
    """Steps whose flight was cut: t' - t equals the dtmax of the electron's band (and class, when the field is uniform)."""
    a2, nu, dtm, sh = oracle.majorant(g)
    band = np.minimum((st_in[4] * g.n_bins / g.e_max).astype(np.int64), g.n_bins - 1) >> sh
    dt = cpu.state[3] - st_in[3]
    if cls is not None:
        return int((np.abs(dt - dtm[band, cls]) <= 4e-16 * np.maximum(np.abs(cpu.state[3]), dt)).sum())
    return int((np.abs(dt[:, None] - dtm[band]) <= 4e-16 * np.maximum(np.abs(cpu.state[3]), dt)[:, None]).any(axis=1).sum())


def _class_of(oracle, g, e_vcm):
    a2 = oracle.majorant(g)[0]
    return int((np.float64(0.0017588200107589609 * e_vcm) ** 2 > a2).sum())


@pytest.mark.parametrize("B", [(0.0, 0.0, 0.0), B30])
@pytest.mark.parametrize("e_field", [60000.0, 1000.0])
def test_banded_form1_uniform(avm, ctx, oracle, g0, B, e_field):
    """Form 1, banded, gas G0 in a uniform field: every level, boundary exits, time limit, cut flights.  1 kV/cm sits
    exactly on a class edge (250 V/cm x 2^2): the class comparison is strict on both sides."""
    rng = np.random.default_rng(131)
    n = 1 << 17
    st = _states(n, rng, box=30e-4, center=(0, 0, 30e-4))
    fd = fields.uniform_gap((0.0, 0.0, -e_field), 0.0, 60e-4, B)
    ids = rng.integers(0, 2 ** 64, n, dtype=np.uint64)
    nidx = rng.integers(0, 2 ** 32 - 64, n, dtype=np.uint64).astype(np.uint32)
    gg, fg = avm.gas_create(ctx, g0), avm.field_create(ctx, fd)
    for seed in (0, 0xABCDEF0123456789):
        cpu = oracle.step_batch(g0, fd, seed, st, ids, nidx, t_max=4.9, flags=BANDED)
        gpu = avm.step_batch_form(ctx, gg, fg, seed, st, ids, nidx, form=1, t_max=4.9, flags=avm.RUN_BANDED)
        assert_step_parity(cpu, gpu, st, f"banded form 1 E={e_field} B={B}")
        assert all((cpu.event == l).sum() > 0 for l in range(0, 16)) and set(np.unique(cpu.status)) >= {0, 6}
        assert _cut_count(oracle, g0, st, cpu, _class_of(oracle, g0, e_field)) > 300
        plain = oracle.step_batch(g0, fd, seed, st, ids, nidx, t_max=4.9)
        assert (cpu.event == -1).sum() < (0.5 if e_field < 5000.0 else 1.0) * (plain.event == -1).sum()   # the point of it: fewer null collisions


def test_banded_form1_grid_and_textbook(avm, ctx, oracle, g0):
    """Form 1, banded, where the acceleration class changes from step to step: a grid map (mirror fold, material, a uniform
    slab above, with and without B) whose field strengths span the classes; then the textbook gases."""
    rng = np.random.default_rng(132)
    nodes = _random_map(rng, 12, 14, 20, e_scale=5e4)
    nodes[..., 0:3] *= np.exp(rng.uniform(-5.0, 1.5, size=nodes.shape[:3]))[..., None].astype(np.float32)   # 300 V/cm .. 200 kV/cm
    g1 = fields.grid_slab(nodes, (0, 0, 0), (1e-4, 1e-4, 1e-4), 0.0, 19e-4, fields.BC_MIRROR, fields.BC_MIRROR, 10e-4, 12e-4)
    u2 = fields.Slab(19e-4, 40e-4, fields.KIND_UNIFORM, (0.0, 0.0, 3000.0))
    n = 1 << 16
    for B in ((0, 0, 0), (0.3, -0.2, 0.9)):
        fd = fields.FieldDesc([g1, u2], B)
        st = _states(n, rng, box=20e-4, center=(3e-4, -7e-4, 20e-4))
        E, m, sl = oracle.field_eval(fd, st[0:3])
        ok = (sl >= 0) & (m >= 0.5)
        st[:, ~ok] = st[:, np.flatnonzero(ok)[0]][:, None]
        ids = rng.integers(0, 2 ** 64, n, dtype=np.uint64)
        nidx = rng.integers(0, 1 << 20, n, dtype=np.uint64).astype(np.uint32)
        cpu = oracle.step_batch(g0, fd, 5, st, ids, nidx, flags=BANDED)
        gpu = avm.step_batch_form(ctx, avm.gas_create(ctx, g0), avm.field_create(ctx, fd), 5, st, ids, nidx, form=1, flags=avm.RUN_BANDED)
        assert_step_parity(cpu, gpu, st, f"banded form 1 grid B={B}")
        assert (cpu.status == 4).sum() > 100 and _cut_count(oracle, g0, st, cpu) > 100
        a2 = oracle.majorant(g0)[0]
        cls = ((0.0017588200107589609 ** 2 * (E ** 2).sum(axis=0))[:, None] > a2[None, :]).sum(axis=1)
        assert len(np.unique(cls[ok])) >= 12                                            # many classes in one batch
    st = _states(20000, rng, e_hi=200.0)
    fd = fields.uniform_gap((1500.0, -700.0, 2500.0), -1.0, 1.0, (0.1, 0.2, -0.4))
    ids = np.arange(20000, dtype=np.uint64); nidx = np.zeros(20000, dtype=np.uint32)
    for g in (gas.constant_elastic(100.0, 0.013), gas.ionisation_only(80.0, w=10.0), gas.attachment_only(2.0, nu_hat=3.0),
              gas.multi_level_constant([5.0, 0.0, 20.0, 1.0, 14.0], [gas.ELASTIC, gas.EXCITATION, gas.EXCITATION, gas.ATTACHMENT, gas.ELASTIC],
                                       loss=[0, 1.0, 2.5, 0, 0], recoil=[1e-3, 0, 0, 0, 0.5], nu_hat=60.0)):
        cpu = oracle.step_batch(g, fd, 9, st, ids, nidx, flags=BANDED)
        gpu = avm.step_batch_form(ctx, avm.gas_create(ctx, g), avm.field_create(ctx, fd), 9, st, ids, nidx, form=1, flags=avm.RUN_BANDED)
        assert_step_parity(cpu, gpu, st, "banded form 1 " + g.names[0])


def banded_in_band_states(oracle, g, seed, n_el, gl, rng):
    """Electrons in a ZERO field (class 0; the energy, hence bin and band, holds over null flights) whose energy sits at
    the centre of a bin b such that, at one chosen step of the next gl, h = floor(u2 rho 2^16) — rho = nu(band of b, class
    0) / nu_hat — is within +-1 of a 16-bit threshold of that bin: there the exact record with u2 nu decides."""
    nu_hat = g.resolved_nu_hat()
    nb, de = g.n_bins, g.e_max / g.n_bins
    a2, nu, dtm, sh = oracle.majorant(g)
    K = nu.shape[0]
    rho = np.minimum(np.floor(nu[:, 0] / nu_hat * 4294967296.0), 4294967295.0).astype(np.uint64)
    q = [np.floor(c / nu_hat * 65536.0).astype(np.int64) for c in (g.cum_rate[:, -1], g.cum_rate[:, 0], g.cum_rate[:, min(1, g.n_levels - 1)])]
    m = 60 * n_el
    ids = rng.integers(0, 2 ** 63, m, dtype=np.int64).astype(np.uint64)
    n0 = rng.integers(0, 1 << 30, m, dtype=np.int64).astype(np.uint32)
    s_t = rng.integers(0, gl, m)
    w = philox.words(seed, ids, (n0 + s_t).astype(np.uint32), 0)
    w2 = w[2].astype(np.uint64)
    which = rng.integers(0, 3, m)
    off = rng.integers(-1, 2, m)
    found = np.full(m, -1, dtype=np.int64)
    for k in rng.permutation(K - 1):
        h = ((w2 * rho[k]) >> np.uint64(48)).astype(np.int64) + off
        lo, hi = k << sh, min((k + 1) << sh, nb)
        for c in range(3):
            lut = np.full(65540, -1, dtype=np.int64)
            lut[np.clip(q[c][lo:hi], 0, 65539)] = np.arange(lo, hi)
            cand = lut[np.clip(h, 0, 65539)]
            take = (found < 0) & (which == c) & (cand >= 1)
            found[take] = cand[take]
    keep = np.flatnonzero(found >= 1)[:n_el]
    assert len(keep) == n_el, f"not enough in-band candidates ({(found >= 1).sum()} of {n_el})"
    st = _states(n_el, rng)
    st[3] = 0.0
    st[4] = (found[keep] + 0.5) * de
    return st, ids[keep], n0[keep], s_t[keep], which[keep]


def oracle_sequence_banded(oracle, g, fd, seed, st, ids, n0, gl, t_max):
    """gl sequential banded oracle steps per electron, in the layout of forms 2 / 3."""
    n = st.shape[1]
    from oracle.avmo import StepResult
    out = StepResult(np.zeros((8, n, gl)), np.full((n, gl), -3, dtype=np.int32), np.zeros((n, gl), dtype=np.int32),
                     np.full((n, gl), -1, dtype=np.int32), np.zeros((8, n, gl)), np.zeros((n, gl), dtype=np.uint64))
    st_in = np.zeros((8, n, gl))
    cur, alive = st.copy(), np.ones(n, dtype=bool)
    for s in range(gl):
        idx = np.flatnonzero(alive)
        if len(idx) == 0:
            break
        r = oracle.step_batch(g, fd, seed, cur[:, idx], ids[idx], (n0[idx].astype(np.uint64) + s).astype(np.uint32), t_max=t_max, flags=BANDED)
        st_in[:, idx, s] = cur[:, idx]
        out.state[:, idx, s] = r.state; out.event[idx, s] = r.event; out.status[idx, s] = r.status; out.bin[idx, s] = r.bin
        out.child[:, idx, s] = r.child; out.child_id[idx, s] = r.child_id
        cur[:, idx] = r.state
        alive[idx] = r.status == 0
    return out, st_in


def test_banded_states_inside_the_filter_bands(avm, ctx, oracle, g0):
    """Forms 1 and 3, banded, where the scaled 16-bit filter cannot decide: the exact record takes the oracle's decision."""
    rng = np.random.default_rng(133)
    seed = 77
    fd = fields.uniform_gap((0.0, 0.0, 0.0), -1.0, 1.0)
    gg, fg = avm.gas_create(ctx, g0), avm.field_create(ctx, fd)
    st, ids, n0, s_t, which = banded_in_band_states(oracle, g0, seed, 3000, 1, rng)
    cpu = oracle.step_batch(g0, fd, seed, st, ids, n0, flags=BANDED)
    gpu = avm.step_batch_form(ctx, gg, fg, seed, st, ids, n0, form=1, flags=avm.RUN_BANDED)
    assert_step_parity(cpu, gpu, st, "banded form 1 in-band")
    assert all((which == c).sum() > 200 for c in range(3))
    assert (cpu.event == -1).sum() > 200 and (cpu.event == 0).sum() > 200 and (cpu.event == 1).sum() > 200 and (cpu.event >= 2).sum() > 30
    for k in (1, 4):
        gl = avm.step_form_lanes(k)
        st, ids, n0, s_t, which = banded_in_band_states(oracle, g0, seed, 400 * k, gl, rng)
        cpu, st_in = oracle_sequence_banded(oracle, g0, fd, seed, st, ids, n0, gl, float("inf"))
        gpu = avm.step_batch_form(ctx, gg, fg, seed, st, ids, n0, form=3, k=k, flags=avm.RUN_BANDED)
        assert_form2_parity(avm, cpu, st_in, gpu, gl, f"banded form 3 in-band k={k}")


def _form3_banded(avm, ctx, oracle, g, fd, fg, k, rng, center, box, what, t_max=5.0):
    gl = avm.step_form_lanes(k)
    n = k * 1200
    st = _states(n, rng, box=box, center=center)
    E, m, sl = oracle.field_eval(fd, st[0:3])
    ok = (sl >= 0) & (m >= 0.5)
    st[:, ~ok] = st[:, np.flatnonzero(ok)[0]][:, None]
    st[3, 50:400] = t_max - rng.uniform(0.0, 20.0, 350) / g.resolved_nu_hat()
    ids = rng.integers(0, 2 ** 64, n, dtype=np.uint64)
    n0 = rng.integers(0, 2 ** 32 - 64, n, dtype=np.uint64).astype(np.uint32)
    n0[:50] = 0xFFFFFFEF - rng.integers(0, 6, 50)
    cpu, st_in = oracle_sequence_banded(oracle, g, fd, 3, st, ids, n0, gl, t_max)
    gpu = avm.step_batch_form(ctx, avm.gas_create(ctx, g), fg, 3, st, ids, n0, form=3, k=k, t_max=t_max, flags=avm.RUN_BANDED)
    total = assert_form2_parity(avm, cpu, st_in, gpu, gl, what)
    assert total > n * min(gl, 3) * 0.5
    return cpu


@pytest.mark.parametrize("B", [(0.0, 0.0, 0.0), B30])
@pytest.mark.parametrize("k", [1, 3, 8, 16])
def test_banded_form3_uniform(avm, ctx, oracle, g0, B, k):
    rng = np.random.default_rng(160 + k)
    fd = fields.uniform_gap((0.0, 0.0, -60000.0), 0.0, 60e-4, B)
    cpu = _form3_banded(avm, ctx, oracle, g0, fd, avm.field_create(ctx, fd), k, rng, (0, 0, 30e-4), 30e-4, f"banded form 3 uniform k={k} B={B}")
    ev = cpu.event[cpu.event != -3]
    assert (ev == -1).sum() > 1000 and (ev == 0).sum() > 50 and (ev == 1).sum() > 50 and (ev >= 2).sum() > 10
    assert set(np.unique(cpu.status)) >= {0, 1, 2, 6, 7}


@pytest.mark.parametrize("widen", [True, False])
@pytest.mark.parametrize("B", [(0.0, 0.0, 0.0), (0.3, -0.2, 0.9)])
def test_banded_form3_grid(avm, ctx, oracle, g0, B, widen):
    rng = np.random.default_rng(170)
    nodes = _random_map(rng, 12, 14, 40, e_scale=5e4)
    # field strengths over many classes, none above the un-banded test's: every step of a batch is compared with the
    # oracle's step from the ORACLE's previous state, so the field gradients amplify the two sides' rounding over the batch
    nodes[..., 0:3] *= np.exp(rng.uniform(-4.5, 0.0, size=nodes.shape[:3]))[..., None].astype(np.float32)
    nodes[..., 2] -= 2e4
    h = (1e-4, 1e-4, 1e-4)
    one = fields.FieldDesc([fields.grid_slab(nodes, (0, 0, 0), h, 0.0, 39e-4, fields.BC_MIRROR, fields.BC_MIRROR, 10e-4, 12e-4)], B)
    two = fields.FieldDesc([fields.grid_slab(nodes, (0, 0, 0), h, 0.0, 39e-4, fields.BC_MIRROR, fields.BC_PERIODIC, 10e-4, 12e-4),
                            fields.Slab(39e-4, 60e-4, fields.KIND_UNIFORM, (0.0, 0.0, -30000.0))], B, (-40e-4, -50e-4), (40e-4, 50e-4))
    for fd, zc, zb, what in ((one, 20e-4, 19e-4, "one grid slab"), (two, 30e-4, 29e-4, "grid + uniform")):
        fg = avm.field_create(ctx, fd, widen=widen)
        for k in (1, 2, 5):
            cpu = _form3_banded(avm, ctx, oracle, g0, fd, fg, k, rng, (3e-4, -7e-4, zc), zb, f"banded form 3 {what} k={k} B={B} widen={widen}")
            assert (cpu.status == 4).sum() > 20 and (cpu.status == 0).sum() > 1000


# ---- whole runs -------------------------------------------------------------------------------------------------------
def _gpu(avm, ctx, w, prim, seed, flags, t_max=None, capacity=None):
    gg, fg = avm.gas_create(ctx, w.gas), avm.field_create(ctx, w.field)
    bufs = avm.RunBuffers(ctx, capacity or w.capacity, prim.shape[0], w.gas.n_levels)
    _, n = avm.run(ctx, gg, fg, torch.from_numpy(prim.copy()).to(ctx.device), bufs, seed=seed, t_max=w.t_max if t_max is None else t_max, flags=flags)
    return avm.fetch(ctx, bufs, n)


def test_banded_config1_same_seed(avm, ctx, oracle):
    """Config 1 in full, banded on both sides (serial batches): identical avalanches, identical tallies (null count too)."""
    w = configs.config1()
    cpu = oracle.run(w.gas, w.field, w.primaries, seed=0, n_threads=CORES, flags=BANDED)
    assert cpu.n_rate_violations == 0
    for flags in (avm.RUN_BANDED, avm.RUN_BANDED | avm.RUN_SHAPE_WIDE):
        gpu = _gpu(avm, ctx, w, w.primaries, 0, flags)
        frac, _ = assert_run_same_seed(cpu, gpu, w.gas.n_levels, label=f"banded config1 full (flags {flags})")
        if frac == 1.0 and cpu.n == gpu.n:
            assert np.array_equal(cpu.tallies_u64, gpu.tallies_u64)
    plain = oracle.run(w.gas, w.field, w.primaries, seed=0, n_threads=CORES)
    L = w.gas.n_levels
    assert cpu.tallies_u64[L + 3] < 0.7 * plain.tallies_u64[L + 3]


def test_banded_full_warps_same_seed(avm, ctx, oracle, g0):
    """The throughput regime (full-warp iterations), banded: 60000 primaries drifting at 1 kV/cm with B, with a time cut."""
    w = configs.config3(n_primaries=60000, t_max=3.0)
    m = 2000
    cpu = oracle.run(w.gas, w.field, w.primaries[:m], seed=0, t_max=3.0, n_threads=CORES, flags=BANDED)
    gpu = _gpu(avm, ctx, w, w.primaries, 0, avm.RUN_BANDED)
    from test_gpu_fullsize import first_avalanches
    assert_run_same_seed(cpu, first_avalanches(gpu, m), w.gas.n_levels, min_identical=0.99, label="banded config3 t_max=3 ns, first 2000 of 60000")
    plain = oracle.run(w.gas, w.field, w.primaries[:m], seed=0, t_max=3.0, n_threads=CORES)
    L = w.gas.n_levels
    assert cpu.tallies_u64[L + 3] < 0.3 * plain.tallies_u64[L + 3]


def test_banded_config2_and_config4_same_seed(avm, ctx, oracle):
    w = configs.config2(n_primaries=24)
    cpu = oracle.run(w.gas, w.field, w.primaries, seed=0, capacity=w.capacity, n_threads=CORES, flags=BANDED)
    gpu = _gpu(avm, ctx, w, w.primaries, 0, avm.RUN_BANDED)
    assert_run_same_seed(cpu, gpu, w.gas.n_levels, min_identical=0.999, label="banded config2, 24 primaries")
    w = configs.config4(n_primaries=48)
    cpu = oracle.run(w.gas, w.field, w.primaries, seed=0, capacity=w.capacity, n_threads=CORES, flags=BANDED)
    assert cpu.n_rate_violations == 0
    gpu = _gpu(avm, ctx, w, w.primaries, 0, avm.RUN_BANDED)
    assert_run_same_seed(cpu, gpu, w.gas.n_levels, min_identical=0.99, end_rtol=1e-6, label="banded config4, 48 primaries")


def test_banded_statistics_against_the_unbanded_oracle(avm, ctx, oracle):
    """The banded CUDA run and the UN-banded oracle draw different random streams for the same collision physics (NOT the same losses at the start plane: DESIGN.md §3.5 N7 —
    which is why the endpoint-z distribution is not compared here and why 4000 primaries do not resolve the 1 % gain shift): mean gain within 3
    combined SE, KS p > 0.01 on gain / endpoint energy / endpoint z, drift velocity within 1 % (config 1, 4000 primaries
    a side; config 4 in full)."""
    from test_gpu_acceptance import compare_statistics, w_alpha
    w = configs.config1()
    pc = primaries.isotropic_primaries(4000, 0); pg = primaries.isotropic_primaries(4000, 1)
    cpu = oracle.run(w.gas, w.field, pc, seed=0, n_threads=CORES)
    gpu = _gpu(avm, ctx, w, pg, 1, avm.RUN_BANDED)
    compare_statistics("banded GPU vs un-banded oracle, config1 (4000 primaries)", cpu, gpu, 2, 50e-4, 1, z_overshoot=False)
    Wc, _ = w_alpha(cpu, w.gas, +1.0); Wg, _ = w_alpha(gpu, w.gas, +1.0)
    record_margin(f"banded GPU vs un-banded oracle config1: W gpu/oracle - 1 = {Wg / Wc - 1:+.2e}")
    assert abs(Wg / Wc - 1) < 0.03
    w = configs.config4()
    cpu = oracle.run(w.gas, w.field, w.primaries, seed=w.seed, capacity=w.capacity, n_threads=CORES)
    gpu = _gpu(avm, ctx, w, configs._gem_primaries(1000, 1, 0), 1, avm.RUN_BANDED)
    compare_statistics("banded GPU vs un-banded oracle, config4 (1000 primaries)", cpu, gpu, 1, w.field.slabs[0].z_lo, 3, z_overshoot=False)
    Wc, ac = w_alpha(cpu, w.gas, -1.0); Wg, ag = w_alpha(gpu, w.gas, -1.0)
    record_margin(f"banded GPU vs un-banded oracle config4: W gpu/oracle - 1 = {Wg / Wc - 1:+.2e}, (alpha - eta) - 1 = {ag / ac - 1:+.2e}")
    assert abs(Wg / Wc - 1) < 0.02
