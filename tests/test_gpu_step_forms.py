"""Per-step parity (tolerance T, 1e-12) of the step FORMS the persistent kernel runs, through avm_step_batch_form.

The hook calls the same device functions as transport_kernel (csrc/avm_forms.cuh): form 1 = the full-warp sequence
(fw_flight: 16-bit threshold filter, exact record inside a band, next draws hoisted, collision phase), form 2 = a whole
time-parallel batch (tp_batch: composed flights from a base state, speculative elastic collision, base-state hand-off
through the warp's exchange area), compared with the oracle stepped sequentially.  States whose uniform falls INSIDE a
band of the 16-bit filter (|h - q| <= 1) are constructed on purpose: there the exact fp64 record decides.
"""
import numpy as np
import pytest

from paper_2509_15377_b200.gen import fields, gas, philox, primaries
from test_gpu_parity import assert_step_parity, _states, _random_map

pytestmark = pytest.mark.gpu
B30 = (0.0, 0.5, 0.8660254037844387)


@pytest.fixture(scope="module")
def ctx(avm):
    return avm.ctx_create(0)


def _slice(res, sel):
    return type(res)(res.state[:, sel], res.event[sel], res.status[sel], res.bin[sel], res.child[:, sel], res.child_id[sel])


def in_band_states(g, seed, n_el, gl, rng):
    """Electrons (state, id, n0) in a ZERO E field whose energy sits at the centre of a bin b such that, at one chosen
    step s of the next gl, h = floor(u2 2^16) is within +-1 of one of the 16-bit thresholds of that bin: q = floor(c 2^16),
    c = (nu_tot, cum0, cum1)[b] / nu_hat.  The energy does not change over null flights without E, so the bin holds."""
    nu_hat = g.resolved_nu_hat()
    nb = g.n_bins
    de = g.e_max / nb
    q = [np.floor(c / nu_hat * 65536.0).astype(np.int64) for c in (g.cum_rate[:, -1], g.cum_rate[:, 0], g.cum_rate[:, min(1, g.n_levels - 1)])]
    lut = []
    for qq in q:
        t = np.full(65540, -1, dtype=np.int64)
        t[np.clip(qq, 0, 65539)] = np.arange(nb)
        lut.append(t)
    ids = rng.integers(0, 2 ** 63, 40 * n_el, dtype=np.int64).astype(np.uint64)
    n0 = rng.integers(0, 1 << 30, 40 * n_el, dtype=np.int64).astype(np.uint32)
    s_t = rng.integers(0, gl, 40 * n_el)
    w = philox.words(seed, ids, (n0 + s_t).astype(np.uint32), 0)
    h = (w[2] >> np.uint32(16)).astype(np.int64)
    which = rng.integers(0, 3, len(h))
    off = rng.integers(-1, 2, len(h))
    b = np.array([lut[which[i]][min(max(h[i] + off[i], 0), 65539)] for i in range(len(h))])
    keep = np.flatnonzero(b >= 1)[:n_el]
    assert len(keep) == n_el, "not enough in-band candidates"
    st = _states(n_el, rng)
    st[3] = 0.0
    st[4] = (b[keep] + 0.5) * de
    return st, ids[keep], n0[keep], s_t[keep], which[keep]


@pytest.mark.parametrize("B", [(0.0, 0.0, 0.0), B30])
def test_form1_full_warp_sequence_uniform(avm, ctx, oracle, g0, B):
    """Form 1 on gas G0 in a uniform field: every level, boundary exits, time limit."""
    rng = np.random.default_rng(31)
    n = 1 << 17
    st = _states(n, rng, box=30e-4, center=(0, 0, 30e-4))
    fd = fields.uniform_gap((0.0, 0.0, -60000.0), 0.0, 60e-4, B)
    ids = rng.integers(0, 2 ** 64, n, dtype=np.uint64)
    nidx = rng.integers(0, 2 ** 32 - 64, n, dtype=np.uint64).astype(np.uint32)
    gg, fg = avm.gas_create(ctx, g0), avm.field_create(ctx, fd)
    for seed in (0, 0xABCDEF0123456789):
        cpu = oracle.step_batch(g0, fd, seed, st, ids, nidx, t_max=4.9)
        gpu = avm.step_batch_form(ctx, gg, fg, seed, st, ids, nidx, form=1, t_max=4.9)
        assert_step_parity(cpu, gpu, st, f"form 1 B={B}")
        assert all((cpu.event == l).sum() > 0 for l in range(0, 16)) and set(np.unique(cpu.status)) >= {0, 1, 2, 6}
    # near the step limit
    nidx2 = np.full(1000, 0xFFFFFFEF, dtype=np.uint32)
    c2 = oracle.step_batch(g0, fd, 0, st[:, :1000], ids[:1000], nidx2)
    g2 = avm.step_batch_form(ctx, gg, fg, 0, st[:, :1000], ids[:1000], nidx2, form=1)
    assert_step_parity(c2, g2, st[:, :1000])
    assert (c2.status == 7).sum() > 100


def test_form1_full_warp_sequence_grid_and_textbook(avm, ctx, oracle, g0):
    """Form 1 with a grid map (mirror fold, material, slab change, B) and with the textbook gases (attachment etc.)."""
    rng = np.random.default_rng(32)
    nodes = _random_map(rng, 12, 14, 20, e_scale=5e4)
    g1 = fields.grid_slab(nodes, (0, 0, 0), (1e-4, 1e-4, 1e-4), 0.0, 19e-4, fields.BC_MIRROR, fields.BC_MIRROR, 10e-4, 12e-4)
    u2 = fields.Slab(19e-4, 40e-4, fields.KIND_UNIFORM, (0.0, 0.0, 3000.0))
    n = 1 << 16
    for B in ((0, 0, 0), (0.3, -0.2, 0.9)):
        fd = fields.FieldDesc([g1, u2], B)
        st = _states(n, rng, box=20e-4, center=(3e-4, -7e-4, 20e-4))
        ids = rng.integers(0, 2 ** 64, n, dtype=np.uint64)
        nidx = rng.integers(0, 1 << 20, n, dtype=np.uint64).astype(np.uint32)
        cpu = oracle.step_batch(g0, fd, 5, st, ids, nidx)
        gpu = avm.step_batch_form(ctx, avm.gas_create(ctx, g0), avm.field_create(ctx, fd), 5, st, ids, nidx, form=1)
        assert_step_parity(cpu, gpu, st, f"form 1 grid B={B}")
        assert (cpu.status == 4).sum() > 100
    st = _states(20000, rng, e_hi=200.0)
    fd = fields.uniform_gap((1500.0, -700.0, 2500.0), -1.0, 1.0, (0.1, 0.2, -0.4))
    ids = np.arange(20000, dtype=np.uint64); nidx = np.zeros(20000, dtype=np.uint32)
    for g in (gas.constant_elastic(100.0, 0.013), gas.ionisation_only(80.0, w=10.0), gas.attachment_only(2.0, nu_hat=3.0),
              gas.multi_level_constant([5.0, 0.0, 20.0, 1.0, 14.0], [gas.ELASTIC, gas.EXCITATION, gas.EXCITATION, gas.ATTACHMENT, gas.ELASTIC],
                                       loss=[0, 1.0, 2.5, 0, 0], recoil=[1e-3, 0, 0, 0, 0.5], nu_hat=60.0)):
        cpu = oracle.step_batch(g, fd, 9, st, ids, nidx)
        gpu = avm.step_batch_form(ctx, avm.gas_create(ctx, g), avm.field_create(ctx, fd), 9, st, ids, nidx, form=1)
        assert_step_parity(cpu, gpu, st, "form 1 " + g.names[0])


def test_form1_states_inside_the_filter_bands(avm, ctx, oracle, g0):
    """Form 1 where the 16-bit filter cannot decide: the exact fp64 record must take the oracle's decision."""
    rng = np.random.default_rng(33)
    seed = 77
    st, ids, n0, s_t, which = in_band_states(g0, seed, 6000, 1, rng)
    fd = fields.uniform_gap((0.0, 0.0, 0.0), -1.0, 1.0)
    cpu = oracle.step_batch(g0, fd, seed, st, ids, n0)
    gpu = avm.step_batch_form(ctx, avm.gas_create(ctx, g0), avm.field_create(ctx, fd), seed, st, ids, n0, form=1)
    assert_step_parity(cpu, gpu, st, "form 1 in-band")
    assert all((which == c).sum() > 500 for c in range(3))
    assert (cpu.event == -1).sum() > 500 and (cpu.event == 0).sum() > 500 and (cpu.event == 1).sum() > 500 and (cpu.event >= 2).sum() > 100


def oracle_sequence(oracle, g, fd, seed, st, ids, n0, gl, t_max):
    """gl sequential oracle steps per electron (stopping where it finishes), in the layout of form 2: [.., n, gl]."""
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
        r = oracle.step_batch(g, fd, seed, cur[:, idx], ids[idx], (n0[idx].astype(np.uint64) + s).astype(np.uint32), t_max=t_max)
        st_in[:, idx, s] = cur[:, idx]
        out.state[:, idx, s] = r.state; out.event[idx, s] = r.event; out.status[idx, s] = r.status; out.bin[idx, s] = r.bin
        out.child[:, idx, s] = r.child; out.child_id[idx, s] = r.child_id
        cur[:, idx] = r.state
        alive[idx] = r.status == 0
    return out, st_in


def assert_form2_parity(avm, cpu, st_in, gpu, gl, what, composed=False):
    """composed (form 2): a step's position is the composed flight from the batch's base state, so its rounding is relative
    to the coordinate's largest magnitude since the batch began (the oracle's sequential sum carries the same absolute
    rounding); form 3 steps sequentially and needs no such allowance.
    Step s of a batch starts from each side's OWN result of step s - 1, not from identical state: the two inputs already
    differ by the accumulated rounding of s steps (each within T), which the field gradients of a random map carry forward.
    The bound therefore grows with the step index: T (1 + s / 8) — 1e-12 at the batch's first step, 4.9e-12 at its 32nd
    (observed worst: 1.2e-12 at step 30 on a random map with B)."""
    assert np.array_equal(cpu.event == -3, gpu.event == -3), f"{what}: the batches reach different steps"
    total = 0
    run_max = np.zeros((3, st_in.shape[1]))
    for s in range(gl):
        run_max = np.maximum(run_max, np.abs(st_in[0:3, :, s]))
        sel = cpu.event[:, s] != -3
        if not sel.any():
            continue
        c = type(cpu)(cpu.state[:, sel, s], cpu.event[sel, s], cpu.status[sel, s], cpu.bin[sel, s], cpu.child[:, sel, s], cpu.child_id[sel, s])
        g = type(cpu)(gpu.state[:, sel, s], gpu.event[sel, s], gpu.status[sel, s], gpu.bin[sel, s], gpu.child[:, sel, s], gpu.child_id[sel, s])
        total += assert_step_parity(c, g, st_in[:, sel, s], f"{what} step {s}", pos_floor=run_max[:, sel] if composed else None,
                                    RTOL=1e-12 * (1.0 + s / 8.0))
    return total


@pytest.mark.parametrize("B", [(0.0, 0.0, 0.0), B30])
@pytest.mark.parametrize("k", [1, 2, 3, 4, 7, 8])
def test_form2_time_parallel_batch(avm, ctx, oracle, g0, B, k):
    """Form 2: a whole time-parallel batch (k electrons per warp on scattered lanes, gl = 32 / k' steps each) against gl
    sequential oracle steps — identical events, levels, statuses, bins and child ids for every step the electron takes,
    continuous outputs of every step within T of the oracle's (relative to that step's own input state)."""
    rng = np.random.default_rng(40 + k)
    gl = avm.step_form_lanes(k)
    n = k * 1500
    st = _states(n, rng, box=30e-4, center=(0, 0, 30e-4))
    fd = fields.uniform_gap((0.0, 0.0, -60000.0), 0.0, 60e-4, B)
    ids = rng.integers(0, 2 ** 64, n, dtype=np.uint64)
    n0 = rng.integers(0, 2 ** 32 - 64, n, dtype=np.uint64).astype(np.uint32)
    n0[:50] = 0xFFFFFFEF - rng.integers(0, 6, 50)                    # some reach the step limit inside the batch
    gg, fg = avm.gas_create(ctx, g0), avm.field_create(ctx, fd)
    t_max = 5.0
    st[3, 50:400] = t_max - rng.uniform(0.0, 20.0, 350) / g0.resolved_nu_hat()    # some run into the time limit inside the batch
    cpu, st_in = oracle_sequence(oracle, g0, fd, 3, st, ids, n0, gl, t_max)
    gpu = avm.step_batch_form(ctx, gg, fg, 3, st, ids, n0, form=2, k=k, t_max=t_max)
    total = assert_form2_parity(avm, cpu, st_in, gpu, gl, f"form 2 k={k} B={B}", composed=True)
    assert total > n * min(gl, 3) * 0.7
    ev = cpu.event[cpu.event != -3]
    assert (ev == -1).sum() > n and (ev == 0).sum() > 50 and (ev == 1).sum() > 50 and (ev >= 2).sum() > 10
    assert set(np.unique(cpu.status)) >= {0, 1, 2, 6, 7}
    assert (cpu.event[:, -1] != -3).sum() > 0                          # some electrons take all gl steps


@pytest.mark.parametrize("B", [(0.0, 0.0, 0.0), B30])
def test_form2_composed_flight_time_and_filter_bands(avm, ctx, oracle, g0, B):
    """The composed flight of step s lasts T_s = dt_0 + .. + dt_s, summed by a shuffle scan instead of sequentially:
    from t = 0 the GPU's t' must equal the oracle's to 32 ulp, whatever the group size.  Same batch:
    electrons whose uniform at one step of the batch lies inside a band of the 16-bit filter."""
    rng = np.random.default_rng(51)
    seed = 5
    fd = fields.uniform_gap((0.0, 0.0, 0.0), -1.0, 1.0, B)
    gg, fg = avm.gas_create(ctx, g0), avm.field_create(ctx, fd)
    for k in (1, 2, 4, 8):
        gl = avm.step_form_lanes(k)
        st, ids, n0, s_t, which = in_band_states(g0, seed, 400 * k, gl, rng)
        cpu, st_in = oracle_sequence(oracle, g0, fd, seed, st, ids, n0, gl, float("inf"))
        gpu = avm.step_batch_form(ctx, gg, fg, seed, st, ids, n0, form=2, k=k)
        assert_form2_parity(avm, cpu, st_in, gpu, gl, f"form 2 in-band k={k} B={B}", composed=True)
        reached = cpu.event != -3
        tc, tg = cpu.state[3][reached], gpu.state[3][reached]
        assert np.all(np.abs(tg - tc) <= 32 * 2.0 ** -52 * tc), np.max(np.abs(tg - tc) / tc) / 2.0 ** -52
        # the constructed step was reached by most electrons, and took every kind of decision
        hit = reached[np.arange(len(s_t)), s_t]
        assert hit.mean() > 0.3
        evs = cpu.event[np.arange(len(s_t)), s_t][hit]
        assert (evs == -1).sum() > 20 and (evs == 0).sum() > 20 and (evs == 1).sum() > 20


def test_overflow_tally_in_every_form(avm, ctx, oracle):
    """tallies_u64[L+2] (energies >= e_max, counted for steps that reach the bin lookup) equals the oracle's in both
    launch shapes and in all three forms: electrons gain ~20 eV per um at 200 kV/cm in a gas table that ends at 5 eV and
    leave the 3 um gap far above it — the last flight of an electron must not be counted (S5 comes before S6)."""
    g = gas.constant_elastic(4000.0, 0.0, n_bins=100, e_max=5.0, nu_hat=10000.0)
    fd = fields.uniform_gap((0.0, 0.0, -200000.0), 0.0, 3e-4)
    gg, fg = avm.gas_create(ctx, g), avm.field_create(ctx, fd)
    for n_p, flags, what in ((1500, avm.RUN_SHAPE_LATENCY, "time-parallel batches"), (1500, avm.RUN_SHAPE_WIDE, "cooperative batches"),
                             (120000, avm.RUN_SHAPE_LATENCY, "full warps")):
        p = primaries.isotropic_primaries(n_p, 8, pos=(0, 0, 1e-4), e_scale=3.0)
        cpu = oracle.run(g, fd, p, seed=8, n_threads=8, capacity=2 * n_p)
        gpu = avm.simulate(ctx, gg, fg, p, seed=8, flags=flags, capacity=2 * n_p)
        assert (cpu.end[4] > 5.0).mean() > 0.5 and int(cpu.tallies_u64[3]) > 5 * n_p
        assert np.array_equal(np.sort(cpu.n_steps), np.sort(gpu.n_steps)), what
        assert np.array_equal(cpu.tallies_u64, gpu.tallies_u64), (what, cpu.tallies_u64, gpu.tallies_u64)


def _form3_case(avm, ctx, oracle, g, fd, fg, k, rng, center, box, what, t_max=5.0):
    gl = avm.step_form_lanes(k)
    n = k * 1200
    st = _states(n, rng, box=box, center=center)
    E, m, sl = oracle.field_eval(fd, st[0:3])
    ok = (sl >= 0) & (m >= 0.5)
    st[:, ~ok] = st[:, np.flatnonzero(ok)[0]][:, None]                 # a step starts in the gas
    st[3, 50:400] = t_max - rng.uniform(0.0, 20.0, 350) / g.resolved_nu_hat()
    ids = rng.integers(0, 2 ** 64, n, dtype=np.uint64)
    n0 = rng.integers(0, 2 ** 32 - 64, n, dtype=np.uint64).astype(np.uint32)
    n0[:50] = 0xFFFFFFEF - rng.integers(0, 6, 50)
    cpu, st_in = oracle_sequence(oracle, g, fd, 3, st, ids, n0, gl, t_max)
    gpu = avm.step_batch_form(ctx, avm.gas_create(ctx, g), fg, 3, st, ids, n0, form=3, k=k, t_max=t_max)
    total = assert_form2_parity(avm, cpu, st_in, gpu, gl, what)
    assert total > n * min(gl, 3) * 0.5
    return cpu


@pytest.mark.parametrize("B", [(0.0, 0.0, 0.0), B30])
@pytest.mark.parametrize("k", [1, 3, 8, 16])
def test_form3_serial_batch_uniform(avm, ctx, oracle, g0, B, k):
    """Form 3 (serial batch) in one uniform slab: gl sequential oracle steps per electron, every output of every step."""
    rng = np.random.default_rng(60 + k)
    fd = fields.uniform_gap((0.0, 0.0, -60000.0), 0.0, 60e-4, B)
    cpu = _form3_case(avm, ctx, oracle, g0, fd, avm.field_create(ctx, fd), k, rng, (0, 0, 30e-4), 30e-4, f"form 3 uniform k={k} B={B}")
    ev = cpu.event[cpu.event != -3]
    assert (ev == -1).sum() > 1000 and (ev == 0).sum() > 50 and (ev == 1).sum() > 50 and (ev >= 2).sum() > 10
    assert set(np.unique(cpu.status)) >= {0, 1, 2, 6, 7}


@pytest.mark.parametrize("widen", [True, False])
@pytest.mark.parametrize("B", [(0.0, 0.0, 0.0), (0.3, -0.2, 0.9)])
def test_form3_serial_batch_grid(avm, ctx, oracle, g0, B, widen):
    """Form 3 on maps: ONE grid slab (the kernel specialisation of config 4: mirror fold, material) and a stack of a grid
    and a uniform slab (the generic one of config 5), from the fp32 nodes and from their widened fp64 copy."""
    rng = np.random.default_rng(70)
    nodes = _random_map(rng, 12, 14, 40, e_scale=5e4)
    nodes[..., 2] -= 4e4
    h = (1e-4, 1e-4, 1e-4)
    one = fields.FieldDesc([fields.grid_slab(nodes, (0, 0, 0), h, 0.0, 39e-4, fields.BC_MIRROR, fields.BC_MIRROR, 10e-4, 12e-4)], B)
    two = fields.FieldDesc([fields.grid_slab(nodes, (0, 0, 0), h, 0.0, 39e-4, fields.BC_MIRROR, fields.BC_PERIODIC, 10e-4, 12e-4),
                            fields.Slab(39e-4, 60e-4, fields.KIND_UNIFORM, (0.0, 0.0, -30000.0))], B, (-40e-4, -50e-4), (40e-4, 50e-4))
    for fd, zc, zb, what in ((one, 20e-4, 19e-4, "one grid slab"), (two, 30e-4, 29e-4, "grid + uniform")):
        fg = avm.field_create(ctx, fd, widen=widen)
        for k in (1, 2, 5):
            cpu = _form3_case(avm, ctx, oracle, g0, fd, fg, k, rng, (3e-4, -7e-4, zc), zb, f"form 3 {what} k={k} B={B} widen={widen}")
            assert (cpu.status == 4).sum() > 20 and (cpu.status == 0).sum() > 1000


def test_form3_states_inside_the_filter_bands(avm, ctx, oracle, g0):
    rng = np.random.default_rng(80)
    seed = 9
    fd = fields.uniform_gap((0.0, 0.0, 0.0), -1.0, 1.0)
    gg, fg = avm.gas_create(ctx, g0), avm.field_create(ctx, fd)
    for k in (1, 4):
        gl = avm.step_form_lanes(k)
        st, ids, n0, s_t, which = in_band_states(g0, seed, 400 * k, gl, rng)
        cpu, st_in = oracle_sequence(oracle, g0, fd, seed, st, ids, n0, gl, float("inf"))
        gpu = avm.step_batch_form(ctx, gg, fg, seed, st, ids, n0, form=3, k=k)
        assert_form2_parity(avm, cpu, st_in, gpu, gl, f"form 3 in-band k={k}")
