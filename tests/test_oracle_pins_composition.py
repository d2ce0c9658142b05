"""Oracle pins, part 3: how the pieces of a step compose (CPU only).

Part 2 pins each piece of oracle/avmo.cpp by a closed form; these pin the places where two pieces meet, which a
piecewise pin cannot see: the excitation loss indexed by the selected level (S9c), the energy bin taken from the energy
AFTER the flight (S6 on eps'), the overflow count (S6, counted only for steps that pass S5), the energy ledger of a whole
avalanche, and — pin C17 of SURVEY.md §8(c) — every output of 1000+ steps against an independent 40-digit
transcription of S0-S9 (tests/transcription_s0_s9.py, which calls nothing under oracle/).
"""
import dataclasses

import numpy as np
import pytest

from paper_2509_15377_b200.gen import fields, gas, philox, primaries

KAPPA = 0.0017588200107589609
C2 = 0.05930969584745753
BIG = 1.0e6


def _open_field(E, B=(0, 0, 0)):
    return fields.uniform_gap(E, -BIG, BIG, B)


def _states(n, rng, e_lo, e_hi):
    k = rng.normal(size=(3, n)); k /= np.linalg.norm(k, axis=0)
    st = np.zeros((8, n))
    st[0:3] = rng.normal(size=(3, n)) * 1e-3
    st[3] = rng.uniform(0, 5, n)
    st[4] = rng.uniform(e_lo, e_hi, n)
    st[5:8] = k
    return st


def test_s9c_excitation_loss_is_the_selected_levels(oracle):
    """S9c / R11: an excitation removes exactly the loss of the SELECTED level.  Excitation-only gas with three levels of
    different losses, nu_hat = nu_tot (every step is real), no field (eps' = eps): eps'' = eps - loss[event].  A wrong
    level index (loss[l-1], loss[0]), a dropped subtraction or a sign error changes eps'' by >= 0.7 eV."""
    loss = np.array([1.0, 2.5, 0.3])
    g = gas.multi_level_constant([10.0, 30.0, 20.0], [gas.EXCITATION] * 3, loss=loss, nu_hat=60.0)
    rng = np.random.default_rng(101)
    n = 20000
    st = _states(n, rng, 3.0, 30.0)
    res = oracle.step_batch(g, _open_field((0, 0, 0)), 3, st, np.arange(n, dtype=np.uint64), np.full(n, 9, dtype=np.uint32))
    assert np.all(res.event >= 0) and all((res.event == l).sum() > 2000 for l in range(3))
    assert np.allclose(res.state[4], st[4] - loss[res.event], rtol=1e-14, atol=0)
    # the guard: a loss above the energy leaves the floor, not a negative energy (R6 keeps real tables away from it)
    st2 = st.copy(); st2[4] = rng.uniform(0.05, 0.25, n)
    r2 = oracle.step_batch(g, _open_field((0, 0, 0)), 3, st2, np.arange(n, dtype=np.uint64), np.full(n, 9, dtype=np.uint32))
    assert np.all(r2.state[4] == 1e-10)
    # the deflection is drawn and applied (isotropic): direction changes, |k| = 1
    assert np.abs(np.linalg.norm(res.state[5:8], axis=0) - 1).max() < 1e-14
    assert np.mean((res.state[5:8] * st[5:8]).sum(0)) < 0.05


def test_s6_bin_uses_the_energy_after_the_flight(oracle):
    """S6: the bin is that of eps' (after the flight), not of the energy the step started with.  Strong field, long
    flights: eps' leaves the starting bin for most states.  eps' is computed here from first principles — the generators'
    Philox for u1, dt = -ln(u1)/nu_hat, v' = v0 - kappa E dt — and the table is zero except in one bin, so `event >= 0`
    reveals the bin the oracle looked up."""
    nb, e_max, nu_hat = 50, 25.0, 10.0
    g = gas.multi_level_constant([nu_hat], [gas.ELASTIC], n_bins=nb, e_max=e_max, nu_hat=nu_hat)
    g.cum_rate[:] = 0.0
    g.cum_rate[7, :] = nu_hat                                         # bin 7 = [3.5, 4.0) eV: always real there, never elsewhere
    rng = np.random.default_rng(102)
    n = 40000
    st = _states(n, rng, 0.5, 8.0)
    E = np.array([300.0, -200.0, -900.0])
    ids = np.arange(n, dtype=np.uint64) + 77
    seed, nidx = 5, 4
    res = oracle.step_batch(g, _open_field(E), seed, st, ids, np.full(n, nidx, dtype=np.uint32))
    u1, _ = philox.uniform_pair(seed, ids, nidx, 0)
    dt = -np.log(u1) / nu_hat
    v1 = C2 * np.sqrt(st[4]) * st[5:8] + (-KAPPA * E)[:, None] * dt
    e1 = (v1 * v1).sum(0) / C2 ** 2
    b1 = np.minimum((e1 * nb / e_max).astype(int), nb - 1)
    b0 = np.minimum((st[4] * nb / e_max).astype(int), nb - 1)
    clear = np.abs(e1 * nb / e_max - np.round(e1 * nb / e_max)) > 1e-9   # away from a bin edge
    assert ((b0 == 7) != (b1 == 7)).sum() > 2000                      # the two readings differ on many states
    assert np.array_equal(res.bin[clear], b1[clear])
    assert np.array_equal((res.event >= 0)[clear], (b1 == 7)[clear])
    # and the work-energy identity gives the same eps' from the oracle's own displacement (C4): eps' = eps - E . dr
    null = res.event == -1
    e1_we = st[4] - (E[:, None] * (res.state[0:3] - st[0:3])).sum(0)
    assert np.allclose(res.state[4][null], e1_we[null], rtol=1e-10)
    assert np.allclose(res.state[4][null], e1[null], rtol=1e-12)


def test_s6_overflow_is_counted_for_steps_that_reach_the_decision(oracle):
    """S6 / R5: energies >= e_max use the last bin and are counted — once per step that passes S5, not for the electron's
    last flight.  (i) Closed form: no field, recoil-free elastic gas (energies never change), time cut: the count is
    sum over electrons with eps >= e_max of (n_steps - 1).  (ii) Strong field: the count of the run equals the count from
    replaying the same electrons step by step (a step reaches the decision iff its status stays 0; eps_out = eps' since
    nothing removes energy) — in a gap whose planes also end electrons above e_max."""
    e_max = 5.0
    g = gas.constant_elastic(40.0, 0.0, n_bins=100, e_max=e_max, nu_hat=100.0)
    L = 1
    p = primaries.isotropic_primaries(400, 7, e_scale=10.0)
    p[:, 4] = np.where(np.abs(p[:, 4] - e_max) < 1e-6, 1.0, p[:, 4])
    r = oracle.run(g, _open_field((0, 0, 0)), p, seed=7, t_max=0.5)
    assert np.all(r.status == 6)
    hot = r.birth[4] >= e_max
    assert hot.sum() > 100 and (~hot).sum() > 100
    assert int(r.tallies_u64[L + 2]) == int((r.n_steps[hot].astype(np.int64) - 1).sum())
    # (ii) field + absorbing planes
    g = gas.constant_elastic(4000.0, 0.0, n_bins=100, e_max=e_max, nu_hat=10000.0)
    fd = fields.uniform_gap((0.0, 0.0, -200000.0), 0.0, 3e-4)
    p = primaries.isotropic_primaries(60, 8, pos=(0, 0, 1e-4), e_scale=3.0)
    r = oracle.run(g, fd, p, seed=8)
    assert set(np.unique(r.status)) <= {1, 2} and (r.end[4] > e_max).sum() > 20   # electrons leave the gap above e_max
    count = 0
    for i in range(60):
        st = p[i].copy()[:, None]
        for n in range(100000):
            s = oracle.step_batch(g, fd, 8, st, np.array([i], dtype=np.uint64), np.array([n], dtype=np.uint32))
            if s.status[0] != 0:
                assert s.bin[0] == -1                                  # the last flight never reaches S6
                break
            assert (s.bin[0] == 99) == (s.state[4, 0] >= e_max * 99 / 100)
            count += int(s.state[4, 0] >= e_max)
            st = s.state
    assert count > 200 and int(r.tallies_u64[L + 2]) == count


def test_energy_ledger_of_whole_avalanches_g0(oracle, g0):
    """Every eV is accounted for, with the level TALLIES as the only record of the losses: gas G0 with recoil 0,
    (sum of all endpoint energies) - (sum of the primaries' energies) = -E . sum(dr) - sum_l N_l loss_l, dr summed over
    every electron's birth-to-end displacement (an ionisation hands eps_s from the parent to the child: it moves energy,
    it removes only the threshold).  A loss taken from the wrong level, a child born with the wrong energy, a primary that keeps the secondary's share
    or a flight that does not conserve energy breaks it."""
    g = dataclasses.replace(g0, level_recoil=np.zeros(g0.n_levels))
    E0 = 60000.0
    fd = fields.uniform_gap((0.0, 0.0, -E0), 0.0, 70e-4)
    p = primaries.isotropic_primaries(40, 9, forward=True); p[:, 2] = 2e-4
    r = oracle.run(g, fd, p, seed=9, capacity=1 << 18, n_threads=4)
    t = r.tallies_u64
    assert r.n > 2000 and int(t[14] + t[15]) == r.n - 40 and sum(int(t[l]) for l in range(2, 14)) > 10000
    gained = E0 * (r.end[2] - r.birth[2]).sum()                       # -E . dr with E = (0, 0, -E0)
    lost = float(sum(int(t[l]) * g.level_loss[l] for l in range(g.n_levels)))
    prim = r.id < 40
    assert prim.sum() == 40
    de = r.end[4].sum() - r.birth[4][prim].sum()
    assert abs(de - (gained - lost)) < 1e-9 * lost, (de, gained, lost)
    # the same ledger with the oracle's own loss sum (tallies_f64[4]) — consistency of the two records
    assert abs(r.tallies_f64[4] - lost) < 1e-9 * lost


# ---- C17 ---------------------------------------------------------------------------------------------------------
def _mixed_gas():
    """All four level types at comparable rates, energy dependent, so that 100 steps meet every branch of S7-S9."""
    nb, e_max = 64, 64.0
    e = (np.arange(nb) + 0.5) * e_max / nb
    rates = np.stack([20.0 + 0.0 * e, 8.0 * (e > 2.0), 6.0 * np.sqrt(e), 25.0 * (e > 12.0), 1.5 + 0.0 * e, 5.0 * (e > 6.0)], axis=1)
    types = [gas.ELASTIC, gas.EXCITATION, gas.ELASTIC, gas.IONISATION, gas.ATTACHMENT, gas.EXCITATION]
    return gas._finish(nb, e_max, rates, types, [0, 2.0, 0, 12.0, 0, 6.0], [1e-3, 0, 0.3, 0, 0, 0], [0, 0, 0, 7.0, 0, 0],
                       [f"l{i}" for i in range(6)], nu_hat=140.0)


def _small_stack(rng, B):
    """A non-uniform 9 x 8 x 12 map (mirror in x, periodic in y, a block of material) between two uniform slabs."""
    nz, ny, nx = 12, 8, 9
    nodes = (rng.normal(size=(nz, ny, nx, 4)) * 3e4).astype(np.float32)
    nodes[..., 2] -= 6e4
    nodes[..., 3] = 1.0
    nodes[4:6, 2:5, 3:6, 3] = 0.0
    h = (1e-4, 1.25e-4, 1e-4)
    g1 = fields.grid_slab(nodes, (-1e-4, 0.5e-4, 0.0), h, 0.0, 11e-4, fields.BC_MIRROR, fields.BC_PERIODIC, 7e-4, 7 * 1.25e-4)
    u0 = fields.Slab(-6e-4, 0.0, fields.KIND_UNIFORM, (500.0, -300.0, -40000.0))
    u2 = fields.Slab(11e-4, 16e-4, fields.KIND_UNIFORM, (0.0, 0.0, -50000.0))
    return fields.FieldDesc([u0, g1, u2], B, (-30e-4, -40e-4), (30e-4, 40e-4))


def _assert_step_equals_transcription(res, i, ref, st_in, rtol=1e-13):
    got = res.state[:, i]
    want = np.array([float(v) for v in ref["state"]])
    assert res.event[i] == ref["event"] and res.status[i] == ref["status"] and res.bin[i] == ref["bin"], \
        (res.event[i], ref["event"], res.status[i], ref["status"], res.bin[i], ref["bin"])
    dr = np.linalg.norm(want[0:3] - st_in[0:3])
    for c in range(3):
        assert abs(got[c] - want[c]) <= rtol * max(abs(st_in[c]), abs(want[c]), dr), (c, got[c], want[c])
    assert abs(got[3] - want[3]) <= rtol * max(abs(want[3]), abs(st_in[3]))
    e_scale = max(st_in[4], want[4]) + (20.0 + float(ref["child"][4]) if ref["child"] is not None else 0.0)
    assert abs(got[4] - want[4]) <= rtol * e_scale, (got[4], want[4])
    assert np.abs(got[5:8] - want[5:8]).max() <= rtol, (got[5:8], want[5:8])
    if ref["child"] is not None:
        ch = np.array([float(v) for v in ref["child"]])
        assert int(res.child_id[i]) == ref["child_id"]
        assert np.abs(res.child[0:4, i] - ch[0:4]).max() <= rtol * max(np.abs(ch[0:4]).max(), dr)
        assert abs(res.child[4, i] - ch[4]) <= rtol * e_scale and np.abs(res.child[5:8, i] - ch[5:8]).max() <= rtol
    else:
        assert res.child_id[i] == 0 and not res.child[:, i].any()


@pytest.mark.parametrize("case", ["g0_grid", "mixed_grid_B", "mixed_uniform_B", "g0_uniform"])
def test_c17_independent_transcription(oracle, g0, case):
    """C17: 10 electrons x 100 steps.  Each step is taken twice from the same fp64 state — by the oracle and by the
    40-digit transcription — and every output must agree: event, status, bin, child id exactly, continuous outputs to
    1e-13 in the sense of tolerance T.  The electron then goes on from the oracle's state (a finished electron is replaced
    by its child or restarted), so the 1000 steps cover the states a real history visits: null and real collisions of
    every type, slab changes, mirror and periodic folds, material and boundary endings, with and without B."""
    import transcription_s0_s9 as T17
    rng = np.random.default_rng({"g0_grid": 1, "mixed_grid_B": 2, "mixed_uniform_B": 3, "g0_uniform": 4}[case])
    B = (0.3, -0.5, 0.8) if case.endswith("_B") else (0.0, 0.0, 0.0)
    g = g0 if case.startswith("g0") else _mixed_gas()
    fd = _small_stack(rng, B) if "grid" in case else fields.uniform_gap((2000.0, -1000.0, -70000.0), 0.0, 4e-4, B)
    seed, t_max = 1234567 + len(case), 0.02
    z_top = fd.slabs[-1].z_hi

    def fresh(j):
        k = rng.normal(size=3); k /= np.linalg.norm(k)
        z = rng.uniform(0.15, 0.85) * z_top
        return np.array([rng.uniform(-2e-4, 2e-4), rng.uniform(-2e-4, 2e-4), z, 0.0, rng.uniform(0.5, 30.0), *k])

    seen_events, seen_status, n_children = set(), set(), 0
    for el in range(10):
        ident, n, st = 1000 + el, 0, fresh(el)
        pending = []                                                    # children wait for their parent to finish
        for _ in range(100):
            res = oracle.step_batch(g, fd, seed, st[:, None], np.array([ident], dtype=np.uint64), np.array([n], dtype=np.uint32), t_max=t_max)
            ref = T17.step(g, fd, seed, t_max, st, ident, n)
            if res.event[0] == -2 and res.status[0] in (1, 2, 3, 4) and ref["status"] == 0:
                pytest.fail("oracle left the domain where the transcription did not")
            _assert_step_equals_transcription(res, 0, ref, st)
            seen_events.add(int(res.event[0])); seen_status.add(int(res.status[0]))
            if ref["child"] is not None:
                pending.append((int(res.child_id[0]), res.child[:, 0].copy())); n_children += 1
            if res.status[0] == 0:
                st, n = res.state[:, 0].copy(), n + 1
            elif pending:
                (ident, st), n = pending.pop(), 0
            else:
                ident, n, st = ident + 100, 0, fresh(el)
    assert -1 in seen_events and 0 in seen_events and 0 in seen_status
    if case.startswith("mixed"):
        assert seen_events >= {-1, 0, 1, 2, 3, 4, 5} and 5 in seen_status and n_children >= 3
    if "grid" in case:
        assert seen_status & {1, 2, 3, 4}
