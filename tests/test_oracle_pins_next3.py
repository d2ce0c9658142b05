"""Oracle pins of NEXT-3 (DESIGN.md §3.6 readings X1-X3), CPU only: anisotropic scattering (X1),
Penning transfer (X2), gas thermal motion (X3).  Each is pinned to closed forms / invariants that a plausible mistake in
oracle/avmo.cpp (wrong table index, a dropped factor, a wrong sign) breaks; the extensions switched off reproduce the base
model bit for bit."""
import copy

import numpy as np
import pytest
from scipy import stats

from paper_2509_15377_b200.gen import fields, gas, primaries

KAPPA = 0.0017588200107589609
C2 = 0.05930969584745753
BIG = 1.0e6


def _open_field(E, B=(0, 0, 0)):
    return fields.uniform_gap(E, -BIG, BIG, B)


def _states(n, rng, e_lo=0.1, e_hi=20.0):
    k = rng.normal(size=(3, n)); k /= np.linalg.norm(k, axis=0)
    st = np.zeros((8, n))
    st[0:3] = rng.normal(size=(3, n)) * 1e-3
    st[3] = rng.uniform(0, 5, n)
    st[4] = rng.uniform(e_lo, e_hi, n)
    st[5:8] = k
    return st


def mean_cos(xi):
    """<cos theta> of cos theta = (c0 + xi) / (1 + xi c0), c0 uniform in (-1, 1): 1/xi - (1 - xi^2) / (2 xi^2) ln((1+xi)/(1-xi))."""
    return 1.0 / xi - (1.0 - xi * xi) / (2.0 * xi * xi) * np.log((1.0 + xi) / (1.0 - xi))


def test_mean_cos_closed_form_against_quadrature():
    from scipy.integrate import quad
    for xi in (-0.7, 0.2, 0.9):
        num = quad(lambda c: 0.5 * (c + xi) / (1 + xi * c), -1, 1)[0]
        assert abs(num - mean_cos(xi)) < 1e-10


# ---- X1 ---------------------------------------------------------------------------------------------------------------
def test_x1_deflection_distribution_and_table_indexing(oracle):
    """cos theta between k' and k'' follows the transformed-uniform law of the (bin, level) entry: the inverse transform
    c0 = (ct - xi) / (1 - xi ct) is uniform in (-1, 1) (KS), <cos theta> is the closed form, the azimuth stays uniform,
    |k''| = 1; xi differs by level AND by energy bin, so a transposed or shifted table index fails."""
    nb = 32
    g = gas.multi_level_constant([60.0, 40.0], [gas.ELASTIC, gas.EXCITATION], loss=[0.0, 0.5], recoil=[0.0, 0.0], n_bins=nb, e_max=32.0)
    xi = np.zeros((nb, 2))
    xi[:16, 0], xi[16:, 0], xi[:16, 1], xi[16:, 1] = 0.8, -0.5, 0.3, 0.95
    g.scat_xi = xi
    rng = np.random.default_rng(1)
    n = 80000
    st = _states(n, rng, e_lo=1.0, e_hi=31.0)
    st[4] = np.where(rng.uniform(size=n) < 0.5, rng.uniform(1.0, 15.5, n), rng.uniform(17.0, 31.0, n))
    res = oracle.step_batch(g, _open_field((0, 0, 0)), 3, st, np.arange(n, dtype=np.uint64), np.full(n, 2, dtype=np.uint32))
    assert np.all(res.event >= 0)
    ct = (st[5:8] * res.state[5:8]).sum(0)                           # E = 0: k' = k
    assert np.allclose(np.linalg.norm(res.state[5:8], axis=0), 1.0, atol=1e-14)
    for lvl in (0, 1):
        for lo, hi, x in ((0.0, 16.0, xi[0, lvl]), (16.0, 32.0, xi[20, lvl])):
            sel = (res.event == lvl) & (st[4] >= lo) & (st[4] < hi)
            assert sel.sum() > 5000
            c0 = (ct[sel] - x) / (1.0 - x * ct[sel])
            assert stats.kstest(c0, stats.uniform(-1, 2).cdf).pvalue > 1e-3, (lvl, lo)
            assert abs(ct[sel].mean() - mean_cos(x)) < 4 * ct[sel].std() / np.sqrt(sel.sum())
    # azimuth about k' is uniform: angle of the perpendicular part of k'' in a fixed basis about k'
    k1, k2 = st[5:8], res.state[5:8]
    perp = k2 - ct * k1
    a = np.cross(k1.T, np.array([0.3, -0.5, 0.81])).T; a /= np.linalg.norm(a, axis=0)
    b = np.cross(k1.T, a.T).T
    phi = np.arctan2((perp * b).sum(0), (perp * a).sum(0))
    assert stats.kstest((phi + np.pi) / (2 * np.pi), "uniform").pvalue > 1e-3
    # the excitation still loses its threshold; the loss-free elastic level keeps the energy
    assert np.allclose(res.state[4][res.event == 1], st[4][res.event == 1] - 0.5, rtol=1e-13)
    assert np.allclose(res.state[4][res.event == 0], st[4][res.event == 0], rtol=1e-13)


def test_x1_xi_zero_is_the_isotropic_model_bit_for_bit(oracle, g0):
    rng = np.random.default_rng(2)
    n = 20000
    st = _states(n, rng, e_hi=39.0)
    ids = rng.integers(0, 2 ** 63, n, dtype=np.int64).astype(np.uint64); nidx = np.zeros(n, dtype=np.uint32)
    f = _open_field((0, 0, -30000.0))
    a = oracle.step_batch(g0, f, 5, st, ids, nidx)
    g = copy.copy(g0); g.scat_xi = np.zeros((g0.n_bins, g0.n_levels))
    b = oracle.step_batch(g, f, 5, st, ids, nidx)
    assert np.array_equal(a.state, b.state) and np.array_equal(a.event, b.event) and np.array_equal(a.child, b.child)


def test_x1_recoil_loss_and_drift_velocity_with_forward_scattering(oracle):
    """Elastic loss follows the ACTUAL deflection: <1 - eps''/eps'> = r (1 - <cos theta>).  Constant collision frequency:
    the momentum balance d<v>/dt = a - nu (1 - <cos theta>) <v> gives W = -(KAPPA / (nu (1 - <cos theta>))) E."""
    x, nu, rec = 0.6, 400.0, 0.02
    g = gas.constant_elastic(nu, rec)
    g.scat_xi = np.full((g.n_bins, 1), x)
    rng = np.random.default_rng(3)
    n = 60000
    st = _states(n, rng)
    res = oracle.step_batch(g, _open_field((0, 0, 0)), 9, st, np.arange(n, dtype=np.uint64), np.full(n, 5, dtype=np.uint32))
    ct = (st[5:8] * res.state[5:8]).sum(0)
    assert np.allclose(res.state[4], st[4] * (1.0 - rec * (1.0 - ct)), rtol=1e-12)
    frac = 1.0 - res.state[4] / st[4]
    assert abs(frac.mean() - rec * (1.0 - mean_cos(x))) < 4 * frac.std() / np.sqrt(n)
    E = np.array([0.0, 0.0, -2000.0])
    p = primaries.isotropic_primaries(1500, 31, e_scale=1.0)
    r = oracle.run(g, _open_field(E), p, seed=31, t_max=4.0, n_threads=8)
    v = (r.end[0:3] - r.birth[0:3]) / (r.end[3] - r.birth[3])
    W, se = v.mean(1), v.std(1, ddof=1) / np.sqrt(1500)
    W_exact = -(KAPPA / (nu * (1.0 - mean_cos(x)))) * E
    # the first 1/(nu_m) of the 4 ns is the approach to the steady state: < 0.2 %
    assert abs(W[2] - W_exact[2]) < 4 * se[2] + 0.003 * abs(W_exact[2]), (W, W_exact, se)
    assert se[2] < 0.01 * abs(W_exact[2])
    W_iso = -(KAPPA / nu) * E
    assert abs(W[2] - W_iso[2]) > 20 * se[2]                        # and it is NOT the isotropic value


# ---- X2 ---------------------------------------------------------------------------------------------------------------
def _penning_gas(p, e_pen, nu=100.0, loss=11.5, nu_hat=0.0):
    g = gas.multi_level_constant([nu], [gas.EXCITATION], loss=[loss], n_bins=16, e_max=100.0, nu_hat=nu_hat)
    g.level_penning_prob = np.array([p]); g.level_penning_eV = np.array([e_pen])
    return g


def test_x2_transfer_probability_energy_and_direction(oracle):
    p, e_pen = 0.37, 4.2
    g = _penning_gas(p, e_pen)
    rng = np.random.default_rng(4)
    n = 60000
    st = _states(n, rng, e_lo=20.0, e_hi=60.0)
    res = oracle.step_batch(g, _open_field((0, 0, -3000.0)), 11, st, np.arange(n, dtype=np.uint64), np.full(n, 1, dtype=np.uint32))
    assert np.all(res.event == 0)
    has = res.child_id != 0
    assert abs(has.mean() - p) < 4 * np.sqrt(p * (1 - p) / n)
    ce = res.child[4][has]
    assert ce.min() > 0 and ce.max() < e_pen and stats.kstest(ce / e_pen, "uniform").pvalue > 1e-3
    assert np.array_equal(res.child[0:4][:, has], res.state[0:4][:, has])            # born where and when the parent is
    assert np.all(res.child[:, ~has] == 0)
    k = res.child[5:8][:, has]
    assert np.allclose(np.linalg.norm(k, axis=0), 1.0, atol=1e-14)
    assert stats.kstest(k[2], stats.uniform(-1, 2).cdf).pvalue > 1e-3
    assert stats.kstest((np.arctan2(k[1], k[0]) + np.pi) / (2 * np.pi), "uniform").pvalue > 1e-3
    # the exciting electron loses the threshold whether or not the transfer happens (work-energy: eps' = eps - E . dr)
    e_after_flight = st[4] + 3000.0 * (res.state[2] - st[2])
    assert np.allclose(res.state[4], np.maximum(e_after_flight - 11.5, 1e-10), rtol=1e-12, atol=1e-11)   # R11: floored
    # the uniform that decides the transfer is independent of the one that sets the energy and of the direction's
    assert abs(np.corrcoef(ce, k[2])[0, 1]) < 0.02


def test_x2_no_transfer_when_probability_zero_or_absent(oracle):
    rng = np.random.default_rng(5)
    n = 5000
    st = _states(n, rng, e_lo=20.0, e_hi=60.0)
    ids = np.arange(n, dtype=np.uint64); nidx = np.zeros(n, dtype=np.uint32)
    base = gas.multi_level_constant([100.0], [gas.EXCITATION], loss=[11.5], n_bins=16, e_max=100.0)
    a = oracle.step_batch(base, _open_field((0, 0, -3000.0)), 1, st, ids, nidx)
    b = oracle.step_batch(_penning_gas(0.0, 4.0), _open_field((0, 0, -3000.0)), 1, st, ids, nidx)
    c = oracle.step_batch(_penning_gas(1.0, 4.0), _open_field((0, 0, -3000.0)), 1, st, ids, nidx)
    assert np.array_equal(a.state, b.state) and np.all(b.child_id == 0)
    assert np.array_equal(a.state, c.state) and np.all(c.child_id != 0)               # the parent's step is the same


def test_x2_charge_conservation_and_yule_furry(oracle):
    """Every transfer creates one electron: electrons = primaries + ionisations + transfers, per avalanche too.  With p = 1
    and no loss an excitation-only gas multiplies exactly like the ionisation-only gas of C13: Yule-Furry."""
    nu, t_max, n_p = 5.0, 0.4, 5000
    g = _penning_gas(1.0, 2.0, nu=nu, loss=0.0, nu_hat=12.0)
    pr = primaries.isotropic_primaries(n_p, 44, e_scale=50.0)
    r = oracle.run(g, _open_field((0, 0, 0)), pr, seed=44, t_max=t_max, capacity=1 << 18)
    L = 1
    assert int(r.tallies_u64[L + 4]) == r.n - n_p == int(r.tallies_u64[0])
    assert np.array_equal(r.per_avalanche[:, 0], np.bincount(r.avalanche, minlength=n_p).astype(np.uint64))
    size = r.per_avalanche[:, 0].astype(np.int64)
    nbar = np.exp(nu * t_max)
    assert abs(size.mean() - nbar) < 4 * np.sqrt(nbar * (nbar - 1) / n_p)
    q = 1 - 1 / nbar
    edges = np.array([1, 2, 3, 4, 5, 6, 8, 10, 13, 17, 22, 30, 10 ** 9])
    obs = np.histogram(size, bins=edges)[0]
    exp = n_p * (q ** (edges[:-1] - 1) - q ** (edges[1:] - 1))
    assert stats.chisquare(obs, exp * obs.sum() / exp.sum()).pvalue > 1e-3
    # p = 0.25: a quarter of the excitations transfer
    g = _penning_gas(0.25, 2.0, nu=nu, loss=0.0, nu_hat=12.0)
    r = oracle.run(g, _open_field((0, 0, 0)), pr, seed=45, t_max=t_max, capacity=1 << 18)
    n_exc, n_pen = int(r.tallies_u64[0]), int(r.tallies_u64[L + 4])
    assert n_pen == r.n - n_p and abs(n_pen / n_exc - 0.25) < 4 * np.sqrt(0.25 * 0.75 / n_exc)


def test_x2_on_g0_with_ionisation_levels(oracle, g0):
    """Gas G0 with Penning transfer on three Ar-like excitation levels: the count still balances with the ionisation and
    attachment levels present, and the gain rises."""
    g = copy.copy(g0)
    pp = np.zeros(g0.n_levels); pe = np.zeros(g0.n_levels)
    exc = np.flatnonzero(g0.level_type == gas.EXCITATION)
    pp[exc[-3:]] = 0.4
    pe[exc[-3:]] = np.maximum(g0.level_loss[exc[-3:]] - 13.8, 0.05)                   # excitation energy - CO2 ionisation potential
    g.level_penning_prob, g.level_penning_eV = pp, pe
    f = fields.uniform_gap((0, 0, -60000.0), 0.0, 60e-4)
    pr = primaries.isotropic_primaries(200, 7, forward=True)
    a = oracle.run(g0, f, pr, seed=7, capacity=1 << 20, n_threads=8)
    b = oracle.run(g, f, pr, seed=7, capacity=1 << 20, n_threads=8)
    L = g0.n_levels
    ion = lambda r: int(sum(r.tallies_u64[l] for l in range(L) if g0.level_type[l] == gas.IONISATION))
    assert int(a.tallies_u64[L + 4]) == 0 and a.n == 200 + ion(a)
    assert int(b.tallies_u64[L + 4]) > 100 and b.n == 200 + ion(b) + int(b.tallies_u64[L + 4])
    assert b.n > 1.1 * a.n


# ---- X3 ---------------------------------------------------------------------------------------------------------------
def thermal_mean(kT, rec):
    """Stationary <eps> of the X3 model at constant collision frequency without field.  Per collision, in energy units:
    <|w|^2> = eps' + 3 s (s = kT r / 4 per component), <|w''|^2> = (1 - r) <|w|^2>, and eps'' = <|w''|^2> + 3 s + 2 <w'' . V> with
    <w'' | w> = m1 w, m1 = <c sqrt(1 - r (1 - c))> over c uniform in (-1, 1) (the deflected speed is correlated with the
    angle), <w . V> = -3 s: eps'' = (1 - r)(eps' + 3 s) + 3 s - 6 m1 s.  Fixed point: (3/2) kT [(1 - r/2) - m1] = 3/2 kT to
    O(m/M) (m1 = r/6 + O(r^2))."""
    from scipy.integrate import quad
    m1 = quad(lambda c: 0.5 * c * np.sqrt(1.0 - rec * (1.0 - c)), -1, 1)[0]
    return 1.5 * kT * ((1.0 - rec / 2) - m1)


def test_x3_thermal_equilibrium(oracle):
    """No field, constant elastic collision frequency: whatever the start energy, the ensemble relaxes to the gas
    temperature: <eps> = thermal_mean (3/2 kT to O(m/M); 250000 electrons resolve the O(r) terms to 4 SE: the mean without
    the m1 term is 5 SE away), and the stationary law of eps is close to the Maxwellian's Gamma(3/2)."""
    nu, rec, kT = 400.0, 0.04, 0.02526
    g = gas.constant_elastic(nu, rec, n_bins=64, e_max=10.0)
    g.kT_eV = kT
    exact = thermal_mean(kT, rec)
    assert abs(exact / (1.5 * kT * (1 - 2 * rec / 3)) - 1) < 1e-3
    for e0, seed, n_el in ((1.0, 61, 250000), (1e-4, 62, 6000)):
        p = primaries.isotropic_primaries(n_el, seed, e_scale=1.0)
        p[:, 4] = e0
        r = oracle.run(g, _open_field((0, 0, 0)), p, seed=seed, t_max=1.2, n_threads=8, capacity=n_el)   # nu r t = 19 relaxation times
        e = r.end[4]
        se = e.std(ddof=1) / np.sqrt(len(e))
        assert abs(e.mean() - exact) < 4 * se, (e.mean(), exact)
        if n_el > 100000:
            assert abs(e.mean() - 1.5 * kT * (1 - rec / 2)) > 3 * se       # the test does resolve the m1 term
        assert abs(e.mean() / (1.5 * kT) - 1) < 0.05
        assert stats.kstest(e[:6000] / (exact / 1.5), stats.gamma(1.5).cdf).pvalue > 1e-3
    # cold gas (kT = 0) loses everything instead
    g.kT_eV = 0.0
    p = primaries.isotropic_primaries(500, 63, e_scale=1.0)
    r = oracle.run(g, _open_field((0, 0, 0)), p, seed=63, t_max=1.2, n_threads=8)
    assert r.end[4].mean() < 1e-3 * kT * 1.5 + 1e-6


def test_x3_energy_balance_in_a_field_and_drift_unchanged(oracle):
    """With a field: W = -(KAPPA / nu) E as in the cold gas (the atom's mean velocity is zero), and the mean energy is the
    cold-gas value of C6 plus the thermal term: <eps> = (a . W) / (KAPPA nu r) + thermal_mean(kT, r)."""
    nu, rec, kT = 400.0, 0.02, 0.05
    E = np.array([0.0, 0.0, -300.0])
    g = gas.constant_elastic(nu, rec)
    g.kT_eV = kT
    p = primaries.isotropic_primaries(3000, 71, e_scale=0.2)
    r = oracle.run(g, _open_field(E), p, seed=71, t_max=4.0, n_threads=8)
    v = (r.end[0:3] - r.birth[0:3]) / (r.end[3] - r.birth[3])
    W, se = v.mean(1), v.std(1, ddof=1) / np.sqrt(3000)
    W_exact = -(KAPPA / nu) * E
    assert np.all(np.abs(W - W_exact) < 4 * se + 1e-12), (W, W_exact, se)
    cold = (-(KAPPA * E) @ W_exact) / (KAPPA * nu * rec)
    exact = cold + thermal_mean(kT, rec)
    e = r.end[4]
    assert abs(e.mean() - exact) < 4 * e.std(ddof=1) / np.sqrt(len(e)), (e.mean(), exact, cold)
    assert 0.75 * kT * (2.0 - rec) > 8 * e.std(ddof=1) / np.sqrt(len(e))                # the thermal term is resolved


def test_x3_one_collision_kinematics(oracle):
    """One thermal collision, checked from the outside: with V recovered from the step's own uniforms (blocks 2 and 3,
    Box-Muller, sigma = c2 sqrt(kT r / 4)), |v'' - V|^2 = |v' - V|^2 (1 - r (1 - cos theta_rel)), theta_rel the angle
    between the relative velocities before and after."""
    nu, rec, kT = 100.0, 0.3, 2.0                                   # heavy recoil, hot gas: every term matters
    g = gas.constant_elastic(nu, rec)
    g.kT_eV = kT
    rng = np.random.default_rng(8)
    n = 4000
    st = _states(n, rng, e_lo=0.05, e_hi=5.0)
    ids = np.arange(n, dtype=np.uint64) + 77; nidx = np.full(n, 9, dtype=np.uint32)
    res = oracle.step_batch(g, _open_field((0, 0, 0)), 13, st, ids, nidx)
    assert np.all(res.event == 0)
    u = np.array([list(oracle.uniform_pair(13, int(i), 9, 2)) + list(oracle.uniform_pair(13, int(i), 9, 3)) for i in ids]).T
    sig = C2 * np.sqrt(kT * rec / 4)
    V = sig * np.array([np.sqrt(-2 * np.log(u[0])) * np.cos(2 * np.pi * u[1]), np.sqrt(-2 * np.log(u[0])) * np.sin(2 * np.pi * u[1]),
                        np.sqrt(-2 * np.log(u[2])) * np.cos(2 * np.pi * u[3])])
    v1 = C2 * np.sqrt(st[4]) * st[5:8]                                # E = 0: the flight leaves v alone
    v2 = C2 * np.sqrt(res.state[4]) * res.state[5:8]
    w1, w2 = v1 - V, v2 - V
    ct = (w1 * w2).sum(0) / np.sqrt((w1 ** 2).sum(0) * (w2 ** 2).sum(0))
    assert np.allclose((w2 ** 2).sum(0), (w1 ** 2).sum(0) * (1 - rec * (1 - ct)), rtol=1e-10)
    assert stats.kstest(ct, stats.uniform(-1, 2).cdf).pvalue > 1e-3   # isotropic in the atom's frame
    # V has the stated variance and no mean
    assert stats.kstest(V.ravel() / sig, "norm").pvalue > 1e-3
