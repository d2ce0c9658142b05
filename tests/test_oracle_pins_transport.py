"""Oracle pins, part 2: free flight, kinematics, collision outcomes, bookkeeping (CPU only).

Closed forms and invariants that a plausible mistake in oracle/avmo.cpp (dropped term, wrong sign or index,
transposed operand) would break.  Pin ids follow SURVEY.md §8(c) / DESIGN.md §5.
"""
import numpy as np
import pytest
from scipy import stats
from scipy.integrate import solve_ivp

from paper_2509_15377_b200.gen import fields, gas, primaries

KAPPA = 0.0017588200107589609      # cm/ns^2 per V/cm  (c^2 / mc^2)
OMEGA1 = 175.88200107589608        # rad/ns/T
C2 = 0.05930969584745753           # cm/ns/sqrt(eV)
INF = float("inf")
BIG = 1.0e6                         # cm: "unbounded" gap


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


def test_c2_free_flight_is_exponential(oracle):
    """C2: dt * nu_hat ~ Exp(1) (null-collision free flight), and dt = -log(u1)/nu_hat with u1 from block 0."""
    g = gas.constant_elastic(50.0, 0.0, nu_hat=200.0)
    rng = np.random.default_rng(10)
    n = 20000
    st = _states(n, rng)
    ids = np.arange(n, dtype=np.uint64) + 1000
    res = oracle.step_batch(g, _open_field((0, 0, 0)), 7, st, ids, np.full(n, 3, dtype=np.uint32))
    dt = res.state[3] - st[3]
    assert stats.kstest(dt * 200.0, "expon").pvalue > 1e-3
    u1 = np.array([oracle.uniform_pair(7, int(i), 3, 0)[0] for i in ids[:200]])
    assert np.allclose(dt[:200], -np.log(u1) / 200.0, rtol=1e-12, atol=1e-15)   # t_in <= 5 limits the relative check
    # real fraction = nu / nu_hat
    frac = np.mean(res.event >= 0)
    assert abs(frac - 0.25) < 4 * np.sqrt(0.25 * 0.75 / n)


@pytest.mark.parametrize("B", [(0.0, 0.0, 0.0), (0.3, -0.4, 0.8), (0.0, 1.5, 0.0)])
def test_flight_matches_lorentz_ode(oracle, B):
    """S3 against the equation of motion itself: m dv/dt = q (E + v x B), q = -e, integrated numerically.
    In our units dv/dt = -KAPPA E - OMEGA1 (v x B).  Pins the sign of the acceleration, the sense of the
    gyration, the E x B drift and the position integral of the helix."""
    g = gas.constant_elastic(1.0, 0.0, nu_hat=30.0)                # few collisions: long flights (theta up to ~ 30 rad)
    rng = np.random.default_rng(11)
    n = 40
    st = _states(n, rng)
    E = np.array([1500.0, -700.0, 2500.0])
    res = oracle.step_batch(g, _open_field(E, B), 3, st, np.arange(n, dtype=np.uint64), np.zeros(n, dtype=np.uint32))
    Bv = np.array(B)

    def rhs(t, y):
        v = y[3:]
        return np.concatenate([v, -KAPPA * E - OMEGA1 * np.cross(v, Bv)])

    for i in range(n):
        if res.event[i] != -1:
            continue                                                 # compare pure flights (null collisions)
        dt = res.state[3, i] - st[3, i]
        v0 = C2 * np.sqrt(st[4, i]) * st[5:8, i]
        sol = solve_ivp(rhs, (0, dt), np.concatenate([st[0:3, i], v0]), rtol=1e-12, atol=1e-16, method="DOP853")
        r1, v1 = sol.y[:3, -1], sol.y[3:, -1]
        dr = np.linalg.norm(r1 - st[0:3, i])
        assert np.linalg.norm(res.state[0:3, i] - r1) < 1e-9 * max(dr, 1e-6)
        e1 = v1 @ v1 / C2 ** 2
        assert abs(res.state[4, i] - e1) < 1e-9 * e1
        assert np.linalg.norm(res.state[5:8, i] - v1 / np.linalg.norm(v1)) < 1e-9


@pytest.mark.parametrize("B", [(0.0, 0.0, 0.0), (0.0, 0.5, 0.8660254037844387)])
def test_c4_work_energy_per_electron(oracle, B):
    """C4: with loss-free collisions, every electron obeys eps_end - eps_birth = -E . (r_end - r_birth) exactly
    (the magnetic force does no work), whatever the number of flights and deflections in between."""
    g = gas.constant_elastic(300.0, 0.0, nu_hat=700.0)
    E = (200.0, -300.0, -1000.0)
    p = primaries.isotropic_primaries(200, 5, e_scale=3.0)
    r = oracle.run(g, _open_field(E, B), p, seed=5, t_max=2.0)
    assert np.all(r.status == 6)
    de = r.end[4] - r.birth[4]
    work = -(np.array(E)[:, None] * (r.end[0:3] - r.birth[0:3])).sum(0)
    assert np.abs(de - work).max() < 1e-10 * np.maximum(np.abs(work), r.end[4]).max()
    # and summed over the run with the tallies: sum(eps_end - eps_birth) = -E . sum(dr) - sum(loss)
    tot = -(np.array(E) * r.tallies_f64[0:3]).sum() - r.tallies_f64[4]
    assert abs(de.sum() - tot) < 1e-9 * abs(tot)
    # the per-flight sums telescope to the endpoints
    assert np.allclose(r.tallies_f64[0:3], (r.end[0:3] - r.birth[0:3]).sum(1), rtol=1e-9, atol=1e-12)
    assert np.isclose(r.tallies_f64[3], (r.end[3] - r.birth[3]).sum(), rtol=1e-12)


def _drift_run(oracle, nu, recoil, E, B, nu_hat, n_el, t_max, seed):
    g = gas.constant_elastic(nu, recoil, nu_hat=nu_hat)
    p = primaries.isotropic_primaries(n_el, seed, e_scale=1.0)
    r = oracle.run(g, _open_field(E, B), p, seed=seed, t_max=t_max, n_threads=8)
    # per-electron mean velocity -> ensemble mean and standard error
    v = (r.end[0:3] - r.birth[0:3]) / (r.end[3] - r.birth[3])
    return r, v.mean(1), v.std(1, ddof=1) / np.sqrt(n_el)


def test_c5_c6_drift_velocity_and_mean_energy_constant_nu(oracle):
    """C5: constant collision frequency + isotropic scattering => W = -(KAPPA/nu) E exactly (= eE/m nu).
    C6: energy balance => <eps> = (a . W) / (KAPPA nu r), sampled at the Poisson event after t_max.
    C3: the result cannot depend on nu_hat."""
    nu, rec, E = 400.0, 0.02, np.array([0.0, 0.0, -2000.0])
    W_exact = -(KAPPA / nu) * E
    eps_exact = (-(KAPPA * E) @ W_exact) / (KAPPA * nu * rec)
    out = []
    for nu_hat, seed in ((400.0, 21), (1000.0, 22)):
        r, W, se = _drift_run(oracle, nu, rec, E, (0, 0, 0), nu_hat, 1500, 4.0, seed)
        assert np.all(np.abs(W - W_exact) < 4 * se + 1e-12), (W, W_exact, se)
        assert se[2] < 0.01 * abs(W_exact[2])                      # the test resolves 1 %
        # equilibrium after ~ 1/(nu r) = 0.125 ns; t_max = 4 ns
        e = r.end[4]
        assert abs(e.mean() - eps_exact) < 4 * e.std(ddof=1) / np.sqrt(len(e)), (e.mean(), eps_exact)
        out.append((W, se))
    assert np.all(np.abs(out[0][0] - out[1][0]) < 4 * np.hypot(out[0][1], out[1][1]) + 1e-12)


def test_c5_drift_with_magnetic_field(oracle):
    """C5 with B: W = -(KAPPA/nu)/(1+beta^2) [E - beta (E x b) + beta^2 (E.b) b], beta = OMEGA1 |B| / nu
    (steady state of dW/dt = -KAPPA E - OMEGA1 W x B - nu W).  E perp B part gives tan(Lorentz angle) = beta."""
    nu, rec = 250.0, 0.02
    E = np.array([0.0, 0.0, -2000.0])
    B = np.array([0.0, 0.5, 0.8660254037844387])                     # 1 T at 30 deg to the field axis
    Bn = np.linalg.norm(B); b = B / Bn
    beta = OMEGA1 * Bn / nu
    W_exact = -(KAPPA / nu) / (1 + beta ** 2) * (E - beta * np.cross(E, b) + beta ** 2 * (E @ b) * b)
    # independent check of the closed form: solve the 3x3 linear steady-state system
    M = nu * np.eye(3) + OMEGA1 * np.array([[0, B[2], -B[1]], [-B[2], 0, B[0]], [B[1], -B[0], 0]])
    assert np.allclose(np.linalg.solve(M, -KAPPA * E), W_exact, rtol=1e-12)
    r, W, se = _drift_run(oracle, nu, rec, E, tuple(B), 600.0, 1500, 4.0, 23)
    assert np.all(np.abs(W - W_exact) < 4 * se + 1e-12), (W, W_exact, se)
    assert np.all(se < 0.02 * np.linalg.norm(W_exact))


def test_c7_recoil_and_isotropic_deflection(oracle):
    """C7 / S9b-d: elastic energy factor 1 - r (1 - cos theta) with theta the angle between k' and k'';
    cos theta uniform in [-1,1], azimuth uniform, |k''| = 1."""
    rec = 0.013
    g = gas.constant_elastic(100.0, rec)                            # nu_hat = nu: every step is a real collision
    rng = np.random.default_rng(12)
    n = 30000
    st = _states(n, rng)
    res = oracle.step_batch(g, _open_field((0, 0, 0)), 9, st, np.arange(n, dtype=np.uint64), np.full(n, 5, dtype=np.uint32))
    assert np.all(res.event == 0)
    k0, k1 = st[5:8], res.state[5:8]
    ct = (k0 * k1).sum(0)
    assert np.abs(np.linalg.norm(k1, axis=0) - 1).max() < 1e-14
    assert np.allclose(res.state[4], st[4] * (1 - rec * (1 - ct)), rtol=1e-12)
    assert abs(np.mean((st[4] - res.state[4]) / st[4]) - rec) < 4 * rec / np.sqrt(3 * n)
    assert stats.kstest((ct + 1) / 2, "uniform").pvalue > 1e-3
    # azimuth of k'' about k' in any fixed frame perpendicular to k': uniform
    a = np.cross(k0.T, np.array([0.3, -0.5, 0.81])); a /= np.linalg.norm(a, axis=1)[:, None]
    b = np.cross(k0.T, a)
    phi = np.arctan2((k1.T * b).sum(1), (k1.T * a).sum(1))
    assert stats.kstest((phi + np.pi) / (2 * np.pi), "uniform").pvalue > 1e-3
    # and the positions/energies before the collision are untouched by it: no field, so |dr| = speed * dt
    dr = np.linalg.norm(res.state[0:3] - st[0:3], axis=0)
    assert np.allclose(dr, C2 * np.sqrt(st[4]) * (res.state[3] - st[3]), rtol=1e-9)


def test_c8_diffusion_closed_form(oracle):
    """C8: constant speed v, isotropic scattering at rate nu, no field:
    <x^2> = 2 D [t - (1 - exp(-nu t))/nu], D = v^2/(3 nu) (velocity autocorrelation exp(-nu t))."""
    nu, e0, t_max, n_el = 100.0, 4.0, 0.5, 6000
    g = gas.constant_elastic(nu, 0.0, nu_hat=150.0)
    p = primaries.isotropic_primaries(n_el, 31, e_scale=0.0)
    p[:, 4] = e0
    r = oracle.run(g, _open_field((0, 0, 0)), p, seed=31, t_max=t_max, n_threads=8)
    v = C2 * np.sqrt(e0)
    t = r.end[3]                                                    # first event after t_max (Poisson: t_max + Exp)
    var_pred = np.mean(2 * v * v / (3 * nu) * (t - (1 - np.exp(-nu * t)) / nu))
    x2 = (r.end[0:3] ** 2).mean(1)
    assert np.all(np.abs(x2 - var_pred) < 4 * var_pred * np.sqrt(2.0 / n_el)), (x2, var_pred)


def test_c9_level_selection_fractions(oracle):
    """C9 / S7-S8: P(level l) = rate_l / nu_hat, P(null) = 1 - nu_tot/nu_hat (chi-square)."""
    rates = [5.0, 0.0, 20.0, 1.0, 14.0]
    types = [gas.ELASTIC, gas.EXCITATION, gas.EXCITATION, gas.ATTACHMENT, gas.ELASTIC]
    g = gas.multi_level_constant(rates, types, nu_hat=60.0)
    rng = np.random.default_rng(13)
    n = 60000
    st = _states(n, rng)
    res = oracle.step_batch(g, _open_field((0, 0, 0)), 11, st, np.arange(n, dtype=np.uint64), np.zeros(n, dtype=np.uint32))
    obs = np.array([(res.event == l).sum() for l in range(5)] + [(res.event == -1).sum()])
    exp = n * np.array(rates + [60.0 - sum(rates)]) / 60.0
    assert obs[1] == 0                                              # a zero-rate level is never selected
    keep = exp > 0
    assert stats.chisquare(obs[keep], exp[keep]).pvalue > 1e-3
    assert np.all(res.status[res.event == 3] == 5) and np.all(res.status[res.event != 3] == 0)
    # energy-bin lookup: a table that is zero except in one bin only collides there
    gb = gas.multi_level_constant([10.0], [gas.ELASTIC], n_bins=50, e_max=25.0, nu_hat=10.0)
    gb.cum_rate[:] = 0.0
    gb.cum_rate[7, :] = 10.0                                        # bin 7 = [3.5, 4.0) eV
    res = oracle.step_batch(gb, _open_field((0, 0, 0)), 1, st, np.arange(n, dtype=np.uint64), np.zeros(n, dtype=np.uint32))
    inside = (st[4] >= 3.5) & (st[4] < 4.0)
    assert np.array_equal(res.event >= 0, inside) and np.array_equal(res.bin, np.minimum((st[4] * 2).astype(int), 49))


def test_c10_opal_beaty_sharing(oracle):
    """C10 / R10: secondary energy CDF F(es) = atan(es/w)/atan(ea/2w) on [0, ea/2]; primary keeps ea - es;
    child direction isotropic; child id = words (w0,w1) of block 0xFFFFFFFF."""
    w, thr, e_in = 10.0, 15.76, 60.0
    g = gas.ionisation_only(80.0, w=w)
    g.level_loss[:] = thr
    n = 30000
    st = np.zeros((8, n)); st[4] = e_in; st[7] = 1.0
    ids = np.arange(n, dtype=np.uint64) * 7 + 3
    res = oracle.step_batch(g, _open_field((0, 0, 0)), 17, st, ids, np.full(n, 2, dtype=np.uint32))
    assert np.all(res.event == 0)
    ea = e_in - thr
    es = res.child[4]
    assert es.max() <= ea / 2 * (1 + 1e-12) and es.min() >= 0
    assert np.allclose(res.state[4] + es, ea, rtol=1e-12)
    assert stats.kstest(np.arctan(es / w) / np.arctan(ea / (2 * w)), "uniform").pvalue > 1e-3
    ck = res.child[5:8]
    assert np.abs(np.linalg.norm(ck, axis=0) - 1).max() < 1e-14
    assert stats.kstest((ck[2] + 1) / 2, "uniform").pvalue > 1e-3
    assert stats.kstest((np.arctan2(ck[1], ck[0]) + np.pi) / (2 * np.pi), "uniform").pvalue > 1e-3
    assert np.array_equal(res.child[0:4], res.state[0:4])            # born at the collision point and time
    for i in range(50):
        wd = oracle.philox(17, int(ids[i]), 2, 0xFFFFFFFF)
        assert int(res.child_id[i]) == int(wd[0]) + (int(wd[1]) << 32)
    assert len(np.unique(res.child_id)) == n


def test_c11_charge_conservation_g0(oracle, g0):
    """C11 on BASELINE config 1: endpoints = primaries + ionisations; attached = attachment tally;
    per-avalanche rows sum to the totals; every id unique; every avalanche has its primary."""
    f = fields.uniform_gap((0, 0, -30000.0), 0.0, 50e-4)
    p = primaries.isotropic_primaries(1000, 0)
    r = oracle.run(g0, f, p, seed=0)
    t = r.tallies_u64
    L = g0.n_levels
    n_ion = int(t[14] + t[15]); n_att = int(t[16])
    assert r.n == 1000 + n_ion
    assert (r.status == 5).sum() == n_att
    assert int(t[L] + t[L + 1]) + int(np.isin(r.status, (1, 2, 3, 4, 6, 7)).sum()) == int(t[L + 3])   # null + real + terminated flights = steps
    assert int(t[:L].sum()) == int(t[L + 1])
    assert r.per_avalanche[:, 0].sum() == r.n and np.all(r.per_avalanche[:, 1] == r.per_avalanche[:, 0] - 1)
    assert r.per_avalanche[:, 2].sum() == n_att
    assert len(np.unique(r.id)) == r.n and set(range(1000)) <= set(r.id.tolist())
    assert np.array_equal(np.bincount(r.avalanche, minlength=1000), r.per_avalanche[:, 0])
    assert int(r.n_steps.sum()) == int(t[L + 3])
    assert np.all(r.status != 0)
    # endpoints are outside the gap or attached; births inside
    out = (r.end[2] < 0) | (r.end[2] > 50e-4)
    assert np.all(out | (r.status == 5)) and np.all((r.birth[2] >= 0) & (r.birth[2] <= 50e-4))


def test_c12_attachment_only(oracle):
    """C12: attachment-only gas: attachment time ~ Exp(nu_att) under null-collision thinning (nu_hat = 4 nu_att);
    survivors at t_max ~ Binomial(N, exp(-nu_att t_max))."""
    nu_att, t_max, n_el = 2.0, 0.4, 8000
    g = gas.attachment_only(nu_att, nu_hat=8.0)
    p = primaries.isotropic_primaries(n_el, 41)
    r = oracle.run(g, _open_field((0, 0, 0)), p, seed=41, t_max=t_max)
    att = r.status == 5
    surv = r.status == 6
    assert att.sum() + surv.sum() == n_el
    ps = np.exp(-nu_att * t_max)
    assert abs(surv.sum() - n_el * ps) < 4 * np.sqrt(n_el * ps * (1 - ps))
    ta = r.end[3][att]                                              # truncated exponential on [0, t_max]
    cdf = (1 - np.exp(-nu_att * ta)) / (1 - ps)
    assert stats.kstest(cdf, "uniform").pvalue > 1e-3


def test_c13_yule_furry_gain_distribution(oracle):
    """C13: energy-independent ionisation rate nu_i, threshold 0, stop at t_max: the avalanche size is
    Yule-Furry, P(n) = (1/nbar)(1 - 1/nbar)^(n-1), nbar = exp(nu_i t_max) — exact gain *distribution*;
    exercises spawn + stack + per-avalanche bookkeeping."""
    nu_i, t_max, n_p = 5.0, 0.4, 5000
    g = gas.ionisation_only(nu_i, nu_hat=12.0)
    p = primaries.isotropic_primaries(n_p, 43, e_scale=50.0)
    r = oracle.run(g, _open_field((0, 0, 0)), p, seed=43, t_max=t_max, capacity=1 << 18)
    size = r.per_avalanche[:, 0].astype(np.int64)
    nbar = np.exp(nu_i * t_max)
    assert abs(size.mean() - nbar) < 4 * np.sqrt(nbar * (nbar - 1) / n_p)
    q = 1 - 1 / nbar
    edges = np.array([1, 2, 3, 4, 5, 6, 8, 10, 13, 17, 22, 30, 10 ** 9])
    obs = np.histogram(size, bins=edges)[0]
    exp = n_p * (q ** (edges[:-1] - 1) - q ** (edges[1:] - 1))
    assert stats.chisquare(obs, exp * obs.sum() / exp.sum()).pvalue > 1e-3
    assert np.all(r.status == 6)


def test_c14_gain_vs_townsend_alpha(oracle, g0):
    """C14: uniform field, gap >> equilibration length: ln(mean gain)/d ~ alpha - eta from the tallies
    (N_ion - N_att) / sum(dz), within 10 %."""
    d = 100e-4
    f = fields.uniform_gap((0, 0, -60000.0), 0.0, d)
    p = primaries.isotropic_primaries(24, 51, forward=True)
    p[:, 2] = 2e-4                                                   # 2 um inside: fewer back-scatter losses
    r = oracle.run(g0, f, p, seed=51, capacity=1 << 20, n_threads=8)
    t = r.tallies_u64
    alpha = (float(t[14] + t[15]) - float(t[16])) / r.tallies_f64[2]
    fw = r.per_avalanche[:, 0][r.per_avalanche[:, 0] > 20].astype(float)   # avalanches that did not die at the cathode
    assert len(fw) >= 12
    a_gain = np.log(fw.mean()) / (d - 2e-4)
    assert abs(a_gain - alpha) < 0.10 * alpha, (a_gain, alpha)


def _transport_stats(r, n_levels):
    """Per-primary gain (mean, SE), drift velocity along the force, ionisations per cm of drift, real collisions per ns."""
    gain = r.per_avalanche[:, 0].astype(float)
    t = r.tallies_u64
    W = r.tallies_f64[2] / r.tallies_f64[3]
    alpha = (float(t[14] + t[15]) - float(t[16])) / r.tallies_f64[2]
    nu_real = float(t[n_levels + 1]) / r.tallies_f64[3]
    return gain.mean(), gain.std(ddof=1) / np.sqrt(len(gain)), W, alpha, nu_real


def test_c3_null_collision_invariance_g0(oracle, g0):
    """C3: the null-collision method is exact for ANY nu_hat >= max total rate — doubling nu_hat doubles the null steps
    and must leave every statistic alone: gain, drift velocity, Townsend alpha and the real-collision rate of gas G0 at
    45 kV/cm (independent streams, so within sampling errors)."""
    import dataclasses
    f = fields.uniform_gap((0, 0, -45000.0), 0.0, 80e-4)
    p = primaries.isotropic_primaries(1500, 61, forward=True)
    p[:, 2] = 2e-4
    g2 = dataclasses.replace(g0, nu_hat=2.0 * g0.resolved_nu_hat())
    a = oracle.run(g0, f, p, seed=61, capacity=1 << 20, n_threads=8)
    b = oracle.run(g2, f, p, seed=62, capacity=1 << 20, n_threads=8)
    L = g0.n_levels
    # the null steps double (real collisions do not)
    null_a, null_b = float(a.tallies_u64[L]), float(b.tallies_u64[L])
    real_a, real_b = float(a.tallies_u64[L + 1]), float(b.tallies_u64[L + 1])
    assert abs((null_b + real_b) / (null_a + real_a) / 2.0 - 1.0) < 0.05
    ga, sa, Wa, aa, na = _transport_stats(a, L)
    gb, sb, Wb, ab, nb = _transport_stats(b, L)
    assert abs(ga - gb) < 3.5 * np.hypot(sa, sb), (ga, gb, sa, sb)
    assert abs(Wb / Wa - 1) < 0.01 and abs(nb / na - 1) < 0.01, (Wa, Wb, na, nb)
    assert abs(ab / aa - 1) < 0.04, (aa, ab)
