"""Oracle pins of NEXT-4 (DESIGN.md §3.7 readings W1-W4), CPU only: induced-signal accumulation
(Shockley-Ramo: q E_w . dr per flight into time bins) and ion drift (explicit midpoint along q mu E).  Pinned to what the
theorem and the mathematics fix: the induced charge of a carrier is the weighting-potential difference it crosses
(exactly, for a uniform weighting field: the sum telescopes to the endpoints), a constant drift velocity gives a flat
current, ions in a uniform field move on straight lines at mu E, the midpoint rule converges with order 2 to the
field-line ODE, and an electron-ion pair that is fully collected induces exactly one elementary charge."""
import numpy as np
import pytest
from scipy import stats
from scipy.integrate import solve_ivp

from paper_2509_15377_b200.gen import fields, gas, primaries

KAPPA = 0.0017588200107589609
BIG = 1.0e6


def _weighting_plate(z_lo, z_hi):
    return fields.uniform_gap((0.0, 0.0, 1.0 / (z_hi - z_lo)), z_lo, z_hi)


def test_w2_ramo_theorem_uniform_weighting(oracle, g0):
    """Parallel plate, E_w = z / d: the electrons' induced charge is -sum over electrons of (z_end - z_birth) / d — the
    per-flight sum telescopes — whatever the multiplication; time bins wide enough hold all of it."""
    d = 50e-4
    fd = fields.uniform_gap((0.0, 0.0, -30000.0), 0.0, d)
    p = primaries.isotropic_primaries(300, 3)
    r = oracle.run(g0, fd, p, seed=3, signal=(_weighting_plate(0.0, d), 0.0, 0.01, 64))
    assert r.n > 330 and r.signal is not None
    exact = -((r.end[2] - r.birth[2]) / d).sum()
    assert abs(r.signal.sum() - exact) < 1e-10 * abs(exact)
    assert r.end[3].max() < 0.64                                      # nothing fell outside the bins
    # the same run without the signal is the same run
    r0 = oracle.run(g0, fd, p, seed=3)
    assert np.array_equal(r0.end, r.end) and r0.signal is None
    # a weighting field that covers only the upper half of the gap sees only the flights that START there
    half = oracle.run(g0, fd, p, seed=3, signal=(_weighting_plate(d / 2, d), 0.0, 0.01, 64))
    assert 0.3 * abs(exact) < abs(half.signal.sum()) * 0.5 < abs(exact)
    # multi-threaded accumulation adds up to the same histogram
    r8 = oracle.run(g0, fd, p, seed=3, n_threads=8, signal=(_weighting_plate(0.0, d), 0.0, 0.01, 64))
    assert np.allclose(r8.signal, r.signal, rtol=1e-9, atol=1e-12)


def test_w2_time_bins_flat_current_and_shift(oracle):
    """Constant collision frequency, no multiplication, open space: after the relaxation the current is flat,
    charge per bin = -N W_z E_w dt_bin with W = -(KAPPA / nu) E (C5).  Shifting t0 by whole bins shifts the histogram;
    flights that start before t0 or after the last bin are dropped."""
    nu, E0, n_el, dtb = 400.0, 2000.0, 4000, 0.1
    g = gas.constant_elastic(nu, 0.02)
    fd = fields.uniform_gap((0.0, 0.0, -E0), -BIG, BIG)
    wf = fields.uniform_gap((0.0, 0.0, 0.5), -BIG, BIG)
    p = primaries.isotropic_primaries(n_el, 5, e_scale=1.0)
    a = oracle.run(g, fd, p, seed=5, t_max=3.0, n_threads=8, signal=(wf, 0.0, dtb, 30))
    Wz = (KAPPA / nu) * E0
    per_bin = -n_el * Wz * 0.5 * dtb
    late = a.signal[5:29]                                              # relaxation time 1 / (nu r) = 0.125 ns
    assert abs(late.mean() / per_bin - 1) < 0.01
    assert np.all(np.abs(late / per_bin - 1) < 0.05)
    b = oracle.run(g, fd, p, seed=5, t_max=3.0, n_threads=8, signal=(wf, 3 * dtb, dtb, 30))
    assert np.allclose(b.signal[:27], a.signal[3:], rtol=1e-6, atol=1e-9 * abs(per_bin))
    assert np.all(b.signal[28:] == 0.0)                               # the run ends at t_max = 3.0 + one flight
    c = oracle.run(g, fd, p, seed=5, t_max=3.0, n_threads=8, signal=(wf, 0.0, dtb, 10))
    assert np.allclose(c.signal, a.signal[:10], rtol=1e-6, atol=1e-9 * abs(per_bin))


def test_w2_the_bin_is_that_of_the_flights_start_time(oracle):
    """Electrons start at t = 0; with t0 a hair above 0 the FIRST flight of each starts before the first bin and is dropped,
    every later flight is kept: total = -sum (z_end - z_1) / d with z_1 the position after the first flight (one oracle
    step from the primaries)."""
    d = 1.0
    g = gas.constant_elastic(500.0, 0.02, nu_hat=800.0)
    fd = fields.uniform_gap((0.0, 0.0, -2000.0), -BIG, BIG)
    wf = fields.uniform_gap((0.0, 0.0, 1.0 / d), -BIG, BIG)
    p = primaries.isotropic_primaries(200, 17, e_scale=2.0, forward=True)
    r = oracle.run(g, fd, p, seed=17, t_max=0.5, signal=(wf, 1e-12, 1.0, 4))
    st = np.ascontiguousarray(p.T)
    one = oracle.step_batch(g, fd, 17, st, np.arange(200, dtype=np.uint64), np.zeros(200, dtype=np.uint32))
    assert np.array_equal(r.id, np.arange(200, dtype=np.uint64))
    exact = -((r.end[2] - one.state[2]) / d).sum()
    first = -((one.state[2] - p[:, 2]) / d).sum()
    assert abs(r.signal.sum() - exact) < 1e-9 * abs(exact) and abs(first) > 1e-4 * abs(exact)


def test_w4_ion_signal_bin_is_that_of_the_steps_start_time(oracle):
    """One ion, uniform field, steps of exactly 1 ns (0.2 um at 2e-5 cm/ns), bins of 1 ns from t0 = -0.5: step k starts at
    t = k and lands in bin k; the bin after the last step stays empty."""
    fd = fields.uniform_gap((0.0, 0.0, -20000.0), 0.0, 1.0)
    wf = fields.uniform_gap((0.0, 0.0, 2.0), 0.0, 1.0)

    class Fake:
        n = 2
        birth = np.array([[0, 0.0], [0, 0.0], [0, 0.5], [0, 0.0], [1, 1]], dtype=float)
        end = np.zeros((8, 2)); status = np.array([1, 1], dtype=np.int32)
    ions = oracle.ion_drift(fd, Fake, 1, 1e-9, 1e-9, 2e-5, max_steps=6, signal=(wf, -0.5, 1.0, 10))
    assert ions.status[1] == 7 and ions.n_steps[1] == 6 and abs(ions.end[3, 1] - 6.0) < 1e-12
    assert np.allclose(ions.signal[:6], -2.0 * 2e-5, rtol=1e-9) and np.all(ions.signal[6:] == 0.0)      # +1 charge moving toward -z


def _potential_map(nx, ny, nz, h):
    """A smooth weighting potential V_w on a grid and E_w = -grad V_w at the nodes (analytic)."""
    x = np.arange(nx) * h; y = np.arange(ny) * h; z = np.arange(nz) * h
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    k = 2 * np.pi / (40 * h)
    V = lambda X, Y, Z: 30.0 * Z + 0.02 * np.sin(k * X) * np.cos(0.7 * k * Y) * np.exp(-k * Z)
    nodes = np.zeros((nz, ny, nx, 4), dtype=np.float32)
    nodes[..., 0] = -0.02 * k * np.cos(k * X) * np.cos(0.7 * k * Y) * np.exp(-k * Z)
    nodes[..., 1] = 0.02 * 0.7 * k * np.sin(k * X) * np.sin(0.7 * k * Y) * np.exp(-k * Z)
    nodes[..., 2] = -30.0 + 0.02 * k * np.sin(k * X) * np.cos(0.7 * k * Y) * np.exp(-k * Z)
    nodes[..., 3] = 1.0
    return nodes, V


def test_w1_nonuniform_weighting_is_the_potential_difference(oracle):
    """E_w from a grid map of -grad V_w: the induced charge of ONE electron is q times minus the potential difference
    it crosses, -1 x -(V_w(end) - V_w(birth)), up to the Riemann sum over its (short) flights and the trilinear
    interpolation — pins the point where E_w is taken, the dot product with dr (not v) and the sign."""
    h = 1e-4
    nodes, V = _potential_map(64, 64, 64, h)
    wf = fields.FieldDesc([fields.grid_slab(nodes, (0, 0, 0), (h, h, h), 0.0, 63 * h)])
    g = gas.constant_elastic(2000.0, 0.02)
    fd = fields.FieldDesc([fields.Slab(2 * h, 61 * h, fields.KIND_UNIFORM, (300.0, -200.0, -3000.0))], (0.0, 0.0, 0.0),
                          (2 * h, 2 * h), (61 * h, 61 * h))
    errs = []
    for i in range(24):
        p = primaries.isotropic_primaries(1, 100 + i, pos=(20 * h + i * h, 45 * h - i * h, 5 * h), e_scale=0.5)
        r = oracle.run(g, fd, p, seed=100 + i, signal=(wf, 0.0, 1.0, 8))
        dV = V(r.end[0, 0], r.end[1, 0], r.end[2, 0]) - V(r.birth[0, 0], r.birth[1, 0], r.birth[2, 0])
        assert abs(dV) > 0.05
        errs.append(r.signal.sum() / dV - 1)
    assert np.max(np.abs(errs)) < 2e-3, errs


# ---- ions -------------------------------------------------------------------------------------------------------------
def test_w3_w4_ions_in_a_uniform_field(oracle, g0):
    """Positive ions start where secondaries were born and move along +E (here -z) at mu E on straight lines; negative ions
    (attached electrons) move the other way.  Arrival time = distance / (mu E) to within one step; which ions exist."""
    d, E0, mu_p, mu_n, step = 50e-4, 30000.0, 1.5e-6, 2.0e-6, 0.5e-4
    fd = fields.uniform_gap((0.0, 0.0, -E0), 0.0, d)
    p = primaries.isotropic_primaries(400, 11)
    g = gas.multi_level_constant([2000.0, 8.0, 4.0], [gas.ELASTIC, gas.IONISATION, gas.ATTACHMENT], recoil=[0.02, 0, 0], w=[0, 10.0, 0],
                                 n_bins=32, e_max=100.0)             # multiplies AND attaches within the gap
    r = oracle.run(g, fd, p, seed=11)
    ions = oracle.ion_drift(fd, r, 400, mu_p, mu_n, step)
    n = r.n
    is_prim = np.arange(n) < 400                                      # outputs are in creation order: primaries first
    assert np.array_equal(r.id[:400], np.arange(400, dtype=np.uint64)) and np.all(r.birth[3][:400] == 0.0) and np.all(r.birth[3][400:] > 0.0)
    pos, neg = ions.status[:n], ions.status[n:]
    assert np.all(pos[is_prim] == -1) and np.all(pos[~is_prim] == 1)          # every secondary left an ion; it reaches z < 0
    att = r.status == 5
    assert att.sum() > 3 and np.all(neg[att] == 2) and np.all(neg[~att] == -1)
    z0 = r.birth[2][~is_prim]
    e = ions.end[:, :n][:, ~is_prim]
    assert np.array_equal(e[0], r.birth[0][~is_prim]) and np.array_equal(e[1], r.birth[1][~is_prim])
    assert np.all(e[2] < 0.0) and np.all(e[2] >= -step * (1 + 1e-9))
    t_exact = r.birth[3][~is_prim] + z0 / (mu_p * E0)
    assert np.all(np.abs(e[3] - t_exact) <= step / (mu_p * E0) * (1 + 1e-9))
    assert np.array_equal(ions.n_steps[:n][~is_prim], np.floor(z0 / step).astype(np.uint32) + 1)
    en = ions.end[:, n:][:, att]
    assert np.all(en[2] > d) and np.all(np.abs(en[3] - (r.end[3][att] + (d - r.end[2][att]) / (mu_n * E0))) <= step / (mu_n * E0) * (1 + 1e-9))


def test_w4_pair_induces_one_elementary_charge(oracle, g0):
    """Uniform weighting field over the gap: electrons + ions together induce sum q (z_end - z_start) / d, and a pair whose
    electron reaches the anode and whose ion reaches the cathode induces -(d + overshoots) / d: one elementary charge."""
    d, E0 = 50e-4, 30000.0
    fd = fields.uniform_gap((0.0, 0.0, -E0), 0.0, d)
    wf = _weighting_plate(-1e-4, d + 1e-4)                            # covers the overshoot of the last flight / step
    p = primaries.isotropic_primaries(300, 13, forward=True)
    sig = (wf, 0.0, 50.0, 200)
    r = oracle.run(g0, fd, p, seed=13, signal=sig)
    ions = oracle.ion_drift(fd, r, 300, 1.5e-9, 2.0e-9, 0.25e-4, signal=sig)      # 1.5, 2 cm^2 / (V s)
    n = r.n
    dd = d + 2e-4
    q_e = -((r.end[2] - r.birth[2]) / dd).sum()
    assert abs(r.signal.sum() - q_e) < 1e-10 * abs(q_e)
    have_p = ions.status[:n] >= 0; have_n = ions.status[n:] >= 0
    q_i = ((ions.end[2, :n] - r.birth[2])[have_p] / dd).sum() - ((ions.end[2, n:] - r.end[2])[have_n] / dd).sum()
    assert abs(ions.signal.sum() - q_i) < 1e-10 * abs(q_i)
    # pairs: the secondary electrons that reached the anode (status 2), with their ions at the cathode
    sec = have_p & (r.status == 2)
    per_pair = -(r.end[2][sec] - r.birth[2][sec]) / dd + (ions.end[2, :n][sec] - r.birth[2][sec]) / dd
    assert np.all(per_pair <= -d / dd) and np.all(per_pair > -d / dd - 0.05) and sec.sum() > 20     # overshoots only add
    # ions are slow: their signal lasts ~ d / (mu E) = 111 ns, the electrons' < 0.1 ns
    assert np.flatnonzero(np.abs(ions.signal) > 0).max() >= 1 and np.flatnonzero(np.abs(r.signal) > 0).max() == 0


def test_w4_midpoint_rule_converges_to_the_field_line(oracle):
    """A curved field (grid map of a smooth analytic field): the ion's path is the field line dr/ds = q E / |E|.  The
    explicit midpoint rule has global order 2: endpoints against scipy's solution of the same ODE through the oracle's own
    trilinear field, error falling ~4x per halving of the step."""
    h = 2e-4
    nodes, _ = _potential_map(64, 64, 64, h)
    nodes[..., 0:3] *= 1000.0                                          # V/cm scale; curvature from the sin / exp term
    nodes[..., 0] += 25000.0 * np.sin(np.arange(64) * 0.1)[None, None, :]     # strong x-dependent transverse field
    fm = fields.FieldDesc([fields.grid_slab(nodes, (0, 0, 0), (h, h, h), 0.0, 63 * h)])

    class Fake:                                                        # a "run" of three electrons: two secondaries, one attached
        n = 3
        birth = np.array([[0, 30 * h, 20 * h], [0, 30 * h, 40 * h], [0, 55 * h, 50 * h], [0, 0.5, 0.7], [1, 1, 1]], dtype=float)
        end = np.zeros((8, 3)); status = np.array([1, 1, 5], dtype=np.int32)
    Fake.end[0:4, 2] = (33 * h, 33 * h, 10 * h, 2.0)

    def field_line(r0, q, length):
        def rhs(s, r):
            E, m, sl = oracle.field_eval(fm, r.reshape(3, 1))
            e = E[:, 0]
            return q * e / np.linalg.norm(e)
        return solve_ivp(rhs, (0, length), r0, rtol=1e-10, atol=1e-13).y[:, -1]

    errs = []
    for step in (2e-4, 1e-4, 0.5e-4):
        n_steps = int(round(40e-4 / step))
        ions = oracle.ion_drift(fm, Fake, 1, 1e-6, 1e-6, step, max_steps=n_steps)
        assert list(ions.status) == [-1, 7, 7, -1, -1, 7] and np.all(ions.n_steps[[1, 2, 5]] == n_steps)
        e = 0.0
        for i, r0, q in ((1, Fake.birth[0:3, 1], 1.0), (2, Fake.birth[0:3, 2], 1.0), (5, Fake.end[0:3, 2], -1.0)):
            e = max(e, np.linalg.norm(ions.end[0:3, i] - field_line(r0, q, n_steps * step)))
        errs.append(e)
    assert errs[2] < 2e-7 and errs[0] > 3.0 * errs[1] > 9.0 * errs[2] * 0.9, errs
    # drift time: dt = step / (mu |E(r_m)|) per step — the midpoint speed, second order too: against the line integral of
    # ds / (mu |E|) along the same field line (|E| varies by ~20 % along these paths)
    def drift_time(r0, q, length, mu):
        def rhs(s, y):
            E, m, sl = oracle.field_eval(fm, y[:3].reshape(3, 1))
            e = E[:, 0]; ne = np.linalg.norm(e)
            return np.concatenate([q * e / ne, [1.0 / (mu * ne)]])
        return solve_ivp(rhs, (0, length), np.concatenate([r0, [0.0]]), rtol=1e-10, atol=1e-13).y[3, -1]
    for i, r0, q, t0 in ((1, Fake.birth[0:3, 1], 1.0, 0.5), (5, Fake.end[0:3, 2], -1.0, 2.0)):
        exact = drift_time(r0, q, n_steps * step, 1e-6)
        assert abs((ions.end[3, i] - t0) / exact - 1) < 2e-5, ((ions.end[3, i] - t0), exact)
    # the ions' induced charge through a curved weighting potential: E_w at the step's MIDPOINT makes the sum second order,
    # q x -(V_w(end) - V_w(start)) to ~1e-5 (E_w at the step's start would leave ~1e-2)
    x = np.arange(64) * h
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    k = 2 * np.pi / (40 * h)
    V = lambda X, Y, Z: 30.0 * Z + 0.05 * np.sin(k * X) * np.cos(0.7 * k * Y) * np.cos(0.5 * k * Z)      # wavy all along the paths
    wnodes = np.zeros((64, 64, 64, 4), dtype=np.float32)
    wnodes[..., 0] = -0.05 * k * np.cos(k * X) * np.cos(0.7 * k * Y) * np.cos(0.5 * k * Z)
    wnodes[..., 1] = 0.05 * 0.7 * k * np.sin(k * X) * np.sin(0.7 * k * Y) * np.cos(0.5 * k * Z)
    wnodes[..., 2] = -30.0 + 0.05 * 0.5 * k * np.sin(k * X) * np.cos(0.7 * k * Y) * np.sin(0.5 * k * Z)
    wnodes[..., 3] = 1.0
    wf = fields.FieldDesc([fields.grid_slab(wnodes, (0, 0, 0), (h, h, h), 0.0, 63 * h)])
    ions = oracle.ion_drift(fm, Fake, 1, 1e-6, 1e-6, step, max_steps=n_steps, signal=(wf, -1.0, 1e9, 1))
    exact = 0.0
    for i, r0, q in ((1, Fake.birth[0:3, 1], 1.0), (2, Fake.birth[0:3, 2], 1.0), (5, Fake.end[0:3, 2], -1.0)):
        exact += -q * (V(*ions.end[0:3, i]) - V(*r0))
    assert abs(ions.signal[0] / exact - 1) < 3e-4, (ions.signal[0], exact)


def test_w4_ions_stop_in_material_and_at_limits(oracle):
    h = 1e-4
    nodes = np.zeros((40, 8, 8, 4), dtype=np.float32)
    nodes[..., 2] = -20000.0; nodes[..., 3] = 1.0
    nodes[:10, :, :, 3] = 0.0                                          # solid below z = 9.5 um (mask interpolates to 0.5 there)
    fm = fields.FieldDesc([fields.grid_slab(nodes, (0, 0, 0), (h, h, h), 0.0, 39 * h)])

    class Fake:
        n = 2
        birth = np.array([[0, 3 * h], [0, 3 * h], [0, 30 * h], [0, 0.0], [1, 1]], dtype=float)
        end = np.zeros((8, 2)); status = np.array([1, 1], dtype=np.int32)
    ions = oracle.ion_drift(fm, Fake, 1, 1e-6, 1e-6, 0.3e-4)
    assert ions.status[1] == 4 and 9.5 * h - 0.3e-4 <= ions.end[2, 1] < 9.5 * h
    late = oracle.ion_drift(fm, Fake, 1, 1e-6, 1e-6, 0.3e-4, t_max=0.05)       # the whole path takes 0.1 ns
    assert late.status[1] == 6 and late.end[3, 1] > 0.05 and late.end[3, 1] < 0.05 + 0.3e-4 / (1e-6 * 20000.0) * 1.001
    few = oracle.ion_drift(fm, Fake, 1, 1e-6, 1e-6, 0.3e-4, max_steps=5)
    assert few.status[1] == 7 and few.n_steps[1] == 5
