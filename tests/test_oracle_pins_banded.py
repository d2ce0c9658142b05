"""Oracle pins, part 4: the energy-banded null-collision rate (readings N1-N6).

The banded mode (flag AVMO_BANDED) draws a flight with the rate of the electron's energy band and of the flight's
acceleration class instead of the global maximum, and cuts flights at the band's validity time.  It is the same
physics with fewer null steps, so every closed form of the global mode must hold unchanged, and the table of banded
rates must bound the total rate of every bin a flight can reach.  CPU only.
"""
import numpy as np
import pytest
from scipy import stats

from paper_2509_15377_b200.gen import fields, gas, primaries

KAPPA = 0.0017588200107589609
C2 = 0.05930969584745753
INV_C2SQ = 284.28150518042008
BIG = 1.0e6


def _open_field(E, B=(0, 0, 0)):
    return fields.uniform_gap(E, -BIG, BIG, B)


def _sawtooth_gas(n_bins=4096, e_max=60.0):
    """Total rate that goes up AND down with energy: a bound built from the band's own bins only (no running maximum
    over the lower bins a decelerating electron reaches, or no look-ahead to the bins an accelerating one reaches) fails."""
    e = (np.arange(n_bins) + 0.5) * e_max / n_bins
    el = 200.0 + 1500.0 * np.abs(np.sin(1.3 * e)) + 40.0 * e
    ion = np.full(n_bins, 5.0)
    return gas._finish(n_bins, e_max, np.stack([el, ion], 1), [gas.ELASTIC, gas.IONISATION], [0.0, 0.0], [1e-4, 0.0],
                       [0.0, 10.0], ["sawtooth elastic", "ionisation"])


def _class_of(a2_edges, a2):
    j = 0
    while j < len(a2_edges) and a2 > a2_edges[j]:
        j += 1
    return j


@pytest.mark.parametrize("which", ["g0", "sawtooth"])
def test_n_banded_rates_bound_every_reachable_bin(oracle, g0, which):
    """N1-N4 by brute force on the kinematics: from any energy of band k, under any acceleration of class j (any
    direction), after any time up to dtmax[k][j], the total rate of the bin the electron is in does not exceed nu[k][j]."""
    g = g0 if which == "g0" else _sawtooth_gas()
    a2e, nu, dtm, shift = oracle.majorant(g)
    K, J1 = nu.shape
    J = J1 - 1
    nb, de = g.n_bins, g.e_max / g.n_bins
    nu_tot = g.cum_rate[:, -1]
    mx = nu_tot.max()
    assert K == (nb + (1 << shift) - 1) >> shift and len(a2e) == J
    assert np.all(nu <= mx * (1 + 1e-15)) and np.allclose(nu[:, J], mx) and np.allclose(nu[K - 1], mx)
    assert np.all(np.isinf(dtm[:, J])) and np.all(np.isinf(dtm[K - 1]))
    assert np.all(a2e[1:] / a2e[:-1] == 2.0) and np.isclose(np.sqrt(a2e[0]), KAPPA * 250.0, rtol=1e-15)
    assert (nu[: K // 2, : J // 2] < 0.8 * mx).mean() > 0.5, "the table buys nothing"
    rng = np.random.default_rng(70)
    n = 400000
    k = rng.integers(0, K - 1, n)
    j = rng.integers(0, J, n)
    b_lo, b_hi = k << shift, np.minimum((k + 1) << shift, nb) - 1
    frac = rng.uniform(0, 1, n); frac[: n // 4] = 1.0 - 1e-12          # a quarter of the samples at the band's upper edge
    eps = (b_lo + frac * (b_hi + 1 - b_lo)) * de
    eps = np.where((eps * (nb / g.e_max)).astype(np.int64) > b_hi, np.nextafter(eps, 0), eps)
    assert np.all((eps * (nb / g.e_max)).astype(np.int64) >> shift == k)
    A = np.sqrt(a2e[j]) * np.where(rng.uniform(size=n) < 0.5, 1.0, rng.uniform(0, 1, n))   # half at the class edge
    kd = rng.normal(size=(3, n)); kd /= np.linalg.norm(kd, axis=0)
    ad = rng.normal(size=(3, n)); ad /= np.linalg.norm(ad, axis=0)
    par = rng.uniform(size=n) < 0.4
    ad = np.where(par, kd, ad)                                          # 40 %: acceleration along the velocity (the worst case)
    dt = dtm[k, j] * np.where(rng.uniform(size=n) < 0.5, 1.0, rng.uniform(0, 1, n))
    v1 = C2 * np.sqrt(eps) * kd + A * ad * dt
    e1 = (v1 * v1).sum(0) * INV_C2SQ
    b1 = np.minimum(nb - 1, (e1 * (nb / g.e_max)).astype(np.int64))
    assert np.all(nu_tot[b1] <= nu[k, j]), "a reachable bin's total rate exceeds the band's null-collision rate"
    # and the bound is not slack by construction only: somewhere the reached rate comes close to it
    assert (nu_tot[b1] / nu[k, j]).max() > 0.9


@pytest.mark.parametrize("E,e_lo,e_hi", [((0.0, 0.0, -30000.0), 1.30, 1.40), ((3000.0, -4000.0, 0.0), 3.85, 3.95),
                                          ((0.0, 0.0, -1000.0), 6.45, 6.50)])
def test_n_banded_flight_time_cut_and_acceptance(oracle, g0, E, e_lo, e_hi):
    """N5, N6 and C2 per band: dt = min(-ln(u1) / nu[k][j], dtmax[k][j]) with k the band of the energy at the start of the
    step and j the class of |a| = kappa |E| (the whole vector, not a component); a cut flight is a null collision whatever
    u2; an uncut one is real with probability nu_tot(bin reached) / nu[k][j]."""
    a2e, nu, dtm, shift = oracle.majorant(g0)
    rng = np.random.default_rng(71)
    n = 60000
    kd = rng.normal(size=(3, n)); kd /= np.linalg.norm(kd, axis=0)
    st = np.zeros((8, n))
    st[3] = rng.uniform(0, 1e-3, n)
    st[4] = rng.uniform(e_lo, e_hi, n)
    st[5:8] = kd
    ids = np.arange(n, dtype=np.uint64) + 77
    nidx = np.full(n, 11, dtype=np.uint32)
    res = oracle.step_batch(g0, _open_field(E), 9, st, ids, nidx, flags=oracle.BANDED)
    ref = oracle.step_batch(g0, _open_field(E), 9, st, ids, nidx)
    inv_de = g0.n_bins / g0.e_max
    k = (st[4] * inv_de).astype(np.int64) >> shift
    a2 = sum((KAPPA * c) ** 2 for c in E)
    j = _class_of(a2e, a2)
    assert 0 < j < len(a2e) and a2e[j - 1] < a2 <= a2e[j]
    nu_k, dt_k = nu[k, j], dtm[k, j]
    assert np.all(nu_k < 0.8 * g0.resolved_nu_hat())                   # banding is at work here
    u1 = np.array([oracle.uniform_pair(9, int(i), 11, 0)[0] for i in ids[:400]])
    dt = res.state[3] - st[3]
    want = np.minimum(-np.log(u1) / nu_k[:400], dt_k[:400])
    assert np.allclose(dt[:400], want, rtol=1e-11, atol=1e-18)
    assert np.all(dt <= dt_k * (1 + 1e-12))
    cut = dt >= dt_k * (1 - 1e-12)
    m = nu_k * dt_k
    assert abs(cut.sum() - np.exp(-m).sum()) < 4.5 * np.sqrt((np.exp(-m) * (1 - np.exp(-m))).sum()) + 1
    assert np.all(res.event[cut] == -1) and np.all(res.status == 0)
    # every step consumes one collision index, the global mode's flights are shorter by the ratio of the rates
    dt_ref = ref.state[3] - st[3]
    assert np.allclose(dt[~cut] * nu_k[~cut], dt_ref[~cut] * g0.resolved_nu_hat(), rtol=1e-11)
    # uncut flights: KS of dt nu against the exponential truncated at m, and acceptance = nu_tot(bin') / nu
    if (~cut).sum() > 2000:
        x = (dt * nu_k)[~cut]
        mm = m[~cut]
        cdf = (1 - np.exp(-x)) / (1 - np.exp(-mm))
        assert stats.kstest(cdf, "uniform").pvalue > 1e-3
    p_real = g0.cum_rate[res.bin[~cut], -1] / nu_k[~cut]
    assert np.all(p_real <= 1.0)
    real = (res.event[~cut] >= 0).sum()
    assert abs(real - p_real.sum()) < 4.5 * np.sqrt((p_real * (1 - p_real)).sum())


def test_n_banded_yule_furry_with_energy_dependent_total_rate(oracle):
    """C13 under banding: constant ionisation rate nu_i (threshold 0) next to an elastic rate that goes up and down with
    energy, in a field that changes the energy during every flight.  The avalanche size at t_max must still be exactly
    Yule-Furry with nbar = exp(nu_i t_max): a band whose rate were used with the wrong acceptance ratio, a cut flight that
    collided, or a dropped / doubled flight segment all shift the ionisation rate."""
    g = _sawtooth_gas()
    nu_i, t_max, n_p = 5.0, 0.4, 6000
    f = _open_field((0.0, 0.0, -8000.0))
    p = primaries.isotropic_primaries(n_p, 44, e_scale=20.0)
    r = oracle.run(g, f, p, seed=44, t_max=t_max, capacity=1 << 18, n_threads=8, flags=oracle.BANDED)
    r0 = oracle.run(g, f, p[:1500], seed=44, t_max=t_max, capacity=1 << 18, n_threads=8)
    assert r.n_rate_violations == 0 and np.all(r.status == 6)
    size = r.per_avalanche[:, 0].astype(np.int64)
    nbar = np.exp(nu_i * t_max)
    assert abs(size.mean() - nbar) < 4 * np.sqrt(nbar * (nbar - 1) / n_p)
    q = 1 - 1 / nbar
    edges = np.array([1, 2, 3, 4, 5, 6, 8, 10, 13, 17, 22, 30, 10 ** 9])
    obs = np.histogram(size, bins=edges)[0]
    exp = n_p * (q ** (edges[:-1] - 1) - q ** (edges[1:] - 1))
    assert stats.chisquare(obs, exp * obs.sum() / exp.sum()).pvalue > 1e-3
    # banding was at work: fewer steps per real collision than with the global rate
    L = g.n_levels
    spr = float(r.tallies_u64[L + 3]) / float(r.tallies_u64[L + 1])
    spr0 = float(r0.tallies_u64[L + 3]) / float(r0.tallies_u64[L + 1])
    assert spr < 0.85 * spr0, (spr, spr0)
    # bookkeeping: every step is null (cut flights included), real, or the electron's last
    t = r.tallies_u64
    assert t[L] + t[L + 1] + (r.n_steps > 0).sum() == t[L + 3] == r.n_steps.sum()


def _stats(r, L):
    gain = r.per_avalanche[:, 0].astype(float)
    t = r.tallies_u64
    W = r.tallies_f64[2] / r.tallies_f64[3]
    alpha = (float(t[14] + t[15]) - float(t[16])) / r.tallies_f64[2]
    return gain.mean(), gain.std(ddof=1) / np.sqrt(len(gain)), W, alpha, float(t[L + 1]) / r.tallies_f64[3]


def test_n_banded_invariance_g0(oracle, g0):
    """C3 for the banded rate: gain, drift velocity, Townsend alpha and the real-collision rate of gas G0 at 45 kV/cm are
    those of the global rate (independent streams: within sampling errors), with fewer null steps."""
    f = fields.uniform_gap((0, 0, -45000.0), 0.0, 80e-4)
    p = primaries.isotropic_primaries(1500, 61, forward=True)
    p[:, 2] = 2e-4
    a = oracle.run(g0, f, p, seed=61, capacity=1 << 20, n_threads=8)
    b = oracle.run(g0, f, p, seed=63, capacity=1 << 20, n_threads=8, flags=oracle.BANDED)
    L = g0.n_levels
    assert b.n_rate_violations == 0
    ga, sa, Wa, aa, na = _stats(a, L)
    gb, sb, Wb, ab, nb = _stats(b, L)
    assert abs(ga - gb) < 3.5 * np.hypot(sa, sb), (ga, gb, sa, sb)
    assert abs(Wb / Wa - 1) < 0.01 and abs(nb / na - 1) < 0.01, (Wa, Wb, na, nb)
    assert abs(ab / aa - 1) < 0.04, (aa, ab)
    null_per_real_a = float(a.tallies_u64[L]) / float(a.tallies_u64[L + 1])
    null_per_real_b = float(b.tallies_u64[L]) / float(b.tallies_u64[L + 1])
    assert null_per_real_b < 0.75 * null_per_real_a, (null_per_real_a, null_per_real_b)
    # charge conservation (C11) holds as before
    assert b.n == len(p) + int(b.tallies_u64[14] + b.tallies_u64[15])
    assert (b.status == 5).sum() == int(b.tallies_u64[16])


def test_n_banded_drift_in_magnetic_field(oracle, g0):
    """Config-3-like (1 kV/cm, 1 T at 30 degrees): the drift velocity vector and the endpoint energies of the banded run
    are those of the global run within 3.5 combined SE per component, with less than a third of the steps."""
    f = fields.uniform_gap((0, 0, -1000.0), -BIG, BIG, (0.0, 0.5, 0.8660254037844387))
    p = primaries.isotropic_primaries(3000, 7)
    out = []
    for fl, seed in ((0, 7), (oracle.BANDED, 8)):
        r = oracle.run(g0, f, p, seed=seed, t_max=6.0, n_threads=16, flags=fl)
        ok = r.status == 6
        v = (r.end[0:3, ok] - r.birth[0:3, ok]) / (r.end[3, ok] - r.birth[3, ok])
        out.append((v.mean(1), v.std(1, ddof=1) / np.sqrt(ok.sum()), r.end[4, ok].mean(),
                    r.end[4, ok].std(ddof=1) / np.sqrt(ok.sum()), float(r.tallies_u64[g0.n_levels + 3]), r.n_rate_violations))
    (va, sa, ea, sea, na, _), (vb, sb, eb, seb, nb, viol) = out
    assert viol == 0
    assert np.all(np.abs(va - vb) < 3.5 * np.hypot(sa, sb)), (va, vb, sa, sb)
    assert abs(ea - eb) < 3.5 * np.hypot(sea, seb), (ea, eb)
    assert abs(va[2]) > 20 * sa[2] and abs(va[0]) > 3 * sa[0]           # the signal is resolved (drift along z, E x B along x)
    assert nb < na / 3.0, (na, nb)


def test_n_banded_constant_map_equals_uniform_field_per_step(oracle, g0):
    """C15 under banding: a grid map holding one constant field vector gives, step by step, what the uniform slab gives —
    the class comes from the interpolated field at r, the band from the energy at the start of the step."""
    E = (1200.0, -800.0, -21000.0)
    nx, ny, nz = 6, 5, 9
    h = (0.01, 0.012, 0.02)
    origin = (-0.03, -0.03, -0.08)
    nodes = np.zeros((nz, ny, nx, 4), dtype=np.float32)
    nodes[..., 0], nodes[..., 1], nodes[..., 2], nodes[..., 3] = E[0], E[1], E[2], 1.0
    fg = fields.FieldDesc([fields.grid_slab(nodes, origin, h, origin[2], origin[2] + (nz - 1) * h[2])])
    fu = fields.uniform_gap(E, origin[2], origin[2] + (nz - 1) * h[2])
    rng = np.random.default_rng(72)
    n = 20000
    kd = rng.normal(size=(3, n)); kd /= np.linalg.norm(kd, axis=0)
    st = np.zeros((8, n))
    st[0] = rng.uniform(-0.02, 0.01, n); st[1] = rng.uniform(-0.02, 0.01, n); st[2] = rng.uniform(-0.07, 0.07, n)
    st[4] = np.exp(rng.uniform(np.log(0.05), np.log(39.0), n)); st[5:8] = kd
    ids = rng.integers(0, 2 ** 63, n, dtype=np.uint64)
    nidx = rng.integers(0, 1 << 20, n, dtype=np.uint64).astype(np.uint32)
    a = oracle.step_batch(g0, fg, 3, st, ids, nidx, flags=oracle.BANDED)
    b = oracle.step_batch(g0, fu, 3, st, ids, nidx, flags=oracle.BANDED)
    assert np.array_equal(a.event, b.event) and np.array_equal(a.bin, b.bin) and np.array_equal(a.child_id, b.child_id)
    same = a.status == b.status
    assert same.mean() > 0.999                                          # x/y faces exist only in the bc-none grid
    assert np.allclose(a.state[:, same], b.state[:, same], rtol=1e-13, atol=1e-300)
    assert (a.event >= 0).sum() > 1000 and (a.event == -1).sum() > 1000
