"""Pins of the GEM map generator (gen/gem.py) and of the oracle's use of it (configs 4 and 5).

The map is an INPUT: these tests fix the recipe against what BASELINE.json config 4 and the mathematics state —
the potential drop across the foil, E = -grad V, the asymptotic drift/induction fields, the hole geometry (R18), the
mirror symmetries the fold (R15) relies on — and check that the oracle reads the node array as laid out.
"""
import numpy as np
import pytest

from paper_2509_15377_b200.gen import configs, fields, gem


@pytest.fixture(scope="module")
def model():
    return gem.GemModel(2000.0, 3000.0, 400.0, 0)


@pytest.fixture(scope="module")
def nodes():
    return gem.gem_nodes(2000.0, 3000.0, 400.0, 0)


def test_potential_drop_across_the_foil_is_400_v(model):
    sx, sy = gem.SOLID_POINT_UM
    v = model.potential_points(np.array([sx, sx]), np.array([sy, sy]), np.array([-30.0, 30.0]))
    assert abs((v[0] - v[1]) - 400.0) < 1e-9
    assert gem.solid_mask(np.array(sx), np.array(sy), 0.0)          # the reference point is in the solid part
    assert model.dvs < 0                                            # potential rises toward -z: electrons go down


def test_field_is_minus_gradient_of_the_potential(model):
    """Central differences of V (independent of the term-by-term derivative used for the nodes)."""
    rng = np.random.default_rng(0)
    n = 40
    x = rng.uniform(0, gem.LX_UM, n); y = rng.uniform(0, gem.LY_UM, n)
    z = rng.uniform(-120, 120, n)
    z = np.where(np.abs(np.abs(z[:, None]) - np.abs(model.zk[None, :])).min(axis=1) < 0.3, z + 0.9, z)  # off the sheets
    d = 1e-3
    for i in range(n):
        ex, ey, ez = model.field_plane(np.array([x[i]]), np.array([y[i]]), z[i])
        gx = (model.potential_points(np.array([x[i] + d]), np.array([y[i]]), np.array([z[i]])) -
              model.potential_points(np.array([x[i] - d]), np.array([y[i]]), np.array([z[i]])))[0] / (2 * d)
        gy = (model.potential_points(np.array([x[i]]), np.array([y[i] + d]), np.array([z[i]])) -
              model.potential_points(np.array([x[i]]), np.array([y[i] - d]), np.array([z[i]])))[0] / (2 * d)
        gz = (model.potential_points(np.array([x[i]]), np.array([y[i]]), np.array([z[i] + d])) -
              model.potential_points(np.array([x[i]]), np.array([y[i]]), np.array([z[i] - d])))[0] / (2 * d)
        got = np.array([ex[0, 0], ey[0, 0], ez[0, 0]]) * gem.UM       # V/um
        ref = -np.array([gx, gy, gz])
        assert np.allclose(got, ref, rtol=2e-5, atol=2e-6 * np.abs(ref).max() + 1e-7), (i, got, ref)


def test_asymptotic_fields_and_hole_field(nodes):
    """2 kV/cm drift above, 3 kV/cm induction below (BASELINE config 4); tens of kV/cm on the hole axis."""
    top, bot = nodes[-1, :, :, :3], nodes[0, :, :, :3]
    assert np.allclose(top[..., 2], 2000.0, rtol=3e-3) and np.allclose(bot[..., 2], 3000.0, rtol=3e-3)
    assert np.abs(top[..., :2]).max() < 1.0 and np.abs(bot[..., :2]).max() < 1.0
    k0 = int(-gem.Z0_UM)                                # z = 0 plane
    assert 4.5e4 < nodes[k0, 121, 70, 2] < 7.0e4        # centre hole
    assert 4.5e4 < nodes[k0, 0, 0, 2] < 7.0e4           # corner hole
    assert np.all(np.isfinite(nodes))


def test_mask_geometry_r18(nodes):
    k0 = int(-gem.Z0_UM)
    m = nodes[..., 3]
    assert set(np.unique(m)) == {0.0, 1.0}
    assert np.all(m[: k0 - 30] == 1.0) and np.all(m[k0 + 31:] == 1.0)       # gas outside |z| <= 30 um
    # along y = 0 from the corner hole centre: radius 25 um at z = 0, 35 um at the polyimide surface and in the copper
    assert m[k0, 0, 25] == 1.0 and m[k0, 0, 26] == 0.0
    assert m[k0 + 25, 0, 35] == 1.0 and m[k0 + 25, 0, 36] == 0.0
    assert m[k0 + 28, 0, 35] == 1.0 and m[k0 + 28, 0, 36] == 0.0 and m[k0 - 30, 0, 36] == 0.0
    assert m[k0 + 12, 0, 29] == 1.0 and m[k0 + 12, 0, 30] == 0.0            # 25 + 10 * 12/25 = 29.8 um
    # open-area fraction of the z = 0 plane = 2 pi 25^2 / (Lx Ly)
    x = np.arange(0, 140, 0.25)[None, :]; y = np.arange(0, gem.LY_UM, 0.25)[:, None]
    open_frac = 1.0 - gem.solid_mask(x, y, 0.0).mean()
    assert abs(open_frac - 2 * np.pi * 25.0 ** 2 / (gem.LX_UM * gem.LY_UM)) < 2e-3


def test_mirror_symmetry_the_fold_relies_on(model, nodes):
    """R15 folds x into [0, P] by reflection: the map must be even in x about 0 and P (Ex odd), likewise y."""
    assert np.abs(nodes[:, :, 0, 0]).max() < 1e-3 and np.abs(nodes[:, :, 140, 0]).max() < 1e-3   # Ex = 0 on the mirrors
    assert np.abs(nodes[:, 0, :, 1]).max() < 1e-3
    assert np.allclose(nodes[:, :, 10, 2], nodes[:, :, 130, 2], atol=1e-2)                      # hexagonal lattice
    x = np.array([13.0]); z = 17.3
    for y in (5.0, 77.7):
        a = model.field_plane(x, np.array([y]), z)
        b = model.field_plane(-x, np.array([y]), z)
        c = model.field_plane(x, np.array([2 * gem.LY_UM - y]), z)
        assert np.isclose(a[0][0, 0], -b[0][0, 0]) and np.isclose(a[2][0, 0], b[2][0, 0])
        assert np.isclose(a[1][0, 0], -c[1][0, 0]) and np.isclose(a[2][0, 0], c[2][0, 0])


def test_sheet_radii_are_seeded_and_bounded():
    r0, r1 = gem.sheet_radii_um(0), gem.sheet_radii_um(1)
    nominal = 25.0 + 10.0 * np.abs(gem.sheet_planes_um()) / 25.0
    assert np.all(np.abs(r0 - nominal) <= 0.5) and np.all(np.abs(r1 - nominal) <= 0.5)
    assert not np.allclose(r0, r1) and np.array_equal(r0, gem.sheet_radii_um(0))


def test_oracle_reads_the_map_as_laid_out(oracle, nodes):
    """Node values are reproduced at node positions, mirror images flip the normal component (config-4 field)."""
    w = configs.config4(n_primaries=4)
    rng = np.random.default_rng(3)
    n = 500
    i = rng.integers(0, gem.NX - 1, n); j = rng.integers(0, 242, n); k = rng.integers(1, gem.NZ - 1, n)
    r = np.vstack([i * gem.UM, j * gem.UM, (gem.Z0_UM + k) * gem.UM]).astype(np.float64)
    E, m, s = oracle.field_eval(w.field, r)
    ref = nodes[k, j, i].astype(np.float64)
    assert np.all(s == 0)
    assert np.allclose(E.T, ref[:, :3], rtol=1e-6, atol=1e-2) and np.allclose(m, ref[:, 3], atol=1e-6)
    # mirror image in x about 0 and a shift by two periods in y
    r2 = r.copy(); r2[0] = -r[0]; r2[1] = r[1] + 2 * 2 * gem.LY_UM * gem.UM
    E2, m2, _ = oracle.field_eval(w.field, r2)
    assert np.allclose(E2[0], -E[0], rtol=1e-6, atol=1e-2) and np.allclose(E2[1:], E[1:], rtol=1e-6, atol=2e-2)


def test_config5_stack_layout():
    w = configs.config5(n_primaries=2)
    s = w.field.slabs
    assert [x.kind for x in s] == [1, 0, 1, 0, 1]
    assert all(s[i].z_hi == s[i + 1].z_lo for i in range(4))
    centres = [0.5 * (s[i].z_lo - configs.GEM_Z_HALF_LO + s[i].z_hi - configs.GEM_Z_HALF_HI) for i in (0, 2, 4)]
    assert np.allclose(np.diff(centres), 2060e-4) and abs(centres[2]) < 1e-12
    assert np.allclose([s[1].z_hi - s[1].z_lo, s[3].z_hi - s[3].z_lo], 1461e-4)
    assert s[1].E == (0.0, 0.0, 3000.0) and np.all(w.primaries[:, 2] == 130e-4)
    assert sum(x.nodes.nbytes for x in s if x.kind == 1) == 3 * 141 * 245 * 600 * 16


def test_config4_oracle_avalanches_conserve_charge(oracle, g0):
    """C11 through the map: endpoints = 1 + ionisations per avalanche; electrons end on the foil (4) or below (1)."""
    w = configs.config4(n_primaries=6)
    r = oracle.run(w.gas, w.field, w.primaries, seed=0, capacity=1 << 14, n_threads=6)
    L = g0.n_levels
    n_ion = int(r.tallies_u64[14] + r.tallies_u64[15])
    assert r.n == 6 + n_ion and int(r.per_avalanche[:, 0].sum()) == r.n
    assert set(np.unique(r.status)) <= {1, 4, 5} and (r.status == 4).sum() > 0
    assert int(r.tallies_u64[L] + r.tallies_u64[L + 1]) > 100000
    assert np.all(r.end[2][r.status == 1] < -300e-4)
    hit = r.status == 4
    assert np.all(np.abs(r.end[2][hit]) < 31e-4)
