"""Oracle pins, part 1: random numbers and field evaluation (CPU only).

Each test fixes a piece of oracle/avmo.cpp against something that is not the oracle: another library's
Philox (C1), exact closed forms (C15, C16).  Pin ids follow SURVEY.md §8(c) / DESIGN.md §5.
"""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

from paper_2509_15377_b200.gen import fields, philox

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def aten_philox(tmp_path_factory):
    import torch
    inc = os.path.join(os.path.dirname(torch.__file__), "include")
    so = str(tmp_path_factory.mktemp("pins") / "philox_aten.so")
    subprocess.run(["g++", "-O1", "-std=c++17", "-shared", "-fPIC", f"-I{inc}", "-o", so,
                    os.path.join(HERE, "pins", "philox_aten.cpp")], check=True)
    return C.CDLL(so)


def test_c1_philox_matches_aten_engine(oracle, aten_philox):
    """C1: Philox4x32-10 + counter layout (n, block, id_lo, id_hi), key = seed — against ATen's engine."""
    rng = np.random.default_rng(1)
    out = (C.c_uint32 * 4)()
    cases = [(0, 0, 0, 0), (0, 1, 0, 0), (0, 0, 1, 0), (0, 0, 0, 1), (1, 0, 0, 0), (1 << 32, 0, 0, 0),
             (0, 1 << 32, 0, 0), (7, 9, 0xFFFFFFFE, 2), (7, 9, 5, 0xFFFFFFFF), (2 ** 64 - 1, 2 ** 64 - 1, 0xFFFFFFFF, 0xFFFFFFFF)]
    for _ in range(300):
        cases.append((int(rng.integers(0, 2 ** 63)) * 2 + int(rng.integers(0, 2)), int(rng.integers(0, 2 ** 63)) * 2 + 1,
                      int(rng.integers(0, 2 ** 32)), int(rng.integers(0, 4))))
    for seed, ident, n, block in cases:
        aten_philox.aten_philox_block(C.c_uint64(seed), C.c_uint64(ident), C.c_uint32(n), C.c_uint32(block), out)
        assert list(out) == list(oracle.philox(seed, ident, n, block)), (seed, ident, n, block)


def test_c1_generator_philox_matches_oracle(oracle):
    """The input generators' numpy Philox is a third, separate implementation; all three must agree."""
    rng = np.random.default_rng(2)
    ids = rng.integers(0, 2 ** 63, size=200).astype(np.uint64)
    ns = rng.integers(0, 2 ** 32, size=200).astype(np.uint32)
    w = philox.words(12345678901234567, ids, ns, 3)
    ua, ub = philox.uniform_pair(12345678901234567, ids, ns, 3)
    for i in range(200):
        o = oracle.philox(12345678901234567, int(ids[i]), int(ns[i]), 3)
        assert [int(w[j][i]) for j in range(4)] == list(o)
        oa, ob = oracle.uniform_pair(12345678901234567, int(ids[i]), int(ns[i]), 3)
        assert oa == ua[i] and ob == ub[i]


def test_uniforms_open_interval_and_exact():
    """u = ((x >> 12) + 0.5) 2^-52: extreme words stay strictly inside (0,1) and are exact in fp64."""
    lo = philox._to_unit(np.uint32(0), np.uint32(0))
    hi = philox._to_unit(np.uint32(0xFFFFFFFF), np.uint32(0xFFFFFFFF))
    assert lo == 2.0 ** -53 and 0.0 < lo
    assert hi == 1.0 - 2.0 ** -53 and hi < 1.0


def test_uniforms_are_uniform(oracle):
    from scipy import stats
    u = np.array([oracle.uniform_pair(3, i, 17, 0) for i in range(20000)])
    assert stats.kstest(u[:, 0], "uniform").pvalue > 1e-3
    assert stats.kstest(u[:, 1], "uniform").pvalue > 1e-3
    assert abs(np.corrcoef(u[:, 0], u[:, 1])[0, 1]) < 0.03


# ---- field evaluation ---------------------------------------------------------------------------------------

def _poly_nodes(nx, ny, nz, origin, h, coef):
    """Nodes sampled from f_c(x,y,z) = sum coef[c][abc] x^a y^b z^c, a,b,c in {0,1} (a trilinear polynomial)."""
    x = origin[0] + h[0] * np.arange(nx)
    y = origin[1] + h[1] * np.arange(ny)
    z = origin[2] + h[2] * np.arange(nz)
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    nodes = np.zeros((nz, ny, nx, 4))
    for c in range(4):
        k = coef[c]
        nodes[..., c] = (k[0] + k[1] * X + k[2] * Y + k[3] * Z + k[4] * X * Y + k[5] * X * Z + k[6] * Y * Z + k[7] * X * Y * Z)
    return nodes


def _poly_eval(coef, r):
    X, Y, Z = r
    return np.stack([k[0] + k[1] * X + k[2] * Y + k[3] * Z + k[4] * X * Y + k[5] * X * Z + k[6] * Y * Z + k[7] * X * Y * Z
                     for k in coef])


def test_c15_trilinear_reproduces_trilinear_polynomial(oracle):
    """C15: trilinear interpolation is exact on trilinear polynomials (up to the fp32 rounding of the nodes)."""
    rng = np.random.default_rng(3)
    nx, ny, nz = 9, 7, 11
    origin, h = (-0.3, 0.2, -1.0), (0.1, 0.15, 0.2)
    coef = rng.normal(size=(4, 8))
    coef[3] = [2.0, 0, 0, 0, 0, 0, 0, 0]                         # mask channel constant (gas everywhere)
    nodes = _poly_nodes(nx, ny, nz, origin, h, coef)
    slab = fields.grid_slab(nodes, origin, h, origin[2], origin[2] + (nz - 1) * h[2])
    f = fields.FieldDesc([slab])
    n = 4000
    r = np.stack([origin[0] + rng.uniform(0, (nx - 1) * h[0], n), origin[1] + rng.uniform(0, (ny - 1) * h[1], n),
                  origin[2] + rng.uniform(0, (nz - 1) * h[2], n)])
    E, m, sl = oracle.field_eval(f, r)
    ref = _poly_eval(coef, r)
    scale = np.abs(nodes[..., :3]).max()
    assert np.all(sl == 0)
    assert np.abs(E - ref[:3]).max() < 4e-7 * scale              # fp32 node rounding only
    assert np.allclose(m, 2.0)
    # exactly on nodes and on the upper faces (index clamp n-2 with weight 1)
    rn = np.array([[origin[0] + 3 * h[0], origin[0] + (nx - 1) * h[0]], [origin[1] + 2 * h[1], origin[1] + (ny - 1) * h[1]],
                   [origin[2] + 5 * h[2], origin[2] + (nz - 1) * h[2]]])
    E2, _, _ = oracle.field_eval(f, rn)
    assert np.abs(E2 - _poly_eval(coef, rn)[:3]).max() < 4e-7 * scale
    # outside a grid with bc none -> not in domain
    ro = np.array([[origin[0] - 1e-6], [origin[1] + 0.1], [origin[2] + 0.1]])
    assert oracle.field_eval(f, ro)[2][0] == -1


def test_c15_axis_order_and_layout(oracle):
    """A map whose channels are exactly (x, y, z, 1) must return the query point: catches a transposed axis
    or a wrong node stride, which a symmetric polynomial would not."""
    nx, ny, nz = 5, 6, 7
    origin, h = (0.0, 0.0, 0.0), (0.5, 0.25, 0.125)              # exactly representable in fp32
    coef = np.zeros((4, 8)); coef[0][1] = 1; coef[1][2] = 1; coef[2][3] = 1; coef[3][0] = 1
    f = fields.FieldDesc([fields.grid_slab(_poly_nodes(nx, ny, nz, origin, h, coef), origin, h, 0.0, (nz - 1) * h[2])])
    rng = np.random.default_rng(4)
    r = np.stack([rng.uniform(0, 2.0, 500), rng.uniform(0, 1.25, 500), rng.uniform(0, 0.75, 500)])
    E, m, _ = oracle.field_eval(f, r)
    assert np.abs(E - r).max() < 1e-14 and np.abs(m - 1).max() < 1e-15


def test_c16_mirror_and_periodic_fold(oracle):
    """C16 / R15: mirror planes at origin + k P: E(x) -> (-Ex, Ey, Ez)(2P k - x); periodic: E(x + P) = E(x)."""
    rng = np.random.default_rng(5)
    nx, ny, nz = 11, 13, 5
    h = (0.1, 0.1, 0.1)
    origin = (0.05, -0.2, 0.0)
    Px, Py = (nx - 1) * h[0], 1.17                                # Py < grid extent 1.2, not on a node
    nodes = rng.normal(size=(nz, ny, nx, 4)).astype(np.float32)
    nodes[..., 3] = 1.0
    slab = fields.grid_slab(nodes, origin, h, 0.0, 0.4, fields.BC_MIRROR, fields.BC_MIRROR, Px, Py)
    f = fields.FieldDesc([slab])
    n = 2000
    x = origin[0] + rng.uniform(0, Px, n); y = origin[1] + rng.uniform(0, Py, n); z = rng.uniform(0, 0.4, n)
    E0, _, _ = oracle.field_eval(f, np.stack([x, y, z]))
    # shift by 2P (any multiple, either sign): identical
    for kx, ky in ((1, 0), (-2, 3), (5, -4)):
        E1, _, sl = oracle.field_eval(f, np.stack([x + 2 * Px * kx, y + 2 * Py * ky, z]))
        assert np.all(sl == 0) and np.abs(E1 - E0).max() < 1e-9 * np.abs(E0).max() + 1e-9
    # reflect about the plane x = origin: Ex flips, Ey, Ez do not
    E2, _, _ = oracle.field_eval(f, np.stack([2 * origin[0] - x, y, z]))
    assert np.abs(E2[0] + E0[0]).max() < 1e-9 and np.abs(E2[1:] - E0[1:]).max() < 1e-9
    # reflect about the plane y = origin + Py
    E3, _, _ = oracle.field_eval(f, np.stack([x, 2 * (origin[1] + Py) - y, z]))
    assert np.abs(E3[1] + E0[1]).max() < 1e-9 and np.abs(E3[[0, 2]] - E0[[0, 2]]).max() < 1e-9
    # periodic
    slab_p = fields.grid_slab(nodes, origin, h, 0.0, 0.4, fields.BC_PERIODIC, fields.BC_NONE, Px, 0.0)
    fp = fields.FieldDesc([slab_p])
    yy = origin[1] + rng.uniform(0, (ny - 1) * h[1], n)
    Ea, _, _ = oracle.field_eval(fp, np.stack([x, yy, z]))
    Eb, _, _ = oracle.field_eval(fp, np.stack([x - 3 * Px, yy, z]))
    assert np.abs(Ea - Eb).max() < 1e-9


def test_slab_dispatch_and_bounds(oracle):
    """Slabs are picked by z; outside z-range / xy bounds is reported as not-in-domain."""
    s0 = fields.Slab(0.0, 1.0, fields.KIND_UNIFORM, (1.0, 2.0, 3.0))
    s1 = fields.Slab(1.0, 3.0, fields.KIND_UNIFORM, (-4.0, 5.0, 6.0))
    f = fields.FieldDesc([s0, s1], xy_lo=(-1.0, -2.0), xy_hi=(1.0, 2.0))
    r = np.array([[0, 0, 0, 0, 0, 1.5, 0], [0, 0, 0, 0, 0, 0, -2.5], [0.0, 0.999, 1.0, 3.0, 3.0001, 0.5, 0.5]])
    E, m, sl = oracle.field_eval(f, r)
    assert list(sl) == [0, 0, 1, 1, -1, -1, -1]
    assert np.allclose(E[:, 1], [1, 2, 3]) and np.allclose(E[:, 2], [-4, 5, 6])
