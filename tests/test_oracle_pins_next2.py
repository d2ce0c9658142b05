"""Oracle pins of NEXT-2 (DESIGN.md §3.8 readings F1-F4), CPU only: unstructured maps of 10-node
tetrahedra.  Pinned to what finite-element theory fixes: quadratic elements reproduce any quadratic potential exactly (so
E = -grad V is exact at every point, whatever the mesh), the element found for a point is the one brute force finds, a point
in no element is solid, the tangential field is continuous across faces, and a mesh that carries a LINEAR potential is a
uniform slab: whole avalanches through it are the uniform-slab avalanches."""
import numpy as np
import pytest

from paper_2509_15377_b200.gen import fields, gas, primaries, tetmesh

H = 2e-4


def _quad(a, b, Q):
    V = lambda x, y, z: a + b[0] * x + b[1] * y + b[2] * z + sum(Q[i][j] * (x, y, z)[i] * (x, y, z)[j] for i in range(3) for j in range(3))
    Qs = np.array(Q) + np.array(Q).T
    E = lambda r: -(np.array(b)[:, None] + Qs @ r)
    return V, E


def _mesh_field(mesh, nx, ny, nz, **kw):
    return fields.FieldDesc([fields.tet_slab(mesh, (0.0, 0.0, 0.0), 0.0, (nz - 1) * H, **kw)])


def test_f1_quadratic_elements_reproduce_quadratic_potentials(oracle):
    nx, ny, nz = 9, 8, 10
    V, E = _quad(3.0, (-2000.0, 500.0, 30000.0), [[4e6, -1e6, 2e6], [0, -3e6, 5e5], [0, 0, 7e6]])
    mesh = tetmesh.kuhn_mesh(nx, ny, nz, (H, H, H), V, seed=3)
    assert mesh.tet_nodes.shape == (6 * 8 * 7 * 9, 10) and len(np.unique(mesh.tet_nodes[:, 4:])) == mesh.node_xyz.shape[0] - nx * ny * nz
    fd = _mesh_field(mesh, nx, ny, nz)
    rng = np.random.default_rng(0)
    r = rng.uniform(0, 1, size=(3, 20000)) * np.array([(nx - 1) * H, (ny - 1) * H, (nz - 1) * H])[:, None]
    Eo, m, sl = oracle.field_eval(fd, r)
    assert np.all(sl == 0) and np.all(m == 1.0)
    exact = E(r)
    assert np.abs(Eo - exact).max() < 1e-9 * np.abs(exact).max()
    # mid-edge nodes sit at the midpoints; every element has positive volume
    xyz, tn = mesh.node_xyz, mesh.tet_nodes
    for k, (a, b) in enumerate([(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)]):
        assert np.allclose(xyz[tn[:, 4 + k]], 0.5 * (xyz[tn[:, a]] + xyz[tn[:, b]]), atol=1e-18)
    vol = np.einsum("ij,ij->i", xyz[tn[:, 0]] - xyz[tn[:, 3]], np.cross(xyz[tn[:, 1]] - xyz[tn[:, 3]], xyz[tn[:, 2]] - xyz[tn[:, 3]]))
    assert vol.min() > 0 and abs(vol.sum() / 6 - 8 * 7 * 9 * H ** 3) < 1e-9 * H ** 3 * 500


def _brute_force(mesh, r):
    """Lowest-index element whose barycentric coordinates of r are all >= -1e-10, or -1 (numpy, all elements at once)."""
    xyz, tn = mesh.node_xyz, mesh.tet_nodes
    p3 = xyz[tn[:, 3]]
    T = np.stack([xyz[tn[:, 0]] - p3, xyz[tn[:, 1]] - p3, xyz[tn[:, 2]] - p3], axis=2)      # columns
    lam = np.linalg.solve(T, (r[None, :] - p3)[:, :, None])[:, :, 0]
    ok = (lam.min(axis=1) >= -1e-10) & (1.0 - lam.sum(axis=1) >= -1e-10)
    idx = np.flatnonzero(ok)
    return (int(idx[0]), lam[idx[0]]) if len(idx) else (-1, None)


def test_f2_point_location_matches_brute_force_and_holes_are_solid(oracle):
    """A cubic potential (NOT reproduced exactly: the field differs from element to element, so picking a wrong element
    shows) on a mesh with solid elements and a removed block: material flag and field of the brute-force element."""
    nx, ny, nz = 8, 8, 9
    V = lambda x, y, z: 3e4 * z + 4e9 * x * y * z + 2e9 * z ** 3
    solid = lambda x, y, z: (x - 7e-4) ** 2 + (y - 7e-4) ** 2 < (2.2e-4) ** 2
    removed = lambda x, y, z: (x > 9e-4) & (y < 5e-4) & (z > 6e-4) & (z < 11e-4)
    mesh = tetmesh.kuhn_mesh(nx, ny, nz, (H, H, H), V, seed=5, solid=solid, removed=removed)
    fd = _mesh_field(mesh, nx, ny, nz)
    rng = np.random.default_rng(1)
    n = 600
    r = rng.uniform(0, 1, size=(3, n)) * np.array([(nx - 1) * H, (ny - 1) * H, (nz - 1) * H])[:, None]
    # some points exactly on vertices, edges and faces
    xyz, tn = mesh.node_xyz, mesh.tet_nodes
    r[:, :20] = xyz[tn[:20, 0]].T
    r[:, 20:40] = xyz[tn[100:120, 5]].T
    r[:, 40:60] = ((xyz[tn[200:220, 0]] + xyz[tn[200:220, 1]] + xyz[tn[200:220, 2]]) / 3).T
    Eo, m, sl = oracle.field_eval(fd, r)
    n_hole = n_solid = 0
    from oracle import avmo
    for i in range(n):
        e, lam = _brute_force(mesh, r[:, i])
        if e < 0:
            assert m[i] == 0.0 and np.all(Eo[:, i] == 0.0); n_hole += 1
            continue
        assert m[i] == float(mesh.tet_gas[e]); n_solid += int(mesh.tet_gas[e] == 0)
        # the element's field from the shape functions, written out independently (numpy)
        l4 = np.append(lam, 1.0 - lam.sum())
        P = xyz[tn[e, :4]]
        G = np.linalg.inv(np.vstack([P.T, np.ones(4)]))[:, :3]                     # grad lambda_a = row a
        Vn = mesh.node_V[tn[e]]
        grad = sum(Vn[a] * (4 * l4[a] - 1) * G[a] for a in range(4))
        for k, (a, b) in enumerate([(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)]):
            grad = grad + 4 * Vn[4 + k] * (l4[b] * G[a] + l4[a] * G[b])
        assert np.abs(Eo[:, i] + grad).max() < 1e-8 * np.abs(grad).max(), i
    assert n_hole > 5 and n_solid > 10


def test_f1_tangential_field_is_continuous_across_faces(oracle):
    """P2 elements: V is continuous across a face, hence so is the tangential part of E; the normal part jumps (the
    potential is cubic).  Two points a hair on either side of interior faces."""
    nx = ny = nz = 6
    V = lambda x, y, z: 3e4 * z + 6e9 * x * y * z + 3e9 * x ** 3
    mesh = tetmesh.kuhn_mesh(nx, ny, nz, (H, H, H), V, seed=7)
    fd = _mesh_field(mesh, nx, ny, nz)
    xyz, tn = mesh.node_xyz, mesh.tet_nodes
    rng = np.random.default_rng(2)
    checked = 0
    jumps = []
    for e in rng.choice(len(tn), 150, replace=False):
        a, b, c, d = xyz[tn[e, :4]]
        w = rng.dirichlet([2, 2, 2])
        pf = w[0] * a + w[1] * b + w[2] * c                                          # on the face opposite vertex 3
        nrm = np.cross(b - a, c - a); nrm /= np.linalg.norm(nrm)
        eps = 1e-9
        pts = np.stack([pf + eps * nrm, pf - eps * nrm], axis=1)
        if pts.min() < 1e-6 or pts.max() > (nx - 1) * H - 1e-6:
            continue
        Eo, m, sl = oracle.field_eval(fd, pts)
        dE = Eo[:, 0] - Eo[:, 1]
        tang = dE - (dE @ nrm) * nrm
        assert np.linalg.norm(tang) < 1e-4 * np.linalg.norm(Eo[:, 0]), (e, tang, Eo)
        jumps.append(abs(dE @ nrm) / np.linalg.norm(Eo[:, 0]))
        checked += 1
    assert checked > 80 and np.max(jumps) > 1e-3


def test_f3_linear_potential_mesh_is_a_uniform_slab(oracle, g0):
    """V = E0 z on a jittered mesh: E = (0, 0, -E0) everywhere (P2 reproduces it), so whole avalanches through the mesh are
    the uniform-slab avalanches: same electrons, same step counts, endpoints to rounding; mirror fold in x / y changes
    nothing; an electron that walks into the solid block stops with status 4."""
    nx, ny, nz = 12, 12, 26
    E0 = 30000.0
    mesh = tetmesh.kuhn_mesh(nx, ny, nz, (4 * H, 4 * H, H), lambda x, y, z: E0 * z, seed=9)
    P = 11 * 4 * H
    fm = fields.FieldDesc([fields.tet_slab(mesh, (0.0, 0.0, 0.0), 0.0, 25 * H, fields.BC_MIRROR, fields.BC_PERIODIC, P, P)])
    fu = fields.uniform_gap((0.0, 0.0, -E0), 0.0, 25 * H)
    p = primaries.isotropic_primaries(40, 3, pos=(0.3 * P, 0.6 * P, 0.0))
    a = oracle.run(g0, fu, p, seed=3).sorted_by_id()
    b = oracle.run(g0, fm, p, seed=3).sorted_by_id()
    assert a.n == b.n and a.n > 44 and np.array_equal(a.id, b.id)
    assert np.array_equal(a.n_steps, b.n_steps) and np.array_equal(a.status, b.status)
    assert np.allclose(a.end, b.end, rtol=1e-8, atol=1e-12)
    solid = lambda x, y, z: z > 20 * H
    mesh2 = tetmesh.kuhn_mesh(nx, ny, nz, (4 * H, 4 * H, H), lambda x, y, z: E0 * z, seed=9, solid=solid)
    fs = fields.FieldDesc([fields.tet_slab(mesh2, (0.0, 0.0, 0.0), 0.0, 25 * H, fields.BC_MIRROR, fields.BC_PERIODIC, P, P)])
    c = oracle.run(g0, fs, p, seed=3)
    assert (c.status == 4).sum() > 20 and np.all(c.end[2][c.status == 4] > 19 * H) and (c.status == 2).sum() == 0
