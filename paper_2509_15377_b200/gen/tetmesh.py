"""Seeded synthetic unstructured tetrahedral meshes with node potentials (inputs only; NEXT-2).

The paper's field maps are ANSYS finite-element meshes of 10-node tetrahedra (Examples/GEM, Examples/Ansys123)
that are not available here.  This generator stands in for them: a lattice of points jittered by a seeded displacement (so
that no two elements are congruent and no face is axis-aligned), every hexahedral cell cut into six tetrahedra along its
main diagonal (Kuhn's subdivision: faces of neighbouring cells match), one mid-edge node per edge, the potential sampled
from a caller-supplied function at every node, elements flagged solid by their centroid, and optionally elements removed
(an unmeshed electrode).
"""
from __future__ import annotations

import itertools

import numpy as np

from . import philox
from .fields import TetMesh

MESH_KEY_XOR = 0x54455421


def kuhn_mesh(nx: int, ny: int, nz: int, h, potential, seed: int = 0, jitter: float = 0.25, solid=None, removed=None,
              warp=None) -> TetMesh:
    """(nx, ny, nz) lattice points with spacings h = (hx, hy, hz); interior points displaced by jitter x h x (2u - 1), u from
    Philox (the boundary stays flat, so the mesh fills its box).  potential(x, y, z) -> V; solid(x, y, z) -> bool at element
    centroids; removed(x, y, z) -> bool at centroids (those elements are dropped).  warp(x, y, z) -> (x, y, z): an
    orientation-preserving map applied to the jittered lattice points before anything else is derived from them (a GRADED
    mesh: e.g. a piecewise-linear stretch of z puts elements ten times taller next to thin ones); edges stay straight, the
    mid-edge nodes are the midpoints of the warped vertices."""
    hx, hy, hz = (float(v) for v in h)
    K, J, I = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    ids = (K * ny + J) * nx + I
    pts = np.stack([I * hx, J * hy, K * hz], axis=-1).astype(np.float64).reshape(-1, 3)
    n0 = pts.shape[0]
    u = [philox.uniform_pair(seed ^ MESH_KEY_XOR, np.arange(n0, dtype=np.uint64), 0, b)[0] for b in range(3)]
    interior = ((I > 0) & (I < nx - 1) & (J > 0) & (J < ny - 1) & (K > 0) & (K < nz - 1)).reshape(-1)
    for a, hh in enumerate((hx, hy, hz)):
        pts[:, a] += np.where(interior, jitter * hh * (2.0 * u[a] - 1.0), 0.0)
    if warp is not None:
        wx, wy, wz = warp(pts[:, 0], pts[:, 1], pts[:, 2])
        pts = np.stack([wx, wy, wz], axis=1).astype(np.float64)
    # six tetrahedra per cell: the paths from corner 000 to corner 111 along the axes in every order
    tets = []
    base = ids[:-1, :-1, :-1].reshape(-1)
    step = {0: 1, 1: nx, 2: nx * ny}
    for perm in itertools.permutations((0, 1, 2)):
        v = [base]
        for ax in perm:
            v.append(v[-1] + step[ax])
        tets.append(np.stack(v, axis=1))
    tv = np.concatenate(tets, axis=0)
    cen = pts[tv].mean(axis=1)
    if removed is not None:
        keep = ~np.asarray(removed(cen[:, 0], cen[:, 1], cen[:, 2]), dtype=bool)
        tv, cen = tv[keep], cen[keep]
    gas_flag = np.ones(tv.shape[0], dtype=np.uint8)
    if solid is not None:
        gas_flag[np.asarray(solid(cen[:, 0], cen[:, 1], cen[:, 2]), dtype=bool)] = 0
    # orientation: positive volume (swap two vertices where needed)
    a, b, c = pts[tv[:, 0]] - pts[tv[:, 3]], pts[tv[:, 1]] - pts[tv[:, 3]], pts[tv[:, 2]] - pts[tv[:, 3]]
    neg = np.einsum("ij,ij->i", a, np.cross(b, c)) < 0
    tv[neg, 0], tv[neg, 1] = tv[neg, 1].copy(), tv[neg, 0].copy()
    # one mid-edge node per edge
    pairs = [(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)]
    e = np.concatenate([np.sort(tv[:, list(pr)], axis=1) for pr in pairs], axis=0)
    key = e[:, 0].astype(np.int64) * n0 + e[:, 1]
    uniq, inv = np.unique(key, return_inverse=True)
    mid = 0.5 * (pts[uniq // n0] + pts[uniq % n0])
    xyz = np.concatenate([pts, mid], axis=0)
    m = tv.shape[0]
    tn = np.concatenate([tv, (n0 + inv.reshape(6, m).T)], axis=1).astype(np.int32)
    V = np.asarray(potential(xyz[:, 0], xyz[:, 1], xyz[:, 2]), dtype=np.float64)
    return TetMesh(xyz, V, tn, gas_flag)
