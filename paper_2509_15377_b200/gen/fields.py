"""Plain-data field descriptions shared by both bindings (inputs only; nobody's arithmetic).

Units (SURVEY.md §8 [PIN]): cm, ns, eV, V/cm, tesla.  A field is a stack of z-slabs, sorted by ascending z
and contiguous; each slab is either a uniform field vector or a regular grid of float32 nodes
(Ex, Ey, Ez, gas-mask) laid out [nz][ny][nx][4].  B is one constant vector for the whole run.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

KIND_UNIFORM, KIND_GRID, KIND_TETMESH = 0, 1, 2
BC_NONE, BC_PERIODIC, BC_MIRROR = 0, 1, 2
INF = float("inf")


@dataclass
class TetMesh:
    """Unstructured mesh of 10-node (quadratic, straight-edged) tetrahedra with node potentials (NEXT-2; the element type
    of the paper's ANSYS maps).  tet_nodes[e] = 4 vertices, then the mid-edge nodes of edges (0,1) (0,2) (0,3)
    (1,2) (1,3) (2,3).  Coordinates are relative to the slab's origin."""
    node_xyz: np.ndarray        # [n_nodes, 3] float64, cm
    node_V: np.ndarray          # [n_nodes] float64, volt
    tet_nodes: np.ndarray       # [n_tets, 10] int32
    tet_gas: np.ndarray         # [n_tets] uint8: 1 gas, 0 solid


@dataclass
class Slab:
    z_lo: float
    z_hi: float
    kind: int = KIND_UNIFORM
    E: tuple = (0.0, 0.0, 0.0)
    nodes: Optional[np.ndarray] = None       # float32 [nz, ny, nx, 4] (host). Grid slabs only.
    origin: tuple = (0.0, 0.0, 0.0)
    spacing: tuple = (1.0, 1.0, 1.0)
    bc_x: int = BC_NONE
    bc_y: int = BC_NONE
    period_x: float = 0.0
    period_y: float = 0.0
    mesh: Optional[TetMesh] = None           # kind 2

    @property
    def shape(self):
        if self.nodes is None:
            return (0, 0, 0)
        nz, ny, nx, _ = self.nodes.shape
        return (nx, ny, nz)


@dataclass
class FieldDesc:
    slabs: list
    B: tuple = (0.0, 0.0, 0.0)
    xy_lo: tuple = (-INF, -INF)
    xy_hi: tuple = (INF, INF)


def uniform_gap(e_vec, z_lo, z_hi, B=(0.0, 0.0, 0.0)) -> FieldDesc:
    return FieldDesc([Slab(float(z_lo), float(z_hi), KIND_UNIFORM, tuple(float(v) for v in e_vec))],
                     tuple(float(v) for v in B))


def grid_slab(nodes, origin, spacing, z_lo, z_hi, bc_x=BC_NONE, bc_y=BC_NONE, period_x=0.0, period_y=0.0) -> Slab:
    nodes = np.ascontiguousarray(nodes, dtype=np.float32)
    assert nodes.ndim == 4 and nodes.shape[3] == 4
    return Slab(float(z_lo), float(z_hi), KIND_GRID, (0.0, 0.0, 0.0), nodes, tuple(map(float, origin)),
                tuple(map(float, spacing)), int(bc_x), int(bc_y), float(period_x), float(period_y))


def tet_slab(mesh: TetMesh, origin, z_lo, z_hi, bc_x=BC_NONE, bc_y=BC_NONE, period_x=0.0, period_y=0.0) -> Slab:
    return Slab(float(z_lo), float(z_hi), KIND_TETMESH, (0.0, 0.0, 0.0), None, tuple(map(float, origin)), (1.0, 1.0, 1.0),
                int(bc_x), int(bc_y), float(period_x), float(period_y), mesh)
