"""Plain-data field descriptions shared by both bindings (inputs only; nobody's arithmetic).

Units (SURVEY.md §8 [PIN]): cm, ns, eV, V/cm, tesla.  A field is a stack of z-slabs, sorted by ascending z
and contiguous; each slab is either a uniform field vector or a regular grid of float32 nodes
(Ex, Ey, Ez, gas-mask) laid out [nz][ny][nx][4].  B is one constant vector for the whole run.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

KIND_UNIFORM, KIND_GRID = 0, 1
BC_NONE, BC_PERIODIC, BC_MIRROR = 0, 1, 2
INF = float("inf")


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
