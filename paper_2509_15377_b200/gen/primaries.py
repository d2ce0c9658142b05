"""Seeded primary electrons (SURVEY.md §8(d) "Primaries").

For p = 0..Np-1: (u_a,u_b) = U(seed, id=p, n=0xFFFFFFFE, block 0), (u_c,u_d) = U(..., block 1),
(u_e,_) = U(..., block 2); direction isotropic from (u_a,u_b), energy u_c * e_scale, t = 0.
Layout: float64 [Np, 8] = x, y, z, t, energy, kx, ky, kz (the boundary's `avm_electron_in`).
"""
from __future__ import annotations

import numpy as np

from . import philox


def isotropic_primaries(n: int, seed: int, pos=(0.0, 0.0, 0.0), e_scale: float = 1.0, id_offset: int = 0,
                        xy_box=None, forward: bool = False) -> np.ndarray:
    ids = np.arange(n, dtype=np.uint64) + np.uint64(id_offset)
    u_a, u_b = philox.uniform_pair(seed, ids, philox.N_PRIMARY, 0)
    u_c, u_d = philox.uniform_pair(seed, ids, philox.N_PRIMARY, 1)
    u_e, _ = philox.uniform_pair(seed, ids, philox.N_PRIMARY, 2)
    out = np.zeros((n, 8), dtype=np.float64)
    out[:, 0], out[:, 1], out[:, 2] = pos
    if xy_box is not None:                     # uniform in [x0,x1] x [y0,y1]
        (x0, x1), (y0, y1) = xy_box
        out[:, 0] = x0 + (x1 - x0) * u_d
        out[:, 1] = y0 + (y1 - y0) * u_e
    out[:, 4] = u_c * e_scale
    st = 2.0 * np.sqrt(u_a * (1.0 - u_a))
    ph = 2.0 * np.pi * u_b
    out[:, 5] = st * np.cos(ph)
    out[:, 6] = st * np.sin(ph)
    out[:, 7] = 1.0 - 2.0 * u_a
    if forward:                                # all launched into +z (C14 pin)
        out[:, 7] = np.abs(out[:, 7])
    return out


def fixed_primaries(n: int, pos=(0.0, 0.0, 0.0), energy: float = 1.0, direction=(0.0, 0.0, 1.0)) -> np.ndarray:
    out = np.zeros((n, 8), dtype=np.float64)
    out[:, 0:3] = pos
    out[:, 4] = energy
    d = np.asarray(direction, dtype=np.float64)
    out[:, 5:8] = d / np.linalg.norm(d)
    return out
