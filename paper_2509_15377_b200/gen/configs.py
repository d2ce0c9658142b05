"""The five BASELINE.json workloads as seeded synthetic inputs.

Inputs only: a gas table, a field description, primaries, a seed and buffer-sizing hints.  The paper's own
workloads are Garfield++'s GEM / triple-GEM examples with ANSYS maps and Magboltz gas, which
are not available; these stand in for them.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from . import fields, gas, primaries

INF = float("inf")


@dataclass
class Workload:
    name: str
    gas: "gas.GasTable"
    field: "fields.FieldDesc"
    primaries: np.ndarray            # [Np, 8]
    seed: int
    t_max: float
    capacity: int                    # electrons ever created (upper bound used to size buffers)
    note: str = ""

    @property
    def n_primaries(self) -> int:
        return int(self.primaries.shape[0])


def config1(n_primaries: int = 1000, seed: int = 0, id_offset: int = 0) -> Workload:
    """Uniform 30 kV/cm, 50 um gap, B = 0, 1000 isotropic primaries at z = 0 (R1: E = (0,0,-E0))."""
    fd = fields.uniform_gap((0.0, 0.0, -30000.0), 0.0, 50e-4)
    p = primaries.isotropic_primaries(n_primaries, seed, id_offset=id_offset)
    return Workload("config1", gas.gas_g0(), fd, p, seed, INF, max(8 * n_primaries, 1 << 14),
                    "uniform E=30 kV/cm, gap 50 um, gas G0, primaries at z=0")


def config2(n_primaries: int = 100, seed: int = 0, id_offset: int = 0) -> Workload:
    """High-gain parallel plate: uniform 60 kV/cm, 128 um gap, B = 0, 100 isotropic primaries at z = 0."""
    fd = fields.uniform_gap((0.0, 0.0, -60000.0), 0.0, 128e-4)
    p = primaries.isotropic_primaries(n_primaries, seed, id_offset=id_offset)
    return Workload("config2", gas.gas_g0(), fd, p, seed, INF, max(4000 * n_primaries, 1 << 16),
                    "uniform E=60 kV/cm, gap 128 um, gas G0, primaries at z=0")


B_CONFIG3 = (0.0, 0.5, 0.8660254037844387)      # 1 T at 30 degrees to the drift axis


def config3(n_primaries: int = 100000, seed: int = 0, t_max: float = INF, id_offset: int = 0) -> Workload:
    """Drift: uniform 1 kV/cm with B = 1 T at 30 degrees, 1 cm gap, primaries at z0 = 0.02 cm (R20)."""
    fd = fields.uniform_gap((0.0, 0.0, -1000.0), 0.0, 1.0, B_CONFIG3)
    p = primaries.isotropic_primaries(n_primaries, seed, pos=(0.0, 0.0, 0.02), id_offset=id_offset)
    return Workload("config3", gas.gas_g0(), fd, p, seed, t_max, max(2 * n_primaries, 1 << 14),
                    "uniform E=1 kV/cm, B=1 T at 30 deg, gap 1 cm, gas G0, primaries at z=0.02 cm")


def replicate(w: Workload, times: int) -> Workload:
    """`times` statistically independent copies of a workload in one batch: copy r uses primary ids
    [r*Np, (r+1)*Np), i.e. different Philox streams (the x64 variant that shows the asymptote)."""
    n = w.n_primaries
    parts = []
    for r in range(times):
        q = w.primaries.copy()
        if r:
            fresh = primaries.isotropic_primaries(n, w.seed, id_offset=r * n)
            q[:, 4:8] = fresh[:, 4:8]            # new direction and energy draws, same start positions
        parts.append(q)
    return Workload(f"{w.name}x{times}", w.gas, w.field, np.concatenate(parts, axis=0), w.seed, w.t_max,
                    w.capacity * times, w.note + f"; {times} independent replicas in one batch")
