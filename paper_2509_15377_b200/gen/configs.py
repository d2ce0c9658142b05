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


# ---- GEM configs (map recipe in gen/gem.py) ------------------------------------
GEM_Z_HALF_LO, GEM_Z_HALF_HI = -300.0e-4, 299.0e-4        # each map covers -300 ... +299 um about its foil centre
GEM_STACK_PITCH = 2060.0e-4                               # foil centres 2 mm + 60 um apart (config 5)
GEM_START_Z = 130.0e-4                                    # 100 um above the top copper surface (z = +30 um)


def _gem_slab(e_above: float, e_below: float, z_centre: float, seed: int, dv: float = 400.0) -> "fields.Slab":
    from . import gem
    nodes = gem.gem_nodes(e_above, e_below, dv, seed)
    return fields.grid_slab(nodes, (0.0, 0.0, z_centre + gem.Z0_UM * gem.UM), (gem.UM, gem.UM, gem.UM),
                            z_centre + GEM_Z_HALF_LO, z_centre + GEM_Z_HALF_HI,
                            fields.BC_MIRROR, fields.BC_MIRROR, gem.LX_UM * gem.UM, gem.LY_UM * gem.UM)


def _gem_primaries(n: int, seed: int, id_offset: int) -> np.ndarray:
    from . import gem
    return primaries.isotropic_primaries(n, seed, pos=(0.0, 0.0, GEM_START_Z), id_offset=id_offset,
                                         xy_box=((0.0, gem.LX_UM * gem.UM), (0.0, gem.LY_UM * gem.UM)))


def config4(n_primaries: int = 1000, seed: int = 0, id_offset: int = 0, dv: float = 400.0) -> Workload:
    """Single GEM: 141 x 245 x 600 fp32 map at 1 um, dV = 400 V, 2 kV/cm drift above, 3 kV/cm induction below,
    mirror-periodic in x/y; primaries 100 um above the foil, uniform over the cell; electrons move toward -z."""
    fd = fields.FieldDesc([_gem_slab(2000.0, 3000.0, 0.0, seed, dv)])
    return Workload("config4", gas.gas_g0(), fd, _gem_primaries(n_primaries, seed, id_offset), seed, INF,
                    max(256 * n_primaries, 1 << 16),
                    "single GEM map 141x245x600 (331.6 MB), dV=400 V, 2/3 kV/cm, gas G0, primaries 100 um above the foil")


def config5(n_primaries: int = 200, seed: int = 0, id_offset: int = 0, dv: float = 400.0, name: str = "config5") -> Workload:
    """Triple GEM: three maps (2->3, 3->3, 3->3 kV/cm) whose foil centres are 2.06 mm apart, uniform 3 kV/cm transfer
    slabs between them; slabs ascend in z, GEM1 (the first the electrons meet) on top at z = 0."""
    slabs = []
    for i, (ea, eb) in enumerate(((3000.0, 3000.0), (3000.0, 3000.0), (2000.0, 3000.0))):    # GEM3, GEM2, GEM1
        zc = -(2 - i) * GEM_STACK_PITCH
        if slabs:
            slabs.append(fields.Slab(slabs[-1].z_hi, zc + GEM_Z_HALF_LO, fields.KIND_UNIFORM, (0.0, 0.0, 3000.0)))
        slabs.append(_gem_slab(ea, eb, zc, seed + (2 - i), dv))
    fd = fields.FieldDesc(slabs)
    return Workload(name, gas.gas_g0(), fd, _gem_primaries(n_primaries, seed, id_offset), seed, INF,
                    max(200000 * n_primaries, 1 << 20),
                    f"triple GEM: 3 maps 141x245x600 (995 MB), dV={dv:g} V, 3 kV/cm transfer gaps, gas G0, primaries 100 um above GEM1")


HG_DV = 500.0


def config5hg(n_primaries: int = 8, seed: int = 0, id_offset: int = 0) -> Workload:
    """High-gain variant of config 5 (NOT a BASELINE config; D4): the same triple-GEM stack with the three maps
    generated at dV = 500 V instead of 400 V.  BASELINE's config 5 asks for "avalanches of 10^4-10^5 electrons each, stressing
    secondary append, compaction and occupancy"; with the synthetic gas G0 the stated 400 V gives ~200 electrons per primary
    (effective gain 3.6 per GEM), 500 V gives ~17 per GEM: 10^4-10^5 electrons per primary (chosen by the oracle on single
    GEMs: 3.6 / 13 / 37 electrons reach the induction side per primary at 400 / 480 / 540 V)."""
    w = config5(n_primaries, seed, id_offset, HG_DV, "config5hg")
    w.capacity = max(400000 * n_primaries, 1 << 21)
    return w
