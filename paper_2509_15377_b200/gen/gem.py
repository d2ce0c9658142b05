"""Seeded analytic GEM field map (inputs only — no transport arithmetic lives here).

BASELINE.json config 4: "regular-grid fp32 E-field map of one hexagonal unit cell (pitch 140 um, hole outer 70 um
and inner 50 um double-conical, foil 50 um thick with 5 um metal layers), dV = 400 V across the foil ... Potential
generated from a seeded analytic dipole-sheet model and sampled on a 141 x 245 x 600 grid at 1 um spacing".
Recipe: SURVEY.md §8(d) "GEM map generator", restated in DESIGN.md §3.4.  The paper's own maps are ANSYS
finite-element files of the Garfield++ examples, which are not available; this stands in for them.

Model.  Rectangular cell Lx = 140 um, Ly = sqrt(3) 140 um with holes at the four corners and the centre (hexagonal
lattice, two holes per cell).  Potential

    V = -Ebar z - dE (sqrt(z^2 + h^2) - h) + sum_{k=1..10} dVs S_k(x, y, z - z_k),

Ebar = (E_above + E_below)/2, dE = (E_above - E_below)/2, h = 30 um; ten dipole sheets at z_k = -22.5 ... +22.5 um
(never on a node plane), each a potential jump dVs across the solid part and none across its circular apertures of
radius R_k = 25 + 10 |z_k| / 25 + 0.5 (2 u_k - 1) um (u_k seeded: the only randomness).  Each sheet is a cosine
series over the cell, S_k = 1/2 sign(zeta) sum_{m,n} p_mn cos(2 pi m x/Lx) cos(2 pi n y/Ly) exp(-|G_mn| |zeta|),
p_00 = 1 - 2 pi R^2/(Lx Ly), p_mn = -(1 + (-1)^(m+n)) 2 pi R J1(|G| R)/(|G| Lx Ly), |m| <= 40, |n| <= 70, with
Lanczos factors sinc(m/41) sinc(n/71).  dVs is fixed by V(solid point, z = -30 um) - V(same, +30 um) = dV.
E = -grad V term by term; node mask 0 inside polyimide/copper (R18), else 1; cast to fp32.

Electrons drift toward -z (E_z > 0): the drift region is above the foil (z > 0), induction below.
"""
from __future__ import annotations

import numpy as np
from scipy.special import j1

from . import philox

UM = 1.0e-4                       # cm per micrometre
PITCH_UM = 140.0
LX_UM = PITCH_UM
LY_UM = PITCH_UM * np.sqrt(3.0)   # 242.4871130596428
NX, NY, NZ = 141, 245, 600
Z0_UM = -300.0                    # first node plane; last = +299 um
H_SMOOTH_UM = 30.0
N_SHEETS = 10
M_MAX, N_MAX = 40, 70
KAPTON_HALF_UM, FOIL_HALF_UM = 25.0, 30.0       # R18: polyimide |z| <= 25 um, copper 25 < |z| <= 30 um
R_INNER_UM, R_OUTER_UM = 25.0, 35.0             # hole radii (50 / 70 um are diameters)
SOLID_POINT_UM = (70.0, 40.4)
GEM_KEY_XOR = 0x47454D21


def sheet_planes_um() -> np.ndarray:
    return -22.5 + 5.0 * np.arange(N_SHEETS)


def sheet_radii_um(seed: int) -> np.ndarray:
    """R_k = 25 + 10 |z_k|/25 + 0.5 (2 u_k - 1) um; u_k = first uniform of Philox counter (k, 0, 0, 0) under the
    separate key (seed_lo, seed_hi ^ GEM_KEY_XOR)."""
    k = np.arange(1, N_SHEETS + 1, dtype=np.uint32)
    u, _ = philox.uniform_pair(seed, np.zeros(N_SHEETS, dtype=np.uint64), k, 0, key_xor_hi=GEM_KEY_XOR)
    return R_INNER_UM + (R_OUTER_UM - R_INNER_UM) * np.abs(sheet_planes_um()) / KAPTON_HALF_UM + 0.5 * (2.0 * u - 1.0)


def hole_radius_um(z_um):
    """Hole radius of the foil at height z (R18): double-conical in the polyimide, 35 um in the copper."""
    az = np.abs(z_um)
    return np.where(az <= KAPTON_HALF_UM, R_INNER_UM + (R_OUTER_UM - R_INNER_UM) * az / KAPTON_HALF_UM, R_OUTER_UM)


def _modes():
    m = np.arange(0, M_MAX + 1, dtype=np.float64)
    n = np.arange(0, N_MAX + 1, dtype=np.float64)
    gx = 2.0 * np.pi * m / LX_UM                      # [M]
    gy = 2.0 * np.pi * n / LY_UM                      # [N]
    G = np.sqrt(gx[:, None] ** 2 + gy[None, :] ** 2)  # [M, N]
    mult = np.where(m > 0, 2.0, 1.0)[:, None] * np.where(n > 0, 2.0, 1.0)[None, :]   # (+-m, +-n) folded onto m, n >= 0
    lanczos = np.sinc(m / (M_MAX + 1.0))[:, None] * np.sinc(n / (N_MAX + 1.0))[None, :]
    parity = 1.0 + (-1.0) ** (m[:, None] + n[None, :])
    return gx, gy, G, mult * lanczos, parity


def _sheet_coefficients(radii_um):
    """p_mn per sheet, with multiplicity and Lanczos factors folded in: [K, M, N]."""
    gx, gy, G, weight, parity = _modes()
    area = LX_UM * LY_UM
    out = np.empty((len(radii_um),) + G.shape)
    Gs = np.where(G > 0, G, 1.0)
    for k, R in enumerate(radii_um):
        p = -parity * 2.0 * np.pi * R * j1(Gs * R) / (Gs * area)
        p[0, 0] = 1.0 - 2.0 * np.pi * R * R / area
        out[k] = p * weight
    return out


class GemModel:
    """The analytic potential: evaluates V and E = -grad V on z-planes of the node grid (or at single points)."""

    def __init__(self, e_above: float, e_below: float, dv: float = 400.0, seed: int = 0):
        self.e_above, self.e_below, self.dv, self.seed = float(e_above), float(e_below), float(dv), int(seed)
        self.ebar = 0.5 * (e_above + e_below) * UM          # V/um
        self.de = 0.5 * (e_above - e_below) * UM
        self.zk = sheet_planes_um()
        self.radii = sheet_radii_um(seed)
        self.gx, self.gy, self.G, _, _ = _modes()
        self.p = _sheet_coefficients(self.radii)
        self.dvs = 1.0
        sx, sy = SOLID_POINT_UM
        lo = self.potential_points(np.array([sx]), np.array([sy]), np.array([-FOIL_HALF_UM]), sheets_only=True)[0]
        hi = self.potential_points(np.array([sx]), np.array([sy]), np.array([+FOIL_HALF_UM]), sheets_only=True)[0]
        bg = self._v_background(-FOIL_HALF_UM) - self._v_background(+FOIL_HALF_UM)
        self.dvs = (self.dv - bg) / (lo - hi)               # one linear solve

    def _v_background(self, z_um):
        return -self.ebar * z_um - self.de * (np.sqrt(z_um ** 2 + H_SMOOTH_UM ** 2) - H_SMOOTH_UM)

    def _plane_coefficients(self, z_um):
        """A[m,n] of V_sheets and of dV_sheets/dz on the plane z."""
        zeta = z_um - self.zk                                     # [K]
        decay = np.exp(-self.G[None] * np.abs(zeta)[:, None, None])
        a_v = self.dvs * np.einsum("k,kmn->mn", 0.5 * np.sign(zeta), self.p * decay)
        a_dz = self.dvs * np.einsum("kmn->mn", -0.5 * self.G[None] * self.p * decay)
        return a_v, a_dz

    def potential_points(self, x_um, y_um, z_um, sheets_only=False):
        out = np.empty(len(x_um))
        for i, (x, y, z) in enumerate(zip(x_um, y_um, z_um)):
            a_v, _ = self._plane_coefficients(z)
            v = np.cos(self.gx * x) @ a_v @ np.cos(self.gy * y)
            out[i] = v if sheets_only else v + self._v_background(z)
        return out

    def field_plane(self, x_um, y_um, z_um):
        """(Ex, Ey, Ez) in V/cm on the plane z over the tensor grid x (x) y: arrays [ny, nx]."""
        a_v, a_dz = self._plane_coefficients(z_um)
        cx, sx = np.cos(np.outer(x_um, self.gx)), np.sin(np.outer(x_um, self.gx))      # [nx, M]
        cy, sy = np.cos(np.outer(y_um, self.gy)), np.sin(np.outer(y_um, self.gy))      # [ny, N]
        ex = (sx * self.gx) @ a_v @ cy.T                       # -dV/dx = +sum g_x sin cos
        ey = cx @ a_v @ (sy * self.gy).T
        ez = -(cx @ a_dz @ cy.T) + self.ebar + self.de * z_um / np.sqrt(z_um ** 2 + H_SMOOTH_UM ** 2)
        return ex.T / UM, ey.T / UM, ez.T / UM


def solid_mask(x_um, y_um, z_um):
    """True where (x, y, z) lies inside polyimide or copper (R18).  x, y broadcastable; z scalar."""
    if abs(z_um) > FOIL_HALF_UM:
        return np.zeros(np.broadcast(x_um, y_um).shape, dtype=bool)
    xr = x_um - LX_UM * np.floor(x_um / LX_UM)
    yr = y_um - LY_UM * np.floor(y_um / LY_UM)
    d2 = np.full(np.broadcast(xr, yr).shape, np.inf)
    for cx, cy in ((0.0, 0.0), (LX_UM, 0.0), (0.0, LY_UM), (LX_UM, LY_UM), (0.5 * LX_UM, 0.5 * LY_UM)):
        d2 = np.minimum(d2, (xr - cx) ** 2 + (yr - cy) ** 2)
    return d2 > float(hole_radius_um(z_um)) ** 2


_CACHE: dict = {}


def gem_nodes(e_above: float, e_below: float, dv: float = 400.0, seed: int = 0, nz: int = NZ, z0_um: float = Z0_UM,
              nx: int = NX, ny: int = NY) -> np.ndarray:
    """float32 [nz, ny, nx, 4] = (Ex, Ey, Ez, gas-mask) on the 1 um grid x = 0..nx-1, y = 0..ny-1, z = z0..z0+nz-1 um.
    Cached per argument tuple for the life of the process (331.6 MB at full size)."""
    key = (float(e_above), float(e_below), float(dv), int(seed), nz, float(z0_um), nx, ny)
    if key in _CACHE:
        return _CACHE[key]
    model = GemModel(e_above, e_below, dv, seed)
    x = np.arange(nx, dtype=np.float64)
    y = np.arange(ny, dtype=np.float64)
    nodes = np.empty((nz, ny, nx, 4), dtype=np.float32)
    for k in range(nz):
        z = z0_um + k
        ex, ey, ez = model.field_plane(x, y, z)
        nodes[k, :, :, 0] = ex
        nodes[k, :, :, 1] = ey
        nodes[k, :, :, 2] = ez
        nodes[k, :, :, 3] = np.where(solid_mask(x[None, :], y[:, None], z), 0.0, 1.0)
    _CACHE[key] = nodes
    return nodes
