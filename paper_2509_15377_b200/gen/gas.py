"""Seeded synthetic gas tables (inputs only — no transport arithmetic lives here).

`gas_g0` is the Ar/CO2 70/30-like table of BASELINE.json config 1 / SURVEY.md §8(d) "Gas G0": 20000 energy
bins over 0-40 eV, 17 levels (2 elastic, 12 excitation, 2 ionisation, 1 attachment), cumulative collision
rates in ns^-1, piecewise constant per bin (value at the bin centre).  The paper's own gas is Magboltz data
that is not available here; this table stands in for it.

The small `*_only` tables are the textbook gases the oracle pins use.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from . import philox

# speed[cm/ns] = C2 * sqrt(energy[eV]);  C2 = c * sqrt(2 / mc^2), c = 29.9792458 cm/ns, mc^2 = 510998.95 eV
C2 = 0.05930969584745753
LOSCHMIDT_293K_1ATM = 2.6867774e19 * (273.15 / 293.15)   # molecules / cm^3

ELASTIC, EXCITATION, IONISATION, ATTACHMENT = 0, 1, 2, 3
GAS_KEY_XOR = 0x47415321
# Excitation amplitude [cm^2].  SURVEY.md §8(d) proposed 2.5e-17 from a numpy-seeded probe and says "rescale once
# and freeze" if the oracle's config-2 forward gain leaves 10^3-10^4: with the Philox-seeded A_k, s_k it did
# (mean forward gain 2.8e4), so the amplitude is frozen at 1.25 x 2.5e-17 (mean forward gain 3.5e3, oracle, seed 0).
EXC_AMPLITUDE = 3.125e-17


@dataclass
class GasTable:
    n_bins: int
    e_max: float
    cum_rate: np.ndarray        # [n_bins, n_levels] float64, ns^-1, non-decreasing along levels
    level_type: np.ndarray      # [n_levels] uint8
    level_loss: np.ndarray      # [n_levels] float64, eV
    level_recoil: np.ndarray    # [n_levels] float64
    level_ob_w: np.ndarray      # [n_levels] float64, eV
    nu_hat: float = 0.0         # <= 0: use max_b cum_rate[b, -1]
    names: list = field(default_factory=list)
    # NEXT-3 extensions, all optional:
    scat_xi: np.ndarray = None             # [n_bins, n_levels] forward-scattering parameter in (-1, 1); None = isotropic
    level_penning_prob: np.ndarray = None  # [n_levels] Penning transfer probability of an excitation level
    level_penning_eV: np.ndarray = None    # [n_levels] energy available to the Penning electron
    kT_eV: float = 0.0                     # gas temperature; 0 = cold gas (R8)

    @property
    def n_levels(self) -> int:
        return int(self.cum_rate.shape[1])

    @property
    def nu_tot(self) -> np.ndarray:
        return self.cum_rate[:, -1]

    def resolved_nu_hat(self) -> float:
        return float(self.nu_hat) if self.nu_hat > 0 else float(self.cum_rate[:, -1].max())

    def level_rates(self) -> np.ndarray:
        return np.diff(self.cum_rate, axis=1, prepend=0.0)


def _finish(n_bins, e_max, rates, types, loss, recoil, w, names, nu_hat=0.0) -> GasTable:
    rates = np.ascontiguousarray(np.asarray(rates, dtype=np.float64))
    cum = np.cumsum(rates, axis=1)
    return GasTable(n_bins, float(e_max), np.ascontiguousarray(cum),
                    np.asarray(types, dtype=np.uint8), np.asarray(loss, dtype=np.float64),
                    np.asarray(recoil, dtype=np.float64), np.asarray(w, dtype=np.float64), float(nu_hat), list(names))


def gas_g0(seed: int = 0, n_bins: int = 20000, e_max: float = 40.0, exc_scale: float = 1.0) -> GasTable:
    """SURVEY.md §8(d) gas G0.  `exc_scale` multiplies EXC_AMPLITUDE (a what-if knob for tests; the configs use 1.0)."""
    de = e_max / n_bins
    lo = np.arange(n_bins, dtype=np.float64) * de            # bin lower edge
    e = (np.arange(n_bins, dtype=np.float64) + 0.5) * de     # bin centre
    n_gas = LOSCHMIDT_293K_1ATM
    f_ar, f_co2 = 0.7, 0.3
    flux = C2 * np.sqrt(e)                                    # cm/ns

    L = 17
    sigma = np.zeros((n_bins, L))
    frac = np.zeros(L)
    types = np.zeros(L, dtype=np.uint8)
    loss = np.zeros(L)
    recoil = np.zeros(L)
    w = np.zeros(L)
    names = [""] * L

    sigma[:, 0] = 1e-16 * (0.15 + np.log(e / 0.23) ** 2) / (1.0 + (e / 25.0) ** 2)
    frac[0], types[0], recoil[0], names[0] = f_ar, ELASTIC, 2.7463945268496799e-05, "Ar elastic"
    sigma[:, 1] = 8e-16 * (e + 0.1) ** -0.4
    frac[1], types[1], recoil[1], names[1] = f_co2, ELASTIC, 2.4929446287114741e-05, "CO2 elastic"

    for k in range(1, 13):
        l = k + 1
        u_a, u_s = philox.uniform_pair(seed, 0, k, 0, key_xor_hi=GAS_KEY_XOR)
        # counter (k,0,0,0): n=k, block=0, id=0
        t_k = 8.0 + 6.0 * (k - 1) / 11.0
        a_k = EXC_AMPLITUDE * exc_scale * (0.5 + float(u_a))
        s_k = 1.0 + 2.0 * float(u_s)
        shape = a_k * (1.0 - np.exp(-((e - t_k) ** 2) / (2.0 * s_k * s_k)))
        sigma[:, l] = np.where(lo >= t_k, shape, 0.0)
        frac[l] = f_ar if l % 2 == 0 else f_co2
        types[l], loss[l] = EXCITATION, t_k
        names[l] = f"{'Ar' if l % 2 == 0 else 'CO2'} excitation {t_k:.3f} eV"

    for l, thr, f, nm in ((14, 15.76, f_ar, "Ar ionisation"), (15, 13.8, f_co2, "CO2 ionisation")):
        sigma[:, l] = np.where(lo >= thr, 4e-16 * (1.0 - thr / e), 0.0)
        frac[l], types[l], loss[l], w[l], names[l] = f, IONISATION, thr, 10.0, nm

    sigma[:, 16] = 4e-21 * np.exp(-((e - 8.0) ** 2) / (2.0 * 0.8 ** 2))
    frac[16], types[16], names[16] = f_co2, ATTACHMENT, "CO2 attachment"

    rates = n_gas * frac[None, :] * sigma * flux[:, None]
    return _finish(n_bins, e_max, rates, types, loss, recoil, w, names)


# ---- textbook gases used by the oracle pins -------------------------------------------------------------

def constant_elastic(nu: float, recoil: float, n_bins: int = 64, e_max: float = 1.0e4, nu_hat: float = 0.0) -> GasTable:
    """One elastic level with energy-independent collision frequency nu [ns^-1] (C5-C8)."""
    rates = np.full((n_bins, 1), nu)
    return _finish(n_bins, e_max, rates, [ELASTIC], [0.0], [recoil], [0.0], ["const elastic"], nu_hat)


def attachment_only(nu_att: float, n_bins: int = 16, e_max: float = 100.0, nu_hat: float = 0.0) -> GasTable:
    rates = np.full((n_bins, 1), nu_att)
    return _finish(n_bins, e_max, rates, [ATTACHMENT], [0.0], [0.0], [0.0], ["attachment"], nu_hat)


def ionisation_only(nu_ion: float, w: float = 10.0, n_bins: int = 16, e_max: float = 1.0e3, nu_hat: float = 0.0) -> GasTable:
    """Threshold-0, energy-independent ionisation: avalanche size at time t is Yule-Furry (C13)."""
    rates = np.full((n_bins, 1), nu_ion)
    return _finish(n_bins, e_max, rates, [IONISATION], [0.0], [0.0], [w], ["ionisation"], nu_hat)


def multi_level_constant(rates_per_level, types, loss=None, recoil=None, w=None, n_bins: int = 32,
                         e_max: float = 100.0, nu_hat: float = 0.0) -> GasTable:
    """Energy-independent rates for several levels (C9 level-selection pin)."""
    L = len(rates_per_level)
    rates = np.tile(np.asarray(rates_per_level, dtype=np.float64)[None, :], (n_bins, 1))
    z = np.zeros(L)
    return _finish(n_bins, e_max, rates, types, z if loss is None else loss, z if recoil is None else recoil,
                   z if w is None else w, [f"level {i}" for i in range(L)], nu_hat)
