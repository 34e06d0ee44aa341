"""Analytic fp32 log-grid cross-section tables (input data for adept_create).

BASELINE.json config 1: "Cross sections are fp32 log-grid tables ... built from
analytic forms (Klein-Nishina total, Bethe-Heitler above 1.022 MeV,
photoelectric ~Z^5/E^3.5, Bethe-Bloch dE/dx, 1/k bremsstrahlung spectrum)".
The forms and constants are DESIGN.md rules T12-T15 (SURVEY.md §8(c) items
12-15).  Everything is evaluated in float64 with numpy and rounded once to
float32; both the oracle and the CUDA library receive the *same* arrays, so
the exact values are inputs, not parity-critical arithmetic.

Units: MeV, mm.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

# physical constants (T15)
MC2 = 0.51099895            # electron rest energy [MeV]
R_E = 2.8179403e-12         # classical electron radius [mm]
ALPHA = 1.0 / 137.035999
N_A = 6.02214076e23
K_BB = 30.7075              # 4 pi N_A r_e^2 mc^2 [MeV mm^2 / mol]
SIGMA_THOMSON = 8.0 * math.pi / 3.0 * R_E * R_E

# quantity indices inside a group
GROUP_GAMMA, GROUP_ELEC = 0, 1
Q_PAIR, Q_COMPT, Q_PHOTO = 0, 1, 2
Q_BREMS, Q_STOP, Q_RANGE = 0, 1, 2


@dataclass(frozen=True)
class Material:
    name: str
    Z: float
    A: float            # g/mol
    rho: float          # g/cm^3
    I_eV: float         # mean excitation energy
    X0: float           # radiation length [mm]

    @property
    def n_atoms(self) -> float:           # atoms / mm^3
        return self.rho * 1e-3 * N_A / self.A


MATERIALS = (
    Material("Pb", 82.0, 207.2, 11.35, 823.0, 5.612),
    Material("lAr", 18.0, 39.948, 1.396, 188.0, 140.0),
)


def klein_nishina_per_electron(E):
    """Textbook Klein-Nishina total cross-section per electron [mm^2]."""
    k = np.asarray(E, dtype=np.float64) / MC2
    l = np.log1p(2.0 * k)
    t1 = (1.0 + k) / (k * k) * (2.0 * (1.0 + k) / (1.0 + 2.0 * k) - l / k)
    t2 = l / (2.0 * k)
    t3 = (1.0 + 3.0 * k) / (1.0 + 2.0 * k) ** 2
    return 2.0 * math.pi * R_E * R_E * (t1 + t2 - t3)


def sigma_compton(mat: Material, E):
    return mat.n_atoms * mat.Z * klein_nishina_per_electron(E)


def sigma_pair(mat: Material, E):
    """Bethe-Heitler: unscreened total over complete-screening total, clamped,
    times the asymptote 7/(9 X0).  Zero for E <= 2 mc^2 (and wherever the
    unscreened form is still negative)."""
    E = np.asarray(E, dtype=np.float64)
    U = (28.0 / 9.0) * np.log(np.maximum(2.0 * E / MC2, 1e-300)) - 218.0 / 27.0
    Sc = (28.0 / 9.0) * math.log(183.0 * mat.Z ** (-1.0 / 3.0)) - 2.0 / 27.0
    v = 7.0 / (9.0 * mat.X0) * np.clip(U / Sc, 0.0, 1.0)
    return np.where(E > 2.0 * MC2, v, 0.0)


def sigma_photo(mat: Material, E):
    E = np.asarray(E, dtype=np.float64)
    return (mat.n_atoms * 4.0 * math.sqrt(2.0) * ALPHA ** 4 * mat.Z ** 5
            * SIGMA_THOMSON * (MC2 / E) ** 3.5)


def _beta2(T):
    gamma = 1.0 + np.asarray(T, dtype=np.float64) / MC2
    return 1.0 - 1.0 / (gamma * gamma)


def _delta_prefactor(mat: Material, T):
    """n Z 2 pi r_e^2 mc^2 / beta^2 [MeV/mm]: prefactor of dSigma/dT_delta = C / T_delta^2."""
    return 0.5 * K_BB * mat.rho * 1e-3 * (mat.Z / mat.A) / _beta2(T)


def sigma_delta(mat: Material, T, e_cut: float):
    """Rule X36: delta-ray production above the cut, the 1/T^2 term common to Moller and Bhabha
    scattering, integrated over [e_cut, T/2]; zero for T <= 2 e_cut."""
    T = np.asarray(T, dtype=np.float64)
    t_max = np.maximum(0.5 * T, e_cut)
    return np.where(T > 2.0 * e_cut, _delta_prefactor(mat, T) * (1.0 / e_cut - 1.0 / t_max), 0.0)


def sigma_annihilation(mat: Material, T):
    """Rule X38: annihilation in flight of a positron of kinetic energy T on an electron at rest,
    Heitler's total cross-section per electron times the electron density [1/mm]."""
    g = 1.0 + np.asarray(T, dtype=np.float64) / MC2
    r = np.sqrt(g * g - 1.0)
    per_e = math.pi * R_E * R_E / (g + 1.0) * ((g * g + 4.0 * g + 1.0) / (g * g - 1.0) * np.log(g + r) - (g + 3.0) / r)
    return mat.n_atoms * mat.Z * per_e


E_SCATTER = 21.2            # Rossi-Greisen scattering energy [MeV]


def sigma_transport(mat: Material, T):
    """Rule X39: transport cross-section of multiple scattering [1/mm], <1 - cos(theta)> per unit path =
    theta_0^2 / 2 with the Rossi-Greisen width theta_0^2 = (E_s / (beta p c))^2 / X0."""
    T = np.asarray(T, dtype=np.float64)
    pc = np.sqrt(T * (T + 2.0 * MC2))
    beta = pc / (T + MC2)
    return (E_SCATTER / (beta * pc)) ** 2 / (2.0 * mat.X0)


def stopping_power(mat: Material, T, e_cut: float, physics: int = 0):
    """Restricted stopping power [MeV/mm]: Bethe-Bloch collision term (no
    density correction) plus the radiative loss to photons below the cut.
    physics 1 (rule X36): minus the energy carried by the delta rays that are
    then produced explicitly, int_{e_cut}^{T/2} T' dSigma = C ln(T / (2 e_cut))."""
    T = np.asarray(T, dtype=np.float64)
    gamma = 1.0 + T / MC2
    beta2 = 1.0 - 1.0 / (gamma * gamma)
    I = mat.I_eV * 1e-6
    col = (K_BB * mat.rho * 1e-3 * (mat.Z / mat.A) / beta2
           * (np.log(2.0 * MC2 * beta2 * gamma * gamma / I) - beta2))
    if physics:
        col = col - np.where(T > 2.0 * e_cut,
                             _delta_prefactor(mat, T) * np.log(np.maximum(0.5 * T, e_cut) / e_cut), 0.0)
    return col + e_cut / mat.X0


def sigma_brems(mat: Material, T, e_cut: float):
    """Integral over k in [e_cut, T] of dSigma/dk = 1/(X0 k)."""
    T = np.asarray(T, dtype=np.float64)
    return np.where(T > e_cut, np.log(np.maximum(T, e_cut) / e_cut) / mat.X0, 0.0)


def csda_range(mat: Material, nodes, e_cut: float, panels: int = 32, physics: int = 0):
    """R(T) = e_cut/S(e_cut) + int_{e_cut}^{T} dT'/S(T') on the table nodes,
    composite Simpson in ln T with `panels` panels per bin."""
    nodes = np.asarray(nodes, dtype=np.float64)
    out = np.empty_like(nodes)
    acc = e_cut / float(stopping_power(mat, e_cut, e_cut, physics))
    prev = e_cut
    for i, T in enumerate(nodes):
        if T > prev:
            lo, hi = math.log(prev), math.log(T)
            x = np.linspace(lo, hi, 2 * panels + 1)
            w = np.ones_like(x)
            w[1:-1:2] = 4.0
            w[2:-1:2] = 2.0
            Tx = np.exp(x)
            acc += float(np.sum(w * Tx / stopping_power(mat, Tx, e_cut, physics))) * (hi - lo) / (6.0 * panels)
            prev = T
        out[i] = acc
    return out


@dataclass
class TableSet:
    """What adept_tables / the oracle receive."""
    n_bins: int
    n_materials: int
    e_min: float
    e_max: float
    e_cut: float
    ln_e_min: np.float32
    inv_dln: np.float32
    nodes: np.ndarray           # float64 [n_bins+1]
    data: np.ndarray            # float32 [mat][group][qty][n_bins+1], C-contiguous
    physics: int = 0            # rule X35: 0 = basic rules; 1 = delta rays (X36), Klein-Nishina sampling (X37), annihilation in flight (X38); 2 = also multiple scattering (X39)
    data_x: np.ndarray | None = None    # physics >= 1: float32 [mat][3][n_bins+1]: Sigma_delta (e+-), Sigma_annihilation (e+), Sigma_transport (e+-)

    def q(self, mat: int, group: int, qty: int) -> np.ndarray:
        return self.data[mat, group, qty]


def build_tables(n_bins: int, e_min: float, e_max: float, e_cut: float,
                 materials=MATERIALS, physics: int = 0) -> TableSet:
    j = np.arange(n_bins + 1, dtype=np.float64)
    nodes = e_min * (e_max / e_min) ** (j / n_bins)
    nodes[0], nodes[-1] = e_min, e_max
    data = np.zeros((len(materials), 2, 3, n_bins + 1), dtype=np.float64)
    for m, mat in enumerate(materials):
        data[m, GROUP_GAMMA, Q_PAIR] = sigma_pair(mat, nodes)
        data[m, GROUP_GAMMA, Q_COMPT] = sigma_compton(mat, nodes)
        data[m, GROUP_GAMMA, Q_PHOTO] = sigma_photo(mat, nodes)
        data[m, GROUP_ELEC, Q_BREMS] = sigma_brems(mat, nodes, e_cut)
        data[m, GROUP_ELEC, Q_STOP] = stopping_power(mat, nodes, e_cut, physics)
        data[m, GROUP_ELEC, Q_RANGE] = csda_range(mat, nodes, e_cut, physics=physics)
    data_x = None
    if physics:
        data_x = np.ascontiguousarray(np.stack([np.stack([sigma_delta(mat, nodes, e_cut), sigma_annihilation(mat, nodes),
                                                          sigma_transport(mat, nodes)])
                                                for mat in materials]).astype(np.float32))
    return TableSet(physics=physics, data_x=data_x,
        n_bins=n_bins, n_materials=len(materials), e_min=e_min, e_max=e_max, e_cut=e_cut,
        ln_e_min=np.float32(math.log(e_min)),
        inv_dln=np.float32(n_bins / math.log(e_max / e_min)),
        nodes=nodes, data=np.ascontiguousarray(data.astype(np.float32)))


def constant_tables(n_bins: int, e_min: float, e_max: float, e_cut: float, *,
                    pair=0.0, compt=0.0, photo=0.0, brems=0.0, stop=0.0, rng=1e30,
                    n_materials: int = 2, physics: int = 0, delta=0.0, annih=0.0, transport=0.0) -> TableSet:
    """Energy-independent tables for closed-form checks (pure absorber,
    vacuum-like geometry tests, brems-only slabs)."""
    j = np.arange(n_bins + 1, dtype=np.float64)
    nodes = e_min * (e_max / e_min) ** (j / n_bins)
    data = np.zeros((n_materials, 2, 3, n_bins + 1), dtype=np.float32)
    data[:, GROUP_GAMMA, Q_PAIR] = pair
    data[:, GROUP_GAMMA, Q_COMPT] = compt
    data[:, GROUP_GAMMA, Q_PHOTO] = photo
    data[:, GROUP_ELEC, Q_BREMS] = brems
    data[:, GROUP_ELEC, Q_STOP] = stop
    data[:, GROUP_ELEC, Q_RANGE] = rng
    data_x = None
    if physics:
        data_x = np.zeros((n_materials, 3, n_bins + 1), dtype=np.float32)
        data_x[:, 0], data_x[:, 1], data_x[:, 2] = delta, annih, transport
    return TableSet(n_bins, n_materials, e_min, e_max, e_cut,
                    np.float32(math.log(e_min)), np.float32(n_bins / math.log(e_max / e_min)),
                    nodes, data, physics, data_x)
