"""Synthetic analytic attenuation tables (input data, not transport arithmetic).

BASELINE.json configs[0]: 200-point log grid 10 keV - 3 MeV; Klein-Nishina Compton per electron x Z;
photoelectric 4.5e-33 * Z^4.5 / E^3 cm^2/atom with a x1/7 step below the Ge K-edge (11.1 keV);
pair production 0 below 1.022 MeV.  configs[1]: plus coherent 7.0e-27 * Z^2.5 / E^2 cm^2/atom.
E in MeV for both power laws.  Pair above threshold: SURVEY.md Q2 (synthetic).
The paper itself uses Livermore data, which is not in this container.

Output layout is the one `gadep_set_materials` takes: mu[n_mat][4][n_grid] float32, linear
attenuation in 1/mm; channel order 0 photoelectric, 1 Compton, 2 coherent, 3 pair.
"""
from __future__ import annotations

import numpy as np

N_GRID = 200
E_MIN_MEV = 0.010
E_MAX_MEV = 3.0

M_E_C2 = 0.51099895          # MeV
R_E_CM = 2.8179403262e-13    # classical electron radius, cm
N_A = 6.02214076e23
ALPHA = 1.0 / 137.035999
GE_K_EDGE_MEV = 0.0111

ELEMENTS = {  # symbol: (Z, A [g/mol])
    "H": (1, 1.008), "C": (6, 12.011), "N": (7, 14.007), "O": (8, 15.999),
    "Al": (13, 26.9815385), "Si": (14, 28.085), "Ar": (18, 39.948),
    "Cu": (29, 63.546), "Ge": (32, 72.630),
}

# material id -> (name, density g/cm^3, {element: mass fraction}, is_scoring)
MATERIALS = [
    ("vacuum", 0.0, {}, 0),
    ("Ge_active", 5.323, {"Ge": 1.0}, 1),
    ("Ge_dead", 5.323, {"Ge": 1.0}, 0),
    ("Al", 2.699, {"Al": 1.0}, 0),
    ("Cu", 8.96, {"Cu": 1.0}, 0),
    ("air", 1.2e-3, {"N": 0.7553, "O": 0.2318, "Ar": 0.0129}, 0),
    ("water", 1.0, {"H": 0.11191, "O": 0.88809}, 0),
    ("polypropylene", 0.9, {"C": 0.85628, "H": 0.14372}, 0),
    ("SiO2", 2.0, {"Si": 0.46744, "O": 0.53256}, 0),
]
MAT = {name: i for i, (name, _, _, _) in enumerate(MATERIALS)}
DENSITY_G_CM3 = np.array([rho for (_, rho, _, _) in MATERIALS], dtype=np.float32)   # input of the electron-range mode
MAT_KILL = -1


def energy_grid(n_grid: int = N_GRID, e_min: float = E_MIN_MEV, e_max: float = E_MAX_MEV) -> np.ndarray:
    i = np.arange(n_grid, dtype=np.float64)
    return e_min * (e_max / e_min) ** (i / (n_grid - 1))


def sigma_kn_total(e_mev) -> np.ndarray:
    """Closed-form Klein-Nishina total cross-section per electron [cm^2]."""
    k = np.asarray(e_mev, dtype=np.float64) / M_E_C2
    l = np.log1p(2.0 * k)
    return 2.0 * np.pi * R_E_CM ** 2 * (
        (1.0 + k) / k ** 2 * (2.0 * (1.0 + k) / (1.0 + 2.0 * k) - l / k)
        + l / (2.0 * k) - (1.0 + 3.0 * k) / (1.0 + 2.0 * k) ** 2)


def element_sigmas(symbol: str, e_mev: np.ndarray, coh_coeff: float) -> np.ndarray:
    """Per-atom cross sections [4][G] in cm^2 at the grid energies."""
    z, _ = ELEMENTS[symbol]
    e = np.asarray(e_mev, dtype=np.float64)
    pe = 4.5e-33 * z ** 4.5 / e ** 3
    if symbol == "Ge":
        pe = np.where(e < GE_K_EDGE_MEV, pe / 7.0, pe)
    compton = z * sigma_kn_total(e)
    coh = coh_coeff * z ** 2.5 / e ** 2
    k = e / M_E_C2
    pair = np.where(k > 2.0, ALPHA * R_E_CM ** 2 * z ** 2 * (2.0 * np.pi / 3.0)
                    * (np.maximum(k - 2.0, 0.0) / k) ** 3, 0.0)
    return np.stack([pe, compton, coh, pair], axis=0)


def make_tables(coh_coeff: float = 7.0e-27, n_grid: int = N_GRID):
    """Returns (mu f32[M,4,G] in 1/mm, is_scoring u8[M], grid f64[G])."""
    grid = energy_grid(n_grid)
    mu = np.zeros((len(MATERIALS), 4, n_grid), dtype=np.float64)
    for m, (_, rho, comp, _) in enumerate(MATERIALS):
        for sym, w in comp.items():
            _, a = ELEMENTS[sym]
            mu[m] += rho * N_A * (w / a) * element_sigmas(sym, grid, coh_coeff)
    mu *= 0.1  # 1/cm -> 1/mm
    is_scoring = np.array([s for (_, _, _, s) in MATERIALS], dtype=np.uint8)
    return np.ascontiguousarray(mu, dtype=np.float32), is_scoring, grid
