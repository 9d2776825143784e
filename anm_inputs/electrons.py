"""Electron stopping-power and range TABLES for the secondary-electron transport (
PAPER.md:L67 "A photon or an electron is transported ... until its energy falls below cutoff energy ... The cutoff
energies for photons and electrons are set to 10 keV and 200 keV").

Input data only.  No electron data of any kind is in the container, so the tables are generated
analytically, like the photon tables: the Bethe collision stopping power for electrons in the Rohrlich-Carlson form
used by ICRU Report 37, without the density-effect correction (a fraction of a percent below 0.5 MeV in these
materials) and without radiative losses (radiation yield ~ 0.1 % at 0.34 MeV in water):

    S_col / rho = 2 pi r_e^2 m c^2 N_A (Z/A) / beta^2 * [ ln( tau^2 (tau + 2) / (2 (I / m c^2)^2) ) + F(tau) ]
    F(tau)      = 1 - beta^2 + [ tau^2 / 8 - (2 tau + 1) ln 2 ] / (tau + 1)^2,      tau = T / m c^2

Mean excitation energies I (eV), the usual ICRU-37 values restated from memory and therefore approximate:
air 85.7, lung 75.3, water 75.0, compact bone 91.9.  Both the oracle and the CUDA path are handed the same arrays;
physical fidelity is approximate and labelled so.

make_electron_tables() returns, on a uniform kinetic-energy grid T_k = T_min + k dT (T_min = the 200 keV electron
cutoff, T_max = 0.512 MeV: a photo-electron takes the whole photon energy E0 = 0.511 MeV; Compton electrons end at 0.3407 MeV):
    stopping[m][k]   S_col/rho at T_k, MeV cm^2 / g
    range[m][k]      residual CSDA range above the cutoff, integral_{T_min}^{T_k} dT / (S_col/rho), g / cm^2
                     (composite Simpson on a 64x finer grid), range[m][0] = 0, increasing.
Both sides read range[m] as a piecewise-linear function of T and invert it as such.
"""
from __future__ import annotations

import numpy as np

from .materials import MATERIALS, ELEMENTS, N_AVOGADRO

MEC2 = 0.51099895                     # MeV
R_E = 2.8179403262e-13                # cm
I_EV = {"air_dry": 85.7, "lung_icrp": 75.3, "water": 75.0, "bone_compact_icru": 91.9}
ELECTRON_CUTOFF_MEV = 0.200
T_MAX_MEV = 0.512                     # >= E0 = 0.51099895 MeV, the largest photo-electron (the Compton edge is 2 E0 / 3)
N_T = 157                             # dT = 2 keV


def z_over_a(mat: dict) -> float:
    return sum(w * ELEMENTS[el][0] / ELEMENTS[el][1] for el, w in mat["w"].items())


def bethe_collision_stopping(T_mev, mat: dict):
    """S_col/rho in MeV cm^2/g (formula in the module docstring)."""
    T = np.asarray(T_mev, np.float64)
    tau = T / MEC2
    beta2 = tau * (tau + 2.0) / (tau + 1.0) ** 2
    I = I_EV[mat["name"]] * 1e-6 / MEC2
    F = 1.0 - beta2 + (tau * tau / 8.0 - (2.0 * tau + 1.0) * np.log(2.0)) / (tau + 1.0) ** 2
    k = 2.0 * np.pi * R_E ** 2 * MEC2 * N_AVOGADRO * z_over_a(mat)
    return k / beta2 * (np.log(tau * tau * (tau + 2.0) / (2.0 * I * I)) + F)


def make_electron_tables() -> dict:
    T = np.linspace(ELECTRON_CUTOFF_MEV, T_MAX_MEV, N_T)
    dT = float(T[1] - T[0])
    nm = len(MATERIALS)
    S = np.empty((nm, N_T), np.float64)
    R = np.zeros((nm, N_T), np.float64)
    sub = 64                                            # Simpson sub-intervals per grid interval (even)
    for m, mat in enumerate(MATERIALS):
        S[m] = bethe_collision_stopping(T, mat)
        for k in range(1, N_T):
            t = np.linspace(T[k - 1], T[k], sub + 1)
            f = 1.0 / bethe_collision_stopping(t, mat)
            h = (T[k] - T[k - 1]) / sub
            R[m, k] = R[m, k - 1] + h / 3.0 * (f[0] + f[-1] + 4.0 * f[1:-1:2].sum() + 2.0 * f[2:-1:2].sum())
    return {"n_materials": nm, "n_t": N_T, "t_min": float(T[0]), "dt": dT,
            "stopping": S.astype(np.float32), "range": R.astype(np.float32)}
