"""Photon cross-section tables, generated analytically.

The paper does not say which photon data library ARCHER uses (PAPER.md:L67 only
names the processes) and none is available in this container, so the tables are
built from closed forms.  Physical fidelity is approximate; parity between the
oracle and the CUDA path is unaffected because both are handed the same arrays.

Layout handed to both sides (all float32, row-major):
  grid       : n_energy points uniform in ln(E/MeV), E from 0.010 to 0.512 MeV,
               lnE_k = lnE_min + k*dlnE; values are interpolated linearly in lnE.
  mu_pe      : [n_materials][n_energy]  photoelectric   mu/rho  (cm^2/g)
  mu_compton : [n_materials][n_energy]  Klein-Nishina   mu/rho  (cm^2/g)
  mu_rayleigh: [n_materials][n_energy]  Rayleigh        mu/rho  (cm^2/g)
  ray_x2     : [n_x2]  momentum-transfer grid x^2 (Angstrom^-2), ray_x2[0] = 0
  ray_cum    : [n_materials][n_x2]  A_m(x^2) = integral_0^{x^2} F_m^2(t) dt,
               per gram up to a constant factor (only ratios are used)
where x = sin(theta/2)/lambda = (E/hc) sin(theta/2).

Models:
  Compton    : electrons/g  x  sigma_KN(E), the closed-form Klein-Nishina total
               cross-section per free electron.
  photoelec. : tau/rho = tau_100 * (0.1 MeV / E)^n, anchors in materials.py.
  Rayleigh   : independent atoms with the screened (hydrogen-like, Thomas-Fermi
               scaled) form factor F(x,Z) = Z / (1 + x^2/x_Z^2)^2,
               x_Z = 0.3 * Z^(1/3) Angstrom^-1; total cross-section
               sigma = pi r_e^2 * integral_{-1}^{1} (1+c^2) F^2(x(c)) dc in closed form.
"""
from __future__ import annotations

import numpy as np

from .materials import MATERIALS, ELEMENTS, N_AVOGADRO, electrons_per_gram

E0_MEV = 0.51099895          # m_e c^2 (MeV): the annihilation photon energy, "0.511 MeV"
R_E_CM = 2.8179403262e-13    # classical electron radius (cm)
HC_KEV_ANGSTROM = 12.398419843

E_MIN_MEV = 0.010            # photon cutoff
E_MAX_MEV = 0.512
N_ENERGY = 512
N_X2 = 256
X2_FIRST = 1.0e-4            # first non-zero grid point of ray_x2 (Angstrom^-2)


def sigma_kn_per_electron(E_mev):
    """Klein-Nishina total cross-section per free electron (cm^2), closed form."""
    a = np.asarray(E_mev, dtype=np.float64) / E0_MEV
    l = np.log1p(2.0 * a)
    t1 = (1.0 + a) / a**2 * (2.0 * (1.0 + a) / (1.0 + 2.0 * a) - l / a)
    t2 = l / (2.0 * a)
    t3 = (1.0 + 3.0 * a) / (1.0 + 2.0 * a) ** 2
    return 2.0 * np.pi * R_E_CM**2 * (t1 + t2 - t3)


def x2_max(E_mev):
    """Largest momentum transfer squared (Angstrom^-2) at photon energy E: (E/hc)^2."""
    return (np.asarray(E_mev, dtype=np.float64) * 1000.0 / HC_KEV_ANGSTROM) ** 2


def _x2_scale(Z: int) -> float:
    return (0.3 * Z ** (1.0 / 3.0)) ** 2      # a = x_Z^2


def _ff2_cum(Z: int, t):
    """integral_0^t Z^2 (1+t'/a)^-4 dt' = Z^2 (a/3) (1 - (1+t/a)^-3)."""
    a = _x2_scale(Z)
    return Z * Z * (a / 3.0) * (1.0 - (1.0 + np.asarray(t, np.float64) / a) ** -3)


def _rayleigh_atom(Z: int, E_mev):
    """Rayleigh cross-section per atom (cm^2) for the screened form factor, closed form.

    sigma = (2 pi r_e^2 / T) * integral_0^T (1+c^2) F^2(t) dt,  c = 1 - 2t/T, T = x_max^2.
    """
    a = _x2_scale(Z)
    T = x2_max(E_mev)
    s = 1.0 + T / a
    i0 = (a / 3.0) * (1.0 - s**-3)
    i1 = a**2 * (1.0 / 6.0 - 0.5 * s**-2 + s**-3 / 3.0)
    i2 = a**3 * (1.0 / 3.0 - 1.0 / s + s**-2 - s**-3 / 3.0)
    integral = Z * Z * (2.0 * i0 - 4.0 * i1 / T + 4.0 * i2 / T**2)
    return 2.0 * np.pi * R_E_CM**2 / T * integral


def energy_grid():
    lnE_min = float(np.log(E_MIN_MEV))
    dlnE = float((np.log(E_MAX_MEV) - np.log(E_MIN_MEV)) / (N_ENERGY - 1))
    E = np.exp(lnE_min + dlnE * np.arange(N_ENERGY))
    return lnE_min, dlnE, E


def make_tables() -> dict:
    """Return the table set as a dict of numpy arrays / scalars (see module docstring)."""
    lnE_min, dlnE, E = energy_grid()
    nm = len(MATERIALS)
    mu_pe = np.zeros((nm, N_ENERGY))
    mu_c = np.zeros((nm, N_ENERGY))
    mu_r = np.zeros((nm, N_ENERGY))
    x2 = np.concatenate([[0.0], np.geomspace(X2_FIRST, float(x2_max(E_MAX_MEV)) * 1.0001, N_X2 - 1)])
    cum = np.zeros((nm, N_X2))
    skn = sigma_kn_per_electron(E)
    for m, mat in enumerate(MATERIALS):
        mu_c[m] = electrons_per_gram(mat) * skn
        mu_pe[m] = mat["pe_tau100"] * (0.1 / E) ** mat["pe_n"]
        for el, w in mat["w"].items():
            Z, A = ELEMENTS[el]
            n_atoms = N_AVOGADRO * w / A
            mu_r[m] += n_atoms * _rayleigh_atom(Z, E)
            cum[m] += (w / A) * _ff2_cum(Z, x2)
        cum[m] /= cum[m, -1]     # only ratios matter; normalise for fp32 headroom
    return {
        "n_materials": nm, "n_energy": N_ENERGY, "lnE_min": lnE_min, "dlnE": dlnE,
        "mu_pe": np.ascontiguousarray(mu_pe, dtype=np.float32),
        "mu_compton": np.ascontiguousarray(mu_c, dtype=np.float32),
        "mu_rayleigh": np.ascontiguousarray(mu_r, dtype=np.float32),
        "n_x2": N_X2,
        "ray_x2": np.ascontiguousarray(x2, dtype=np.float32),
        "ray_cum": np.ascontiguousarray(cum, dtype=np.float32),
    }


def interp_lnE(table_row, E_mev, lnE_min, dlnE):
    """Reference reader of a table row: linear in ln E (used by tests to form expectations)."""
    n = len(table_row)
    t = (np.log(E_mev) - lnE_min) / dlnE
    i = int(np.clip(np.floor(t), 0, n - 2))
    f = t - i
    return float((1.0 - f) * float(table_row[i]) + f * float(table_row[i + 1]))
