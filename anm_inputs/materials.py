"""The four phantom materials of PAPER.md:L65 (§2.1): dry air, lung (ICRP),
water, compact bone (ICRU).  The paper names them and gives no numbers; the
elemental mass fractions are the usual ICRU-44 / NIST ones.
Material ids: 0 air, 1 lung, 2 water (also all soft tissue), 3 bone.
"""
from __future__ import annotations

N_AVOGADRO = 6.02214076e23

# Z, A (g/mol)
ELEMENTS = {
    "H": (1, 1.008), "C": (6, 12.011), "N": (7, 14.007), "O": (8, 15.999),
    "Na": (11, 22.990), "Mg": (12, 24.305), "P": (15, 30.974), "S": (16, 32.06),
    "Cl": (17, 35.45), "Ar": (18, 39.948), "K": (19, 39.098), "Ca": (20, 40.078),
}

MATERIALS = [
    {   # 0
        "name": "air_dry",
        "w": {"C": 0.000124, "N": 0.755268, "O": 0.231781, "Ar": 0.012827},
        # photoelectric anchor: tau/rho at 100 keV (cm^2/g) and power-law exponent
        "pe_tau100": 0.0026, "pe_n": 3.25,
    },
    {   # 1
        "name": "lung_icrp",
        "w": {"H": 0.103, "C": 0.105, "N": 0.031, "O": 0.749, "Na": 0.002,
              "P": 0.002, "S": 0.003, "Cl": 0.003, "K": 0.002},
        "pe_tau100": 0.0029, "pe_n": 3.27,
    },
    {   # 2
        "name": "water",
        "w": {"H": 0.111894, "O": 0.888106},
        "pe_tau100": 0.00277, "pe_n": 3.27,
    },
    {   # 3
        "name": "bone_compact_icru",
        "w": {"H": 0.034, "C": 0.155, "N": 0.042, "O": 0.435, "Na": 0.001,
              "Mg": 0.002, "P": 0.103, "S": 0.003, "Ca": 0.225},
        "pe_tau100": 0.026, "pe_n": 3.1,
    },
]
MATERIAL_IDS = {m["name"]: i for i, m in enumerate(MATERIALS)}
AIR, LUNG, WATER, BONE = 0, 1, 2, 3


def electrons_per_gram(mat: dict) -> float:
    """N_A * sum_i w_i Z_i / A_i."""
    return N_AVOGADRO * sum(w * ELEMENTS[el][0] / ELEMENTS[el][1] for el, w in mat["w"].items())
