"""Synthetic CT (HU, int16) and PET (Bq/mL, float32) IMAGES for the image front end.

Input data only (no arithmetic of the method's forward path): the default HU ramp's numbers and a generator that
turns one of the synthetic phantoms of phantoms.py into the pair of images a PET/CT scanner would deliver --
a CT on its own, finer grid ("The CT images are resampled to obtain the same size as the PET
images") and a PET image in Bq/mL on the simulation grid.

Stand-in notice: the paper's patient PET/CT is private clinical data; these images are synthetic.

DEFAULT_HU_RAMP.  The paper cites its "HU-to-density conversion curve [39]" without printing it (a dangling
citation) and names four materials with the references Schneider et al. 2000 and
Kawrakow & Walters 2006.  The default here is a four-segment continuous ramp of that family -- air / lung / soft
tissue (water, as in the paper) / compact bone -- with node values restated from memory of the usual DOSXYZnrc
ctcreate default and therefore APPROXIMATE; it is a parameter of the library (anm_hu_ramp), not a constant of the
method.  include/anm.h's anm_default_hu_ramp holds the same numbers (tests/test_cabi_host.py checks they agree).
"""
from __future__ import annotations

import numpy as np

from .materials import AIR, LUNG, WATER, BONE
from .phantoms import TOTAL_ACTIVITY_BQ, GENERATOR_SEED

DEFAULT_HU_RAMP = {
    "hu": [-1024.0, -974.0, -724.0, 101.0, 1976.0],
    "rho": [0.001, 0.044, 0.302, 1.101, 2.088],
    "material": [AIR, LUNG, WATER, BONE],
    "hu_outside": -1024.0,
}


def _hash_normal(idx: np.ndarray, seed: int) -> np.ndarray:
    """Counter-based N(0,1) per voxel index: two rounds of a 64-bit mix -> two uniforms -> Box-Muller."""
    def mix(v):
        v = (v ^ (v >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        v = (v ^ (v >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return v ^ (v >> np.uint64(31))
    with np.errstate(over="ignore"):
        a = mix(idx.astype(np.uint64) + np.uint64(seed) * np.uint64(0x9E3779B97F4A7C15))
        b = mix(a + np.uint64(0x9E3779B97F4A7C15))
    u1 = ((a >> np.uint64(11)).astype(np.float64) + 0.5) / 2.0 ** 53
    u2 = ((b >> np.uint64(11)).astype(np.float64) + 0.5) / 2.0 ** 53
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


def density_to_hu(rho, material, ramp: dict = DEFAULT_HU_RAMP) -> np.ndarray:
    """The HU a scanner would show for (material, density): the ramp read backwards inside the material's own
    segment (generator only; the forward map is the method's)."""
    rho = np.asarray(rho, np.float64)
    material = np.asarray(material)
    hu_n, rho_n = np.asarray(ramp["hu"], np.float64), np.asarray(ramp["rho"], np.float64)
    out = np.empty(rho.shape, np.float64)
    for k, m in enumerate(ramp["material"]):
        sel = material == m
        r = np.clip(rho[sel], rho_n[k], rho_n[k + 1])
        out[sel] = hu_n[k] + (r - rho_n[k]) / (rho_n[k + 1] - rho_n[k]) * (hu_n[k + 1] - hu_n[k])
    return out


def make_ct_pet(cfg: dict, ct_shape=None, ct_margin_mm=(0.0, 0.0, 0.0), noise_hu: float = 8.0,
                ramp: dict = DEFAULT_HU_RAMP, seed: int = GENERATOR_SEED) -> dict:
    """CT + PET images of the phantom in `cfg` (a make_config dict with an activity map).

    CT: `ct_shape` = (cnx, cny, cnz) voxels (default: 2x finer in x and y, 1.5x in z, rounded) covering the
    simulation grid plus `ct_margin_mm` on every side (so its corner sits at -margin: part of the CT lies outside the
    simulation grid, and with a negative margin part of the grid lies outside the CT).  The HU of a CT voxel is
    that of the phantom voxel containing its centre (air outside), plus N(0, noise_hu) noise hashed from the voxel
    index, rounded to int16 and clipped to [-1024, 3071].
    PET: Bq/mL on the simulation grid (the PET grid IS the simulation grid), scaled so that the
    whole-body activity is TOTAL_ACTIVITY_BQ.
    """
    nx, ny, nz = cfg["shape"]
    sp = cfg["spacing_mm"]
    if ct_shape is None:
        ct_shape = (2 * nx, 2 * ny, int(round(1.5 * nz)))
    ext = [n * d + 2.0 * m for n, d, m in zip((nx, ny, nz), sp, ct_margin_mm)]
    ct_sp = tuple(e / n for e, n in zip(ext, ct_shape))
    ct_off = tuple(-float(m) for m in ct_margin_mm)
    hu_sim = density_to_hu(cfg["density"], cfg["material"], ramp)
    idx = []
    inside = []
    for a in range(3):
        c = ct_off[a] + (np.arange(ct_shape[a]) + 0.5) * ct_sp[a]
        i = np.floor(c / sp[a]).astype(np.int64)
        inside.append((i >= 0) & (i < (nx, ny, nz)[a]))
        idx.append(np.clip(i, 0, (nx, ny, nz)[a] - 1))
    hu = hu_sim[np.ix_(idx[2], idx[1], idx[0])]
    ok = inside[2][:, None, None] & inside[1][None, :, None] & inside[0][None, None, :]
    hu = np.where(ok, hu, float(ramp["hu_outside"]))
    lin = np.arange(hu.size, dtype=np.uint64).reshape(hu.shape)
    hu = hu + noise_hu * _hash_normal(lin, seed + 17)
    hu = np.clip(np.rint(hu), -1024, 3071).astype(np.int16)

    act = np.asarray(cfg["activity"], np.float64)
    vox_ml = sp[0] * sp[1] * sp[2] / 1000.0
    bqml = (act * (TOTAL_ACTIVITY_BQ / act.sum()) / vox_ml).astype(np.float32)
    return {"ct_hu": hu, "ct_shape": tuple(int(v) for v in ct_shape), "ct_spacing_mm": ct_sp, "ct_offset_mm": ct_off,
            "pet_bqml": bqml, "pet_shape": (nx, ny, nz), "pet_spacing_mm": tuple(sp), "pet_offset_mm": (0.0, 0.0, 0.0),
            "ramp": ramp, "total_activity_bq": float(bqml.astype(np.float64).sum() * vox_ml)}
