"""Synthetic phantoms for the five BASELINE.json configs (SURVEY.md §8(d) recipe).

Every array is indexed [iz][iy][ix] in C order, so the linear voxel index is
ix + nx*(iy + ny*iz) (the C-ABI's layout, include/anm.h).  Densities are rounded
to the 2^-20 g/cm^3 grid of the packed texel BEFORE they are handed out, so the
oracle and the CUDA path see identical values.

`make_config(k, scale=s)` divides the voxel counts by s and multiplies the
spacing by s (same physical extent): the small variants the parity tests use.

Stand-in notice: cfg3/cfg4 replace the paper's private patient PET/CT and
DeepViewer contours; organ NAMES follow Table 1
(PAPER.md:L142-170), shapes and placement are invented here and frozen.
"""
from __future__ import annotations

import numpy as np

from .materials import AIR, LUNG, WATER, BONE

GENERATOR_SEED = 2111
DENSITY_STEP = 2.0 ** -20
DENSITY_STEP_16 = 2.0 ** -12          # cfg4: on this grid a 16-bit texel holds every density exactly (reading C18)

CONFIG_NAMES = ["cfg0_point_sanity", "cfg1_water_validation", "cfg2_slabs",
                "cfg3_patient", "cfg4_fullres"]

# Table 1 order; label id = position + 1
ORGAN_NAMES = [
    "Bladder", "Bowel", "Brain", "Brain_Stem", "Esophagus", "Eye_Left", "Eye_Right", "Heart",
    "Kidney_Left", "Kidney_Right", "Larynx", "Liver", "Lung_Left", "Lung_Right", "Optic_Chiasm",
    "Optical_Nerve_Left", "Optical_Nerve_Right", "Pancreas", "Parotid_Left", "Parotid_Right",
    "Pelvis", "Pituitary", "Rectum", "Spinal_Cord", "Spleen", "Stomach", "Thyroid_Gland",
]
_LABEL = {n: i + 1 for i, n in enumerate(ORGAN_NAMES)}

# (name, centre x,y,z mm, semi-axes a,b,c mm); x left(+)/right(-), y front(-)/back(+), z from the feet,
# in the cfg3 frame (body axis 1600 mm).  Later entries override earlier ones.
_ELLIPSOIDS = [
    ("Brain", 0, 0, 1520, 65, 80, 55), ("Brain_Stem", 0, 25, 1465, 12, 12, 25),
    ("Pituitary", 0, -5, 1490, 5, 5, 5), ("Optic_Chiasm", 0, -15, 1495, 7, 4, 3),
    ("Optical_Nerve_Left", 15, -45, 1495, 3, 18, 3), ("Optical_Nerve_Right", -15, -45, 1495, 3, 18, 3),
    ("Eye_Left", 32, -78, 1495, 12, 12, 12), ("Eye_Right", -32, -78, 1495, 12, 12, 12),
    ("Parotid_Left", 62, 10, 1440, 12, 18, 25), ("Parotid_Right", -62, 10, 1440, 12, 18, 25),
    ("Larynx", 0, -40, 1360, 15, 15, 22), ("Thyroid_Gland", 0, -45, 1325, 22, 10, 15),
    ("Esophagus", 0, 25, 1180, 8, 8, 130), ("Spinal_Cord", 0, 70, 1050, 6, 6, 380),
    ("Lung_Left", 75, 0, 1180, 55, 70, 120), ("Lung_Right", -75, 0, 1180, 55, 70, 120),
    ("Heart", 15, -25, 1130, 45, 40, 55), ("Liver", -70, -10, 985, 75, 65, 70),
    ("Stomach", 60, -30, 965, 40, 35, 50), ("Spleen", 105, 40, 975, 28, 35, 50),
    ("Pancreas", 10, -5, 925, 55, 15, 18), ("Kidney_Left", 60, 50, 895, 25, 22, 50),
    ("Kidney_Right", -60, 50, 895, 25, 22, 50), ("Bowel", 0, -25, 790, 110, 60, 80),
    ("Bladder", 0, -35, 640, 35, 30, 30), ("Rectum", 0, 45, 630, 15, 15, 40),
]
_UPTAKE_FACTOR = {"Brain": 8.0, "Heart": 6.0, "Bladder": 20.0, "Kidney_Left": 3.0, "Kidney_Right": 3.0}
_BODY_A, _BODY_B = 170.0, 110.0
_SPINE = dict(x=0.0, y=70.0, r=20.0, z0=660.0, z1=1440.0)
_PELVIS = dict(ao=140.0, bo=90.0, ai=115.0, bi=68.0, z0=560.0, z1=700.0)
_BODY_Z = 1600.0

# 8.0 mCi injected, scan after 60 min; 18F half-life 109.77 min
TOTAL_ACTIVITY_BQ = 8.0 * 3.7e7 * float(np.exp(-np.log(2.0) * 60.0 / 109.77))


def quantize_density(rho, step=DENSITY_STEP):
    """Densities on the grid both sides are handed (reading C18): multiples of `step` g/cm^3 -- 2^-20, the 32-bit
    texel's grid, or DENSITY_STEP_16 = 2^-12, on which a 16-bit texel holds the value exactly (cfg4)."""
    return (np.round(np.asarray(rho, np.float64) / step) * step).astype(np.float32)


def _patient_params():
    rng = np.random.Generator(np.random.Philox(key=GENERATOR_SEED))
    base_rho = {n: float(rng.uniform(1.00, 1.06)) for n in ORGAN_NAMES}
    uptake = {n: float(np.exp(rng.normal(0.0, 0.5))) * _UPTAKE_FACTOR.get(n, 1.0) for n in ORGAN_NAMES}
    lesions = []
    while len(lesions) < 5:
        x, y, z = rng.uniform(-100, 100), rng.uniform(-50, 50), rng.uniform(750, 1250)
        if (x / (_BODY_A - 12)) ** 2 + (y / (_BODY_B - 12)) ** 2 < 1.0:
            lesions.append((float(x), float(y), float(z)))
    return base_rho, uptake, lesions


def _patient_slice(x, y, z, params):
    """Analytic patient at points (x[None,:], y[:,None]) of one z plane (cfg3 frame, mm).

    Returns material u8, density f64 (no noise), noise flag bool, label u8, activity f32: all [ny][nx].
    """
    base_rho, uptake, lesions = params
    X, Y = np.meshgrid(x, y)                      # [ny][nx]
    shape = X.shape
    body = (X / _BODY_A) ** 2 + (Y / _BODY_B) ** 2 <= 1.0
    mat = np.where(body, WATER, AIR).astype(np.uint8)
    rho = np.where(body, 1.03, 0.0012)
    noisy = body.copy()
    lab = np.zeros(shape, np.uint8)
    act = np.where(body, 1.0, 0.0).astype(np.float32)
    # bones first (structures), organs afterwards
    sp = _SPINE
    if sp["z0"] <= z <= sp["z1"]:
        r = np.sqrt((X - sp["x"]) ** 2 + (Y - sp["y"]) ** 2) / sp["r"]
        m = (r <= 1.0) & body
        mat[m] = BONE
        rho = np.where(m, 1.4 + 0.5 * np.clip((r - 0.5) / 0.5, 0.0, 1.0), rho)
        noisy &= ~m
    pv = _PELVIS
    if pv["z0"] <= z <= pv["z1"]:
        q = np.sqrt((X / pv["ao"]) ** 2 + (Y / pv["bo"]) ** 2)
        m = (q <= 1.0) & ((X / pv["ai"]) ** 2 + (Y / pv["bi"]) ** 2 >= 1.0) & body
        mat[m] = BONE
        rho = np.where(m, 1.4 + 0.5 * np.clip((q - 0.8) / 0.2, 0.0, 1.0), rho)
        noisy &= ~m
        lab[m] = _LABEL["Pelvis"]
        act[m] = uptake["Pelvis"]
    for name, cx, cy, cz, a, b, c in _ELLIPSOIDS:
        dz2 = ((z - cz) / c) ** 2
        if dz2 > 1.0:
            continue
        m = (((X - cx) / a) ** 2 + ((Y - cy) / b) ** 2 + dz2 <= 1.0) & body
        if not m.any():
            continue
        lab[m] = _LABEL[name]
        act[m] = uptake[name]
        if name.startswith("Lung"):
            mat[m] = LUNG
            rho = np.where(m, 0.26, rho)
            noisy &= ~m
        else:
            mat[m] = WATER
            rho = np.where(m, base_rho[name], rho)
            noisy |= m
    for lx, ly, lz in lesions:
        if abs(z - lz) > 10.0:
            continue
        m = ((X - lx) ** 2 + (Y - ly) ** 2 + (z - lz) ** 2 <= 100.0) & body
        act[m] = 15.0
    return mat, rho, noisy, lab, act


def _patient_volume(nx, ny, nz, dx, dy, dz, z_stretch=1.0, with_activity=True, density_step=DENSITY_STEP):
    """Sample the analytic patient on an (nx,ny,nz) grid centred in-plane; z in mm from the grid bottom,
    divided by z_stretch to land in the cfg3 frame."""
    params = _patient_params()
    x = (np.arange(nx) + 0.5) * dx - 0.5 * nx * dx
    y = (np.arange(ny) + 0.5) * dy - 0.5 * ny * dy
    mat = np.empty((nz, ny, nx), np.uint8)
    rho = np.empty((nz, ny, nx), np.float32)
    lab = np.empty((nz, ny, nx), np.uint8)
    act = np.empty((nz, ny, nx), np.float32) if with_activity else None
    for iz in range(nz):
        z = (iz + 0.5) * dz / z_stretch
        m, r, noisy, l, a = _patient_slice(x, y, z, params)
        g = np.random.Generator(np.random.Philox(key=np.array([GENERATOR_SEED, iz], dtype=np.uint64)))
        noise = g.standard_normal(size=r.shape) * 0.02
        r = np.where(noisy, np.maximum(r + noise, 0.9), r)
        mat[iz], rho[iz], lab[iz] = m, quantize_density(r, density_step), l
        if with_activity:
            act[iz] = a
    return mat, rho, lab, act


def _trilinear_activity(nx, ny, nz, dx, dy, dz, z_stretch):
    """cfg4 (reading C21): activity lives on a 192x192x300 PET grid (4 x 4 x 6 mm) centred on the CT
    volume and is sampled trilinearly at the CT voxel centres; zero outside the PET grid."""
    pnx, pny, pnz, pdx, pdy, pdz = 192, 192, 300, 4.0, 4.0, 6.0
    params = _patient_params()
    px = (np.arange(pnx) + 0.5) * pdx - 0.5 * pnx * pdx
    py = (np.arange(pny) + 0.5) * pdy - 0.5 * pny * pdy
    z_off = 0.5 * (pnz * pdz - nz * dz)          # PET grid bottom relative to CT bottom (= 0 for cfg4)
    pet = np.empty((pnz, pny, pnx), np.float32)
    for iz in range(pnz):
        z = ((iz + 0.5) * pdz - z_off) / z_stretch
        pet[iz] = _patient_slice(px, py, z, params)[4] if 0.0 <= z <= _BODY_Z else 0.0

    def axis(n, d, pn, pd, off):
        c = ((np.arange(n) + 0.5) * d + off) / pd - 0.5      # continuous PET index of each CT centre
        i0 = np.floor(c).astype(np.int64)
        w = (c - i0).astype(np.float32)
        valid = (i0 >= 0) & (i0 + 1 < pn)
        return np.clip(i0, 0, pn - 2), w, valid

    ix0, wx, vx = axis(nx, dx, pnx, pdx, 0.5 * (pnx * pdx - nx * dx))
    iy0, wy, vy = axis(ny, dy, pny, pdy, 0.5 * (pny * pdy - ny * dy))
    iz0, wz, vz = axis(nz, dz, pnz, pdz, z_off)
    act = np.zeros((nz, ny, nx), np.float32)
    for iz in range(nz):
        if not vz[iz]:
            continue
        pl = (1.0 - wz[iz]) * pet[iz0[iz]] + wz[iz] * pet[iz0[iz] + 1]           # [pny][pnx]
        rows = (1.0 - wy)[:, None] * pl[iy0] + wy[:, None] * pl[iy0 + 1]         # [ny][pnx]
        sl = (1.0 - wx)[None, :] * rows[:, ix0] + wx[None, :] * rows[:, ix0 + 1]  # [ny][nx]
        sl[~vy, :] = 0.0
        sl[:, ~vx] = 0.0
        act[iz] = sl
    return act


def _radial_shells(n, d_mm, centre_mm, width_mm, n_shells):
    """Label volume of concentric shells around centre_mm (label 1 = innermost), by voxel-centre distance;
    the 'dose-distance curve' of PAPER.md:L109 read out through the organ tally."""
    c = (np.arange(n) + 0.5) * d_mm
    Z, Y, X = np.meshgrid(c - centre_mm[2], c - centre_mm[1], c - centre_mm[0], indexing="ij")
    k = np.floor(np.sqrt(X * X + Y * Y + Z * Z) / width_mm).astype(np.int64) + 1
    return np.where(k <= n_shells, k, 0).astype(np.uint8)


def _base(name, shape_xyz, spacing_mm, n_decays, seed, n_batches, photons_per_decay, positron_ke=0.0):
    return {
        "name": name, "shape": tuple(int(v) for v in shape_xyz),
        "spacing_mm": tuple(float(v) for v in spacing_mm),
        "n_decays": int(n_decays), "seed": int(seed), "n_batches": int(n_batches),
        "photons_per_decay": int(photons_per_decay), "rayleigh_on": 1,
        "photon_cutoff_mev": 0.010, "positron_ke_mev": float(positron_ke),
        "activity": None, "point_source_mm": None, "labels": None, "n_organs": 0,
        "organ_names": [], "total_activity_bq": TOTAL_ACTIVITY_BQ,
    }


def make_patient_on_grid(shape_xyz, spacing_mm, n_decays: int = 1_000_000_000) -> dict:
    """The cfg3 analytic patient sampled on an arbitrary grid (body axis stretched to the grid's height), e.g. the
    paper's PET grid 168 x 168 x 219 at 4.063 x 4.063 x 5 mm."""
    nx, ny, nz = (int(v) for v in shape_xyz)
    sp = tuple(float(v) for v in spacing_mm)
    c = _base("patient_%dx%dx%d" % (nx, ny, nz), (nx, ny, nz), sp, n_decays, 42, 100, 2, positron_ke=0.2498)
    mat, rho, lab, act = _patient_volume(nx, ny, nz, *sp, z_stretch=(nz * sp[2]) / _BODY_Z)
    c.update(material=mat, density=rho, activity=act, labels=lab, n_organs=27, organ_names=list(ORGAN_NAMES))
    c["scale"] = 1
    return c


def make_config(k: int, scale: int = 1) -> dict:
    """Build config k (0..4) of BASELINE.json; `scale` coarsens the grid (tests)."""
    s = int(scale)
    if k == 0:
        n, d = 32 // s, 4.0 * s
        c = _base(CONFIG_NAMES[0], (n, n, n), (d, d, d), 1_000_000, 1, 10, 1)
        c["material"] = np.full((n, n, n), WATER, np.uint8)
        c["density"] = quantize_density(np.full((n, n, n), 1.0))
        c["point_source_mm"] = (64.0, 64.0, 64.0)          # exact centre (a voxel corner, C11)
        c.update(labels=_radial_shells(n, d, (64.0, 64.0, 64.0), 8.0, 8), n_organs=8,
                 organ_names=["shell_%02d" % i for i in range(8)])
    elif k == 1:
        n, d = 100 // s, 2.0 * s
        c = _base(CONFIG_NAMES[1], (n, n, n), (d, d, d), 100_000_000, 1, 100, 1)
        c["material"] = np.full((n, n, n), WATER, np.uint8)
        c["density"] = quantize_density(np.full((n, n, n), 1.0))
        act = np.zeros((n, n, n), np.float32)
        act[n // 2, n // 2, n // 2] = 1.0                   # the paper's construction
        c["activity"] = act
        ctr = ((n // 2 + 0.5) * d,) * 3
        c.update(labels=_radial_shells(n, d, ctr, 4.0, 25), n_organs=25,
                 organ_names=["shell_%02d" % i for i in range(25)])
    elif k == 2:
        n, d = 128 // s, 3.0 * s
        t = n // 4
        c = _base(CONFIG_NAMES[2], (n, n, n), (d, d, d), 100_000_000, 1, 100, 2)
        mat = np.empty((n, n, n), np.uint8)
        rho = np.empty((n, n, n), np.float64)
        lab = np.empty((n, n, n), np.uint8)
        for i, (m, r) in enumerate([(WATER, 1.00), (LUNG, 0.26), (BONE, 1.92), (WATER, 1.00)]):
            mat[i * t:(i + 1) * t], rho[i * t:(i + 1) * t], lab[i * t:(i + 1) * t] = m, r, i + 1
        act = np.zeros((n, n, n), np.float32)
        b0, b1 = (56 * n) // 128, (72 * n) // 128
        act[(8 * n) // 128:(24 * n) // 128, b0:b1, b0:b1] = 1.0
        c.update(material=mat, density=quantize_density(rho), activity=act, labels=lab, n_organs=4,
                 organ_names=["slab_water_0", "slab_lung", "slab_bone", "slab_water_1"])
    elif k == 3:
        nx, ny, nz = 256 // s, 256 // s, 400 // s
        sp = (2.0 * s, 2.0 * s, 4.0 * s)
        c = _base(CONFIG_NAMES[3], (nx, ny, nz), sp, 1_000_000_000, 42, 100, 2, positron_ke=0.2498)
        mat, rho, lab, act = _patient_volume(nx, ny, nz, *sp)
        c.update(material=mat, density=rho, activity=act, labels=lab, n_organs=27,
                 organ_names=list(ORGAN_NAMES))
    elif k == 4:
        nx, ny, nz = 512 // s, 512 // s, 600 // s
        sp = (0.98 * s, 0.98 * s, 3.0 * s)
        c = _base(CONFIG_NAMES[4], (nx, ny, nz), sp, 10_000_000_000, 42, 100, 2, positron_ke=0.2498)
        stretch = (nz * sp[2]) / _BODY_Z
        mat, rho, lab, _ = _patient_volume(nx, ny, nz, *sp, z_stretch=stretch, with_activity=False, density_step=DENSITY_STEP_16)
        act = _trilinear_activity(nx, ny, nz, *sp, z_stretch=stretch)
        c.update(material=mat, density=rho, activity=act, labels=lab, n_organs=27,
                 organ_names=list(ORGAN_NAMES))
    else:
        raise ValueError("config index must be 0..4")
    c["scale"] = s
    return c
