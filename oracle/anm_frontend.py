"""CPU oracle of the image front end -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this module.  It imports
nothing from paper_2111_11687_b200/ (the CUDA path) and shares no code with it.

What it computes, in fp64 numpy, each step the plain definition written out:

  PAPER.md:L81 (§2.2)  "The CT images are resampled to obtain the same size as the PET images."
      resample_mean(): the value of a destination voxel is the MEAN over that voxel's volume of the source
      image read as a piecewise-constant field (source voxel j covers [off + j d, off + (j+1) d) on each axis);
      whatever part of the destination voxel lies outside the source image counts with `fill`.
      (The paper does not name the resampling kernel; reading C26 takes the volume-weighted mean,
      the one that conserves the integral of the image.)
  PAPER.md:L65 (§2.1)  "The CT images are converted into mass density and material composition using the
      Hounsfield unit (HU)-to-density conversion curve.  ... four materials, each having a density specified
      by the HU ..."
      hu_to_material_density(): a continuous piecewise-linear density ramp over HU nodes, one material per
      HU interval (reading C27).
  PAPER.md:L65  "The PET images indicate the intensity distribution of radionuclides expressed in Bq/mL ...
      The probability density distribution of the decay events ... is constructed through a linear conversion
      of the PET value."
      pet_to_activity(): activity of a voxel [Bq] = concentration [Bq/mL] x voxel volume [mL]; their sum is
      the whole-body activity A(t_s) of Eq. 1.

Arrays are [nz][ny][nx] (x fastest), spacings and offsets are (x, y, z) in mm.
"""
from __future__ import annotations

import numpy as np

DENSITY_STEP = 2.0 ** -20      # g/cm^3: the texel grid of DESIGN.md reading C18


def overlap_weights(n_dst: int, d_dst: float, n_src: int, d_src: float, off_src: float) -> np.ndarray:
    """W[i, j] = length of (destination voxel i  intersect  source voxel j) / d_dst on one axis.

    Destination voxel i spans [i d_dst, (i+1) d_dst); source voxel j spans [off_src + j d_src, off_src + (j+1) d_src).
    Row sums are <= 1; 1 - row sum is the fraction of the destination voxel outside the source image.
    """
    W = np.zeros((n_dst, n_src), np.float64)
    for i in range(n_dst):
        a, b = i * d_dst, (i + 1) * d_dst
        for j in range(n_src):
            lo, hi = off_src + j * d_src, off_src + (j + 1) * d_src
            W[i, j] = max(0.0, min(b, hi) - max(a, lo)) / d_dst
    return W


def resample_mean(src, src_spacing, src_offset, dst_shape, dst_spacing, fill: float) -> np.ndarray:
    """Volume-weighted mean of the piecewise-constant source image over every destination voxel.

    src: [snz][sny][snx]; dst_shape: (nx, ny, nz).  out[k,j,i] = sum_{c,b,a} Wz[k,c] Wy[j,b] Wx[i,a] src[c,b,a]
    + (1 - sum of those weights) * fill.
    """
    src = np.asarray(src, np.float64)
    snz, sny, snx = src.shape
    nx, ny, nz = dst_shape
    Wx = overlap_weights(nx, dst_spacing[0], snx, src_spacing[0], src_offset[0])
    Wy = overlap_weights(ny, dst_spacing[1], sny, src_spacing[1], src_offset[1])
    Wz = overlap_weights(nz, dst_spacing[2], snz, src_spacing[2], src_offset[2])
    out = np.einsum("kc,jb,ia,cba->kji", Wz, Wy, Wx, src, optimize=True)
    inside = np.einsum("k,j,i->kji", Wz.sum(1), Wy.sum(1), Wx.sum(1))
    return out + (1.0 - inside) * fill


def hu_to_material_density(hu, ramp: dict):
    """ramp = {"hu": [h_0 < h_1 < ... < h_{n-1}], "rho": [r_0 .. r_{n-1}], "material": [m_0 .. m_{n-2}]}.

    density(h) = linear interpolation of (hu, rho), clamped to r_0 below h_0 and to r_{n-1} above h_{n-1};
    material(h) = m_k for h in [h_k, h_{k+1}), m_0 below h_0, m_{n-2} at and above h_{n-1}.
    Returns (material uint8, density float64), same shape as hu.
    """
    h = np.asarray(hu, np.float64)
    nodes = np.asarray(ramp["hu"], np.float64)
    rho_n = np.asarray(ramp["rho"], np.float64)
    mats = np.asarray(ramp["material"], np.int64)
    assert nodes.ndim == 1 and nodes.size >= 2 and np.all(np.diff(nodes) > 0)
    assert rho_n.size == nodes.size and mats.size == nodes.size - 1
    k = np.clip(np.searchsorted(nodes, h, side="right") - 1, 0, nodes.size - 2)   # interval index
    hc = np.clip(h, nodes[0], nodes[-1])
    f = (hc - nodes[k]) / (nodes[k + 1] - nodes[k])
    rho = rho_n[k] + f * (rho_n[k + 1] - rho_n[k])
    return mats[k].astype(np.uint8), rho


def quantize_density(rho, bits: int = 20) -> np.ndarray:
    """DESIGN.md reading C18: densities live on the 2^-20 g/cm^3 texel grid (round to nearest, at most 2^24 - 1 counts).
    Reading C30: bits = 12 rounds to the 2^-12 g/cm^3 grid instead (to nearest, at most 2^16 - 1 steps) -- every value is
    then also on the 2^-20 grid, with its low 8 bits zero."""
    assert bits in (12, 20)
    step = 2.0 ** -bits
    counts = np.minimum(np.rint(np.asarray(rho, np.float64) / step), float(2 ** (bits + 4) - 1))
    return (counts * step).astype(np.float32)


def ct_to_phantom(hu_ct, ct_spacing, ct_offset, shape, spacing, ramp: dict):
    """PAPER.md:L81 then L65: resample the CT to the simulation grid, then HU -> (material, density).
    ramp["density_bits"] (absent or 0: 20) chooses the density grid, reading C30.
    Returns (material uint8 [nz][ny][nx], density float32 on the texel grid, resampled HU float64)."""
    hu = resample_mean(hu_ct, ct_spacing, ct_offset, shape, spacing, float(ramp["hu_outside"]))
    mat, rho = hu_to_material_density(hu, ramp)
    return mat, quantize_density(rho, int(ramp.get("density_bits", 0)) or 20), hu


def pet_to_activity(bqml_pet, pet_spacing, pet_offset, shape, spacing):
    """decay pdf = linear conversion of the PET value.  The PET image (Bq/mL) is resampled to the
    simulation grid by the volume-weighted mean (0 outside the PET image) and multiplied by the voxel volume in mL:
    activity [Bq] per voxel; their sum is A(t_s) of Eq. 1.  Returns (activity float64, total Bq)."""
    conc = resample_mean(bqml_pet, pet_spacing, pet_offset, shape, spacing, 0.0)
    vox_ml = spacing[0] * spacing[1] * spacing[2] / 1000.0          # mm^3 -> mL
    act = conc * vox_ml
    return act, float(act.sum())
