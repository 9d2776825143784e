"""Pins of the image front end's CPU oracle (oracle/anm_frontend.py) against what the
definitions fix: brute-force point sampling on a lattice commensurate with both grids, block means (numpy),
conservation of the image integral, identity, constants, and the ramp's node / midpoint / clamp values."""
import numpy as np
import pytest

import anm_inputs
from oracle import anm_frontend as fe


def test_overlap_weights_rows_and_columns():
    # dst 5 voxels of 2.0, src 4 voxels of 3.0 starting at -1.0: src covers [-1, 11), dst covers [0, 10)
    W = fe.overlap_weights(5, 2.0, 4, 3.0, -1.0)
    assert np.allclose(W.sum(1), 1.0)                           # every dst voxel fully inside the source
    assert np.allclose(W.sum(0) * 2.0, [2.0, 3.0, 3.0, 2.0])    # covered length of each src voxel: [0,2), [2,5), [5,8), [8,10)
    # dst voxel 2 = [4,6): src 1 = [2,5) -> 1, src 2 = [5,8) -> 1
    assert np.allclose(W[2], [0, 0.5, 0.5, 0])


def test_resample_brute_force_lattice():
    """Point sampling at the centres of a 0.5 mm lattice is exact when 0.5 divides both spacings and the offset."""
    rng = np.random.default_rng(5)
    src = rng.normal(size=(5, 4, 6))                            # [z][y][x]
    s_sp, s_off = (1.5, 3.0, 2.5), (-1.0, 0.5, -2.0)
    d_shape, d_sp = (4, 5, 3), (2.0, 2.5, 3.5)
    fill = -7.0
    got = fe.resample_mean(src, s_sp, s_off, d_shape, d_sp, fill)
    h = 0.5
    want = np.zeros((d_shape[2], d_shape[1], d_shape[0]))
    for k in range(d_shape[2]):
        for j in range(d_shape[1]):
            for i in range(d_shape[0]):
                acc, n = 0.0, 0
                for zz in np.arange(k * d_sp[2] + h / 2, (k + 1) * d_sp[2], h):
                    for yy in np.arange(j * d_sp[1] + h / 2, (j + 1) * d_sp[1], h):
                        for xx in np.arange(i * d_sp[0] + h / 2, (i + 1) * d_sp[0], h):
                            a = int(np.floor((xx - s_off[0]) / s_sp[0])); b = int(np.floor((yy - s_off[1]) / s_sp[1]))
                            c = int(np.floor((zz - s_off[2]) / s_sp[2]))
                            ok = 0 <= a < 6 and 0 <= b < 4 and 0 <= c < 5
                            acc += src[c, b, a] if ok else fill
                            n += 1
                want[k, j, i] = acc / n
    assert np.allclose(got, want, rtol=0, atol=1e-12)


def test_resample_block_mean_identity_constant_and_integral():
    rng = np.random.default_rng(6)
    src = rng.uniform(size=(6, 8, 12))
    # integer ratio (3, 2, 2) downsample == block mean
    got = fe.resample_mean(src, (1.0, 1.0, 1.0), (0, 0, 0), (4, 4, 3), (3.0, 2.0, 2.0), 0.0)
    want = src.reshape(3, 2, 4, 2, 4, 3).mean(axis=(1, 3, 5))
    assert np.allclose(got, want, atol=1e-14)
    # same grid == identity
    assert np.allclose(fe.resample_mean(src, (2.0, 1.0, 3.0), (0, 0, 0), (12, 8, 6), (2.0, 1.0, 3.0), 9.0), src, atol=1e-14)
    # a constant image stays constant whatever the grids, also partly outside when fill equals it
    c = fe.resample_mean(np.full((3, 3, 3), 4.25), (1.7, 2.3, 0.9), (-0.4, 0.3, 1.1), (5, 4, 6), (1.1, 1.3, 0.7), 4.25)
    assert np.allclose(c, 4.25, atol=1e-13)
    # integral conserved when the destination covers the source (fill 0): sum(dst) V_dst == sum(src) V_src
    src2 = rng.uniform(size=(4, 5, 3))
    d = fe.resample_mean(src2, (1.3, 0.7, 2.1), (1.0, 0.5, 0.25), (7, 6, 11), (1.0, 1.0, 1.0), 0.0)
    assert d.sum() * 1.0 == pytest.approx(src2.sum() * 1.3 * 0.7 * 2.1, rel=1e-13)


def test_hu_ramp_nodes_midpoints_clamps_materials():
    ramp = anm_inputs.DEFAULT_HU_RAMP
    hu = np.array(ramp["hu"])
    mat, rho = fe.hu_to_material_density(hu, ramp)
    assert np.allclose(rho, ramp["rho"], atol=1e-15)
    assert list(mat) == [0, 1, 2, 3, 3]                          # [h_k, h_{k+1}) -> m_k; the last node belongs to the last segment
    mid = 0.5 * (hu[:-1] + hu[1:])
    matm, rhom = fe.hu_to_material_density(mid, ramp)
    assert np.allclose(rhom, 0.5 * (np.array(ramp["rho"])[:-1] + np.array(ramp["rho"])[1:]), atol=1e-15)
    assert list(matm) == ramp["material"]
    m2, r2 = fe.hu_to_material_density(np.array([-5000.0, 5000.0, np.nextafter(-974.0, -np.inf)]), ramp)
    assert list(m2) == [0, 3, 0] and r2[0] == 0.001 and r2[1] == 2.088
    # "All voxels in CT images are assigned a value of 0 to simulate the water box": HU 0 must be water at ~1 g/cm^3
    m0, r0 = fe.hu_to_material_density(np.array([0.0]), ramp)
    assert m0[0] == anm_inputs.MATERIAL_IDS["water"] and abs(r0[0] - 1.0) < 0.01
    # hand value: 0.302 + 724/825 * 0.799
    assert r0[0] == pytest.approx(0.302 + 724.0 / 825.0 * 0.799, abs=1e-15)
    # monotone
    h = np.linspace(-1100, 2100, 3201)
    assert np.all(np.diff(fe.hu_to_material_density(h, ramp)[1]) >= 0)


def test_density_quantisation_and_pet_linear_conversion():
    q = fe.quantize_density(np.array([0.0, 1.0, 1.0 + 0.4 * 2.0 ** -20, 1.0 + 0.6 * 2.0 ** -20, 20.0]))
    assert q[0] == 0 and q[1] == 1 and q[2] == 1 and q[3] == np.float32(1.0 + 2.0 ** -20) and q[4] == np.float32((2 ** 24 - 1) * 2.0 ** -20)
    # Bq/mL x mL: a 2 x 2 x 4 mm voxel is 0.016 mL (SURVEY P12's voxel); same-grid PET
    pet = np.zeros((3, 3, 3)); pet[1, 1, 1] = 1000.0
    act, tot = fe.pet_to_activity(pet, (2.0, 2.0, 4.0), (0, 0, 0), (3, 3, 3), (2.0, 2.0, 4.0))
    assert act[1, 1, 1] == pytest.approx(16.0, rel=1e-15) and tot == pytest.approx(16.0, rel=1e-15)
    # a PET image on a coarser, shifted grid: total activity conserved when the grid covers it
    pet2 = np.random.default_rng(3).uniform(size=(2, 3, 2)) * 5e3
    act2, tot2 = fe.pet_to_activity(pet2, (4.0, 3.0, 5.0), (1.0, 2.0, 0.5), (10, 12, 11), (1.0, 1.0, 1.0))
    assert tot2 == pytest.approx(pet2.sum() * 4.0 * 3.0 * 5.0 / 1000.0, rel=1e-13)


def test_round_trip_recovers_the_phantom():
    """A noise-free CT made from a phantom by nearest-neighbour upsampling at an integer ratio comes back exactly
    (block mean of equal values), so ct_to_phantom must return the phantom's materials and densities."""
    cfg = anm_inputs.make_config(3, 16)
    nx, ny, nz = cfg["shape"]
    img = anm_inputs.make_ct_pet(cfg, ct_shape=(2 * nx, 2 * ny, 2 * nz), noise_hu=0.0)
    hu = anm_inputs.density_to_hu(cfg["density"], cfg["material"]).repeat(2, 0).repeat(2, 1).repeat(2, 2)
    mat, rho, _ = fe.ct_to_phantom(hu, img["ct_spacing_mm"], img["ct_offset_mm"], cfg["shape"], cfg["spacing_mm"], img["ramp"])
    ramp = img["ramp"]
    # densities outside their material's segment were clipped by the generator; compare where they were not
    lo = np.array(ramp["rho"])[:-1][cfg["material"]]; hi = np.array(ramp["rho"])[1:][cfg["material"]]
    ok = (cfg["density"] > lo) & (cfg["density"] < hi)
    assert ok.mean() > 0.9
    assert np.array_equal(mat[ok], cfg["material"][ok])
    assert np.max(np.abs(rho[ok].astype(np.float64) - cfg["density"][ok])) <= 2.0 ** -20 + 1e-12
    act, tot = fe.pet_to_activity(img["pet_bqml"], img["pet_spacing_mm"], img["pet_offset_mm"], cfg["shape"], cfg["spacing_mm"])
    assert tot == pytest.approx(anm_inputs.phantoms.TOTAL_ACTIVITY_BQ, rel=1e-6)
    assert np.allclose(act / act.sum(), cfg["activity"].astype(np.float64) / cfg["activity"].astype(np.float64).sum(), rtol=1e-6, atol=0)


def test_density_grid_of_reading_c30():
    """quantize_density(rho, 12): every value on the 2^-12 g/cm^3 grid (hence on the 2^-20 grid with the low 8 bits of its
    count zero: the word the 16-bit texel holds exactly), to nearest (error <= 2^-13), ties and the cap as for 20 bits;
    the default is unchanged; ct_to_phantom takes the choice from ramp["density_bits"] and changes nothing else."""
    rho = np.concatenate([np.random.default_rng(5).uniform(0.0, 2.2, 20000), [0.0, 0.0012, 1.0, 1.0 + 0.4 * 2.0 ** -12, 1.0 + 0.6 * 2.0 ** -12, 40.0]])
    q12 = fe.quantize_density(rho, 12).astype(np.float64)
    c20 = q12 * 2.0 ** 20
    assert np.array_equal(c20, np.rint(c20)) and np.all(c20.astype(np.int64) % 256 == 0)
    inside = rho < 15.9
    assert np.max(np.abs(q12[inside] - rho[inside])) <= 2.0 ** -13 + 1e-15
    assert q12[-3] == 1.0 and q12[-2] == 1.0 + 2.0 ** -12 and q12[-1] == (2 ** 16 - 1) * 2.0 ** -12
    assert q12[-5] == round(0.0012 * 4096) / 4096                       # air: 5 steps of 2^-12 = 0.00122 g/cm^3
    assert np.array_equal(fe.quantize_density(rho), fe.quantize_density(rho, 20))
    assert np.max(np.abs(fe.quantize_density(rho, 20).astype(np.float64)[inside] - rho[inside])) <= 2.0 ** -21 + 2.0 ** -24   # + float32 storage
    # through ct_to_phantom: same materials, same resampled HU, densities = the fine ones re-rounded from the SAME rho(HU)
    hu = np.random.default_rng(6).integers(-1024, 1700, size=(7, 6, 5)).astype(np.int16)
    ramp = {"hu": [-1024.0, -974.0, -724.0, 101.0, 1976.0], "rho": [0.001, 0.044, 0.302, 1.101, 2.088], "material": [0, 1, 2, 3], "hu_outside": -1024.0}
    m20, r20, h20 = fe.ct_to_phantom(hu, (2.0, 2.0, 2.0), (0, 0, 0), (5, 6, 7), (2.0, 2.0, 2.0), ramp)
    m12, r12, h12 = fe.ct_to_phantom(hu, (2.0, 2.0, 2.0), (0, 0, 0), (5, 6, 7), (2.0, 2.0, 2.0), dict(ramp, density_bits=12))
    assert np.array_equal(m20, m12) and np.array_equal(h20, h12)
    _, rho_exact = fe.hu_to_material_density(h12, ramp)
    assert np.array_equal(r12, fe.quantize_density(rho_exact, 12))
    assert np.max(np.abs(r12.astype(np.float64) - r20)) <= 2.0 ** -13 + 2.0 ** -20
    assert abs(r12.astype(np.float64).sum() / r20.astype(np.float64).sum() - 1.0) < 2.0 ** -13      # total mass: within the per-voxel bound
