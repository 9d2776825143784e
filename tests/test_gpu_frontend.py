"""Parity of the CUDA image front end (anm_load_ct / anm_load_pet) with its CPU oracle
(oracle/anm_frontend.py), element by element on the same synthetic CT / PET images, through the C ABI.

Bar: material ids bit-exact (a voxel whose mean HU sits within 1e-9 HU of a ramp node may fall on either side: both
sides sum in fp64 but in a different order); density within one texel count (2^-20 g/cm^3); activity equal to the
oracle's fp64 value rounded to fp32 within 1 ulp; A(t_s) within 1e-12 relative.  Then the whole path from the images:
run on the GPU from anm_load_ct / anm_load_pet against the transport oracle run on the oracle front end's volumes."""
import numpy as np
import pytest

import anm_inputs
from oracle import anm_frontend as fe
from oracle import anm_oracle as O

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def anm():
    import paper_2111_11687_b200 as pkg
    return pkg


@pytest.fixture(scope="module")
def tables():
    return anm_inputs.make_tables()


def compare_front_end(anm, cfg, img, device_inputs=False):
    shape, sp = cfg["shape"], cfg["spacing_mm"]
    mat_o, rho_o, hu_o = fe.ct_to_phantom(img["ct_hu"], img["ct_spacing_mm"], img["ct_offset_mm"], shape, sp, img["ramp"])
    act_o, tot_o = fe.pet_to_activity(img["pet_bqml"], img["pet_spacing_mm"], img["pet_offset_mm"], shape, sp)
    with anm.Simulation(0) as sim:
        sim.set_grid(shape, sp)
        if device_inputs:
            import torch
            hu_d = torch.from_numpy(img["ct_hu"]).cuda()
            pet_d = torch.from_numpy(img["pet_bqml"]).cuda()
            act_d = torch.empty(sim.V, dtype=torch.float32, device="cuda")
            sim.load_ct(hu_d, img["ct_shape"], img["ct_spacing_mm"], img["ct_offset_mm"], img["ramp"])
            tot_g = sim.load_pet(pet_d, img["pet_shape"], img["pet_spacing_mm"], img["pet_offset_mm"], out_activity=act_d)
            torch.cuda.synchronize()
            act_g = act_d.cpu().numpy()
        else:
            sim.load_ct(img["ct_hu"], img["ct_shape"], img["ct_spacing_mm"], img["ct_offset_mm"], img["ramp"])
            act_g = np.empty(sim.V, np.float32)
            tot_g = sim.load_pet(img["pet_bqml"], img["pet_shape"], img["pet_spacing_mm"], img["pet_offset_mm"], out_activity=act_g)
        mat_g, rho_g = sim.get_phantom()
        st = sim.get_stats()
    nodes = np.asarray(img["ramp"]["hu"])
    near_node = np.min(np.abs(hu_o[..., None] - nodes), axis=-1) < 1e-9
    diff = mat_g != mat_o
    assert not (diff & ~near_node).any(), int((diff & ~near_node).sum())
    assert diff.sum() <= 4
    bits = int(img["ramp"].get("density_bits", 0)) or 20       # the density grid (reading C30); counts in ITS steps
    counts_g = rho_g.astype(np.float64) * 2 ** bits
    counts_o = rho_o.astype(np.float64) * 2 ** bits
    assert np.array_equal(counts_g, np.rint(counts_g)) and np.array_equal(counts_o, np.rint(counts_o))     # both on the grid
    assert np.max(np.abs(counts_g - counts_o)[~diff]) <= 1
    assert (counts_g != counts_o).mean() < 1e-3           # a 1-count difference needs rho*2^20 within ~1e-9 of a half-integer
    a32 = act_o.astype(np.float32).reshape(-1)
    ulp = np.spacing(np.maximum(np.abs(a32), np.float32(1e-30)))
    assert np.all(np.abs(act_g - a32) <= ulp), float(np.max(np.abs(act_g - a32) / ulp))
    assert (act_g != a32).mean() < 1e-3
    assert tot_g == pytest.approx(tot_o, rel=1e-12)
    assert st["ms_load_ct"] > 0 and st["ms_load_pet"] > 0
    return mat_o, rho_o, act_o, tot_o, st


@pytest.mark.parametrize("device_inputs", [False, True])
def test_front_end_small_ragged(anm, device_inputs):
    """cfg3 / 4 (64 x 64 x 100 voxels); the CT grid is incommensurate with the simulation grid, overhangs it on two
    axes and falls short on the third (hu_outside fills the rest); several resample tiles and a ragged tail."""
    cfg = anm_inputs.make_config(3, 4)
    img = anm_inputs.make_ct_pet(cfg, ct_shape=(151, 131, 173), ct_margin_mm=(13.0, -9.0, 5.5))
    compare_front_end(anm, cfg, img, device_inputs)


def test_front_end_on_the_coarse_density_grid_reaches_the_16_bit_texels(anm, tables):
    """anm_hu_ramp.density_bits = 12 (reading C30): material ids as before, densities exactly the oracle's on the
    2^-12 g/cm^3 grid -- and a phantom made from a CT image then runs on the exact 16-bit texel copy
    (anm_stats.texel_bits), which the 2^-20 grid never allows.  The synthetic patient stays below 2 g/cm^3."""
    cfg = anm_inputs.make_config(3, 4)
    img = anm_inputs.make_ct_pet(cfg, ct_shape=(151, 131, 173), ct_margin_mm=(13.0, -9.0, 5.5))
    img12 = dict(img, ramp=dict(img["ramp"], density_bits=12))
    _, rho_o, _, _, _ = compare_front_end(anm, cfg, img12)
    assert float(np.max(rho_o)) < 2.0
    bits = {}
    for name, im in (("fine", img), ("coarse", img12)):
        with anm.Simulation(0) as sim:
            sim.set_grid(cfg["shape"], cfg["spacing_mm"])
            sim.load_ct(im["ct_hu"], im["ct_shape"], im["ct_spacing_mm"], im["ct_offset_mm"], im["ramp"])
            sim.load_pet(im["pet_bqml"], im["pet_shape"], im["pet_spacing_mm"], im["pet_offset_mm"])
            sim.set_physics_tables(tables)
            sim.set_options(n_batches=10, collect_stats=1, positron_ke_MeV=0.2498)
            sim.run(200_000, 9)
            st = sim.get_stats()
            bits[name] = (int(st["texel_bits"]), st["deposited_MeV"])
    assert bits["fine"][0] == 32 and bits["coarse"][0] == 16
    assert abs(bits["coarse"][1] / bits["fine"][1] - 1.0) < 5e-3        # densities moved by <= 1.2e-4 g/cm^3: the same physics
    with anm.Simulation(0) as sim:
        sim.set_grid(cfg["shape"], cfg["spacing_mm"])
        with pytest.raises(anm.AnmError) as ei:
            sim.load_ct(img["ct_hu"], img["ct_shape"], img["ct_spacing_mm"], img["ct_offset_mm"], dict(img["ramp"], density_bits=16))
        assert ei.value.code == -1


def test_front_end_pet_on_its_own_grid(anm):
    """PET image on a coarser grid that covers only part of the simulation grid (0 outside)."""
    cfg = anm_inputs.make_config(3, 8)
    img = anm_inputs.make_ct_pet(cfg)
    rng = np.random.default_rng(11)
    img["pet_bqml"] = (rng.uniform(size=(20, 17, 13)) * 4e3).astype(np.float32)
    img["pet_shape"], img["pet_spacing_mm"], img["pet_offset_mm"] = (13, 17, 20), (31.0, 23.0, 57.0), (40.0, 61.0, 120.0)
    *_, tot_o, _ = compare_front_end(anm, cfg, img)
    # the image lies inside the grid: the integral of the image is conserved
    assert tot_o == pytest.approx(float(img["pet_bqml"].astype(np.float64).sum()) * 31.0 * 23.0 * 57.0 / 1000.0, rel=1e-12)


def test_front_end_at_the_papers_sizes(anm):
    """PET grid 168 x 168 x 219 at 4.063 x 4.063 x 5 mm; a 512 x 512 x 365 CT resampled onto it."""
    cfg = anm_inputs.make_patient_on_grid((168, 168, 219), (4.063, 4.063, 5.0))
    img = anm_inputs.make_ct_pet(cfg, ct_shape=(512, 512, 365))
    *_, st = compare_front_end(anm, cfg, img, device_inputs=True)
    print("load_ct %.3f ms, load_pet resample %.3f ms" % (st["ms_load_ct"], st["ms_load_pet"]))


def test_whole_path_from_the_images(anm, tables):
    """Images -> anm_load_ct / anm_load_pet -> run -> organ doses and dose rate, against the transport oracle fed with
    the oracle front end's volumes (north_star tolerances)."""
    cfg = anm_inputs.make_config(3, 4)
    img = anm_inputs.make_ct_pet(cfg, ct_shape=(150, 140, 170), ct_margin_mm=(6.0, 6.0, 0.0))
    mat_o, rho_o, _ = fe.ct_to_phantom(img["ct_hu"], img["ct_spacing_mm"], img["ct_offset_mm"], cfg["shape"], cfg["spacing_mm"], img["ramp"])
    act_o, tot_o = fe.pet_to_activity(img["pet_bqml"], img["pet_spacing_mm"], img["pet_offset_mm"], cfg["shape"], cfg["spacing_mm"])
    n, B = 2_000_000, 100
    with anm.Simulation(0) as sim:
        sim.set_grid(cfg["shape"], cfg["spacing_mm"])
        sim.load_ct(img["ct_hu"], img["ct_shape"], img["ct_spacing_mm"], img["ct_offset_mm"])      # default ramp
        tot_g = sim.load_pet(img["pet_bqml"], img["pet_shape"], img["pet_spacing_mm"], img["pet_offset_mm"])
        sim.load_organs(cfg["labels"], cfg["n_organs"])
        sim.set_physics_tables(tables)
        sim.set_options(n_batches=B, photons_per_decay=2, rayleigh_on=1, photon_cutoff_MeV=0.010, positron_ke_MeV=0.2498, collect_stats=1)
        sim.run(n, 42)
        organs = sim.get_organ_doses()
        st = sim.get_stats()
        rate = sim.get_dose_rate(tot_g).astype(np.float64)
        dose = sim.get_dose().astype(np.float64)
    ocfg = dict(cfg, material=mat_o, density=rho_o, activity=act_o.astype(np.float32))
    o = O.Oracle(ocfg, tables, n_decays=n, n_batches=B, seed=1042)
    r = o.run_parallel(min(32, __import__("os").cpu_count() or 1))
    f = o.finalize(r, total_activity_bq=tot_o)
    assert abs(st["deposited_MeV"] + st["escaped_MeV"] - st["emitted_MeV"]) < 2e-5 * st["emitted_MeV"]
    assert st["deposited_MeV"] / r["stats"]["deposited"] == pytest.approx(1.0, abs=2e-3)
    big = f["organs"]["n_voxels"] >= 20
    gm, gs = organs["mean_Gy_per_decay"][big], organs["sigma_mean"][big]
    om, osig = f["organs"]["mean"][big], f["organs"]["sigma_mean"][big]
    assert np.all(np.abs(gm - om) <= np.maximum(0.01 * om, 3.0 * np.sqrt(gs ** 2 + osig ** 2)))
    # Eq. 1: dose rate = dose per decay x A(t_s), A(t_s) from the PET image
    assert np.allclose(rate, dose * tot_g, rtol=1e-6, atol=0)
    assert tot_g == pytest.approx(anm_inputs.phantoms.TOTAL_ACTIVITY_BQ, rel=1e-6)


def test_front_end_error_codes(anm):
    import ctypes as C
    from paper_2111_11687_b200 import binding
    cfg = anm_inputs.make_config(3, 16)
    img = anm_inputs.make_ct_pet(cfg)
    with anm.Simulation(0) as sim:
        with pytest.raises(anm.AnmError) as e:
            sim.load_ct(img["ct_hu"], img["ct_shape"], img["ct_spacing_mm"])
        assert e.value.code == -2                       # before anm_set_grid
        sim.set_grid(cfg["shape"], cfg["spacing_mm"])
        with pytest.raises(anm.AnmError) as e:
            sim.get_phantom()
        assert e.value.code == -2
        bad = dict(img["ramp"], hu=[-1024.0, -974.0, -974.0, 101.0, 1976.0])
        with pytest.raises(anm.AnmError) as e:
            sim.load_ct(img["ct_hu"], img["ct_shape"], img["ct_spacing_mm"], img["ct_offset_mm"], bad)
        assert e.value.code == -1
        bad = dict(img["ramp"], material=[0, 1, 2, 9])
        with pytest.raises(anm.AnmError) as e:
            sim.load_ct(img["ct_hu"], img["ct_shape"], img["ct_spacing_mm"], img["ct_offset_mm"], bad)
        assert e.value.code == -1
        with pytest.raises(anm.AnmError) as e:
            sim.load_ct(img["ct_hu"], img["ct_shape"], (1.0, -1.0, 1.0))
        assert e.value.code == -1
        L = binding.load()
        assert L.anm_load_ct(sim._ctx, None, 2, 2, 2, 1.0, 1.0, 1.0, 0.0, 0.0, 0.0, None, 0) == -1
        assert L.anm_load_pet(sim._ctx, None, 2, 2, 2, 1.0, 1.0, 1.0, 0.0, 0.0, 0.0, 0, None, None, 0) == -1
        neg = img["pet_bqml"].copy(); neg[3, 3, 3] = -1.0
        with pytest.raises(anm.AnmError) as e:
            sim.load_pet(neg, img["pet_shape"], img["pet_spacing_mm"])
        assert e.value.code == -1
        nan = img["pet_bqml"].copy(); nan[2, 3, 3] = np.nan
        with pytest.raises(anm.AnmError) as e:
            sim.load_pet(nan, img["pet_shape"], img["pet_spacing_mm"])
        assert e.value.code == -1
        with pytest.raises(anm.AnmError) as e:       # an image entirely outside the grid leaves no activity
            sim.load_pet(img["pet_bqml"], img["pet_shape"], img["pet_spacing_mm"], (1e5, 0.0, 0.0))
        assert e.value.code == -1
        sim.load_ct(img["ct_hu"], img["ct_shape"], img["ct_spacing_mm"], img["ct_offset_mm"])
        m, r = sim.get_phantom()
        assert m.shape == cfg["material"].shape and r.dtype == np.float32
