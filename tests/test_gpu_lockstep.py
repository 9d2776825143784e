"""History-by-history parity of the CUDA transport with the oracle's LOCKSTEP mode:
the oracle restates the documented algorithm and draw schedule of the CUDA path in fp64, so with the same seed both
follow the same histories up to fp32 rounding.  One decay per batch makes the organ rows of a run a per-history
fingerprint: with 255 interleaved labels (neighbouring voxels always differ) a history matches only if every deposit
went to the same voxel with the same energy.  A few histories in a thousand legitimately part ways where an fp32
rounding flips a decision (a voxel face, an accept test); after that the two are different samples of the same physics."""
import numpy as np
import pytest

import anm_inputs
from oracle import anm_oracle as O

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("photons,rayleigh,positron,hull,scale,src", [
    (2, 1, 0.2498, True, 2, (271.0, 231.0, 1130.0)),      # in the heart, hull majorant on (the default)
    (2, 1, 0.2498, False, 4, (271.0, 231.0, 1130.0)),     # global majorant only
    (1, 0, 0.0, True, 4, (256.0, 150.0, 640.0)),          # single photons, no Rayleigh, source in the skin of the pelvis
])
def test_histories_match_one_by_one(photons, rayleigh, positron, hull, scale, src):
    import paper_2111_11687_b200 as pkg
    tables = anm_inputs.make_tables()
    base = anm_inputs.make_config(3, scale)                   # 4: 64 x 64 x 100 voxels of 8 x 8 x 16 mm; four materials
    nx, ny, nz = base["shape"]
    iz, iy, ix = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    labels = (1 + (ix + 7 * iy + 13 * iz) % 255).astype(np.uint8)
    cfg = dict(base, activity=None, point_source_mm=src, labels=labels, n_organs=255,
               photons_per_decay=photons, rayleigh_on=rayleigh, positron_ke_mev=positron)
    n, seed = 20_000, 77
    with pkg.Simulation(0) as sim:
        sim.load_config(cfg, tables, n_batches=n, collect_stats=1, hull_majorant=1 if hull else 2)
        sim.run(n, seed)
        st = sim.get_stats()
        rows_g = sim.get_tally_buffers()[2].cpu().numpy()[:, 1:256].copy()
    o = O.Oracle(cfg, tables, n_decays=n, n_batches=n, seed=seed, tracking=3 if hull else 2)
    r = o.run_parallel(8)
    rows_o = r["organ_batch"][:, 1:256]
    so = r["stats"]
    assert rows_g.shape == rows_o.shape == (n, 255)
    scale = rows_o.max()
    same = np.all(np.abs(rows_g - rows_o) <= 2e-4 * np.abs(rows_o) + 1e-7 * scale, axis=1)
    frac = same.mean()
    rel = np.abs(rows_g - rows_o)[same] / (np.abs(rows_o)[same] + 1e-7 * scale)
    print("histories identical: %.4f (%d of %d differ); largest relative deviation among them %.1e" % (frac, int((~same).sum()), n, rel.max()))
    assert frac > 0.998
    # totals: the same algorithm on the same random numbers -> the event counts agree far inside the statistical noise
    assert st["n_steps"] == pytest.approx(so["n_substeps"], rel=2e-3)
    assert st["n_compton"] == pytest.approx(so["n_compton"], rel=2e-3)
    assert st["n_pe"] == pytest.approx(so["n_pe"], rel=0.02)
    assert st["deposited_MeV"] == pytest.approx(so["deposited"], rel=1e-3)
    # and the histories that differ are not systematically different: their mean deposit is unbiased
    if (~same).sum() > 20:
        dg, do = rows_g[~same].sum(1).mean(), rows_o[~same].sum(1).mean()
        assert dg == pytest.approx(do, rel=0.35)


@pytest.mark.parametrize("case", ["patient", "fine_water"])
def test_histories_match_with_electron_transport(case):
    """The same with secondary electrons transported (NEXT-2): the walk draws no random numbers, so the histories stay in
    step; in 0.5 mm voxels most electrons cross voxel faces, which the interleaved labels register."""
    import paper_2111_11687_b200 as pkg
    tables = anm_inputs.make_tables()
    et = anm_inputs.make_electron_tables()
    if case == "patient":
        base = anm_inputs.make_config(3, 4)
        src = (271.0, 231.0, 1130.0)
    else:
        nv = 64
        base = dict(anm_inputs.make_config(0, 1), shape=(nv,) * 3, spacing_mm=(0.5,) * 3,
                    material=np.full((nv,) * 3, 2, np.uint8), density=anm_inputs.phantoms.quantize_density(np.full((nv,) * 3, 1.0)))
        src = (16.2, 15.9, 16.1)
    nx, ny, nz = base["shape"]
    iz, iy, ix = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    labels = (1 + (ix + 7 * iy + 13 * iz) % 255).astype(np.uint8)
    cfg = dict(base, activity=None, point_source_mm=src, labels=labels, n_organs=255, photons_per_decay=2, rayleigh_on=1,
               positron_ke_mev=0.0)
    n, seed = 20_000 if case == "patient" else 60_000, 5
    with pkg.Simulation(0) as sim:
        sim.load_config(cfg, tables, n_batches=n, collect_stats=1)
        sim.set_electron_tables(et)
        sim.set_options(n_batches=n, collect_stats=1, electron_transport=1, photons_per_decay=2, rayleigh_on=1,
                        photon_cutoff_MeV=0.010, positron_ke_MeV=0.0)
        sim.run(n, seed)
        st = sim.get_stats()
        rows_g = sim.get_tally_buffers()[2].cpu().numpy()[:, 1:256].copy()
    o = O.Oracle(cfg, tables, n_decays=n, n_batches=n, seed=seed, tracking=3, electron_tables=et)
    r = o.run_parallel(8)
    rows_o = r["organ_batch"][:, 1:256]
    hit = rows_o.sum(1) > 0
    scale = rows_o.max()
    # fp32 positions (1e-6 cm) shift what a grazed voxel receives by ~1e-5 of the largest deposit: absolute floor 2e-5
    same = np.all(np.abs(rows_g - rows_o) <= 5e-4 * np.abs(rows_o) + 2e-5 * scale, axis=1)
    print("%s: histories with deposits %d, identical %.4f, electrons %d (oracle %d, %d voxel crossings)"
          % (case, int(hit.sum()), same[hit].mean(), st["n_electrons"], r["stats"]["n_electrons"], r["stats"]["n_electron_crossings"]))
    assert hit.sum() > 2000
    assert same[hit].mean() > 0.99
    assert st["n_electrons"] == pytest.approx(r["stats"]["n_electrons"], rel=2e-3)
    if case == "fine_water":
        assert r["stats"]["n_electron_crossings"] > 0.5 * r["stats"]["n_electrons"]


def test_histories_match_from_the_activity_map():
    """The bench workload's shape: decays drawn from the patient's activity map through the alias table (which the oracle
    rebuilds by the ordered sweep from the same activity volume), uniform point in the voxel, pairs, positron energy,
    Rayleigh, hull majorant.  Every step of SURVEY.md §8(a) A1-A9 is then followed history by history."""
    import paper_2111_11687_b200 as pkg
    tables = anm_inputs.make_tables()
    base = anm_inputs.make_config(3, 4)
    nx, ny, nz = base["shape"]
    iz, iy, ix = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    labels = (1 + (ix + 7 * iy + 13 * iz) % 255).astype(np.uint8)
    cfg = dict(base, labels=labels, n_organs=255)
    n, seed = 30_000, 42
    with pkg.Simulation(0) as sim:
        sim.load_config(cfg, tables, n_batches=n, collect_stats=1)
        alias_g = sim.get_alias_table()
        sim.run(n, seed)
        st = sim.get_stats()
        rows_g = sim.get_tally_buffers()[2].cpu().numpy()[:, 1:256].copy()
    o = O.Oracle(cfg, tables, n_decays=n, n_batches=n, seed=seed, tracking=3)
    r = o.run_parallel(8)
    rows_o = r["organ_batch"][:, 1:256]
    scale = rows_o.max()
    same = np.all(np.abs(rows_g - rows_o) <= 2e-4 * np.abs(rows_o) + 1e-7 * scale, axis=1)
    print("activity source: histories identical %.4f (%d of %d differ)" % (same.mean(), int((~same).sum()), n))
    assert same.mean() > 0.998
    assert st["n_steps"] == pytest.approx(r["stats"]["n_substeps"], rel=2e-3)
    assert st["deposited_MeV"] == pytest.approx(r["stats"]["deposited"], rel=1e-3)
    assert alias_g.shape[0] == int((base["activity"] > 0).sum())


def test_energy_and_hbh_sigma_maps_voxel_by_voxel():
    """With the histories in step the tallies themselves can be compared element by element: the energy map and the
    history-by-history sigma map (NEXT-4) of a 200 000-decay run, voxel by voxel, against the lockstep oracle's."""
    import paper_2111_11687_b200 as pkg
    tables = anm_inputs.make_tables()
    cfg = anm_inputs.make_config(3, 4)
    n, B, seed = 200_000, 10, 42
    with pkg.Simulation(0) as sim:
        sim.load_config(cfg, tables, n_batches=B, collect_stats=1, uncertainty=1)
        sim.run(n, seed)
        e_g = sim.get_energy().astype(np.float64)
        rel_g = sim.get_uncertainty().astype(np.float64)
        organs = sim.get_organ_doses()
    o = O.Oracle(cfg, tables, n_decays=n, n_batches=B, seed=seed, tracking=3)
    r = o.run_parallel(10, hbh=True)
    f = o.finalize(r)
    e_o, rel_o = f["energy"], f["rel_sigma_hbh"]
    hit = (e_o > 0) | (e_g > 0)
    ok = np.abs(e_g - e_o) <= 1e-4 * e_o + 1e-9
    print("voxels with energy %d, energy identical in %.5f, sum ratio %.7f" % (int(hit.sum()), ok[hit].mean(), e_g.sum() / e_o.sum()))
    assert ok[hit].mean() > 0.999                      # a history that parts ways touches a handful of voxels
    assert e_g.sum() == pytest.approx(e_o.sum(), rel=2e-5)
    both = ok & (e_o > 0)
    assert np.allclose(rel_g[both], rel_o[both], rtol=2e-3, atol=1e-6)
    # organ doses (Eq. 2) and their batch sigma from the same histories: equal, not merely compatible
    big = f["organs"]["n_voxels"] >= 20
    assert np.allclose(organs["mean_Gy_per_decay"][big], f["organs"]["mean"][big], rtol=2e-4)
    assert np.allclose(organs["sigma_mean"][big], f["organs"]["sigma_mean"][big], rtol=5e-3)


def test_full_size_patient_in_the_bench_configuration():
    """BASELINE.json cfg3 at full size (256 x 256 x 400 voxels) in the configuration bench.py times -- 100 batches, the
    default event-pool kernel, hull majorant, launch pipeline, positron energy -- on 1e6 of its decays: the lockstep
    oracle follows the same histories, so the energy map is compared voxel by voxel and the 27 organ doses number by number."""
    import paper_2111_11687_b200 as pkg
    tables = anm_inputs.make_tables()
    cfg = anm_inputs.make_config(3)
    n, B, seed = 1_000_000, 100, cfg["seed"]
    with pkg.Simulation(0) as sim:
        sim.load_config(cfg, tables, n_batches=B)
        sim.run(n, seed)
        e_g = sim.get_energy().astype(np.float64)
        organs = sim.get_organ_doses()
    o = O.Oracle(cfg, tables, n_decays=n, n_batches=B, seed=seed, tracking=3)
    r = o.run_parallel(10)
    f = o.finalize(r)
    e_o = f["energy"]
    hit = (e_o > 0) | (e_g > 0)
    ok = np.abs(e_g - e_o) <= 1e-4 * e_o + 1e-9
    print("full size: voxels with energy %d, identical %.5f, sum ratio %.7f" % (int(hit.sum()), ok[hit].mean(), e_g.sum() / e_o.sum()))
    assert hit.sum() > 1_000_000
    assert ok[hit].mean() > 0.999
    assert e_g.sum() == pytest.approx(e_o.sum(), rel=2e-5)
    nz_ = f["organs"]["n_voxels"] > 0
    assert np.array_equal(organs["n_voxels"][nz_].astype(np.int64), f["organs"]["n_voxels"][nz_].astype(np.int64))
    assert np.allclose(organs["mean_Gy_per_decay"][nz_], f["organs"]["mean"][nz_], rtol=1e-3, atol=1e-4 * f["organs"]["mean"].max())
    big = f["organs"]["n_voxels"] >= 1000
    assert np.allclose(organs["mean_Gy_per_decay"][big], f["organs"]["mean"][big], rtol=2e-4)


@pytest.mark.parametrize("k,scale", [(0, 1), (1, 2), (2, 2)])
def test_other_configs_voxel_by_voxel(k, scale):
    """cfg0 (point source, full size), cfg1 (single active voxel, one photon per history) and cfg2 (water / lung / bone
    slabs, activity box, pairs) at half resolution: energy map voxel by voxel against the lockstep oracle."""
    import paper_2111_11687_b200 as pkg
    tables = anm_inputs.make_tables()
    cfg = anm_inputs.make_config(k, scale)
    n, B, seed = 200_000, 10, cfg["seed"]
    with pkg.Simulation(0) as sim:
        sim.load_config(cfg, tables, n_batches=B, collect_stats=1)
        sim.run(n, seed)
        e_g = sim.get_energy().astype(np.float64)
        st = sim.get_stats()
    o = O.Oracle(cfg, tables, n_decays=n, n_batches=B, seed=seed, tracking=3)
    r = o.run_parallel(10)
    e_o = r["sum"]
    hit = (e_o > 0) | (e_g > 0)
    ok = np.abs(e_g - e_o) <= 1e-4 * e_o + 1e-9
    print("cfg%d: voxels with energy %d, identical %.5f, sum ratio %.7f" % (k, int(hit.sum()), ok[hit].mean(), e_g.sum() / e_o.sum()))
    assert ok[hit].mean() > 0.998
    assert e_g.sum() == pytest.approx(e_o.sum(), rel=5e-5)
    assert st["escaped_MeV"] == pytest.approx(r["stats"]["escaped"], rel=5e-5)
    assert st["n_compton"] == pytest.approx(r["stats"]["n_compton"], rel=1e-3)


def test_the_papers_configuration_electrons_and_history_by_history():
    """PAPER.md:L67 as a whole: secondary electrons followed down to 200 keV AND the history-by-history uncertainty.
    0.5 mm water voxels (the paper's water test, L79), point source; energy map and sigma map voxel by voxel."""
    import paper_2111_11687_b200 as pkg
    tables = anm_inputs.make_tables()
    et = anm_inputs.make_electron_tables()
    nv = 64
    cfg = dict(anm_inputs.make_config(0, 1), shape=(nv,) * 3, spacing_mm=(0.5,) * 3, material=np.full((nv,) * 3, 2, np.uint8),
               density=anm_inputs.phantoms.quantize_density(np.full((nv,) * 3, 1.0)), point_source_mm=(16.2, 15.9, 16.1),
               labels=None, n_organs=0, photons_per_decay=2, positron_ke_mev=0.0)
    n, B, seed = 2_000_000, 10, 3
    with pkg.Simulation(0) as sim:
        sim.load_config(cfg, tables, n_batches=B)
        sim.set_electron_tables(et)
        sim.set_options(n_batches=B, collect_stats=1, electron_transport=1, uncertainty=1, photons_per_decay=2, rayleigh_on=1,
                        photon_cutoff_MeV=0.010, positron_ke_MeV=0.0)
        sim.run(n, seed)
        e_g = sim.get_energy().astype(np.float64)
        rel_g = sim.get_uncertainty().astype(np.float64)
        st = sim.get_stats()
    o = O.Oracle(cfg, tables, n_decays=n, n_batches=B, seed=seed, tracking=3, electron_tables=et)
    r = o.run_parallel(10, hbh=True)
    f = o.finalize(r)
    e_o, rel_o = f["energy"], f["rel_sigma_hbh"]
    assert st["n_hbh_overflow"] == 0 and st["n_electrons"] == pytest.approx(r["stats"]["n_electrons"], rel=1e-3)
    hit = (e_o > 0) | (e_g > 0)
    ok = np.abs(e_g - e_o) <= 2e-4 * e_o + 2e-5
    print("electrons + HbH: voxels with energy %d, identical %.5f, sum ratio %.7f" % (int(hit.sum()), ok[hit].mean(), e_g.sum() / e_o.sum()))
    assert ok[hit].mean() > 0.995
    assert e_g.sum() == pytest.approx(e_o.sum(), rel=5e-5)
    both = ok & (e_o > 0.5)                       # voxels hit by several histories
    assert both.sum() > 1000
    assert np.allclose(rel_g[both], rel_o[both], rtol=5e-3, atol=1e-6)
