"""BASELINE.json cfg4 (512 x 512 x 600 voxels of 0.98 x 0.98 x 3 mm; the fp32 tally, 630 MB, exceeds the L2): a parity
case, not the bench workload.  Half-resolution variant against the live oracle (north_star tolerances), and the
full-size grid on what holds at any size: energy balance, positron energy in the decay voxels, totals per decay equal
to the half-resolution run's (the same analytic patient), every counter equal between the two schedules."""
import os

import numpy as np
import pytest

import anm_inputs
from oracle import anm_oracle as O

pytestmark = pytest.mark.gpu
NPROC = min(32, os.cpu_count() or 1)


@pytest.fixture(scope="module")
def anm():
    import paper_2111_11687_b200 as pkg
    return pkg


@pytest.fixture(scope="module")
def tables():
    return anm_inputs.make_tables()


def test_cfg4_half_resolution_vs_oracle(anm, tables):
    cfg = anm_inputs.make_config(4, 4)                   # 128 x 128 x 150 voxels of 3.92 x 3.92 x 12 mm
    n, B = 2_000_000, 100
    with anm.Simulation(0) as sim:
        sim.load_config(cfg, tables, n_batches=B, collect_stats=1)
        sim.run(n, cfg["seed"])
        st, organs = sim.get_stats(), sim.get_organ_doses()
    o = O.Oracle(cfg, tables, n_decays=n, n_batches=B, seed=cfg["seed"] + 1000)
    r = o.run_parallel(NPROC)
    f = o.finalize(r)
    assert abs(st["deposited_MeV"] + st["escaped_MeV"] - st["emitted_MeV"]) < 2e-5 * st["emitted_MeV"]
    assert st["deposited_MeV"] / r["stats"]["deposited"] == pytest.approx(1.0, abs=2e-3)
    big = f["organs"]["n_voxels"] >= 20
    gm, gs = organs["mean_Gy_per_decay"][big], organs["sigma_mean"][big]
    om, osig = f["organs"]["mean"][big], f["organs"]["sigma_mean"][big]
    assert np.all(np.abs(gm - om) <= np.maximum(0.01 * om, 3.0 * np.sqrt(gs ** 2 + osig ** 2)))


def test_cfg4_full_size_properties(anm, tables):
    cfg = anm_inputs.make_config(4)                      # 157 M voxels; tally volumes of 630 MB each
    assert cfg["shape"] == (512, 512, 600)
    n, B = 20_000_000, 100
    res = {}
    with anm.Simulation(0) as sim:
        sim.load_config(cfg, tables, n_batches=B, collect_stats=1)
        for sched in (2, 1):
            sim.set_options(n_batches=B, collect_stats=1, schedule=sched, photons_per_decay=2, rayleigh_on=1,
                            photon_cutoff_MeV=0.010, positron_ke_MeV=cfg["positron_ke_mev"])
            sim.run(n, cfg["seed"])
            res[sched] = sim.get_stats()
        e = sim.get_energy()
        organs = sim.get_organ_doses()
    a, b = res[2], res[1]
    for k in ("n_steps", "n_real", "n_pe", "n_compton", "n_rayleigh", "n_escaped", "n_cutoff"):
        assert a[k] == b[k], k
    for st in (a, b):
        assert abs(st["deposited_MeV"] + st["escaped_MeV"] - st["emitted_MeV"]) < 2e-5 * st["emitted_MeV"]
    assert float(e.sum(dtype=np.float64)) == pytest.approx(b["deposited_MeV"], rel=1e-5)
    # positron energy lands where the activity is: no energy in voxels farther than a few cm from the body
    air_far = ((cfg["material"] == 0) & (cfg["activity"] == 0)).reshape(-1)
    assert e[air_far].sum(dtype=np.float64) < 2e-3 * b["deposited_MeV"]      # 1.2 mg/cm^3 air absorbs almost nothing
    # the same analytic patient at half the resolution absorbs the same fraction of the emitted energy (within 1 %)
    half = anm_inputs.make_config(4, 2)
    with anm.Simulation(0) as sim:
        sim.load_config(half, tables, n_batches=B, collect_stats=1)
        sim.run(4_000_000, half["seed"])
        sh = sim.get_stats()
        oh = sim.get_organ_doses()
    assert (a["deposited_MeV"] / a["emitted_MeV"]) / (sh["deposited_MeV"] / sh["emitted_MeV"]) == pytest.approx(1.0, abs=0.01)
    big = organs["n_voxels"] > 20000
    assert big.sum() >= 8
    assert np.allclose(organs["mean_Gy_per_decay"][big], oh["mean_Gy_per_decay"][big], rtol=0.05)
    print("cfg4 full size: %.3e decays/s (schedule 2), steps/decay %.2f" % (n / ((a["ms_transport"] + a["ms_fold"]) * 1e-3), a["n_steps"] / n))


def test_cfg4_full_size_voxel_by_voxel(anm, tables):
    """The full 157 M-voxel grid against the lockstep oracle (same histories): energy map voxel by voxel on
    2e5 of its decays, 100 batches."""
    cfg = anm_inputs.make_config(4)
    n, B, seed = 200_000, 100, cfg["seed"]
    with anm.Simulation(0) as sim:
        sim.load_config(cfg, tables, n_batches=B)
        sim.run(n, seed)
        e_g = sim.get_energy().astype(np.float64)
    o = O.Oracle(cfg, tables, n_decays=n, n_batches=B, seed=seed, tracking=3)
    r = o.run_parallel(2)
    e_o = r["sum"]
    hit = (e_o > 0) | (e_g > 0)
    ok = np.abs(e_g - e_o) <= 1e-4 * e_o + 1e-9
    print("cfg4 full size: voxels with energy %d, identical %.5f, sum ratio %.7f" % (int(hit.sum()), ok[hit].mean(), e_g.sum() / e_o.sum()))
    # 0.98 mm voxels, coordinates up to 180 cm: an fp32 position (ulp 1.5e-5 cm) lands across a voxel face more often
    # than on the 2 mm grid (measured 99.79 %); a displaced deposit shows up in two voxels
    assert ok[hit].mean() > 0.995
    assert e_g.sum() == pytest.approx(e_o.sum(), rel=5e-5)
