"""Parity of the CUDA history-by-history uncertainty (anm_options.uncertainty = 1, Walters et al. 2002;
SURVEY.md §8(f) NEXT-4) with the oracle and with what the estimator's definition fixes, through the C ABI."""
import os

import numpy as np
import pytest

import anm_inputs
from oracle import anm_oracle as O

pytestmark = pytest.mark.gpu
E0 = 0.51099895
NPROC = min(32, os.cpu_count() or 1)


@pytest.fixture(scope="module")
def anm():
    import paper_2111_11687_b200 as pkg
    return pkg


@pytest.fixture(scope="module")
def tables():
    return anm_inputs.make_tables()


def _run(anm, cfg, tables, n, B, mode, seed=None, **opts):
    with anm.Simulation(0) as sim:
        sim.load_config(cfg, tables, n_batches=B, collect_stats=1, uncertainty=mode, **opts)
        sim.run(n, cfg["seed"] if seed is None else seed)
        out = {"energy": sim.get_energy().astype(np.float64), "rel": sim.get_uncertainty().astype(np.float64),
               "stats": sim.get_stats()}
        if cfg.get("n_organs"):
            out["organs"] = sim.get_organ_doses()
    return out


def test_same_histories_same_energy_and_one_history_per_batch(anm, tables):
    """Scoring history by history changes only how a decay's deposits reach the tally (merged per voxel first): the
    energy map is the batch run's up to fp32 summation order, every counter is equal; and with ONE decay per batch the
    batch estimator is the history-by-history estimator, so the two uncertainty maps must coincide."""
    cfg = anm_inputs.make_config(3, 8)
    n = 20_000
    b = _run(anm, cfg, tables, n, n, 0)            # B = N: one decay per batch
    h = _run(anm, cfg, tables, n, 50, 1)
    for k in ("n_steps", "n_real", "n_pe", "n_compton", "n_rayleigh", "n_escaped", "n_cutoff"):
        assert b["stats"][k] == h["stats"][k], k
    assert h["stats"]["n_hbh_overflow"] == 0
    assert np.allclose(h["energy"], b["energy"], rtol=2e-6, atol=1e-6)
    hit = b["energy"] > 0
    assert hit.sum() > 1000
    assert np.allclose(h["rel"][hit], b["rel"][hit], rtol=2e-4, atol=1e-6)
    assert np.all(h["rel"][~hit] == 0)


def test_photoelectric_only_closed_form(anm, tables):
    """Every collision absorbs the photon (Compton, Rayleigh 1e-30 in the tables), one photon per history: X_h is 0 or
    E0, so rel sigma^2 = (1/p - 1) / (N - 1) with p = hits / N, exactly."""
    t = dict(tables)
    t["mu_compton"] = np.full_like(tables["mu_compton"], 1e-30)
    t["mu_rayleigh"] = np.full_like(tables["mu_rayleigh"], 1e-30)
    t["mu_pe"] = tables["mu_pe"] * 50.0
    cfg = anm_inputs.make_config(0, 2)
    n = 200_000
    h = _run(anm, cfg, t, n, 10, 1)
    assert h["stats"]["n_compton"] == 0 and h["stats"]["n_pe"] > 500
    hit = h["energy"] > 0
    p = h["energy"][hit] / E0 / n
    assert np.allclose(np.rint(p * n), p * n, atol=1e-2)                 # whole numbers of photons
    assert np.allclose(h["rel"][hit] ** 2, (1.0 / p - 1.0) / (n - 1.0), rtol=1e-4)


def test_a_decay_is_one_history(anm, tables):
    """One 100 m voxel, point source at its centre, pairs + positron energy: every decay leaves 2 E0 + 0.2498 MeV in
    the voxel, so the variance is zero -- only if positron, photon A and photon B are scored as ONE history."""
    cfg = {"name": "one_voxel", "shape": (1, 1, 1), "spacing_mm": (1e5, 1e5, 1e5), "material": np.full((1, 1, 1), 2, np.uint8),
           "density": np.full((1, 1, 1), 1.0, np.float32), "activity": None, "point_source_mm": (5e4, 5e4, 5e4),
           "labels": None, "n_organs": 0, "n_decays": 5000, "n_batches": 5, "seed": 2, "photons_per_decay": 2,
           "rayleigh_on": 1, "photon_cutoff_mev": 0.010, "positron_ke_mev": 0.2498}
    h = _run(anm, cfg, tables, 5000, 5, 1)
    assert h["stats"]["n_escaped"] == 0
    assert h["energy"][0] == pytest.approx(5000 * (2 * E0 + 0.2498), rel=1e-5)
    # fp32 tallies: S and sum X^2 carry ~1e-5 relative rounding after 5000 RED.ADDs, i.e. rel sigma ~ sqrt(1e-5 / N) = 5e-5;
    # separate photon histories would give 0.57 / sqrt(N) = 8e-3
    assert h["rel"][0] < 0.04 * 0.57 / np.sqrt(5000)


def test_hbh_sigma_vs_oracle_patient(anm, tables):
    """cfg3 / 4, 2e6 decays: the history-by-history sigma maps of the two sides estimate the same quantity; over the
    voxels above 10 % of the maximum dose their ratio is 1 on average (each side's estimate scatters by ~1/sqrt(2 hits))."""
    cfg = anm_inputs.make_config(3, 4)
    n, B = 2_000_000, 100
    g = _run(anm, cfg, tables, n, B, 1)
    o = O.Oracle(cfg, tables, n_decays=n, n_batches=B, seed=cfg["seed"] + 1000)
    r = o.run_parallel(NPROC, hbh=True)
    f = o.finalize(r)
    assert g["stats"]["n_hbh_overflow"] == 0
    mass = cfg["density"].reshape(-1).astype(np.float64)
    # population chosen on the mean of the two dose estimates (reading C25: a cut on one side's own noisy value
    # biases the comparison); ratio of the sums, not the mean of the ratios (E[1/x] > 1/E[x] for a noisy denominator)
    dose_m = np.where(cfg["material"].reshape(-1) != 0, 0.5 * (f["energy"] + g["energy"]) / np.maximum(mass, 1e-9), 0.0)
    sel = dose_m > 0.1 * dose_m.max()
    assert sel.sum() > 2000
    assert g["rel"][sel].sum() / f["rel_sigma_hbh"][sel].sum() == pytest.approx(1.0, abs=0.01)
    assert np.std(g["rel"][sel] / f["rel_sigma_hbh"][sel]) < 0.15
    # the history-by-history and the batch estimate of one run agree on average; Eq. 3 (organ RMS of the voxel sigmas)
    # follows the chosen estimator, the organ's sigma of the mean stays the batch one
    gb = _run(anm, cfg, tables, n, B, 0)
    assert np.sqrt((g["rel"][sel] ** 2).sum() / (gb["rel"][sel] ** 2).sum()) == pytest.approx(1.0, abs=0.02)
    big = g["organs"]["n_voxels"] >= 50
    assert np.allclose(g["organs"]["rms_voxel_rel_sigma"][big], gb["organs"]["rms_voxel_rel_sigma"][big], rtol=0.1)
    assert not np.array_equal(g["organs"]["rms_voxel_rel_sigma"][big], gb["organs"]["rms_voxel_rel_sigma"][big])
    assert np.allclose(g["organs"]["sigma_mean"][big], gb["organs"]["sigma_mean"][big], rtol=1e-3)
    assert np.allclose(g["organs"]["rms_voxel_rel_sigma"][big], f["organs"]["rms_voxel_rel_sigma"][big], rtol=0.2)


def test_hbh_error_codes(anm, tables):
    cfg = anm_inputs.make_config(3, 16)
    with anm.Simulation(0) as sim:
        sim.load_config(cfg, tables, n_batches=4)
        with pytest.raises(anm.AnmError) as e:
            sim.set_options(n_batches=4, uncertainty=2)
        assert e.value.code == -1
        with pytest.raises(anm.AnmError) as e:
            sim.set_options(n_batches=4, uncertainty=1, schedule=1)
        assert e.value.code == -5
        sim.set_options(n_batches=4, uncertainty=1)
        sim.run(4000, 1)
        # back to the batch estimator on the same ctx
        sim.set_options(n_batches=4, uncertainty=0)
        sim.run(4000, 1)
        assert sim.get_uncertainty().max() > 0
