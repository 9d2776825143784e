"""Pins of the oracle's history-by-history uncertainty ("the corresponding uncertainty is evaluated using
the history-by-history method (Walters et al., 2002)") against what the definition fixes:
s^2 of the mean = (sum_h X_h^2 / N - (sum_h X_h / N)^2) / (N - 1), X_h = the energy history h leaves in the voxel."""
import numpy as np
import pytest

import anm_inputs
from oracle import anm_oracle as O

E0 = 0.51099895


@pytest.fixture(scope="module")
def tables():
    return anm_inputs.make_tables()


def test_one_history_per_batch_is_the_same_estimator(tables):
    """With one decay per batch the batch tally's sum of squares IS sum_h X_h^2: an independent route to the same
    number (the batch fold shares no bookkeeping with the last-history / temp arrays)."""
    cfg = anm_inputs.make_config(3, 16)
    n = 3000
    o = O.Oracle(cfg, tables, n_decays=n, n_batches=n, seed=11)
    r = o.run(hbh=True)
    assert r["sumsq"].sum() > 0
    assert np.allclose(r["hbh_sumsq"], r["sumsq"], rtol=1e-12, atol=0)
    # and with coarser batches the two differ (several histories share a batch) while the sums agree
    r2 = O.Oracle(cfg, tables, n_decays=n, n_batches=10, seed=11).run(hbh=True)
    assert np.allclose(r2["hbh_sumsq"], r["hbh_sumsq"], rtol=1e-12, atol=0)
    assert np.allclose(r2["sum"], r["sum"], rtol=1e-12, atol=0)
    assert r2["sumsq"].sum() > 1.5 * r2["hbh_sumsq"].sum()


def test_photoelectric_only_is_bernoulli(tables):
    """Compton and Rayleigh switched off in the tables (1e-30): every collision absorbs the photon, so with one photon
    per history X_h is 0 or E0 and sum X^2 = E0 sum X exactly; rel sigma^2 = (1/p - 1) / (N - 1) with p = hits / N."""
    t = dict(tables)
    t["mu_compton"] = np.full_like(tables["mu_compton"], 1e-30)
    t["mu_rayleigh"] = np.full_like(tables["mu_rayleigh"], 1e-30)
    t["mu_pe"] = tables["mu_pe"] * 50.0
    cfg = anm_inputs.make_config(0, 2)
    n = 20000
    o = O.Oracle(cfg, t, n_decays=n, n_batches=4, seed=3)
    r = o.run(hbh=True)
    f = o.finalize(r)
    assert r["stats"]["n_compton"] == 0 and r["stats"]["n_pe"] > 0
    assert np.allclose(r["hbh_sumsq"], E0 * r["sum"], rtol=1e-12, atol=0)
    hit = r["sum"] > 0
    p = r["sum"][hit] / E0 / n
    assert np.allclose(f["rel_sigma_hbh"][hit] ** 2, (1.0 / p - 1.0) / (n - 1.0), rtol=1e-9)


def test_a_decay_is_one_history(tables):
    """One enormous voxel: every decay leaves positron energy + both photons in it, X_h = 0.2498 + 2 E0 for every h, so
    the variance is zero.  (Scoring the two photons as separate histories would give sum X^2 = N (KE^2 + 2 E0^2).)"""
    cfg = {"shape": (1, 1, 1), "spacing_mm": (1e9, 1e9, 1e9), "material": np.full((1, 1, 1), 2, np.uint8),
           "density": np.full((1, 1, 1), 1.0, np.float32), "activity": np.ones((1, 1, 1), np.float32),
           "point_source_mm": None, "labels": None, "n_organs": 0, "n_decays": 500, "n_batches": 5, "seed": 2,
           "photons_per_decay": 2, "rayleigh_on": 1, "photon_cutoff_mev": 0.010, "positron_ke_mev": 0.2498}
    o = O.Oracle(cfg, tables)
    # the decay point is uniform in the 1000 km voxel: a photon born within a few mean free paths of a face could leave
    r = o.run(hbh=True)
    x = 0.2498 + 2 * E0
    if r["stats"]["n_escaped"] == 0:
        assert r["hbh_sumsq"][0] == pytest.approx(500 * x * x, rel=1e-12)
        assert o.finalize(r)["rel_sigma_hbh"][0] < 1e-6
    else:
        pytest.skip("a photon escaped the voxel")


def test_hbh_sigma_is_calibrated_and_agrees_with_the_batch_sigma(tables):
    """K independent runs: the spread of a voxel's mean over the runs equals the history-by-history sigma each run
    reports (ratio 1 +- 0.15 averaged over voxels), and the batch sigma estimates the same quantity."""
    cfg = anm_inputs.make_config(1, 10)            # 10^3 voxels of 20 mm water, single active centre voxel
    K, n, B = 24, 20000, 20
    means, s_h, s_b = [], [], []
    for k in range(K):
        o = O.Oracle(cfg, tables, n_decays=n, n_batches=B, seed=100 + k)
        f = o.finalize(o.run(hbh=True))
        means.append(f["energy"] / n)
        s_h.append(f["rel_sigma_hbh"] * f["energy"] / n)
        s_b.append(f["rel_sigma"] * f["energy"] / n)
    means, s_h, s_b = np.array(means), np.array(s_h), np.array(s_b)
    sel = means.mean(0) > 0.02 * means.mean(0).max()
    emp = means.std(0, ddof=1)[sel]
    rms_h = np.sqrt((s_h ** 2).mean(0))[sel]
    rms_b = np.sqrt((s_b ** 2).mean(0))[sel]
    assert sel.sum() >= 20
    assert np.mean(emp / rms_h) == pytest.approx(1.0, abs=0.1)
    assert np.mean(rms_b / rms_h) == pytest.approx(1.0, abs=0.05)
    # the HbH estimate has N - 1 degrees of freedom, the batch estimate only B - 1: it scatters far less from run to run
    assert np.mean(s_h.std(0)[sel] / rms_h) < 0.5 * np.mean(s_b.std(0)[sel] / rms_b)


def test_parallel_runs_add_up(tables):
    cfg = anm_inputs.make_config(3, 16)
    o = O.Oracle(cfg, tables, n_decays=4000, n_batches=8, seed=5)
    a = o.run(hbh=True)
    b = o.run_parallel(4, hbh=True)
    assert np.allclose(a["hbh_sumsq"], b["hbh_sumsq"], rtol=1e-12, atol=0)
    assert np.allclose(a["sum"], b["sum"], rtol=1e-12, atol=0)
