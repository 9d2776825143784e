"""Pins of the oracle's LOCKSTEP mode (tracking = 2 / 3: Woodcock tracking with the CUDA path's documented draw schedule,
without / with the hull majorant; SURVEY.md §8(c) "lockstep", pin P6 "Woodcock vs exact DDA") against the oracle's own
exact voxel-boundary transport: different algorithms, same distribution.  What lockstep is FOR -- following the CUDA
path history by history -- is tested on the GPU (tests/test_gpu_lockstep.py); here it must first be right."""
import numpy as np
import pytest

import anm_inputs
from oracle import anm_oracle as O


@pytest.fixture(scope="module")
def tables():
    return anm_inputs.make_tables()


def _point_cfg(scale=8, src=(271.0, 231.0, 1130.0), **kw):
    base = anm_inputs.make_config(3, scale)
    return dict(base, activity=None, point_source_mm=src, **kw)


@pytest.mark.parametrize("tracking", [2, 3])
def test_lockstep_agrees_with_exact_tracking(tables, tracking):
    cfg = _point_cfg()
    n, B = 200_000, 20
    a = O.Oracle(cfg, tables, n_decays=n, n_batches=B, seed=11)
    ra = a.run_parallel(8); fa = a.finalize(ra)
    b = O.Oracle(cfg, tables, n_decays=n, n_batches=B, seed=12, tracking=tracking)
    rb = b.run_parallel(8); fb = b.finalize(rb)
    sa, sb = ra["stats"], rb["stats"]
    assert sb["max_history_residual"] < 2e-9 and sa["max_history_residual"] < 2e-9       # energy conservation per history
    # total deposited energy: per-decay spread <= 0.6 MeV
    assert abs(sa["deposited"] - sb["deposited"]) / n < 4.0 * np.sqrt(2.0) * 0.6 / np.sqrt(n)
    for k in ("n_compton", "n_pe", "n_rayleigh", "n_escaped"):
        assert sa[k] == pytest.approx(sb[k], rel=4.0 / np.sqrt(min(sa[k], sb[k])) + 1e-3), k
    big = fa["organs"]["n_voxels"] >= 4
    d = np.abs(fa["organs"]["mean"][big] - fb["organs"]["mean"][big])
    s = np.sqrt(fa["organs"]["sigma_mean"][big] ** 2 + fb["organs"]["sigma_mean"][big] ** 2)
    assert np.all(d <= 4.5 * s + 1e-3 * fa["organs"]["mean"][big])


def test_hull_majorant_changes_the_steps_not_the_physics(tables):
    """Source in the skin: many photons leave the body at once.  With the hull majorant they take fewer sub-steps in the
    air margin; the deposits follow the same distribution."""
    cfg = _point_cfg(src=(256.0, 150.0, 640.0))
    n, B = 100_000, 10
    r2 = O.Oracle(cfg, tables, n_decays=n, n_batches=B, seed=3, tracking=2).run_parallel(8)
    r3 = O.Oracle(cfg, tables, n_decays=n, n_batches=B, seed=3, tracking=3).run_parallel(8)
    assert r3["stats"]["n_substeps"] < 0.8 * r2["stats"]["n_substeps"]          # every Woodcock sub-step, real or virtual
    assert abs(r2["stats"]["deposited"] - r3["stats"]["deposited"]) / n < 4.0 * np.sqrt(2.0) * 0.6 / np.sqrt(n)
    assert r2["stats"]["n_compton"] == pytest.approx(r3["stats"]["n_compton"], rel=0.01)


def test_lockstep_source_follows_the_activity_pdf(tables):
    """The lockstep source (alias table rebuilt by the ordered sweep, bucket from 64 random bits) must draw decay voxels
    with probability a_v / sum(a) like the oracle's own inverse-CDF pick (P8).  Near-vacuum phantom: the photons leave
    without interacting, the 1 MeV 'positron energy' stays in the decay voxel, so the energy map counts the decays."""
    cfg = anm_inputs.make_config(3, 16)
    cfg = dict(cfg, density=np.full_like(cfg["density"], 1e-4), material=np.zeros_like(cfg["material"]),
               positron_ke_mev=1.0, photons_per_decay=1)
    n = 400_000
    r = O.Oracle(cfg, tables, n_decays=n, n_batches=4, seed=9, tracking=2).run_parallel(4)
    assert r["stats"]["n_collisions"] < 400
    counts = r["sum"]
    a = cfg["activity"].astype(np.float64).reshape(-1)
    expect = n * a / a.sum()
    assert counts[a == 0].sum() < 400 * 0.6            # nothing where there is no activity (a stray collision aside)
    sel = expect > 5
    chi2 = ((counts[sel] - expect[sel]) ** 2 / expect[sel]).sum()
    dof = sel.sum() - 1
    assert abs(chi2 - dof) < 5.0 * np.sqrt(2.0 * dof), (chi2, dof)
    # the hottest voxels individually
    top = np.argsort(expect)[-20:]
    assert np.all(np.abs(counts[top] - expect[top]) < 5.0 * np.sqrt(expect[top]))
