"""Pins of two steps of the oracle's history that nothing else observes from outside ("softest spot"):
  * the two annihilation photons leave in exactly opposite directions ("two 0.511 MeV photons are emitted
    in opposite directions"), and
  * the deflection of a Compton-scattered photon, cos(theta) = 1 + 1/alpha - 1/(alpha eps).
Both are read off the GEOMETRY of the deposits the oracle's own transport leaves in a fine voxel grid, with cross
sections crafted so that every history has a known structure; neither test restates the oracle's formula for the
quantity it checks against: the angle comes from voxel positions, the energies from the tally."""
import numpy as np
import pytest

import anm_inputs
from oracle import anm_oracle as O

E0 = 0.51099895
WATER = 2


def _grid_cfg(n, d_mm, rho, photons):
    mat = np.full((n, n, n), WATER, np.uint8)
    dens = np.full((n, n, n), rho, np.float32)
    c = 0.5 * n * d_mm
    return {"shape": (n, n, n), "spacing_mm": (d_mm,) * 3, "material": mat, "density": dens, "activity": None,
            "point_source_mm": (c, c, c), "labels": None, "n_organs": 0, "seed": 1, "photons_per_decay": photons,
            "rayleigh_on": 1, "photon_cutoff_mev": 0.010, "positron_ke_mev": 0.0}


def _crafted_tables(pe, compton_at_e0, compton_below):
    """Copies of the standard tables with constant coefficients (cm^2/g): photoelectric `pe` everywhere below 0.5 MeV,
    Compton `compton_at_e0` on the last grid points (E >= 0.5 MeV, where a fresh annihilation photon sits) and
    `compton_below` elsewhere; Rayleigh negligible."""
    t = dict(anm_inputs.make_tables())
    E = np.exp(t["lnE_min"] + t["dlnE"] * np.arange(t["n_energy"]))
    hi = E >= 0.5
    t["mu_pe"] = np.where(hi, 1e-9 if compton_at_e0 > 1e-6 else pe, pe)[None, :].repeat(t["n_materials"], 0).astype(np.float32)
    t["mu_compton"] = np.where(hi, compton_at_e0, compton_below)[None, :].repeat(t["n_materials"], 0).astype(np.float32)
    t["mu_rayleigh"] = np.full_like(t["mu_pe"], 1e-12)
    return t


def _voxel_centres(idx, n, d_cm):
    iz, rem = np.divmod(idx, n * n)
    iy, ix = np.divmod(rem, n)
    return (np.stack([ix, iy, iz], axis=-1) + 0.5) * d_cm


def test_annihilation_photons_are_back_to_back():
    """Pure absorber (photoelectric only, mean free path 2 cm): each photon of a pair leaves all of its 0.511 MeV in the
    voxel of its first collision.  Seen from the decay point the two voxels must lie in opposite directions -- within the
    angle a 1 mm voxel subtends at >= 1 cm -- while their distances are independent draws."""
    n, d_mm = 128, 1.0
    cfg = _grid_cfg(n, d_mm, 5.0, photons=2)
    t = _crafted_tables(pe=0.1, compton_at_e0=1e-9, compton_below=1e-9)
    N = 300
    o = O.Oracle(cfg, t, n_decays=N, n_batches=N, seed=21)
    src = np.array(cfg["point_source_mm"]) / 10.0
    cosines, ratios = [], []
    for k in range(N):
        e = o.run(k, k + 1)["sum"]
        idx = np.nonzero(e)[0]
        if len(idx) != 2 or not np.allclose(e[idx], E0, rtol=1e-12):
            continue                                   # a photon escaped, or both stopped in one voxel
        r = _voxel_centres(idx, n, d_mm / 10.0) - src
        dist = np.linalg.norm(r, axis=1)
        if dist.min() < 1.0:
            continue
        cosines.append(float(r[0] @ r[1] / (dist[0] * dist[1])))
        ratios.append(dist[0] / dist[1])
    cosines, ratios = np.array(cosines), np.array(ratios)
    assert len(cosines) > 100
    assert np.all(cosines < -0.985), cosines.max()     # a 1 mm voxel at 1 cm: < 0.1 rad off the axis, cos < -0.995 typically
    assert np.median(cosines) < -0.998
    assert np.std(np.log(ratios)) > 0.3                # the two path lengths are NOT mirrored


def test_compton_deflection_matches_the_energy_split():
    """Compton only at E0, photoelectric only below it: a single photon scatters once at r1 (leaving T = E0 - E') and is
    absorbed at r2 (leaving E').  The first-collision recorder gives T and |r1 - s|, which identify r1 without using any
    angle; then the angle between (r1 - s) and (r2 - r1), read off the voxel positions, must satisfy the Compton
    relation with eps = E' / E0 taken from the tally:  1 - cos(theta) = (1 / eps - 1) / alpha."""
    n, d_mm = 128, 1.5
    cfg = _grid_cfg(n, d_mm, 5.0, photons=1)
    t = _crafted_tables(pe=0.1, compton_at_e0=0.1, compton_below=1e-9)
    N = 700
    o = O.Oracle(cfg, t, n_decays=N, n_batches=N, seed=33)
    src = np.array(cfg["point_source_mm"]) / 10.0
    d_cm = d_mm / 10.0
    geo, kin = [], []
    for k in range(N):
        r = o.run(k, k + 1, first_collision=True)
        e = r["sum"]
        idx = np.nonzero(e)[0]
        T = float(r["fc_dep"][0])
        if len(idx) != 2 or not (0.0 < T < E0) or abs(e[idx].sum() - E0) > 1e-9:
            continue                                   # escaped, scattered twice, or both deposits in one voxel
        i1 = idx[np.argmin(np.abs(e[idx] - T))]
        i2 = idx[0] if idx[1] == i1 else idx[1]
        if abs(e[i1] - T) > 1e-9:
            continue
        p1, p2 = _voxel_centres(np.array([i1, i2]), n, d_cm)
        a, b = p1 - src, p2 - p1
        la, lb = np.linalg.norm(a), np.linalg.norm(b)
        assert abs(la - float(r["fc_dist"][0])) < 0.87 * d_cm + 1e-9       # r1 really is the first collision site
        if la < 1.5 or lb < 1.5:
            continue                                   # too short a lever for a 1.5 mm voxel
        eps = float(e[i2]) / E0
        geo.append(float(a @ b / (la * lb)))
        kin.append(1.0 - (1.0 / eps - 1.0) / 1.0)      # alpha = E0 / m c^2 = 1
    geo, kin = np.array(geo), np.array(kin)
    assert len(geo) > 100
    assert np.all(np.abs(geo - kin) < 0.2), np.abs(geo - kin).max()
    assert np.mean(np.abs(geo - kin)) < 0.05
    assert np.corrcoef(geo, kin)[0, 1] > 0.99
    assert kin.min() < -0.5 and kin.max() > 0.8        # forward and backward scatters are both in the sample
