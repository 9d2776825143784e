"""Pin of the oracle's run-level statistical-uncertainty figure ("0.47 %", L117 "1.19 %": one figure per
run, definition not given; reading C17: RMS of the voxels' relative sigma over the NON-AIR voxels whose dose
exceeds 10 % / 50 % of the largest non-air voxel dose).  The finalize arithmetic is checked on a hand-worked example
whose every number can be verified by eye, and against an explicit Python loop on random tallies."""
import numpy as np
import pytest

import anm_inputs
from oracle import anm_oracle as O

AIR, WATER = 0, 2


def _oracle(mat, rho, n_decays, B):
    n = len(mat)
    cfg = {"shape": (n, 1, 1), "spacing_mm": (10.0, 10.0, 10.0), "material": np.asarray(mat, np.uint8).reshape(1, 1, n),
           "density": np.asarray(rho, np.float32).reshape(1, 1, n), "activity": None, "point_source_mm": (5.0, 5.0, 5.0),
           "labels": None, "n_organs": 0, "n_decays": n_decays, "n_batches": B, "seed": 1, "photons_per_decay": 1,
           "rayleigh_on": 1, "photon_cutoff_mev": 0.010, "positron_ke_mev": 0.0}
    return O.Oracle(cfg, anm_inputs.make_tables())


def test_hand_worked_example():
    """Five 1 cm^3 voxels, B = 2 batches of one decay each.  Batch energies (MeV):
         voxel      0 (air)   1 (water)  2 (water)  3 (water, rho 2)  4 (water)
         batch 0    50        6          1          8                 0.2
         batch 1    50        4          3          12                0.2
       sum          100       10         4          20                0.4
       dose ~ S/rho (air rho 0.001: 1e5 -- would dominate the maximum; it is excluded)
                    --        10         4          10                0.4     -> max = 10
       rel sigma = sqrt((B Q / S^2 - 1) / (B - 1)), Q = sum of squares:
         voxel 1: Q = 52,  2*52/100 - 1 = 0.04 -> 0.2      voxel 2: Q = 10, 2*10/16 - 1 = 0.25 -> 0.5
         voxel 3: Q = 208, 2*208/400 - 1 = 0.04 -> 0.2     voxel 4: Q = 0.08, 2*0.08/0.16 - 1 = 0 -> 0
       > 10 % of max (dose > 1): voxels 1, 2, 3 -> RMS = sqrt((0.04 + 0.25 + 0.04) / 3) = 0.331662...
       > 50 % of max (dose > 5): voxels 1, 3    -> RMS = 0.2"""
    o = _oracle([AIR, WATER, WATER, WATER, WATER], [0.001, 1.0, 1.0, 2.0, 1.0], 2, 2)
    b0 = np.array([50.0, 6.0, 1.0, 8.0, 0.2]); b1 = np.array([50.0, 4.0, 3.0, 12.0, 0.2])
    f = o.finalize({"sum": b0 + b1, "sumsq": b0 ** 2 + b1 ** 2})
    assert f["n_voxels_gt10"] == 3 and f["n_voxels_gt50"] == 2
    assert f["rms_rel_sigma_gt10"] == pytest.approx(np.sqrt(0.33 / 3.0), rel=1e-12)
    assert f["rms_rel_sigma_gt50"] == pytest.approx(0.2, rel=1e-12)
    # the maximum is voxel 1's (or 3's) dose: 10 MeV in 1 g over 2 decays
    assert f["max_dose"] == pytest.approx(10.0 * 1.602176634e-10 / 2.0, rel=1e-12)
    # with the air voxel counted as body (material 2) its huge dose would set the maximum and empty the population
    o2 = _oracle([WATER, WATER, WATER, WATER, WATER], [0.001, 1.0, 1.0, 2.0, 1.0], 2, 2)
    f2 = o2.finalize({"sum": b0 + b1, "sumsq": b0 ** 2 + b1 ** 2})
    assert f2["n_voxels_gt10"] == 1 and f2["rms_rel_sigma_gt10"] == 0.0


def test_against_an_explicit_loop():
    rng = np.random.default_rng(5)
    n, B, N = 400, 20, 2000
    mat = rng.choice([AIR, 1, WATER, 3], size=n).astype(np.uint8)
    rho = np.where(mat == AIR, 0.0012, rng.uniform(0.2, 1.9, n)).astype(np.float32)
    xb = rng.gamma(2.0, 1.0, size=(B, n)) * rng.uniform(0.0, 1.0, n) ** 3       # a wide range of doses
    S, Q = xb.sum(0), (xb ** 2).sum(0)
    f = _oracle(mat, rho, N, B).finalize({"sum": S, "sumsq": Q})
    dose = [S[i] / float(rho[i]) for i in range(n)]
    dmax = max(dose[i] for i in range(n) if mat[i] != AIR)
    for name, frac in (("gt10", 0.1), ("gt50", 0.5)):
        acc, cnt = 0.0, 0
        for i in range(n):
            if mat[i] == AIR or not dose[i] > frac * dmax:
                continue
            yb = xb[:, i] / (N / B)
            sem = np.std(yb, ddof=1) / np.sqrt(B)                  # standard error of the mean over batches
            acc += (sem / yb.mean()) ** 2; cnt += 1
        assert f["n_voxels_" + name] == cnt and cnt > 0
        assert f["rms_rel_sigma_" + name] == pytest.approx(np.sqrt(acc / cnt), rel=1e-9)
