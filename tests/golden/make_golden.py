"""Writes the stored oracle results under tests/golden/ -- calls ONLY oracle/ and anm_inputs/.

    python tests/golden/make_golden.py --cfg 3 --decays 100000000 --procs 8
    python tests/golden/make_golden.py --cfg 3 --decays 1000000000 --procs 6 --tag _1e9     (the north-star target size)

For config k at full size this runs the CPU oracle (oracle/anm_oracle.cpp) on N decays in 100 batches
with seed 1000 + (the config's seed) -- deliberately NOT the seed the CUDA run uses, so the two
estimates are statistically independent -- and writes
  cfg<k>_oracle_meta.json     run parameters, counters, total deposited / escaped energy, wall time
  cfg<k>_oracle_organs.csv    per organ: Eq. 2 mean (Gy/decay), batch sigma of the mean, Eq. 3 RMS,
                              mass-weighted dose, voxel counts
  cfg<k>_oracle_voxels.csv    a seeded random sample of the non-air voxels (material != 0; the paper sets the
                              dose in air to zero) with oracle dose > 5 % of their maximum:
                              linear index, sum_b x, sum_b x^2 (MeV, MeV^2)  ->  per-voxel z-scores.
                              The 5 % pre-selection is deliberately wider than north_star's "> 10 % of max":
                              the test applies the 10 % cut to the MEAN of the two estimates, which is
                              uncorrelated with their difference; cutting on the oracle's own noisy value
                              would select its upward fluctuations and bias z (regression to the mean).
No value in these files comes from the CUDA path.
"""
import argparse
import json
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import anm_inputs                         # noqa: E402
from oracle import anm_oracle as O        # noqa: E402


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--cfg", type=int, required=True)
    ap.add_argument("--decays", type=float, default=1e8)
    ap.add_argument("--procs", type=int, default=os.cpu_count())
    ap.add_argument("--sample", type=int, default=20000)
    ap.add_argument("--tag", default="", help="file-name suffix, e.g. _1e9 -> cfg3_1e9_oracle_*.{json,csv} (keeps the 1e8 files)")
    a = ap.parse_args()
    cfg = anm_inputs.make_config(a.cfg)
    tables = anm_inputs.make_tables()
    n = int(a.decays)
    seed = 1000 + cfg["seed"]
    o = O.Oracle(cfg, tables, n_decays=n, n_batches=100, seed=seed)
    r = o.run_parallel(a.procs)
    f = o.finalize(r)
    tag = os.path.join(HERE, "cfg%d%s_oracle" % (a.cfg, a.tag))
    meta = {"config": cfg["name"], "shape": cfg["shape"], "spacing_mm": cfg["spacing_mm"], "n_decays": n,
            "n_batches": 100, "seed": seed, "cores": r["cores"], "wall_seconds": r["seconds"],
            "stats": r["stats"], "max_dose_gy_per_decay_non_air": float(np.where(o.material != 0, f["dose"], 0.0).max()),
            "voxel_preselection": "non-air, oracle dose > 0.05 * max_dose_gy_per_decay_non_air",
            "written_by": "tests/golden/make_golden.py (oracle only)"}
    json.dump(meta, open(tag + "_meta.json", "w"), indent=1)
    if "organs" in f:
        og = f["organs"]
        with open(tag + "_organs.csv", "w") as fh:
            fh.write("label,name,mean_gy_per_decay,sigma_mean,rms_voxel_rel_sigma,mass_weighted_gy_per_decay,mass_g,n_voxels,n_voxels_nonzero\n")
            for i, name in enumerate(cfg["organ_names"]):
                fh.write("%d,%s,%.9e,%.9e,%.9e,%.9e,%.9e,%d,%d\n" % (
                    i + 1, name, og["mean"][i], og["sigma_mean"][i], og["rms_voxel_rel_sigma"][i],
                    og["mass_weighted"][i], og["mass_g"][i], og["n_voxels"][i], og["n_voxels_nonzero"][i]))
    dose_na = np.where(o.material != 0, f["dose"], 0.0)
    pop = np.nonzero(dose_na > 0.05 * dose_na.max())[0]
    rng = np.random.default_rng(2111)
    pick = np.sort(rng.choice(pop, size=min(a.sample, pop.size), replace=False))
    with open(tag + "_voxels.csv", "w") as fh:
        fh.write("voxel,sum_mev,sumsq_mev2\n")
        for v in pick:
            fh.write("%d,%.9e,%.9e\n" % (v, r["sum"][v], r["sumsq"][v]))
    print(json.dumps(meta))


if __name__ == "__main__":
    main()
