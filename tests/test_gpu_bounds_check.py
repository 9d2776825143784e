"""compute-sanitizer is closed on this pool (profiles/r2_sanitizer.md), so the out-of-range accesses it would look for are
looked for by the library itself: a build with -DANM_BOUNDS_CHECK tests every index the transport kernels form (voxel,
material, energy-grid cell, alias bucket, pool slot, ring fill, deposit-list and electron-array position, local batch)
and counts violations in anm_stats.n_check_violations.  This test compiles that build into a temporary file and runs
every kernel variant on it in a separate process (tests/bounds_check_smoke.py): 0 violations."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_no_index_out_of_range_in_any_kernel_variant(tmp_path):
    from paper_2111_11687_b200 import build
    lib = build.build(out=str(tmp_path / "libanm_check.so"), extra=["-DANM_BOUNDS_CHECK"])
    env = dict(os.environ, ANM_LIBRARY=lib, SAN_N="100000")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "bounds_check_smoke.py")], env=env, cwd=ROOT,
                       capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-2000:]
    assert "TOTAL check violations: 0" in r.stdout, r.stdout[-2000:]
    assert r.stdout.count("0 check violations") >= 11          # one line per kernel variant
    # and the normal build reports the field as zero, always
    import anm_inputs
    from paper_2111_11687_b200 import Simulation
    cfg = anm_inputs.make_config(0, 4)
    with Simulation(0) as sim:
        sim.load_config(cfg, anm_inputs.make_tables(), n_batches=10, collect_stats=1)
        sim.run(10_000, 1)
        assert sim.get_stats()["n_check_violations"] == 0
