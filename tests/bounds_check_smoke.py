"""Smoke-sized run of every kernel variant of libanm.so: every schedule / tally / estimator combination, the merge, the
parity hooks, a point source, the image front end and the roofline microbenchmarks.  Written for the bounds-checking
build (-DANM_BOUNDS_CHECK; profiles/r2_sanitizer.md): it adds up anm_stats.n_check_violations and prints the total.

    ANM_LIBRARY=<a build of the library> python tests/bounds_check_smoke.py       (run by tests/test_gpu_bounds_check.py)

Not a pytest module (no test_ prefix); exits non-zero on any API error."""
import os, sys
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import numpy as np
import anm_inputs
VIOL = 0
from paper_2111_11687_b200 import Simulation
tables = anm_inputs.make_tables(); et = anm_inputs.make_electron_tables()
cfg = anm_inputs.make_config(3, 8)       # 32 x 32 x 50 patient
n = int(os.environ.get("SAN_N", "20000"))
variants = [dict(schedule=1), dict(schedule=1, warp_aggregate=1), dict(schedule=2), dict(schedule=2, warp_aggregate=1),
            dict(schedule=2, tally=2), dict(schedule=2, electron_transport=1), dict(schedule=2, uncertainty=1),
            dict(schedule=2, electron_transport=1, uncertainty=1), dict(schedule=2, batch_pipeline=1), dict(schedule=2, hull_majorant=2),
            dict(schedule=2, collect_stats=0)]
with Simulation(0) as sim:
    sim.load_config(cfg, tables, n_batches=10)
    sim.set_electron_tables(et)
    for v in variants:
        kw = dict(n_batches=10, photons_per_decay=2, rayleigh_on=1, positron_ke_MeV=cfg["positron_ke_mev"], collect_stats=1); kw.update(v)
        sim.set_options(**kw)
        sim.run(n, 42)
        st = sim.get_stats()
        e = sim.get_energy(); d = sim.get_dose(); u = sim.get_uncertainty(); o = sim.get_organ_doses()
        VIOL += st["n_check_violations"]
        print("variant %s: deposited %.1f MeV, %d launches, %d check violations" % (v, st["deposited_MeV"], st["n_launches"], st["n_check_violations"]), flush=True)
    # merge path (emulated second shard: merge with itself is refused unless counts fit; use anm_merge on own rows)
    s, q, rows = sim.get_tally_buffers()
    sim.merge(n, 10, rows.cpu().numpy(), sim.get_stats())
    print("merge ok", flush=True)
    # parity hooks
    sim.philox_blocks(1, np.arange(64, dtype=np.uint32).reshape(16, 4))
    el = np.array([[10.0, 10.0, 10.0, 1.0, 0.0, 0.0, 0.3], [20.0, 20.0, 40.0, 0.0, 0.6, 0.8, 0.5]], np.float32)
    sim.trace_electrons(el)
    a = sim.get_alias_table()
    print("hooks ok, alias entries", len(a), flush=True)
# point source + single photons (cfg0-like) both schedules
cfg0 = anm_inputs.make_config(0, 2)
with Simulation(0) as sim:
    for sch in (1, 2):
        sim.load_config(cfg0, tables, n_batches=10, schedule=sch, collect_stats=1, positron_ke_MeV=0.2498)
        sim.run(n, 1)
    print("cfg0 ok", flush=True)
# front end
img = anm_inputs.make_ct_pet(cfg, ct_shape=(48, 40, 60))
with Simulation(0) as sim:
    sim.set_grid(cfg["shape"], cfg["spacing_mm"])
    sim.load_ct(img["ct_hu"], img["ct_shape"], img["ct_spacing_mm"], img["ct_offset_mm"])
    sim.load_pet(img["pet_bqml"], img["pet_shape"], img["pet_spacing_mm"], img["pet_offset_mm"])
    m, r = sim.get_phantom()
    sim.load_organs(cfg["labels"], cfg["n_organs"])
    sim.set_physics_tables(tables); sim.set_options(n_batches=10)
    sim.run(n, 3)
    print("front end ok", flush=True)
    p = sim.measure_peaks(1 << 20, 1 << 22)
    print("peaks ok", flush=True)
print("TOTAL check violations:", VIOL)
