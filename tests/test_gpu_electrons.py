"""Parity of the CUDA secondary-electron transport (anm_options.electron_transport, SURVEY.md §8(f) NEXT-2;
PAPER.md:L67) with the CPU oracle, through the C ABI.

The electron walk is deterministic, so it is compared voxel by voxel on given electrons (anm_trace_electrons vs the
oracle's walk; fp32 vs fp64: 5e-5 MeV per voxel).  Whole runs are compared statistically like the photon path
(north_star tolerances), and exactly where the method fixes it: electron transport draws no random numbers, so the
photon histories -- every counter -- are the same with it on and off."""
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


@pytest.fixture(scope="module")
def etab():
    return anm_inputs.make_electron_tables()


def _random_electrons(cfg, n, seed, t_lo=0.2005, t_hi=0.51099):      # up to a photo-electron's E0 (reading C28)
    rng = np.random.default_rng(seed)
    ext = np.array(cfg["shape"], np.float64) * np.array(cfg["spacing_mm"], np.float64)
    pos = rng.uniform(0.02, 0.98, size=(n, 3)) * ext
    d = rng.normal(size=(n, 3)); d /= np.linalg.norm(d, axis=1, keepdims=True)
    d[: n // 8, 1:] = 0.0; d[: n // 8, 0] = np.sign(d[: n // 8, 0] + 1e-30)       # some axis-parallel ones
    T = rng.uniform(t_lo, t_hi, size=(n, 1))
    return np.concatenate([pos, d, T], axis=1).astype(np.float32)


def _oracle_trace(cfg, tables, etab, electrons):
    o = O.Oracle(dict(cfg, n_decays=10, n_batches=2), tables, electron_tables=etab)
    vol = np.zeros(int(np.prod(cfg["shape"])), np.float64)
    esc = 0.0
    for e in electrons.astype(np.float64):
        dep, out = o.electron_walk(e[:3] / 10.0, e[3:6] / np.linalg.norm(e[3:6]), e[6])
        for v, x in dep:
            vol[v] += x
        esc += out
    return vol, esc


@pytest.mark.parametrize("case", ["patient_coarse", "fine_slabs"])
def test_electron_walk_voxel_by_voxel(anm, tables, etab, case):
    if case == "patient_coarse":
        cfg = anm_inputs.make_config(3, 8)                # 32 x 32 x 50 voxels of 16 x 16 x 32 mm, four materials
        n = 4000
    else:                                                 # 0.25 mm voxels: every electron crosses several voxels
        nx, ny, nz = 48, 40, 36
        mat = np.full((nz, ny, nx), 2, np.uint8); rho = np.full((nz, ny, nx), 1.0, np.float32)
        mat[:, :, 16:32], rho[:, :, 16:32] = 1, 0.26      # lung slab
        mat[:, :, 32:], rho[:, :, 32:] = 3, 1.92          # bone slab
        mat[:8], rho[:8] = 0, 0.0012                      # air layer
        cfg = {"shape": (nx, ny, nz), "spacing_mm": (0.25, 0.25, 0.3), "material": mat, "density": anm_inputs.phantoms.quantize_density(rho),
               "activity": None, "point_source_mm": (1.0, 1.0, 1.0), "labels": None, "n_organs": 0, "seed": 1,
               "photons_per_decay": 2, "rayleigh_on": 1, "photon_cutoff_mev": 0.010, "positron_ke_mev": 0.0}
        n = 3000
    el = _random_electrons(cfg, n, 5)
    with anm.Simulation(0) as sim:
        sim.set_grid(cfg["shape"], cfg["spacing_mm"])
        sim.load_phantom(cfg["material"], cfg["density"])
        sim.set_electron_tables(etab)
        vol_g, esc_g = sim.trace_electrons(el)
    vol_o, esc_o = _oracle_trace(cfg, tables, etab, el)
    vol_g = vol_g.reshape(-1).astype(np.float64)
    assert vol_g.sum() + esc_g == pytest.approx(float(el[:, 6].astype(np.float64).sum()), rel=2e-6)      # energy conservation
    assert esc_g == pytest.approx(esc_o, abs=2e-4 + 1e-5 * esc_o)
    # a start point that fp32 rounds across a voxel face moves one electron's first deposit to the neighbour
    bad = np.abs(vol_g - vol_o) > 5e-5
    assert bad.sum() <= 4, (int(bad.sum()), float(np.abs(vol_g - vol_o).max()))
    assert np.abs(vol_g - vol_o).sum() < 1e-3 * vol_o.sum()
    if case == "fine_slabs":
        assert (vol_o > 0).sum() > 3 * n                 # the walks really spread over voxels


def _run_gpu(anm, cfg, tables, etab, n, B, electrons, **opts):
    with anm.Simulation(0) as sim:
        sim.load_config(cfg, tables, n_batches=B, collect_stats=1, electron_transport=0, **opts)
        if electrons:
            sim.set_electron_tables(etab)
            sim.set_options(n_batches=B, collect_stats=1, electron_transport=1, photons_per_decay=cfg["photons_per_decay"],
                            rayleigh_on=cfg["rayleigh_on"], photon_cutoff_MeV=cfg["photon_cutoff_mev"],
                            positron_ke_MeV=cfg["positron_ke_mev"], **opts)
        sim.run(n, cfg["seed"])
        out = {"energy": sim.get_energy().astype(np.float64), "dose": sim.get_dose().astype(np.float64),
               "rel": sim.get_uncertainty().astype(np.float64), "stats": sim.get_stats()}
        if cfg.get("n_organs"):
            out["organs"] = sim.get_organ_doses()
    return out


def test_photon_histories_do_not_change(anm, tables, etab):
    cfg = anm_inputs.make_config(3, 4)
    n, B = 400_000, 10
    off = _run_gpu(anm, cfg, tables, etab, n, B, False)
    on = _run_gpu(anm, cfg, tables, etab, n, B, True)
    for k in ("n_steps", "n_real", "n_pe", "n_compton", "n_rayleigh", "n_escaped", "n_cutoff"):
        assert off["stats"][k] == on["stats"][k], k
    assert off["stats"]["n_electrons"] == 0 and on["stats"]["n_electrons"] > 0
    s0, s1 = off["stats"], on["stats"]
    assert abs(s1["deposited_MeV"] + s1["escaped_MeV"] - s1["emitted_MeV"]) < 2e-5 * s1["emitted_MeV"]
    assert s1["deposited_MeV"] + s1["escaped_MeV"] == pytest.approx(s0["deposited_MeV"] + s0["escaped_MeV"], rel=2e-5)
    moved = np.abs(on["energy"] - off["energy"]).sum() / off["energy"].sum()
    assert 1e-4 < moved < 0.2


def test_run_with_electrons_vs_oracle_patient(anm, tables, etab):
    cfg = anm_inputs.make_config(3, 4)
    n, B = 2_000_000, 100
    g = _run_gpu(anm, cfg, tables, etab, n, B, True)
    o = O.Oracle(cfg, tables, n_decays=n, n_batches=B, seed=cfg["seed"] + 1000, electron_tables=etab)
    r = o.run_parallel(NPROC)
    f = o.finalize(r)
    st = g["stats"]
    assert abs(st["deposited_MeV"] + st["escaped_MeV"] - st["emitted_MeV"]) < 2e-5 * st["emitted_MeV"]
    assert st["deposited_MeV"] / r["stats"]["deposited"] == pytest.approx(1.0, abs=2e-3)
    assert st["n_electrons"] / r["stats"]["n_electrons"] == pytest.approx(1.0, abs=0.01)
    big = f["organs"]["n_voxels"] >= 20
    gm, gs = g["organs"]["mean_Gy_per_decay"][big], g["organs"]["sigma_mean"][big]
    om, osig = f["organs"]["mean"][big], f["organs"]["sigma_mean"][big]
    assert np.all(np.abs(gm - om) <= np.maximum(0.01 * om, 3.0 * np.sqrt(gs ** 2 + osig ** 2)))


def test_fine_voxels_where_electrons_matter(anm, tables, etab):
    """The paper's water test has 0.5 mm voxels: there the electron range (~0.55 mm) spreads the dose.
    Point source in 64^3 voxels of 0.5 mm; radial energy profile in 0.5 mm shells, GPU vs oracle, and both clearly
    different from local deposition."""
    nvox = 64
    base = anm_inputs.make_config(0, 1)
    cfg = dict(base, shape=(nvox,) * 3, spacing_mm=(0.5,) * 3, material=np.full((nvox,) * 3, 2, np.uint8),
               density=anm_inputs.phantoms.quantize_density(np.full((nvox,) * 3, 1.0)), point_source_mm=(16.0, 16.0, 16.0),
               labels=None, n_organs=0, photons_per_decay=1)
    n, B = 4_000_000, 20
    g = _run_gpu(anm, cfg, tables, etab, n, B, True)
    g_local = _run_gpu(anm, cfg, tables, etab, n, B, False)
    o = O.Oracle(cfg, tables, n_decays=n, n_batches=B, seed=2001, electron_tables=etab)
    r = o.run_parallel(NPROC)
    c = (np.arange(nvox) + 0.5) * 0.5 - 16.0
    rr = np.sqrt(c[:, None, None] ** 2 + c[None, :, None] ** 2 + c[None, None, :] ** 2).reshape(-1)
    shell = np.minimum((rr / 0.5).astype(int), 31)
    eg = np.bincount(shell, weights=g["energy"], minlength=32)[:24]
    el = np.bincount(shell, weights=g_local["energy"], minlength=32)[:24]
    eo = np.bincount(shell, weights=r["sum"], minlength=32)[:24]
    # Poisson-like noise of a shell sum: each deposit <= 0.34 MeV, so var <= 0.34 * sum (MeV^2)
    sig = np.sqrt(0.34 * (eg + eo))
    assert np.all(np.abs(eg - eo) < 5.0 * sig + 1e-3 * eo), (np.abs(eg - eo) / sig)
    assert abs(eg[0] - el[0]) > 10.0 * sig[0]            # the innermost shell loses energy to its neighbours
    assert g["stats"]["deposited_MeV"] / r["stats"]["deposited"] == pytest.approx(1.0, abs=3e-3)


def test_electron_error_codes(anm, tables, etab):
    cfg = anm_inputs.make_config(3, 16)
    with anm.Simulation(0) as sim:
        sim.load_config(cfg, tables, n_batches=2)
        sim.set_options(n_batches=2, electron_transport=1)
        with pytest.raises(anm.AnmError) as e:
            sim.run(1000, 1)
        assert e.value.code == -2                        # no electron tables
        with pytest.raises(anm.AnmError) as e:
            sim.set_options(n_batches=2, electron_transport=1, schedule=1)
        assert e.value.code == -5
        with pytest.raises(anm.AnmError) as e:
            sim.set_options(n_batches=2, electron_transport=2)
        assert e.value.code == -1
        bad = dict(etab, range=etab["range"].copy()); bad["range"][1, 5] = bad["range"][1, 4]
        with pytest.raises(anm.AnmError) as e:
            sim.set_electron_tables(bad)
        assert e.value.code == -1
        short = dict(etab, n_t=10, range=etab["range"][:, :10].copy())
        with pytest.raises(anm.AnmError) as e:
            sim.set_electron_tables(short)
        assert e.value.code == -1                        # does not reach E0 (photo-electrons)
        with pytest.raises(anm.AnmError) as e:
            sim.trace_electrons(np.array([[1.0, 1.0, 1.0, 1.0, 0.0, 0.0, 0.3]]))
        assert e.value.code == -2                        # no tables yet
        sim.set_electron_tables(etab)
        with pytest.raises(anm.AnmError) as e:
            sim.trace_electrons(np.array([[-1.0, 1.0, 1.0, 1.0, 0.0, 0.0, 0.3]]))
        assert e.value.code == -1
        with pytest.raises(anm.AnmError) as e:
            sim.trace_electrons(np.array([[1.0, 1.0, 1.0, 1.0, 0.0, 0.0, 0.1]]))
        assert e.value.code == -1
        sim.run(1000, 1)
        assert sim.get_stats()["n_decays"] == 1000
