"""Pins of the oracle's secondary-electron transport (reading C28)
and of the electron tables, against what the physics fixes independently of the oracle's own code:
published collision stopping powers and CSDA ranges of water, direct numerical integration of the Bethe formula,
the textbook Compton electron angle, energy conservation, and the invariance of the photon histories."""
import ctypes as C

import numpy as np
import pytest
from scipy import integrate

import anm_inputs
from anm_inputs import electrons as el
from oracle import anm_oracle as O

WATER, LUNG, BONE = 2, 1, 3


@pytest.fixture(scope="module")
def tables():
    return anm_inputs.make_tables()


@pytest.fixture(scope="module")
def etab():
    return anm_inputs.make_electron_tables()


def _slab_problem(tables, etab, n=(40, 3, 3), d_mm=(0.1, 10.0, 10.0), mats=None, rhos=None, **over):
    nx, ny, nz = n
    mat = np.full((nz, ny, nx), WATER, np.uint8)
    rho = np.full((nz, ny, nx), 1.0, np.float32)
    if mats is not None:
        mat[:, :, :] = np.asarray(mats, np.uint8)[None, None, :]
        rho[:, :, :] = np.asarray(rhos, np.float32)[None, None, :]
    cfg = {"shape": n, "spacing_mm": d_mm, "material": mat, "density": rho, "activity": None,
           "point_source_mm": (0.05, 15.0, 15.0), "labels": None, "n_organs": 0, "n_decays": 100, "n_batches": 2,
           "seed": 1, "photons_per_decay": 1, "rayleigh_on": 1, "photon_cutoff_mev": 0.010, "positron_ke_mev": 0.0}
    return O.Oracle(cfg, tables, electron_tables=etab, **over)


def test_bethe_table_against_published_water_values(etab):
    """NIST ESTAR, liquid water, collision stopping power (MeV cm^2/g) and CSDA range (g/cm^2), values as printed in
    the standard tables: 0.2 MeV 2.793 / 0.04488, 0.3 MeV 2.355 / 0.08421, 0.4 MeV 2.148 / 0.1288."""
    w = anm_inputs.MATERIALS[WATER]
    for T, S in ((0.1, 4.115), (0.2, 2.793), (0.3, 2.355), (0.4, 2.148), (0.5, 2.034)):
        assert el.bethe_collision_stopping(T, w) == pytest.approx(S, rel=3e-3)
    k300 = int(round((0.3 - etab["t_min"]) / etab["dt"]))
    assert etab["t_min"] + k300 * etab["dt"] == pytest.approx(0.3, abs=1e-12)
    assert float(etab["range"][WATER, k300]) == pytest.approx(0.08421 - 0.04488, rel=1e-2)
    assert etab["t_min"] == 0.2 and etab["t_min"] + etab["dt"] * (etab["n_t"] - 1) >= 0.51099895     # photo-electrons: all of E0
    assert np.all(np.diff(etab["range"], axis=1) > 0) and np.all(etab["range"][:, 0] == 0)
    # the table is the integral of 1/S: check one entry per material by adaptive quadrature
    for m, mat in enumerate(anm_inputs.MATERIALS):
        q, _ = integrate.quad(lambda t: 1.0 / el.bethe_collision_stopping(t, mat), 0.2, 0.34)
        k = int(round((0.34 - 0.2) / etab["dt"]))
        assert float(etab["range"][m, k]) == pytest.approx(q, rel=2e-6)


def test_range_and_its_inverse(tables, etab):
    o = _slab_problem(tables, etab)
    R = etab["range"].astype(np.float64)
    for m in (0, 1, 2, 3):
        for k in (0, 1, 17, etab["n_t"] - 1):
            T = etab["t_min"] + k * etab["dt"]
            assert o.electron_range(m, T) == pytest.approx(R[m, k], abs=1e-15)
            assert o.electron_energy(m, R[m, k]) == pytest.approx(T, abs=1e-12)
        T = etab["t_min"] + 10.25 * etab["dt"]
        r = o.electron_range(m, T)
        assert r == pytest.approx(0.75 * R[m, 10] + 0.25 * R[m, 11], rel=1e-14)
        assert o.electron_energy(m, r) == pytest.approx(T, abs=1e-12)
        assert o.electron_range(m, 0.1) == 0.0 and o.electron_energy(m, -1.0) == etab["t_min"]


def _csda_energy_after(mat, T0, mass_path):
    """Independent of the tables: integrate dT/ds = -S(T) over a mass path (g/cm^2) with an ODE solver."""
    sol = integrate.solve_ivp(lambda s, T: -el.bethe_collision_stopping(T, mat), (0.0, mass_path), [T0], rtol=1e-10, atol=1e-12)
    return float(sol.y[0, -1])


def test_walk_in_water_matches_direct_integration(tables, etab):
    """0.1 mm voxels of water, electron of 0.34 MeV along +x from x = 0.05 mm: the deposit in each voxel equals
    T(entry) - T(exit) from integrating the Bethe formula directly; the walk ends where the energy reaches 0.2 MeV and
    everything left is deposited there."""
    o = _slab_problem(tables, etab)
    T0 = 0.34
    dep, esc = o.electron_walk((0.005, 1.5, 1.5), (1.0, 0.0, 0.0), T0)
    assert esc == 0.0
    assert sum(e for _, e in dep) == pytest.approx(T0, abs=1e-12)
    w = anm_inputs.MATERIALS[WATER]
    T = T0
    edges = [0.005] + [0.01 * (i + 1) for i in range(40)]
    for i, (v, e) in enumerate(dep):
        assert v == 40 * (1 + 3 * 1) + i                       # iy = iz = 1, ix = i
        T_next = _csda_energy_after(w, T, 1.0 * (edges[i + 1] - edges[i]))
        if i < len(dep) - 1:
            assert e == pytest.approx(T - T_next, abs=3e-6)     # table interpolation error only
            T = T_next
        else:
            assert T_next < 0.2 + 3e-6 and e == pytest.approx(T, abs=1e-5)
    # CSDA path length from 0.34 to 0.2 MeV in water: ~0.55 mm
    q, _ = integrate.quad(lambda t: 1.0 / el.bethe_collision_stopping(t, w), 0.2, T0)
    assert len(dep) == int(np.floor((0.005 + q) / 0.01)) + 1
    assert 0.05 < q < 0.06


def test_photo_electron_walk_matches_direct_integration(tables, etab):
    """A photo-electron takes the whole photon energy (reading C28): up to E0 = 0.511 MeV, beyond the Compton edge.
    0.1 mm voxels of water, electron of 0.51099895 MeV along +x: every voxel's deposit equals T(entry) - T(exit) from
    integrating the Bethe formula directly (no table), the walk ends where the energy reaches the 0.2 MeV cutoff; the
    CSDA path 0.511 -> 0.2 MeV is the difference of the published water ranges (ESTAR: 0.5 MeV 0.1766, 0.2 MeV 0.04488
    g/cm^2, so a little over 1.3 mm).  The range table must therefore cover E0 (orc_run refuses one that does not)."""
    o = _slab_problem(tables, etab)
    T0 = 0.51099895
    dep, esc = o.electron_walk((0.005, 1.5, 1.5), (1.0, 0.0, 0.0), T0)
    assert esc == 0.0 and sum(e for _, e in dep) == pytest.approx(T0, abs=1e-12)
    w = anm_inputs.MATERIALS[WATER]
    T = T0
    edges = [0.005] + [0.01 * (i + 1) for i in range(40)]
    for i, (v, e) in enumerate(dep):
        assert v == 40 * (1 + 3 * 1) + i
        T_next = _csda_energy_after(w, T, edges[i + 1] - edges[i])
        if i < len(dep) - 1:
            assert e == pytest.approx(T - T_next, abs=3e-6), i
            T = T_next
        else:
            assert T_next < 0.2 + 3e-6 and e == pytest.approx(T, abs=1e-5)
    q, _ = integrate.quad(lambda t: 1.0 / el.bethe_collision_stopping(t, w), 0.2, T0)
    assert len(dep) == int(np.floor((0.005 + q) / 0.01)) + 1
    assert q == pytest.approx(0.1766 + (0.51099895 - 0.5) / 2.034 - 0.04488, rel=1.5e-2)       # published ranges
    # a table that stops at the Compton edge is refused: the walk would extrapolate its last segment
    short = dict(etab, n_t=77, range=etab["range"][:, :77].copy())
    assert short["t_min"] + short["dt"] * 76 > 2 * 0.51099895 / 3
    bad = _slab_problem(tables, short)
    with pytest.raises(Exception):
        bad.run()


def test_walk_across_materials_and_out_of_the_grid(tables, etab):
    """water | lung 0.26 | bone 1.92 in 0.2 mm slabs; oblique direction; then an electron that leaves the grid."""
    mats = [WATER] * 1 + [LUNG] * 2 + [BONE] * 37
    rhos = [1.0] * 1 + [0.26] * 2 + [1.92] * 37
    o = _slab_problem(tables, etab, d_mm=(0.2, 10.0, 10.0), mats=mats, rhos=rhos)
    d = np.array([0.8, 0.6, 0.0])
    T0 = 0.335
    dep, esc = o.electron_walk((0.01, 1.2, 1.5), d, T0)
    assert esc == 0.0 and sum(e for _, e in dep) == pytest.approx(T0, abs=1e-12)
    T = T0
    x = 0.01
    for i, (v, e) in enumerate(dep[:-1]):
        chord = (0.02 * (i + 1) - x) / d[0]
        x = 0.02 * (i + 1)
        T_next = _csda_energy_after(anm_inputs.MATERIALS[mats[i]], T, rhos[i] * chord)
        assert e == pytest.approx(T - T_next, abs=5e-6), i
        T = T_next
    assert len(dep) == 4 and mats[len(dep) - 1] == BONE         # through the water and the lung, stops in the bone
    # leaving the grid: start 0.05 mm from the low-x face, heading out
    dep2, esc2 = o.electron_walk((0.005, 1.5, 1.5), (-1.0, 0.0, 0.0), 0.3)
    assert len(dep2) == 1 and esc2 > 0.28 and dep2[0][1] + esc2 == pytest.approx(0.3, abs=1e-12)
    assert esc2 == pytest.approx(_csda_energy_after(anm_inputs.MATERIALS[WATER], 0.3, 0.005), abs=3e-6)


def test_compton_electron_direction_is_the_textbook_angle():
    """cot(phi_e) = (1 + alpha) tan(theta / 2); electron, incident and scattered photon are coplanar."""
    L = O.lib()
    rng = np.random.default_rng(2)
    for _ in range(50):
        E = rng.uniform(0.05, 0.511)
        a = E / 0.51099895
        eps = rng.uniform(1.0 / (1.0 + 2.0 * a), 1.0)
        cos_t = 1.0 + 1.0 / a - 1.0 / (a * eps)
        d = rng.normal(size=3); d /= np.linalg.norm(d)
        nd = np.zeros(3); out = np.zeros(3)
        L.orc_rotate(d.ctypes.data, C.c_double(cos_t), C.c_double(rng.uniform(0, 2 * np.pi)), nd.ctypes.data)
        L.orc_compton_electron_direction(C.c_double(E), C.c_double(eps), d.ctypes.data, nd.ctypes.data, out.ctypes.data)
        assert np.linalg.norm(out) == pytest.approx(1.0, abs=1e-12)
        theta = np.arccos(np.clip(cos_t, -1, 1))
        phi = np.arccos(np.clip(out @ d, -1, 1))
        assert 1.0 / np.tan(phi) == pytest.approx((1.0 + a) * np.tan(theta / 2.0), rel=1e-6)
        assert abs(np.dot(np.cross(d, nd), out)) < 1e-9
        # transverse momentum balance: the electron goes to the other side of the beam
        assert (out - (out @ d) * d) @ (nd - (nd @ d) * d) <= 1e-12


def test_histories_conserve_energy_and_photons_do_not_change(tables, etab):
    """Electron transport draws no random numbers: photon histories are identical with it on or off, so every counter
    agrees, emitted = deposited + escaped per history to 1e-9, and only WHERE the energy lands changes."""
    cfg = anm_inputs.make_config(3, 8)
    kw = dict(n_decays=20_000, n_batches=4, seed=7)
    off = O.Oracle(cfg, tables, **kw); r0 = off.run()
    on = O.Oracle(cfg, tables, electron_tables=etab, **kw); r1 = on.run()
    s0, s1 = r0["stats"], r1["stats"]
    for k in ("n_photons", "n_collisions", "n_pe", "n_compton", "n_rayleigh", "n_escaped", "n_cutoff", "n_crossings"):
        assert s0[k] == s1[k], k
    assert s0["n_electrons"] == 0 and s1["n_electrons"] > 0.1 * s1["n_compton"] * 0.5
    assert s1["max_history_residual"] < 1e-9 * 1.3 and s0["max_history_residual"] < 1e-9 * 1.3
    assert s1["emitted"] == s0["emitted"]
    assert s1["deposited"] + s1["escaped"] == pytest.approx(s0["deposited"] + s0["escaped"], rel=1e-12)
    moved = np.abs(r1["sum"] - r0["sum"]).sum() / r0["sum"].sum()
    assert 1e-4 < moved < 0.2                      # 16 x 16 x 32 mm voxels: few electrons cross a face
    # fine voxels (the paper's 0.5 mm water test): many electrons cross
    fine = anm_inputs.make_config(0, 1)
    fine = dict(fine, spacing_mm=(0.5, 0.5, 0.5), point_source_mm=(8.0, 8.0, 8.0))
    a = O.Oracle(fine, tables, n_decays=20_000, n_batches=4, seed=3).run()
    b = O.Oracle(fine, tables, electron_tables=etab, n_decays=20_000, n_batches=4, seed=3).run()
    assert b["stats"]["n_electron_crossings"] > 0.5 * b["stats"]["n_electrons"]
    assert b["stats"]["deposited"] + b["stats"]["escaped"] == pytest.approx(a["stats"]["deposited"] + a["stats"]["escaped"], rel=1e-12)


def test_huge_voxels_reduce_to_local_deposition(tables, etab):
    """P6-style limit: in 250 cm voxels no electron reaches a face, so the tallies equal local deposition exactly."""
    n = 4
    cfg = {"shape": (n, n, n), "spacing_mm": (2500.0,) * 3, "material": np.full((n, n, n), WATER, np.uint8),
           "density": np.full((n, n, n), 1.0, np.float32), "activity": None, "point_source_mm": (6250.0, 6250.0, 6250.0),
           "labels": None, "n_organs": 0, "n_decays": 4000, "n_batches": 2, "seed": 5, "photons_per_decay": 2,
           "rayleigh_on": 1, "photon_cutoff_mev": 0.010, "positron_ke_mev": 0.0}
    a = O.Oracle(cfg, tables).run()
    b = O.Oracle(cfg, tables, electron_tables=etab).run()
    assert b["stats"]["n_electron_crossings"] == 0 and b["stats"]["n_electrons"] > 0
    assert np.allclose(a["sum"], b["sum"], rtol=1e-13, atol=0)
