"""Pins for the CPU oracle (oracle/): each checks it against something the paper or the mathematics
fixes -- never against the CUDA path and never against the oracle's own formula retyped.
Pin numbers follow SURVEY.md §8(c) / DESIGN.md.
"""
import ctypes as C
import os

import numpy as np
import pytest
from scipy import integrate, stats

import anm_inputs
from anm_inputs import tables as T
from oracle import anm_oracle as O

E0 = 0.51099895
HERE = os.path.dirname(os.path.abspath(__file__))


def _ptr(a):
    return a.ctypes.data


def _homog(n=8, d_mm=10.0, mat=2, rho=1.0, **kw):
    c = {"name": "t", "shape": (n, n, n), "spacing_mm": (d_mm,) * 3,
         "material": np.full((n, n, n), mat, np.uint8), "density": np.full((n, n, n), rho, np.float32),
         "activity": None, "point_source_mm": (n * d_mm / 2,) * 3, "labels": None, "n_organs": 0,
         "n_decays": 1000, "seed": 1, "n_batches": 1, "photons_per_decay": 1, "rayleigh_on": 1,
         "photon_cutoff_mev": 0.010, "positron_ke_mev": 0.0}
    c.update(kw)
    return c


def _mu_water(tables, E, rayleigh=True):
    m = 2
    return sum(T.interp_lnE(tables[k][m], E, tables["lnE_min"], tables["dlnE"])
               for k in (("mu_pe", "mu_compton", "mu_rayleigh") if rayleigh else ("mu_pe", "mu_compton")))


# ------------------------------------------------------------------------------------------ P1
def test_p1_philox_known_answers():
    """Philox4x32-10 known answers, read from tests/golden/philox4x32_10_kat.txt (Random123 KAT vectors,
    restated in SURVEY.md §8(c) P1)."""
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "philox4x32_10_kat.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        assert [int(x) for x in O.philox4x32_10(v[0:4], v[4:6])] == v[6:10]


def test_table_reader_matches_definition(tables):
    row = tables["mu_compton"][2]
    for E in (0.010, 0.0123, 0.2, 0.511, 0.512):
        got = O.lib().orc_interp(_ptr(row), len(row), tables["lnE_min"], tables["dlnE"], E)
        # independent: numpy's piecewise-linear interpolation on the ln E grid
        lnE = tables["lnE_min"] + tables["dlnE"] * np.arange(len(row))
        assert abs(got - np.interp(np.log(E), lnE, row.astype(np.float64))) < 1e-12


# ------------------------------------------------------------------------------------------ P3
def _kn_pdf(eps, a):
    c = 1 + 1 / a - 1 / (a * eps)
    return eps + 1 / eps - (1 - c * c)


@pytest.mark.parametrize("E,mean_T_frac", [(0.010, 0.018764), (0.050, 0.080708), (0.100, 0.138003),
                                           (0.200, 0.216352), (0.300, 0.269654), (0.400, 0.309627),
                                           (E0, 0.344482)])
def test_p3_kn_sampler(E, mean_T_frac):
    """Klein-Nishina sampler: KS against the CDF obtained by numerical quadrature of the Klein-Nishina
    density, and the mean energy-transfer fraction against the values printed in SURVEY.md §8(c) P3."""
    a = E / E0
    emin = 1 / (1 + 2 * a)
    n = 200_000
    eps = np.zeros(n)
    O.lib().orc_kn_sample_many(E, 77, n, _ptr(eps))
    assert eps.min() >= emin - 1e-15 and eps.max() <= 1.0
    norm = integrate.quad(_kn_pdf, emin, 1, args=(a,), epsrel=1e-12)[0]
    # mean fraction: quadrature reproduces the printed value, sampler agrees within 5 sigma
    mt = integrate.quad(lambda e: (1 - e) * _kn_pdf(e, a), emin, 1, epsrel=1e-12)[0] / norm
    assert abs(mt - mean_T_frac) < 2e-6
    assert abs((1 - eps).mean() - mean_T_frac) < 5 * (1 - eps).std() / np.sqrt(n)
    grid = np.linspace(emin, 1, 4001)
    cdf = integrate.cumulative_trapezoid(_kn_pdf(grid, a), grid, initial=0)
    cdf /= cdf[-1]
    d = stats.kstest(eps, lambda x: np.interp(x, grid, cdf)).statistic
    assert d < 1.95 / np.sqrt(n)
    if E == E0:     # eps_min = 1/3, T_max = 0.340667 MeV
        assert abs(emin - 1 / 3) < 1e-15 and abs(E * (1 - emin) - 0.340667) < 1.5e-6


def test_p3_kn_closed_form_cdf():
    """The closed-form antiderivative quoted in SURVEY.md P3 agrees with quadrature (pins the pdf used above)."""
    a = 1.0
    k = 1 + 1 / a
    G = lambda e: e * e / 2 + np.log(e) - e + k * k * e - (2 * k / a) * np.log(e) - 1 / (a * a * e)   # noqa: E731
    for e in (0.4, 0.7, 0.95):
        num = integrate.quad(_kn_pdf, 1 / 3, e, args=(a,), epsrel=1e-12)[0]
        assert abs(num - (G(e) - G(1 / 3))) < 1e-10


# ------------------------------------------------------------------------------------------ rotation
def test_rotate_geometry():
    rng = np.random.default_rng(5)
    for _ in range(200):
        d = rng.normal(size=3)
        d /= np.linalg.norm(d)
        if rng.random() < 0.2:
            d = np.array([0.0, 0.0, rng.choice([-1.0, 1.0])])
        ct, phi = rng.uniform(-1, 1), rng.uniform(0, 2 * np.pi)
        out = np.zeros(3)
        O.lib().orc_rotate(_ptr(d), ct, phi, _ptr(out))
        assert abs(np.linalg.norm(out) - 1) < 1e-12 and abs(out @ d - ct) < 1e-9
    # azimuth: at fixed polar angle the rotated vectors average to cos(theta) d and fill the cone evenly
    d = np.array([0.3, -0.5, np.sqrt(1 - 0.09 - 0.25)])
    phis = (np.arange(3600) + 0.5) * 2 * np.pi / 3600
    outs = np.zeros((3600, 3))
    for i, ph in enumerate(phis):
        O.lib().orc_rotate(_ptr(d), 0.25, float(ph), _ptr(outs[i]))
    assert np.allclose(outs.mean(axis=0), 0.25 * d, atol=1e-9)
    # equal azimuth steps -> equal chord between neighbours
    ch = np.linalg.norm(np.diff(outs, axis=0), axis=1)
    assert ch.std() / ch.mean() < 1e-6


# ------------------------------------------------------------------------------------------ P8
def test_p8_isotropy():
    n = 300_000
    d = np.zeros((n, 3))
    O.lib().orc_isotropic_many(11, n, _ptr(d))
    assert np.allclose(np.linalg.norm(d, axis=1), 1, atol=1e-12)
    assert np.all(np.abs(d.mean(axis=0)) < 4 / np.sqrt(3 * n))
    assert np.all(np.abs((d ** 2).mean(axis=0) - 1 / 3) < 4 * np.sqrt(4 / 45 / n))
    for a in range(3):     # Archimedes: each component of an isotropic unit vector is U(-1,1)
        assert stats.kstest(d[:, a], stats.uniform(-1, 2).cdf).statistic < 1.95 / np.sqrt(n)
    phi = np.arctan2(d[:, 1], d[:, 0])
    assert stats.kstest(phi, stats.uniform(-np.pi, 2 * np.pi).cdf).statistic < 1.95 / np.sqrt(n)
    # cross moments vanish
    assert abs((d[:, 0] * d[:, 1]).mean()) < 4 * np.sqrt(1 / 15 / n)


def test_p8_voxel_pick_and_position(tables):
    rng = np.random.default_rng(3)
    nx, ny, nz = 5, 4, 3
    act = rng.uniform(0.1, 3.0, size=(nz, ny, nx)).astype(np.float32)
    act[rng.random(act.shape) < 0.3] = 0.0
    act[0, 0, 0] = 0.0
    act[-1, -1, -1] = 2.0
    c = _homog()
    c.update(shape=(nx, ny, nz), spacing_mm=(2.0, 3.0, 5.0), material=np.full((nz, ny, nx), 2, np.uint8),
             density=np.ones((nz, ny, nx), np.float32), activity=act, point_source_mm=None)
    o = O.Oracle(c, tables)
    n = 400_000
    pos, dirs, vox = np.zeros((n, 3)), np.zeros((n, 3)), np.zeros(n, np.int64)
    O.lib().orc_sample_source_many(C.byref(o.p), 0, n, _ptr(pos), _ptr(dirs), _ptr(vox))
    cnt = np.bincount(vox, minlength=act.size)
    p = act.reshape(-1).astype(np.float64) / act.sum(dtype=np.float64)
    assert np.all(cnt[p == 0] == 0)
    chi2 = ((cnt[p > 0] - n * p[p > 0]) ** 2 / (n * p[p > 0])).sum()
    assert stats.chi2.sf(chi2, (p > 0).sum() - 1) > 1e-4
    # position: inside the picked voxel, uniform
    h = np.array([0.2, 0.3, 0.5])
    idx = np.stack([vox % nx, (vox // nx) % ny, vox // (nx * ny)], axis=1)
    frac = pos / h - idx
    assert frac.min() > 0 and frac.max() < 1
    for a in range(3):
        assert stats.kstest(frac[:, a], "uniform").statistic < 1.95 / np.sqrt(n)
    assert np.allclose(np.linalg.norm(dirs, axis=1), 1, atol=1e-12)


def test_pick_voxel_edges():
    cdf = np.cumsum(np.array([0, 0, 1.0, 0, 3.0, 0], np.float64))
    L = O.lib()
    assert L.orc_pick_voxel(_ptr(cdf), 6, 0.0) == 2
    assert L.orc_pick_voxel(_ptr(cdf), 6, 0.2499999) == 2
    assert L.orc_pick_voxel(_ptr(cdf), 6, 0.25) == 4
    assert L.orc_pick_voxel(_ptr(cdf), 6, 1 - 2 ** -53) == 4


# ------------------------------------------------------------------------------------------ P4
def _mu_field(o, tables, E):
    mu_m = np.array([sum(T.interp_lnE(tables[k][m], E, tables["lnE_min"], tables["dlnE"])
                         for k in ("mu_pe", "mu_compton", "mu_rayleigh")) for m in range(4)])
    return o.density.astype(np.float64) * mu_m[o.material]


def test_p4_flight_line_integral(tables):
    """orc_flight with a GIVEN optical depth: the brute-force line integral of mu along the ray up to
    the returned point equals that optical depth; rays that leave the grid have a smaller total."""
    rng = np.random.default_rng(9)
    nx, ny, nz = 7, 6, 5
    h = np.array([0.3, 0.5, 0.4])
    c = _homog()
    c.update(shape=(nx, ny, nz), spacing_mm=tuple(10 * h), material=rng.integers(0, 4, (nz, ny, nx)).astype(np.uint8),
             density=anm_inputs.phantoms.quantize_density(rng.uniform(0.2, 2.0, (nz, ny, nx))))
    o = O.Oracle(c, tables)
    E = 0.2
    mu = _mu_field(o, tables, E)
    L = O.lib()
    n_hit = n_esc = 0
    for _ in range(300):
        p0 = rng.uniform(0.02, 0.98, 3) * h * [nx, ny, nz]
        d = rng.normal(size=3)
        d /= np.linalg.norm(d)
        if rng.random() < 0.15:
            d = np.eye(3)[rng.integers(3)] * rng.choice([-1, 1])
        tau = rng.exponential(1.0) * 0.6
        out, vox, dist = np.zeros(3), np.zeros(1, np.int64), np.zeros(1)
        hit = L.orc_flight(C.byref(o.p), _ptr(p0), _ptr(d), E, tau, _ptr(out), _ptr(vox), _ptr(dist))
        s = (np.arange(200_000) + 0.5) / 200_000 * dist[0]
        pts = p0[None, :] + s[:, None] * d[None, :]
        ijk = np.floor(pts / h).astype(int)
        ok = np.all((ijk >= 0) & (ijk < [nx, ny, nz]), axis=1)
        ijk = np.clip(ijk, 0, [nx - 1, ny - 1, nz - 1])
        integral = (mu[ijk[:, 0] + nx * (ijk[:, 1] + ny * ijk[:, 2])] * ok).sum() * dist[0] / 200_000
        assert np.allclose(out, p0 + dist[0] * d, atol=1e-12)
        if hit:
            n_hit += 1
            assert abs(integral - tau) < 2e-4 * max(tau, 0.05)
            ihit = np.floor(out / h).astype(int)
            # the reported voxel contains the point (up to a face)
            v = int(vox[0])
            vi = np.array([v % nx, (v // nx) % ny, v // (nx * ny)])
            assert np.all(np.abs((vi + 0.5) * h - out) <= 0.5 * h + 1e-9), (ihit, vi)
        else:
            n_esc += 1
            assert integral < tau + 2e-4
            eps = 1e-9
            assert np.any((out <= eps) | (out >= h * [nx, ny, nz] - eps))
    assert n_hit > 50 and n_esc > 50


def test_p4_slab_transmission(tables):
    """Narrow beam through the cfg2 slab stack (water/lung/bone/water): uncollided fraction = exp(-sum mu_i L_i)."""
    c = anm_inputs.make_config(2, 8)          # 16^3 voxels of 24 mm, slabs 4 voxels thick
    o = O.Oracle(c, tables)
    mu = _mu_field(o, tables, E0)
    nx = 16
    col = mu[8 + nx * (8 + nx * np.arange(16))]
    h = 2.4
    L = O.lib()
    p0 = np.array([8.5 * h, 8.5 * h, 1e-9])
    d = np.array([0.0, 0.0, 1.0])
    total = col.sum() * h
    out, vox, dist = np.zeros(3), np.zeros(1, np.int64), np.zeros(1)
    assert L.orc_flight(C.byref(o.p), _ptr(p0), _ptr(d), E0, total * 1.000001, _ptr(out), _ptr(vox), _ptr(dist)) == 0
    assert L.orc_flight(C.byref(o.p), _ptr(p0), _ptr(d), E0, total * 0.999999, _ptr(out), _ptr(vox), _ptr(dist)) == 1
    assert int(vox[0]) // (nx * nx) == 15
    # half-way through the bone slab
    tau = col[:8].sum() * h + 2.5 * h * col[8]
    assert L.orc_flight(C.byref(o.p), _ptr(p0), _ptr(d), E0, tau, _ptr(out), _ptr(vox), _ptr(dist)) == 1
    assert abs(out[2] - (8 + 2.5) * h) < 1e-7 and int(vox[0]) // (nx * nx) == 10


def test_p4_p6_p7_water_point_source(tables):
    """Point source in a large water block:
       P4  first-collision distance ~ Exp(mu) (KS) and survival exp(-mu x);
       P6  infinite medium: nothing escapes, deposited = emitted;
       P7  mean first-collision deposit = E0 (mu_C <T>/E0 + mu_PE)/mu_tot with <T>/E0 = 0.344482 (P3)."""
    n = 200_000
    c = _homog(n=4, d_mm=2500.0, n_decays=n)
    o = O.Oracle(c, tables)
    r = o.run(first_collision=True)
    st = r["stats"]
    mu = _mu_water(tables, E0)
    assert st["n_escaped"] == 0 and st["escaped"] == 0.0
    assert abs(st["deposited"] / (n * E0) - 1) < 1e-10 and abs(r["sum"].sum() / (n * E0) - 1) < 1e-10
    dist = r["fc_dist"]
    assert dist.min() > 0
    assert stats.kstest(dist, stats.expon(scale=1 / mu).cdf).statistic < 1.95 / np.sqrt(n)
    for x in (5.0, 10.44, 25.0):
        t = np.exp(-mu * x)
        assert abs((dist > x).mean() - t) < 4 * np.sqrt(t * (1 - t) / n)
    m = 2
    parts = [T.interp_lnE(tables[k][m], E0, tables["lnE_min"], tables["dlnE"]) for k in ("mu_pe", "mu_compton", "mu_rayleigh")]
    f = (parts[1] * 0.344482 + parts[0]) / sum(parts)
    dep = r["fc_dep"]
    assert abs(dep.mean() - f * E0) < 4 * dep.std() / np.sqrt(n)
    # interaction-type fractions at the FIRST collision are mu_i/mu_tot; over all collisions only bounds hold
    assert abs((dep == E0).mean() - parts[0] / sum(parts)) < 4 * np.sqrt(parts[0] / sum(parts) / n) + 1e-6
    # P7 shells: first-collision energy in [r1, r2) = N f E0 (exp(-mu r1) - exp(-mu r2))
    for r1, r2 in ((0, 2), (2, 6), (6, 15), (15, 40)):
        sel = (dist >= r1) & (dist < r2)
        want = n * f * E0 * (np.exp(-mu * r1) - np.exp(-mu * r2))
        sig = np.sqrt(n * (dep ** 2).mean() * (np.exp(-mu * r1) - np.exp(-mu * r2)))
        assert abs(dep[sel].sum() - want) < 4 * sig


def test_p4_transmission_without_rayleigh(tables):
    n = 100_000
    c = _homog(n=4, d_mm=2500.0, n_decays=n, rayleigh_on=0)
    r = O.Oracle(c, tables).run(first_collision=True)
    mu = _mu_water(tables, E0, rayleigh=False)
    t = np.exp(-mu * 10.0)
    assert abs((r["fc_dist"] > 10.0).mean() - t) < 4 * np.sqrt(t * (1 - t) / n)
    assert r["stats"]["n_rayleigh"] == 0


# ------------------------------------------------------------------------------------------ P5
@pytest.mark.parametrize("k,scale", [(0, 2), (2, 4), (3, 8)])
def test_p5_energy_conservation(tables, k, scale):
    c = anm_inputs.make_config(k, scale)
    n = 20_000
    o = O.Oracle(c, tables, n_decays=n, n_batches=10)
    r = o.run()
    st = r["stats"]
    per = E0 * c["photons_per_decay"] + c["positron_ke_mev"]
    assert abs(st["emitted"] - n * per) < 1e-9 * n * per
    assert st["max_history_residual"] <= 1e-9 * per
    assert abs(st["deposited"] + st["escaped"] - st["emitted"]) <= 1e-9 * st["emitted"]
    assert abs(r["sum"].sum() - st["deposited"]) <= 1e-9 * st["deposited"]
    assert st["n_photons"] == n * c["photons_per_decay"]
    assert st["n_collisions"] == st["n_pe"] + st["n_compton"] + st["n_rayleigh"]
    assert st["n_photons"] == st["n_escaped"] + st["n_pe"] + st["n_cutoff"]


def test_cutoff_deposits_locally(tables):
    """below the cutoff the remaining energy is deposited locally.  With a 0.3 MeV cutoff
    most first Compton scatters end the photon; energy is still conserved and cutoffs are counted."""
    c = _homog(n=4, d_mm=2500.0, n_decays=20_000, photon_cutoff_mev=0.3)
    r = O.Oracle(c, tables).run()
    st = r["stats"]
    assert st["n_cutoff"] > 5000 and st["n_escaped"] == 0
    assert abs(st["deposited"] / st["emitted"] - 1) < 1e-10


# ------------------------------------------------------------------------------------------ P6b
def test_p6_woodcock_cross_check(tables):
    """Exact stepping and Woodcock tracking (cross-check mode) give the same per-voxel energies on a
    4^3 random-material grid, within statistics."""
    rng = np.random.default_rng(21)
    n = 4
    c = _homog(n=n, d_mm=40.0)
    c.update(material=rng.integers(0, 4, (n, n, n)).astype(np.uint8),
             density=anm_inputs.phantoms.quantize_density(rng.uniform(0.3, 1.9, (n, n, n))),
             activity=rng.uniform(0, 1, (n, n, n)).astype(np.float32), point_source_mm=None,
             photons_per_decay=2, n_decays=200_000, n_batches=20)
    ra = O.Oracle(c, tables, seed=5)
    rb = O.Oracle(c, tables, seed=6, tracking=1)
    fa, fb = ra.finalize(ra.run_parallel(4)), rb.finalize(rb.run_parallel(4))
    z = (fa["dose"] - fb["dose"]) / np.sqrt(fa["dose_sigma"] ** 2 + fb["dose_sigma"] ** 2)
    assert np.abs(z).max() < 4.5 and abs(z.mean()) < 4 / np.sqrt(z.size) * 1.5
    assert abs(fa["energy"].sum() / fb["energy"].sum() - 1) < 3e-3


# ------------------------------------------------------------------------------------------ P9
def test_p9_rayleigh_thomson_limit(tables):
    """With a constant form factor the Rayleigh sampler must reduce to Thomson scattering:
    CDF(c) = 1/2 + (3/8)(c + c^3/3)."""
    t = dict(tables)
    t["ray_cum"] = np.tile(tables["ray_x2"] / tables["ray_x2"][-1], (4, 1)).astype(np.float32)
    keep = []
    ts = O.tables_struct(t, keep)
    n = 200_000
    cs = np.zeros(n)
    O.lib().orc_rayleigh_sample_many(C.byref(ts), 2, 0.1, 4, n, _ptr(cs))
    cdf = lambda c: 0.5 + 0.375 * (c + c ** 3 / 3)   # noqa: E731
    assert stats.kstest(cs, cdf).statistic < 1.95 / np.sqrt(n)


@pytest.mark.parametrize("E,m", [(0.03, 2), (0.2, 3)])
def test_p9_rayleigh_form_factor_distribution(tables, E, m):
    """Sampled cos(theta) against the density (1+c^2) F_m^2(x^2(c)) integrated numerically, F from the
    analytic form factor of anm_inputs/tables.py."""
    from anm_inputs.materials import MATERIALS, ELEMENTS
    n = 200_000
    keep = []
    ts = O.tables_struct(tables, keep)
    cs = np.zeros(n)
    O.lib().orc_rayleigh_sample_many(C.byref(ts), m, E, 8, n, _ptr(cs))
    Tm = float(T.x2_max(E))

    def pdf(c):
        x2 = Tm * (1 - c) / 2
        f2 = sum(w / ELEMENTS[el][1] * ELEMENTS[el][0] ** 2 * (1 + x2 / (0.3 * ELEMENTS[el][0] ** (1 / 3)) ** 2) ** -4
                 for el, w in MATERIALS[m]["w"].items())
        return (1 + c * c) * f2

    # forward-peaked: integrate on a grid uniform in log(1-c)
    g = 1 - np.geomspace(1e-9, 2, 6000)[::-1]
    g[0] = -1
    cdf = integrate.cumulative_trapezoid(pdf(g), g, initial=0)
    cdf /= cdf[-1]
    d = stats.kstest(cs, lambda x: np.interp(x, g, cdf)).statistic
    assert d < 1.95 / np.sqrt(n) + 2e-3     # + table interpolation error


# ------------------------------------------------------------------------------------------ P10
def test_p10_batch_sigma_calibration(tables):
    """The reported batch standard error matches the spread over independent runs; sigma ~ 1/sqrt(N)."""
    c = anm_inputs.make_config(0, 4)        # 8^3 voxels of 16 mm
    K, n = 32, 20_000
    doses, sig = [], []
    for s in range(K):
        o = O.Oracle(c, tables, n_decays=n, n_batches=10, seed=100 + s)
        f = o.finalize(o.run())
        doses.append(f["dose"]); sig.append(f["dose_sigma"])
    doses, sig = np.array(doses), np.array(sig)
    core = doses.mean(axis=0) > 0.05 * doses.mean(axis=0).max()
    ratio = doses.std(axis=0, ddof=1)[core] / np.sqrt((sig ** 2).mean(axis=0))[core]
    assert abs(ratio.mean() - 1) < 0.15 and core.sum() > 50
    o = O.Oracle(c, tables, n_decays=4 * n, n_batches=10, seed=7)
    f4 = o.finalize(o.run())
    r = (np.sqrt((sig ** 2).mean(axis=0))[core] / doses.mean(axis=0)[core]).mean() / f4["rel_sigma"][core].mean()
    assert abs(r - 2) < 0.3


# ------------------------------------------------------------------------------------------ P11
def test_p11_symmetry(tables):
    """cfg0 geometry (point source at the exact centre of a homogeneous cube): the energy map is
    invariant under mirrors and axis permutations within statistics -- pins the index arithmetic."""
    c = anm_inputs.make_config(0, 4)
    n = 200_000
    o = O.Oracle(c, tables, n_decays=n, n_batches=10)
    r = o.run_parallel(4)
    e = r["sum"].reshape(8, 8, 8)
    tot = e.sum()
    # per-deposit relative noise: compare octant sums (each ~ tot/8)
    oct_sums = [e[z:z + 4, y:y + 4, x:x + 4].sum() for z in (0, 4) for y in (0, 4) for x in (0, 4)]
    rel = np.std(oct_sums) / np.mean(oct_sums)
    assert rel < 4 * np.sqrt(8 / (n * 0.6)) * 0.6      # ~0.6 deposits of ~0.15 MeV per history, loose 4 sigma
    sig = (o.finalize(r)["rel_sigma"] * r["sum"]).reshape(8, 8, 8)      # batch sigma of the voxel energies
    for tr in (lambda a: a.transpose(1, 0, 2), lambda a: a.transpose(2, 1, 0), lambda a: a.transpose(0, 2, 1),
               lambda a: a[::-1], lambda a: a[:, ::-1], lambda a: a[:, :, ::-1]):
        den = np.sqrt(sig ** 2 + tr(sig) ** 2)
        ok = (den > 0) & (e > 0.01 * e.max())
        z = ((e - tr(e))[ok] / den[ok])
        assert np.abs(z).max() < 7 and np.sqrt((z ** 2).mean()) < 1.6       # t-distributed (B = 10), loose
    assert abs(e[:, :, :4].sum() - e[:, :, 4:].sum()) / tot < 0.01
    assert abs(e[:4].sum() - e[4:].sum()) / tot < 0.01


# ------------------------------------------------------------------------------------------ P12 + post-processing
def test_p12_units_and_batch_statistics(tables):
    """finalize(): 1 MeV in a 2x2x4 mm water voxel = 1.0014e-8 Gy; the batch standard
    error equals numpy's std(ddof=1)/sqrt(B) of the batch means; Eq. 2/3 by explicit loops."""
    rng = np.random.default_rng(2)
    nx, ny, nz, B, nb = 3, 2, 2, 7, 50
    c = _homog()
    rho = anm_inputs.phantoms.quantize_density(rng.uniform(0.5, 1.5, (nz, ny, nx)))
    rho[0, 0, 0] = 1.0
    lab = rng.integers(0, 3, (nz, ny, nx)).astype(np.uint8)
    lab[0, 0, 0], lab[0, 0, 1] = 1, 2
    c.update(shape=(nx, ny, nz), spacing_mm=(2.0, 2.0, 4.0), material=np.full((nz, ny, nx), 2, np.uint8), density=rho,
             labels=lab, n_organs=2, n_decays=B * nb, n_batches=B)
    o = O.Oracle(c, tables)
    x = rng.uniform(0, 2, (B, nx * ny * nz))
    x[:, 5] = 0.0                                    # a voxel that never scores
    vox_cm3 = 0.2 * 0.2 * 0.4
    mass = rho.reshape(-1).astype(np.float64) * vox_cm3
    ob = np.zeros((B, 3))
    for b in range(B):
        for v in range(x.shape[1]):
            ob[b, lab.reshape(-1)[v]] += x[b, v] / mass[v]
    f = o.finalize({"sum": x.sum(0), "sumsq": (x ** 2).sum(0), "organ_batch": ob}, total_activity_bq=2.0e8)
    # P12
    one = o.finalize({"sum": np.eye(1, x.shape[1], 0)[0] * 1.0, "sumsq": np.zeros(x.shape[1]), "organ_batch": ob * 0})
    assert abs(one["dose"][0] * (B * nb) - 1.602176634e-10 / 0.016) < 1e-20
    assert abs(1.602176634e-10 / 0.016 - 1.0014e-8) < 1e-12
    # batch statistics against numpy
    y = x / nb
    se = y.std(axis=0, ddof=1) / np.sqrt(B)
    assert np.allclose(f["rel_sigma"][y.mean(0) > 0], (se / y.mean(0).clip(1e-300))[y.mean(0) > 0], rtol=1e-9)
    assert f["rel_sigma"][5] == 0 and f["dose"][5] == 0
    k = 1.602176634e-10
    dose = x.sum(0) * k / (B * nb * mass)
    assert np.allclose(f["dose"], dose, rtol=1e-12)
    assert np.allclose(f["dose_rate"], dose * 2.0e8, rtol=1e-12)            # Eq. 1
    for oid in (1, 2):
        vs = [v for v in range(x.shape[1]) if lab.reshape(-1)[v] == oid]
        assert abs(f["organs"]["mean"][oid - 1] - np.mean([dose[v] for v in vs])) < 1e-12 * dose.max()      # Eq. 2
        nzv = [v for v in vs if dose[v] > 0]
        assert abs(f["organs"]["rms_voxel_rel_sigma"][oid - 1]
                   - np.sqrt(np.mean([f["rel_sigma"][v] ** 2 for v in nzv]))) < 1e-12                        # Eq. 3
        dob = np.array([np.mean([x[b, v] * k / (nb * mass[v]) for v in vs]) for b in range(B)])
        assert abs(f["organs"]["sigma_mean"][oid - 1] - dob.std(ddof=1) / np.sqrt(B)) < 1e-9 * dob.mean()
        assert f["organs"]["n_voxels"][oid - 1] == len(vs) and f["organs"]["n_voxels_nonzero"][oid - 1] == len(nzv)
        assert abs(f["organs"]["mass_weighted"][oid - 1] - sum(x.sum(0)[v] for v in vs) * k / (B * nb) / sum(mass[v] for v in vs)) < 1e-12 * dose.max()


def test_run_argument_checks(tables):
    c = _homog(n_decays=1000, n_batches=7)
    with pytest.raises(ValueError):
        O.Oracle(c, tables).run()                    # N % B != 0 (reading C15)
    c = _homog(n_decays=1000, n_batches=10)
    o = O.Oracle(c, tables)
    r = o.run(2, 5)
    assert r["stats"]["n_histories"] == 300


def test_batches_partition_is_exact(tables):
    """Histories are keyed by index: running batches in pieces gives the same sums as one run."""
    c = anm_inputs.make_config(2, 8)
    o = O.Oracle(c, tables, n_decays=4000, n_batches=8)
    a = o.run()
    b1, b2 = o.run(0, 3), o.run(3, 8)
    assert np.allclose(a["sum"], b1["sum"] + b2["sum"], rtol=1e-13, atol=0)
    assert np.allclose(a["sumsq"], b1["sumsq"] + b2["sumsq"], rtol=1e-13, atol=0)
    p = o.run_parallel(3)
    assert np.allclose(a["sum"], p["sum"], rtol=1e-12) and np.allclose(a["organ_batch"], p["organ_batch"], rtol=1e-12)


def test_positron_energy_in_decay_voxel(tables):
    """cfg3 option: the constant positron kinetic energy lands in the decay voxel.  In near-vacuum all
    photons escape and exactly N * 0.2498 MeV stays, distributed like the activity."""
    n = 4
    act = np.zeros((n, n, n), np.float32)
    act[1, 2, 3], act[0, 0, 0] = 3.0, 1.0
    c = _homog(n=n, d_mm=1.0, mat=0, rho=1e-6, n_decays=40_000, n_batches=4, photons_per_decay=2,
               positron_ke_mev=0.2498, activity=act, point_source_mm=None)
    r = O.Oracle(c, tables).run()
    e = r["sum"].reshape(n, n, n)
    assert abs(e.sum() - 40_000 * 0.2498) < 1e-6
    assert set(zip(*np.nonzero(e))) == {(1, 2, 3), (0, 0, 0)}
    assert abs(e[1, 2, 3] / e.sum() - 0.75) < 4 * np.sqrt(0.75 * 0.25 / 40_000)
    assert r["stats"]["n_photons"] == 80_000 and r["stats"]["n_escaped"] == 80_000
