"""Pins for the input generators (anm_inputs): cross-section tables and phantoms.

P2: the Klein-Nishina total cross-section against (i) the values printed in the
survey and (ii) direct numerical integration of the differential cross-section.
"""
import numpy as np
import pytest
from scipy import integrate

import anm_inputs
from anm_inputs import tables as T
from anm_inputs.materials import MATERIALS, ELEMENTS, N_AVOGADRO

BARN = 1e-24


def test_p2_kn_total_printed_values():
    # SURVEY.md §8(c) P2, barns per electron
    E = [0.010, 0.030, 0.050, 0.100, 0.200, 0.300, 0.400, 0.51099895]
    want = [0.640470, 0.597494, 0.561507, 0.492748, 0.406482, 0.353450, 0.316680, 0.286540]
    got = anm_inputs.sigma_kn_per_electron(np.array(E)) / BARN
    assert np.allclose(got, want, rtol=0, atol=2e-6)
    # Thomson limit 8 pi r_e^2 / 3 = 0.665246 b
    a = 1e-3                                      # low-energy expansion sigma_T (1 - 2a + 26a^2/5)
    got = anm_inputs.sigma_kn_per_electron(a * T.E0_MEV) / BARN
    assert abs(got - 0.665246 * (1 - 2 * a + 5.2 * a * a)) < 2e-6


@pytest.mark.parametrize("E", [0.01, 0.08, 0.3, 0.511])
def test_p2_kn_total_vs_quadrature(E):
    a = E / T.E0_MEV

    def dsdo(c):   # Klein-Nishina d(sigma)/d(Omega), integrated over azimuth
        k = 1.0 / (1.0 + a * (1.0 - c))
        return 2 * np.pi * 0.5 * T.R_E_CM ** 2 * k * k * (k + 1.0 / k - (1.0 - c * c))

    num, _ = integrate.quad(dsdo, -1, 1, epsabs=0, epsrel=1e-11)
    assert abs(num / anm_inputs.sigma_kn_per_electron(E) - 1.0) < 1e-9


def test_water_compton_at_511(tables):
    # water 0.09578 cm^2/g at 0.511 MeV; total 0.096-0.097 (C6 sanity)
    m = anm_inputs.MATERIAL_IDS["water"]
    mc = T.interp_lnE(tables["mu_compton"][m], T.E0_MEV, tables["lnE_min"], tables["dlnE"])
    assert abs(mc - 0.09578) < 2e-5
    tot = mc + sum(T.interp_lnE(tables[k][m], T.E0_MEV, tables["lnE_min"], tables["dlnE"])
                   for k in ("mu_pe", "mu_rayleigh"))
    assert 0.0955 < tot < 0.0975


def test_electron_densities():
    want = {"water": 3.3428e23, "air_dry": 3.0062e23, "bone_compact_icru": 3.1001e23, "lung_icrp": 3.3151e23}
    for m in MATERIALS:
        assert abs(anm_inputs.electrons_per_gram(m) / want[m["name"]] - 1) < 2e-4
        assert abs(sum(m["w"].values()) - 1.0) < 2e-3


@pytest.mark.parametrize("E", [0.012, 0.06, 0.511])
def test_rayleigh_total_vs_quadrature(tables, E):
    """mu_rayleigh (closed form) against numerical integration of (1+c^2) F^2 over the sphere."""
    for mi, mat in enumerate(MATERIALS):
        Tm = float(T.x2_max(E))
        tot = 0.0
        for el, w in mat["w"].items():
            Z, A = ELEMENTS[el]
            a = (0.3 * Z ** (1 / 3)) ** 2
            f = lambda c: (1 + c * c) * Z * Z * (1 + Tm * (1 - c) / 2 / a) ** -4   # noqa: E731
            # forward peak: split the interval
            pts = [1 - 2 * min(1.0, k * a / Tm) for k in (1, 10, 100)]
            num, _ = integrate.quad(f, -1, 1, points=sorted(set(pts)), epsabs=0, epsrel=1e-10, limit=400)
            tot += N_AVOGADRO * w / A * np.pi * T.R_E_CM ** 2 * num
        got = T.interp_lnE(tables["mu_rayleigh"][mi], E, tables["lnE_min"], tables["dlnE"])
        assert abs(got / tot - 1) < 2e-4     # fp32 storage + lnE interpolation of a smooth curve


def test_rayleigh_cum_monotone_and_grid(tables):
    x2, cum = tables["ray_x2"], tables["ray_cum"]
    assert x2[0] == 0 and np.all(np.diff(x2) > 0) and x2[-1] >= T.x2_max(0.512)
    assert np.all(cum[:, 0] == 0) and np.all(np.diff(cum, axis=1) >= 0)


def test_energy_grid(tables):
    lnE = tables["lnE_min"] + tables["dlnE"] * np.arange(tables["n_energy"])
    assert abs(np.exp(lnE[0]) - 0.010) < 1e-12 and abs(np.exp(lnE[-1]) - 0.512) < 1e-9
    for k in ("mu_pe", "mu_compton", "mu_rayleigh"):
        assert tables[k].shape == (4, 512) and tables[k].dtype == np.float32 and np.all(tables[k] > 0)


def test_configs_small():
    c0 = anm_inputs.make_config(0)
    assert c0["shape"] == (32, 32, 32) and c0["spacing_mm"] == (4.0, 4.0, 4.0)
    assert c0["point_source_mm"] == (64.0, 64.0, 64.0) and c0["photons_per_decay"] == 1 and c0["n_batches"] == 10
    c1 = anm_inputs.make_config(1, 2)
    assert c1["activity"].sum() == 1.0 and c1["activity"][25, 25, 25] == 1.0
    c2 = anm_inputs.make_config(2, 2)
    assert c2["shape"] == (64, 64, 64)
    assert [int(c2["material"][z, 0, 0]) for z in (0, 16, 32, 48)] == [2, 1, 3, 2]
    assert np.allclose([c2["density"][z, 0, 0] for z in (0, 16, 32, 48)], [1.0, 0.26, 1.92, 1.0], atol=1e-6)
    assert c2["activity"].sum() == 8 ** 3 and c2["activity"][4:12, 28:36, 28:36].all()


def test_config3_structure():
    c = anm_inputs.make_config(3, 4)
    nx, ny, nz = c["shape"]
    assert (nx, ny, nz) == (64, 64, 100) and c["spacing_mm"] == (8.0, 8.0, 16.0)
    mat, rho, lab, act = c["material"], c["density"], c["labels"], c["activity"]
    assert mat.shape == (nz, ny, nx) and lab.dtype == np.uint8 and act.dtype == np.float32
    body = mat != 0
    frac = body.mean()
    assert abs(frac - np.pi * 170 * 110 / 512 ** 2) < 0.01           # elliptical cylinder in the 512 mm square
    assert np.allclose(rho[~body], 0.0012, atol=1e-6) and np.all(act[~body] == 0)
    assert np.all(rho[mat == 1] == rho[mat == 1][0]) and abs(rho[mat == 1][0] - 0.26) < 1e-6
    assert rho[mat == 3].min() >= 1.4 - 1e-6 and rho[mat == 3].max() <= 1.9 + 1e-6
    soft = (mat == 2)
    assert 0.9 <= rho[soft].min() and rho[soft].max() < 1.2 and 1.0 < rho[soft].mean() < 1.06
    # densities sit on the texel grid
    k = rho.astype(np.float64) * 2 ** 20
    assert np.all(k == np.round(k))
    assert lab.max() <= 27 and act.max() > 15.0     # bladder x20
    # same seeds -> identical volumes
    c2 = anm_inputs.make_config(3, 4)
    assert np.array_equal(c2["density"], rho) and np.array_equal(c2["activity"], act)
