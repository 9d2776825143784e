"""ctypes front end of the CPU oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from paper_2111_11687_b200/ (the CUDA path).

The transport itself is oracle/anm_oracle.cpp (plain single-threaded fp64 C++).  This file adds
  * build():   g++ -O2 -shared  ->  oracle/liboracle.so
  * Oracle:    problem set-up, single-process and multi-process (whole batches per process,
               SURVEY.md §8(d) "Timing the oracle beside it") runs
  * finalize(): the paper's post-processing written out in numpy --
                Eq. 1 dose rate = D / N_evts x A(t_s),
                Eq. 2 organ mean = unweighted mean of the organ's voxel doses,
                Eq. 3 organ uncertainty = RMS of the voxel uncertainties,
                and the batch-method standard error of the mean (north_star (c); reading C1).
"""
from __future__ import annotations

import ctypes as C
import multiprocessing as mp
import os
import subprocess
import time

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "anm_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")

MEV_PER_G_TO_GY = 1.602176634e-10     # 1 MeV/g in Gy (P12)


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


class OrcTables(C.Structure):
    _fields_ = [("n_materials", C.c_int32), ("n_energy", C.c_int32), ("lnE_min", C.c_double),
                ("dlnE", C.c_double), ("mu_pe", C.c_void_p), ("mu_compton", C.c_void_p),
                ("mu_rayleigh", C.c_void_p), ("n_x2", C.c_int32), ("pad_", C.c_int32),
                ("ray_x2", C.c_void_p), ("ray_cum", C.c_void_p)]


class OrcProblem(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("pad0_", C.c_int32),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
                ("material", C.c_void_p), ("density", C.c_void_p), ("cdf", C.c_void_p),
                ("use_point_source", C.c_int32), ("pad1_", C.c_int32),
                ("px", C.c_double), ("py", C.c_double), ("pz", C.c_double),
                ("labels", C.c_void_p), ("n_organs", C.c_int32), ("photons_per_decay", C.c_int32),
                ("rayleigh_on", C.c_int32), ("tracking", C.c_int32),
                ("photon_cutoff", C.c_double), ("positron_ke", C.c_double),
                ("n_total", C.c_uint64), ("n_batches", C.c_int32), ("pad2_", C.c_int32),
                ("seed", C.c_uint64), ("t", OrcTables),
                ("electron_on", C.c_int32), ("n_t", C.c_int32), ("electron_cutoff", C.c_double),
                ("t_min", C.c_double), ("dt", C.c_double), ("e_range", C.c_void_p), ("activity", C.c_void_p)]


class OrcStats(C.Structure):
    _fields_ = [("emitted", C.c_double), ("deposited", C.c_double), ("escaped", C.c_double),
                ("max_history_residual", C.c_double)] + [
        (n, C.c_uint64) for n in ("n_histories", "n_photons", "n_crossings", "n_collisions", "n_pe",
                                  "n_compton", "n_rayleigh", "n_escaped", "n_cutoff", "n_virtual",
                                  "n_electrons", "n_electron_crossings", "n_substeps")]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_interp.restype = C.c_double
        L.orc_interp.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_double]
        L.orc_pick_voxel.restype = C.c_uint64
        L.orc_pick_voxel.argtypes = [C.c_void_p, C.c_uint64, C.c_double]
        L.orc_build_cdf.argtypes = [C.c_void_p, C.c_uint64, C.c_void_p]
        L.orc_philox4x32_10.argtypes = [C.c_void_p] * 3
        L.orc_isotropic_many.argtypes = [C.c_uint64, C.c_uint64, C.c_void_p]
        L.orc_kn_sample_many.argtypes = [C.c_double, C.c_uint64, C.c_uint64, C.c_void_p]
        L.orc_rayleigh_sample_many.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_uint64, C.c_uint64, C.c_void_p]
        L.orc_rotate.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_void_p]
        L.orc_sample_source_many.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_flight.restype = C.c_int
        L.orc_flight.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_double,
                                 C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_compton_electron_direction.argtypes = [C.c_double, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_e_range.restype = C.c_double
        L.orc_e_range.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.orc_e_energy.restype = C.c_double
        L.orc_e_energy.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.orc_electron_walk.restype = C.c_int
        L.orc_electron_walk.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        L.orc_run.restype = C.c_int
        L.orc_run.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64] + [C.c_void_p] * 7
        _lib = L
    return _lib


def _ptr(a):
    return a.ctypes.data if a is not None else None


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, np.uint32)
    k = np.asarray(key, np.uint32)
    out = np.zeros(4, np.uint32)
    lib().orc_philox4x32_10(_ptr(c), _ptr(k), _ptr(out))
    return out


def tables_struct(tables: dict, keep: list) -> OrcTables:
    t = OrcTables()
    t.n_materials, t.n_energy = tables["n_materials"], tables["n_energy"]
    t.lnE_min, t.dlnE, t.n_x2 = tables["lnE_min"], tables["dlnE"], tables["n_x2"]
    for name in ("mu_pe", "mu_compton", "mu_rayleigh", "ray_x2", "ray_cum"):
        a = np.ascontiguousarray(tables[name], np.float32)
        keep.append(a)
        setattr(t, name, _ptr(a))
    return t


class Oracle:
    """One problem (phantom + source + tables + run parameters) for the CPU oracle.

    cfg: a dict from anm_inputs.make_config (arrays [nz][ny][nx]); overrides: n_decays, n_batches,
    seed, rayleigh_on, positron_ke_mev, photons_per_decay, tracking.
    """

    def __init__(self, cfg: dict, tables: dict, **over):
        self._keep = []
        nx, ny, nz = cfg["shape"]
        self.shape = (nx, ny, nz)
        self.V = nx * ny * nz
        self.spacing_cm = tuple(s / 10.0 for s in cfg["spacing_mm"])
        get = lambda k: over.get(k, cfg.get(k))   # noqa: E731
        self.n_decays = int(get("n_decays"))
        self.n_batches = int(get("n_batches"))
        self.material = np.ascontiguousarray(cfg["material"], np.uint8).reshape(-1)
        self.density = np.ascontiguousarray(cfg["density"], np.float32).reshape(-1)
        assert self.material.size == self.V and self.density.size == self.V
        assert int(self.material.max()) < tables["n_materials"]
        self.labels = None
        self.n_organs = int(cfg.get("n_organs") or 0)
        if cfg.get("labels") is not None:
            self.labels = np.ascontiguousarray(cfg["labels"], np.uint8).reshape(-1)
            assert int(self.labels.max()) <= self.n_organs
        p = OrcProblem()
        p.nx, p.ny, p.nz = nx, ny, nz
        p.dx, p.dy, p.dz = self.spacing_cm
        p.material, p.density, p.labels = _ptr(self.material), _ptr(self.density), _ptr(self.labels)
        p.n_organs = self.n_organs
        if cfg.get("point_source_mm") is not None:
            p.use_point_source = 1
            p.px, p.py, p.pz = (c / 10.0 for c in cfg["point_source_mm"])
            self.cdf = None
        else:
            act = np.ascontiguousarray(cfg["activity"], np.float32).reshape(-1)
            assert act.size == self.V and float(act.min()) >= 0.0 and float(act.max()) > 0.0
            self.activity = act
            p.activity = _ptr(act)
            self.cdf = np.zeros(self.V, np.float64)
            lib().orc_build_cdf(_ptr(act), self.V, _ptr(self.cdf))
            p.cdf = _ptr(self.cdf)
        p.photons_per_decay = int(get("photons_per_decay"))
        p.rayleigh_on = int(get("rayleigh_on"))
        p.tracking = int(over.get("tracking", 0))
        p.photon_cutoff = float(get("photon_cutoff_mev"))
        p.positron_ke = float(get("positron_ke_mev"))
        p.n_total, p.n_batches, p.seed = self.n_decays, self.n_batches, int(get("seed"))
        p.t = tables_struct(tables, self._keep)
        # secondary-electron transport (NEXT-2): electron_tables = anm_inputs.make_electron_tables()
        et = over.get("electron_tables")
        p.electron_on = int(bool(over.get("electron_on", et is not None)))
        if et is not None:
            rng = np.ascontiguousarray(et["range"], np.float32)
            assert rng.shape == (tables["n_materials"], et["n_t"])
            self._keep.append(rng)
            p.n_t, p.t_min, p.dt, p.e_range = int(et["n_t"]), float(et["t_min"]), float(et["dt"]), _ptr(rng)
            p.electron_cutoff = float(over.get("electron_cutoff_mev", et["t_min"]))
        self.p = p
        self.tables = tables

    # ------------------------------------------------------------------ runs
    def run(self, b0: int = 0, b1: int | None = None, first_collision: bool = False, hbh: bool = False) -> dict:
        """Run batches [b0, b1) in this process.  hbh: also score sum over histories of X_h^2 per voxel (NEXT-4)."""
        b1 = self.n_batches if b1 is None else b1
        nb = self.n_decays // self.n_batches
        h0, h1 = b0 * nb, b1 * nb
        s = np.zeros(self.V, np.float64)
        q = np.zeros(self.V, np.float64)
        ob = np.zeros((self.n_batches, self.n_organs + 1), np.float64)
        st = OrcStats()
        fcd = np.zeros(h1 - h0, np.float64) if first_collision else None
        fce = np.zeros(h1 - h0, np.float64) if first_collision else None
        t0 = time.perf_counter()
        hq = np.zeros(self.V, np.float64) if hbh else None
        rc = lib().orc_run(C.byref(self.p), h0, h1, _ptr(s), _ptr(q), _ptr(ob), C.byref(st), _ptr(fcd), _ptr(fce), _ptr(hq))
        dt = time.perf_counter() - t0
        if rc != 0:
            raise ValueError("orc_run: bad arguments (N %% B != 0, or range not on batch boundaries)")
        out = {"sum": s, "sumsq": q, "organ_batch": ob, "stats": st.as_dict(), "seconds": dt,
               "n_decays_run": h1 - h0}
        if first_collision:
            out["fc_dist"], out["fc_dep"] = fcd, fce
        if hbh:
            out["hbh_sumsq"] = hq
        return out

    def run_parallel(self, n_procs: int | None = None, hbh: bool = False) -> dict:
        """All batches, split as whole batches over n_procs forked single-threaded processes."""
        n_procs = min(n_procs or os.cpu_count() or 1, self.n_batches)
        if n_procs <= 1:
            r = self.run(hbh=hbh)
            r["cores"] = 1
            return r
        ctx = mp.get_context("fork")
        V, B, no = self.V, self.n_batches, self.n_organs + 1
        sh_sum, sh_sq = ctx.RawArray("d", V), ctx.RawArray("d", V)
        sh_ob = ctx.RawArray("d", B * no)
        sh_hq = ctx.RawArray("d", V) if hbh else None
        lock = ctx.Lock()
        qout = ctx.Queue()
        bounds = np.linspace(0, B, n_procs + 1).astype(int)

        def work(i):
            r = self.run(int(bounds[i]), int(bounds[i + 1]), hbh=hbh)
            with lock:
                if hbh:
                    np.frombuffer(sh_hq, np.float64)[:] += r["hbh_sumsq"]
                np.frombuffer(sh_sum, np.float64)[:] += r["sum"]
                np.frombuffer(sh_sq, np.float64)[:] += r["sumsq"]
                np.frombuffer(sh_ob, np.float64)[:] += r["organ_batch"].reshape(-1)
            qout.put((r["stats"], r["seconds"]))

        t0 = time.perf_counter()
        procs = [ctx.Process(target=work, args=(i,)) for i in range(n_procs)]
        for pr in procs:
            pr.start()
        res = [qout.get() for _ in procs]
        for pr in procs:
            pr.join()
        wall = time.perf_counter() - t0
        stats = {k: (max(r[0][k] for r in res) if k == "max_history_residual" else sum(r[0][k] for r in res))
                 for k in res[0][0]}
        out = {"sum": np.frombuffer(sh_sum, np.float64).copy(), "sumsq": np.frombuffer(sh_sq, np.float64).copy(),
               "organ_batch": np.frombuffer(sh_ob, np.float64).reshape(B, no).copy(), "stats": stats,
               "seconds": wall, "cpu_seconds": sum(r[1] for r in res), "cores": n_procs,
               "n_decays_run": self.n_decays}
        if hbh:
            out["hbh_sumsq"] = np.frombuffer(sh_hq, np.float64).copy()
        return out

    # ------------------------------------------------------------------ electron pins
    def electron_range(self, m: int, T: float) -> float:
        return float(lib().orc_e_range(C.byref(self.p), int(m), float(T)))

    def electron_energy(self, m: int, r: float) -> float:
        return float(lib().orc_e_energy(C.byref(self.p), int(m), float(r)))

    def electron_walk(self, pos_cm, direction, T: float, cap: int = 4096):
        """One CSDA straight-line walk: ([(voxel, MeV), ...] in path order, escaped MeV)."""
        pos = np.asarray(pos_cm, np.float64); d = np.asarray(direction, np.float64)
        vox = np.zeros(cap, np.int64); dep = np.zeros(cap, np.float64); esc = C.c_double(0.0)
        n = lib().orc_electron_walk(C.byref(self.p), _ptr(pos), _ptr(d), float(T), _ptr(vox), _ptr(dep), cap, C.byref(esc))
        assert n <= cap
        return list(zip(vox[:n].tolist(), dep[:n].tolist())), float(esc.value)

    # ------------------------------------------------------------------ post-processing
    def finalize(self, r: dict, total_activity_bq: float | None = None) -> dict:
        """SURVEY.md §8(c) step 7, written out.  r: result of run()/run_parallel() over ALL batches."""
        N, B = float(self.n_decays), self.n_batches
        nb = N / B
        vox_cm3 = self.spacing_cm[0] * self.spacing_cm[1] * self.spacing_cm[2]
        mass = self.density.astype(np.float64) * vox_cm3                       # g
        S, Q = r["sum"], r["sumsq"]
        dose = S * MEV_PER_G_TO_GY / (N * mass)                                # Gy per decay
        ybar = S / N                                                           # MeV per decay
        var = (Q / (nb * nb) / B - ybar * ybar) / (B - 1) if B > 1 else np.zeros_like(S)
        s_abs = np.sqrt(np.maximum(var, 0.0))                                  # standard error of ybar
        rel = np.divide(s_abs, ybar, out=np.zeros_like(S), where=ybar > 0)
        out = {"energy": S, "dose": dose, "rel_sigma": rel, "dose_sigma": dose * rel}
        if "hbh_sumsq" in r:
            # history-by-history (Walters et al. 2002): s^2 of the mean = (sum X^2 / N - (sum X / N)^2) / (N - 1)
            var_h = (r["hbh_sumsq"] / N - ybar * ybar) / (N - 1.0)
            out["rel_sigma_hbh"] = np.divide(np.sqrt(np.maximum(var_h, 0.0)), ybar, out=np.zeros_like(S), where=ybar > 0)
        # run-level "statistical uncertainty" (PAPER.md:L109, L117 quote one figure per run without defining it; reading
        # C17): RMS of the relative sigma over the non-air voxels (material id 0 = air) whose dose exceeds
        # 10 % / 50 % of the largest non-air voxel dose
        body = self.material != 0
        dmax = float(dose[body].max()) if body.any() else 0.0
        out["max_dose"] = dmax
        for name, frac in (("gt10", 0.1), ("gt50", 0.5)):
            sel = body & (dose > frac * dmax)
            out["n_voxels_" + name] = int(sel.sum())
            out["rms_rel_sigma_" + name] = float(np.sqrt(np.mean(rel[sel] ** 2))) if sel.any() else 0.0
        if total_activity_bq is not None:
            out["dose_rate"] = dose * total_activity_bq                        # Eq. 1
        if self.labels is not None and self.n_organs > 0:
            no = self.n_organs
            lab = self.labels
            n_vox = np.bincount(lab, minlength=no + 1).astype(np.float64)[: no + 1]
            with np.errstate(divide="ignore", invalid="ignore"):
                d_ob = r["organ_batch"] * MEV_PER_G_TO_GY / (nb * n_vox[None, :])   # [B][no+1] organ mean per batch
                d_o = d_ob.mean(axis=0)                                             # Eq. 2
                sig_o = np.sqrt(np.maximum((d_ob ** 2).mean(axis=0) - d_o ** 2, 0.0) / (B - 1)) if B > 1 else 0 * d_o
                nz = dose > 0
                n_nz = np.bincount(lab[nz], minlength=no + 1).astype(np.float64)[: no + 1]
                rms = np.sqrt(np.bincount(lab[nz], weights=rel[nz] ** 2, minlength=no + 1)[: no + 1] / n_nz)  # Eq. 3
                m_o = np.bincount(lab, weights=mass, minlength=no + 1)[: no + 1]
                e_o = np.bincount(lab, weights=S, minlength=no + 1)[: no + 1]
                mw = e_o * MEV_PER_G_TO_GY / (N * m_o)
            fix = lambda a: np.nan_to_num(a, nan=0.0, posinf=0.0, neginf=0.0)   # noqa: E731
            out["organs"] = {"mean": fix(d_o)[1:], "sigma_mean": fix(sig_o)[1:], "rms_voxel_rel_sigma": fix(rms)[1:],
                             "mass_weighted": fix(mw)[1:], "mass_g": m_o[1:], "n_voxels": n_vox[1:],
                             "n_voxels_nonzero": n_nz[1:]}
        return out
