"""ctypes binding of libanm.so -- argument marshalling only; every step of the path runs in the CUDA kernels.

The low-level functions keep the C names (`load().anm_run(...)`); `Simulation` wraps one `anm_ctx` with
methods named after the calls (set_grid, load_phantom, load_activity, set_point_source, load_organs,
set_physics_tables, set_options, set_stream, run, get_energy, get_dose, get_dose_rate, get_uncertainty,
get_organ_doses, get_stats).  Volume arguments may be numpy arrays (host) or CUDA torch tensors (device
pointers are passed through, `on_device=1`).  torch is used only for device memory and streams.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))

ANM_SYMBOLS = [
    "anm_create", "anm_destroy", "anm_last_error", "anm_set_stream", "anm_set_grid", "anm_load_phantom",
    "anm_load_activity", "anm_set_point_source", "anm_load_organs", "anm_set_physics_tables", "anm_set_options",
    "anm_default_options", "anm_run", "anm_get_energy", "anm_get_dose", "anm_get_dose_rate", "anm_get_uncertainty",
    "anm_get_organ_doses", "anm_get_stats", "anm_get_tally_buffers", "anm_merge", "anm_get_alias_table",
    "anm_default_hu_ramp", "anm_load_ct", "anm_get_phantom", "anm_load_pet",
    "anm_set_electron_tables", "anm_trace_electrons", "anm_philox_blocks", "anm_measure_peaks",
    "anm_organ_summary_static", "anm_set_tally_budget",
]

STATUS = {0: "ANM_OK", -1: "ANM_E_ARG", -2: "ANM_E_STATE", -3: "ANM_E_CUDA", -4: "ANM_E_NOMEM", -5: "ANM_E_UNSUPPORTED"}


class AnmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("%s: %s" % (STATUS.get(code, code), msg))
        self.code = code


class anm_tables(C.Structure):
    _fields_ = [("n_materials", C.c_int32), ("n_energy", C.c_int32), ("lnE_min", C.c_double), ("dlnE", C.c_double),
                ("mu_pe", C.c_void_p), ("mu_compton", C.c_void_p), ("mu_rayleigh", C.c_void_p),
                ("n_x2", C.c_int32), ("reserved0", C.c_int32), ("ray_x2", C.c_void_p), ("ray_cum", C.c_void_p)]


class anm_options(C.Structure):
    _fields_ = [("n_batches", C.c_int32), ("photons_per_decay", C.c_int32), ("rayleigh_on", C.c_int32),
                ("zero_air_dose", C.c_int32), ("photon_cutoff_MeV", C.c_double), ("positron_ke_MeV", C.c_double),
                ("schedule", C.c_int32), ("collect_stats", C.c_int32), ("warp_aggregate", C.c_int32),
                ("hull_majorant", C.c_int32), ("history_offset", C.c_uint64),
                ("electron_transport", C.c_int32), ("uncertainty", C.c_int32),
                ("batch_pipeline", C.c_int32), ("tally", C.c_int32),
                ("batches_per_launch", C.c_int32), ("texel_bits", C.c_int32)]


class anm_electron_tables(C.Structure):
    _fields_ = [("n_materials", C.c_int32), ("n_t", C.c_int32), ("t_min", C.c_double), ("dt", C.c_double),
                ("range", C.c_void_p)]


class anm_organ(C.Structure):
    _fields_ = [("mean_Gy_per_decay", C.c_double), ("sigma_mean", C.c_double), ("rms_voxel_rel_sigma", C.c_double),
                ("mass_weighted_Gy_per_decay", C.c_double), ("mass_g", C.c_double),
                ("n_voxels", C.c_uint64), ("n_voxels_nonzero", C.c_uint64)]


class anm_stats(C.Structure):
    _fields_ = [("emitted_MeV", C.c_double), ("deposited_MeV", C.c_double), ("escaped_MeV", C.c_double)] + [
        (n, C.c_uint64) for n in ("n_decays", "n_steps", "n_real", "n_pe", "n_compton", "n_rayleigh", "n_escaped", "n_cutoff", "n_electrons", "n_hbh_overflow")] + [
        ("ms_transport", C.c_double), ("ms_fold", C.c_double), ("ms_finalize", C.c_double), ("ms_setup", C.c_double),
        ("n_launches", C.c_uint64), ("ms_load_ct", C.c_double), ("ms_load_pet", C.c_double),
        ("tally_binned", C.c_uint64), ("n_tally_overflow", C.c_uint64),
        ("rms_rel_sigma_gt10", C.c_double), ("rms_rel_sigma_gt50", C.c_double), ("n_voxels_gt10", C.c_uint64),
        ("n_voxels_gt50", C.c_uint64), ("max_dose_Gy_per_decay", C.c_double), ("batches_per_launch", C.c_uint64),
        ("n_fly_trips", C.c_uint64), ("n_compton_tries", C.c_uint64), ("n_rayleigh_tries", C.c_uint64),
        ("texel_bits", C.c_uint64), ("n_check_violations", C.c_uint64)]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


class anm_peaks(C.Structure):
    _fields_ = [("issue_gtis", C.c_double), ("issue_sm_mhz", C.c_double), ("philox_gblocks", C.c_double), ("gather_gps", C.c_double * 2),
                ("red_gps", C.c_double * 2), ("bytes", C.c_uint64 * 2), ("mix_gps", C.c_double * 2),
                ("gather_in_flight", C.c_int32 * 2), ("red_in_flight", C.c_int32 * 2)]


ANM_MAX_RAMP_NODES = 16


class anm_hu_ramp(C.Structure):
    _fields_ = [("n_nodes", C.c_int32), ("density_bits", C.c_int32), ("hu", C.c_double * ANM_MAX_RAMP_NODES),
                ("rho", C.c_double * ANM_MAX_RAMP_NODES), ("material", C.c_int32 * ANM_MAX_RAMP_NODES),
                ("hu_outside", C.c_double)]

    @classmethod
    def from_dict(cls, ramp: dict) -> "anm_hu_ramp":
        r = cls()
        n = len(ramp["hu"])
        if n > ANM_MAX_RAMP_NODES or len(ramp["rho"]) != n or len(ramp["material"]) != n - 1:
            raise ValueError("ramp: need n HU nodes, n densities and n - 1 materials, n <= %d" % ANM_MAX_RAMP_NODES)
        r.n_nodes = n
        for k in range(n):
            r.hu[k], r.rho[k] = float(ramp["hu"][k]), float(ramp["rho"][k])
        for k in range(n - 1):
            r.material[k] = int(ramp["material"][k])
        r.hu_outside = float(ramp["hu_outside"])
        r.density_bits = int(ramp.get("density_bits", 0))
        return r

    def as_dict(self) -> dict:
        n = self.n_nodes
        d = {"hu": [self.hu[k] for k in range(n)], "rho": [self.rho[k] for k in range(n)],
             "material": [self.material[k] for k in range(n - 1)], "hu_outside": self.hu_outside}
        if self.density_bits:
            d["density_bits"] = int(self.density_bits)
        return d


def lib_path() -> str:
    """The library to load: paper_2111_11687_b200/libanm.so, or the build named by ANM_LIBRARY (e.g. the bounds-checking
    build of tests/test_gpu_bounds_check.py)."""
    return os.environ.get("ANM_LIBRARY") or os.path.join(_PKG, "libanm.so")


_lib = None


def load(build_if_missing: bool = True):
    """dlopen libanm.so and declare the prototypes.  Fails loudly (no fallback) if it cannot be built or loaded."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if build_if_missing:
        from . import build as _b
        if _b.needs_build():
            _b.build()
    if not os.path.exists(path):
        raise RuntimeError("libanm.so is missing (%s): build it with `python -m paper_2111_11687_b200.build`; "
                           "there is no CPU fallback" % path)
    L = C.CDLL(path)
    vp, i32, u64, dbl, sz = C.c_void_p, C.c_int, C.c_uint64, C.c_double, C.c_size_t
    protos = {
        "anm_create": (i32, [C.POINTER(vp), i32]), "anm_destroy": (i32, [vp]), "anm_last_error": (C.c_char_p, [vp]),
        "anm_set_stream": (i32, [vp, vp]), "anm_set_grid": (i32, [vp, i32, i32, i32, dbl, dbl, dbl]),
        "anm_load_phantom": (i32, [vp, vp, vp, i32]), "anm_load_activity": (i32, [vp, vp, i32]),
        "anm_set_point_source": (i32, [vp, dbl, dbl, dbl]), "anm_load_organs": (i32, [vp, vp, i32, i32]),
        "anm_set_physics_tables": (i32, [vp, C.POINTER(anm_tables)]), "anm_set_options": (i32, [vp, C.POINTER(anm_options)]),
        "anm_default_options": (i32, [C.POINTER(anm_options)]), "anm_run": (i32, [vp, u64, u64]),
        "anm_get_energy": (i32, [vp, vp, sz, i32]), "anm_get_dose": (i32, [vp, vp, sz, i32]),
        "anm_get_dose_rate": (i32, [vp, dbl, vp, sz, i32]), "anm_get_uncertainty": (i32, [vp, vp, sz, i32]),
        "anm_get_organ_doses": (i32, [vp, C.POINTER(anm_organ), i32]), "anm_get_stats": (i32, [vp, C.POINTER(anm_stats)]),
        "anm_get_tally_buffers": (i32, [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(sz), C.POINTER(vp), C.POINTER(i32)]),
        "anm_merge": (i32, [vp, u64, i32, vp, C.POINTER(anm_stats)]),
        "anm_get_alias_table": (i32, [vp, vp, sz, C.POINTER(sz)]),
        "anm_set_electron_tables": (i32, [vp, C.POINTER(anm_electron_tables)]),
        "anm_trace_electrons": (i32, [vp, vp, sz, vp, sz, C.POINTER(dbl)]),
        "anm_philox_blocks": (i32, [vp, u64, vp, sz, vp]),
        "anm_measure_peaks": (i32, [vp, u64, u64, C.POINTER(anm_peaks)]),
        "anm_default_hu_ramp": (i32, [C.POINTER(anm_hu_ramp)]),
        "anm_load_ct": (i32, [vp, vp, i32, i32, i32, dbl, dbl, dbl, dbl, dbl, dbl, C.POINTER(anm_hu_ramp), i32]),
        "anm_get_phantom": (i32, [vp, vp, vp, sz, i32]),
        "anm_load_pet": (i32, [vp, vp, i32, i32, i32, dbl, dbl, dbl, dbl, dbl, dbl, i32, C.POINTER(dbl), vp, sz]),
        "anm_set_tally_budget": (i32, [vp, u64]),
        "anm_organ_summary_static": (i32, [vp, vp, vp, sz, i32, dbl, vp, vp, C.c_char_p, sz]),
    }
    for name, (res, args) in protos.items():
        f = getattr(L, name)
        f.restype, f.argtypes = res, args
    _lib = L
    return L


def organ_summary_static(d_sum, d_sumsq, d_labels, n_organs: int, n_samples: float, d_out, stream=None, n_voxels=None):
    """anm_organ_summary_static (include/anm.h): the per-organ summary for callers that cannot let the library allocate
    device memory (their own allocator owns the card, or they are on a thread that must not call cudaMalloc).  No
    anm_ctx, no allocation: every argument is a CUDA torch tensor the caller already owns -- d_sum / d_sumsq float32,
    d_labels uint8 (None with n_organs = 0), d_out float64 with 3 * (n_organs + 1) elements, overwritten with
    {RMS relative sigma, voxels with energy, energy in MeV} per label (row 0: total energy in its third word).  The
    work is queued on `stream` (torch stream, raw handle or None); all calls on a device share one built-in scratch
    array, so keep them ordered on the GPU.  Marshalling only: this wrapper creates no tensor."""
    L = load()
    for t in (d_sum, d_sumsq, d_out) + ((d_labels,) if d_labels is not None else ()):
        if not (_is_torch(t) and t.is_cuda and t.is_contiguous()):
            raise ValueError("organ_summary_static takes contiguous CUDA tensors")
    if d_sum.dtype.itemsize != 4 or d_sumsq.dtype.itemsize != 4 or d_out.dtype.itemsize != 8 or (d_labels is not None and d_labels.dtype.itemsize != 1):
        raise ValueError("organ_summary_static: float32 sums, uint8 labels, float64 out")
    n = int(n_voxels) if n_voxels is not None else int(d_sum.numel())
    if d_sumsq.numel() < n or d_sum.numel() < n or (d_labels is not None and d_labels.numel() < n):
        raise ValueError("organ_summary_static: a volume is shorter than n_voxels")
    if 0 <= int(n_organs) <= 255 and d_out.numel() < 3 * (int(n_organs) + 1):
        raise ValueError("organ_summary_static: d_out needs 3 * (n_organs + 1) float64")
    h = getattr(stream, "cuda_stream", stream)
    err = C.create_string_buffer(512)
    rc = L.anm_organ_summary_static(C.c_void_p(d_sum.data_ptr()), C.c_void_p(d_sumsq.data_ptr()),
                                    C.c_void_p(d_labels.data_ptr()) if d_labels is not None else None, n, int(n_organs),
                                    float(n_samples), C.c_void_p(d_out.data_ptr()), C.c_void_p(int(h) if h else None), err, len(err))
    if rc != 0:
        raise AnmError(rc, err.value.decode())


def _is_torch(a) -> bool:
    return type(a).__module__.startswith("torch")


def _in_ptr(a, dtype, n, keep):
    """(pointer, on_device) of an input volume: numpy -> host pointer; CUDA torch tensor -> device pointer."""
    if _is_torch(a):
        import torch
        want = {np.uint8: torch.uint8, np.float32: torch.float32, np.int16: torch.int16}[dtype]
        if a.dtype != want or not a.is_contiguous() or a.numel() != n:
            raise ValueError("tensor must be contiguous %s with %d elements" % (want, n))
        keep.append(a)
        if a.is_cuda:
            return a.data_ptr(), 1
        return a.data_ptr(), 0
    arr = np.ascontiguousarray(a, dtype=dtype).reshape(-1)
    if arr.size != n:
        raise ValueError("array has %d elements, the grid has %d voxels" % (arr.size, n))
    keep.append(arr)
    return arr.ctypes.data, 0


class Simulation:
    """One anm_ctx.  Shapes are (nx, ny, nz); volumes are indexed [iz][iy][ix] (C order)."""

    def __init__(self, device: int = 0):
        self._L = load()
        self._ctx = C.c_void_p()
        rc = self._L.anm_create(C.byref(self._ctx), int(device))
        if rc != 0:
            raise AnmError(rc, "anm_create failed: no usable CUDA device %d (there is no CPU fallback)" % device)
        self.device = int(device)
        self.shape = None
        self.V = 0
        self.n_organs = 0
        self._keep = []

    def close(self):
        if getattr(self, "_ctx", None):
            self._L.anm_destroy(self._ctx)
            self._ctx = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def _ck(self, rc):
        if rc != 0:
            raise AnmError(rc, (self._L.anm_last_error(self._ctx) or b"").decode())

    # ---- inputs
    def set_stream(self, stream):
        """stream: a torch.cuda.Stream, a raw cudaStream_t integer, or None (default stream)."""
        h = getattr(stream, "cuda_stream", stream)
        self._ck(self._L.anm_set_stream(self._ctx, C.c_void_p(int(h) if h else None)))

    def set_grid(self, shape, spacing_mm):
        nx, ny, nz = (int(v) for v in shape)
        self._ck(self._L.anm_set_grid(self._ctx, nx, ny, nz, *(float(s) for s in spacing_mm)))
        self.shape, self.V = (nx, ny, nz), nx * ny * nz

    def set_tally_budget(self, n_bytes: int):
        """Bytes of per-batch tallies this ctx may keep in flight (default 4 GiB); call before set_grid (anm_set_tally_budget)."""
        self._ck(self._L.anm_set_tally_budget(self._ctx, int(n_bytes)))

    def load_phantom(self, material, density):
        keep = []
        pm, d1 = _in_ptr(material, np.uint8, self.V, keep)
        pr, d2 = _in_ptr(density, np.float32, self.V, keep)
        if d1 != d2:
            raise ValueError("material and density must both be host or both be device arrays")
        self._ck(self._L.anm_load_phantom(self._ctx, pm, pr, d1))

    def load_activity(self, activity):
        keep = []
        p, d = _in_ptr(activity, np.float32, self.V, keep)
        self._ck(self._L.anm_load_activity(self._ctx, p, d))

    def load_ct(self, hu, shape, spacing_mm, offset_mm=(0.0, 0.0, 0.0), ramp: dict | None = None):
        """CT image of int16 HU on its own grid (shape = (cnx, cny, cnz), [iz][iy][ix]) -> the phantom (anm_load_ct)."""
        cn = tuple(int(v) for v in shape)
        keep = []
        p, d = _in_ptr(hu, np.int16, cn[0] * cn[1] * cn[2], keep)
        r = anm_hu_ramp.from_dict(ramp) if ramp is not None else None
        self._ck(self._L.anm_load_ct(self._ctx, p, *cn, *(float(v) for v in spacing_mm), *(float(v) for v in offset_mm),
                                     C.byref(r) if r is not None else None, d))

    def load_pet(self, bq_per_ml, shape, spacing_mm, offset_mm=(0.0, 0.0, 0.0), out_activity=None) -> float:
        """PET image of float32 Bq/mL on its own grid -> the decay pdf (anm_load_pet).  Returns A(t_s) in Bq;
        out_activity (numpy float32 [V] for host input, CUDA tensor for device input) receives Bq per voxel."""
        pn = tuple(int(v) for v in shape)
        keep = []
        p, d = _in_ptr(bq_per_ml, np.float32, pn[0] * pn[1] * pn[2], keep)
        total = C.c_double(0.0)
        po, n = None, 0
        if out_activity is not None:
            if _is_torch(out_activity):
                po, d_out = _in_ptr(out_activity, np.float32, self.V, keep)
            else:
                if not (isinstance(out_activity, np.ndarray) and out_activity.dtype == np.float32 and
                        out_activity.flags.c_contiguous and out_activity.size == self.V):
                    raise ValueError("out_activity must be a C-contiguous float32 array with one element per voxel")
                po, d_out = out_activity.ctypes.data, 0
            if d_out != d:
                raise ValueError("out_activity must live in the same memory space as the image")
            n = self.V
        self._ck(self._L.anm_load_pet(self._ctx, p, *pn, *(float(v) for v in spacing_mm), *(float(v) for v in offset_mm),
                                      d, C.byref(total), po, n))
        return float(total.value)

    def get_phantom(self):
        """(material uint8 [nz][ny][nx], density float32) the ctx holds, on the host."""
        nx, ny, nz = self.shape
        m, r = np.empty(self.V, np.uint8), np.empty(self.V, np.float32)
        self._ck(self._L.anm_get_phantom(self._ctx, m.ctypes.data, r.ctypes.data, self.V, 0))
        return m.reshape(nz, ny, nx), r.reshape(nz, ny, nx)

    def default_hu_ramp(self) -> dict:
        r = anm_hu_ramp()
        self._ck(self._L.anm_default_hu_ramp(C.byref(r)))
        return r.as_dict()

    def set_point_source(self, xyz_mm):
        self._ck(self._L.anm_set_point_source(self._ctx, *(float(v) for v in xyz_mm)))

    def load_organs(self, labels, n_organs: int):
        keep = []
        p, d = _in_ptr(labels, np.uint8, self.V, keep)
        self._ck(self._L.anm_load_organs(self._ctx, p, int(n_organs), d))
        self.n_organs = int(n_organs)

    def set_physics_tables(self, tables: dict):
        t = anm_tables()
        keep = []
        t.n_materials, t.n_energy, t.n_x2 = int(tables["n_materials"]), int(tables["n_energy"]), int(tables["n_x2"])
        t.lnE_min, t.dlnE = float(tables["lnE_min"]), float(tables["dlnE"])
        for name, n in (("mu_pe", t.n_materials * t.n_energy), ("mu_compton", t.n_materials * t.n_energy),
                        ("mu_rayleigh", t.n_materials * t.n_energy), ("ray_x2", t.n_x2), ("ray_cum", t.n_materials * t.n_x2)):
            a = np.ascontiguousarray(tables[name], np.float32).reshape(-1)
            if a.size != n:
                raise ValueError("%s has %d elements, expected %d" % (name, a.size, n))
            keep.append(a)
            setattr(t, name, a.ctypes.data)
        self._ck(self._L.anm_set_physics_tables(self._ctx, C.byref(t)))

    def set_electron_tables(self, et: dict):
        """et = anm_inputs.make_electron_tables(): {"n_materials", "n_t", "t_min", "dt", "range" [nm][n_t]}."""
        t = anm_electron_tables()
        rng = np.ascontiguousarray(et["range"], np.float32).reshape(-1)
        t.n_materials, t.n_t, t.t_min, t.dt = int(et["n_materials"]), int(et["n_t"]), float(et["t_min"]), float(et["dt"])
        if rng.size != t.n_materials * t.n_t:
            raise ValueError("range must hold n_materials * n_t values")
        t.range = rng.ctypes.data
        self._ck(self._L.anm_set_electron_tables(self._ctx, C.byref(t)))

    def trace_electrons(self, electrons):
        """electrons: [n][7] = x, y, z (mm), unit direction, T (MeV).  Returns (energy per voxel [nz][ny][nx], escaped MeV)."""
        e = np.ascontiguousarray(electrons, np.float32).reshape(-1, 7)
        nx, ny, nz = self.shape
        out = np.zeros(self.V, np.float32)
        esc = C.c_double(0.0)
        self._ck(self._L.anm_trace_electrons(self._ctx, e.ctypes.data, e.shape[0], out.ctypes.data, self.V, C.byref(esc)))
        return out.reshape(nz, ny, nx), float(esc.value)

    def philox_blocks(self, seed: int, counters) -> np.ndarray:
        """Device Philox4x32-10 blocks for counters [n][4] (uint32) under key = seed: [n][4] uint32."""
        ctr = np.ascontiguousarray(counters, np.uint32).reshape(-1, 4)
        out = np.zeros_like(ctr)
        self._ck(self._L.anm_philox_blocks(self._ctx, int(seed), ctr.ctypes.data, ctr.shape[0], out.ctypes.data))
        return out

    def default_options(self) -> anm_options:
        o = anm_options()
        self._L.anm_default_options(C.byref(o))
        return o

    def set_options(self, **kw):
        o = self.default_options()
        for k, v in kw.items():
            if not hasattr(o, k):
                raise TypeError("unknown option %r" % k)
            setattr(o, k, v)
        self._ck(self._L.anm_set_options(self._ctx, C.byref(o)))
        return o

    # ---- run
    def run(self, n_decays: int, seed: int):
        self._ck(self._L.anm_run(self._ctx, int(n_decays), int(seed)))

    # ---- results
    def _out(self, out):
        if out is None:
            out = np.empty(self.V, np.float32)
        if _is_torch(out):
            import torch
            if out.dtype != torch.float32 or not out.is_contiguous() or out.numel() != self.V:
                raise ValueError("output tensor must be contiguous float32 with %d elements" % self.V)
            return out, out.data_ptr(), 1 if out.is_cuda else 0
        if out.dtype != np.float32 or not out.flags.c_contiguous or out.size != self.V:
            raise ValueError("output array must be contiguous float32 with %d elements" % self.V)
        return out, out.ctypes.data, 0

    def get_energy(self, out=None):
        out, p, d = self._out(out)
        self._ck(self._L.anm_get_energy(self._ctx, p, self.V, d))
        return out

    def get_dose(self, out=None):
        out, p, d = self._out(out)
        self._ck(self._L.anm_get_dose(self._ctx, p, self.V, d))
        return out

    def get_dose_rate(self, total_activity_bq: float, out=None):
        out, p, d = self._out(out)
        self._ck(self._L.anm_get_dose_rate(self._ctx, float(total_activity_bq), p, self.V, d))
        return out

    def get_uncertainty(self, out=None):
        out, p, d = self._out(out)
        self._ck(self._L.anm_get_uncertainty(self._ctx, p, self.V, d))
        return out

    def get_organ_doses(self) -> dict:
        arr = (anm_organ * self.n_organs)()
        self._ck(self._L.anm_get_organ_doses(self._ctx, arr, self.n_organs))
        names = [n for n, _ in anm_organ._fields_]
        return {n: np.array([getattr(o, n) for o in arr]) for n in names}

    def get_stats(self) -> dict:
        s = anm_stats()
        self._ck(self._L.anm_get_stats(self._ctx, C.byref(s)))
        return s.as_dict()

    def measure_peaks(self, small_bytes: int = 104_857_600, large_bytes: int = 629_145_600) -> dict:
        """Roofline microbenchmarks of this device (include/anm.h anm_measure_peaks)."""
        pk = anm_peaks()
        self._ck(self._L.anm_measure_peaks(self._ctx, int(small_bytes), int(large_bytes), C.byref(pk)))
        return {"issue_gtis": pk.issue_gtis, "issue_sm_mhz": pk.issue_sm_mhz, "philox_gblocks": pk.philox_gblocks,
                "gather_gps": [pk.gather_gps[0], pk.gather_gps[1]], "red_gps": [pk.red_gps[0], pk.red_gps[1]],
                "bytes": [int(pk.bytes[0]), int(pk.bytes[1])], "mix_gps": [pk.mix_gps[0], pk.mix_gps[1]],
                "gather_in_flight": [pk.gather_in_flight[0], pk.gather_in_flight[1]],
                "red_in_flight": [pk.red_in_flight[0], pk.red_in_flight[1]]}

    def get_alias_table(self) -> np.ndarray:
        """uint32 [n_entries][4] = {threshold, own voxel, alias voxel, 0} of the loaded activity map."""
        n = C.c_size_t()
        self._ck(self._L.anm_get_alias_table(self._ctx, None, 0, C.byref(n)))
        out = np.empty((n.value, 4), np.uint32)
        self._ck(self._L.anm_get_alias_table(self._ctx, out.ctypes.data, n.value, C.byref(n)))
        return out

    # ---- one logical run over several GPUs (include/anm.h, "one logical run over several GPUs")
    def get_tally_buffers(self):
        """Zero-copy torch views of the ctx-owned device buffers: (sum f32[Vpad], sumsq f32[Vpad], organ_rows f64[B][256])."""
        import torch
        ps, pq, pr = C.c_void_p(), C.c_void_p(), C.c_void_p()
        n, rows = C.c_size_t(), C.c_int()
        self._ck(self._L.anm_get_tally_buffers(self._ctx, C.byref(ps), C.byref(pq), C.byref(n), C.byref(pr), C.byref(rows)))

        class _View:   # the CUDA array interface is what torch.as_tensor reads: no copy, the ctx keeps ownership
            def __init__(self, ptr, shape, typestr):
                self.__cuda_array_interface__ = {"shape": shape, "typestr": typestr, "data": (int(ptr), False), "version": 3}

        dev = torch.device("cuda", self.device)
        return (torch.as_tensor(_View(ps.value, (n.value,), "<f4"), device=dev),
                torch.as_tensor(_View(pq.value, (n.value,), "<f4"), device=dev),
                torch.as_tensor(_View(pr.value, (rows.value, 256), "<f8"), device=dev))

    def merge(self, total_decays: int, total_batches: int, organ_rows_all=None, summed_stats: dict | None = None):
        rows = None
        if organ_rows_all is not None:
            rows = np.ascontiguousarray(organ_rows_all, np.float64)
            if rows.shape != (int(total_batches), 256):
                raise ValueError("organ_rows_all must be [total_batches][256]")
        st = None
        if summed_stats is not None:
            st = anm_stats()
            for k, v in summed_stats.items():
                setattr(st, k, type(getattr(st, k))(v))
        self._ck(self._L.anm_merge(self._ctx, int(total_decays), int(total_batches),
                                   rows.ctypes.data if rows is not None else None, C.byref(st) if st is not None else None))

    # ---- convenience: everything a config dict (anm_inputs.make_config) describes
    def load_config(self, cfg: dict, tables: dict, **options):
        self.set_grid(cfg["shape"], cfg["spacing_mm"])
        self.load_phantom(cfg["material"], cfg["density"])
        if cfg.get("point_source_mm") is not None:
            self.set_point_source(cfg["point_source_mm"])
        else:
            self.load_activity(cfg["activity"])
        if cfg.get("labels") is not None and cfg.get("n_organs"):
            self.load_organs(cfg["labels"], cfg["n_organs"])
        self.set_physics_tables(tables)
        opts = dict(n_batches=cfg["n_batches"], photons_per_decay=cfg["photons_per_decay"],
                    rayleigh_on=cfg["rayleigh_on"], photon_cutoff_MeV=cfg["photon_cutoff_mev"],
                    positron_ke_MeV=cfg["positron_ke_mev"])
        opts.update(options)
        self.set_options(**opts)
