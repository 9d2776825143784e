"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol that
include/anm.h declares; structure layouts of the binding match the header; no-GPU behaviour is a loud error."""
import ctypes as C
import os
import re

import pytest

import paper_2111_11687_b200 as pkg
from paper_2111_11687_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    txt = open(os.path.join(ROOT, "include", "anm.h")).read()
    return sorted(set(re.findall(r"^(?:int|const char\*)\s+(anm_[a-z_]+)\s*\(", txt, flags=re.M)))


def test_header_symbols_exported():
    lib = binding.load()
    names = _declared()
    assert len(names) >= 19
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(pkg.ANM_SYMBOLS) == names


def test_library_is_sm100a_cuda():
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", binding.lib_path()], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_struct_sizes_match_header():
    # sizes implied by include/anm.h on LP64
    assert C.sizeof(binding.anm_tables) == 8 + 16 + 24 + 8 + 16
    assert C.sizeof(binding.anm_options) == 16 + 16 + 16 + 8 + 8 + 8 + 8
    assert C.sizeof(binding.anm_electron_tables) == 8 + 16 + 8
    assert C.sizeof(binding.anm_organ) == 5 * 8 + 2 * 8
    assert C.sizeof(binding.anm_stats) == 3 * 8 + 10 * 8 + 4 * 8 + 8 + 2 * 8 + 2 * 8 + 11 * 8
    assert C.sizeof(binding.anm_hu_ramp) == 8 + 16 * 8 + 16 * 8 + 16 * 4 + 8
    assert C.sizeof(binding.anm_peaks) == 3 * 8 + 2 * 8 + 2 * 8 + 2 * 8 + 2 * 8 + 4 * 4


def test_default_options():
    lib = binding.load()
    o = binding.anm_options()
    assert lib.anm_default_options(C.byref(o)) == 0
    assert (o.n_batches, o.photons_per_decay, o.rayleigh_on) == (100, 2, 1)
    assert abs(o.photon_cutoff_MeV - 0.010) < 1e-15 and o.positron_ke_MeV == 0.0 and o.history_offset == 0
    assert lib.anm_default_options(None) == -1


def test_default_hu_ramp_matches_the_input_module():
    """include/anm.h's default HU ramp and anm_inputs.DEFAULT_HU_RAMP (which the oracle is handed) hold the same numbers."""
    import anm_inputs
    lib = binding.load()
    r = binding.anm_hu_ramp()
    assert lib.anm_default_hu_ramp(C.byref(r)) == 0
    assert r.as_dict() == {k: list(v) if isinstance(v, list) else v for k, v in anm_inputs.DEFAULT_HU_RAMP.items()}
    assert lib.anm_default_hu_ramp(None) == -1
    back = binding.anm_hu_ramp.from_dict(anm_inputs.DEFAULT_HU_RAMP).as_dict()
    assert back == r.as_dict()


def test_no_gpu_is_a_loud_error():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(pkg.AnmError) as ei:
        pkg.Simulation(0)
    assert ei.value.code == -3          # ANM_E_CUDA: no CPU fallback


def test_null_ctx_calls_do_not_crash():
    lib = binding.load()
    assert lib.anm_destroy(None) == 0
    assert lib.anm_run(None, 10, 1) == -1
    assert lib.anm_last_error(None) == b"null context"
    assert lib.anm_set_tally_budget(None, 1 << 30) == -1


def test_static_summary_checks_its_arguments_before_it_touches_the_gpu():
    """anm_organ_summary_static validates sizes and pointers first: these refusals need no device."""
    lib = binding.load()
    err = C.create_string_buffer(256)
    assert lib.anm_organ_summary_static(None, None, None, 16, 256, 10.0, None, None, err, len(err)) == -1
    assert b"at most 255 organs" in err.value
    assert lib.anm_organ_summary_static(None, None, None, 16, 4, 10.0, None, None, err, len(err)) == -1
    assert b"must not be NULL" in err.value
    assert lib.anm_organ_summary_static(None, None, None, 16, 4, 10.0, None, None, None, 0) == -1     # no buffer: still no crash


def test_product_does_not_import_oracle():
    """The CUDA path must not route through the oracle or the input generators' arithmetic."""
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2111_11687_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "liboracle" not in txt, f
                assert "anm_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_2111_11687_b200", txt, flags=re.M)
            assert "libanm" not in txt and "anm_kernels" not in txt
