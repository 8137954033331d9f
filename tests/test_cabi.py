"""The C-ABI library loads and exports every symbol include/mg5b200.h declares (no compute calls without a GPU)."""
import ctypes as C
import os
import re

from paper_2507_21039_b200 import binding as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "mg5b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mg_[a-z_0-9]+)\s*\(", text)))


def test_every_declared_symbol_is_exported_and_bound():
    names = _declared()
    assert "mg_create" in names and "mg_compute" in names and "mg_filter_helicities" in names and "mg_sample_rambo" in names
    lib = B.lib()
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(B.EXPORTS) == names


def test_no_torch_types_in_signatures():
    text = open(os.path.join(ROOT, "include", "mg5b200.h")).read()
    assert "torch" not in text and "at::" not in text and "std::" not in text
    assert 'extern "C"' in text


def test_error_codes_without_gpu():
    lib = B.lib()
    assert lib.mg_strerror(0) == b"success"
    assert b"mg_filter_helicities" in lib.mg_strerror(B.MG_ENOTFILTERED)
    h = C.c_void_p()
    sm = B.mg_sm_params(91.188, 2.441404, 173.0, 1.4915, 132.507, 1.16639e-5, 0.118)
    # argument validation happens before any CUDA call
    assert lib.mg_create(C.byref(h), 10, C.byref(sm), 0, 0) == B.MG_EINVAL      # ids 1..9 exist
    assert lib.mg_create(C.byref(h), 2, C.byref(sm), 7, 0) == B.MG_EINVAL
    assert lib.mg_create(None, 2, C.byref(sm), 0, 0) == B.MG_EINVAL
    assert lib.mg_create(C.byref(h), 1, C.byref(sm), B.MG_FP32, 0) == B.MG_EINVAL      # config 1 is FP64 only
    assert lib.mg_destroy(None) == 0
    assert lib.mg_get_info(None, None) == B.MG_EINVAL
    assert lib.mg_launch_count(None) == 0


def test_product_path_does_not_use_the_oracle():
    pkg = os.path.join(ROOT, "paper_2507_21039_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".inc")):
                text = open(os.path.join(dirpath, f)).read()
                for needle in ("import oracle", "from oracle", "libmg_oracle", "mg_oracle", "orc_"):
                    assert needle not in text, (dirpath, f, needle)
