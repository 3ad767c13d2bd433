"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/nms.h declares; without a CUDA device the product fails loudly (no CPU fallback)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "nms.h")).read()
    return sorted(set(re.findall(r"^NMS_API\s+[\w\s\*]+?\b(nms_\w+)\s*\(", text, flags=re.M)))


def test_header_declares_the_north_star_entry_points():
    names = _declared_symbols()
    for must in ["nms_create", "nms_set_sample", "nms_amplitudes", "nms_response", "nms_azimuthal_average",
                 "nms_correlation", "nms_form_factor_split", "nms_compute", "nms_run_host", "nms_destroy"]:
        assert must in names


def test_library_exports_every_declared_symbol():
    import paper_2601_18444_b200 as nms
    lib = C.CDLL(nms.LIB_PATH)
    declared = _declared_symbols()
    assert len(declared) >= 20
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in include/nms.h but not exported by libnms.so"
    assert sorted(nms.EXPORTS) == declared


def test_binding_has_same_names():
    import paper_2601_18444_b200 as nms
    for name in _declared_symbols():
        assert callable(getattr(nms, name)), name


def test_no_cpu_fallback_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    import paper_2601_18444_b200 as nms
    with pytest.raises(nms.NmsError) as e:
        nms.nms_create(0)
    assert e.value.status == nms.NMS_E_CUDA
    # the raw entry point reports NMS_E_CUDA too and leaves *out NULL
    lib = C.CDLL(nms.LIB_PATH)
    out = C.c_void_p(123)
    assert lib.nms_create(C.byref(out), 0, None) == nms.NMS_E_CUDA
    assert out.value is None


def test_null_context_is_an_argument_error():
    import paper_2601_18444_b200 as nms
    lib = C.CDLL(nms.LIB_PATH)
    assert lib.nms_synchronize(None) == nms.NMS_E_ARG
    assert lib.nms_create(None, 0, None) == nms.NMS_E_ARG
    lib.nms_destroy(None)   # allowed


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2601_18444_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "nmso" not in text, f
