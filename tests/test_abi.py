"""The C-ABI library loads without a GPU and exports every symbol include/csf.h declares; compute entry points fail
loudly (CSF_ECUDA) when no CUDA device is present. No compute call is made here."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2410_02754_b200 import build
    return C.CDLL(build.build())


def _declared():
    src = open(os.path.join(ROOT, "include", "csf.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(csf_[a-zA-Z0-9_]+)\s*\(", src)))


def test_header_declares_the_boundary_calls():
    names = _declared()
    for need in ["csf_create", "csf_destroy", "csf_num_nodes", "csf_node_coords", "csf_mass_diag", "csf_set_potential", "csf_set_projectors",
                 "csf_workspace_bytes", "csf_apply_H", "csf_filter", "csf_filter_host", "csf_last_error"]:
        assert need in names


def test_library_exports_every_declared_symbol(lib):
    for name in _declared():
        assert hasattr(lib, name), f"libcsf.so does not export {name}"


def test_binding_lists_the_same_names():
    from paper_2410_02754_b200 import binding
    assert sorted(binding.EXPORTS) == _declared()


def test_no_cpu_fallback(lib):
    """Without a CUDA device csf_create must fail with CSF_ECUDA (-3), never fall back to host code."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    h = C.c_void_p()
    nc = (C.c_int * 3)(2, 2, 2); bx = (C.c_double * 3)(1.0, 1.0, 1.0); bc = (C.c_int * 3)(0, 0, 0)
    rc = lib.csf_create(C.byref(h), nc, bx, C.c_int(3), bc, C.c_int(0), None)
    assert rc == -3 and not h.value
    lib.csf_last_error.restype = C.c_char_p
    assert b"CUDA" in lib.csf_last_error(None)
    # argument errors are still reported before any device work
    nc0 = (C.c_int * 3)(2, 0, 2)
    assert lib.csf_create(C.byref(h), nc0, bx, C.c_int(3), bc, C.c_int(0), None) == -1
    bcf = (C.c_int * 3)(0, 0, 2)
    assert lib.csf_create(C.byref(h), nc, bx, C.c_int(3), bcf, C.c_int(0), None) == -5
