"""The C-ABI library builds, loads, and exports every symbol include/*.h declares.
No compute calls here (no GPU on this box)."""
import ctypes
import glob
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_1011_4687_b200 import build
    return build.build()


def declared_symbols():
    names = []
    for hdr in glob.glob(os.path.join(ROOT, "include", "*.h")):
        text = re.sub(r"/\*.*?\*/", "", open(hdr).read(), flags=re.S)
        names += re.findall(r"\b(qmmm_[a-z_0-9]+)\s*\(", text)
    return sorted(set(names))


def test_header_declares_the_north_star_calls():
    syms = declared_symbols()
    for must in ("qmmm_field_create", "qmmm_field_eval", "qmmm_field_destroy"):
        assert must in syms


def test_library_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(lib_path)
    for name in declared_symbols():
        assert hasattr(lib, name), f"{name} declared in include/*.h but not exported"


def test_binding_lists_the_same_symbols(lib_path):
    from paper_1011_4687_b200 import binding
    assert sorted(binding.EXPORTED_SYMBOLS) == declared_symbols()


def test_header_compiles_as_plain_c(tmp_path):
    """The boundary is a C ABI: the header must be valid C (no C++/CUDA types)."""
    import subprocess
    src = tmp_path / "t.c"
    src.write_text('#include "qmmm_field.h"\nint main(void){qmmm_plan p={0,0,0,0};return p.slices;}\n')
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"),
                    "-c", str(src), "-o", str(tmp_path / "t.o")], check=True)


def test_argument_errors_without_gpu(lib_path):
    """Argument validation happens before any CUDA call: safe on a CPU box."""
    from paper_1011_4687_b200 import binding
    lib = binding._lib
    out = ctypes.c_void_p()
    assert lib.qmmm_field_create(None, None, -1, None, None, 0, 8, ctypes.byref(out)) == 1
    assert b"negative" in lib.qmmm_last_error()
    assert lib.qmmm_field_create(None, None, 4, None, None, 0, 8, ctypes.byref(out)) == 1
    assert lib.qmmm_field_create(None, None, 0, None, None, 0, 0, ctypes.byref(out)) == 1
    assert lib.qmmm_field_create(None, None, 0, None, None, 0, 8, None) == 1
    assert lib.qmmm_field_eval(None, None, 1, 1, None, None, 0, None) == 1
    assert lib.qmmm_field_destroy(None) == 0


def test_grid_argument_errors_without_gpu(lib_path):
    """qmmm_field_create_grid / set_layout validate their arguments before any CUDA call."""
    from paper_1011_4687_b200 import binding
    lib = binding._lib
    out = ctypes.c_void_p()
    org = (ctypes.c_double * 3)(0.0, 0.0, 0.0)
    n = (ctypes.c_int64 * 3)(4, 4, 4)
    q = (ctypes.c_double * 64)()
    qp = ctypes.cast(q, ctypes.c_void_p)
    assert lib.qmmm_field_create_grid(None, 0.3, n, qp, None, None, 0, 8, ctypes.byref(out)) == 1
    assert lib.qmmm_field_create_grid(org, 0.0, n, qp, None, None, 0, 8, ctypes.byref(out)) == 1
    assert b"spacing" in lib.qmmm_last_error()
    assert lib.qmmm_field_create_grid(org, float("nan"), n, qp, None, None, 0, 8, ctypes.byref(out)) == 1
    bad = (ctypes.c_int64 * 3)(4, 0, 4)
    assert lib.qmmm_field_create_grid(org, 0.3, bad, qp, None, None, 0, 8, ctypes.byref(out)) == 1
    huge = (ctypes.c_int64 * 3)(65536, 65536, 2)
    assert lib.qmmm_field_create_grid(org, 0.3, huge, qp, None, None, 0, 8, ctypes.byref(out)) == 1
    assert lib.qmmm_field_create_grid(org, 0.3, n, None, None, None, 0, 8, ctypes.byref(out)) == 1
    assert lib.qmmm_field_create_grid(org, 0.3, n, qp, None, None, 2, 8, ctypes.byref(out)) == 1   # K > 0, NULL nuclei
    assert lib.qmmm_field_create_grid(org, 0.3, n, qp, None, None, 0, 0, ctypes.byref(out)) == 1   # max_points < 1
    assert lib.qmmm_field_create_grid(org, 0.3, n, qp, None, None, 0, 8, None) == 1
    assert out.value is None
    assert lib.qmmm_field_set_layout(None, 0) == 1
    assert lib.qmmm_field_share(None, 8, ctypes.byref(out)) == 1
    assert lib.qmmm_field_eval_energy(None, None, 1, 1, None, 0, None) == 1
    assert lib.qmmm_field_get_grid_info(None, None) == 1
