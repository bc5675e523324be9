"""CPU-only checks of the C-ABI boundary: libhprmat.so builds/loads, exports every symbol include/hprmat.h declares,
validates arguments, and refuses to compute without a CUDA device (there is no CPU fallback)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "hprmat.h")
PROFILE_HEADER = os.path.join(ROOT, "include", "hprmat_profile.h")


@pytest.fixture(scope="module")
def lib():
    from paper_2512_11590_b200 import build
    path = build.build()
    return C.CDLL(path)


def _declared_functions(header=HEADER):
    src = open(header).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(hprmat_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_boundary_calls():
    names = _declared_functions()
    for must in ["hprmat_setup", "hprmat_mesh", "hprmat_solve", "hprmat_solve_host", "hprmat_get_x", "hprmat_get_matrix",
                 "hprmat_destroy", "hprmat_zsolve", "hprmat_zgetrf", "hprmat_zgetrs", "hprmat_zgemm",
                 "hprmat_workspace_bytes", "hprmat_strerror"]:
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    missing = [n for n in _declared_functions() if not hasattr(lib, n)]
    assert not missing, f"declared in hprmat.h but not exported: {missing}"


def test_measurement_aids_live_outside_the_product_interface(lib):
    """include/hprmat_profile.h: the timing record and the launch counter are exported by libhprmat.so, the FP64 peak probe
    only by libhprmat_bench.so; hprmat.h declares none of them."""
    product = set(_declared_functions())
    aids = _declared_functions(PROFILE_HEADER)
    assert aids and not (product & set(aids))
    from paper_2512_11590_b200 import build
    bench = C.CDLL(build.BENCH_LIB)
    for n in aids:
        if n.startswith("hprmat_bench_"):
            assert hasattr(bench, n) and not hasattr(lib, n), n
        else:
            assert hasattr(lib, n), n


def test_strerror_and_argument_validation(lib):
    lib.hprmat_strerror.restype = C.c_char_p
    assert b"singular" in lib.hprmat_strerror(1)
    assert b"converge" in lib.hprmat_strerror(2)
    assert b"invalid" in lib.hprmat_strerror(-3)
    h = C.c_void_p()
    lv = np.zeros(2, dtype=np.int32)
    et = np.zeros(2)
    args = lambda nch, nb, a, h2m: (C.byref(h), C.c_int(nch), C.c_int(nb), C.c_double(a), C.c_double(h2m),
                                   lv.ctypes.data_as(C.c_void_p), et.ctypes.data_as(C.c_void_p), C.c_int(0), None)
    assert lib.hprmat_setup(*args(0, 10, 1.0, 1.0)) == -2
    assert lib.hprmat_setup(*args(2, 1, 1.0, 1.0)) == -3
    assert lib.hprmat_setup(*args(2, 10, -1.0, 1.0)) == -4
    assert lib.hprmat_setup(*args(2, 10, 1.0, 0.0)) == -5
    assert lib.hprmat_zgemm(None, C.c_int(-1), C.c_int(1), C.c_int(1), C.c_double(1), None, C.c_int(1), None, C.c_int(1),
                            C.c_double(0), None, C.c_int(1)) == -2
    lib.hprmat_workspace_bytes.restype = C.c_size_t
    assert lib.hprmat_workspace_bytes(C.c_int(1000), C.c_int(4), C.c_int(1)) > 0


def test_no_cpu_fallback(lib):
    """Without a CUDA device the compute entries must fail loudly with HPRMAT_ECUDA, never compute on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    h = C.c_void_p()
    lv = np.zeros(2, dtype=np.int32)
    et = np.zeros(2)
    rc = lib.hprmat_setup(C.byref(h), C.c_int(2), C.c_int(10), C.c_double(5.0), C.c_double(20.0),
                          lv.ctypes.data_as(C.c_void_p), et.ctypes.data_as(C.c_void_p), C.c_int(0), None)
    assert rc == 4
    lib.hprmat_last_cuda_error.restype = C.c_char_p
    assert b"no CUDA device" in lib.hprmat_last_cuda_error()


def test_product_does_not_import_the_oracle():
    """The CUDA path and its binding share no code with oracle/ (only workloads.py, which holds no arithmetic)."""
    pkg = os.path.join(ROOT, "paper_2512_11590_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "hprmat_oracle" not in txt, f
