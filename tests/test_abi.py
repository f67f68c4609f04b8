"""The C-ABI boundary without a GPU: libsph_b200.so builds for sm_100a, loads, and exports every
entry point include/sph.h declares (and the Python binding wraps exactly those).  No compute call is
made here; the product path has no CPU fallback and must say so loudly."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "sph.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sph_[a-z_]+)\s*\(", text)))


@pytest.fixture(scope="module")
def lib():
    from paper_2310_03596_b200 import build
    return C.CDLL(build.build())


def test_header_declares_the_seven_stage_calls():
    names = _declared()
    for want in ("sph_hash", "sph_sort", "sph_cell_ranges", "sph_comm_hash", "sph_interact",
                 "sph_integrate", "sph_step"):        # BASELINE.json north_star's list
        assert want in names


def test_library_exports_every_declared_symbol(lib):
    for name in _declared():
        assert getattr(lib, name) is not None, name


def test_binding_wraps_exactly_the_declared_symbols():
    from paper_2310_03596_b200 import sph
    assert sorted(sph.EXPORTS) == _declared()
    for name in ("sph_hash", "sph_sort", "sph_reorder", "sph_cell_ranges", "sph_comm_hash", "sph_interact",
                 "sph_integrate", "sph_step", "sph_step_host"):
        assert callable(getattr(sph, name))


def test_strerror_and_null_arguments(lib):
    lib.sph_strerror.restype = C.c_char_p
    assert lib.sph_strerror(0) and lib.sph_strerror(-1) and lib.sph_strerror(-2)
    # a NULL ctx / params is an argument error, never a crash
    lib.sph_create.restype = C.c_int
    assert lib.sph_create(None, None, C.c_int64(0), None) == -1
    lib.sph_destroy.restype = C.c_int
    assert lib.sph_destroy(None) in (0, -1)


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2310_03596_b200 import sph
    with pytest.raises(Exception):
        sph.Context(origin=(0.0, 0.0, 0.0), dims=(2, 2, 2), h=1.0)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2310_03596_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "sph_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            for line in open(os.path.join(ROOT, "oracle", f)):
                code = line.split("#")[0]
                assert not re.search(r"^\s*(import|from)\s+paper_2310_03596_b200", code), (f, line)
                assert not re.search(r'#include\s+"(sph\.h|.*csrc)', line), (f, line)


def test_create_refuses_dims_whose_coordinates_are_not_exact_in_fp32(lib):
    """dims[a] > 2^24: clamp(floorf(u), 0, n - 1) is no longer the same in fp32 and in integers
    (the argument checks come before any CUDA call, so this runs without a GPU)."""
    from paper_2310_03596_b200 import sph
    p = sph._Params()
    p.h, p.K, p.G, p.n_owners = 1.0, 1.0, 0.5, 1
    p.dims[0], p.dims[1], p.dims[2] = (1 << 24) + 1, 1, 1
    h = C.c_void_p()
    lib.sph_create.restype = C.c_int
    assert lib.sph_create(C.byref(h), C.byref(p), C.c_int64(4), None) == sph.SPH_EINVAL
