"""CPU-side checks of the C-ABI boundary: the library builds for sm_100a with nvcc (no GPU needed),
loads, and exports every symbol include/dwf.h declares.  No compute calls here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2203_17119_b200 import build
    return build.build()


def header_symbols():
    txt = open(os.path.join(ROOT, "include", "dwf.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(dwf_[a-z0-9_]+)\s*\(", txt)))


def test_header_declares_the_north_star_entry_points():
    syms = header_symbols()
    for name in ("dwf_create", "dwf_dhop", "dwf_mooee_inv", "dwf_mpc", "dwf_mdagm", "dwf_cg"):
        assert name in syms


def test_library_exports_every_declared_symbol(libpath):
    lib = ctypes.CDLL(libpath)
    for name in header_symbols():
        assert hasattr(lib, name), name


def test_binding_lists_the_same_symbols(libpath):
    from paper_2203_17119_b200 import api
    assert sorted(api.SYMBOLS) == header_symbols()
    lib = api.load_library()
    assert lib.dwf_version().decode().startswith("dwf_b200")


def test_binding_has_no_torch_types_in_the_abi():
    txt = open(os.path.join(ROOT, "include", "dwf.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)     # declarations only
    assert "torch" not in txt.lower()
    assert "at::" not in txt and "#include <cuda" not in txt


def test_product_path_never_touches_the_oracle():
    pkg = os.path.join(ROOT, "paper_2203_17119_b200")
    for dp, _, fns in os.walk(pkg):
        if "build" in os.path.relpath(dp, pkg).split(os.sep)[:1] and dp != pkg:
            continue
        for fn in fns:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dp, fn)).read()
                assert "import oracle" not in src and "from oracle" not in src and "dwf_oracle" not in src, fn


def test_cuda_required_and_loud(libpath):
    import torch
    from paper_2203_17119_b200 import api
    if torch.cuda.is_available():
        pytest.skip("GPU box: covered by the gpu tests")
    with pytest.raises(RuntimeError):
        api.Dwf((4, 4, 4, 4), 4, 1.8, 0.1, 1.0, 0.0)


def test_create_rejects_bad_arguments_without_touching_cuda(libpath):
    """Error behaviour stated in include/dwf.h: integer status, never abort; argument validation precedes every CUDA call,
    so these run on the CPU-only box."""
    from paper_2203_17119_b200 import api
    lib = api.load_library()

    def create(dims, Ls, cut=(0, 0, 0, 0), M5=1.8, b5=1.5):
        h = ctypes.c_void_p()
        st = lib.dwf_create(ctypes.byref(h), (ctypes.c_int * 4)(*dims), Ls, M5, 0.01, b5, 0.5, (ctypes.c_int * 4)(*cut))
        assert st != api.OK and not h.value
        return st

    assert create((4, 4, 4, 5), 8) == api.EINVAL            # odd extent
    assert create((4, 4, 4, 0), 8) == api.EINVAL
    assert create((4, 4, 4, 4), 0) == api.EINVAL            # Ls < 1
    assert create((4, 4, 4, 4), 33) == api.EINVAL           # Ls beyond the table size
    assert create((4, 4, 4, 8), 8, cut=(0, 0, 0, 3)) == api.EINVAL    # cut does not divide Lt
    assert create((4, 4, 4, 8), 8, cut=(0, 0, 0, -4)) == api.EINVAL
    assert create((4, 4, 4, 4), 8, M5=5.0, b5=1.0) == api.EINVAL      # bee = 1 + b5 (4 - M5) = 0: Mee singular
    assert create((256, 256, 256, 256), 16) == api.EINVAL             # beyond the 32-bit vector index range
    assert lib.dwf_create(None, None, 8, 1.8, 0.01, 1.5, 0.5, None) == api.EINVAL
    assert lib.dwf_destroy(None) == api.EINVAL
    assert lib.dwf_launch_count(None) == 0
    lib.dwf_last_error.restype = ctypes.c_char_p
    assert lib.dwf_last_error(None) == b"null context"
