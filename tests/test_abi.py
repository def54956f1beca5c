"""The C-ABI library builds, loads without a GPU and exports every symbol include/comet.h declares."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_1911_09340_b200.build import build
    return build()


def _declared():
    hdr = open(os.path.join(ROOT, "include", "comet.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    return sorted(set(re.findall(r"\b(comet_[a-z0-9_]+)\s*\(", hdr)))


def test_every_declared_symbol_is_exported(libpath):
    L = ctypes.CDLL(libpath)
    names = _declared()
    assert {"comet_seed_extrapolate", "comet_dca_rss", "comet_select_and_classify"} <= set(names)
    for n in names:
        assert hasattr(L, n), n


def test_binding_lists_the_same_symbols(libpath):
    from paper_1911_09340_b200 import binding
    assert sorted(binding.EXPORTED_SYMBOLS) == _declared()
    binding.load_library()


def test_host_only_entry_points(libpath):
    L = ctypes.CDLL(libpath)
    L.comet_status_string.restype = ctypes.c_char_p
    assert L.comet_status_string(0) == b"ok"
    assert L.comet_status_string(-1) == b"invalid argument"
    L.comet_track_bytes.restype = ctypes.c_size_t
    L.comet_track_bytes.argtypes = [ctypes.c_int64, ctypes.c_int32]
    # two planes x ceil(S/32) chunks x (n_steps+1 rounded up to 64) rows x 3 components x 32 lanes x 8 bytes
    assert L.comet_track_bytes(8192, 400) == 2 * 256 * 448 * 3 * 32 * 8
    assert L.comet_track_bytes(33, 10) == 2 * 2 * 64 * 3 * 32 * 8
    assert L.comet_track_bytes(33, 63) == 2 * 2 * 64 * 3 * 32 * 8
    assert L.comet_track_bytes(33, 64) == 2 * 2 * 128 * 3 * 32 * 8
    assert L.comet_track_bytes(0, 10) == 0
    assert L.comet_track_bytes(10, 0) == 0 and L.comet_track_bytes(-1, 10) == 0
    # argument errors are reported before any CUDA call
    assert L.comet_create(None, 0) == -1
    assert L.comet_destroy(None) == -1
    # comet_argmin_static: more partitions than its static scratch holds is refused with a status of its own, and
    # negative sizes as invalid arguments -- both before any CUDA call
    L.comet_argmin_static.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int32, ctypes.c_void_p,
                                      ctypes.c_void_p, ctypes.c_void_p]
    assert L.comet_argmin_static(None, 0, None, 65, None, None, None) == -4
    assert b"statically allocated scratch" in L.comet_status_string(-4)
    assert L.comet_argmin_static(None, -1, None, 1, None, None, None) == -1
    assert L.comet_argmin_static(None, 0, None, 0, None, None, None) == 0


def test_no_gpu_means_loud_failure(libpath):
    """The product path has no CPU fallback."""
    import torch
    from paper_1911_09340_b200 import Comet, CometError
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(CometError):
        Comet(0)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1911_09340_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"oracle", src, flags=re.I), f
