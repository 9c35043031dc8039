"""CPU-side checks of the C-ABI boundary: the library builds for sm_100a, loads, and exports every symbol
include/wave2d.h declares; the binding's export list, the header and the library agree; and the product
path has no route into oracle/ and no CPU fallback.  No compute call is made here (no GPU).
"""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PKG = os.path.join(ROOT, "paper_2006_10142_b200")


def _header_functions():
    src = open(os.path.join(ROOT, "include", "wave2d.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(wave2d_[a-z_0-9]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_2006_10142_b200 import build
    return build.build()


def test_header_declares_the_north_star_calls():
    names = _header_functions()
    for need in ("wave2d_create", "wave2d_set_initial", "wave2d_set_speed", "wave2d_set_source", "wave2d_run",
                 "wave2d_get", "wave2d_destroy"):
        assert need in names


def test_library_exports_every_declared_symbol(lib_path):
    L = ctypes.CDLL(lib_path)
    missing = [n for n in _header_functions() if not hasattr(L, n)]
    assert not missing, missing


def test_binding_export_list_matches_header():
    from paper_2006_10142_b200 import binding
    assert sorted(binding.EXPORTS) == _header_functions()


def test_status_strings_without_a_device(lib_path):
    L = ctypes.CDLL(lib_path)
    L.wave2d_strerror.restype = ctypes.c_char_p
    L.wave2d_strerror.argtypes = [ctypes.c_int]
    seen = {L.wave2d_strerror(s) for s in range(0, -7, -1)}
    assert len(seen) == 7 and b"ok" in seen
    assert L.wave2d_strerror(-99) == b"unknown status"
    L.wave2d_destroy.argtypes = [ctypes.c_void_p]
    L.wave2d_destroy(None)   # NULL-safe


def test_create_fails_loudly_without_gpu(lib_path):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2006_10142_b200 import Wave2D, Wave2DError
    with pytest.raises(Wave2DError) as e:
        Wave2D(16, 16, 1.0, 0.01, 4)
    assert e.value.status == -4   # WAVE2D_ERR_CUDA: no device, no other code path


def test_product_path_never_touches_the_oracle_or_work_dir():
    bad = []
    files = [os.path.join(ROOT, "bench.py")]
    for d, _, fs in os.walk(PKG):
        files += [os.path.join(d, f) for f in fs if f.endswith((".py", ".cu", ".cuh", ".h"))]
    for p in files:
        if not os.path.exists(p):
            continue
        txt = open(p).read()
        if re.search(r"_work[/\\\"']", txt):
            bad.append((p, "_work"))
        if p.startswith(PKG) and re.search(r"^\s*(from|import)\s+oracle|oracle/|liboracle", txt, flags=re.M):
            bad.append((p, "oracle"))
    assert not bad, bad


def test_sass_has_tma_and_no_legacy_tensor_path(lib_path):
    """The sweep kernels move tiles with TMA (UTMALDG / UTMASTG in SASS, B200_PROFILING.md)."""
    import shutil
    import subprocess
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    sass = subprocess.run([cuobjdump, "-sass", lib_path], capture_output=True, text=True).stdout
    assert "sm_100a" in sass
    assert "UTMALDG" in sass and "UTMASTG" in sass
    assert "HMMA" not in sass
