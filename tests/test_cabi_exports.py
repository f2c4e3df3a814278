"""The C-ABI library builds for sm_100a, loads without a GPU and exports every symbol that
include/rts.h declares (no compute calls here)."""
import ctypes
import os
import re

from paper_2107_08145_b200 import build as rts_build
from paper_2107_08145_b200 import rts

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    with open(os.path.join(ROOT, "include", "rts.h")) as fh:
        text = fh.read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rts_[a-z_0-9]+)\s*\(", text)))


def test_header_declares_the_boundary_of_the_north_star():
    names = _declared_symbols()
    for must in ("rts_create", "rts_set_tables", "rts_solve", "rts_destroy"):
        assert must in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    lib_path = rts_build.build()
    assert os.path.exists(lib_path)
    lib = ctypes.CDLL(lib_path)
    for name in _declared_symbols():
        assert hasattr(lib, name), f"{name} declared in include/rts.h but not exported"


def test_python_binding_names_match_the_header():
    assert sorted(rts.EXPORTS) == _declared_symbols()
    lib = rts.load_library()
    for name in rts.EXPORTS:
        assert getattr(lib, name).argtypes is not None


def test_create_fails_loudly_without_a_device():
    import torch
    if torch.cuda.is_available():
        return
    lib = rts.load_library()
    ctx = ctypes.c_void_p()
    rc = lib.rts_create(ctypes.byref(ctx), 8, 8, 8, 1e5, 1e5, 1e5, 1)
    assert rc == -3 and not ctx.value                     # RTS_ECUDA, no context: no CPU fallback
    assert b"CUDA" in lib.rts_last_error(None) or b"device" in lib.rts_last_error(None)
    try:
        rts.RTS(8, 8, 8, 1e5, 1e5, 1e5, 1)
    except rts.RTSError:
        pass
    else:
        raise AssertionError("RTS() must raise without a CUDA device")


def test_product_path_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2107_08145_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                with open(os.path.join(dirpath, f)) as fh:
                    src = fh.read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
                assert "rts_oracle" not in src, f
