"""The C-ABI library loads and exports every symbol include/fdemri.h declares (no compute calls: no GPU here)."""
import ctypes
import os
import re

from paper_2307_12585_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "fdemri.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(fdemri_[a-z0-9_]+)\s*\(", src)))


def test_library_builds_and_exports_all_declared_symbols():
    path = build.build()
    L = ctypes.CDLL(path)
    names = declared_symbols()
    assert set(names) == set(binding.EXPORTS)
    for n in names:
        assert hasattr(L, n), n


def test_strerror_and_version_without_gpu():
    L = binding.lib()
    assert L.fdemri_strerror(0) == b"ok"
    assert b"sm_100a" in L.fdemri_version()
    # argument validation that needs no device
    assert L.fdemri_workspace_bytes(None) == 0
    assert L.fdemri_destroy(None) == 1


def test_sass_is_sm100a_fp64():
    """The shipped cubin is sm_100a and the hot kernel is FP64 (DFMA), not a PTX-JIT fallback."""
    import shutil
    import subprocess
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    out = subprocess.run([cuobjdump, "-lelf", build.build()], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    sass = subprocess.run([cuobjdump, "-sass", build.build()], capture_output=True, text=True).stdout
    body = sass.split("Function : _Z10k_tile_sum7SumArgs")[1].split("Function : ")[0]
    assert body.count("DFMA") > 50
