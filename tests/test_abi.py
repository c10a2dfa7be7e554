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


def test_plan_argument_validation_without_gpu():
    """fdemri_plan / fdemri_plan_kerr reject bad arguments before touching the device (host logic only)."""
    import numpy as np
    L = binding.lib()
    h = ctypes.c_void_p()
    ip = ctypes.POINTER(ctypes.c_int32)
    fake = ctypes.c_void_p(256)                          # a non-NULL "device pointer": never dereferenced on these paths

    def plan(fn, modes, n_batch=1, n_knots=10, n_freq=1000, df=1e-6, flags=0, t=fake):
        a = np.ascontiguousarray(modes, dtype=np.int32)
        return fn(ctypes.byref(h), a.shape[0], a.ctypes.data_as(ip), n_batch, n_knots, t, n_freq, None, 0.0, df, flags)

    INVALID = 1
    for fn, good, bads in (
            (L.fdemri_plan, [(2, 2, 0)], [[(1, 0, 0)], [(2, 3, 0)], [(2, -1, 0)], [(2, 2, 200000)], [(61, 0, 0)]]),
            (L.fdemri_plan_kerr, [(2, 2, 1, 0)], [[(1, 0, 0, 0)], [(2, 3, 0, 0)], [(2, -1, 0, 0)], [(2, 2, 200000, 0)],
                                                  [(2, 2, 0, 200000)]])):
        for bad in bads:
            assert plan(fn, bad) == INVALID and not h.value, bad
        assert plan(fn, good, n_knots=3) == INVALID            # fewer than 4 knots: no not-a-knot spline
        assert plan(fn, good, n_knots=513) == INVALID
        assert plan(fn, good, n_freq=0) == INVALID
        assert plan(fn, good, df=0.0) == INVALID               # uniform grid needs df > 0
        assert plan(fn, good, t=None) == INVALID
        assert plan(fn, good, flags=2 | 4) == INVALID          # bin-major and tile-major at once
    assert L.fdemri_plan_kerr(None, 1, None, 1, 10, fake, 1000, None, 0.0, 1e-6, 0) == INVALID
    assert L.fdemri_build_splines_kerr(None, fake, fake, fake, fake, fake, fake, fake, None) == INVALID
    assert L.fdemri_build_splines(None, fake, fake, fake, fake, fake, None) == INVALID


def test_select_modes_static_validates_before_touching_the_device():
    """fdemri_select_modes_static (the entry point that allocates nothing): bad arguments and sizes beyond its static
    scratch are refused on the host, before any CUDA call."""
    L = binding.lib()
    fake = ctypes.c_void_p(256)
    INVALID, STATIC_SCRATCH = 1, 6
    assert L.fdemri_select_modes_static(0, 4, 10, fake, 0.1, fake, fake, None) == INVALID
    assert L.fdemri_select_modes_static(1, 4, 10, None, 0.1, fake, fake, None) == INVALID
    assert L.fdemri_select_modes_static(1, 4, 10, fake, -1.0, fake, fake, None) == INVALID
    assert L.fdemri_select_modes_static(1, 4, 10, fake, float("nan"), fake, fake, None) == INVALID
    lim = binding.FDEMRI_STATIC_MAX_TOTALS
    assert L.fdemri_select_modes_static(lim // 100 + 1, 4, 100, fake, 0.1, fake, fake, None) == STATIC_SCRATCH
    assert L.fdemri_select_modes_static(1 << 20, 4, 1 << 20, fake, 0.1, fake, fake, None) == STATIC_SCRATCH
    assert b"static scratch" in L.fdemri_strerror(STATIC_SCRATCH)
    assert binding.STATUS[STATIC_SCRATCH] == "FDEMRI_ERR_STATIC_SCRATCH"
