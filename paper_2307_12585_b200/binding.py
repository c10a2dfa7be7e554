"""Thin ctypes binding of libfdemri.so (include/fdemri.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; PyTorch is used for device memory and
streams.  There is no CPU fallback: if the shared library is missing and cannot be built, importing the
functions raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))

FDEMRI_OK = 0
FDEMRI_FLAG_TIMING, FDEMRI_FLAG_BIN_MAJOR, FDEMRI_FLAG_TILE_MAJOR = 1, 2, 4
STATUS = {0: "FDEMRI_OK", 1: "FDEMRI_ERR_INVALID_ARG", 2: "FDEMRI_ERR_WORKSPACE", 3: "FDEMRI_ERR_CUDA",
          4: "FDEMRI_ERR_NOT_BUILT", 5: "FDEMRI_ERR_UNSUPPORTED", 6: "FDEMRI_ERR_STATIC_SCRATCH"}
FDEMRI_STATIC_MAX_TOTALS = 32768

EXPORTS = ["fdemri_plan", "fdemri_plan_kerr", "fdemri_build_splines_kerr", "fdemri_workspace_bytes", "fdemri_workspace_bytes_min", "fdemri_set_workspace", "fdemri_build_splines", "fdemri_sum", "fdemri_td_sum", "fdemri_sum_inner", "fdemri_select_modes", "fdemri_select_modes_rule", "fdemri_select_modes_static", "fdemri_set_mode_mask",
           "fdemri_get_stats", "fdemri_get_item_evals", "fdemri_get_coeffs", "fdemri_get_kernel_ms", "fdemri_measure_fp64_peak", "fdemri_measure_fp64_peak_3reg", "fdemri_measure_issue_ns", "fdemri_destroy", "fdemri_strerror", "fdemri_version"]


class FdemriStats(C.Structure):
    _fields_ = [("n_items", C.c_uint64), ("reserved", C.c_uint64), ("n_evals", C.c_uint64),
                ("n_turnover", C.c_uint64), ("n_airy", C.c_uint64), ("flags", C.c_uint64), ("n_slow", C.c_uint64), ("n_pairs", C.c_uint64)]


class FdemriError(RuntimeError):
    def __init__(self, fn, status):
        super().__init__(f"{fn} -> {STATUS.get(status, status)}")
        self.status = status


_LIB = None


def lib() -> C.CDLL:
    """Loads (building first if stale) paper_2307_12585_b200/libfdemri.so.  Raises if it cannot."""
    global _LIB
    if _LIB is None:
        path = _build.LIB
        if _build.is_stale():
            path = _build.build()
        L = C.CDLL(path)
        vp, dp, ip = C.c_void_p, C.c_void_p, C.POINTER(C.c_int32)
        L.fdemri_plan.restype = C.c_int
        L.fdemri_plan.argtypes = [C.POINTER(vp), C.c_int, ip, C.c_int, C.c_int, dp, C.c_int64, dp, C.c_double,
                                  C.c_double, C.c_uint32]
        L.fdemri_workspace_bytes.restype = C.c_size_t
        L.fdemri_workspace_bytes.argtypes = [vp]
        L.fdemri_workspace_bytes_min.restype = C.c_size_t
        L.fdemri_workspace_bytes_min.argtypes = [vp]
        L.fdemri_set_workspace.restype = C.c_int
        L.fdemri_set_workspace.argtypes = [vp, vp, C.c_size_t]
        L.fdemri_build_splines.restype = C.c_int
        L.fdemri_build_splines.argtypes = [vp, dp, dp, dp, dp, dp, vp]
        L.fdemri_plan_kerr.restype = C.c_int
        L.fdemri_plan_kerr.argtypes = L.fdemri_plan.argtypes
        L.fdemri_build_splines_kerr.restype = C.c_int
        L.fdemri_build_splines_kerr.argtypes = [vp, dp, dp, dp, dp, dp, dp, dp, vp]
        L.fdemri_sum.restype = C.c_int
        L.fdemri_sum.argtypes = [vp, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double), dp, dp, vp]
        L.fdemri_td_sum.restype = C.c_int
        L.fdemri_td_sum.argtypes = [vp, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_int64, C.c_double, C.c_double,
                                    dp, dp, vp]
        L.fdemri_sum_inner.restype = C.c_int
        L.fdemri_sum_inner.argtypes = [vp, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double), dp, dp, dp, C.c_int, dp, dp, dp,
                                       vp]
        L.fdemri_select_modes.restype = C.c_int
        L.fdemri_select_modes.argtypes = [vp, dp, C.c_double, vp, vp, vp]
        L.fdemri_select_modes_rule.restype = C.c_int
        L.fdemri_select_modes_rule.argtypes = [vp, dp, C.c_double, C.c_int, vp, vp, vp]
        L.fdemri_select_modes_static.restype = C.c_int
        L.fdemri_select_modes_static.argtypes = [C.c_int, C.c_int, C.c_int, dp, C.c_double, vp, vp, vp]
        L.fdemri_set_mode_mask.restype = C.c_int
        L.fdemri_set_mode_mask.argtypes = [vp, vp]
        L.fdemri_get_stats.restype = C.c_int
        L.fdemri_get_stats.argtypes = [vp, C.POINTER(FdemriStats)]
        L.fdemri_get_item_evals.restype = C.c_int
        L.fdemri_get_item_evals.argtypes = [vp, C.POINTER(C.c_uint64)]
        L.fdemri_get_coeffs.restype = C.c_int
        L.fdemri_get_coeffs.argtypes = [vp, dp, dp, dp]
        L.fdemri_get_kernel_ms.restype = C.c_int
        L.fdemri_get_kernel_ms.argtypes = [vp, C.POINTER(C.c_float)]
        L.fdemri_measure_fp64_peak.restype = C.c_int
        L.fdemri_measure_fp64_peak.argtypes = [C.c_int, C.POINTER(C.c_double)]
        L.fdemri_measure_fp64_peak_3reg.restype = C.c_int
        L.fdemri_measure_fp64_peak_3reg.argtypes = [C.c_int, C.POINTER(C.c_double)]
        L.fdemri_measure_issue_ns.restype = C.c_int
        L.fdemri_measure_issue_ns.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_double)]
        L.fdemri_destroy.restype = C.c_int
        L.fdemri_destroy.argtypes = [vp]
        L.fdemri_strerror.restype = C.c_char_p
        L.fdemri_strerror.argtypes = [C.c_int]
        L.fdemri_version.restype = C.c_char_p
        _LIB = L
    return _LIB


def _chk(fn, rc):
    if rc != FDEMRI_OK:
        raise FdemriError(fn, rc)


def _ptr(t):
    """Device pointer of a contiguous float64 CUDA tensor (or None)."""
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous() and t.dtype.is_floating_point and t.element_size() == 8, \
        "expected a contiguous float64 CUDA tensor"
    return C.c_void_p(t.data_ptr())


def _stream_ptr(stream):
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


# ---- the C calls, same names ---------------------------------------------------------------------------
def fdemri_plan(lmn, n_batch, n_knots, t_knots, n_freq, freq=None, f0=0.0, df=0.0, flags=0):
    lmn = np.ascontiguousarray(lmn, dtype=np.int32)
    assert lmn.ndim == 2 and lmn.shape[1] == 3
    assert tuple(t_knots.shape) == (n_batch, n_knots)
    h = C.c_void_p()
    rc = lib().fdemri_plan(C.byref(h), lmn.shape[0], lmn.ctypes.data_as(C.POINTER(C.c_int32)), n_batch, n_knots,
                           _ptr(t_knots), int(n_freq), _ptr(freq), float(f0), float(df), int(flags))
    _chk("fdemri_plan", rc)
    return h


def fdemri_plan_kerr(lmkn, n_batch, n_knots, t_knots, n_freq, freq=None, f0=0.0, df=0.0, flags=0):
    lmkn = np.ascontiguousarray(lmkn, dtype=np.int32)
    assert lmkn.ndim == 2 and lmkn.shape[1] == 4
    assert tuple(t_knots.shape) == (n_batch, n_knots)
    h = C.c_void_p()
    rc = lib().fdemri_plan_kerr(C.byref(h), lmkn.shape[0], lmkn.ctypes.data_as(C.POINTER(C.c_int32)), n_batch, n_knots,
                                _ptr(t_knots), int(n_freq), _ptr(freq), float(f0), float(df), int(flags))
    _chk("fdemri_plan_kerr", rc)
    return h


def fdemri_workspace_bytes(plan) -> int:
    return int(lib().fdemri_workspace_bytes(plan))


def fdemri_workspace_bytes_min(plan) -> int:
    return int(lib().fdemri_workspace_bytes_min(plan))


def fdemri_set_workspace(plan, ws):
    _chk("fdemri_set_workspace", lib().fdemri_set_workspace(plan, C.c_void_p(ws.data_ptr()), ws.numel() * ws.element_size()))


def fdemri_build_splines(plan, f_phi, f_r, Phi_phi, Phi_r, amp, stream=None):
    _chk("fdemri_build_splines", lib().fdemri_build_splines(plan, _ptr(f_phi), _ptr(f_r), _ptr(Phi_phi), _ptr(Phi_r),
                                                            _ptr(amp), _stream_ptr(stream)))


def fdemri_sum(plan, theta, phi, hplus, hcross, stream=None):
    th = np.atleast_1d(np.asarray(theta, dtype=np.float64))
    ph = np.atleast_1d(np.asarray(phi, dtype=np.float64))
    assert th.shape == ph.shape
    dp = C.POINTER(C.c_double)
    _chk("fdemri_sum", lib().fdemri_sum(plan, th.shape[0], th.ctypes.data_as(dp), ph.ctypes.data_as(dp), _ptr(hplus),
                                        _ptr(hcross), _stream_ptr(stream)))


def fdemri_td_sum(plan, theta, phi, n_samples, t0, dt, hplus_td, hcross_td, stream=None):
    """hplus_td, hcross_td: float64 CUDA tensors [n_batch][n_samples]."""
    th = np.atleast_1d(np.asarray(theta, dtype=np.float64))
    ph = np.atleast_1d(np.asarray(phi, dtype=np.float64))
    assert th.shape == ph.shape
    dp = C.POINTER(C.c_double)
    _chk("fdemri_td_sum", lib().fdemri_td_sum(plan, th.shape[0], th.ctypes.data_as(dp), ph.ctypes.data_as(dp), int(n_samples),
                                              float(t0), float(dt), _ptr(hplus_td), _ptr(hcross_td), _stream_ptr(stream)))


def fdemri_sum_inner(plan, theta, phi, inner_out, weight=None, data_plus=None, data_cross=None, hann=False, hplus=None,
                     hcross=None, stream=None):
    th = np.atleast_1d(np.asarray(theta, dtype=np.float64))
    ph = np.atleast_1d(np.asarray(phi, dtype=np.float64))
    assert th.shape == ph.shape
    dp = C.POINTER(C.c_double)
    _chk("fdemri_sum_inner", lib().fdemri_sum_inner(plan, th.shape[0], th.ctypes.data_as(dp), ph.ctypes.data_as(dp),
                                                    _ptr(weight), _ptr(data_plus), _ptr(data_cross), int(bool(hann)),
                                                    _ptr(hplus), _ptr(hcross), _ptr(inner_out), _stream_ptr(stream)))


def fdemri_select_modes(plan, amp, eps, keep, n_keep, stream=None):
    """keep: uint8 CUDA tensor [n_batch][n_modes]; n_keep: int32 CUDA tensor [n_batch]."""
    assert keep.is_cuda and keep.is_contiguous() and keep.element_size() == 1
    assert n_keep.is_cuda and n_keep.is_contiguous() and n_keep.element_size() == 4
    _chk("fdemri_select_modes", lib().fdemri_select_modes(plan, _ptr(amp), float(eps), C.c_void_p(keep.data_ptr()),
                                                          C.c_void_p(n_keep.data_ptr()), _stream_ptr(stream)))


FDEMRI_SELECT_OWN_POWER, FDEMRI_SELECT_CUMULATIVE = 0, 1


def fdemri_select_modes_rule(plan, amp, eps, rule, keep, n_keep, stream=None):
    """As fdemri_select_modes with the reading of L60 chosen by `rule` (FDEMRI_SELECT_OWN_POWER / _CUMULATIVE)."""
    assert keep.is_cuda and keep.is_contiguous() and keep.element_size() == 1
    assert n_keep.is_cuda and n_keep.is_contiguous() and n_keep.element_size() == 4
    _chk("fdemri_select_modes_rule", lib().fdemri_select_modes_rule(plan, _ptr(amp), float(eps), int(rule), C.c_void_p(keep.data_ptr()),
                                                                    C.c_void_p(n_keep.data_ptr()), _stream_ptr(stream)))


def fdemri_select_modes_static(amp, eps, keep, n_keep, stream=None):
    """fdemri_select_modes without a plan or a work space: the scratch is a static device array of the library, so the call
    allocates nothing (include/fdemri.h).  amp: float64 CUDA tensor [n_batch][n_modes][n_knots][2]; keep, n_keep as there.
    Raises FdemriError(FDEMRI_ERR_STATIC_SCRATCH) when n_batch * n_knots > FDEMRI_STATIC_MAX_TOTALS."""
    assert amp.dim() == 4 and amp.shape[3] == 2
    n_batch, n_modes, n_knots = (int(x) for x in amp.shape[:3])
    assert keep.is_cuda and keep.is_contiguous() and keep.element_size() == 1 and keep.numel() == n_batch * n_modes
    assert n_keep.is_cuda and n_keep.is_contiguous() and n_keep.element_size() == 4 and n_keep.numel() == n_batch
    _chk("fdemri_select_modes_static", lib().fdemri_select_modes_static(n_batch, n_modes, n_knots, _ptr(amp), float(eps),
                                                                        C.c_void_p(keep.data_ptr()), C.c_void_p(n_keep.data_ptr()),
                                                                        _stream_ptr(stream)))


def fdemri_set_mode_mask(plan, keep):
    _chk("fdemri_set_mode_mask", lib().fdemri_set_mode_mask(plan, None if keep is None else C.c_void_p(keep.data_ptr())))


def fdemri_get_stats(plan, check=True) -> dict:
    s = FdemriStats()
    rc = lib().fdemri_get_stats(plan, C.byref(s))
    if check:
        _chk("fdemri_get_stats", rc)
    out = {k: int(getattr(s, k)) for k, _ in FdemriStats._fields_}
    out["status"] = rc
    return out


def fdemri_get_item_evals(plan, n_batch) -> np.ndarray:
    out = np.zeros(int(n_batch), dtype=np.uint64)
    _chk("fdemri_get_item_evals", lib().fdemri_get_item_evals(plan, out.ctypes.data_as(C.POINTER(C.c_uint64))))
    return out


def fdemri_get_coeffs(plan, shared_hi=None, shared_lo=None, amp_coef=None):
    _chk("fdemri_get_coeffs", lib().fdemri_get_coeffs(plan, _ptr(shared_hi), _ptr(shared_lo), _ptr(amp_coef)))


def fdemri_get_kernel_ms(plan) -> float:
    ms = C.c_float()
    _chk("fdemri_get_kernel_ms", lib().fdemri_get_kernel_ms(plan, C.byref(ms)))
    return float(ms.value)


def fdemri_measure_fp64_peak(n_iters=1 << 16) -> float:
    tf = C.c_double()
    _chk("fdemri_measure_fp64_peak", lib().fdemri_measure_fp64_peak(int(n_iters), C.byref(tf)))
    return float(tf.value)


def fdemri_measure_fp64_peak_3reg(n_iters=1 << 16) -> float:
    tf = C.c_double()
    _chk("fdemri_measure_fp64_peak_3reg", lib().fdemri_measure_fp64_peak_3reg(int(n_iters), C.byref(tf)))
    return float(tf.value)


def fdemri_measure_issue_ns(variant, n_iters=1 << 15) -> float:
    ns = C.c_double()
    _chk("fdemri_measure_issue_ns", lib().fdemri_measure_issue_ns(int(variant), int(n_iters), C.byref(ns)))
    return float(ns.value)


def fdemri_destroy(plan):
    _chk("fdemri_destroy", lib().fdemri_destroy(plan))


def fdemri_version() -> str:
    return lib().fdemri_version().decode()


def fdemri_build_splines_kerr(plan, f_phi, f_theta, f_r, Phi_phi, Phi_theta, Phi_r, amp, stream=None):
    _chk("fdemri_build_splines_kerr",
         lib().fdemri_build_splines_kerr(plan, _ptr(f_phi), _ptr(f_theta), _ptr(f_r), _ptr(Phi_phi), _ptr(Phi_theta),
                                         _ptr(Phi_r), _ptr(amp), _stream_ptr(stream)))


# ---- convenience: one object owning the torch buffers ---------------------------------------------------
class Waveform:
    """Owns the device buffers of one plan.  `lmn` with four columns (l, m, k, n) makes a plan of general voices
    (fdemri_plan_kerr); build_splines then wants f_theta and Phi_theta too."""

    def __init__(self, lmn, t_knots, n_freq, freqs=None, f0=0.0, df=0.0, device="cuda:0", flags=0):
        import torch
        self.torch = torch
        self.dev = torch.device(device)
        t_knots = np.atleast_2d(np.asarray(t_knots, dtype=np.float64))
        self.n_batch, self.n_knots = t_knots.shape
        self.n_freq = int(n_freq)
        self.lmn = np.ascontiguousarray(lmn, dtype=np.int32)
        self.n_modes = self.lmn.shape[0]
        self.t_knots = torch.from_numpy(t_knots).to(self.dev)
        self.freqs = None if freqs is None else torch.from_numpy(np.ascontiguousarray(freqs, dtype=np.float64)).to(self.dev)
        self.polar = self.lmn.shape[1] == 4
        make = fdemri_plan_kerr if self.polar else fdemri_plan
        self.plan = make(self.lmn, self.n_batch, self.n_knots, self.t_knots, self.n_freq, self.freqs, f0, df, flags)
        self._alloc_workspace(fdemri_workspace_bytes(self.plan))
        self.hplus = torch.empty((self.n_batch, self.n_freq, 2), dtype=torch.float64, device=self.dev)
        self.hcross = torch.empty_like(self.hplus)
        self._inputs = None

    def _alloc_workspace(self, nbytes):
        torch = self.torch
        self.ws = None                                      # release the old buffer first
        self.ws = torch.empty((nbytes + 255) // 8 + 32, dtype=torch.float64, device=self.dev)
        off = (-self.ws.data_ptr()) % 256
        self.ws_view = self.ws.view(torch.uint8)[off:off + nbytes]
        self.ws_bytes = nbytes
        fdemri_set_workspace(self.plan, self.ws_view)

    def ensure_capacity(self, stream=None) -> bool:
        """Kept for callers of the first release: there is no work list that could outgrow the work space any more
        (the sum kernels find their entries from the bands of the map), so there is never anything to grow."""
        return False

    def _build(self, stream):
        if self.polar:
            fp, fr, Pp, Pr, am, ft, Pt = self._inputs
            fdemri_build_splines_kerr(self.plan, fp, ft, fr, Pp, Pt, Pr, am, stream=stream)
        else:
            fdemri_build_splines(self.plan, *self._inputs, stream=stream)

    def build_splines(self, f_phi, f_r, Phi_phi, Phi_r, amp, stream=None, f_theta=None, Phi_theta=None):
        """Arguments: CUDA tensors, or numpy arrays (copied to the device first)."""
        torch = self.torch
        conv = lambda a: a if torch.is_tensor(a) else torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).to(self.dev)
        ins = [f_phi, f_r, Phi_phi, Phi_r, amp]
        if self.polar:
            assert f_theta is not None and Phi_theta is not None
            ins += [f_theta, Phi_theta]
        self._inputs = tuple(conv(a) for a in ins)
        self._build(stream)

    def sum(self, theta, phi, stream=None):
        fdemri_sum(self.plan, theta, phi, self.hplus, self.hcross, stream=stream)
        return self.hplus, self.hcross

    def stats(self, check=True):
        return fdemri_get_stats(self.plan, check=check)

    def item_evals(self) -> np.ndarray:
        return fdemri_get_item_evals(self.plan, self.n_batch)

    def coeffs(self):
        torch = self.torch
        S = self.n_knots - 1
        hi = torch.empty((self.n_batch, 4, S, 4), dtype=torch.float64, device=self.dev)
        lo = torch.empty_like(hi)
        am = torch.empty((self.n_batch, self.n_modes, 2, S, 4), dtype=torch.float64, device=self.dev)
        fdemri_get_coeffs(self.plan, hi, lo, am)
        torch.cuda.synchronize()
        return hi.cpu().numpy(), lo.cpu().numpy(), am.cpu().numpy()

    def result(self):
        """(hplus, hcross) as complex128 numpy arrays [n_batch][n_freq]."""
        self.torch.cuda.synchronize()
        hp = self.hplus.cpu().numpy().view(np.complex128)[..., 0]
        hx = self.hcross.cpu().numpy().view(np.complex128)[..., 0]
        return hp, hx

    def close(self):
        if self.plan is not None:
            fdemri_destroy(self.plan)
            self.plan = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def waveform_from_workload(w, device="cuda:0", flags=0) -> Waveform:
    polar = getattr(w, "lmkn", None) is not None
    wf = Waveform(w.lmkn if polar else w.lmn, w.t_knots, w.n_freq, freqs=w.freqs, f0=w.f0, df=w.df, device=device,
                  flags=flags)
    if polar:
        wf.build_splines(w.f_phi, w.f_r, w.Phi_phi, w.Phi_r, w.amp, f_theta=w.f_theta, Phi_theta=w.Phi_theta)
    else:
        wf.build_splines(w.f_phi, w.f_r, w.Phi_phi, w.Phi_r, w.amp)
    wf.ensure_capacity()
    return wf
