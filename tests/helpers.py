"""Shared test helpers: parity statistics (R11) and closed forms that do not come from either
implementation."""
import math

import numpy as np


def y2(m, theta, phi):
    """Closed-form spin-weight -2 harmonics for l = 2."""
    c, s = math.cos(theta), math.sin(theta)
    tab = {2: math.sqrt(5 / (64 * math.pi)) * (1 + c) ** 2, 1: math.sqrt(5 / (16 * math.pi)) * s * (1 + c),
           0: math.sqrt(15 / (32 * math.pi)) * s * s, -1: math.sqrt(5 / (16 * math.pi)) * s * (1 - c),
           -2: math.sqrt(5 / (64 * math.pi)) * (1 - c) ** 2}
    return tab[m] * np.exp(1j * m * phi)


def weights_l2(m, theta, phi):
    """W+, Wx of DESIGN.md O2 for l = 2."""
    Y = y2(m, theta, phi)
    if m > 0:
        Ym = np.conj(y2(-m, theta, phi))
        return 0.5 * (Y + Ym), 0.5j * (Y - Ym)
    return 0.5 * Y, 0.5j * Y


def one_minus_overlap(ap, ax, bp, bx):
    """R11: flat-noise mismatch over both polarisations, as 1/2 |a^ - b^|^2 with unit-normalised vectors."""
    a = np.concatenate([ap, ax]).astype(np.complex128)
    b = np.concatenate([bp, bx]).astype(np.complex128)
    na = math.sqrt(math.fsum((a.real ** 2 + a.imag ** 2).tolist()))
    nb = math.sqrt(math.fsum((b.real ** 2 + b.imag ** 2).tolist()))
    if na == 0.0 and nb == 0.0:
        return 0.0
    d = a / na - b / nb
    return 0.5 * math.fsum((d.real ** 2 + d.imag ** 2).tolist())


def max_rel_err(ap, ax, bp, bx, mask=None):
    """max_bin |delta h| / max|h| over both polarisations (north_star tolerance 1e-10)."""
    scale = max(np.max(np.abs(bp)), np.max(np.abs(bx)))
    dp, dx = np.abs(ap - bp), np.abs(ax - bx)
    if mask is not None:
        dp, dx = dp[mask], dx[mask]
    if scale == 0.0:
        return float(max(dp.max(initial=0.0), dx.max(initial=0.0)))
    return float(max(dp.max(initial=0.0), dx.max(initial=0.0)) / scale)


def zigzag_case():
    """R5 test input: a zig-zag f_r through 5..8 random knots (seed 7) whose spline has a segment with TWO interior
    extrema (asserted with scipy), i.e. the paper's "at most one turnover per segment" (L105) does not hold."""
    from scipy.interpolate import CubicSpline
    from paper_2307_12585_b200 import synth
    rng = np.random.default_rng(7)
    N = int(rng.integers(5, 9))
    T = 3.0e6
    t = np.sort(np.concatenate([[0, T], rng.uniform(0.05, 0.95, N - 2) * T]))
    f_r = 1.3e-3 + 3e-4 * rng.uniform(-1, 1, N)
    cs = CubicSpline(t, f_r)
    two = 0
    for k in range(N - 1):
        r = np.roots([3 * cs.c[0, k], 2 * cs.c[1, k], cs.c[2, k]])
        r = r[np.isreal(r)].real
        two += int(np.sum((r > 0) & (r < t[k + 1] - t[k])) == 2)
    assert two >= 1
    f_phi = 2.0e-3 + 4.0e-4 * (t / T)
    Phi_r = 2 * np.pi * np.concatenate([[0.0], np.cumsum(0.5 * (f_r[1:] + f_r[:-1]) * np.diff(t))])
    Phi_phi = 2 * np.pi * (2.0e-3 * t + 2.0e-4 * t ** 2 / T)
    lmn = np.array([[2, 0, 1], [3, 1, -1], [2, 2, 2]], dtype=np.int32)
    amp = synth.amplitudes(np.random.Generator(np.random.PCG64(3)), lmn, t, "n2")
    n_freq = 24000
    return synth.Workload("two-extrema", lmn, t[None], f_phi[None], f_r[None], Phi_phi[None], Phi_r[None], amp[None],
                          n_freq, 0.0, 1.0 / T, None, 1.1, -0.4, {})
