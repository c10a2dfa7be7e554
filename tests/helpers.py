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
