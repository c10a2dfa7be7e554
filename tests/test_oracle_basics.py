"""Pins P1 (splines), P2 (-2Y_lm), P5 (g(X)) for the CPU oracle.  SURVEY.md section 8(c)."""
import math
import os

import mpmath as mp
import numpy as np
import pytest
from scipy.interpolate import CubicSpline

from paper_2307_12585_b200 import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")


def golden():
    out = {}
    for line in open(GOLD):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


def test_table2_bin_count():
    """N_f = 6 311 631 at T = 4 yr, dt = 10 s pins the year and the N/2+1 layout (G1)."""
    g = golden()
    n_freq, f0, df = synth.dft_grid(g["table2_T_years"] * synth.YEAR_S, g["table2_dt_seconds"])
    assert n_freq == int(g["table2_n_freq"])
    assert f0 == 0.0


# ---- P1 --------------------------------------------------------------------------------------
def test_spline_reproduces_cubic(orc):
    rng = np.random.default_rng(1)
    t = np.sort(rng.uniform(0, 5e6, 40))
    t[0] = 0.0
    c = np.array([0.3, -2e-7, 5e-14, 3e-21])
    y = c[0] + c[1] * t + c[2] * t ** 2 + c[3] * t ** 3
    hi, lo = orc.build_splines(t, y[None])
    co = hi[0] + lo[0]
    for k in range(len(t) - 1):
        tk = t[k]
        exact = [c[0] + c[1] * tk + c[2] * tk ** 2 + c[3] * tk ** 3, c[1] + 2 * c[2] * tk + 3 * c[3] * tk ** 2,
                 c[2] + 3 * c[3] * tk, c[3]]
        # scale of each coefficient times h^j compared against |y|
        h = t[k + 1] - tk
        for j in range(4):
            assert abs(co[k, j] - exact[j]) * h ** j < 1e-13 * np.max(np.abs(y))


def test_spline_matches_scipy_not_a_knot(orc):
    rng = np.random.default_rng(2)
    t = np.cumsum(rng.uniform(0.2, 3.0, 60))
    y = np.sin(0.3 * t) + 0.1 * t + rng.normal(0, 0.01, t.size)
    hi, lo = orc.build_splines(t, y[None])
    cs = CubicSpline(t, y, bc_type="not-a-knot")          # c[3-j] is the tau^j coefficient
    ref = np.stack([cs.c[3], cs.c[2], cs.c[1], cs.c[0]], axis=1)
    np.testing.assert_allclose(hi[0], ref, rtol=0, atol=2e-12)
    # interpolation and C2 continuity
    co = hi[0] + lo[0]
    h = np.diff(t)
    end = co[:, 0] + co[:, 1] * h + co[:, 2] * h ** 2 + co[:, 3] * h ** 3
    np.testing.assert_allclose(end, y[1:], atol=1e-13)
    d1 = co[:, 1] + 2 * co[:, 2] * h + 3 * co[:, 3] * h ** 2
    np.testing.assert_allclose(d1[:-1], co[1:, 1], atol=1e-12)
    d2 = 2 * co[:, 2] + 6 * co[:, 3] * h
    np.testing.assert_allclose(d2[:-1], 2 * co[1:, 2], atol=1e-12)
    # not-a-knot: third derivative continuous at t_1 and t_{N-2}
    assert abs(co[0, 3] - co[1, 3]) < 1e-13 and abs(co[-1, 3] - co[-2, 3]) < 1e-13


# ---- P2 --------------------------------------------------------------------------------------
@pytest.mark.parametrize("theta,phi", [(math.pi / 3, math.pi / 4), (0.3, 2.0), (2.5, -1.0), (0.0, 0.7), (math.pi, 0.2)])
def test_ylm_l2_closed_forms(orc, theta, phi):
    c = math.cos(theta)
    s = math.sin(theta)
    ref = {
        (2, 2): math.sqrt(5 / (64 * math.pi)) * (1 + c) ** 2 * np.exp(2j * phi),
        (2, 1): math.sqrt(5 / (16 * math.pi)) * s * (1 + c) * np.exp(1j * phi),
        (2, 0): math.sqrt(15 / (32 * math.pi)) * s ** 2,
        (2, -1): math.sqrt(5 / (16 * math.pi)) * s * (1 - c) * np.exp(-1j * phi),
        (2, -2): math.sqrt(5 / (64 * math.pi)) * (1 - c) ** 2 * np.exp(-2j * phi),
    }
    for (l, m), v in ref.items():
        assert abs(orc.ylm(l, m, theta, phi) - v) < 1e-14


def test_ylm_orthonormal_and_phase(orc):
    # Gauss-Legendre in cos(theta); phi-dependence e^{i m phi} checked separately
    x, w = np.polynomial.legendre.leggauss(48)
    th = np.arccos(x)
    for m in (0, 1, 2, 3, 7):
        ls = [l for l in range(2, 11) if l >= m]
        Y = np.array([[orc.ylm(l, m, t, 0.0).real for t in th] for l in ls])
        G = 2 * math.pi * (Y * w) @ Y.T
        np.testing.assert_allclose(G, np.eye(len(ls)), atol=2e-13)
    y = orc.ylm(7, 3, 1.1, 0.9)
    assert abs(y - orc.ylm(7, 3, 1.1, 0.0) * np.exp(3j * 0.9)) < 1e-15
    assert abs(orc.ylm(7, 3, 1.1, 0.0).imag) == 0.0


def test_ylm_conjugation_symmetry(orc):
    """conj(sY_lm) = (-1)^{s+m} (-s)Y_{l,-m}; for s=-2 use the parity relation
    -2Y_lm(pi-theta, phi+pi) = (-1)^l  +2Y_lm(theta,phi) = (-1)^{l+m} conj(-2Y_{l,-m}(theta,phi))."""
    for l, m in [(2, 1), (3, -2), (5, 4), (10, -7), (6, 0)]:
        th, ph = 0.8, 0.3
        lhs = orc.ylm(l, m, math.pi - th, ph + math.pi)
        rhs = (-1) ** (l + m) * np.conj(orc.ylm(l, -m, th, ph))
        assert abs(lhs - rhs) < 1e-14


# ---- P5 --------------------------------------------------------------------------------------
def g_mp(X):
    mp.mp.dps = 40
    ax = mp.mpf(abs(X))
    g = mp.sqrt(mp.pi * ax / 2) * mp.e ** (1j * mp.pi / 6) * mp.e ** (-1j * ax) * mp.hankel1(mp.mpf(1) / 3, ax)
    return complex(g) if X > 0 else complex(mp.conj(g))


@pytest.mark.parametrize("X", [1e-9, 1e-6, 1e-3, 0.1, 0.5, 1.0, 3.0, 7.0, 12.46, 25.0, 29.999, 30.001, 45.0, 100.0, 1e3,
                               1e4, 1e6, -0.2, -7.0, -29.0, -31.0, -5e4])
def test_g_vs_mpmath_hankel(orc, X):
    assert abs(orc.g(X) - g_mp(X)) < 2e-14


def test_g_limits(orc):
    g = golden()
    ph = g["spa_limit_phase_over_pi"] * math.pi
    assert abs(orc.g(1e12) - np.exp(1j * ph)) < 1e-12           # L119: standard SPA limit
    assert abs(orc.g(-1e12) - np.exp(-1j * ph)) < 1e-12
    # first correction of the large-|X| series: g ~ e^{-i pi/4}(1 - 5i/(72 X))
    X = 2e4
    assert abs(orc.g(X) - np.exp(-1j * math.pi / 4) * (1 - 5j / (72 * X) - 385 / (10368 * X * X))) < 1e-13


def test_g_over_sqrt_is_contour_integral_half(orc):
    """Eq. 7's integral  I = int exp(-i pi (Fd t^2 + Fdd t^3/3)) dt  equals the Airy form
    2 pi (pi|Fdd|)^{-1/3} Ai(-y) e^{-iX}; the per-root factor is its single-stationary-point half, and the two
    halves (roots Fd and -Fd of the same turnover) sum to it (R3)."""
    mp.mp.dps = 30
    Fd, Fdd = 0.9, 0.35
    X = 2 * mp.pi * Fd ** 3 / (3 * Fdd ** 2)
    y = (3 * X / 2) ** (mp.mpf(2) / 3)
    full = mp.e ** (-1j * X) * 2 * mp.pi * (mp.pi * Fdd) ** (-mp.mpf(1) / 3) * mp.airyai(-y)
    own = orc.g_over_sqrt(Fd, Fdd)
    # the other stationary point of the same cubic phase sits at t' = -2 Fd/Fdd with slope -Fd; its term carries
    # the phase offset exp(-2iX):  pi*(-Fd)*t'^2 ... = exp(-i*2X) relative to the own point
    other = orc.g_over_sqrt(-Fd, Fdd) * complex(mp.e ** (-2j * X))
    assert abs(own + other - complex(full)) < 1e-13
    # and the integral itself by rotated-contour quadrature (t = s e^{-i pi/6} for s>0, s e^{-5 i pi/6}... use mp.quadosc-free form)
    f = lambda t: mp.e ** (-1j * mp.pi * (Fd * t * t + Fdd * t ** 3 / 3))
    r1 = mp.e ** (-1j * mp.pi / 6)
    r2 = mp.e ** (-5j * mp.pi / 6)
    I = mp.quad(lambda s: f(s * r1) * r1, [0, 2, 6, 12]) - mp.quad(lambda s: f(s * r2) * r2, [0, 2, 6, 12])
    assert abs(complex(I) - complex(full)) < 1e-12


def test_eq8_identity_real_alpha():
    """Eq. 8 (L113) for real alpha > 0 by direct quadrature."""
    mp.mp.dps = 25
    a, b = mp.mpf("0.7"), mp.mpf("1.3")
    lhs = mp.quad(lambda t: mp.e ** (-a * t * t / 2 - 1j * b * t ** 3 / 6), list(range(-16, 17)))
    z = a ** 3 / (3 * b * b)
    rhs = 2 / mp.sqrt(3) * a / abs(b) * mp.e ** z * mp.besselk(mp.mpf(1) / 3, z)
    assert abs(lhs - rhs) < 1e-15


def test_regular_form_at_zero_slope(orc):
    mp.mp.dps = 30
    Fdd = -2.3e-18
    v = orc.g_over_sqrt(0.0, Fdd)
    ref = mp.pi * (mp.pi * abs(Fdd)) ** (-mp.mpf(1) / 3) * (mp.airyai(0) - 1j * mp.airybi(0))
    assert abs(v - complex(ref)) < 1e-13 * abs(ref)
    # continuity across the small-|X| switch
    for Fd in (1e-16, 3e-15, 1e-13):
        a = orc.g_over_sqrt(Fd, Fdd)
        X = 2 * mp.pi * mp.mpf(Fd) ** 3 / (3 * mp.mpf(Fdd) ** 2)
        y = (3 * X / 2) ** (mp.mpf(2) / 3)
        ref = mp.e ** (-1j * X) * mp.pi * (mp.pi * abs(Fdd)) ** (-mp.mpf(1) / 3) * (mp.airyai(-y) - 1j * mp.airybi(-y))
        assert abs(a - complex(ref)) < 1e-13 * abs(ref)


def test_inner_product_is_the_weighted_dot_product(orc):
    """Pin of fdemri_oracle_inner (Eq. 12): equals numpy's vdot on random arrays (library
    routine); <h|h> = sum |h|^2 for w = 1; Hermitian: <d|h> = conj <h|d>; linear in w."""
    rng = np.random.default_rng(5)
    n = 1000
    hp, hx, dp, dx = (rng.standard_normal(n) + 1j * rng.standard_normal(n) for _ in range(4))
    w = rng.uniform(0.1, 2.0, n)
    hh, dh = orc.inner(hp, hx, dp, dx, w)
    want_hh = np.sum(w * (np.abs(hp) ** 2 + np.abs(hx) ** 2))
    want_dh = np.vdot(hp, w * dp) + np.vdot(hx, w * dx)            # vdot conjugates its first argument
    assert abs(hh - want_hh) <= 1e-12 * want_hh and abs(dh - want_dh) <= 1e-12 * abs(want_dh)
    hh1, _ = orc.inner(hp, hx)
    assert abs(hh1 - (np.vdot(hp, hp) + np.vdot(hx, hx)).real) <= 1e-12 * hh1
    _, hd = orc.inner(dp, dx, hp, hx, w)
    assert abs(hd - np.conj(dh)) <= 1e-12 * abs(dh)
    hh2, dh2 = orc.inner(hp, hx, dp, dx, 3.0 * w)
    assert abs(hh2 - 3.0 * hh) <= 1e-12 * hh2 and abs(dh2 - 3.0 * dh) <= 1e-12 * abs(dh2)


def test_hann_filter_is_the_dft_of_the_windowed_series(orc):
    """Pin of the 3-point filter (the Hann window on the time series is a convolution of the
    frequency-domain waveform with the window's DFT): for a series whose spectrum vanishes at both ends of the
    grid, DFT(hann * x)_k = X_k/2 - X_{k-1}/4 - X_{k+1}/4 exactly, so the oracle's filtered <h|h> must equal the
    sum over the FFT of the windowed series."""
    rng = np.random.default_rng(9)
    N = 512
    X = np.zeros(N, dtype=complex)
    X[3:200] = rng.standard_normal(197) + 1j * rng.standard_normal(197)      # zero at the grid ends: no wrap-around
    x = np.fft.ifft(X)
    n = np.arange(N)
    win = 0.5 * (1.0 - np.cos(2.0 * np.pi * n / N))
    Xw = np.fft.fft(win * x)
    want = np.sum(np.abs(Xw[:256]) ** 2)
    zeros = np.zeros(256, dtype=complex)
    got, _ = orc.inner(X[:256], zeros, hann=True)
    assert abs(got - want) <= 1e-12 * want
    d = rng.standard_normal(256) + 1j * rng.standard_normal(256)
    _, dh = orc.inner(X[:256], zeros, d, zeros, hann=True)
    assert abs(dh - np.vdot(Xw[:256], d)) <= 1e-12 * abs(dh)


def test_mode_selection_reading():
    """Pins of oracle.select_modes: the sorted-array walk equals the direct threshold on every mode's
    own power; eps = 0 keeps every mode, eps > 1 none; the kept set shrinks as eps grows; a mode that dominates at a
    single time step only is kept (the union over time steps)."""
    import oracle
    rng = np.random.default_rng(4)
    V, N = 60, 17
    amp = rng.standard_normal((V, N, 2)) * np.exp(rng.uniform(-8, 0, (V, 1, 1)))
    amp[7, :, :] = 1e-9
    amp[7, 5, :] = 30.0                                          # dominant at one step only
    power = amp[..., 0] ** 2 + amp[..., 1] ** 2
    prev = None
    for eps in (0.0, 1e-8, 1e-5, 1e-2, 0.3, 1.5):
        keep, total = oracle.select_modes(amp, eps)
        direct = np.any(power >= eps * power.sum(axis=0)[None, :], axis=1)
        assert np.array_equal(keep, direct)
        assert np.allclose(total, power.sum(axis=0), rtol=1e-14)
        if prev is not None:
            assert np.all(prev | ~keep)                          # monotone: kept at larger eps => kept at smaller
        prev = keep
    assert oracle.select_modes(amp, 0.0)[0].all() and not oracle.select_modes(amp, 1.5)[0].any()
    assert oracle.select_modes(amp, 0.3)[0][7]
