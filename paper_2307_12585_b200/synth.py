"""Seeded synthetic inputs for the five BASELINE.json configs (rules G1-G8).

This module serves BOTH the CUDA path and the CPU oracle, so it holds none of the method's
arithmetic (no splines, no root finding, no SPA terms): it only manufactures the *inputs* of
`fdemri_plan / fdemri_build_splines / fdemri_sum` -- a sparse inspiral trajectory
(~100 non-uniform points of t, Omega_phi, Omega_r, Phi_phi, Phi_r), complex mode
amplitudes at the knots (L60), a mode list, a frequency array (L141, L218) and viewing angles (L66).

The paper's real inputs come from FEW's flux grids and Teukolsky amplitude data (L58-60), which do
not exist here; these inputs stand in for them with the same shapes and sizes.  Only numpy/scipy.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np
from scipy.special import ellipe, ellipk, elliprf, elliprj

# G1 constants --------------------------------------------------------------------------------
MSUN_S = 4.925490947641267e-6          # G M_sun / c^3 in seconds
YEAR_S = 31558149.763545603            # sidereal year; pinned by Table 2's N_f = 6 311 631 (L236)
SEED0 = 230712585


def dft_grid(T_s: float, dt: float):
    """Uniform DFT grid (L141): N = ceil(T/dt) rounded up to even, bins i = 0..N/2, f_i = i*df."""
    N = int(math.ceil(T_s / dt))
    N += N & 1
    n_freq = N // 2 + 1
    df = 1.0 / (N * dt)
    return n_freq, 0.0, df


def uniform_freqs(n_freq: int, f0: float, df: float) -> np.ndarray:
    """The doubles f_i = f0 + (double)i*df (product rounded, then sum rounded)."""
    return f0 + np.arange(n_freq, dtype=np.float64) * df


# G3: Schwarzschild fundamental frequencies (dimensionless, per M) ------------------------------
def _ellippi(n, m):
    return elliprf(0.0, 1.0 - m, 1.0) + n / 3.0 * elliprj(0.0, 1.0 - m, 1.0, 1.0 - n)


def schwarzschild_omegas(p, e):
    """Omega_phi, Omega_r for bound Schwarzschild geodesics (p > 6 + 2e).

    T_r = int_0^2pi dt/dchi dchi and Delta_phi = int_0^2pi sqrt(p/(p-6-2e cos chi)) dchi with
    dt/dchi = p^2 sqrt((p-2)^2-4e^2) / [(p-2-2e cos chi)(1+e cos chi)^2 sqrt(p-6-2e cos chi)],
    reduced to Legendre K, E, Pi by chi = 2 theta + pi and partial fractions in sin^2 theta.
    Checked against periodic-trapezoid quadrature in tests/test_synth.py.
    """
    p = np.asarray(p, dtype=np.float64)
    e = np.maximum(np.asarray(e, dtype=np.float64), 1e-14)   # e -> 0 limit is regular; avoid 0/0
    m = 4.0 * e / (p - 6.0 + 2.0 * e)
    n1 = -2.0 * e / (1.0 - e)
    n2 = 4.0 * e / (p - 2.0 + 2.0 * e)
    K = ellipk(m)
    E = ellipe(m)
    P1 = _ellippi(n1, m)
    P2 = _ellippi(n2, m)
    # int dtheta / ((1 - n s^2)^2 Delta) = Pi + n dPi/dn
    P1sq = P1 + (n1 * E + (m - n1) * K + (n1 * n1 - m) * P1) / (2.0 * (m - n1) * (n1 - 1.0))
    a = 1.0 / (1.0 - n1 / n2) ** 2
    c = 1.0 / (1.0 - n2 / n1)
    b = 1.0 - a - c
    pref = 4.0 * p * p * np.sqrt((p - 2.0) ** 2 - 4.0 * e * e) / (
        (p - 2.0 + 2.0 * e) * (1.0 - e) ** 2 * np.sqrt(p - 6.0 + 2.0 * e))
    T_r = pref * (a * P2 + b * P1 + c * P1sq)
    dphi = 4.0 * np.sqrt(p / (p - 6.0 + 2.0 * e)) * K
    return dphi / T_r, 2.0 * np.pi / T_r


# G2: leading-order Peters-Mathews fluxes, in units of M ------------------------------------------
def _pe_rhs(p, e, q):
    one_me2 = (1.0 - e * e) ** 1.5
    dp = -(64.0 / 5.0) * q * one_me2 * (1.0 + 7.0 * e * e / 8.0) / p ** 3
    de = -(304.0 / 15.0) * q * e * one_me2 * (1.0 + 121.0 * e * e / 304.0) / p ** 4
    return dp, de


def _time_to_stop(p0, e0, q, nsteps=2000):
    """Time (units of M) from (p0,e0) to the stop surface p = 6 + 2e + 0.1, RK4 in x = p-6-2e."""
    p0 = np.asarray(p0, dtype=np.float64)
    e0 = np.asarray(e0, dtype=np.float64)
    x0 = p0 - 6.0 - 2.0 * e0
    hx = (0.1 - x0) / nsteps

    def rhs(x, e):
        p = x + 6.0 + 2.0 * e
        dp, de = _pe_rhs(p, e, q)
        dx = dp - 2.0 * de
        return de / dx, 1.0 / dx

    e = e0.copy()
    t = np.zeros_like(e)
    x = x0.copy()
    for _ in range(nsteps):
        k1e, k1t = rhs(x, e)
        k2e, k2t = rhs(x + 0.5 * hx, e + 0.5 * hx * k1e)
        k3e, k3t = rhs(x + 0.5 * hx, e + 0.5 * hx * k2e)
        k4e, k4t = rhs(x + hx, e + hx * k3e)
        e = e + hx / 6.0 * (k1e + 2 * k2e + 2 * k3e + k4e)
        t = t + hx / 6.0 * (k1t + 2 * k2t + 2 * k3t + k4t)
        x = x + hx
    return t


def plunge_p0(M, mu, e0, T_s):
    """G4: p0 in [6+2e0+0.2, 40] such that the inspiral reaches p = 6+2e+0.1 at t = T (bisection).
    If even the lower bound lasts longer than T (heavy M) the lower bound is returned."""
    M = np.atleast_1d(np.asarray(M, dtype=np.float64))
    e0 = np.atleast_1d(np.asarray(e0, dtype=np.float64))
    q = mu / M
    T_M = T_s / (M * MSUN_S)
    lo = 6.0 + 2.0 * e0 + 0.2
    hi = np.full_like(lo, 40.0)
    t_lo = _time_to_stop(lo, e0, q)
    stuck = t_lo >= T_M
    for _ in range(60):
        mid = 0.5 * (lo + hi)
        t_mid = _time_to_stop(mid, e0, q)
        too_long = t_mid > T_M
        hi = np.where(too_long, mid, hi)
        lo = np.where(too_long, lo, mid)
    p0 = 0.5 * (lo + hi)
    return np.where(stuck, 6.0 + 2.0 * e0 + 0.2, p0)


def trajectory(M, mu, p0, e0, t_knots, substeps=200):
    """G2: classical RK4 on (p, e, Phi_phi, Phi_r) with `substeps` equal steps per knot interval,
    Phi(0)=0.  Vectorised over a leading batch axis.  Returns dict of [B][N] arrays: f_phi, f_r in
    Hz (= Omega/(2 pi M), L94), Phi_phi, Phi_r in rad, p, e."""
    M = np.atleast_1d(np.asarray(M, dtype=np.float64))
    p = np.atleast_1d(np.asarray(p0, dtype=np.float64)).copy()
    e = np.atleast_1d(np.asarray(e0, dtype=np.float64)).copy()
    t_knots = np.atleast_2d(np.asarray(t_knots, dtype=np.float64))
    B, N = t_knots.shape
    q = mu / M
    Msec = M * MSUN_S
    php = np.zeros(B)
    phr = np.zeros(B)
    out = {k: np.empty((B, N)) for k in ("f_phi", "f_r", "Phi_phi", "Phi_r", "p", "e")}

    def rhs(p, e):
        dp, de = _pe_rhs(p, e, q)
        om_phi, om_r = schwarzschild_omegas(p, e)
        return dp, de, om_phi, om_r

    def record(k):
        om_phi, om_r = schwarzschild_omegas(p, e)
        out["f_phi"][:, k] = om_phi / (2.0 * np.pi * Msec)
        out["f_r"][:, k] = om_r / (2.0 * np.pi * Msec)
        out["Phi_phi"][:, k] = php
        out["Phi_r"][:, k] = phr
        out["p"][:, k] = p
        out["e"][:, k] = e

    record(0)
    for k in range(N - 1):
        h = (t_knots[:, k + 1] - t_knots[:, k]) / Msec / substeps
        for _ in range(substeps):
            a1 = rhs(p, e)
            a2 = rhs(p + 0.5 * h * a1[0], e + 0.5 * h * a1[1])
            a3 = rhs(p + 0.5 * h * a2[0], e + 0.5 * h * a2[1])
            a4 = rhs(p + h * a3[0], e + h * a3[1])
            p = p + h / 6.0 * (a1[0] + 2 * a2[0] + 2 * a3[0] + a4[0])
            e = e + h / 6.0 * (a1[1] + 2 * a2[1] + 2 * a3[1] + a4[1])
            php = php + h / 6.0 * (a1[2] + 2 * a2[2] + 2 * a3[2] + a4[2])
            phr = phr + h / 6.0 * (a1[3] + 2 * a2[3] + 2 * a3[3] + a4[3])
        record(k + 1)
    return out


def knots_uniform(T_s, n):
    return np.linspace(0.0, T_s, n)


def knots_plunge(T_s, n):
    """G5: t_k = T [1 - (1 - k/(N-1))^2] -- denser toward plunge, non-uniform like an adaptive stepper (L58)."""
    u = np.arange(n, dtype=np.float64) / (n - 1)
    return T_s * (1.0 - (1.0 - u) ** 2)


# G8 mode list -----------------------------------------------------------------------------------
def mode_list(l_min, l_max, m_values, n_max):
    """(l, m, n) int32 rows: l ascending, m in m_values(l) ascending, n = -n_max..n_max."""
    rows = []
    for l in range(l_min, l_max + 1):
        for m in m_values(l):
            for n in range(-n_max, n_max + 1):
                rows.append((l, m, n))
    return np.asarray(rows, dtype=np.int32)


# G6 amplitudes ------------------------------------------------------------------------------------
def amplitudes(rng, lmn, t_knots, scale_rule):
    """A_v(t) = a_v [P_re(s) cos th_v + i P_im(s) sin th_v], s = t/t_end, P(s) = 1+c1 s+c2 s^2+c3 s^3.
    Draw order per call: z[n_modes] normal, th[n_modes] U[0,2pi), c[n_modes][2][3] U(-.5,.5).
    Returns [n_modes][N][2] float64 (re, im)."""
    n_modes = lmn.shape[0]
    z = rng.standard_normal(n_modes)
    th = rng.uniform(0.0, 2.0 * np.pi, n_modes)
    c = rng.uniform(-0.5, 0.5, (n_modes, 2, 3))
    l = lmn[:, 0].astype(np.float64)
    n = np.abs(lmn[:, 2]).astype(np.float64)
    if scale_rule == "n2":
        scale = np.exp(-n / 2.0)
    elif scale_rule == "n4l":
        scale = np.exp(-n / 4.0) * np.exp(-(l - 2.0))
    else:
        raise ValueError(scale_rule)
    a = np.exp(0.5 * z) * scale
    s = (t_knots / t_knots[-1])[None, :]
    P = 1.0 + c[:, :, 0, None] * s[:, None, :] + c[:, :, 1, None] * s[:, None, :] ** 2 \
        + c[:, :, 2, None] * s[:, None, :] ** 3                       # [n_modes][2][N]
    amp = np.empty((n_modes, t_knots.shape[0], 2))
    amp[:, :, 0] = a[:, None] * P[:, 0, :] * np.cos(th)[:, None]
    amp[:, :, 1] = a[:, None] * P[:, 1, :] * np.sin(th)[:, None]
    return amp


@dataclasses.dataclass
class Workload:
    """One call's worth of inputs, host side (numpy).  Batch axis first."""
    name: str
    lmn: np.ndarray            # [n_modes][3] int32
    t_knots: np.ndarray        # [B][N]
    f_phi: np.ndarray          # [B][N] Hz
    f_r: np.ndarray            # [B][N] Hz
    Phi_phi: np.ndarray        # [B][N] rad
    Phi_r: np.ndarray          # [B][N] rad
    amp: np.ndarray            # [B][n_modes][N][2]
    n_freq: int
    f0: float
    df: float
    freqs: np.ndarray | None   # explicit array (arbitrary grid) or None for uniform
    theta: float
    phi: float
    meta: dict
    # general voices (l, m, k, n) of Eq. 1 (L64); None for the Schwarzschild workloads
    lmkn: np.ndarray | None = None        # [n_modes][4] int32; lmn then holds the columns (l, m, n) of the same rows
    f_theta: np.ndarray | None = None     # [B][N] Hz
    Phi_theta: np.ndarray | None = None   # [B][N] rad

    @property
    def n_batch(self):
        return self.t_knots.shape[0]

    @property
    def n_knots(self):
        return self.t_knots.shape[1]

    def freq_array(self) -> np.ndarray:
        return self.freqs if self.freqs is not None else uniform_freqs(self.n_freq, self.f0, self.df)


THETA = math.pi / 3.0
PHI = math.pi / 4.0


def _single(name, idx, M, mu, e0, T_yr, n_knots, lmn, scale_rule, p0=None, uniform_knots=False,
            dt=10.0, substeps=200):
    T_s = T_yr * YEAR_S
    rng = np.random.Generator(np.random.PCG64(SEED0 + idx))
    if p0 is None:
        p0 = float(plunge_p0(M, mu, e0, T_s)[0])
    t = knots_uniform(T_s, n_knots) if uniform_knots else knots_plunge(T_s, n_knots)
    tr = trajectory(M, mu, p0, e0, t[None, :], substeps=substeps)
    amp = amplitudes(rng, lmn, t, scale_rule)
    n_freq, f0, df = dft_grid(T_s, dt)
    return Workload(name, lmn, t[None, :], tr["f_phi"], tr["f_r"], tr["Phi_phi"], tr["Phi_r"],
                    amp[None], n_freq, f0, df, None, THETA, PHI,
                    dict(M=M, mu=mu, p0=p0, e0=e0, T_s=T_s, dt=dt, p_end=float(tr["p"][0, -1]),
                         e_end=float(tr["e"][0, -1]), scale_rule=scale_rule))


def config0():
    lmn = mode_list(2, 2, lambda l: (1, 2), 3)
    return _single("config0", 0, 1e6, 10.0, 0.2, 0.1, 50, lmn, "n2", p0=10.0, uniform_knots=True)


def config1():
    lmn = mode_list(2, 4, lambda l: range(0, l + 1), 10)
    return _single("config1", 1, 5e5, 10.0, 0.3, 1.0, 100, lmn, "n2")


def config2():
    lmn = mode_list(2, 10, lambda l: range(0, l + 1), 30)
    return _single("config2", 2, 2e6, 10.0, 0.4, 2.0, 150, lmn, "n4l")


def config3():
    w = config2()
    i = np.arange(10000, dtype=np.float64)
    w.freqs = 1e-5 * 5000.0 ** (i / 9999.0)
    w.n_freq = 10000
    w.name = "config3"
    return w


def config4_params(n_items=1024):
    rng = np.random.Generator(np.random.PCG64(SEED0 + 4))
    logM = rng.uniform(5.0, 7.0, n_items)
    e0 = rng.uniform(0.0, 0.5, n_items)
    return 10.0 ** logM, e0, rng


def config4(items=None, n_items=1024, substeps=200):
    """Batched config.  `items` selects a subset of the 1024 parameter sets (same draws as the full
    set: every item's amplitudes come from its own generator seeded SEED0 + 4 + 1000*(item+1))."""
    M, e0, _ = config4_params(n_items)
    if items is None:
        items = np.arange(n_items)
    items = np.asarray(items)
    M = M[items]
    e0 = e0[items]
    T_s = 1.0 * YEAR_S
    lmn = mode_list(2, 10, lambda l: range(0, l + 1), 30)
    p0 = plunge_p0(M, 10.0, e0, T_s)
    t = knots_plunge(T_s, 100)
    tk = np.broadcast_to(t, (len(items), 100)).copy()
    tr = trajectory(M, 10.0, p0, e0, tk, substeps=substeps)
    amp = np.empty((len(items), lmn.shape[0], 100, 2))
    for j, it in enumerate(items):
        rng = np.random.Generator(np.random.PCG64(SEED0 + 4 + 1000 * (int(it) + 1)))
        amp[j] = amplitudes(rng, lmn, t, "n4l")
    n_freq, f0, df = dft_grid(T_s, 10.0)
    return Workload("config4", lmn, tk, tr["f_phi"], tr["f_r"], tr["Phi_phi"], tr["Phi_r"], amp,
                    n_freq, f0, df, None, THETA, PHI,
                    dict(M=M, mu=10.0, p0=p0, e0=e0, T_s=T_s, dt=10.0, items=items))


CONFIGS = {0: config0, 1: config1, 2: config2, 3: config3, 4: config4}


def small_case(seed=1, n_knots=12, n_freq=30000, modes=((2, 2, 0), (2, 1, -2), (3, 0, 1), (2, 2, -3)),
               T_s=3.0e6, turnover=True):
    """A few-voice case for unit tests: analytic smooth f_phi(t), f_r(t) (f_r with a maximum inside
    the span when `turnover`), phases by exact integration of the analytic forms, random smooth
    amplitudes, uniform grid.  Cheap (no ODE)."""
    rng = np.random.Generator(np.random.PCG64(SEED0 + 100 + seed))
    u = np.sort(np.concatenate([[0.0, 1.0], rng.uniform(0.02, 0.98, n_knots - 2)]))
    t = T_s * u
    s = t / T_s
    # f_phi rising; f_r rising then falling (turnover near s = 0.6)
    fphi0, fphi1, fphi2 = 2.0e-3, 6.0e-4, 3.0e-4
    f_phi = fphi0 + fphi1 * s + fphi2 * s ** 2
    Phi_phi = 2 * np.pi * T_s * (fphi0 * s + fphi1 * s ** 2 / 2 + fphi2 * s ** 3 / 3)
    if turnover:
        fr0, fr1, fr2 = 1.2e-3, 2.4e-4, -2.0e-4
    else:
        fr0, fr1, fr2 = 1.2e-3, 1.0e-4, 0.5e-4
    f_r = fr0 + fr1 * s + fr2 * s ** 2
    Phi_r = 2 * np.pi * T_s * (fr0 * s + fr1 * s ** 2 / 2 + fr2 * s ** 3 / 3)
    lmn = np.asarray(modes, dtype=np.int32)
    amp = amplitudes(rng, lmn, t, "n2")
    df = 1.0 / T_s
    return Workload("small", lmn, t[None], f_phi[None], f_r[None], Phi_phi[None], Phi_r[None], amp[None],
                    n_freq, 0.0, df, None, THETA, PHI, dict(T_s=T_s))


# G9: general voices (l, m, k, n) -------------------------------------------------------------------------
KERR_MIX = (0.8137, 0.1542)     # f_theta = a f_phi + b f_r: between f_r and f_phi, as for prograde Kerr orbits


def with_polar_voices(w: Workload, k_max: int, seed: int = 0, k_decay: float = 1.0) -> Workload:
    """A workload of general voices (l, m, k, n), k = -k_max..k_max, on the trajectory of `w` (Eq. 1; the paper
    has no Kerr inputs: L252 expects "an order of magnitude" more modes).  The polar frequency is the fixed mix
    f_theta = a f_phi + b f_r (KERR_MIX), so that Phi_theta = a Phi_phi + b Phi_r is its exact integral; amplitudes are
    drawn like G6 with an extra factor exp(-k_decay |k|).  Rows: every (l, m, n) row of w.lmn, k ascending inside."""
    a, b = KERR_MIX
    ks = np.arange(-k_max, k_max + 1, dtype=np.int32)
    n0 = w.lmn.shape[0]
    lmn = np.repeat(w.lmn, ks.shape[0], axis=0)
    kk = np.tile(ks, n0)
    lmkn = np.stack([lmn[:, 0], lmn[:, 1], kk, lmn[:, 2]], axis=1).astype(np.int32)
    rng = np.random.Generator(np.random.PCG64(SEED0 + 900 + seed))
    amp = np.empty((w.n_batch, lmn.shape[0], w.n_knots, 2))
    rule = w.meta.get("scale_rule", "n2")
    for i in range(w.n_batch):
        amp[i] = amplitudes(rng, lmn, w.t_knots[i], rule) * np.exp(-k_decay * np.abs(kk))[:, None, None]
    meta = dict(w.meta, k_max=k_max, mix=KERR_MIX)
    return dataclasses.replace(w, name=w.name + "+k", lmn=lmn, amp=amp, meta=meta, lmkn=lmkn,
                               f_theta=a * w.f_phi + b * w.f_r, Phi_theta=a * w.Phi_phi + b * w.Phi_r)


def small_case_kerr(seed=1, n_knots=12, n_freq=30000,
                    modes=((2, 2, 0, 0), (2, 1, 1, -2), (3, 0, -1, 1), (2, 2, 2, -3), (3, 2, -1, 0), (4, 3, 1, 1)),
                    T_s=3.0e6):
    """small_case with a polar frequency of its own (analytic quadratic, exact phase), voices (l, m, k, n)."""
    modes = np.asarray(modes, dtype=np.int32)
    w = small_case(seed=seed, n_knots=n_knots, n_freq=n_freq, modes=modes[:, [0, 1, 3]], T_s=T_s)
    s = w.t_knots[0] / T_s
    c0, c1, c2 = 1.7e-3, 4.1e-4, 1.0e-4
    f_theta = c0 + c1 * s + c2 * s ** 2
    Phi_theta = 2 * np.pi * T_s * (c0 * s + c1 * s ** 2 / 2 + c2 * s ** 3 / 3)
    return dataclasses.replace(w, name="small+k", lmkn=modes, f_theta=f_theta[None], Phi_theta=Phi_theta[None])


def config5():
    """Not a BASELINE config: config 2's trajectory and grid with the polar harmonics k = -5..5 on every (l, m, n), the
    "order of magnitude" more modes the paper expects of Kerr (L252): 42273 voices."""
    return with_polar_voices(config2(), k_max=5)


CONFIGS[5] = config5
