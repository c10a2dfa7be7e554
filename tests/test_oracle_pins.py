"""More pins of the CPU oracle (round 2): the level-A entry fdemri_oracle_sum, the membership / root-count logic (R5-R8)
against an implementation that shares nothing with it (scipy's piecewise-polynomial root finder), the half-open rule at
a knot (R6) on a constructed case whose knot values fall exactly on bins, and both readings of the mode selection."""
import math

import numpy as np
import pytest
from scipy.interpolate import CubicSpline

from paper_2307_12585_b200 import synth
from helpers import weights_l2, zigzag_case

TH, PH = math.pi / 3, math.pi / 4


def _waveform(orc, w, freq=None):
    freq = w.freq_array() if freq is None else freq
    return orc.waveform(w.lmn, w.t_knots[0], w.f_phi[0], w.f_r[0], w.Phi_phi[0], w.Phi_r[0], w.amp[0], freq, w.theta, w.phi)


# ---- fdemri_oracle_sum (the level-A entry) -------------------------------------------------------------------
@pytest.mark.parametrize("case", ["small", "config0"])
def test_sum_of_built_splines_is_the_waveform_bit_for_bit(orc, case):
    """fdemri_oracle_sum fed the oracle's own long-double coefficients (as hi + lo doubles: exact, a long double has 64
    mantissa bits) must give fdemri_oracle_waveform bit for bit: pins the coefficient layouts [4][N-1][4] and
    [n_modes][2][N-1][4], the hi + lo reassembly and the argument order of the level-A entry."""
    w = synth.small_case(seed=2, n_knots=14) if case == "small" else synth.config0()
    t = w.t_knots[0]
    freq = w.freq_array()
    a = _waveform(orc, w)
    sh_hi, sh_lo = orc.build_splines(t, np.stack([w.f_phi[0], w.f_r[0], w.Phi_phi[0], w.Phi_r[0]]))
    V, N = w.lmn.shape[0], t.shape[0]
    comp = np.ascontiguousarray(np.transpose(w.amp[0], (0, 2, 1))).reshape(2 * V, N)       # rows: (voice, re/im)
    am_hi, am_lo = orc.build_splines(t, comp)
    am_hi, am_lo = am_hi.reshape(V, 2, N - 1, 4), am_lo.reshape(V, 2, N - 1, 4)
    b = orc.sum(w.lmn, t, w.f_phi[0], w.f_r[0], sh_hi, sh_lo, am_hi, am_lo, freq, w.theta, w.phi)
    assert a["n_evals"] == b["n_evals"] > 0
    assert np.array_equal(a["nterms"], b["nterms"]) and np.array_equal(a["ambiguous"], b["ambiguous"])
    assert np.array_equal(a["hplus"].view(np.uint64), b["hplus"].view(np.uint64))
    assert np.array_equal(a["hcross"].view(np.uint64), b["hcross"].view(np.uint64))
    # and the hi parts alone are not the same thing (the lo parts are really used)
    c = orc.sum(w.lmn, t, w.f_phi[0], w.f_r[0], sh_hi, None, am_hi, None, freq, w.theta, w.phi)
    assert not np.array_equal(a["hplus"], c["hplus"])
    # a transposed amplitude layout ([2][n_modes] instead of [n_modes][2]) must be visible
    if V > 1:
        bad = np.ascontiguousarray(np.transpose(am_hi, (1, 0, 2, 3))).reshape(V, 2, N - 1, 4)
        d = orc.sum(w.lmn, t, w.f_phi[0], w.f_r[0], sh_hi, sh_lo, bad, None, freq, w.theta, w.phi)
        assert np.max(np.abs(d["hplus"] - a["hplus"])) > 1e-3 * np.max(np.abs(a["hplus"]))


# ---- root counts and membership against scipy's piecewise-polynomial solver -------------------------------------
def _independent_root_counts(w, freq):
    """Number of real roots t in [t_0, t_{N-1}) of F_v(t) = s f for every bin, summed over list voices and both signs.
    F_v = the scipy not-a-knot spline through the knot doubles F_k = fl(fl(m f_phi,k) + fl(n f_r,k)) (the spline is linear
    in its data, L103); roots from scipy's PPoly.solve (closed-form / companion-matrix roots per piece).  Also returns the
    bins whose count is ill-conditioned for this method: a root within 1e-7 of the span from either end of the
    trajectory, or two roots closer than 1e-6 of the span (a bin sitting on an extremum value)."""
    t = w.t_knots[0]
    T = t[-1] - t[0]
    cnt = np.zeros(freq.size, dtype=np.int64)
    unsure = np.zeros(freq.size, dtype=bool)
    for (l, m, n) in w.lmn:
        Fk = float(m) * w.f_phi[0] + float(n) * w.f_r[0]
        cs = CubicSpline(t, Fk, bc_type="not-a-knot")
        fine = cs(np.linspace(t[0], t[-1], 4001))
        for s in (1, -1):
            lo, hi = (s * fine).min(), (s * fine).max()
            pad = 0.05 * (hi - lo) + 1e-9
            for i in np.flatnonzero((freq > 0) & (freq >= lo - pad) & (freq <= hi + pad)):
                x = s * freq[i]
                if x == Fk[-1]:
                    unsure[i] = True                   # decided by rule R6/R14 below, not by a computed root
                    continue
                r = np.sort(cs.solve(x, extrapolate=False))
                r = r[np.isfinite(r)]
                if r.size and (r[0] - t[0] < 1e-7 * T and x != Fk[0] or t[-1] - r[-1] < 1e-7 * T):
                    unsure[i] = True
                if r.size > 1 and np.min(np.diff(r)) < 1e-6 * T:
                    unsure[i] = True
                cnt[i] += int(np.sum(r < t[-1]))
    return cnt, unsure


@pytest.mark.parametrize("case", ["turnover", "zigzag"])
def test_root_counts_against_scipy_ppoly(orc, case):
    """The per-bin number of accumulated terms of the oracle (R5-R8: piece splitting at extrema, half-open membership on
    the knot doubles, both signs, f > 0) equals the number of real roots found by an unrelated solver, on a single-turnover
    trajectory and on the zig-zag with a two-extrema segment.  Excluded: the oracle's own boundary-ambiguous bins (R8) and
    the bins the independent count marks ill-conditioned -- together a handful."""
    w = synth.small_case(seed=2, n_knots=14) if case == "turnover" else zigzag_case()
    freq = w.freq_array()
    out = _waveform(orc, w)
    cnt, unsure = _independent_root_counts(w, freq)
    keep = (out["ambiguous"] == 0) & ~unsure
    assert (~keep).sum() <= 6
    assert out["n_evals"] > 5000 and out["max_roots"] >= (2 if case == "turnover" else 3)
    assert np.array_equal(cnt[keep], out["nterms"][keep])
    # every multiplicity the oracle reports is seen by the independent count too
    assert set(np.unique(out["nterms"][keep])) == set(np.unique(cnt[keep]))
    assert cnt[keep].max() >= 3


# ---- R6: a root on a knot is counted once; the last knot is excluded ------------------------------------------------
@pytest.mark.parametrize("slope", [+1, -1])
def test_knot_values_exactly_on_bins(orc, slope):
    """Linear chirp with dyadic numbers throughout: df = 2^-22 Hz, knots t_k = k 2^18 s (k = 0..16), F(t) = F_0 + kappa t
    with kappa = +-2^-32 Hz/s and F_0 a multiple of df, so that every knot value F_k is EXACTLY a bin frequency.  R6
    (half-open in time, "one or two segments per voice"): every bin between F(t_0) and F(t_16) gets exactly
    one term -- also the sixteen bins that sit on a knot, each shared by two segments -- the bin of the first knot is
    included, the bin of the last knot is not.  Values against the closed-form SPA (L119) on all of them."""
    df = 2.0 ** -22
    kappa = slope * 2.0 ** -32
    tk = np.arange(17, dtype=np.float64) * 2.0 ** 18
    T = tk[-1]
    F0 = 2.0 ** -9 if slope > 0 else 2.0 ** -9 + 2.0 ** -10       # F runs 2^-9 .. 2^-9 + 2^-10 (up) or back (down)
    F = F0 + kappa * tk                                            # exact in double
    assert np.all(np.round(F / df) == F / df)
    # voice (2, 2, 0): F = 2 f_phi.  Phases: Phi_v = 2 pi (F0 t + kappa t^2 / 2), rounded once from extended precision
    L = np.longdouble
    two_pi = 2 * L("3.14159265358979323846264338327950288")
    Phi = (two_pi * (L(F0) * tk.astype(L) + L(kappa) * tk.astype(L) ** 2 / 2)).astype(float)
    f_phi, P_phi = F / 2, Phi / 2
    f_r, P_r = np.full_like(tk, 1e-3), 2 * np.pi * 1e-3 * tk
    A0 = 0.6 - 0.35j
    amp = np.tile(np.array([A0.real, A0.imag]), (1, tk.size, 1))
    n_freq = 2 ** 14
    freq = np.arange(n_freq, dtype=np.float64) * df
    out = orc.waveform(np.array([[2, 2, 0]], np.int32), tk, f_phi, f_r, P_phi, P_r, amp, freq, TH, PH)
    i_first, i_last = int(round(F[0] / df)), int(round(F[-1] / df))
    lo, hi = min(i_first, i_last), max(i_first, i_last)
    want = np.zeros(n_freq, dtype=np.int32)
    want[lo:hi + 1] = 1
    want[i_last] = 0                                               # t_{N-1} is excluded (R6, R14)
    assert want[i_first] == 1
    assert np.array_equal(out["nterms"], want)
    assert out["ambiguous"].sum() == 0 and out["max_roots"] == 1
    knot_bins = np.round(F[:-1] / df).astype(int)
    assert np.all(out["nterms"][knot_bins] == 1)
    # closed form: A |kappa|^-1/2 exp{i [pi (f - F0)^2 / kappa - pi/4 sgn kappa]} W, on every bin with a term
    Wp, Wx = weights_l2(2, TH, PH)
    sel = want == 1
    S = A0 / math.sqrt(abs(kappa)) * np.exp(1j * (math.pi * (freq[sel] - F0) ** 2 / kappa - math.pi / 4 * slope))
    scale = abs(A0) / math.sqrt(abs(kappa)) * abs(Wp)
    assert np.max(np.abs(out["hplus"][sel] - S * Wp)) < 3e-11 * scale
    assert np.max(np.abs(out["hcross"][sel] - S * Wx)) < 3e-11 * scale
    assert np.all(out["hplus"][~sel] == 0)


# ---- mode selection: the two readings of L60 (R15) -----------------------------------------------------
def test_mode_selection_hand_computed_five_modes():
    """Five modes, two time steps, powers chosen by hand (squares of small integers, exact in binary):
         step 0: 16, 8, 4, 2, 1   (total 31)        step 1: 1, 2, 64, 2, 1   (total 70)
       eps = 0.2.  "own": p >= eps total -> step 0: p >= 6.2 keeps modes {0, 1}; step 1: p >= 14 keeps {2}; union {0,1,2}.
       "cumulative": shortest sorted prefix reaching (1 - eps) total -> step 0: target 24.8, sums 16, 24, 28 -> {0,1,2};
       step 1: target 56, sums 64 -> {2}; union {0,1,2}.  With eps = 0.25: own: step 0 p >= 7.75 -> {0,1}, step 1 p >= 17.5
       -> {2}: union {0,1,2};  cumulative: step 0 target 23.25, sums 16, 24 -> {0,1}; step 1 target 52.5 -> {2}.
       eps = 0.04: own: step 0 p >= 1.24 -> {0,1,2,3}; step 1 p >= 2.8 -> {2}; union {0,1,2,3}.  cumulative: step 0 target
       29.76: sums 16, 24, 28, 30 -> {0,1,2,3}; step 1 target 67.2: sums 64, 66 (mode 1: stable order among the 2s),
       68 (mode 3) -> {2,1,3}; union {0,1,2,3}.
       eps = 0.1: own: step 0 p >= 3.1 -> {0,1,2}; step 1 p >= 7 -> {2}.  cumulative: step 0 target 27.9: 16, 24, 28 ->
       {0,1,2}; step 1 target 63 -> {2}.
       The two readings differ at eps = 0.2 restricted to step 0 alone ({0,1} against {0,1,2})."""
    import oracle
    amp = np.zeros((5, 2, 2))
    amp[:, 0, 0] = [4, 2, 2, 1, 1]
    amp[:, 0, 1] = [0, 2, 0, 1, 0]
    amp[:, 1, 0] = [1, 1, 8, 1, 1]
    amp[:, 1, 1] = [0, 1, 0, 1, 0]
    m = lambda *idx: np.isin(np.arange(5), idx)
    for eps, own, cum in ((0.2, m(0, 1, 2), m(0, 1, 2)), (0.25, m(0, 1, 2), m(0, 1, 2)), (0.04, m(0, 1, 2, 3), m(0, 1, 2, 3)),
                          (0.1, m(0, 1, 2), m(0, 1, 2))):
        k1, tot = oracle.select_modes(amp, eps, rule="own")
        k2, _ = oracle.select_modes(amp, eps, rule="cumulative")
        assert np.array_equal(tot, [31.0, 70.0])
        assert np.array_equal(k1, own), (eps, k1)
        assert np.array_equal(k2, cum), (eps, k2)
    one = amp[:, :1, :]
    assert np.array_equal(oracle.select_modes(one, 0.2, rule="own")[0], m(0, 1))
    assert np.array_equal(oracle.select_modes(one, 0.2, rule="cumulative")[0], m(0, 1, 2))
    assert np.array_equal(oracle.select_modes(one, 0.25, rule="cumulative")[0], m(0, 1))
    # the cumulative reading bounds the discarded power by eps total at every step; the own-power reading does not
    rng = np.random.default_rng(8)
    big = rng.standard_normal((400, 9, 2)) * np.exp(rng.uniform(-6, 0, (400, 1, 1)))
    power = big[..., 0] ** 2 + big[..., 1] ** 2
    for eps in (1e-3, 1e-2, 0.1):
        keep, total = oracle.select_modes(big, eps, rule="cumulative")
        assert np.all(power[~keep].sum(axis=0) <= eps * total * (1 + 1e-12))
        keep_own, _ = oracle.select_modes(big, eps, rule="own")
        assert keep_own.sum() < keep.sum()                       # many small modes add up: the own-power rule drops more
    assert np.any(power[~oracle.select_modes(big, 1e-2, rule="own")[0]].sum(axis=0) > 1e-2 * total)
    assert not oracle.select_modes(big, 1.0, rule="cumulative")[0].any()
    assert oracle.select_modes(big, 0.0, rule="cumulative")[0].sum() >= 395      # all but modes below the rounding of the sum
