"""Pins P3, P4, P6, P7, P8 for the oracle's harmonic sum."""
import math

import numpy as np
import pytest
from scipy.interpolate import CubicSpline
from scipy.special import airy

from paper_2307_12585_b200 import synth
from helpers import one_minus_overlap, weights_l2

TH, PH = math.pi / 3, math.pi / 4


def _run(orc, lmn, t, f_phi, f_r, P_phi, P_r, amp, freq, theta=TH, phi=PH):
    return orc.waveform(np.asarray(lmn, np.int32), t, f_phi, f_r, P_phi, P_r, amp, freq, theta, phi)


# ---- P3: linear chirp, single voice, closed-form SPA ---------------------------------------------
@pytest.mark.parametrize("l,m,n,aphi,bphi,ar,br", [
    (2, 2, 0, 1.5e-3, 2.0e-10, 1.0e-3, 1.0e-11),      # rising, F>0  (s=+1)
    (2, 2, 0, 2.5e-3, -1.5e-10, 1.0e-3, 1.0e-11),     # falling
    (2, 1, -3, 1.0e-3, 1.0e-10, 1.2e-3, 2.0e-11),     # F<0 everywhere -> contributes through s=-1
    (2, 0, 2, 1.0e-3, 1.0e-10, 1.2e-3, 2.0e-10),      # m=0 voice (R1)
    (2, 1, -1, 1.0e-3, 2.0e-10, 1.3e-3, 0.0),         # F crosses zero: both signs contribute
])
def test_linear_chirp_closed_form(orc, l, m, n, aphi, bphi, ar, br):
    T = 4.0e6
    rng = np.random.default_rng(5)
    # jittered knots (no nearly-coincident pair: those amplify the 1/2-ulp rounding of the Phi knot values)
    t = T * (np.arange(20) + np.concatenate([[0.0], rng.uniform(-0.3, 0.3, 18), [0.0]])) / 19.0
    f_phi, f_r = aphi + bphi * t, ar + br * t
    # knot values rounded once from extended precision, so that the inputs are the exact chirp to 1/2 ulp
    tl = t.astype(np.longdouble)
    two_pi = 2 * np.longdouble("3.14159265358979323846264338327950288")
    L = np.longdouble
    f_phi, f_r = (L(aphi) + L(bphi) * tl).astype(float), (L(ar) + L(br) * tl).astype(float)
    P_phi = (two_pi * (L(aphi) * tl + L(bphi) * tl * tl / 2)).astype(float)
    P_r = (two_pi * (L(ar) * tl + L(br) * tl * tl / 2)).astype(float)
    ca = np.array([1.0, 2e-7, -3e-14, 1e-21]) * 0.7
    cb = np.array([-0.4, 1e-7, 2e-14, -2e-21])
    A = lambda x: (ca[0] + ca[1] * x + ca[2] * x ** 2 + ca[3] * x ** 3) + 1j * (cb[0] + cb[1] * x + cb[2] * x ** 2 + cb[3] * x ** 3)
    amp = np.stack([A(t).real, A(t).imag], axis=-1)[None]
    df = 1.0 / T
    freq = np.arange(0, 30000) * df
    out = _run(orc, [(l, m, n)], t, f_phi, f_r, P_phi, P_r, amp, freq)
    F0, kap = m * aphi + n * ar, m * bphi + n * br
    Wp, Wx = weights_l2(m, TH, PH)
    hp = np.zeros(freq.size, complex)
    hx = np.zeros(freq.size, complex)
    for s in (+1, -1):
        ts = (s * freq - F0) / kap
        ok = (ts >= 0) & (ts < T) & (freq > 0)
        # keep clear of the end bins where membership is decided by rounding of knot values
        ok &= (ts > 1e-3) & (ts < T - 1e-3)
        S = A(ts) / math.sqrt(abs(kap)) * np.exp(1j * (math.pi * (s * freq - F0) ** 2 / kap - math.pi / 4 * np.sign(kap)))
        S = np.where(ok, S, 0)
        hp += S * Wp if s > 0 else np.conj(S * Wp)
        hx += S * Wx if s > 0 else np.conj(S * Wx)
    assert np.count_nonzero(hp) > 100
    scale = np.max(np.abs(hp))
    edge = np.zeros(freq.size, bool)
    for s in (+1, -1):
        ts = (s * freq - F0) / kap
        edge |= (np.abs(ts) < 2e-3) | (np.abs(ts - T) < 2e-3)
    keep = ~edge
    # phases reach ~1e5 rad and the knot values of Phi are rounded doubles: 3e-11 ("limited by R9")
    assert np.max(np.abs(out["hplus"] - hp)[keep]) < 3e-11 * scale
    assert np.max(np.abs(out["hcross"] - hx)[keep]) < 3e-11 * scale
    assert out["max_roots"] == 1


# ---- P4: quadratic chirp (turnover) = Airy closed form ----------------------------------------------
@pytest.mark.parametrize("Fdd", [-3.0e-17, 2.0e-17])
def test_quadratic_chirp_airy(orc, Fdd):
    T = 4.0e6
    te, Fe = 0.55 * T, 3.0e-3
    rng = np.random.default_rng(7)
    t = T * (np.arange(16) + np.concatenate([[0.0], rng.uniform(-0.3, 0.3, 14), [0.0]])) / 15.0
    u = t - te
    F = Fe + 0.5 * Fdd * u ** 2                       # voice (2,2,0): F = 2 f_phi
    Phi = 2 * np.pi * (Fe * u + Fdd * u ** 3 / 6)     # Phi_v = 2 Phi_phi
    f_phi, P_phi = F / 2, Phi / 2
    f_r, P_r = 1e-3 + 0 * t, 2 * np.pi * 1e-3 * t
    A0 = 0.8 - 0.3j
    amp = np.tile(np.array([A0.real, A0.imag]), (1, t.size, 1))
    df = 1.0 / T
    freq = np.arange(0, 14000) * df
    out = _run(orc, [(2, 2, 0)], t, f_phi, f_r, P_phi, P_r, amp, freq)
    Wp, Wx = weights_l2(2, TH, PH)
    x = np.sign(Fdd) * 2 * np.pi * (freq - Fe) / (np.pi * abs(Fdd)) ** (1 / 3)
    ai = airy(-x)[0]
    Phi_e = 0.0                                         # Phi(t_e) = 0 by construction (u = 0)
    full = A0 * np.exp(1j * (2 * np.pi * freq * te - Phi_e)) * 2 * np.pi * (np.pi * abs(Fdd)) ** (-1 / 3) * ai
    # bins where both roots lie inside [0, T): |u*| < min(te, T - te), on the oscillatory side
    ustar2 = 2 * (freq - Fe) / Fdd
    both = (ustar2 > 1e6) & (np.sqrt(np.abs(ustar2)) < 0.98 * min(te, T - te))
    assert both.sum() > 50
    assert out["max_roots"] == 2
    assert np.all(out["nterms"][both] == 2)
    scale = np.max(np.abs(full[both]))
    # Phi's knot values carry the rounding of 2 pi Fe u ~ 4e4 rad -> 1e-11 rad
    assert np.max(np.abs(out["hplus"][both] - full[both] * Wp)) < 1e-10 * scale
    assert np.max(np.abs(out["hcross"][both] - full[both] * Wx)) < 1e-10 * scale
    # beyond the extremum: no term at all (R7, L147)
    beyond = (freq - Fe) * np.sign(Fdd) < -4 * df
    assert np.all(out["nterms"][beyond] == 0) and np.all(out["hplus"][beyond] == 0)


# ---- P6: brute-force FFT of the time-domain voice sum ------------------------------------------------
def _td_case():
    N = 2 ** 19
    dt = 10.0
    T = N * dt
    modes = [(2, 2, 0), (2, 1, 1), (2, 2, -2), (3, 0, 2), (3, 3, -1), (2, 1, -4), (4, 2, 1), (2, 0, -1), (3, 1, -2)]
    w = synth.small_case(seed=3, n_knots=24, n_freq=N // 2 + 1, modes=modes, T_s=T)
    return w, N, dt


def _td_waveform(w, N, dt, theta, phi, orc):
    """h(t_j) = sum_V A_V Y_V exp(-i Phi_V) over the list AND the implied partners (Eq. 1-2), with scipy splines."""
    t = w.t_knots[0]
    tj = np.arange(N) * dt
    sp = lambda y: CubicSpline(t, y, bc_type="not-a-knot")(tj)
    Pp, Pr = sp(w.Phi_phi[0]), sp(w.Phi_r[0])
    h = np.zeros(N, complex)
    for v, (l, m, n) in enumerate(w.lmn):
        A = sp(w.amp[0, v, :, 0]) + 1j * sp(w.amp[0, v, :, 1])
        Phi = m * Pp + n * Pr
        h += A * orc.ylm(int(l), int(m), theta, phi) * np.exp(-1j * Phi)
        if m > 0:
            h += (-1) ** l * np.conj(A) * orc.ylm(int(l), -int(m), theta, phi) * np.exp(+1j * Phi)
    return h


def test_brute_force_fft(orc):
    w, N, dt = _td_case()
    freq = w.freq_array()
    out = orc.waveform(w.lmn, w.t_knots[0], w.f_phi[0], w.f_r[0], w.Phi_phi[0], w.Phi_r[0], w.amp[0], freq, TH, PH)
    assert out["max_roots"] == 2                                  # the case has turnover voices
    h = _td_waveform(w, N, dt, TH, PH, orc)
    # Eq. 3 sign: h~(f) = int h e^{+2 pi i f t} dt  ->  N dt ifft
    Hp = (N * dt * np.fft.ifft(h.real))[: N // 2 + 1]
    Hx = (N * dt * np.fft.ifft(-h.imag))[: N // 2 + 1]            # h = h+ - i hx (L64)
    sl = slice(1, N // 2)
    m_raw = one_minus_overlap(out["hplus"][sl], out["hcross"][sl], Hp[sl], Hx[sl])
    hann = 0.5 * (1 - np.cos(2 * np.pi * np.arange(N) / N))       # L145: Hann on the TD signal ...
    Hpw = (N * dt * np.fft.ifft(h.real * hann))[: N // 2 + 1]
    Hxw = (N * dt * np.fft.ifft(-h.imag * hann))[: N // 2 + 1]
    filt = lambda H: 0.5 * H[1:-1] - 0.25 * H[:-2] - 0.25 * H[2:]  # ... = 3-point convolution of the FD signal
    m_win = one_minus_overlap(filt(out["hplus"]), filt(out["hcross"]), Hpw[1:-1], Hxw[1:-1])
    assert m_raw < 1e-2, m_raw
    assert m_win < 2e-3, m_win
    # sensitivity: a conjugation or overall-sign mistake gives O(1)
    assert one_minus_overlap(np.conj(out["hplus"][sl]), out["hcross"][sl], Hp[sl], Hx[sl]) > 0.2
    assert one_minus_overlap(-out["hplus"][sl], -out["hcross"][sl], Hp[sl], Hx[sl]) > 1.5


# ---- P7: (l,-m,-n) <-> (-1)^l conj symmetry ---------------------------------------------------------
def test_partner_symmetry(orc):
    w = synth.small_case(seed=4, n_knots=16, modes=((2, 2, 0), (2, 1, -2), (3, 2, 1), (3, 0, 1), (4, 3, -3)))
    freq = w.freq_array()
    args = (w.t_knots[0], w.f_phi[0], w.f_r[0], w.Phi_phi[0], w.Phi_r[0])
    a = orc.waveform(w.lmn, *args, w.amp[0], freq, TH, PH)
    lmn2, amp2 = [], []
    for v, (l, m, n) in enumerate(w.lmn):
        lmn2.append((l, m, n)); amp2.append(w.amp[0, v])
        if m > 0:
            lmn2.append((l, -m, -n))
            p = w.amp[0, v].copy() * (-1) ** l
            p[:, 1] *= -1
            amp2.append(p)
    try:
        orc.set_explicit(True)
        b = orc.waveform(np.asarray(lmn2, np.int32), *args, np.asarray(amp2), freq, TH, PH)
    finally:
        orc.set_explicit(False)
    scale = np.max(np.abs(a["hplus"]))
    assert scale > 0
    assert np.max(np.abs(a["hplus"] - b["hplus"])) < 1e-13 * scale
    assert np.max(np.abs(a["hcross"] - b["hcross"])) < 1e-13 * scale
    # explicit enumeration counts a partner's root as its own term: every m>0 term appears twice
    n_m0 = sum(1 for (l, m, n) in w.lmn if m == 0)
    assert n_m0 == 1 and b["n_evals"] > a["n_evals"]


# ---- P8: zero outside support; root counts ------------------------------------------------------------
def test_zero_outside_support_and_root_count(orc):
    w = synth.small_case(seed=2, n_knots=14)
    freq = w.freq_array()
    out = orc.waveform(w.lmn, w.t_knots[0], w.f_phi[0], w.f_r[0], w.Phi_phi[0], w.Phi_r[0], w.amp[0], freq, TH, PH)
    assert out["hplus"][0] == 0 and out["hcross"][0] == 0            # R13
    # support from a dense scan of the voice frequencies (independent of the root finder)
    t = w.t_knots[0]
    tt = np.linspace(t[0], t[-1], 200001)
    fp = CubicSpline(t, w.f_phi[0])(tt)
    fr = CubicSpline(t, w.f_r[0])(tt)
    df = w.df
    cover = np.zeros(freq.size, bool)
    for l, m, n in w.lmn:
        F = m * fp + n * fr
        for s in (1, -1):
            lo, hi = (s * F).min(), (s * F).max()
            cover |= (freq >= lo - 2 * df) & (freq <= hi + 2 * df)
    outside = ~cover
    assert outside.sum() > 1000
    assert np.all(out["hplus"][outside] == 0) and np.all(out["hcross"][outside] == 0)
    assert np.all(out["nterms"][outside] == 0)
    assert out["max_roots"] == 2          # golden: N in {1,2} (L105, L111)
    assert out["n_evals"] == int(out["nterms"].sum())
    inside = out["nterms"] > 0
    assert np.all(np.abs(out["hplus"][inside]) > 0)


# ---- general voices (l, m, k, n) of Eq. 1 (L64; R16) ------------------------------------------------
def _run_kerr(orc, w, freq=None, lmkn=None, amp=None):
    freq = w.freq_array() if freq is None else freq
    return orc.waveform_kerr(w.lmkn if lmkn is None else lmkn, w.t_knots[0], w.f_phi[0], w.f_theta[0], w.f_r[0],
                             w.Phi_phi[0], w.Phi_theta[0], w.Phi_r[0], w.amp[0] if amp is None else amp, freq, TH, PH)


def test_kerr_voices_with_k_zero_are_the_schwarzschild_sum(orc):
    """k = 0 on every voice: bit for bit the (l, m, n) sum, whatever f_theta is."""
    w = synth.small_case_kerr(seed=5)
    lmkn = w.lmkn.copy()
    lmkn[:, 2] = 0
    a = _run_kerr(orc, w, lmkn=lmkn)
    b = _run(orc, lmkn[:, [0, 1, 3]], w.t_knots[0], w.f_phi[0], w.f_r[0], w.Phi_phi[0], w.Phi_r[0], w.amp[0], w.freq_array())
    assert np.max(np.abs(b["hplus"])) > 0
    assert np.array_equal(a["hplus"], b["hplus"]) and np.array_equal(a["hcross"], b["hcross"])
    assert a["n_evals"] == b["n_evals"]


def test_kerr_voices_polar_equal_radial(orc):
    """f_theta = f_r, Phi_theta = Phi_r: the voice (l, m, k, n) has the frequency and phase of (l, m, n + k), and for
    even k the same partner sign, so the two sums agree (up to the rounding of the knot values: bins whose membership
    hinges on it are left out)."""
    w = synth.small_case_kerr(seed=6, modes=((2, 2, 2, -1), (2, 1, -2, 0), (3, 0, 4, -3), (3, 3, 0, 1), (4, 2, -4, 2)))
    w.f_theta, w.Phi_theta = w.f_r.copy(), w.Phi_r.copy()
    a = _run_kerr(orc, w)
    lmn = np.stack([w.lmkn[:, 0], w.lmkn[:, 1], w.lmkn[:, 3] + w.lmkn[:, 2]], axis=1)
    b = _run(orc, lmn, w.t_knots[0], w.f_phi[0], w.f_r[0], w.Phi_phi[0], w.Phi_r[0], w.amp[0], w.freq_array())
    ok = (a["ambiguous"] == 0) & (b["ambiguous"] == 0)
    assert ok.sum() > 0.99 * ok.size and np.array_equal(a["nterms"][ok], b["nterms"][ok])
    scale = np.max(np.abs(b["hplus"]))
    assert scale > 0
    assert np.max(np.abs(a["hplus"][ok] - b["hplus"][ok])) < 1e-11 * scale
    assert np.max(np.abs(a["hcross"][ok] - b["hcross"][ok])) < 1e-11 * scale
    # odd k flips the partner's sign, (-1)^(l+k): the same comparison must then fail for an m > 0 voice
    w2 = synth.small_case_kerr(seed=6, modes=((2, 2, 1, -1),))
    w2.f_theta, w2.Phi_theta = w2.f_r.copy(), w2.Phi_r.copy()
    a2 = _run_kerr(orc, w2)
    b2 = _run(orc, np.asarray([(2, 2, 0)], np.int32), w2.t_knots[0], w2.f_phi[0], w2.f_r[0], w2.Phi_phi[0], w2.Phi_r[0],
              w2.amp[0], w2.freq_array())
    assert np.max(np.abs(a2["hplus"] - b2["hplus"])) > 1e-3 * np.max(np.abs(b2["hplus"]))


def test_kerr_partner_symmetry(orc):
    """The implied partner of (l, m, k, n) is (l, -m, -k, -n) with amplitude (-1)^(l+k) conj A (R16): listing it
    explicitly gives the same sum."""
    w = synth.small_case_kerr(seed=7)
    a = _run_kerr(orc, w)
    rows, amps = [], []
    for v, (l, m, k, n) in enumerate(w.lmkn):
        rows.append((l, m, k, n)); amps.append(w.amp[0, v])
        if m > 0:
            rows.append((l, -m, -k, -n))
            p = w.amp[0, v].copy() * (-1) ** (l + k)
            p[:, 1] *= -1
            amps.append(p)
    try:
        orc.set_explicit(True)
        b = _run_kerr(orc, w, lmkn=np.asarray(rows, np.int32), amp=np.asarray(amps))
    finally:
        orc.set_explicit(False)
    scale = np.max(np.abs(a["hplus"]))
    assert scale > 0 and b["n_evals"] > a["n_evals"]
    assert np.max(np.abs(a["hplus"] - b["hplus"])) < 1e-13 * scale
    assert np.max(np.abs(a["hcross"] - b["hcross"])) < 1e-13 * scale


def test_kerr_brute_force_fft(orc):
    """Eq. 1 with its k Phi_theta term, summed in the time domain over the list and the implied partners and
    Fourier-transformed, against the stationary-phase sum of the same voices."""
    N, dt = 2 ** 19, 10.0
    modes = [(2, 2, 0, 0), (2, 1, 1, 1), (2, 2, -1, -2), (3, 0, 2, 2), (3, 3, 1, -1), (2, 1, -2, -4), (4, 2, 1, 1),
             (2, 0, -1, -1), (3, 1, 3, -2)]
    w = synth.small_case_kerr(seed=3, n_knots=24, n_freq=N // 2 + 1, modes=modes, T_s=N * dt)
    out = _run_kerr(orc, w)
    t = w.t_knots[0]
    tj = np.arange(N) * dt
    sp = lambda y: CubicSpline(t, y, bc_type="not-a-knot")(tj)
    Pp, Pt, Pr = sp(w.Phi_phi[0]), sp(w.Phi_theta[0]), sp(w.Phi_r[0])
    h = np.zeros(N, complex)
    for v, (l, m, k, n) in enumerate(w.lmkn):
        A = sp(w.amp[0, v, :, 0]) + 1j * sp(w.amp[0, v, :, 1])
        Phi = m * Pp + k * Pt + n * Pr
        h += A * orc.ylm(int(l), int(m), TH, PH) * np.exp(-1j * Phi)
        if m > 0:
            h += (-1) ** (l + k) * np.conj(A) * orc.ylm(int(l), -int(m), TH, PH) * np.exp(+1j * Phi)
    hann = 0.5 * (1 - np.cos(2 * np.pi * np.arange(N) / N))
    Hpw = (N * dt * np.fft.ifft(h.real * hann))[: N // 2 + 1]
    Hxw = (N * dt * np.fft.ifft(-h.imag * hann))[: N // 2 + 1]
    filt = lambda H: 0.5 * H[1:-1] - 0.25 * H[:-2] - 0.25 * H[2:]
    m_win = one_minus_overlap(filt(out["hplus"]), filt(out["hcross"]), Hpw[1:-1], Hxw[1:-1])
    assert m_win < 2e-3, m_win
    # sensitivity: dropping the k Phi_theta term, or the (-1)^k of the partner, is seen
    lm0 = w.lmkn.copy(); lm0[:, 2] = 0
    bad = _run_kerr(orc, w, lmkn=lm0)
    assert one_minus_overlap(filt(bad["hplus"]), filt(bad["hcross"]), Hpw[1:-1], Hxw[1:-1]) > 0.2


# ---- the time-domain voice sum (Eq. 1 / Eq. 2) of the oracle -----------------------------------------------------
def test_td_sum_against_numpy_and_fft(orc):
    """fdemri_oracle_td (long double, C++) against the plain numpy sum with scipy's not-a-knot splines used by P6 above
    (phases reach 1e5 rad, so the double-precision scipy splines limit the agreement to ~1e-10); zero outside
    [t_0, t_{N-1}); h+ = Re h, hx = -Im h; and the FFT of the oracle's own time series against its own stationary-phase
    sum at the convention-check level of P6 (Hann-filtered mismatch < 2e-3)."""
    w, N, dt = _td_case()
    h = _td_waveform(w, N, dt, TH, PH, orc)
    hp, hx = orc.td(w.lmn, w.t_knots[0], w.Phi_phi[0], w.Phi_r[0], w.amp[0], N, 0.0, dt, TH, PH)
    scale = np.abs(h).max()
    assert np.max(np.abs(hp - h.real)) < 3e-10 * scale and np.max(np.abs(hx + h.imag)) < 3e-10 * scale
    # samples before t_0 and from t_{N-1} on are exactly zero; inside they are not
    hp2, hx2 = orc.td(w.lmn, w.t_knots[0], w.Phi_phi[0], w.Phi_r[0], w.amp[0], 64, -20 * dt, dt, TH, PH)
    assert np.all(hp2[:20] == 0) and np.all(hx2[:20] == 0) and np.all(hp2[20:] != 0)
    T = w.t_knots[0][-1]
    hp3, _ = orc.td(w.lmn, w.t_knots[0], w.Phi_phi[0], w.Phi_r[0], w.amp[0], 8, T - 4 * dt, dt, TH, PH)
    assert np.all(hp3[:4] != 0) and np.all(hp3[4:] == 0)
    # Eq. 3 convention and the Hann filter, now from the oracle's own time series
    out = orc.waveform(w.lmn, w.t_knots[0], w.f_phi[0], w.f_r[0], w.Phi_phi[0], w.Phi_r[0], w.amp[0], w.freq_array(), TH, PH)
    hann = 0.5 * (1 - np.cos(2 * np.pi * np.arange(N) / N))
    Hpw = (N * dt * np.fft.ifft(hp * hann))[: N // 2 + 1]
    Hxw = (N * dt * np.fft.ifft(hx * hann))[: N // 2 + 1]
    filt = lambda H: 0.5 * H[1:-1] - 0.25 * H[:-2] - 0.25 * H[2:]
    assert one_minus_overlap(filt(out["hplus"]), filt(out["hcross"]), Hpw[1:-1], Hxw[1:-1]) < 2e-3


def test_td_sum_general_voices(orc):
    """The k Phi_theta term and the (-1)^(l+k) of the partner in the time-domain sum: against the numpy sum of
    test_kerr_brute_force_fft's kind on a small case."""
    w = synth.small_case_kerr(seed=3, n_knots=16, n_freq=1024)
    t = w.t_knots[0]
    N, dt = 4096, t[-1] / 4096
    tj = np.arange(N) * dt
    sp = lambda y: CubicSpline(t, y, bc_type="not-a-knot")(tj)
    Pp, Pt, Pr = sp(w.Phi_phi[0]), sp(w.Phi_theta[0]), sp(w.Phi_r[0])
    h = np.zeros(N, complex)
    for v, (l, m, k, n) in enumerate(w.lmkn):
        A = sp(w.amp[0, v, :, 0]) + 1j * sp(w.amp[0, v, :, 1])
        Phi = m * Pp + k * Pt + n * Pr
        h += A * orc.ylm(int(l), int(m), TH, PH) * np.exp(-1j * Phi)
        if m > 0:
            h += (-1) ** (l + k) * np.conj(A) * orc.ylm(int(l), -int(m), TH, PH) * np.exp(+1j * Phi)
    hp, hx = orc.td(w.lmkn, t, w.Phi_phi[0], w.Phi_r[0], w.amp[0], N, 0.0, dt, TH, PH, Phi_theta=w.Phi_theta[0])
    scale = np.abs(h).max()
    assert np.max(np.abs(hp - h.real)) < 3e-10 * scale and np.max(np.abs(hx + h.imag)) < 3e-10 * scale
