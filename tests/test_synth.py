"""Input generator (paper_2307_12585_b200/synth.py): the closed-form Schwarzschild
frequencies against quadrature and the circular limit, the DFT grid against the paper's Table 2, determinism."""
import numpy as np

from paper_2307_12585_b200 import synth


def _omegas_quadrature(p, e, n=512):
    chi = 2.0 * np.pi * (np.arange(n) + 0.5) / n                 # periodic midpoint rule: spectrally accurate
    dt = p * p * np.sqrt((p - 2.0) ** 2 - 4.0 * e * e) / (
        (p - 2.0 - 2.0 * e * np.cos(chi)) * (1.0 + e * np.cos(chi)) ** 2 * np.sqrt(p - 6.0 - 2.0 * e * np.cos(chi)))
    dphi = np.sqrt(p / (p - 6.0 - 2.0 * e * np.cos(chi)))
    T_r = dt.sum() * 2.0 * np.pi / n
    return dphi.sum() * 2.0 * np.pi / n / T_r, 2.0 * np.pi / T_r


def test_frequencies_match_quadrature():
    for p, e in ((10.0, 0.2), (7.723, 0.4), (12.0, 0.05), (8.0, 0.45)):
        om_phi, om_r = synth.schwarzschild_omegas(p, e)
        q_phi, q_r = _omegas_quadrature(p, e)
        assert abs(om_phi / q_phi - 1.0) < 1e-12 and abs(om_r / q_r - 1.0) < 1e-12


def test_survey_probe_values_and_circular_limit():
    om_phi, om_r = synth.schwarzschild_omegas(10.0, 0.2)
    assert abs(om_phi - 0.030310185430) < 1e-11 and abs(om_r - 0.019133771077) < 1e-11
    p = 9.0
    om_phi, om_r = synth.schwarzschild_omegas(p, 0.0)
    assert abs(om_phi - p ** -1.5) < 1e-12 and abs(om_r - p ** -1.5 * np.sqrt(1.0 - 6.0 / p)) < 1e-10


def test_dft_grid_reproduces_table2():
    n_freq, f0, df = synth.dft_grid(4.0 * synth.YEAR_S, 10.0)     # N_f = 6 311 631
    assert n_freq == 6311631 and f0 == 0.0
    for T_yr, want in ((0.1, 157792), (1.0, 1577909), (2.0, 3155816)):
        assert synth.dft_grid(T_yr * synth.YEAR_S, 10.0)[0] == want


def test_config0_is_deterministic_and_well_formed():
    a, b = synth.config0(), synth.config0()
    for name in ("t_knots", "f_phi", "f_r", "Phi_phi", "Phi_r", "amp"):
        assert np.array_equal(getattr(a, name), getattr(b, name))
    assert a.lmn.shape == (14, 3) and a.amp.shape == (1, 14, 50, 2)
    assert np.all(np.diff(a.t_knots[0]) > 0) and np.all(np.diff(a.Phi_phi[0]) > 0)
    assert a.n_freq == 157792
