"""GPU parity: libfdemri (through the C ABI) against the CPU oracle, element by element.

Bar (BASELINE.json north_star): per bin |delta h| <= 1e-10 max|h|, and 1 - overlap <= 1e-12 (flat noise,
both polarisations).  Bins the oracle marks boundary-ambiguous (R8: within 16 ulp of an
extremum value F_e) are excluded from the per-bin check (expected count: 0; MAX_AMBIGUOUS = 2 tolerated per waveform).  Level C = independent spline builds; level A = oracle fed the GPU's coefficients.
"""
import functools
import math

import numpy as np
import pytest

from helpers import max_rel_err, one_minus_overlap

pytestmark = pytest.mark.gpu

TOL_BIN = 1e-10
TOL_MISMATCH = 1e-12
MAX_AMBIGUOUS = 2          # DESIGN.md R8


@pytest.fixture(scope="module")
def fd():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2307_12585_b200 as pkg
    return pkg


@functools.lru_cache(maxsize=None)
def workload(idx):
    from paper_2307_12585_b200 import synth
    return synth.CONFIGS[idx]()


def oracle_c(orc, w, freq, b=0):
    if getattr(w, "lmkn", None) is not None:
        return orc.waveform_kerr(w.lmkn, w.t_knots[b], w.f_phi[b], w.f_theta[b], w.f_r[b], w.Phi_phi[b], w.Phi_theta[b],
                                 w.Phi_r[b], w.amp[b], freq, w.theta, w.phi)
    return orc.waveform(w.lmn, w.t_knots[b], w.f_phi[b], w.f_r[b], w.Phi_phi[b], w.Phi_r[b], w.amp[b], freq,
                        w.theta, w.phi)


def check(gp, gx, ref, label):
    keep = ref["ambiguous"] == 0
    assert (~keep).sum() <= MAX_AMBIGUOUS, f"{label}: {(~keep).sum()} ambiguous bins"
    err = max_rel_err(gp, gx, ref["hplus"], ref["hcross"], mask=keep)
    mm = one_minus_overlap(gp[keep], gx[keep], ref["hplus"][keep], ref["hcross"][keep])
    print(f"[parity] {label}: max|dh|/max|h| = {err:.3e}, 1-overlap = {mm:.3e}, bins = {keep.sum()}")
    assert np.all(np.isfinite(gp)) and np.all(np.isfinite(gx))
    assert err <= TOL_BIN, f"{label}: per-bin {err}"
    assert mm <= TOL_MISMATCH, f"{label}: mismatch {mm}"
    # exact zeros where the oracle has no term (P8)
    zero = (ref["nterms"] == 0) & keep
    assert np.all(gp[zero] == 0) and np.all(gx[zero] == 0), f"{label}: non-zero outside support"
    return err, mm


def run_gpu(fd, w):
    wf = fd.waveform_from_workload(w)
    wf.sum(w.theta, w.phi)
    hp, hx = wf.result()
    st = wf.stats()
    return wf, hp, hx, st


def test_small_case_levels_A_and_C(fd, orc):
    from paper_2307_12585_b200 import synth
    w = synth.small_case(seed=2, n_knots=14)
    wf, hp, hx, st = run_gpu(fd, w)
    freq = w.freq_array()
    ref = oracle_c(orc, w, freq)
    assert ref["max_roots"] == 2
    check(hp[0], hx[0], ref, "small level C")
    assert st["n_evals"] == ref["n_evals"]                      # P9
    assert st["n_airy"] > 0 and st["n_turnover"] > 0
    # level A: the oracle's sum on the GPU-built coefficients
    hi, lo, am = wf.coeffs()
    refA = orc.sum(w.lmn, w.t_knots[0], w.f_phi[0], w.f_r[0], hi[0], lo[0], am[0], None, freq, w.theta, w.phi)
    check(hp[0], hx[0], refA, "small level A")
    # level B: coefficients themselves (phase increments over a segment, relative amplitude deviation)
    ohi, olo = orc.build_splines(w.t_knots[0], np.stack([w.f_phi[0], w.f_r[0], w.Phi_phi[0], w.Phi_r[0]]))
    h = np.diff(w.t_knots[0])
    dco = (hi[0] - ohi) + (lo[0] - olo)
    for c in (2, 3):
        inc = np.abs(dco[c, :, 1] * h) + np.abs(dco[c, :, 2] * h ** 2) + np.abs(dco[c, :, 3] * h ** 3)
        assert inc.max() < 1e-12, f"phase-increment deviation {inc.max()} rad"
    wf.close()


def test_small_case_no_turnover_other_angles(fd, orc):
    from paper_2307_12585_b200 import synth
    w = synth.small_case(seed=5, n_knots=9, turnover=False, modes=((2, 2, 0), (3, 1, 2), (4, 0, 3), (5, 5, -1), (10, 7, -2)))
    w.theta, w.phi = 2.1, -0.7
    wf, hp, hx, st = run_gpu(fd, w)
    ref = oracle_c(orc, w, w.freq_array())
    check(hp[0], hx[0], ref, "no-turnover")
    assert st["n_evals"] == ref["n_evals"]
    wf.close()


def test_config0_full(fd, orc):
    w = workload(0)
    wf, hp, hx, st = run_gpu(fd, w)
    ref = oracle_c(orc, w, w.freq_array())
    check(hp[0], hx[0], ref, "config0")
    assert st["n_evals"] == ref["n_evals"]
    wf.close()


def test_config1_full(fd, orc):
    w = workload(1)
    wf, hp, hx, st = run_gpu(fd, w)
    ref = oracle_c(orc, w, w.freq_array())
    check(hp[0], hx[0], ref, "config1")
    assert st["n_evals"] == ref["n_evals"]
    assert ref["max_roots"] == 2
    wf.close()


def _sampled_bins(n_freq, n, seed, hi_frac=0.36):
    rng = np.random.default_rng(seed)
    a = rng.integers(1, int(n_freq * hi_frac), size=n)
    edge = np.array([0, 1, 2, 255, 256, 257, n_freq - 2, n_freq - 1])
    return np.unique(np.concatenate([a, edge]))


def test_config2_sampled_bins_full_size(fd, orc):
    """BASELINE config 2 at full size in the launch configuration bench.py times; the oracle computes sampled
    bins one by one (an arbitrary grid holding exactly those frequencies)."""
    w = workload(2)
    wf, hp, hx, st = run_gpu(fd, w)
    idx = _sampled_bins(w.n_freq, 6000, 11)
    freq = w.freq_array()[idx]
    ref = oracle_c(orc, w, freq)
    # scale by the full waveform's maximum, as the tolerance is stated
    scale = max(np.abs(hp[0]).max(), np.abs(hx[0]).max())
    keep = ref["ambiguous"] == 0
    dp = np.abs(hp[0][idx] - ref["hplus"])[keep].max() / scale
    dx = np.abs(hx[0][idx] - ref["hcross"])[keep].max() / scale
    mm = one_minus_overlap(hp[0][idx][keep], hx[0][idx][keep], ref["hplus"][keep], ref["hcross"][keep])
    print(f"[parity] config2 sampled: {dp:.3e} {dx:.3e} mismatch {mm:.3e}; evals {st['n_evals']:.4g} items {st['n_items']}")
    assert max(dp, dx) <= TOL_BIN and mm <= TOL_MISMATCH
    assert 2.5e8 < st["n_evals"] < 4e8            # ~3.15e8 evaluations
    # properties that hold at any size: zero beyond the highest voice frequency, f = 0 bin zero
    assert hp[0][0] == 0 and hx[0][0] == 0
    assert np.all(hp[0][int(0.5 * w.n_freq):] == 0)
    wf.close()


def test_config3_arbitrary_grid(fd, orc):
    w = workload(3)
    wf, hp, hx, st = run_gpu(fd, w)
    ref = oracle_c(orc, w, w.freq_array())
    check(hp[0], hx[0], ref, "config3")
    assert st["n_evals"] == ref["n_evals"]
    wf.close()


def test_deterministic_bitwise(fd):
    w = workload(1)
    wf = fd.waveform_from_workload(w)
    wf.sum(w.theta, w.phi)
    a = [x.copy() for x in wf.result()]
    for _ in range(2):
        wf.sum(w.theta, w.phi)
        b = wf.result()
        assert np.array_equal(a[0].view(np.uint64), b[0].view(np.uint64))
        assert np.array_equal(a[1].view(np.uint64), b[1].view(np.uint64))
    wf.close()


def test_batched_config4_eight_items(fd, orc):
    """BASELINE config 4 on the inputs bench.py times (substeps = 200, the seeded parameter sets): 8 of the 1024 items
    spanning the M range (1e5 .. 1e7: 3.9e9 .. 2e6 evaluations each) in one plan, per-item viewing angles.
      * >= 1e5 random (item, bin) samples in total against the oracle, bar 1e-10 per bin relative to the item's max|h|;
      * the three cheapest items (2e6, 1.5e7 and 1e8 evaluations) element by element over EVERY bin, with the per-item
        evaluation count of the map (fdemri_get_item_evals) equal to the oracle's count of accumulated terms (P9)."""
    from paper_2307_12585_b200 import synth
    M, e0, _ = synth.config4_params()
    order = np.argsort(M)
    pick = [0, 146, 292, 438, 585, 731, 877, 1023]
    items = [int(order[i]) for i in pick]
    w = synth.config4(items=items)                                   # substeps = 200, as bench.py --config 4
    wf = fd.waveform_from_workload(w)
    rng = np.random.default_rng(404)
    th = np.concatenate([[w.theta], rng.uniform(0.2, 2.9, len(items) - 1)])
    ph = np.concatenate([[w.phi], rng.uniform(-3.0, 3.0, len(items) - 1)])
    wf.sum(th, ph)
    hp, hx = wf.result()
    st = wf.stats()
    per_item = wf.item_evals()
    assert st["flags"] == 0 and int(per_item.sum()) == st["n_evals"] and np.all(per_item > 0)
    # the three cheapest items (fewest evaluations): every bin
    cheap = [int(i) for i in np.argsort(per_item)[:3]]
    n_samples = 0
    freq_all = w.freq_array()
    for b in range(len(items)):
        full = b in cheap
        idx = np.arange(w.n_freq) if full else _sampled_bins(w.n_freq, 14000, 40 + b, hi_frac=0.95)
        ref = orc.waveform(w.lmn, w.t_knots[b], w.f_phi[b], w.f_r[b], w.Phi_phi[b], w.Phi_r[b], w.amp[b], freq_all[idx],
                           float(th[b]), float(ph[b]))
        scale = max(np.abs(hp[b]).max(), np.abs(hx[b]).max())
        keep = ref["ambiguous"] == 0
        assert (~keep).sum() <= MAX_AMBIGUOUS
        err = max(np.abs(hp[b][idx] - ref["hplus"])[keep].max(), np.abs(hx[b][idx] - ref["hcross"])[keep].max()) / scale
        mm = one_minus_overlap(hp[b][idx][keep], hx[b][idx][keep], ref["hplus"][keep], ref["hcross"][keep])
        zero = (ref["nterms"] == 0) & keep
        assert np.all(hp[b][idx][zero] == 0) and np.all(hx[b][idx][zero] == 0)
        counts = f"map count {int(per_item[b])}"
        if full:
            assert int(per_item[b]) == ref["n_evals"], (items[b], int(per_item[b]), ref["n_evals"])
            counts += f" = oracle count {ref['n_evals']} (every bin)"
        print(f"[parity] config4 item {items[b]} (M = {M[items[b]]:.3g}, e0 = {e0[items[b]]:.2f}): max|dh|/max|h| = {err:.3e}, "
              f"1-overlap = {mm:.3e}, {len(idx)} bins, {counts}")
        assert err <= TOL_BIN and mm <= TOL_MISMATCH
        n_samples += len(idx)
    assert n_samples >= 100000
    wf.close()


def test_edge_cases(fd, orc):
    import torch
    from paper_2307_12585_b200 import synth
    w = synth.small_case(seed=6, n_knots=4, n_freq=1)           # minimum knots; only the f = 0 bin
    wf, hp, hx, st = run_gpu(fd, w)
    assert hp.shape == (1, 1) and hp[0, 0] == 0 and hx[0, 0] == 0 and st["n_evals"] == 0
    wf.close()
    w = synth.small_case(seed=6, n_knots=4, n_freq=777)         # ragged tile; grid entirely below every voice
    wf, hp, hx, st = run_gpu(fd, w)
    ref = oracle_c(orc, w, w.freq_array())
    assert ref["n_evals"] == st["n_evals"]
    check(hp[0], hx[0], ref, "ragged")
    wf.close()
    w = synth.small_case(seed=7, n_knots=5, n_freq=20001)       # 4 segments, ragged tail, turnover
    wf, hp, hx, st = run_gpu(fd, w)
    ref = oracle_c(orc, w, w.freq_array())
    check(hp[0], hx[0], ref, "n_knots=5")
    assert ref["n_evals"] == st["n_evals"] and st["n_evals"] > 0
    wf.close()
    # error behaviour
    t = torch.zeros((1, 3), dtype=torch.float64, device="cuda")
    with pytest.raises(fd.FdemriError):
        fd.fdemri_plan(np.array([[2, 2, 0]], np.int32), 1, 3, t, 10, None, 0.0, 1e-6)      # n_knots < 4
    t = torch.zeros((1, 8), dtype=torch.float64, device="cuda")
    with pytest.raises(fd.FdemriError):
        fd.fdemri_plan(np.array([[2, 3, 0]], np.int32), 1, 8, t, 10, None, 0.0, 1e-6)      # m > l
    p = fd.fdemri_plan(np.array([[2, 2, 0]], np.int32), 1, 8, t, 10, None, 0.0, 1e-6)
    out = torch.zeros((1, 10, 2), dtype=torch.float64, device="cuda")
    with pytest.raises(fd.FdemriError) as ei:
        fd.fdemri_sum(p, 0.1, 0.2, out, out)                                               # no work space
    assert ei.value.status == 2
    fd.fdemri_destroy(p)


def test_work_space_is_exact_and_too_small_is_refused(fd, orc):
    """There is no work list any more (the sum kernels find their entries from the bands of the map), so the work
    space has no optional part: the minimum is the size, a smaller buffer is refused by fdemri_set_workspace, and
    the exact size is enough for the heaviest list the old design knew (config 0 through both kernels)."""
    import torch
    w = workload(0)
    for flags in (fd.FDEMRI_FLAG_TILE_MAJOR, fd.FDEMRI_FLAG_BIN_MAJOR):
        wf = fd.Waveform(w.lmn, w.t_knots, w.n_freq, freqs=w.freqs, f0=w.f0, df=w.df, flags=flags)
        need = fd.fdemri_workspace_bytes(wf.plan)
        assert fd.fdemri_workspace_bytes_min(wf.plan) == need
        small = torch.empty(need // 8, dtype=torch.float64, device=wf.dev)
        off = (-small.data_ptr()) % 256
        with pytest.raises(fd.FdemriError) as ei:
            fd.fdemri_set_workspace(wf.plan, small.view(torch.uint8)[off:off + need - 256])
        assert ei.value.status == 2
        wf._alloc_workspace(need)
        wf.build_splines(w.f_phi, w.f_r, w.Phi_phi, w.Phi_r, w.amp)
        assert wf.ensure_capacity() is False
        wf.sum(w.theta, w.phi)
        hp, hx = wf.result()
        ref = oracle_c(orc, w, w.freq_array())
        check(hp[0], hx[0], ref, f"config0, exact work space (flags={flags})")
        st = wf.stats()
        assert st["n_evals"] == ref["n_evals"] and st["flags"] == 0
        wf.close()


def test_many_voices_in_one_tile(fd, orc):
    """Far more entries in a tile / block than the shared-memory queues of the item scan hold (512 staged entries in
    the tile-major producer; 8 x 256 collected entries per round in the bin-major kernel): the scan must hand them out
    in rounds, in the same fixed order.  9000 voices (l = 2, m = 2, n = 0) all cover the same bins."""
    from paper_2307_12585_b200 import synth
    base = synth.small_case(seed=3, n_knots=6, n_freq=3000, modes=((2, 2, 0),), turnover=False)
    base.f0 = 4.0e-3                                             # F = 2 f_phi sweeps 4.0 .. 5.8 mHz
    nv = 9000
    base.lmn = np.repeat(base.lmn, nv, axis=0)
    rng = np.random.Generator(np.random.PCG64(7))
    scale = rng.uniform(0.5, 1.5, (1, nv, 1, 1))
    base.amp = np.ascontiguousarray(np.repeat(base.amp, nv, axis=1) * scale)
    wf, hp, hx, st = run_gpu(fd, base)
    ref = oracle_c(orc, base, base.freq_array())
    check(hp[0], hx[0], ref, "9000 voices in one tile")
    assert st["n_evals"] == ref["n_evals"] and st["n_evals"] >= nv * 2000 and st["n_pairs"] >= 4 * nv
    assert st["n_items"] <= st["n_pairs"] <= st["n_items"] + 9000 * 3    # every entry once, plus once per tile border it crosses
    wf2, hp2, hx2, _ = run_gpu(fd, base)                         # and it is reproducible bit for bit
    assert np.array_equal(hp, hp2) and np.array_equal(hx, hx2)
    wf.close(); wf2.close()
    hb = []
    for _ in range(2):                                           # per-bin lists of 9000 keys, twice: same bits
        wf3 = fd.waveform_from_workload(base, flags=fd.FDEMRI_FLAG_BIN_MAJOR)
        wf3.sum(base.theta, base.phi)
        hb.append(wf3.result())
        st3 = wf3.stats()
        assert st3["n_evals"] == ref["n_evals"] == st3["n_pairs"]     # terms accumulated = terms of the map (P9)
        wf3.close()
    check(hb[0][0][0], hb[0][1][0], ref, "9000 voices per bin, bin-major")
    assert np.array_equal(hb[0][0], hb[1][0]) and np.array_equal(hb[0][1], hb[1][1])


def test_fused_inner_products_eq12(fd, orc):
    """fdemri_sum_inner (Eq. 12) against the oracle: the oracle's own waveform, its own inner product.
    Data = the oracle-independent seeded noise + a scaled copy of a *different* small waveform; weights random.
    Checked with and without writing the waveform, and bit-for-bit reproducible."""
    import torch
    w = workload(1)
    freq = w.freq_array()
    ref = oracle_c(orc, w, freq)
    rng = np.random.default_rng(11)
    n = w.n_freq
    scale = np.abs(ref["hplus"]).max()
    dplus = scale * (rng.standard_normal(n) + 1j * rng.standard_normal(n))
    dcross = scale * (rng.standard_normal(n) + 1j * rng.standard_normal(n))
    weight = rng.uniform(0.2, 3.0, n)
    want_hh, want_dh = orc.inner(ref["hplus"], ref["hcross"], dplus, dcross, weight)
    want_hh1, _ = orc.inner(ref["hplus"], ref["hcross"])
    wf = fd.waveform_from_workload(w)
    dev = wf.dev
    t_w = torch.from_numpy(weight).to(dev)
    t_dp = torch.from_numpy(np.ascontiguousarray(dplus).view(np.float64).reshape(n, 2)).to(dev)
    t_dx = torch.from_numpy(np.ascontiguousarray(dcross).view(np.float64).reshape(n, 2)).to(dev)
    out = torch.zeros((1, 4), dtype=torch.float64, device=dev)
    # (1) inner products only: no waveform leaves the kernel
    fd.fdemri_sum_inner(wf.plan, w.theta, w.phi, out, weight=t_w, data_plus=t_dp, data_cross=t_dx)
    torch.cuda.synchronize()
    o1 = out.cpu().numpy()[0].copy()
    assert abs(o1[0] - want_hh) <= 1e-10 * want_hh
    assert abs(complex(o1[1], o1[2]) - want_dh) <= 1e-10 * np.sqrt(want_hh * orc.inner(dplus, dcross, w=weight)[0])
    # (2) with the waveform written as well: same numbers bit for bit, waveform as in fdemri_sum
    out2 = torch.zeros_like(out)
    fd.fdemri_sum_inner(wf.plan, w.theta, w.phi, out2, weight=t_w, data_plus=t_dp, data_cross=t_dx, hplus=wf.hplus,
                        hcross=wf.hcross)
    hp, hx = wf.result()
    assert np.array_equal(out2.cpu().numpy()[0], o1)
    check(hp[0], hx[0], ref, "config1 via fdemri_sum_inner")
    # (3) w = 1, no data: <h|h> = sum |h|^2
    out3 = torch.zeros_like(out)
    fd.fdemri_sum_inner(wf.plan, w.theta, w.phi, out3)
    torch.cuda.synchronize()
    o3 = out3.cpu().numpy()[0]
    assert abs(o3[0] - want_hh1) <= 1e-10 * want_hh1 and o3[1] == 0.0 and o3[2] == 0.0
    # (4) Hann window as the 3-point frequency-domain filter (L145), including the bins at warp and tile borders
    want_hh4, want_dh4 = orc.inner(ref["hplus"], ref["hcross"], dplus, dcross, weight, hann=True)
    out4 = torch.zeros_like(out)
    fd.fdemri_sum_inner(wf.plan, w.theta, w.phi, out4, weight=t_w, data_plus=t_dp, data_cross=t_dx, hann=True)
    torch.cuda.synchronize()
    o4 = out4.cpu().numpy()[0]
    assert abs(o4[0] - want_hh4) <= 1e-10 * want_hh4 and abs(want_hh4 - want_hh) > 1e-3 * want_hh
    assert abs(complex(o4[1], o4[2]) - want_dh4) <= 1e-10 * np.sqrt(want_hh4 * orc.inner(dplus, dcross, w=weight)[0])
    print(f"[parity] fused inner products, Hann filter: <h|h> rel {abs(o4[0] - want_hh4) / want_hh4:.2e}, "
          f"<d|h> rel {abs(complex(o4[1], o4[2]) - want_dh4) / abs(want_dh4):.2e}")
    print(f"[parity] fused inner products: <h|h> rel {abs(o1[0] - want_hh) / want_hh:.2e}, "
          f"<d|h> rel {abs(complex(o1[1], o1[2]) - want_dh) / abs(want_dh):.2e}")
    wf.close()


def test_fused_inner_ragged_grid_with_hann(fd, orc):
    """Ragged grid (20001 bins: the last warp range and the last tile are partial) with the Hann filter and w = 1."""
    import torch
    from paper_2307_12585_b200 import synth
    w = synth.small_case(seed=7, n_knots=5, n_freq=20001)
    ref = oracle_c(orc, w, w.freq_array())
    rng = np.random.default_rng(3)
    d = np.abs(ref["hplus"]).max() * (rng.standard_normal((2, w.n_freq)) + 1j * rng.standard_normal((2, w.n_freq)))
    wf = fd.waveform_from_workload(w)
    t_d = [torch.from_numpy(np.ascontiguousarray(x).view(np.float64).reshape(-1, 2)).to(wf.dev) for x in d]
    out = torch.zeros((1, 4), dtype=torch.float64, device=wf.dev)
    for hann in (False, True):
        want_hh, want_dh = orc.inner(ref["hplus"], ref["hcross"], d[0], d[1], hann=hann)
        fd.fdemri_sum_inner(wf.plan, w.theta, w.phi, out, data_plus=t_d[0], data_cross=t_d[1], hann=hann)
        torch.cuda.synchronize()
        o = out.cpu().numpy()[0]
        assert abs(o[0] - want_hh) <= 1e-10 * want_hh
        assert abs(complex(o[1], o[2]) - want_dh) <= 1e-10 * np.sqrt(want_hh * orc.inner(d[0], d[1])[0])
    wf.close()


def test_random_small_cases_sweep(fd, orc):
    """Twenty seeded small cases with random knot counts, mode sets (m = 0, negative n, high l), grids (offset f0,
    ragged sizes), angles and with/without a turnover: per-bin parity, evaluation counts (P9) and exact zeros outside
    the support (P8) on every one of them."""
    from paper_2307_12585_b200 import synth
    rng = np.random.default_rng(20230712)
    worst, newton = 0.0, 0
    for case in range(20):
        n_knots = int(rng.integers(4, 40))
        n_modes = int(rng.integers(1, 9))
        modes = []
        for _ in range(n_modes):
            l = int(rng.integers(2, 11))
            modes.append((l, int(rng.integers(0, l + 1)), int(rng.integers(-6, 7))))
        n_freq = int(rng.integers(500, 40000))
        w = synth.small_case(seed=100 + case, n_knots=n_knots, n_freq=n_freq, modes=tuple(modes),
                             turnover=bool(case & 1))
        if case % 3 == 0:
            w.f0 = float(rng.uniform(0.0, 2e-3))
        w.theta, w.phi = float(rng.uniform(0.05, 3.0)), float(rng.uniform(-3.0, 3.0))
        wf = fd.waveform_from_workload(w)
        wf.sum(w.theta, w.phi)
        hp, hx = wf.result()
        st = wf.stats()
        assert st["status"] == 0 and (st["flags"] & ~8) == 0     # (8 = FDEMRI_BAD_NEWTON: counted below)
        newton += bool(st["flags"] & 8)
        ref = oracle_c(orc, w, w.freq_array())
        assert st["n_evals"] == ref["n_evals"], (case, modes)
        if ref["n_evals"] == 0:
            assert not hp.any() and not hx.any()
        else:
            keep = ref["ambiguous"] == 0
            assert (~keep).sum() <= MAX_AMBIGUOUS
            err = max_rel_err(hp[0], hx[0], ref["hplus"], ref["hcross"], mask=keep)
            zero = (ref["nterms"] == 0) & keep
            assert np.all(hp[0][zero] == 0) and np.all(hx[0][zero] == 0)
            assert err <= TOL_BIN, (case, modes, err)
            worst = max(worst, err)
        wf.close()
    print(f"[parity] 20 random small cases: worst max|dh|/max|h| = {worst:.3e}; iteration cap reported in {newton} of them")
    assert newton == 0


def test_random_wide_sweep_both_kernels(fd, orc):
    """Eighty seeded cases wider than the sweep above -- up to 24 modes (repeats allowed), 4 to 120 knots, 300 to 80 000 bins,
    offset grids -- through BOTH sum kernels: per-bin parity on every bin the oracle does not mark boundary-ambiguous (R8),
    exact zeros outside the support, no flag raised, and evaluation counts that differ from the oracle's by at most the
    pair of roots an ambiguous bin may gain or lose.  With many voices that have a turnover, more than MAX_AMBIGUOUS bins
    of a waveform can sit within 16 ulp of an extremum value; the allowance here is one per voice and sign."""
    from paper_2307_12585_b200 import synth
    rng = np.random.default_rng(230712585)
    worst, n_amb, n_ev = 0.0, 0, 0
    for case in range(80):
        n_knots = int(rng.choice([rng.integers(4, 40), rng.integers(40, 121)]))
        modes = []
        for _ in range(int(rng.integers(1, 25))):
            l = int(rng.integers(2, 11))
            modes.append((l, int(rng.integers(0, l + 1)), int(rng.integers(-8, 9))))
        n_freq = int(rng.choice([rng.integers(300, 5000), rng.integers(5000, 80000)]))
        w = synth.small_case(seed=3000 + case, n_knots=n_knots, n_freq=n_freq, modes=tuple(modes), turnover=bool(rng.integers(0, 2)))
        if case % 3 == 0:
            w.f0 = float(rng.uniform(0.0, 2e-3))
        w.theta, w.phi = float(rng.uniform(0.05, 3.0)), float(rng.uniform(-3.0, 3.0))
        ref = oracle_c(orc, w, w.freq_array())
        keep = ref["ambiguous"] == 0
        amb = int((~keep).sum())
        assert amb <= 2 * len(modes), (case, amb)
        zero = (ref["nterms"] == 0) & keep
        for flag in (fd.FDEMRI_FLAG_TILE_MAJOR, fd.FDEMRI_FLAG_BIN_MAJOR):
            wf = fd.waveform_from_workload(w, flags=flag)
            wf.sum(w.theta, w.phi)
            hp, hx = wf.result()
            st = wf.stats()
            wf.close()
            assert st["status"] == 0 and st["flags"] == 0, (case, flag, st["flags"])
            assert abs(st["n_evals"] - ref["n_evals"]) <= 2 * amb, (case, flag, st["n_evals"], ref["n_evals"], amb)
            if ref["n_evals"] == 0:
                assert not hp.any() and not hx.any()
                continue
            err = max_rel_err(hp[0], hx[0], ref["hplus"], ref["hcross"], mask=keep)
            assert np.all(hp[0][zero] == 0) and np.all(hx[0][zero] == 0), (case, flag)
            assert err <= TOL_BIN, (case, flag, modes, err)
            worst = max(worst, err)
        n_amb += amb
        n_ev += ref["n_evals"]
    print(f"[parity] 80 random wide cases x 2 kernels ({n_ev:.3g} evaluations): worst max|dh|/max|h| = {worst:.3e}; "
          f"{n_amb} boundary-ambiguous bins in all")


@pytest.mark.parametrize("mode", ["bin", "tile"])
def test_both_sum_kernels_on_the_same_inputs(fd, orc, mode):
    """The bin-major kernel (sparse grids, section 3.3) and the tile-major kernel forced on the same inputs:
    a small turnover case, and config 3 (the 10^4 log-spaced frequencies) -- each against the oracle."""
    from paper_2307_12585_b200 import synth
    flag = fd.FDEMRI_FLAG_BIN_MAJOR if mode == "bin" else fd.FDEMRI_FLAG_TILE_MAJOR
    for label, w in (("small", synth.small_case(seed=2, n_knots=14)), ("config3", workload(3))):
        wf = fd.waveform_from_workload(w, flags=flag)
        wf.sum(w.theta, w.phi)
        hp, hx = wf.result()
        st = wf.stats()
        ref = oracle_c(orc, w, w.freq_array())
        check(hp[0], hx[0], ref, f"{label}, {mode}-major")
        assert st["n_evals"] == ref["n_evals"]
        if mode == "bin":
            assert st["n_pairs"] == ref["n_evals"]            # terms the kernel accumulated = terms of the oracle (P9)
        wf.close()


@pytest.mark.parametrize("mode", ["bin", "tile"])
def test_empty_work_list_every_mode_masked_out(fd, orc, mode):
    """Degenerate case: the mode mask of L60 drops every mode, so the segment -> bin map has no entry and the work list
    is empty.  Both sum kernels must still write every bin (exact zeros, buffers pre-filled with NaN), count no
    evaluation, and the fused inner products of the empty waveform are exactly 0; with the mask removed the same plan
    gives the oracle's waveform again."""
    import torch
    from paper_2307_12585_b200 import synth
    w = synth.small_case(seed=2, n_knots=14)
    flag = fd.FDEMRI_FLAG_BIN_MAJOR if mode == "bin" else fd.FDEMRI_FLAG_TILE_MAJOR
    wf = fd.waveform_from_workload(w, flags=flag)
    keep = torch.zeros((1, w.lmn.shape[0]), dtype=torch.uint8, device=wf.dev)
    fd.fdemri_set_mode_mask(wf.plan, keep)
    wf.build_splines(w.f_phi, w.f_r, w.Phi_phi, w.Phi_r, w.amp)
    wf.hplus.fill_(float("nan")); wf.hcross.fill_(float("nan"))
    wf.sum(w.theta, w.phi)
    hp, hx = wf.result()
    st = wf.stats()
    assert st["n_evals"] == 0 and st["n_pairs"] == 0 and st["flags"] == 0
    assert np.all(hp == 0) and np.all(hx == 0)
    out = torch.full((1, 4), float("nan"), dtype=torch.float64, device=wf.dev)
    fd.fdemri_sum_inner(wf.plan, w.theta, w.phi, out, hann=True)
    torch.cuda.synchronize()
    assert np.all(out.cpu().numpy()[0, :3] == 0.0)
    fd.fdemri_set_mode_mask(wf.plan, None)
    wf.build_splines(w.f_phi, w.f_r, w.Phi_phi, w.Phi_r, w.amp)
    wf.sum(w.theta, w.phi)
    hp, hx = wf.result()
    ref = oracle_c(orc, w, w.freq_array())
    check(hp[0], hx[0], ref, f"small case after removing an all-zero mask, {mode}-major")
    assert wf.stats()["n_evals"] == ref["n_evals"] > 0
    wf.close()


def test_degenerate_constant_frequencies_and_zero_amplitudes(fd, orc):
    """Two degenerate inputs.  (a) f_phi and f_r constant in time: every segment of every voice has F_k = F_{k+1}, so
    under R6 (half-open intervals decided on the knot doubles) no bin belongs to any segment -- no entry, no
    evaluation, exact zeros on both sides (the delta-function limit is not SPA, R10).  (b) A = 0 at every knot: the
    map and the evaluation count are those of the non-zero case, every term is exactly 0."""
    import dataclasses
    from paper_2307_12585_b200 import synth
    w = synth.small_case(seed=2, n_knots=14)
    t = w.t_knots
    wc = dataclasses.replace(w, f_phi=np.full_like(w.f_phi, 2.0e-3), f_r=np.full_like(w.f_r, 1.2e-3),
                             Phi_phi=2 * np.pi * 2.0e-3 * t, Phi_r=2 * np.pi * 1.2e-3 * t)
    wf, hp, hx, st = run_gpu(fd, wc)
    ref = oracle_c(orc, wc, wc.freq_array())
    assert ref["n_evals"] == 0 and st["n_evals"] == 0 and st["flags"] == 0
    assert np.all(hp == 0) and np.all(hx == 0) and np.all(ref["hplus"] == 0)
    wf.close()
    wz = dataclasses.replace(w, amp=np.zeros_like(w.amp))
    wf, hp, hx, st = run_gpu(fd, wz)
    ref = oracle_c(orc, wz, wz.freq_array())
    assert st["n_evals"] == ref["n_evals"] > 0 and st["flags"] == 0
    assert np.all(hp == 0) and np.all(hx == 0) and np.all(ref["hplus"] == 0) and np.all(ref["hcross"] == 0)
    wf.close()


def test_bin_major_config1_and_fused_inner(fd, orc):
    """Config 1 (a dense grid: 4.9e7 evaluations) forced through the bin-major kernel: parity, accumulated-term count,
    and the Eq. 12 inner products formed on the fly from the blocks' accumulators -- with and without the waveform
    buffers, with and without the Hann filter and data (49 310 blocks of 32 bins, the last one ragged)."""
    import torch
    w = workload(1)
    wf = fd.waveform_from_workload(w, flags=fd.FDEMRI_FLAG_BIN_MAJOR)
    ref = oracle_c(orc, w, w.freq_array())
    rng = np.random.default_rng(12)
    n = w.n_freq
    scale = np.abs(ref["hplus"]).max()
    dplus = scale * (rng.standard_normal(n) + 1j * rng.standard_normal(n))
    dcross = scale * (rng.standard_normal(n) + 1j * rng.standard_normal(n))
    weight = rng.uniform(0.2, 3.0, n)
    t_w = torch.from_numpy(weight).to(wf.dev)
    t_dp = torch.from_numpy(np.ascontiguousarray(dplus).view(np.float64).reshape(n, 2)).to(wf.dev)
    t_dx = torch.from_numpy(np.ascontiguousarray(dcross).view(np.float64).reshape(n, 2)).to(wf.dev)
    out = torch.zeros((1, 4), dtype=torch.float64, device=wf.dev)
    fd.fdemri_sum_inner(wf.plan, w.theta, w.phi, out, hann=True, hplus=wf.hplus, hcross=wf.hcross)
    hp, hx = wf.result()
    check(hp[0], hx[0], ref, "config1, bin-major")
    st = wf.stats()
    assert st["n_pairs"] == ref["n_evals"] == st["n_evals"]
    want_hh, _ = orc.inner(ref["hplus"], ref["hcross"], hann=True)
    o_with = out.cpu().numpy()[0].copy()
    assert abs(o_with[0] - want_hh) <= 1e-10 * want_hh
    out.zero_()
    fd.fdemri_sum_inner(wf.plan, w.theta, w.phi, out, hann=True)            # no waveform buffers: same bits
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy()[0], o_with)
    dd = orc.inner(dplus, dcross, w=weight)[0]
    for hann in (False, True):
        want_hh, want_dh = orc.inner(ref["hplus"], ref["hcross"], dplus, dcross, weight, hann=hann)
        fd.fdemri_sum_inner(wf.plan, w.theta, w.phi, out, weight=t_w, data_plus=t_dp, data_cross=t_dx, hann=hann)
        torch.cuda.synchronize()
        o = out.cpu().numpy()[0]
        assert abs(o[0] - want_hh) <= 1e-10 * want_hh
        assert abs(complex(o[1], o[2]) - want_dh) <= 1e-10 * np.sqrt(want_hh * dd)
    wf.close()


def test_config2_every_bin(fd, orc):
    """BASELINE config 2 element by element over all 3 155 816 bins (the oracle needs ~20 s on the box's host cores):
    per-bin parity, mismatch, evaluation count (P9), exact zeros wherever the oracle has no term (P8)."""
    w = workload(2)
    wf, hp, hx, st = run_gpu(fd, w)
    ref = oracle_c(orc, w, w.freq_array())
    check(hp[0], hx[0], ref, "config2, every bin")
    assert st["n_evals"] == ref["n_evals"] and ref["max_roots"] == 2
    wf.close()


def test_segment_with_two_interior_extrema(fd, orc):
    """R5: the paper assumes at most one turnover per spline segment (L105).  A zig-zag f_r through 8 random knots
    (seed 7: one segment's cubic has TWO interior extrema; checked with scipy below) must be summed all the same, on
    its three monotone branches, by both kernels."""
    from helpers import zigzag_case
    w = zigzag_case()
    ref = oracle_c(orc, w, w.freq_array())
    assert ref["max_roots"] >= 3
    for flag in (fd.FDEMRI_FLAG_TILE_MAJOR, fd.FDEMRI_FLAG_BIN_MAJOR):
        wf = fd.waveform_from_workload(w, flags=flag)
        wf.sum(w.theta, w.phi)
        hp, hx = wf.result()
        st = wf.stats()
        assert st["flags"] == 0 and st["n_evals"] == ref["n_evals"]
        check(hp[0], hx[0], ref, f"two interior extrema in a segment (flags={flag})")
        wf.close()


def test_table2_grid_4yr(fd, orc):
    """The grid of the paper's Table 2 (T = 4 yr, dt = 10 s: N_f = 6 311 631 bins) with the full
    3843-mode content on a 4-yr plunging trajectory: sampled bins against the oracle, properties at full size."""
    from paper_2307_12585_b200 import synth
    lmn = synth.mode_list(2, 10, lambda l: range(0, l + 1), 30)
    w = synth._single("table2-grid", 7, 2e6, 10.0, 0.4, 4.0, 150, lmn, "n4l")
    assert w.n_freq == 6311631
    wf, hp, hx, st = run_gpu(fd, w)
    idx = _sampled_bins(w.n_freq, 4000, 5, hi_frac=0.2)
    ref = oracle_c(orc, w, w.freq_array()[idx])
    scale = max(np.abs(hp[0]).max(), np.abs(hx[0]).max())
    keep = ref["ambiguous"] == 0
    err = max(np.abs(hp[0][idx] - ref["hplus"])[keep].max(), np.abs(hx[0][idx] - ref["hcross"])[keep].max()) / scale
    mm = one_minus_overlap(hp[0][idx][keep], hx[0][idx][keep], ref["hplus"][keep], ref["hcross"][keep])
    print(f"[parity] Table-2 grid (6 311 631 bins, {st['n_evals']:.4g} evaluations, {st['n_pairs']} pairs): {err:.3e}, mismatch {mm:.3e}")
    assert err <= TOL_BIN and mm <= TOL_MISMATCH and st["flags"] == 0
    assert hp[0][0] == 0 and np.all(hp[0][int(0.5 * w.n_freq):] == 0) and np.all(np.isfinite(hp[0]))
    wf.close()


def test_mode_selection_feeds_the_sum(fd, orc):
    """fdemri_select_modes against oracle.select_modes (modes whose decision hinges
    on the rounding of the total are left out of the comparison), then the masked sum against the oracle run on the
    selected mode list only."""
    import torch
    import oracle
    w = workload(1)
    amp = w.amp[0]
    wf = fd.Waveform(w.lmn, w.t_knots, w.n_freq, freqs=w.freqs, f0=w.f0, df=w.df)
    d_amp = torch.from_numpy(np.ascontiguousarray(w.amp)).to(wf.dev)
    keep = torch.zeros((1, w.lmn.shape[0]), dtype=torch.uint8, device=wf.dev)
    n_keep = torch.zeros(1, dtype=torch.int32, device=wf.dev)
    power = amp[..., 0] ** 2 + amp[..., 1] ** 2
    for eps in (0.0, 1e-5, 1e-2):
        fd.fdemri_select_modes(wf.plan, d_amp, eps, keep, n_keep)
        torch.cuda.synchronize()
        got = keep.cpu().numpy()[0].astype(bool)
        want, total = oracle.select_modes(amp, eps)
        margin = np.min(np.abs(power - eps * total[None, :]) / total[None, :], axis=1)     # distance from the threshold
        sure = margin > 1e-12
        assert np.array_equal(got[sure], want[sure]) and sure.sum() >= len(sure) - 2
        assert int(n_keep.item()) == int(got.sum())
        if eps == 0.0:
            assert got.all()
    assert 0 < got.sum() < len(got)                               # eps = 1e-2 drops some of the 252 modes
    # the masked sum = the oracle on the selected modes alone
    fd.fdemri_set_mode_mask(wf.plan, keep)
    wf.build_splines(w.f_phi, w.f_r, w.Phi_phi, w.Phi_r, w.amp)
    wf.sum(w.theta, w.phi)
    hp, hx = wf.result()
    st = wf.stats()
    sel = np.flatnonzero(got)
    ref = orc.waveform(w.lmn[sel], w.t_knots[0], w.f_phi[0], w.f_r[0], w.Phi_phi[0], w.Phi_r[0], amp[sel], w.freq_array(),
                       w.theta, w.phi)
    check(hp[0], hx[0], ref, f"config1 with mode selection eps = 1e-2 ({len(sel)} of {len(got)} modes)")
    assert st["n_evals"] == ref["n_evals"]
    fd.fdemri_set_mode_mask(wf.plan, None)
    wf.close()


def test_many_knots(fd, orc):
    """400 knots: the cyclic-reduction solvers run with 416 threads and more than 48 KB of shared memory (the plan limit
    is 512 knots); level B of the splines (phase increments against the oracle's long-double build) and level C."""
    from paper_2307_12585_b200 import synth
    w = synth.small_case(seed=11, n_knots=400, n_freq=20000)
    wf, hp, hx, st = run_gpu(fd, w)
    ref = oracle_c(orc, w, w.freq_array())
    check(hp[0], hx[0], ref, "400 knots")
    assert st["n_evals"] == ref["n_evals"]
    hi, lo, am = wf.coeffs()
    ohi, olo = orc.build_splines(w.t_knots[0], np.stack([w.f_phi[0], w.f_r[0], w.Phi_phi[0], w.Phi_r[0]]))
    h = np.diff(w.t_knots[0])
    dco = (hi[0] - ohi) + (lo[0] - olo)
    for c in (2, 3):
        inc = np.abs(dco[c, :, 1] * h) + np.abs(dco[c, :, 2] * h ** 2) + np.abs(dco[c, :, 3] * h ** 3)
        assert inc.max() < 1e-12, f"phase-increment deviation {inc.max()} rad"
    wf.close()


def test_tile_major_merged_passes_short_segments(fd, orc):
    """Segments much shorter than a consumer warp's 64 bins (300 knots, ~18 bins per segment of the (2,2,0) voice; fewer
    for the slow voices), tile-major forced: every warp range holds several segment boundaries, so the consumers' merged
    passes -- consecutive items with disjoint bins evaluated in one pass, each (lane, slot) with the item that covers its
    bin -- run with runs of two and more items, rising and falling voices, both signs."""
    from paper_2307_12585_b200 import synth
    modes = ((2, 2, 0), (2, 1, -2), (3, 0, 1), (2, 2, -3), (4, 3, 2), (5, 1, -4), (3, 2, -1))
    for seed, nk in ((13, 300), (14, 97)):
        w = synth.small_case(seed=seed, n_knots=nk, n_freq=30000, modes=modes)
        wf = fd.waveform_from_workload(w, flags=fd.FDEMRI_FLAG_TILE_MAJOR)
        wf.sum(w.theta, w.phi)
        hp, hx = wf.result()
        st = wf.stats()
        ref = oracle_c(orc, w, w.freq_array())
        check(hp[0], hx[0], ref, f"short segments, {nk} knots, tile-major")
        assert st["n_evals"] == ref["n_evals"] and st["flags"] == 0
        assert st["n_evals"] / st["n_items"] < 64            # on average several entries per warp range
        again = [x.copy() for x in (hp, hx)]
        wf.sum(w.theta, w.phi)
        hp2, hx2 = wf.result()
        assert np.array_equal(again[0].view(np.uint64), hp2.view(np.uint64)) and np.array_equal(again[1].view(np.uint64), hx2.view(np.uint64))
        wf.close()


@pytest.mark.parametrize("mode", ["bin", "tile"])
def test_explicit_grid_changed_between_builds(fd, orc, mode):
    """Explicit frequency arrays go through a bucket table that the first build after fdemri_set_workspace writes into the
    work space (fdemri_map.cuh).  The array is then replaced IN PLACE by a different one -- other spacing, other range -- and
    the splines rebuilt: the table is stale, every lookup through it is checked against the array and repeated by plain
    search where the check fails, so the result is at parity for the new array (and the counts are the oracle's)."""
    import torch
    from paper_2307_12585_b200 import synth
    w = synth.small_case(seed=21, n_knots=40)
    n = 6000
    grids = [np.geomspace(2e-4, 9e-3, n), np.concatenate([[0.0], np.linspace(1.1e-3, 7e-3, n - 1) ** 1.0]),
             np.sort(np.random.default_rng(5).uniform(5e-4, 8e-3, n))]
    flag = fd.FDEMRI_FLAG_BIN_MAJOR if mode == "bin" else fd.FDEMRI_FLAG_TILE_MAJOR
    wf = fd.Waveform(w.lmn, w.t_knots, n, freqs=grids[0], flags=flag)
    for i, g in enumerate(grids):
        wf.freqs.copy_(torch.from_numpy(g))
        wf.build_splines(w.f_phi, w.f_r, w.Phi_phi, w.Phi_r, w.amp)
        wf.sum(w.theta, w.phi)
        hp, hx = wf.result()
        st = wf.stats()
        ref = orc.waveform(w.lmn, w.t_knots[0], w.f_phi[0], w.f_r[0], w.Phi_phi[0], w.Phi_r[0], w.amp[0], g, w.theta, w.phi)
        check(hp[0], hx[0], ref, f"explicit grid {i} ({mode}-major), table built for grid 0")
        assert st["n_evals"] == ref["n_evals"] and st["flags"] == 0
    wf.close()


# ---- general voices (l, m, k, n) of Eq. 1: fdemri_plan_kerr / fdemri_build_splines_kerr -----------
def test_kerr_voices_small(fd, orc):
    from paper_2307_12585_b200 import synth
    w = synth.small_case_kerr(seed=2, n_knots=14)
    wf, hp, hx, st = run_gpu(fd, w)
    ref = oracle_c(orc, w, w.freq_array())
    check(hp[0], hx[0], ref, "general voices, small")
    assert st["n_evals"] == ref["n_evals"] and st["n_evals"] > 0
    # the two build calls belong to their own kind of plan
    with pytest.raises(fd.FdemriError):
        fd.fdemri_build_splines(wf.plan, *wf._inputs[:5])
    wf.close()
    w0 = synth.small_case(seed=2, n_knots=14)
    wf0 = fd.waveform_from_workload(w0)
    with pytest.raises(fd.FdemriError):
        fd.fdemri_build_splines_kerr(wf0.plan, wf0._inputs[0], wf0._inputs[0], wf0._inputs[1], wf0._inputs[2],
                                     wf0._inputs[2], wf0._inputs[3], wf0._inputs[4])
    wf0.close()


def test_kerr_voices_k_zero_bitwise(fd):
    """k = 0 on every voice: the same bits as the (l, m, n) plan, whatever f_theta holds."""
    import dataclasses
    from paper_2307_12585_b200 import synth
    w = synth.small_case_kerr(seed=4, n_knots=20, n_freq=50000)
    lmkn = w.lmkn.copy()
    lmkn[:, 2] = 0
    wk = dataclasses.replace(w, lmkn=lmkn)
    w0 = dataclasses.replace(w, lmkn=None, f_theta=None, Phi_theta=None)
    _, hpk, hxk, stk = run_gpu(fd, wk)
    _, hp0, hx0, st0 = run_gpu(fd, w0)
    assert np.max(np.abs(hp0)) > 0
    assert np.array_equal(hpk, hp0) and np.array_equal(hxk, hx0)
    assert stk["n_evals"] == st0["n_evals"]


def test_kerr_voices_config1_scale(fd, orc):
    """Config 1's trajectory and grid with eleven polar harmonics per (l, m, n), both sum kernels."""
    from paper_2307_12585_b200 import synth
    w = synth.with_polar_voices(synth.config1(), k_max=5)
    assert w.lmkn.shape == (11 * synth.config1().lmn.shape[0], 4)
    freq = w.freq_array()
    ref = oracle_c(orc, w, freq)
    assert ref["max_roots"] >= 1
    for flags, label in ((0, "tile-major"), (fd.FDEMRI_FLAG_BIN_MAJOR, "bin-major")):
        wf = fd.waveform_from_workload(w, flags=flags)
        wf.sum(w.theta, w.phi)
        hp, hx = wf.result()
        st = wf.stats()
        check(hp[0], hx[0], ref, f"general voices, config 1 x 11 k, {label}")
        assert st["n_evals"] == ref["n_evals"]
        wf.close()


def test_kerr_voices_batch_and_odd_k_weights(fd, orc):
    """Two batch items with different trajectories; voices with odd k and m > 0 (partner sign (-1)^(l+k))."""
    import dataclasses
    from paper_2307_12585_b200 import synth
    modes = ((2, 2, 1, 0), (2, 1, -1, 1), (3, 2, 3, -2), (3, 3, -3, 1), (4, 1, 2, 0), (2, 0, 1, -1))
    a = synth.small_case_kerr(seed=8, n_knots=16, modes=modes)
    b = synth.small_case_kerr(seed=9, n_knots=16, modes=modes)
    cat = lambda x, y: np.concatenate([x, y], axis=0)
    w = dataclasses.replace(a, t_knots=cat(a.t_knots, b.t_knots), f_phi=cat(a.f_phi, b.f_phi), f_r=cat(a.f_r, b.f_r),
                            Phi_phi=cat(a.Phi_phi, b.Phi_phi), Phi_r=cat(a.Phi_r, b.Phi_r), amp=cat(a.amp, b.amp),
                            f_theta=cat(a.f_theta, b.f_theta), Phi_theta=cat(a.Phi_theta, b.Phi_theta))
    wf, hp, hx, st = run_gpu(fd, w)
    tot = 0
    for i in range(2):
        ref = oracle_c(orc, w, w.freq_array(), b=i)
        check(hp[i], hx[i], ref, f"general voices, batch item {i}")
        tot += ref["n_evals"]
    assert st["n_evals"] == tot
    wf.close()


def test_kerr_voices_selection_and_fused_inner(fd, orc):
    """General voices through the rest of the path: mode selection (L60; in the paper's words over |A_lmkn|^2) feeding
    the work list, then the Eq. 12 inner products with the Hann filter formed on the fly."""
    import torch
    import oracle
    from paper_2307_12585_b200 import synth
    w = synth.with_polar_voices(synth.small_case(seed=12, n_knots=18, n_freq=40000,
                                                 modes=((2, 2, 0), (2, 1, -1), (3, 2, 1), (3, 0, 2), (4, 4, -2))), k_max=3)
    amp = w.amp[0]
    wf = fd.Waveform(w.lmkn, w.t_knots, w.n_freq, freqs=w.freqs, f0=w.f0, df=w.df)
    d_amp = torch.from_numpy(np.ascontiguousarray(w.amp)).to(wf.dev)
    keep = torch.zeros((1, w.lmkn.shape[0]), dtype=torch.uint8, device=wf.dev)
    n_keep = torch.zeros(1, dtype=torch.int32, device=wf.dev)
    eps = 3e-3
    fd.fdemri_select_modes(wf.plan, d_amp, eps, keep, n_keep)
    torch.cuda.synchronize()
    got = keep.cpu().numpy()[0].astype(bool)
    want, total = oracle.select_modes(amp, eps)
    power = amp[..., 0] ** 2 + amp[..., 1] ** 2
    sure = np.min(np.abs(power - eps * total[None, :]) / total[None, :], axis=1) > 1e-12
    assert np.array_equal(got[sure], want[sure]) and 0 < got.sum() < len(got)
    fd.fdemri_set_mode_mask(wf.plan, keep)
    wf.build_splines(w.f_phi, w.f_r, w.Phi_phi, w.Phi_r, w.amp, f_theta=w.f_theta, Phi_theta=w.Phi_theta)
    sel = np.flatnonzero(got)
    ref = orc.waveform_kerr(w.lmkn[sel], w.t_knots[0], w.f_phi[0], w.f_theta[0], w.f_r[0], w.Phi_phi[0], w.Phi_theta[0],
                            w.Phi_r[0], amp[sel], w.freq_array(), w.theta, w.phi)
    rng = np.random.default_rng(5)
    d = np.abs(ref["hplus"]).max() * (rng.standard_normal((2, w.n_freq)) + 1j * rng.standard_normal((2, w.n_freq)))
    t_d = [torch.from_numpy(np.ascontiguousarray(x).view(np.float64).reshape(-1, 2)).to(wf.dev) for x in d]
    out = torch.zeros((1, 4), dtype=torch.float64, device=wf.dev)
    fd.fdemri_sum_inner(wf.plan, w.theta, w.phi, out, data_plus=t_d[0], data_cross=t_d[1], hann=True, hplus=wf.hplus,
                        hcross=wf.hcross)
    hp, hx = wf.result()
    check(hp[0], hx[0], ref, f"general voices, {len(sel)} of {len(got)} selected")
    assert wf.stats()["n_evals"] == ref["n_evals"]
    want_hh, want_dh = orc.inner(ref["hplus"], ref["hcross"], d[0], d[1], hann=True)
    o = out.cpu().numpy()[0]
    assert abs(o[0] - want_hh) <= 1e-10 * want_hh
    assert abs(complex(o[1], o[2]) - want_dh) <= 1e-10 * np.sqrt(want_hh * orc.inner(d[0], d[1])[0])
    wf.close()


def test_step_is_capturable_in_a_cuda_graph(fd, orc):
    """build_splines + sum enqueue only (kernels, memsets, one small copy, an event fork/join onto the plan's side
    stream): the sequence captures into a CUDA graph, and a replay on fresh inputs gives the bits of the stream launch."""
    import torch
    from paper_2307_12585_b200 import synth
    w = synth.small_case(seed=13, n_knots=20, n_freq=40000)
    wf = fd.waveform_from_workload(w)
    ins = wf._inputs
    s = torch.cuda.Stream()

    def step():
        fd.fdemri_build_splines(wf.plan, *ins)
        fd.fdemri_sum(wf.plan, w.theta, w.phi, wf.hplus, wf.hcross)

    with torch.cuda.stream(s):
        step()
    hp0, hx0 = wf.result()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        step()
    # new amplitudes in the captured input buffer: the replay must follow them
    ins[4].mul_(-2.0)
    wf.hplus.zero_(); wf.hcross.zero_()
    g.replay()
    hp1, hx1 = wf.result()
    assert np.array_equal(hp1, -2.0 * hp0) and np.array_equal(hx1, -2.0 * hx0)
    ref = oracle_c(orc, w, w.freq_array())
    check(hp1[0] / -2.0, hx1[0] / -2.0, ref, "graph replay")
    del g
    wf.close()


@pytest.mark.parametrize("mode", ["tile", "bin"])
def test_guard_bands_and_garbage_in_the_work_space(fd, orc, mode):
    """compute-sanitizer is closed on this pool, so the library is checked with means of its own.  (memcheck) the work
    space and both output buffers sit between guard bands of a known byte pattern, which must be intact after build +
    sum + fused inner products on three cases (small turnover case, the zig-zag with a two-extrema segment, 2000 voices
    in one tile / block -- more than the scan queues hold); (initcheck) the work space is filled with garbage (0xFF: NaN
    as doubles, -1 as integers) or with zeros before the plan touches it, and both runs must give the same bits, equal to
    the oracle within the bar: nothing is read before it is written."""
    import torch
    from helpers import zigzag_case
    from paper_2307_12585_b200 import synth
    flag = fd.FDEMRI_FLAG_BIN_MAJOR if mode == "bin" else fd.FDEMRI_FLAG_TILE_MAJOR
    many = synth.small_case(seed=3, n_knots=6, n_freq=3000, modes=((2, 2, 0),), turnover=False)
    many.f0 = 4.0e-3
    many.lmn = np.repeat(many.lmn, 2000, axis=0)
    many.amp = np.ascontiguousarray(np.repeat(many.amp, 2000, axis=1))
    G = 1 << 16                                                   # guard bytes on either side
    for label, w in (("small", synth.small_case(seed=2, n_knots=14)), ("zigzag", zigzag_case()), ("2000 voices", many)):
        ref = oracle_c(orc, w, w.freq_array())
        results = []
        for fill in (0xFF, 0x00):
            wf = fd.Waveform(w.lmn, w.t_knots, w.n_freq, freqs=w.freqs, f0=w.f0, df=w.df, flags=flag)
            need = fd.fdemri_workspace_bytes(wf.plan)
            raw = torch.full((need + 2 * G + 512,), 0xA5, dtype=torch.uint8, device=wf.dev)
            off = G + ((-(raw.data_ptr() + G)) % 256)
            raw[off:off + need] = fill
            wf.ws, wf.ws_view = raw, raw[off:off + need]
            fd.fdemri_set_workspace(wf.plan, wf.ws_view)
            nout = w.n_freq * 2
            obuf = torch.full((2 * nout + 3 * (G // 8),), float("inf"), dtype=torch.float64, device=wf.dev)
            g8 = G // 8
            hp = obuf[g8:g8 + nout].view(1, w.n_freq, 2)
            hx = obuf[2 * g8 + nout:2 * g8 + 2 * nout].view(1, w.n_freq, 2)
            wf.build_splines(w.f_phi, w.f_r, w.Phi_phi, w.Phi_r, w.amp)
            fd.fdemri_sum(wf.plan, w.theta, w.phi, hp, hx)
            inner = torch.zeros((1, 4), dtype=torch.float64, device=wf.dev)
            fd.fdemri_sum_inner(wf.plan, w.theta, w.phi, inner, hann=True, hplus=hp, hcross=hx)
            torch.cuda.synchronize()
            assert bool((raw[:off] == 0xA5).all()) and bool((raw[off + need:] == 0xA5).all()), f"{label}: work-space guard"
            guards = torch.cat([obuf[:g8], obuf[g8 + nout:2 * g8 + nout], obuf[2 * g8 + 2 * nout:]])
            assert bool(torch.isinf(guards).all()), f"{label}: output guard"
            a = hp.cpu().numpy().view(np.complex128)[0, :, 0]
            b = hx.cpu().numpy().view(np.complex128)[0, :, 0]
            check(a, b, ref, f"{label}, {mode}-major, work space pre-filled with {fill:#04x}")
            assert wf.stats()["n_evals"] == ref["n_evals"]
            results.append((a.copy(), b.copy(), inner.cpu().numpy().copy()))
            wf.close()
        for x, y in zip(results[0], results[1]):
            assert np.array_equal(x.view(np.uint64) if x.dtype != np.float64 else x, y.view(np.uint64) if y.dtype != np.float64 else y)


def _cumulative_margin(amp, eps):
    """Modes whose cumulative-cut decision is clear at every time step: |sum before the mode - (1 - eps) total| > 1e-12 total."""
    power = amp[..., 0] ** 2 + amp[..., 1] ** 2
    sure = np.ones(power.shape[0], dtype=bool)
    for k in range(power.shape[1]):
        order = np.argsort(-power[:, k], kind="stable")
        cum = np.cumsum(power[order, k])
        before = np.concatenate([[0.0], cum[:-1]])
        sure[order[np.abs(before - (1.0 - eps) * cum[-1]) <= 1e-12 * cum[-1]]] = False
    return sure


def test_mode_selection_cumulative_cut(fd, orc):
    """The second reading of L60 (R15 (b)): fdemri_select_modes_rule(FDEMRI_SELECT_CUMULATIVE) -- a descending sort
    and a cumulative sum per (item, time step) on the device -- against oracle.select_modes(rule="cumulative") on config 1
    (252 modes) and on config 2's amplitudes (3843 modes, 150 time steps), two batch items with different amplitudes; the
    two readings differ; the cumulative mask feeds the sum like the other one."""
    import torch
    import oracle
    for idx in (1, 2):
        w = workload(idx)
        amp2 = np.stack([w.amp[0], w.amp[0][::-1] * 0.5 + 0.1 * w.amp[0]])          # a second item with other amplitudes
        tk = np.repeat(w.t_knots, 2, axis=0)
        wf = fd.Waveform(w.lmn, tk, 4096, f0=0.0, df=w.df)
        d_amp = torch.from_numpy(np.ascontiguousarray(amp2)).to(wf.dev)
        keep = torch.zeros((2, w.lmn.shape[0]), dtype=torch.uint8, device=wf.dev)
        n_keep = torch.zeros(2, dtype=torch.int32, device=wf.dev)
        for eps in (1e-5, 1e-2, 0.3):
            fd.fdemri_select_modes_rule(wf.plan, d_amp, eps, fd.FDEMRI_SELECT_CUMULATIVE, keep, n_keep)
            torch.cuda.synchronize()
            for b in range(2):
                got = keep.cpu().numpy()[b].astype(bool)
                want, _ = oracle.select_modes(amp2[b], eps, rule="cumulative")
                sure = _cumulative_margin(amp2[b], eps)
                assert np.array_equal(got[sure], want[sure]) and sure.sum() >= len(sure) - 3, (idx, eps, b)
                assert int(n_keep.cpu().numpy()[b]) == int(got.sum())
                own, _ = oracle.select_modes(amp2[b], eps, rule="own")
                assert want.sum() >= own.sum()
            print(f"[select] config {idx} amplitudes, eps = {eps}: cumulative cut keeps {int(got.sum())} of {len(got)} modes "
                  f"(own-power rule: {int(own.sum())})")
        wf.close()
    # the mask feeds the sum
    w = workload(1)
    wf = fd.Waveform(w.lmn, w.t_knots, w.n_freq, freqs=w.freqs, f0=w.f0, df=w.df)
    d_amp = torch.from_numpy(np.ascontiguousarray(w.amp)).to(wf.dev)
    keep = torch.zeros((1, w.lmn.shape[0]), dtype=torch.uint8, device=wf.dev)
    n_keep = torch.zeros(1, dtype=torch.int32, device=wf.dev)
    fd.fdemri_select_modes_rule(wf.plan, d_amp, 1e-2, fd.FDEMRI_SELECT_CUMULATIVE, keep, n_keep)
    fd.fdemri_set_mode_mask(wf.plan, keep)
    wf.build_splines(w.f_phi, w.f_r, w.Phi_phi, w.Phi_r, w.amp)
    wf.sum(w.theta, w.phi)
    hp, hx = wf.result()
    sel = np.flatnonzero(keep.cpu().numpy()[0])
    assert 0 < len(sel) < w.lmn.shape[0]
    ref = orc.waveform(w.lmn[sel], w.t_knots[0], w.f_phi[0], w.f_r[0], w.Phi_phi[0], w.Phi_r[0], w.amp[0][sel], w.freq_array(),
                       w.theta, w.phi)
    check(hp[0], hx[0], ref, f"config1 with the cumulative cut at eps = 1e-2 ({len(sel)} of {w.lmn.shape[0]} modes)")
    assert wf.stats()["n_evals"] == ref["n_evals"]
    # more modes than the shared-memory sort takes: the call says so
    big = fd.Waveform(np.repeat(w.lmn, 70, axis=0), w.t_knots, 1024, f0=0.0, df=w.df)
    k2 = torch.zeros((1, 70 * w.lmn.shape[0]), dtype=torch.uint8, device=wf.dev)
    with pytest.raises(fd.FdemriError) as ei:
        fd.fdemri_select_modes_rule(big.plan, d_amp, 1e-2, fd.FDEMRI_SELECT_CUMULATIVE, k2, n_keep)
    assert ei.value.status == 5
    big.close()
    fd.fdemri_set_mode_mask(wf.plan, None)
    wf.close()


# ---- the time-domain voice sum of Eq. 1 / Eq. 2: fdemri_td_sum ---------------------------------
def test_td_sum_parity_and_fd_against_fft_of_td(fd, orc):
    """(1) fdemri_td_sum element by element against the oracle's time-domain sum (fdemri_oracle_td) on a 2^19-sample
    case with nine voices (F < 0, m = 0 and turnover voices among them), on a ragged general-voice case with two batch
    items and per-item angles, and with a mode mask.  (2) On the box, the check the paper makes (L141-147): the
    frequency-domain waveform of fdemri_sum against the FFT of the time-domain one (cuFFT through torch.fft, Eq. 3's sign:
    N dt ifft), mismatch with and without the Hann window, at the levels of the oracle's own convention check P6."""
    import dataclasses
    import torch
    from paper_2307_12585_b200 import synth
    N, dt = 2 ** 19, 10.0
    modes = [(2, 2, 0), (2, 1, 1), (2, 2, -2), (3, 0, 2), (3, 3, -1), (2, 1, -4), (4, 2, 1), (2, 0, -1), (3, 1, -2)]
    w = synth.small_case(seed=3, n_knots=24, n_freq=N // 2 + 1, modes=modes, T_s=N * dt)
    wf = fd.waveform_from_workload(w)
    wf.sum(w.theta, w.phi)
    Hp, Hx = wf.result()
    tp = torch.full((1, N), float("nan"), dtype=torch.float64, device=wf.dev)
    tx = torch.full_like(tp, float("nan"))
    fd.fdemri_td_sum(wf.plan, w.theta, w.phi, N, 0.0, dt, tp, tx)
    torch.cuda.synchronize()
    ref_p, ref_x = orc.td(w.lmn, w.t_knots[0], w.Phi_phi[0], w.Phi_r[0], w.amp[0], N, 0.0, dt, w.theta, w.phi)
    scale = max(np.abs(ref_p).max(), np.abs(ref_x).max())
    err = max(np.abs(tp.cpu().numpy()[0] - ref_p).max(), np.abs(tx.cpu().numpy()[0] - ref_x).max()) / scale
    print(f"[parity] time-domain sum, 2^19 samples x 9 voices: max|dh|/max|h| = {err:.3e}")
    assert err <= TOL_BIN
    # (2) FD against N dt ifft(TD), on the device
    win = 0.5 * (1.0 - torch.cos(2.0 * math.pi * torch.arange(N, dtype=torch.float64, device=wf.dev) / N))
    fft = lambda x: (N * dt * torch.fft.ifft(x)).cpu().numpy()[: N // 2 + 1]
    sl = slice(1, N // 2)
    m_raw = one_minus_overlap(Hp[0][sl], Hx[0][sl], fft(tp[0])[sl], fft(tx[0])[sl])
    filt = lambda H: 0.5 * H[1:-1] - 0.25 * H[:-2] - 0.25 * H[2:]
    m_win = one_minus_overlap(filt(Hp[0]), filt(Hx[0]), fft(tp[0] * win)[1:-1], fft(tx[0] * win)[1:-1])
    print(f"[fd vs fft(td)] mismatch without window {m_raw:.3e}, with the Hann window {m_win:.3e} (paper, one system: 8e-4 -> 4e-6, L147)")
    assert m_raw < 1e-2 and m_win < 2e-3 and m_win < m_raw
    assert one_minus_overlap(np.conj(Hp[0][sl]), Hx[0][sl], fft(tp[0])[sl], fft(tx[0])[sl]) > 0.2
    # with a mode mask: the masked voices are left out of the time-domain sum too
    keep = torch.ones((1, len(modes)), dtype=torch.uint8, device=wf.dev)
    keep[0, 1] = 0; keep[0, 4] = 0
    fd.fdemri_set_mode_mask(wf.plan, keep)
    wf.build_splines(w.f_phi, w.f_r, w.Phi_phi, w.Phi_r, w.amp)
    a = torch.empty((1, 4096), dtype=torch.float64, device=wf.dev); b = torch.empty_like(a)
    fd.fdemri_td_sum(wf.plan, w.theta, w.phi, 4096, 1.0e5, 777.0, a, b)
    torch.cuda.synchronize()
    sel = [i for i in range(len(modes)) if i not in (1, 4)]
    rp, rx = orc.td(w.lmn[sel], w.t_knots[0], w.Phi_phi[0], w.Phi_r[0], w.amp[0][sel], 4096, 1.0e5, 777.0, w.theta, w.phi)
    assert max(np.abs(a.cpu().numpy()[0] - rp).max(), np.abs(b.cpu().numpy()[0] - rx).max()) <= TOL_BIN * scale
    fd.fdemri_set_mode_mask(wf.plan, None)
    wf.close()
    # general voices, two batch items, per-item angles, a grid that starts before t_0 and runs past t_{N-1}
    modes4 = ((2, 2, 1, 0), (2, 1, -1, 1), (3, 2, 3, -2), (3, 3, -3, 1), (4, 1, 2, 0), (2, 0, 1, -1))
    a_ = synth.small_case_kerr(seed=8, n_knots=16, modes=modes4)
    b_ = synth.small_case_kerr(seed=9, n_knots=16, modes=modes4)
    cat = lambda x, y: np.concatenate([x, y], axis=0)
    w2 = dataclasses.replace(a_, t_knots=cat(a_.t_knots, b_.t_knots), f_phi=cat(a_.f_phi, b_.f_phi), f_r=cat(a_.f_r, b_.f_r),
                             Phi_phi=cat(a_.Phi_phi, b_.Phi_phi), Phi_r=cat(a_.Phi_r, b_.Phi_r), amp=cat(a_.amp, b_.amp),
                             f_theta=cat(a_.f_theta, b_.f_theta), Phi_theta=cat(a_.Phi_theta, b_.Phi_theta))
    wf2 = fd.waveform_from_workload(w2)
    ns, t0s, dts = 5001, -3.0e4, 613.7
    th, ph = np.array([0.7, 2.2]), np.array([-1.0, 0.4])
    o1 = torch.empty((2, ns), dtype=torch.float64, device=wf2.dev); o2 = torch.empty_like(o1)
    fd.fdemri_td_sum(wf2.plan, th, ph, ns, t0s, dts, o1, o2)
    torch.cuda.synchronize()
    for i in range(2):
        rp, rx = orc.td(w2.lmkn, w2.t_knots[i], w2.Phi_phi[i], w2.Phi_r[i], w2.amp[i], ns, t0s, dts, float(th[i]), float(ph[i]),
                        Phi_theta=w2.Phi_theta[i])
        sc = max(np.abs(rp).max(), np.abs(rx).max())
        e = max(np.abs(o1.cpu().numpy()[i] - rp).max(), np.abs(o2.cpu().numpy()[i] - rx).max()) / sc
        assert e <= TOL_BIN and np.all(o1.cpu().numpy()[i][rp == 0] == 0) and (rp == 0).sum() > 40
    wf2.close()


def test_interleaved_builds_of_plans_with_different_knot_counts(fd, orc):
    """The dynamic shared-memory limit of the spline kernels is an attribute of the kernel, not of a plan: two live plans
    with 150 and 40 knots (and one with 400), built in turn and again, must all keep working (round-1 advice)."""
    from paper_2307_12585_b200 import synth
    cases = [synth.small_case(seed=21, n_knots=150, n_freq=20000), synth.small_case(seed=22, n_knots=40, n_freq=20000),
             synth.small_case(seed=23, n_knots=400, n_freq=20000)]
    wfs = [fd.Waveform(w.lmn, w.t_knots, w.n_freq, f0=w.f0, df=w.df) for w in cases]
    refs = [oracle_c(orc, w, w.freq_array()) for w in cases]
    for order in ((0, 1, 2), (1, 0, 2), (2, 1, 0)):
        for i in order:
            w, wf = cases[i], wfs[i]
            wf.build_splines(w.f_phi, w.f_r, w.Phi_phi, w.Phi_r, w.amp)
        for i in order:
            w, wf = cases[i], wfs[i]
            wf.sum(w.theta, w.phi)
            hp, hx = wf.result()
            check(hp[0], hx[0], refs[i], f"plan with {w.n_knots} knots, build order {order}")
            assert wf.stats()["n_evals"] == refs[i]["n_evals"]
    for wf in wfs:
        wf.close()
