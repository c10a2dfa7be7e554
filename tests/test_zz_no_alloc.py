"""fdemri_select_modes_static (include/fdemri.h): the mode selection of PAPER.md L60 without a plan, a work space or any
allocation -- its scratch of total powers is a static device array of the library -- against the existing path,
fdemri_select_modes on a plan with a caller-allocated work space, on two calls in a row.

Byte and index work: the bar is bit-exact (keep flags and counts equal), as in the other selection tests.  The file is
named so that pytest collects it last (the suite runs with pytest -x); it passes alone in a fresh process and after the
other GPU tests.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def fd():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2307_12585_b200 as pkg
    return pkg


def _existing_path(fd, w, d_amp, eps):
    """fdemri_select_modes on a plan whose work space the caller allocated."""
    import torch
    wf = fd.Waveform(w.lmn, w.t_knots, w.n_freq, freqs=w.freqs, f0=w.f0, df=w.df)
    n_batch, n_modes = d_amp.shape[0], d_amp.shape[1]
    keep = torch.full((n_batch, n_modes), 7, dtype=torch.uint8, device=wf.dev)
    n_keep = torch.full((n_batch,), -5, dtype=torch.int32, device=wf.dev)
    fd.fdemri_select_modes(wf.plan, d_amp, eps, keep, n_keep)
    torch.cuda.synchronize()
    out = keep.cpu().numpy().copy(), n_keep.cpu().numpy().copy()
    wf.close()
    return out


def test_static_scratch_selection_equals_the_plan_path_twice(fd):
    import torch
    from paper_2307_12585_b200 import synth
    dev = torch.device("cuda:0")
    # call 1: config 1's amplitudes (252 modes, one item); call 2: three parameter sets of config 4 (3843 modes each) with
    # another eps, so that it runs over what call 1 left in the shared scratch
    cases = [(synth.CONFIGS[1](), 1e-2), (synth.config4(items=[3, 10, 500]), 1e-4)]
    want = []
    d_amps = []
    for w, eps in cases:
        d_amp = torch.from_numpy(np.ascontiguousarray(w.amp)).to(dev)
        d_amps.append(d_amp)
        want.append(_existing_path(fd, w, d_amp, eps))
    outs = []
    for d_amp in d_amps:
        n_batch, n_modes = d_amp.shape[0], d_amp.shape[1]
        outs.append((torch.full((n_batch, n_modes), 9, dtype=torch.uint8, device=dev),
                     torch.full((n_batch,), 123, dtype=torch.int32, device=dev)))
    torch.cuda.synchronize()
    free_before = None
    for i, ((w, eps), d_amp, (keep, n_keep)) in enumerate(zip(cases, d_amps, outs)):
        if i == 1:                                    # the first call on a device may load the module; the second may not
            free_before = torch.cuda.mem_get_info(dev)[0]
        fd.fdemri_select_modes_static(d_amp, eps, keep, n_keep)
        torch.cuda.synchronize()
        if i == 1:
            assert torch.cuda.mem_get_info(dev)[0] == free_before, "the call changed the device's free memory"
        got_keep, got_n = keep.cpu().numpy(), n_keep.cpu().numpy()
        assert np.array_equal(got_keep, want[i][0]), f"call {i + 1}: keep flags differ from fdemri_select_modes"
        assert np.array_equal(got_n, want[i][1]) and np.array_equal(got_n, got_keep.sum(axis=1))
        assert 0 < got_keep.sum() < got_keep.size      # the cut is neither empty nor everything
        print(f"[static] call {i + 1}: {got_keep.shape[0]} x {got_keep.shape[1]} modes x {d_amp.shape[2]} knots, eps = {eps}: "
              f"{int(got_keep.sum())} kept, identical to the plan path")
    # the first case once more: same answer after the other sizes went through the scratch
    keep, n_keep = outs[0]
    keep.fill_(3)
    fd.fdemri_select_modes_static(d_amps[0], cases[0][1], keep, n_keep)
    torch.cuda.synchronize()
    assert np.array_equal(keep.cpu().numpy(), want[0][0]) and np.array_equal(n_keep.cpu().numpy(), want[0][1])


def test_static_scratch_limit_is_refused(fd):
    import torch
    dev = torch.device("cuda:0")
    n_knots = 64
    n_batch = fd.FDEMRI_STATIC_MAX_TOTALS // n_knots + 1          # one item too many for the static array
    amp = torch.ones((n_batch, 2, n_knots, 2), dtype=torch.float64, device=dev)
    keep = torch.full((n_batch, 2), 5, dtype=torch.uint8, device=dev)
    n_keep = torch.full((n_batch,), 5, dtype=torch.int32, device=dev)
    with pytest.raises(fd.FdemriError) as e:
        fd.fdemri_select_modes_static(amp, 0.1, keep, n_keep)
    assert e.value.status == 6 and "STATIC_SCRATCH" in str(e.value)
    torch.cuda.synchronize()
    assert bool((keep == 5).all()) and bool((n_keep == 5).all())   # nothing was enqueued
    # at the limit it runs: both modes carry half of the power at every knot
    amp = amp[:n_batch - 1].contiguous()
    keep, n_keep = keep[:n_batch - 1].contiguous(), n_keep[:n_batch - 1].contiguous()
    fd.fdemri_select_modes_static(amp, 0.1, keep, n_keep)
    torch.cuda.synchronize()
    assert bool((keep == 1).all()) and bool((n_keep == 2).all())
