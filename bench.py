#!/usr/bin/env python
"""bench.py -- throughput of the FD EMRI harmonic sum (arXiv:2307.12585) on B200, FP64.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2]

One "step" = one pass of the whole hot path (S0-S4: fdemri_build_splines + fdemri_sum) over one synthetic
waveform of BASELINE.json config 2 (3843 modes, 2 yr, dt = 10 s).  Prints ONE JSON
line.  `value` = waveforms/s with inputs resident in HBM; `e2e` = the same through host buffers (pinned H2D of
the inputs and D2H of both polarisations inside the timed region).  N > 1 (torchrun): independent replicas,
one per GPU, no data-path collective; value = N waveforms / max-over-ranks time.
`--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "waveforms/s, 3843-mode 2-yr FD sum (FP64)"
FLOP_PER_EVAL = 200.0          # SURVEY.md 8(d) / DESIGN.md: algorithmic FP64 flop per mode-bin evaluation
# (DRAM traffic and the executed-flop fraction of the dominant kernel come from an ncu capture, which this program never
# runs under: the line reports null for both and points to the profile that holds them.)
NCU_PROFILE = "profiles/r2_final.md"
KERNELS_PER_STEP = 5           # k_spline_amp, k_spline_shared, k_records | k_weights, k_tile_sum (or k_bin_sum)


def workload_name(idx, w):
    if idx == 2:
        return (f"BASELINE config 2: 3843 modes l=2..10,n=-30..30; M=2e6, e0=0.4, 2 yr, 150 knots; uniform grid "
                f"{w.n_freq} bins (dt=10 s)")
    if idx == 5:
        return (f"general voices (l,m,k,n) of Eq. 1, not a BASELINE config: config 2's trajectory and grid ({w.n_freq} bins) "
                f"with polar harmonics k=-5..5, {w.lmn.shape[0]} voices (SURVEY 8(f) rank 4)")
    return f"BASELINE config {idx}"


def workload_inputs(w):
    """Host arrays in the order the binding keeps them: f_phi, f_r, Phi_phi, Phi_r, amp (, f_theta, Phi_theta)."""
    arrs = [w.f_phi, w.f_r, w.Phi_phi, w.Phi_r, w.amp]
    if w.lmkn is not None:
        arrs += [w.f_theta, w.Phi_theta]
    return [np.ascontiguousarray(a, dtype=np.float64) for a in arrs]


def build_call(fd, wf, ins):
    if wf.polar:
        fp, fr, Pp, Pr, am, ft, Pt = ins
        fd.fdemri_build_splines_kerr(wf.plan, fp, ft, fr, Pp, Pt, Pr, am)
    else:
        fd.fdemri_build_splines(wf.plan, *ins)


def oracle_waveform(orc, w, freq, **kw):
    if w.lmkn is not None:
        return orc.waveform_kerr(w.lmkn, w.t_knots[0], w.f_phi[0], w.f_theta[0], w.f_r[0], w.Phi_phi[0], w.Phi_theta[0],
                                 w.Phi_r[0], w.amp[0], freq, w.theta, w.phi, **kw)
    return orc.waveform(w.lmn, w.t_knots[0], w.f_phi[0], w.f_r[0], w.Phi_phi[0], w.Phi_r[0], w.amp[0], freq,
                        w.theta, w.phi, **kw)


def load_workload(idx):
    from paper_2307_12585_b200 import synth
    return synth.CONFIGS[idx]()


class ClockSampler:
    """SM clock and throttle reasons sampled DURING the timed region (B200_PROFILING.md), through NVML from a
    polling thread (every ~2 ms: the timed region of the default run lasts tens of milliseconds, too short for
    `nvidia-smi -lms`)."""

    def __init__(self, index=0):
        self.index = index
        self.sm, self.reasons, self.mx = [], set(), None
        self.stop_flag = threading.Event()
        self.th = None
        self.err = None

    def _run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.mx = float(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
            names = {"hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
                     "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
                     "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
                     "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4)}
            get_reasons = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or \
                getattr(nv, "nvmlDeviceGetCurrentClocksThrottleReasons")
            while not self.stop_flag.is_set():
                self.sm.append(float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)))
                r = int(get_reasons(h))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
                time.sleep(0.002)
            nv.nvmlShutdown()
        except Exception as e:                              # noqa: BLE001
            self.err = repr(e)

    def start(self):
        self.th = threading.Thread(target=self._run, daemon=True)
        self.th.start()
        time.sleep(0.02)                                    # let NVML initialise before the timed region starts

    def stop(self):
        self.stop_flag.set()
        if self.th:
            self.th.join(timeout=5)
        if not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.mx, "reasons": ["nvml unavailable: %s" % self.err], "samples": 0}
        return {"sm_mhz": float(np.median(self.sm)), "sm_max_mhz": self.mx, "reasons": sorted(self.reasons),
                "samples": len(self.sm)}


def cpu_oracle_sample(w, total_evals, n_bins=500000, seed=0):
    """The oracle as it stands, on a seeded random sample of the covered bins of the same workload."""
    import oracle
    orc = oracle.load()
    rng = np.random.default_rng(seed)
    idx = np.unique(rng.integers(1, int(w.n_freq * 0.36), size=n_bins))
    freq = w.freq_array()[idx]
    t0 = time.perf_counter()
    r = oracle_waveform(orc, w, freq, extra=False)
    dt = time.perf_counter() - t0
    cores = orc.num_threads                                 # read before the one-thread pass below resets it
    frac = r["n_evals"] / float(total_evals) if total_evals else float("nan")
    # one thread, on a smaller sample (single-thread time beside the all-cores one)
    idx1 = idx[:: max(1, len(idx) // 12000)]
    t1 = time.perf_counter()
    r1 = oracle_waveform(orc, w, w.freq_array()[idx1], extra=False, n_threads=1)
    dt1 = time.perf_counter() - t1
    single = {"evals_per_s": r1["n_evals"] / dt1, "waveforms_per_s": (r1["n_evals"] / float(total_evals)) / dt1 if total_evals else None,
              "seconds": dt1, "bins": int(len(idx1))}
    return {"single_thread": single, "value": frac / dt, "unit": "waveforms/s", "cores": cores, "kind": "oracle",
            "sample": f"{len(idx)} random bins of the covered band ({r['n_evals']} of {int(total_evals)} mode-bin "
                      f"evaluations) incl. the oracle's spline build, {dt:.2f} s wall; scaled by evaluation count",
            "evals_per_s": r["n_evals"] / dt, "seconds": dt}


def run_reference(args):
    """--impl reference: the CPU oracle on bounded samples of the workload (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    w = load_workload(args.config)
    import oracle
    orc = oracle.load()
    # evaluation count of the full workload from a coarse oracle pass is too slow; use the count of the sample and
    # the covered-band fraction: report evaluations/s and the waveforms/s it implies with SURVEY's count
    total_evals = 3.299e8 if args.config == 2 else None
    times, evals, cores = [], 0, orc.num_threads
    for i in range(args.warmup + args.steps):
        r = cpu_oracle_sample(w, total_evals or 1.0, n_bins=200000, seed=i)
        cores = r["cores"]
        if i >= args.warmup:
            times.append(r["seconds"]); evals += r["evals_per_s"] * r["seconds"]
    tot = sum(times)
    val = (evals / total_evals) / tot if total_evals else evals / tot
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "waveforms/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / max(1, args.steps),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f80 (x87 long double)",
            "data": "synthetic",
            "config": {"workload": workload_name(args.config, w), "sample": "200000 random bins of the covered band per step"},
            "cpu_baseline": {"value": val, "unit": "waveforms/s", "cores": cores, "kind": "oracle",
                             "sample": "each step: 200000 random bins of the covered band incl. spline build, scaled by "
                                       "evaluation count (3.299e8 per waveform)"},
            "e2e": {"value": val, "unit": "waveforms/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "evals_per_s": evals / tot}
    print(json.dumps(line))


def run_batched(args, fd, fdist, torch, dev, rank, world, local, barrier, quiet=False):
    """BASELINE config 4: many parameter sets, evaluated chunk by chunk in one launch sequence.  A "step" is one
    pass over this rank's share of the items (S1-S4 for every chunk, inputs resident in HBM)."""
    from paper_2307_12585_b200 import synth
    mine = fdist.shard_range(args.items, world, rank)
    chunk = args.chunk
    chunks = [list(mine)[i:i + chunk] for i in range(0, len(mine), chunk)]
    # generate and upload all chunks first (untimed); every input and output stays resident in HBM, the work
    # space is ONE buffer shared by the plans of all chunks (a chunk's sum is enqueued right after its build)
    loads = []
    ws = None
    ws_bytes = 0

    def give_workspace(plan, need):
        nonlocal ws, ws_bytes
        if need > ws_bytes:
            ws = None
            ws_bytes = int(need * 1.25) + (1 << 20)
            ws = torch.empty(ws_bytes // 8 + 64, dtype=torch.float64, device=dev)
            for ld in loads:                                # re-point the plans made so far
                fd.fdemri_set_workspace(ld["plan"], ws_view())
        fd.fdemri_set_workspace(plan, ws_view())

    def ws_view():
        off = (-ws.data_ptr()) % 256
        return ws.view(torch.uint8)[off:off + ws_bytes]

    for ids in chunks:
        w = synth.config4(items=ids)
        t_knots = torch.from_numpy(np.ascontiguousarray(w.t_knots)).to(dev)
        plan = fd.fdemri_plan(w.lmn, w.n_batch, w.n_knots, t_knots, w.n_freq, None, w.f0, w.df, 0)
        dev_in = [torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).to(dev)
                  for a in (w.f_phi, w.f_r, w.Phi_phi, w.Phi_r, w.amp)]
        hp = torch.empty((w.n_batch, w.n_freq, 2), dtype=torch.float64, device=dev)
        hx = torch.empty_like(hp)
        ld = dict(plan=plan, t_knots=t_knots, dev_in=dev_in, hp=hp, hx=hx, theta=w.theta, phi=w.phi)
        give_workspace(plan, fd.fdemri_workspace_bytes(plan))
        fd.fdemri_build_splines(plan, *dev_in)
        st = fd.fdemri_get_stats(plan, check=True)
        ld["n_evals"] = st["n_evals"]
        loads.append(ld)
        del w
    stream = torch.cuda.current_stream()

    def one_pass():
        for ld in loads:
            fd.fdemri_build_splines(ld["plan"], *ld["dev_in"])
            fd.fdemri_sum(ld["plan"], ld["theta"], ld["phi"], ld["hp"], ld["hx"])

    for _ in range(max(1, args.warmup)):
        one_pass()
    torch.cuda.synchronize()
    evals = sum(ld["n_evals"] for ld in loads)
    peak_tf = fd.fdemri_measure_fp64_peak(1 << 16)
    sampler = ClockSampler(local)
    if rank == 0 and not quiet:
        sampler.start()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        one_pass()
    e1.record(stream)
    e1.synchronize()
    barrier()
    clocks = sampler.stop() if (rank == 0 and not quiet) else None
    total_ms = fdist.max_over_ranks(e0.elapsed_time(e1), device=dev)
    all_items = fdist.sum_over_ranks(len(mine), device=dev)
    all_evals = fdist.sum_over_ranks(evals, device=dev)
    if rank == 0:
        secs = total_ms * 1e-3 / args.steps
        achieved = all_evals * FLOP_PER_EVAL / secs * 1e-12 / world
        line = {"metric": "waveforms/s, batched 3843-mode 1-yr FD sums (FP64)", "value": all_items / secs,
                "unit": "waveforms/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": f"BASELINE config 4: first {args.items} of the 1024 seeded parameter sets (M log-uniform "
                                       f"1e5..1e7, e0 0..0.5, T = 1 yr, 100 knots, 3843 modes, 1577909 bins), chunks of {chunk}",
                           "step": "fdemri_build_splines + fdemri_sum per chunk, one launch sequence",
                           "l2": "inputs and outputs of a pass exceed L2", "parallelism": "items sharded over ranks, no collective"},
                "evals_per_step": all_evals, "evals_per_s": all_evals / secs,
                "gpu_launches": KERNELS_PER_STEP * args.steps * len(chunks),
                "roofline": {"bound": "alu", "kernel": "whole pass (k_tile_sum dominates)", "achieved": achieved, "peak": peak_tf,
                             "unit": "TFLOP/s", "frac": achieved / peak_tf, "traffic": None, "flop_per_eval": FLOP_PER_EVAL},
                "clocks": clocks}
        for ld in loads:
            fd.fdemri_destroy(ld["plan"])
        return line
    return None


def measure_single(fd, torch, dev, idx, steps, warmup, flush, latency_reps=0, inner=False):
    """One workload through fdemri_build_splines + fdemri_sum, inputs resident in HBM, L2 flushed between steps.
    Returns the numbers of the line for that workload (no collectives; the caller takes the max over ranks)."""
    w = load_workload(idx)
    wf = fd.Waveform(w.lmkn if w.lmkn is not None else w.lmn, w.t_knots, w.n_freq, freqs=w.freqs, f0=w.f0, df=w.df,
                     device=dev, flags=fd.FDEMRI_FLAG_TIMING)
    host = workload_inputs(w)
    dev_in = [torch.from_numpy(a).to(dev) for a in host]
    stream = torch.cuda.current_stream()

    def step_device():
        build_call(fd, wf, dev_in)
        fd.fdemri_sum(wf.plan, w.theta, w.phi, wf.hplus, wf.hcross)

    for _ in range(max(3, warmup)):
        step_device()
    torch.cuda.synchronize()
    st = wf.stats()
    step_ms, sum_ms, kern_ms = [], [], []
    for _ in range(steps):
        flush.fill_(1.0)
        e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        e0.record(stream)
        build_call(fd, wf, dev_in)
        e1.record(stream)
        fd.fdemri_sum(wf.plan, w.theta, w.phi, wf.hplus, wf.hcross)
        e2.record(stream)
        e2.synchronize()
        step_ms.append(e0.elapsed_time(e2))
        sum_ms.append(e1.elapsed_time(e2))
        kern_ms.append(fd.fdemri_get_kernel_ms(wf.plan))
    out = {"w": w, "wf": wf, "host": host, "dev_in": dev_in, "stats": st, "step_ms": step_ms, "sum_ms": sum_ms,
           "kern_ms": kern_ms, "bin_major": w.n_freq < 256 * (w.n_knots - 1)}
    if latency_reps:
        # one waveform at a time, nothing overlapped: pinned H2D of the inputs, S0-S4, pinned D2H of both polarisations,
        # synchronise -- what a sampler that needs the waveform on the host before its next call sees
        pin_in = [torch.from_numpy(a).pin_memory() for a in host]
        pin_out = [torch.empty(wf.hplus.shape, dtype=torch.float64).pin_memory() for _ in range(2)]
        lat = []
        for i in range(latency_reps + 2):
            flush.fill_(1.0)
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0 = time.perf_counter()
            a.record(stream)
            for d, p_ in zip(dev_in, pin_in):
                d.copy_(p_, non_blocking=True)
            build_call(fd, wf, dev_in)
            fd.fdemri_sum(wf.plan, w.theta, w.phi, wf.hplus, wf.hcross)
            pin_out[0].copy_(wf.hplus, non_blocking=True)
            pin_out[1].copy_(wf.hcross, non_blocking=True)
            b.record(stream)
            b.synchronize()
            wall = (time.perf_counter() - t0) * 1e3
            if i >= 2:
                lat.append((a.elapsed_time(b), wall))
        out["e2e_latency_ms"] = float(np.median([x[0] for x in lat]))
        out["e2e_latency_wall_ms"] = float(np.median([x[1] for x in lat]))
    return out


def sub_record(fd, m, peak_tf, world=1):
    """The entry of `configs` for one workload."""
    k_ms = float(np.mean(m["kern_ms"]))
    ms = float(np.mean(m["step_ms"]))
    n_evals = m["stats"]["n_evals"]
    achieved = n_evals * FLOP_PER_EVAL / (k_ms * 1e-3) * 1e-12
    rec = {"ms_per_step": ms, "waveforms_per_s": world * 1e3 / ms, "evals_per_waveform": n_evals,
           "evals_per_s": world * n_evals / (ms * 1e-3), "ms_build_splines": ms - float(np.mean(m["sum_ms"])),
           "ms_sum": float(np.mean(m["sum_ms"])), "kernel": "k_bin_sum" if m["bin_major"] else "k_tile_sum", "kernel_ms": k_ms,
           "roofline": {"bound": "alu", "achieved": achieved, "peak": peak_tf, "unit": "TFLOP/s", "frac": achieved / peak_tf},
           "steps": len(m["step_ms"])}
    if "e2e_latency_ms" in m:
        rec["e2e_latency_ms"] = m["e2e_latency_ms"]
        rec["e2e_latency_wall_ms"] = m["e2e_latency_wall_ms"]
    return rec


def issue_model(fd):
    """The issue-cost microbenchmarks of profiles/r2_dispatch_model.md, in SM cycles at the clock NVML reports."""
    names = ["dfma_1reg", "dfma_2reg", "dfma_2reg_cbank", "dfma_3reg", "dmul_2reg", "dadd_2reg", "dfma_2reg+2int",
             "dfma_2reg+4int", "dfma_1reg+ffma", "dfma_3reg+ffma"]
    return {n: fd.fdemri_measure_issue_ns(i) for i, n in enumerate(names)}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-configs", action="store_true", help="skip the `configs` sub-records (configs 1, 3, 4, 5)")
    ap.add_argument("--items", type=int, default=64, help="config 4: parameter sets (of the 1024) to evaluate")
    ap.add_argument("--chunk", type=int, default=16, help="config 4: parameter sets per plan / launch sequence")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    import paper_2307_12585_b200 as fd

    from paper_2307_12585_b200 import dist as fdist
    rank, world, local = fdist.env_world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    def barrier():
        fdist.barrier()
        torch.cuda.synchronize()

    if args.config == 4:
        line = run_batched(args, fd, fdist, torch, dev, rank, world, local, barrier)
        if rank == 0:
            print(json.dumps(line))
        if world > 1:
            dist.destroy_process_group()
        return

    flush = torch.empty(512 * 1024 * 1024 // 8, dtype=torch.float64, device=dev)     # 512 MB > 126 MB L2
    stream = torch.cuda.current_stream()
    peak_tf = fd.fdemri_measure_fp64_peak(1 << 16)
    peak3_tf = fd.fdemri_measure_fp64_peak_3reg(1 << 16)

    # ---- timed: K steps of the headline workload, L2 flushed between steps, CUDA events on the launching stream ----
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    barrier()
    m = measure_single(fd, torch, dev, args.config, args.steps, args.warmup, flush,
                       latency_reps=0 if args.no_e2e else 5)
    barrier()
    w, wf, host, dev_in, st = m["w"], m["wf"], m["host"], m["dev_in"], m["stats"]
    n_evals = st["n_evals"]
    total_ms = fdist.max_over_ranks(float(sum(m["step_ms"])), device=dev)

    # the same step with the inner products of Eq. 12 formed on the fly and no waveform written
    gen = torch.Generator(device=dev); gen.manual_seed(230712585)
    inner_w = torch.rand(w.n_freq, dtype=torch.float64, device=dev, generator=gen) + 0.5
    inner_dp = torch.randn((w.n_freq, 2), dtype=torch.float64, device=dev, generator=gen)
    inner_dx = torch.randn((w.n_freq, 2), dtype=torch.float64, device=dev, generator=gen)
    inner_out = torch.zeros((w.n_batch, 4), dtype=torch.float64, device=dev)
    inner_ms = []
    for i in range(3 + args.steps):
        flush.fill_(1.0)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        build_call(fd, wf, dev_in)
        fd.fdemri_sum_inner(wf.plan, w.theta, w.phi, inner_out, weight=inner_w, data_plus=inner_dp, data_cross=inner_dx)
        e1.record(stream)
        e1.synchronize()
        if i >= 3:
            inner_ms.append(e0.elapsed_time(e1))
    fused_inner = {"ms_per_step": float(np.mean(inner_ms)), "waveforms_per_s": 1e3 / float(np.mean(inner_ms)),
                   "what": "fdemri_build_splines + fdemri_sum_inner: <h|h> and <d|h> of Eq. 12 per waveform, no waveform "
                           "written (32 B leave the GPU)", "inner": inner_out.cpu().numpy()[0, :3].tolist()}

    # ---- end to end through host buffers (pinned H2D of inputs, D2H of both polarisations) ----
    e2e = None
    if not args.no_e2e:
        # Throughput pipeline over two sets of buffers and three streams: the upload stream brings the inputs of step
        # i+1 (pinned H2D, 9 MB), the compute stream runs S0-S4 of step i, the download stream takes the polarisations
        # of step i-1 home (pinned D2H, 101 MB: the PCIe link, not the kernels, would otherwise set the pace).  Every
        # byte in and out crosses inside the timed region; the region ends when the last download has landed.
        pin_in = [torch.from_numpy(a).pin_memory() for a in host]
        ins = [dev_in, [torch.empty_like(t) for t in dev_in]]
        outs = [(wf.hplus, wf.hcross), (torch.empty_like(wf.hplus), torch.empty_like(wf.hcross))]
        pin_out = [[torch.empty(wf.hplus.shape, dtype=torch.float64).pin_memory() for _ in range(2)] for _ in range(2)]
        h2d = sum(a.numel() * 8 for a in pin_in)
        d2h = sum(a.numel() * 8 for a in pin_out[0])
        copy_stream = torch.cuda.Stream(device=dev)
        up_stream = torch.cuda.Stream(device=dev)
        in_ready = [torch.cuda.Event() for _ in range(2)]
        comp_done = [torch.cuda.Event() for _ in range(2)]
        copy_done = [torch.cuda.Event() for _ in range(2)]

        def run_e2e(n):
            for i in range(n):
                k = i & 1
                with torch.cuda.stream(up_stream):
                    up_stream.wait_event(comp_done[k])      # the splines of step i-2 have consumed input buffer k
                    for d, p in zip(ins[k], pin_in):
                        d.copy_(p, non_blocking=True)
                    in_ready[k].record(up_stream)
                stream.wait_event(in_ready[k])
                stream.wait_event(copy_done[k])             # output buffer k free again (its last download landed)
                build_call(fd, wf, ins[k])
                fd.fdemri_sum(wf.plan, w.theta, w.phi, outs[k][0], outs[k][1])
                comp_done[k].record(stream)
                with torch.cuda.stream(copy_stream):
                    copy_stream.wait_event(comp_done[k])
                    pin_out[k][0].copy_(outs[k][0], non_blocking=True)
                    pin_out[k][1].copy_(outs[k][1], non_blocking=True)
                    copy_done[k].record(copy_stream)

        for ev in comp_done:
            ev.record(stream)
        for ev in copy_done:
            ev.record(copy_stream)
        run_e2e(3)
        torch.cuda.synchronize()
        barrier()
        flush.fill_(1.0)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        run_e2e(args.steps)
        stream.wait_stream(copy_stream)
        b.record(stream)
        b.synchronize()
        ems = a.elapsed_time(b)
        barrier()
        ems = fdist.max_over_ranks(ems, device=dev)
        assert np.array_equal(pin_out[(args.steps - 1) & 1][0].numpy(), outs[(args.steps - 1) & 1][0].cpu().numpy())
        e2e = {"value": world * args.steps / (ems * 1e-3), "unit": "waveforms/s", "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "ms_per_step": ems / args.steps,
               "how": "two-deep pipeline on three streams: pinned H2D of the next step's inputs, S0-S4, pinned D2H of the "
                      f"previous step's polarisations ({d2h / 1e6:.1f} MB per step)",
               "latency_ms_one_waveform": m.get("e2e_latency_ms"),
               "latency_how": "nothing overlapped: pinned H2D of the inputs, fdemri_build_splines + fdemri_sum, pinned D2H "
                              "of both polarisations, synchronise (CUDA events; median of 5)"}
        del pin_in, pin_out, ins, outs

    clocks = sampler.stop() if rank == 0 else None          # sampled over both timed regions (device and e2e)

    # ---- the other workloads, fewer steps each: driver-visible numbers for every figure DESIGN.md / README.md quote ----
    configs = None
    launches_extra = 0
    if rank == 0 and world == 1 and not args.no_configs and args.config == 2:
        configs = {}
        sub_steps = max(5, args.steps // 2)
        m.pop("wf").close()
        del wf, dev_in
        torch.cuda.empty_cache()
        for idx in (1, 3, 5):
            ms_ = measure_single(fd, torch, dev, idx, sub_steps, 3, flush, latency_reps=5 if idx == 3 else 0)
            configs[str(idx)] = dict(sub_record(fd, ms_, peak_tf), workload=workload_name(idx, ms_["w"]))
            launches_extra += KERNELS_PER_STEP * (sub_steps + (7 if idx == 3 else 0))
            ms_.pop("wf").close()
            del ms_
            torch.cuda.empty_cache()
        args4 = argparse.Namespace(**vars(args))
        args4.items, args4.chunk, args4.steps, args4.warmup = 64, 16, 1, 3
        l4 = run_batched(args4, fd, fdist, torch, dev, rank, world, local, barrier, quiet=True)
        configs["4"] = {"ms_per_step": l4["ms_per_step"], "waveforms_per_s": l4["value"], "items": 64,
                        "evals_per_step": l4["evals_per_step"], "evals_per_s": l4["evals_per_s"], "roofline": l4["roofline"],
                        "workload": l4["config"]["workload"], "steps": 1}
        launches_extra += l4["gpu_launches"]
        configs["issue_ns"] = issue_model(fd)

    if rank == 0:
        k_ms = float(np.mean(m["kern_ms"]))
        achieved = n_evals * FLOP_PER_EVAL / (k_ms * 1e-3) * 1e-12
        n_timed_steps = args.steps * 2 + 3 + (0 if args.no_e2e else args.steps + 3 + 7)
        line = {
            "metric": METRIC, "value": world * args.steps / (total_ms * 1e-3), "unit": "waveforms/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": total_ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.config, w),
                       "step": "fdemri_build_splines + fdemri_sum (S0-S4)", "l2": "flushed between steps (512 MB fill)",
                       "parallelism": "replicas, one waveform per GPU, no collective"},
            "ms_per_waveform": total_ms / args.steps, "evals_per_waveform": n_evals,
            "evals_per_s": world * n_evals * args.steps / (total_ms * 1e-3),
            "ms_build_splines": float(np.mean(m["step_ms"]) - np.mean(m["sum_ms"])), "ms_sum": float(np.mean(m["sum_ms"])),
            "gpu_launches": KERNELS_PER_STEP * args.steps,
            "gpu_launches_whole_run": KERNELS_PER_STEP * n_timed_steps + launches_extra,
            "roofline": {"bound": "alu", "kernel": "k_bin_sum" if m["bin_major"] else "k_tile_sum", "achieved": achieved,
                         "peak": peak_tf, "unit": "TFLOP/s",
                         "frac": achieved / peak_tf, "traffic": None,
                         "traffic_note": "dram__bytes_read.sum + dram__bytes_write.sum need ncu, which this program never runs "
                                         "under: see " + NCU_PROFILE + " (bytes are context: the bound is the FP64 pipe)",
                         "executed_flop_frac_ncu": None,
                         "executed_flop_frac_note": "frac counts SURVEY 8(d)'s 200 algorithmic flop per evaluation; the executed-"
                                                    "instruction fraction (2 DFMA + DADD + DMUL per cycle, ncu) is in " + NCU_PROFILE,
                         "kernel_ms": k_ms,
                         "flop_per_eval": FLOP_PER_EVAL,
                         "peak_source": "FP64 DFMA loop measured live (fdemri_measure_fp64_peak); nominal 148 SM x 64 "
                                        "lanes x 2 x 1.965 GHz = 37.2 TFLOP/s; MEASURED_PEAKS.json has no FP64 entry",
                         "peak_3reg": peak3_tf,
                         "peak_3reg_note": "context, not a roof for `achieved` (which counts algorithmic, not executed, flops): the "
                                           "same loop with three distinct register operands per DFMA -- an FP64 instruction "
                                           "costs max(2, distinct register operands) issue cycles, and integer / FP32 "
                                           "instructions do not issue in its shadow (profiles/r2_dispatch_model.md)"},
            "clocks": clocks, "stats": st, "fused_inner": fused_inner,
        }
        if e2e:
            line["e2e"] = e2e
        if configs:
            line["configs"] = configs
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_oracle_sample(w, n_evals)
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
