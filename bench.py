#!/usr/bin/env python
"""bench.py — throughput of the fused NLL + analytic-gradient hot path on B200.

Workload (BASELINE.json configs[1], "C1"): the 1D Gaussian+exponential mass model, N = 1,000,000
fp64 events, 4 free parameters, "repeated NLL+gradient calls at 1,000 random parameter points within
+-3 sigma_stat of truth".  One STEP = one complete SWEEP of the hot path over that workload: all 1,000
seeded lambda points evaluated on one dataset replica (S2 parameter-only constants on the host, S3
per-event value + gradient, S4/S5 reductions, S6 K+2 doubles out per point) = 1e9 event evaluations,
issued as ONE mf_nll_grad_points call of 1,000 points (= one kernel launch; consecutive calls overlap on the GPU, so the
number does not depend on how a sweep is cut into calls).  `value` = events/s;
`us_per_evaluation` = ms_per_step / 1000 points is printed beside it.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl mine|reference]

Timing rules followed: W >= 3 warm-up steps of the SAME call shape as the timed ones; the steps rotate
over R = 32 dataset replicas (256 MB > the 126 MB L2), so every sweep first reads its events from HBM
("l2" in config); CUDA events on the launching stream; max over ranks; SM clocks and throttle reasons
sampled (NVML, separate process) during the timed region.  The number does not depend on --steps: the
driver's `--steps 20 --warmup 5` times 20 launches (~31 ms).

`e2e` is the same step through the public API with HOST inputs: mf_dataset_upload from pinned host memory,
mf_model_create, mf_nll_grad_sweep (1,000 host lambda points in, 1,000 x (K+1) host results out), destroy.
`roofline` is for the dominant kernel nll_grad_batch_kernel<MassModel> (ALU bound);
`cpu_baseline` is the fp64 oracle on this box's host cores on a bounded sample.

--impl reference times the CPU oracle itself (there is no reference implementation to install:
/root/reference holds only the paper), on the same config, metric and unit.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import mf_datagen as dg  # noqa: E402

N_EVENTS = 1_000_000
N_POINTS = 1000          # lambda points of one sweep = one step
N_REPLICAS = 32
K_PARAMS = 4
METRIC = "nll_grad_event_evals_per_s"
UNIT = "events/s"
WORKLOAD = "C1: 1D Gaussian+exponential mass model, N=1e6 fp64 events, K=4, NLL+gradient at 1000 seeded lambda points"
# fp64-pipe thread-instructions per event of the shipped mass kernel's fast path, counted in its SASS (177 DFMA/DMUL/DADD
# per 8-event call = 22.1 per event, DESIGN.md §7 "Roofline"); the shipped kernel's count, never more than
# the plain two-exponential form's hand count (100).  Round 1 credited 26 (that kernel's count).
MASS_FP64_INSTR_PER_EVENT = 22.1
POINTS_PER_CALL = 1000  # evaluations per mf_nll_grad_points call (ONE launch: CTA tile = (point, event chunk))
NOMINAL_FP64_LANES_PER_SM = 64  # B200: 4 SMSPs x 16 fp64 FMA lanes
SINGLE_LAUNCH_STEPS = 4000      # evaluations of the one-launch-per-evaluation leg (fixed, whatever --steps says)
REF_POINTS_PER_STEP = 8         # reference arm: lambda points of the sweep evaluated per step (bounded sample)

# the same dict in both arms (the driver compares the arms' configs)
CONFIG = {"workload": WORKLOAD, "n_events": N_EVENTS, "n_params": K_PARAMS, "lambda_points": N_POINTS,
          "step": "one sweep: all 1000 lambda points on one 1e6-event dataset = 1e9 event evaluations",
          "l2": "inputs larger than L2: the steps rotate over 32 x 8 MB dataset replicas (256 MB > 126 MB), so each sweep first "
                "reads its events from HBM; the 1000 evaluations of a sweep re-read them from L2 by design (8 B/event, ALU bound)"}


def _clock_sampler_main(index: int, path: str) -> None:
    """Child process: appends 't sm_mhz sm_max_mhz reasons_bitmask' lines to `path` until stdin closes."""
    import select

    import pynvml
    pynvml.nvmlInit()
    h = pynvml.nvmlDeviceGetHandleByIndex(index)
    mx = pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM)
    with open(path, "w", buffering=1) as fh:
        while True:
            if select.select([sys.stdin], [], [], 0.002)[0]:
                break
            sm = pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)
            rs = pynvml.nvmlDeviceGetCurrentClocksEventReasons(h)
            fh.write(f"{time.time():.6f} {sm} {mx} {rs}\n")


class ClockSampler:
    """SM clock and throttle reasons sampled by NVML in a separate process during the timed region."""
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x100: "display_clock_setting",
               0x10: "sync_boost"}

    def __init__(self, index: int):
        import tempfile
        self.path = os.path.join(tempfile.gettempdir(), f"mf_clocks_{os.getpid()}.txt")
        self.p = None
        try:
            self.p = subprocess.Popen([sys.executable, os.path.abspath(__file__), "--clock-sampler", str(index), self.path],
                                      stdin=subprocess.PIPE, stdout=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def wait_ready(self, timeout: float = 30.0) -> None:
        t = time.time()
        while self.p is not None and time.time() - t < timeout:
            if os.path.exists(self.path) and os.path.getsize(self.path) > 0:
                return
            if self.p.poll() is not None:
                return
            time.sleep(0.01)

    def stop(self, t0: float, t1: float) -> dict:
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["sampler unavailable"]}
        try:
            self.p.communicate(b"q\n", timeout=10)
        except Exception:
            self.p.kill()
        sm, mx, bits, n_all = [], None, 0, 0
        try:
            with open(self.path) as fh:
                lines = fh.read().splitlines()
            os.remove(self.path)
        except Exception:
            lines = []
        for line in lines:
            try:
                t, s, m, r = line.split()
            except ValueError:
                continue
            n_all += 1
            mx = int(m)
            if t0 <= float(t) <= t1:
                sm.append(int(s))
                bits |= int(r)
        reasons = [name for bit, name in self.REASONS.items() if bits & bit]
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": mx, "reasons": reasons,
                "samples_in_region": len(sm), "samples": n_all}


def _dist_setup(n_gpus: int):
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch
        import torch.distributed as dist
        torch.cuda.set_device(local)
        dist.init_process_group(backend="nccl", device_id=torch.device("cuda", local))
    return rank, world, local


def _barrier(world: int):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def _max_over_ranks(x: float, world: int) -> float:
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device="cuda")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def _cpu_baseline(sample_events: int, repeats: int) -> dict:
    """The oracle as it stands on this box's host cores, on the first `sample_events` events of C1."""
    import oracle
    m = dg.gen_mass(N_EVENTS, seed=1)[:sample_events]
    pts = dg.gen_lambda_points(N_POINTS, 1001, dg.MASS_TRUTH, 3 * dg.mass_sigma_stat(N_EVENTS))
    best = {}
    for nt in sorted({1, oracle.max_threads()}):
        oracle.nll_grad(oracle.MASS, m[:1000], pts[0], dg.MASS_LO, dg.MASS_HI, nthreads=nt)
        t = time.perf_counter()
        for i in range(repeats):
            oracle.nll_grad(oracle.MASS, m, pts[i % N_POINTS], dg.MASS_LO, dg.MASS_HI, nthreads=nt)
        best[nt] = sample_events * repeats / (time.perf_counter() - t)
    nt = max(best, key=best.get)
    return {"value": best[nt], "unit": UNIT, "cores": nt, "kind": "oracle",
            "sample": f"{repeats} NLL+gradient calls (lambda points 0..{repeats - 1} of the sweep) on all {sample_events} events "
                      "of the C1 dataset (seed 1)",
            "single_thread_value": best[1], "host_cores": os.cpu_count()}


def run_reference(args) -> None:
    """--impl reference: the CPU oracle timed as the reference arm (rank 0 only).  Same config, metric and unit as the
    GPU arm; each step is a bounded sample of the sweep: its first REF_POINTS_PER_STEP lambda points (rotating through the
    1000) on ALL 1e6 events."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    m = dg.gen_mass(N_EVENTS, seed=1)
    pts = dg.gen_lambda_points(N_POINTS, 1001, dg.MASS_TRUTH, 3 * dg.mass_sigma_stat(N_EVENTS))
    nt = oracle.max_threads()
    steps = min(args.steps, 400)   # each step ~ 0.1 s of CPU on 16 cores: keeps the arm within minutes
    warm = min(args.warmup, 5)

    def step(i: int):
        for q in range(REF_POINTS_PER_STEP):
            oracle.nll_grad(oracle.MASS, m, pts[(i * REF_POINTS_PER_STEP + q) % N_POINTS], dg.MASS_LO, dg.MASS_HI, nthreads=nt)

    for i in range(warm):
        step(i)
    t = time.perf_counter()
    for i in range(steps):
        step(warm + i)
    dt = time.perf_counter() - t
    value = N_EVENTS * REF_POINTS_PER_STEP * steps / dt
    desc = (f"each step = {REF_POINTS_PER_STEP} of the sweep's 1000 lambda points (oracle NLL+gradient calls) on all {N_EVENTS} "
            f"events of C1 ({nt} threads)")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": warm, "ms_per_step": 1e3 * dt / steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": CONFIG,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": nt, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def _time_points(torch, models, lam, K, n_calls: int) -> float:
    """us per evaluation: n_calls back-to-back evaluations at lam rotating over `models` (CUDA events)."""
    out = torch.zeros((8, K + 2), dtype=torch.float64, device="cuda")
    lams = np.tile(np.asarray(lam, dtype=np.float64), (8, 1))
    per = 1 if len(models) > 1 else 8   # several replicas: a different one every evaluation; < 16 per call = one launch each

    def go(n):
        i = 0
        while i < n:
            c = min(per, n - i)
            models[(i // per) % len(models)].nll_grad_points(lams[:c], out.data_ptr())
            i += c

    go(20)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    go(n_calls)
    e1.record()
    torch.cuda.synchronize()
    if not np.all(np.isfinite(out.cpu().numpy()[0, :K + 1])):
        raise RuntimeError("non-finite result in an extra workload")
    return float(e0.elapsed_time(e1)) * 1e3 / n_calls


def _other_workloads(torch, mf, ctx, peaks, traffic_all) -> dict:
    """The other BASELINE.json configs, each timed the same way (device-resident inputs, CUDA events,
    inputs larger than the 126 MB L2 or rotated over replicas that are).  Parity for these is in tests/."""
    # HBM peak: the driver's measured copy bandwidth, else the profiling guide's stated fallback (6.65 TB/s, "of fallback")
    hbm = float(peaks.get("hbm_gbs", 0.0)) or 6650.0
    hbm_how = "MEASURED_PEAKS.json hbm_gbs" if peaks.get("hbm_gbs") else "fallback of B200_PROFILING.md (6.65 TB/s)"
    res = {"hbm_peak_source": hbm_how}
    n_sm_ = torch.cuda.get_device_properties(0).multi_processor_count
    sm_mhz_ = float(peaks.get("sm_max_mhz", 1965.0))
    # C2: 3D angular, N = 1e6, nine cached basis columns = 72 B/event (HBM bound)
    ev = dg.gen_angular(1_000_000, seed=2)
    ms = [ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ctx.dataset_upload(ev)) for _ in range(6)]   # 6 x 72 MB = 432 MB > 3 x L2
    us = _time_points(torch, ms, dg.ANG_TRUTH, 8, 600)
    gbs = 72.0 * 1_000_000 / us / 1e3
    res["C2_angular_1e6"] = {"us_per_eval": us, "events_per_s": 1e6 / (us * 1e-6), "kernel": "nll_grad_tma_kernel<AngularModel>",
                             "roofline": {"bound": "hbm", "achieved": gbs, "peak": hbm, "unit": "GB/s",
                                          "frac": gbs / hbm if hbm else None, "bytes_per_event": 72,
                                          "traffic": traffic_all.get("nll_grad_tma_kernel<AngularModel>")},
                             "l2": "6 model replicas x 72 MB = 432 MB (> 3 x L2) rotated, a different one every evaluation"}
    # the same evaluation repeated on ONE model: its 72 MB of basis columns stay in the 126 MB L2 (what a fit sees)
    us_l2 = _time_points(torch, ms[:1], dg.ANG_TRUTH, 8, 600)
    res["C2_angular_1e6"]["l2_resident"] = {"us_per_eval": us_l2, "read_gbs": 72.0 * 1_000_000 / us_l2 / 1e3,
                                            "what": "one model evaluated back to back (north_star: basis terms cached in L2 when the "
                                                    "dataset fits); not a roofline claim against HBM"}
    t = time.perf_counter()
    r = ms[0].fit(dg.ANG_TRUTH)
    res["C2_angular_1e6"]["fit_s"] = time.perf_counter() - t
    res["C2_angular_1e6"]["fit_calls"] = r.n_calls
    # many parameter points in ONE pass over the data: two fp64 tensor-core contractions, 64 points per pass
    mp = {}
    for M in (64, 1000):
        ptsM = np.tile(np.array(dg.ANG_TRUTH), (M, 1)) + np.random.default_rng(5).uniform(-0.03, 0.03, (M, 8))
        oM = torch.zeros((M, 10), dtype=torch.float64, device="cuda")
        for _ in range(3):
            ms[0].nll_grad_points(ptsM, oM.data_ptr())
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = 20
        e0.record()
        for i_ in range(reps):
            ms[i_ % len(ms)].nll_grad_points(ptsM, oM.data_ptr())
        e1.record()
        torch.cuda.synchronize()
        usM = float(e0.elapsed_time(e1)) * 1e3 / reps / M
        if not np.all(np.isfinite(oM.cpu().numpy()[:, :9])):
            raise RuntimeError("non-finite result in the angular many-points workload")
        # pipe work per (point, event) pair: 4/64 DMMA of 256 FMAs + reciprocal (3 DFMA) + 1 DMUL = 20 FMA-equivalents
        mp[f"us_per_evaluation_{M}_points"] = usM
        mp[f"frac_of_fp64_peak_{M}_points"] = 20.0 * 1e6 / (usM * 1e-6) / (n_sm_ * NOMINAL_FP64_LANES_PER_SM * sm_mhz_ * 1e6)
    mp["kernel"] = "angular_points_mma_kernel<4> + angular_points_combine_kernel (mf_nll_grad_points), 32 points per pass"
    mp["bound"] = "alu (fp64 pipe, DMMA shares it with DFMA): 20 FMA-equivalents per (point, event) pair incl. tile padding"
    res["C2_angular_1e6"]["many_points"] = mp
    del ms, ev
    # C3: 4D, N = 2e6, 12 columns = 96 B/event (192 MB > L2)
    ev = dg.gen_4d(2_000_000, seed=3)
    m4s = [ctx.model_create(mf.MF_MASS_X_ANGULAR, ctx.dataset_upload(ev, dg.MASS_LO, dg.MASS_HI)) for _ in range(2)]
    m4 = m4s[0]
    us = _time_points(torch, m4s, dg.FOURD_TRUTH, 16, 400)   # 2 x 192 MB of columns, alternating
    gbs = 96.0 * 2_000_000 / us / 1e3
    res["C3_4d_2e6"] = {"us_per_eval": us, "events_per_s": 2e6 / (us * 1e-6), "kernel": "nll_grad_tma_kernel<FourDModel>",
                        "roofline": {"bound": "hbm", "achieved": gbs, "peak": hbm, "unit": "GB/s",
                                     "frac": gbs / hbm if hbm else None, "bytes_per_event": 96,
                                     "traffic": traffic_all.get("nll_grad_tma_kernel<FourDModel>")},
                        "l2": "2 model replicas x 192 MB of columns, alternating every evaluation"}
    # many parameter points in ONE pass over the data per 16 points (mf_points4d.cuh)
    mp4 = {}
    for M in (64, 256):
        ptsM = np.tile(np.array(dg.FOURD_TRUTH), (M, 1))
        ptsM += np.random.default_rng(6).uniform(-1, 1, (M, 16)) * np.array([0.02, 0.002, 0.001, 0.2] + [0.03] * 8 + [0.05] * 4)
        oM = torch.zeros((M, 18), dtype=torch.float64, device="cuda")
        for _ in range(2):
            m4.nll_grad_points(ptsM, oM.data_ptr())
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for i_ in range(6):
            m4s[i_ % 2].nll_grad_points(ptsM, oM.data_ptr())
        e1.record()
        torch.cuda.synchronize()
        if not np.all(np.isfinite(oM.cpu().numpy()[:, :17])):
            raise RuntimeError("non-finite result in the 4D many-points workload")
        mp4[f"us_per_evaluation_{M}_points"] = float(e0.elapsed_time(e1)) * 1e3 / 6 / M
    mp4["kernel"] = "fourd_points_mma_kernel<2> + fourd_points_combine_kernel (mf_nll_grad_points), 16 points per pass"
    mp4["single_launch_us_per_evaluation"] = us
    res["C3_4d_2e6"]["many_points"] = mp4
    m4.fit(dg.FOURD_TRUTH)
    t = time.perf_counter()
    r = m4.fit(dg.FOURD_TRUTH)
    res["C3_4d_2e6"]["fit_s"] = time.perf_counter() - t
    res["C3_4d_2e6"]["fit_calls"] = r.n_calls
    res["C3_4d_2e6"]["fit"] = "mf_fit: Newton steps on the analytic Hessian (second-order kernel: S^T S by fp64 tensor-core contraction) + HESSE"
    # value + gradient + analytic Hessian (136 second derivatives), and with the Fisher matrix, per synchronous call
    def sync_us(f, n=20):
        f()
        t0 = time.perf_counter()
        for _ in range(n):
            f()
        return (time.perf_counter() - t0) / n * 1e6
    res["C3_4d_2e6"]["second_order"] = {
        "kernel": "nll_second_kernel<FourDSecond, 1|2> + second_combine_kernel",
        "us_per_call_value_gradient_hessian": sync_us(lambda: m4.nll_grad_hess(dg.FOURD_TRUTH)),
        "us_per_call_with_fisher_matrix": sync_us(lambda: m4.nll_grad_hess_fisher(dg.FOURD_TRUTH)),
        "us_per_call_value_gradient": sync_us(lambda: m4.nll_grad(dg.FOURD_TRUTH)),
        "what": "synchronous host calls (launch pair + D2H of the result row + stream synchronise included)"}
    # weighted fit of the same events: every evaluation through the second-order kernel, sandwich covariance
    dsw = ctx.dataset_upload(ev, dg.MASS_LO, dg.MASS_HI)
    dsw.set_weights(np.random.default_rng(77).uniform(0.5, 1.5, ev.shape[1]))
    m4w = ctx.model_create(mf.MF_MASS_X_ANGULAR, dsw)
    m4w.fit(dg.FOURD_TRUTH)
    t = time.perf_counter()
    rw = m4w.fit(dg.FOURD_TRUTH)
    res["C3_4d_2e6"]["weighted_fit"] = {"fit_s": time.perf_counter() - t, "fit_calls": rw.n_calls, "converged": bool(rw.converged),
                                        "us_per_call_value_gradient": sync_us(lambda: m4w.nll_grad(dg.FOURD_TRUTH)),
                                        "what": "weights uniform in [0.5, 1.5]; covariance = H^-1 F H^-1 (mf_nll_grad_hess_fisher at the minimum)"}
    del m4, m4s, m4w, dsw, ev
    # C4: 4096 toys x 1e4 events (328 MB > L2), one launch for all toys; then all toys fitted concurrently
    T, n = 4096, 10_000
    toys = dg.gen_mass_toys(T, n, first_seed=0)
    bm = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(toys, dg.MASS_LO, dg.MASS_HI, n_toys=T))
    lams = np.tile(np.array(dg.MASS_TRUTH), (T, 1))
    for _ in range(3):
        bm.nll_grad_batch(lams)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps = 30
    e0.record()
    for _ in range(reps):
        bm.nll_grad_batch(lams)
    e1.record()
    torch.cuda.synchronize()
    us_call = float(e0.elapsed_time(e1)) * 1e3 / reps
    # the same evaluation with lambda and the results resident on the device (mf_nll_grad_batch_async)
    d_lam = torch.from_numpy(lams).cuda()
    d_out = torch.zeros((T, 6), dtype=torch.float64, device="cuda")
    for _ in range(3):
        bm.nll_grad_batch_async(d_lam.data_ptr(), d_out.data_ptr())
    torch.cuda.synchronize()
    e0.record()
    for _ in range(reps):
        bm.nll_grad_batch_async(d_lam.data_ptr(), d_out.data_ptr())
    e1.record()
    torch.cuda.synchronize()
    us = float(e0.elapsed_time(e1)) * 1e3 / reps
    chk = d_out.cpu().numpy()
    if not (np.all(np.isfinite(chk[:, :5])) and np.all(chk[:, 5] == 0)):
        raise RuntimeError("non-finite result in the batched-toy workload")
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    peak_tf = 2.0 * n_sm * NOMINAL_FP64_LANES_PER_SM * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6 / 1e12
    ach_tf = 2.0 * MASS_FP64_INSTR_PER_EVENT * T * n / (us * 1e-6) / 1e12
    # value + gradient + analytic Hessian for all toys (host call), the evaluation the toy fits use
    for _ in range(2):
        bm.nll_grad_hess_batch(lams)
    e0.record()
    for _ in range(10):
        bm.nll_grad_hess_batch(lams)
    e1.record()
    torch.cuda.synchronize()
    us_hess_call = float(e0.elapsed_time(e1)) * 1e3 / 10
    bm.fit_batch(np.array(dg.MASS_TRUTH))
    t = time.perf_counter()
    fr = bm.fit_batch(np.array(dg.MASS_TRUTH))
    fit_s = time.perf_counter() - t
    ofd = mf.default_fit_opts()
    ofd.analytic_hessian = 0
    t = time.perf_counter()
    fr_fd = bm.fit_batch(np.array(dg.MASS_TRUTH), opts=ofd)
    fit_fd_s = time.perf_counter() - t
    pulls = ((fr.lam - np.array(dg.MASS_TRUTH)) / fr.sigma)[fr.converged]
    res["C4_toys_4096x1e4"] = {
        "us_per_batch_eval": us, "events_per_s": T * n / (us * 1e-6), "kernel": "nll_grad_batch_kernel<MassModel>",
        "what": "mf_nll_grad_batch_async (lambda and results on the device): batch_consts_kernel + nll_grad_batch_kernel, back to back",
        "us_per_host_call": us_call, "host_call_events_per_s": T * n / (us_call * 1e-6),
        "host_call": "mf_nll_grad_batch: H2D of 4096 lambda vectors + the two launches + D2H of 4096 x 6 doubles + synchronise",
        "roofline": {"bound": "alu", "achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s", "frac": ach_tf / peak_tf,
                     "fp64_instr_per_event": MASS_FP64_INSTR_PER_EVENT,
                     "traffic": traffic_all.get("nll_grad_batch_kernel<MassModel>"),
                     "hbm_side_gbs": 8.0 * T * n / us / 1e3},
        "us_per_host_call_with_hessian": us_hess_call,
        "fits_per_s": T / fit_s, "fit_batch_s": fit_s, "converged": int(fr.converged.sum()),
        "mean_calls_per_toy": float(fr.n_calls.mean()),
        "fit": "mf_fit_batch, all 4096 toys concurrently from the truth, Newton steps on the analytic Hessian + HESSE",
        "fits_per_s_finite_difference_hessian": T / fit_fd_s, "mean_calls_per_toy_finite_difference": float(fr_fd.n_calls.mean()),
        "pull_mean": pulls.mean(0).round(4).tolist(), "pull_width": pulls.std(0).round(4).tolist()}
    del bm, toys
    # the paper's own protocol (time per pseudo-experiment = generation + fit + HESSE), all on the device
    def toy_study(seed0):
        return ctx.toy_study_mass(seed0, T, n, dg.MASS_TRUTH, dg.MASS_LO, dg.MASS_HI)
    toy_study(1)
    t = time.perf_counter()
    ts = toy_study(100_000)
    ts_s = time.perf_counter() - t
    e0.record()
    gds = ctx.generate_mass(7, T, n, dg.MASS_TRUTH, dg.MASS_LO, dg.MASS_HI)
    e1.record()
    torch.cuda.synchronize()
    gen_us = float(e0.elapsed_time(e1)) * 1e3
    gds.close()
    # the other two generators (accept-reject under the paper's get_max() envelope, ~10 % acceptance for the angular PDF)
    gen_other = {}
    for name, n_gen, make in (("angular_1e6", 1_000_000, lambda sd: ctx.generate_angular(sd, 1, 1_000_000, dg.ANG_TRUTH)),
                              ("4d_2e6", 2_000_000, lambda sd: ctx.generate_4d(sd, 1, 2_000_000, dg.FOURD_TRUTH, dg.MASS_LO, dg.MASS_HI))):
        make(11).close()
        e0.record()
        g_ = make(12)
        e1.record()
        torch.cuda.synchronize()
        g_us = float(e0.elapsed_time(e1)) * 1e3
        g_.close()
        gen_other[name] = {"generation_us": g_us, "generated_events_per_s": n_gen / (g_us * 1e-6)}
    res["generators"] = gen_other
    res["toy_study_4096x1e4_on_device"] = {
        "ms_per_toy": 1e3 * ts_s / T, "toys_per_s": T / ts_s, "converged": int(ts.converged.sum()),
        "what": "mf_toy_study_mass: mf_generate_mass (4096 toys x 1e4 events, Philox4x32-10) + mf_model_create + mf_fit_batch "
                "(Newton on the analytic Hessian + HESSE); no event crosses PCIe",
        "generation_us": gen_us, "generated_events_per_s": T * n / (gen_us * 1e-6),
        "paper_context": "MoreFit OpenCL GPU (analytic), Titan V: 1.62 ms per toy at 1e4 events (PAPER.md:191); another machine"}
    # the paper's second benchmark (Table 3): angular pseudo-experiments, generation + fit + HESSE
    Ta = 1024
    ctx.toy_study_angular(1, Ta, n, dg.ANG_TRUTH)
    t = time.perf_counter()
    tsa = ctx.toy_study_angular(200_000, Ta, n, dg.ANG_TRUTH)
    tsa_s = time.perf_counter() - t
    res["toy_study_angular_1024x1e4_on_device"] = {
        "ms_per_toy": 1e3 * tsa_s / Ta, "toys_per_s": Ta / tsa_s, "converged": int(tsa.converged.sum()),
        "mean_calls_per_toy": float(tsa.n_calls.mean()),
        "what": "mf_toy_study_angular: mf_generate_angular (accept-reject, 1024 toys x 1e4 events) + mf_model_create (basis cache) + "
                "mf_fit_batch (Newton on the analytic Hessian + HESSE); no event crosses PCIe",
        "paper_context": "MoreFit OpenCL GPU (analytic), Titan V: 2.39 ms per toy at 1e4 events (PAPER.md:224); another machine, other truth values"}
    # C0: N = 1e4, one call + full fit (latency bound: no roofline claim)
    m0 = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(dg.gen_mass(10_000, seed=0), dg.MASS_LO, dg.MASS_HI))
    m0.nll_grad(dg.MASS_START)
    t = time.perf_counter()
    for _ in range(200):
        m0.nll_grad(dg.MASS_START)
    lat = (time.perf_counter() - t) / 200
    m0.fit(dg.MASS_START)     # first fit on a model: sets up the resident kernel's stream and scratch
    t = time.perf_counter()
    r = m0.fit(dg.MASS_START)
    fit_s0 = time.perf_counter() - t
    m0.serve(True)          # resident evaluation kernel: no launch, no completion latency per call (mf_server.cuh)
    for _ in range(50):
        m0.nll_grad(dg.MASS_START)
    t = time.perf_counter()
    for _ in range(200):
        m0.nll_grad(dg.MASS_START)
    lat_served = (time.perf_counter() - t) / 200
    m0.serve(False)
    res["C0_mass_1e4"] = {"sync_call_us": lat * 1e6, "served_call_us": lat_served * 1e6, "fit_s": fit_s0, "fit_calls": r.n_calls,
                          "converged": bool(r.converged),
                          "what": "Python-level synchronous mf_nll_grad calls (ctypes marshalling included; from C: 13.0 us by launch, "
                                  "8.5 us served, profiles/r2_server_latency.md); mf_fit serves its own evaluations"}
    # C1's full fit from the BASELINE start point (N = 1e6)
    m1 = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(dg.gen_mass(N_EVENTS, seed=1), dg.MASS_LO, dg.MASS_HI))
    m1.fit(dg.MASS_START)
    t = time.perf_counter()
    r = m1.fit(dg.MASS_START)
    res["C1_full_fit"] = {"fit_s": time.perf_counter() - t, "fit_calls": r.n_calls, "converged": bool(r.converged),
                          "pull": ((r.lam - np.array(dg.MASS_TRUTH)) / r.sigma).round(3).tolist()}
    return res


def run_mine(args) -> None:
    import torch

    import paper_2505_12414_b200 as mf
    from paper_2505_12414_b200 import build as mf_build

    if int(os.environ.get("LOCAL_RANK", "0")) == 0:
        mf_build.build()   # no-op when the library is newer than its sources
    rank, world, local = _dist_setup(args.gpus)
    _barrier(world)
    torch.cuda.set_device(local)
    sampler = ClockSampler(local) if rank == 0 else None   # started early: it needs ~1 s to come up
    ctx = mf.Context(local)  # borrows torch's current stream on this device
    K = K_PARAMS

    # ---- inputs: R replicas of C1 (seeds 1, 2, ...; rank r uses its own seeds), resident in HBM
    pts = dg.gen_lambda_points(N_POINTS, 1001, dg.MASS_TRUTH, 3 * dg.mass_sigma_stat(N_EVENTS))
    models, host0 = [], None
    for r in range(N_REPLICAS):
        m = dg.gen_mass(N_EVENTS, seed=1 + r + 1000 * rank)
        if r == 0:
            host0 = m
        models.append(ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(m, dg.MASS_LO, dg.MASS_HI)))
    out = torch.zeros((N_POINTS, K + 2), dtype=torch.float64, device="cuda")
    out_ptrs = [out[i].data_ptr() for i in range(N_POINTS)]
    pts_c = np.ascontiguousarray(pts)
    calls_per_step = (N_POINTS + POINTS_PER_CALL - 1) // POINTS_PER_CALL

    def run_steps(first: int, count: int):
        """Steps first .. first+count-1: step s = the full sweep (all 1000 lambda points) on dataset replica s % 32,
        issued as mf_nll_grad_points calls of POINTS_PER_CALL points (one kernel launch each)."""
        for s_ in range(first, first + count):
            md = models[s_ % N_REPLICAS]
            for p in range(0, N_POINTS, POINTS_PER_CALL):
                md.nll_grad_points(pts_c[p:p + POINTS_PER_CALL], out_ptrs[p])

    run_steps(0, args.warmup)
    torch.cuda.synchronize()

    if sampler:
        sampler.wait_ready()
    launches0 = ctx.kernel_launches
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    _barrier(world)
    torch.cuda.synchronize()
    t_host0 = time.time()
    e0.record()
    run_steps(args.warmup, args.steps)
    e1.record()
    torch.cuda.synchronize()
    _barrier(world)
    t_host1 = time.time()
    ms = _max_over_ranks(float(e0.elapsed_time(e1)), world)
    launches = ctx.kernel_launches - launches0
    clocks = sampler.stop(t_host0, t_host1) if sampler else None

    res = out.cpu().numpy()
    if not (np.all(np.isfinite(res)) and np.all(res[:, K + 1] == 0)):
        raise RuntimeError("non-finite NLL / gradient in the timed steps")

    ms_per_step = ms / args.steps
    us_per_eval = 1e3 * ms_per_step / N_POINTS
    value = world * N_EVENTS * N_POINTS * args.steps / (ms * 1e-3)

    # the same evaluations as ONE KERNEL LAUNCH PER EVALUATION (7 points per call -> pipelined single evaluations, every
    # launch reading its replica's events from HBM): the number a minimiser sees when its points arrive one at a time.
    # Always SINGLE_LAUNCH_STEPS launches, whatever --steps says.
    def run_single_launch_steps(count: int):
        i = 0
        while i < count:
            p = i % N_POINTS
            c = min(7 - p % 7, count - i, N_POINTS - p)   # < 8 points per call: the library launches them one by one
            models[(i // 7) % N_REPLICAS].nll_grad_points(pts_c[p:p + c], out_ptrs[p])
            i += c

    n_single = SINGLE_LAUNCH_STEPS
    run_single_launch_steps(400)
    torch.cuda.synchronize()
    l0 = ctx.kernel_launches
    e0.record()
    run_single_launch_steps(n_single)
    e1.record()
    torch.cuda.synchronize()
    single_us = _max_over_ranks(float(e0.elapsed_time(e1)), world) * 1e3 / n_single
    single_launches = ctx.kernel_launches - l0

    # ---- e2e: the same step through the public API with HOST (pinned) inputs and HOST results, every step:
    # mf_dataset_upload (8 MB pinned host -> device) + mf_model_create + mf_nll_grad_sweep (1000 host lambda points in,
    # 1000 x (K+1) host results out through the library's pinned staging) + destroy
    pinned = torch.from_numpy(host0).pin_memory()
    host_view = pinned.numpy()
    e2e_steps = max(3, min(args.steps, 30))

    e2e_parts = []   # host seconds of the pieces of every timed step: upload, model, sweep, destroy

    def e2e_step(i: int):
        t0 = time.perf_counter()
        ds = ctx.dataset_upload(host_view, dg.MASS_LO, dg.MASS_HI)
        t1 = time.perf_counter()
        md = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ds)
        t2 = time.perf_counter()
        nll, g, nbad = md.nll_grad_sweep(pts_c)
        t3 = time.perf_counter()
        md.close()
        ds.close()
        e2e_parts.append((t1 - t0, t2 - t1, t3 - t2, time.perf_counter() - t3))
        return nll, nbad

    # warm-up: at least 3 steps and at least 0.3 s of them.  The PCIe link of an otherwise busy GPU takes some tens of ms of
    # host<->device traffic to reach its full speed (measured on this pool: the 8 MB upload takes 0.35-0.7 ms for the first
    # 30-100 ms after the traffic starts, 0.19 ms afterwards; the device-only phases before this point move no data)
    t_w = time.perf_counter()
    i = 0
    while i < 3 or time.perf_counter() - t_w < 0.3:
        e2e_step(i)
        i += 1
    e2e_warmup_steps = i
    torch.cuda.synchronize()
    _barrier(world)
    t = time.perf_counter()
    e2e_parts.clear()
    for i in range(e2e_steps):
        nll_h, nbad = e2e_step(i)
    torch.cuda.synchronize()
    e2e_s = _max_over_ranks(time.perf_counter() - t, world)
    e2e_median_ms = [round(float(v) * 1e3, 4) for v in np.median(np.array(e2e_parts), axis=0)]
    if nbad or not np.all(np.isfinite(nll_h)):
        raise RuntimeError("non-finite NLL in the e2e steps")
    # the smallest e2e unit a minimiser sees: upload + model + ONE synchronous evaluation + destroy
    def e2e_single(i: int):
        ds = ctx.dataset_upload(host_view, dg.MASS_LO, dg.MASS_HI)
        md = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ds)
        nll, g = md.nll_grad(pts_c[i % N_POINTS])
        md.close()
        ds.close()
    for i in range(3):
        e2e_single(i)
    t = time.perf_counter()
    for i in range(20):
        e2e_single(i)
    e2e_single_ms = 1e3 * (time.perf_counter() - t) / 20
    e2e = {"value": world * N_EVENTS * N_POINTS * e2e_steps / e2e_s, "unit": UNIT,
           "h2d_bytes_per_step": 8 * N_EVENTS + 8 * K * N_POINTS, "d2h_bytes_per_step": 8 * (K + 2) * N_POINTS,
           "steps": e2e_steps, "ms_per_step": 1e3 * e2e_s / e2e_steps,
           "what": "per step: mf_dataset_upload (pinned host -> device, 8 MB) + mf_model_create + mf_nll_grad_sweep "
                   "(1000 host lambda points -> 1000 x (-lnL, gradient) on the host) + destroy",
           "upload_plus_one_evaluation_ms": e2e_single_ms,
           "median_ms_upload_model_sweep_destroy": e2e_median_ms, "warmup_steps": e2e_warmup_steps}

    if rank != 0:
        return

    # ---- roofline of the dominant kernel (ALU bound; fp64-pipe instruction = 1 DFMA = 2 flop)
    from paper_2505_12414_b200 import probe
    peaks = {}
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            peaks = json.load(fh)
    except Exception:
        pass
    sm_max_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    n_sm = torch.cuda.get_device_properties(local).multi_processor_count
    peak_tflops = 2.0 * n_sm * NOMINAL_FP64_LANES_PER_SM * sm_max_mhz * 1e6 / 1e12
    measured_rate = probe.fp64_rate(local, torch.cuda.current_stream(local).cuda_stream)
    dmma = probe.dmma_rate(local, torch.cuda.current_stream(local).cuda_stream)   # fp64 tensor-core rate, DMMA + DFMA mix
    n_launches_timed = max(int(launches), 1)
    us_per_launch = 1e3 * ms / n_launches_timed
    achieved_tflops = 2.0 * MASS_FP64_INSTR_PER_EVENT * N_EVENTS * POINTS_PER_CALL / (us_per_launch * 1e-6) / 1e12
    traffic_all = {}
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as fh:
            traffic_all = json.load(fh)
    except Exception:
        pass
    roofline = {
        "bound": "alu", "achieved": achieved_tflops, "peak": peak_tflops, "unit": "TFLOP/s",
        "frac": achieved_tflops / peak_tflops, "traffic": traffic_all.get("nll_grad_batch_kernel<MassModel>/points"),
        "kernel": "nll_grad_batch_kernel<MassModel> (points mode)", "fp64_instr_per_event": MASS_FP64_INSTR_PER_EVENT,
        "launches_timed": n_launches_timed, "us_per_launch": us_per_launch, "evaluations_per_launch": POINTS_PER_CALL,
        "peak_how": f"derived: {n_sm} SMs x {NOMINAL_FP64_LANES_PER_SM} fp64 lanes x {sm_max_mhz:.0f} MHz x 2 flop",
        "peak_measured_dfma_chain": 2.0 * measured_rate / 1e12,
        "peak_measured_dmma": 2.0 * dmma["dmma_fma_per_s"] / 1e12,
        "dmma_plus_dfma_time_over_sum_of_times": dmma["mix_4dmma_8dfma_vs_sum"],
        "frac_of_measured_dfma_chain": achieved_tflops / (2.0 * measured_rate / 1e12),
        "one_launch_per_evaluation": {"us_per_evaluation": single_us, "evaluations": n_single, "gpu_launches": int(single_launches),
                                      "events_per_s": world * N_EVENTS / (single_us * 1e-6),
                                      "frac": 2.0 * MASS_FP64_INSTR_PER_EVENT * N_EVENTS / (single_us * 1e-6) / 1e12 / peak_tflops,
                                      "kernel": "nll_grad_kernel<MassModel>, programmatic dependent launch between evaluations"},
        "hbm_side": {"bytes_per_event": 8, "achieved_gbs": 8.0 * N_EVENTS / (us_per_eval * 1e-6) / 1e9,
                     "peak_gbs": peaks.get("hbm_gbs")},
    }
    in_region = (clocks or {}).get("samples_in_region", 0)
    headline_ok = bool(n_launches_timed >= 3 and in_region and in_region > 0)

    cpu = _cpu_baseline(sample_events=N_EVENTS, repeats=40)
    others = None
    if world == 1 and not args.no_extras:
        del models
        others = _other_workloads(torch, mf, ctx, peaks, traffic_all)

    launch_cfg = {"replicas": N_REPLICAS, "points_per_call": POINTS_PER_CALL,
                  "launch": f"{calls_per_step} nll_grad_batch_kernel<MassModel> launches per step (mf_nll_grad_points, "
                            f"{POINTS_PER_CALL} lambda points each; CTA tile = (lambda point, event chunk))"}
    print(json.dumps({
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": CONFIG, "launch_config": launch_cfg, "us_per_evaluation": us_per_eval,
        "headline_ok": headline_ok,
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu,
        "other_workloads": others,
    }))


def main() -> None:
    if len(sys.argv) >= 4 and sys.argv[1] == "--clock-sampler":
        _clock_sampler_main(int(sys.argv[2]), sys.argv[3])
        return
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=60, help="timed steps; one step = one sweep of 1000 lambda points (~2.3 ms)")
    ap.add_argument("--warmup", type=int, default=8)
    ap.add_argument("--impl", choices=["mine", "reference"], default="mine")
    ap.add_argument("--no-extras", action="store_true", help="skip the C0/C2/C3/C4 summary (other_workloads)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    args.steps = max(args.steps, 1)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_mine(args)


if __name__ == "__main__":
    main()
