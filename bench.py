#!/usr/bin/env python
"""bench.py — throughput of the fused NLL + analytic-gradient hot path on B200.

Workload (BASELINE.json configs[1], "C1"): the 1D Gaussian+exponential mass model, N = 1,000,000
fp64 events, 4 free parameters; one STEP = one complete pass of the hot path (S2 parameter-only
constants on the host, S3 per-event value + gradient, S4/S5 reductions, S6 K+2 doubles out) at a
new parameter point drawn within +-3 sigma_stat of the truth (1,000 seeded points, cycled).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl mine|reference]

Timing rules followed: W >= 3 warm-up steps; the timed steps rotate over R dataset replicas whose
total size (R x 8 MB = 256 MB) exceeds the 126 MB L2, so every step reads its events from HBM
("l2": "inputs larger than L2" in config); CUDA events on the launching stream; max over ranks;
SM clocks and throttle reasons sampled (NVML, separate process) during the timed region.

`value` is events/s with the data resident in HBM; `e2e` is the same metric through the public API
with HOST inputs (pinned), i.e. mf_dataset_upload + mf_model_create + mf_nll_grad every step.
`roofline` is for the dominant kernel nll_grad_kernel<MassModel> (ALU bound);
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
N_POINTS = 1000
N_REPLICAS = 32
METRIC = "nll_grad_event_evals_per_s"
UNIT = "events/s"
WORKLOAD = "C1: 1D Gaussian+exponential mass model, N=1e6 fp64 events, K=4, NLL+gradient at 1000 seeded lambda points"
# fp64-pipe thread-instructions per event of the shipped mass kernel's fast path (counted from
# SASS); never more than the plain two-exponential form's hand count (100).
MASS_FP64_INSTR_PER_EVENT = 26.0
POINTS_PER_CALL = 500  # evaluations per mf_nll_grad_points call (ONE launch: CTA tile = (point, event chunk))
NOMINAL_FP64_LANES_PER_SM = 64  # B200: 4 SMSPs x 16 fp64 FMA lanes


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
            "sample": f"{repeats} NLL+gradient calls on the first {sample_events} events of the C1 dataset (seed 1)",
            "single_thread_value": best[1], "host_cores": os.cpu_count()}


def run_reference(args) -> None:
    """--impl reference: the CPU oracle timed as the reference arm (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    sample = 200_000
    m = dg.gen_mass(N_EVENTS, seed=1)[:sample]
    pts = dg.gen_lambda_points(N_POINTS, 1001, dg.MASS_TRUTH, 3 * dg.mass_sigma_stat(N_EVENTS))
    nt = oracle.max_threads()
    steps = min(args.steps, 400)   # each step ~ 0.05-0.1 s of CPU: keeps the arm within minutes
    warm = min(args.warmup, 5)
    for i in range(warm):
        oracle.nll_grad(oracle.MASS, m, pts[i % N_POINTS], dg.MASS_LO, dg.MASS_HI, nthreads=nt)
    t = time.perf_counter()
    for i in range(steps):
        oracle.nll_grad(oracle.MASS, m, pts[i % N_POINTS], dg.MASS_LO, dg.MASS_HI, nthreads=nt)
    dt = time.perf_counter() - t
    value = sample * steps / dt
    desc = f"each step = one oracle NLL+gradient call on the first {sample} events of C1 ({nt} threads)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": warm, "ms_per_step": 1e3 * dt / steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "n_events": N_EVENTS, "sample": desc},
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


def _other_workloads(torch, mf, ctx, peaks) -> dict:
    """The other BASELINE.json configs, each timed the same way (device-resident inputs, CUDA events,
    inputs larger than the 126 MB L2 or rotated over replicas that are).  Parity for these is in tests/."""
    # HBM peak: the driver's measured copy bandwidth, else the profiling guide's stated fallback (6.65 TB/s, "of fallback")
    hbm = float(peaks.get("hbm_gbs", 0.0)) or 6650.0
    hbm_how = "MEASURED_PEAKS.json hbm_gbs" if peaks.get("hbm_gbs") else "fallback of B200_PROFILING.md (6.65 TB/s)"
    res = {"hbm_peak_source": hbm_how}
    # C2: 3D angular, N = 1e6, nine cached basis columns = 72 B/event (HBM bound)
    ev = dg.gen_angular(1_000_000, seed=2)
    ms = [ctx.model_create(mf.MF_ANGULAR_KSTMUMU, ctx.dataset_upload(ev)) for _ in range(3)]   # 3 x 72 MB > L2
    us = _time_points(torch, ms, dg.ANG_TRUTH, 8, 600)
    gbs = 72.0 * 1_000_000 / us / 1e3
    res["C2_angular_1e6"] = {"us_per_eval": us, "events_per_s": 1e6 / (us * 1e-6), "kernel": "nll_grad_tma_kernel<AngularModel>",
                             "roofline": {"bound": "hbm", "achieved": gbs, "peak": hbm, "unit": "GB/s",
                                          "frac": gbs / hbm if hbm else None, "bytes_per_event": 72},
                             "l2": "3 model replicas x 72 MB rotated"}
    t = time.perf_counter()
    r = ms[0].fit(dg.ANG_TRUTH)
    res["C2_angular_1e6"]["fit_s"] = time.perf_counter() - t
    res["C2_angular_1e6"]["fit_calls"] = r.n_calls
    del ms, ev
    # C3: 4D, N = 2e6, 12 columns = 96 B/event (192 MB > L2)
    ev = dg.gen_4d(2_000_000, seed=3)
    m4s = [ctx.model_create(mf.MF_MASS_X_ANGULAR, ctx.dataset_upload(ev, dg.MASS_LO, dg.MASS_HI)) for _ in range(2)]
    m4 = m4s[0]
    us = _time_points(torch, m4s, dg.FOURD_TRUTH, 16, 400)   # 2 x 192 MB of columns, alternating
    gbs = 96.0 * 2_000_000 / us / 1e3
    res["C3_4d_2e6"] = {"us_per_eval": us, "events_per_s": 2e6 / (us * 1e-6), "kernel": "nll_grad_tma_kernel<FourDModel>",
                        "roofline": {"bound": "hbm", "achieved": gbs, "peak": hbm, "unit": "GB/s",
                                     "frac": gbs / hbm if hbm else None, "bytes_per_event": 96},
                        "l2": "2 model replicas x 192 MB of columns, alternating every evaluation"}
    t = time.perf_counter()
    r = m4.fit(dg.FOURD_TRUTH)
    res["C3_4d_2e6"]["fit_s"] = time.perf_counter() - t
    res["C3_4d_2e6"]["fit_calls"] = r.n_calls
    del m4, m4s, ev
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
    res["toy_study_4096x1e4_on_device"] = {
        "ms_per_toy": 1e3 * ts_s / T, "toys_per_s": T / ts_s, "converged": int(ts.converged.sum()),
        "what": "mf_toy_study_mass: mf_generate_mass (4096 toys x 1e4 events, Philox4x32-10) + mf_model_create + mf_fit_batch "
                "(Newton on the analytic Hessian + HESSE); no event crosses PCIe",
        "generation_us": gen_us, "generated_events_per_s": T * n / (gen_us * 1e-6),
        "paper_context": "MoreFit OpenCL GPU (analytic), Titan V: 1.62 ms per toy at 1e4 events (PAPER.md:191); another machine"}
    # C0: N = 1e4, one call + full fit (latency bound: no roofline claim)
    m0 = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(dg.gen_mass(10_000, seed=0), dg.MASS_LO, dg.MASS_HI))
    m0.nll_grad(dg.MASS_START)
    t = time.perf_counter()
    for _ in range(200):
        m0.nll_grad(dg.MASS_START)
    lat = (time.perf_counter() - t) / 200
    t = time.perf_counter()
    r = m0.fit(dg.MASS_START)
    res["C0_mass_1e4"] = {"sync_call_us": lat * 1e6, "fit_s": time.perf_counter() - t, "fit_calls": r.n_calls,
                          "converged": bool(r.converged)}
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
    K = 4

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
    lam_rows = [np.ascontiguousarray(pts[i]) for i in range(N_POINTS)]
    pts_c = np.ascontiguousarray(pts)

    def run_steps(first: int, count: int):
        """Steps first .. first+count-1: step i = one NLL+gradient evaluation at lambda point i % 1000 on dataset
        replica (i // 500) % 32; 500 steps per mf_nll_grad_points call."""
        i, end = first, first + count
        while i < end:
            p = i % N_POINTS
            c = min(POINTS_PER_CALL - p % POINTS_PER_CALL, end - i, N_POINTS - p)
            models[(i // POINTS_PER_CALL) % N_REPLICAS].nll_grad_points(pts_c[p:p + c], out_ptrs[p])
            i += c

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
    n_done = min(args.steps + args.warmup, N_POINTS)
    if not (np.all(np.isfinite(res[:n_done])) and np.all(res[:n_done, K + 1] == 0)):
        raise RuntimeError("non-finite NLL / gradient in the timed steps")

    ms_per_step = ms / args.steps
    value = world * N_EVENTS * args.steps / (ms * 1e-3)

    # the same steps as ONE KERNEL LAUNCH PER STEP (8 points per call -> pipelined single evaluations, every launch
    # reading its replica's events from HBM): the number a minimiser sees when its points arrive one at a time
    def run_single_launch_steps(count: int):
        i = 0
        while i < count:
            p = i % N_POINTS
            c = min(8 - p % 8, count - i)
            models[(i // 8) % N_REPLICAS].nll_grad_points(pts_c[p:p + c], out_ptrs[p])
            i += c

    n_single = min(args.steps, 4000)
    run_single_launch_steps(200)
    torch.cuda.synchronize()
    l0 = ctx.kernel_launches
    e0.record()
    run_single_launch_steps(n_single)
    e1.record()
    torch.cuda.synchronize()
    single_us = _max_over_ranks(float(e0.elapsed_time(e1)), world) * 1e3 / n_single
    single_launches = ctx.kernel_launches - l0

    # ---- e2e: public API with HOST (pinned) inputs, upload + model + evaluation every step
    pinned = torch.from_numpy(host0).pin_memory()
    host_view = pinned.numpy()
    e2e_steps = max(3, min(args.steps, 100))

    def e2e_step(i: int):
        ds = ctx.dataset_upload(host_view, dg.MASS_LO, dg.MASS_HI)
        md = ctx.model_create(mf.MF_MASS_GAUSS_EXP, ds)
        nll, g = md.nll_grad(lam_rows[i % N_POINTS])
        md.close()
        ds.close()
        return nll

    for i in range(3):
        e2e_step(i)
    torch.cuda.synchronize()
    _barrier(world)
    t = time.perf_counter()
    for i in range(e2e_steps):
        e2e_step(i)
    torch.cuda.synchronize()
    e2e_s = _max_over_ranks(time.perf_counter() - t, world)
    e2e = {"value": world * N_EVENTS * e2e_steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": 8 * N_EVENTS,
           "d2h_bytes_per_step": 8 * (K + 2), "steps": e2e_steps, "ms_per_step": 1e3 * e2e_s / e2e_steps,
           "what": "mf_dataset_upload (pinned host -> device) + mf_model_create + mf_nll_grad + destroy, every step"}

    if rank != 0:
        return

    # ---- roofline of the dominant kernel (ALU bound; fp64-pipe instruction = 1 DFMA = 2 flop)
    peaks = {}
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            peaks = json.load(fh)
    except Exception:
        pass
    sm_max_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    n_sm = torch.cuda.get_device_properties(local).multi_processor_count
    peak_tflops = 2.0 * n_sm * NOMINAL_FP64_LANES_PER_SM * sm_max_mhz * 1e6 / 1e12
    measured_rate = ctx.probe_fp64_rate()
    achieved_tflops = 2.0 * MASS_FP64_INSTR_PER_EVENT * N_EVENTS / (ms_per_step * 1e-3) / 1e12
    traffic = None
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as fh:
            traffic = json.load(fh).get("nll_grad_batch_kernel<MassModel>/points")
    except Exception:
        pass
    roofline = {
        "bound": "alu", "achieved": achieved_tflops, "peak": peak_tflops, "unit": "TFLOP/s",
        "frac": achieved_tflops / peak_tflops, "traffic": traffic,
        "kernel": "nll_grad_batch_kernel<MassModel> (points mode)", "fp64_instr_per_event": MASS_FP64_INSTR_PER_EVENT,
        "peak_how": f"derived: {n_sm} SMs x {NOMINAL_FP64_LANES_PER_SM} fp64 lanes x {sm_max_mhz:.0f} MHz x 2 flop",
        "peak_measured_dfma_chain": 2.0 * measured_rate / 1e12,
        "frac_of_measured_dfma_chain": achieved_tflops / (2.0 * measured_rate / 1e12),
        "one_launch_per_step": {"us_per_step": single_us, "steps": n_single, "gpu_launches": int(single_launches),
                                "events_per_s": world * N_EVENTS / (single_us * 1e-6),
                                "frac": 2.0 * MASS_FP64_INSTR_PER_EVENT * N_EVENTS / (single_us * 1e-6) / 1e12 / peak_tflops,
                                "kernel": "nll_grad_kernel<MassModel>, programmatic dependent launch between steps"},
        "hbm_side": {"bytes_per_event": 8, "achieved_gbs": 8.0 * N_EVENTS / (ms_per_step * 1e-3) / 1e9,
                     "peak_gbs": peaks.get("hbm_gbs")},
    }

    cpu = _cpu_baseline(sample_events=N_EVENTS, repeats=40)
    others = None
    if world == 1 and not args.no_extras:
        del models
        others = _other_workloads(torch, mf, ctx, peaks)

    print(json.dumps({
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "n_events": N_EVENTS, "n_params": K, "lambda_points": N_POINTS,
                   "replicas": N_REPLICAS, "points_per_call": POINTS_PER_CALL,
                   "l2": "inputs larger than L2: calls rotate over 32 x 8 MB dataset replicas, so each call first reads its "
                         "events from HBM; the 500 evaluations of one call re-read them from L2 by design (8 B/event, ALU bound)",
                   "launch": "one nll_grad_batch_kernel<MassModel> launch per mf_nll_grad_points call of 500 steps "
                             "(CTA tile = (lambda point, event chunk))"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu,
        "other_workloads": others,
    }))


def main() -> None:
    if len(sys.argv) >= 4 and sys.argv[1] == "--clock-sampler":
        _clock_sampler_main(int(sys.argv[2]), sys.argv[3])
        return
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20000)
    ap.add_argument("--warmup", type=int, default=100)
    ap.add_argument("--impl", choices=["mine", "reference"], default="mine")
    ap.add_argument("--no-extras", action="store_true", help="skip the C0/C2/C3/C4 summary (other_workloads)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_mine(args)


if __name__ == "__main__":
    main()
