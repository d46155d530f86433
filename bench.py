#!/usr/bin/env python
"""bench.py -- split-step throughput of libspgpe on BASELINE.json's metric workload (config 4: 2048 x 2048,
two components, complex128, real time, dt = 2.5e-4), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload 4|4c64|3|2|1]

A "step" is one Strang step of the whole hot path (a6 in imaginary time).
  value      : grid-point-steps/s (P = nx*ny counted once, not per component) over all N replicas, state and
               fields resident in HBM, CUDA events around ONE spgpe_step(K) call, max over ranks; --repeats (5)
               such regions of exactly K steps are timed and the median one is reported with the MAD (`repeats`).
  e2e        : the same metric through the C ABI with HOST buffers: set_potential/raman/zeeman_host +
               set_psi_host (pinned) -> spgpe_step(K) -> get_psi_host, copies inside the timed region (the
               paper's usage: order parameter in, M steps, order parameter out).
  roofline   : dominant kernel (the longer of the row pass and the column pass), timed per launch with CUDA
               events on the handle's stream (spgpe_profile) over a second region of K steps.
  cpu_baseline: the oracle as it stands, on this box's host cores, a bounded sample of the same workload.
  cufft_comparison: context only -- the paper's own formulation (torch.fft.fft2 = cuFFT, Hadamard products as torch
               elementwise operations) timed on this GPU for the same workload, and the relative L2 difference between
               the library and that independent GPU path after the same steps (N = 1, states up to 256 MiB).
Multi-GPU: replicas only: every rank steps its own copy of the workload, no collective
on the data path; value = N * P * K / max-over-ranks time.
--impl reference times the oracle (oracle/) on the host cores; rank 0 only.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "split-step grid-point-steps/s"
UNIT = "grid-point-steps/s"
# algorithmic bytes per grid point per launch: psi read + written once per
# pass; the row pass also reads the fields in use (one real per point each)
WORKLOADS = {
    "4": dict(cfg=4, dtype="c128"), "4c64": dict(cfg=4, dtype="c64"), "3": dict(cfg=3, dtype="c128"),
    "2": dict(cfg=2, dtype="c128"), "1": dict(cfg=1, dtype="c128"), "5": dict(cfg=5, dtype="c64"),
}


KERNEL_SOURCES = ("common.cuh", "radix.cuh", "line_fft.cuh", "su2.cuh", "pass_x.cuh", "pass_y.cuh", "launch.cuh")


def kernel_source_sha16() -> str:
    """Hash of the sources the two pass kernels are compiled from (stamps profiles/r2_traffic.json)."""
    import hashlib
    h = hashlib.sha256()
    for name in KERNEL_SOURCES:
        with open(os.path.join(ROOT, "paper_2010_15069_b200", "csrc", name), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def read_traffic(workload: str, kernel: str):
    """(bytes, source): dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu --set full
    summary profiles/r2_traffic.json.  The file names the commit and the hash of the kernel sources it was captured
    from; when those sources have changed since, the number is stale and None is reported instead."""
    path = os.path.join(ROOT, "profiles", "r2_traffic.json")
    try:
        with open(path) as f:
            d = json.load(f)
        if d.get("workload") != workload:
            return None, f"profiles/r2_traffic.json holds {d.get('workload')}, not this workload"
        if d.get("kernel_source_sha16") != kernel_source_sha16():
            return None, "profiles/r2_traffic.json is stale (kernel sources changed since the capture)"
        return d["kernels"][kernel]["bytes_per_launch"], (f"ncu --set full at commit {d.get('captured_at_commit')}, "
                                                           "profiles/r2_ncu_full.md")
    except Exception as e:
        return None, f"no traffic record ({type(e).__name__})"


def read_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """SM clock and throttle reasons sampled through NVML while the timed regions run."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz, self.ok = [], set(), None, False
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.dev = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.dev, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:  # NVML missing: report that, do not fail the bench
            self.err = repr(e)

    def _run(self):
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4),
            "hw_power_brake": getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80),
        }
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.dev, nv.NVML_CLOCK_SM)))
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.dev))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.dev))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.005)

    def start(self):
        if self.ok:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        if self._thr:
            self._stop.set()
            self._thr.join()
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "note": "NVML unavailable"}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def oracle_sample(w_cfg: int, dtype: str, budget_s: float, steps: int, threads: int = 0):
    """Times the oracle on a proxy grid of the same recipe, chosen so that `steps` steps fit the budget.
    threads = 0: every host core (OpenMP), else that many.  Returns (grid-point-steps/s, threads, description,
    seconds per step)."""
    import oracle as orc
    import workloads as wl
    all_threads = orc.max_threads()
    orc.set_threads(threads or all_threads)
    threads = threads or all_threads
    full = wl.CONFIGS[w_cfg]["n"]
    n, sec = 64, None
    while True:
        w = wl.make_workload(w_cfg, n=n, dtype=dtype)
        p = orc.params_of(w)
        cnt, dt, imag = w.schedule[0]
        t0 = time.perf_counter()
        orc.step(w.psi0, w.V, w.Omega, w.delta, p, 1, dt, imag)
        sec = time.perf_counter() - t0
        if n >= full or 4.2 * sec * steps > budget_s:  # the next size costs ~4.2x
            break
        n *= 2
    steps = int(min(200, max(steps, 0.5 * budget_s / max(sec, 1e-3))))  # about half the budget of CPU work
    t0 = time.perf_counter()
    orc.step(w.psi0, w.V, w.Omega, w.delta, p, steps, dt, imag)
    sec = (time.perf_counter() - t0) / steps
    orc.set_threads(all_threads)
    what = (f"{steps} oracle steps (fp64, own radix-2 FFT, {threads} OpenMP thread{'s' if threads > 1 else ''}) of "
            f"config {w_cfg}'s recipe on a {n}x{n} grid (full size {full}x{full}), "
            f"{'imaginary' if imag else 'real'} time")
    return n * n / sec, threads, what, sec


def cufft_comparison(w, spec, steps: int, warmup: int, ours_after_steps=None):
    """The paper's own formulation of the same step, timed on this GPU as CONTEXT (BASELINE.json north_star: "a
    cuFFT-plus-elementwise-kernel version of the same step may be timed as a comparison"; PyTorch
    arrays, torch.fft (cuFFT) and Hadamard products): torch.fft.fft2 / ifft2 on a [2, ny, nx] array, the k-space phase
    and the closed 2x2 real-space factor as plain torch elementwise operations.  Not part of the product path and not
    the oracle; bench.py only.  Returns a dict for the JSON line.  ours_after_steps: the library's psi (numpy
    [ny, nx, 2]) after `steps` steps from the same initial state, for a cross-check of the two GPU paths."""
    import torch
    dev = torch.device("cuda", torch.cuda.current_device())
    cdt = torch.complex128 if spec["dtype"] == "c128" else torch.complex64
    rdt = torch.float64 if spec["dtype"] == "c128" else torch.float32
    cnt, dt, imag = w.schedule[0]
    tau = 0.5 * dt
    ny, nx = w.ny, w.nx
    def field(f):
        return torch.zeros((ny, nx), dtype=rdt, device=dev) if f is None else torch.from_numpy(np.ascontiguousarray(f)).to(dev, rdt)
    V, Om, De = field(w.V), field(w.Omega), field(w.delta)
    psi = torch.from_numpy(np.ascontiguousarray(np.moveaxis(w.psi0, 2, 0))).to(dev, cdt)  # [2, ny, nx]
    kx = torch.from_numpy(2.0 * np.pi * np.fft.fftfreq(nx, d=w.Lx / nx)).to(dev)
    ky = torch.from_numpy(2.0 * np.pi * np.fft.fftfreq(ny, d=w.Ly / ny)).to(dev)
    K = torch.stack([0.5 * ((kx + w.k_L) ** 2)[None, :] + 0.5 * (ky ** 2)[:, None],
                     0.5 * ((kx - w.k_L) ** 2)[None, :] + 0.5 * (ky ** 2)[:, None]])          # [2, ny, nx] fp64
    kphase = (torch.exp(-K * dt) if imag else torch.exp(-1j * K * dt)).to(cdt)
    cell = (w.Lx / nx) * (w.Ly / ny)
    targets = cell * (psi.abs() ** 2).sum(dim=(1, 2))

    def half(psi):
        u, d = psi[0], psi[1]
        nu, nd = u.real ** 2 + u.imag ** 2, d.real ** 2 + d.imag ** 2
        d_up = V + w.g_uu * nu + w.g_ud * nd + 0.5 * De
        d_dn = V + w.g_dd * nd + w.g_ud * nu - 0.5 * De
        a, bz, bx = 0.5 * (d_up + d_dn), 0.5 * (d_up - d_dn), 0.5 * Om
        th = torch.sqrt(bx * bx + bz * bz) * tau
        if imag:
            c = torch.cosh(th)
            s = tau * torch.where(th.abs() < 1e-4, 1.0 + th * th / 6.0, torch.sinh(th) / th)
            e = torch.exp(-a * tau)
            return torch.stack([e * (c * u - s * (bz * u + bx * d)), e * (c * d - s * (bx * u - bz * d))])
        c = torch.cos(th)
        s = tau * torch.sinc(th / np.pi)          # sin(theta)/|b|
        ph = torch.polar(torch.ones_like(a), -a * tau)
        return torch.stack([ph * (c * u - 1j * s * (bz * u + bx * d)), ph * (c * d - 1j * s * (bx * u - bz * d))])

    def step(psi):
        psi = half(psi)
        psi = torch.fft.ifft2(torch.fft.fft2(psi, dim=(1, 2)) * kphase, dim=(1, 2))
        psi = half(psi)
        if imag:
            n = cell * (psi.abs() ** 2).sum(dim=(1, 2))
            sc = torch.sqrt(targets / n) if w.norm_mode == 0 else torch.sqrt(targets.sum() / n.sum()).expand(2)
            psi = psi * sc[:, None, None].to(rdt)
        return psi

    q = psi
    for _ in range(warmup):
        q = step(q)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    q = psi
    e0.record()
    for _ in range(steps):
        q = step(q)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    out = {"kind": "torch.fft (cuFFT) + torch elementwise operations: the paper's formulation of the step, this GPU",
           "ms_per_step": ms, "value": w.points / (ms * 1e-3), "unit": UNIT, "steps": steps,
           "note": "context, not part of the product path; library calls only"}
    if ours_after_steps is not None:
        ref = np.moveaxis(q.cpu().numpy(), 0, 2).astype(np.complex128)
        got = ours_after_steps.astype(np.complex128)
        out["rel_l2_ours_vs_this"] = float(np.linalg.norm((got - ref).ravel()) / np.linalg.norm(ref.ravel()))
    return out


def whole_job_value(points: int, steps: int, ms_local: float, world: int, group=None):
    """(value, ms) of the replicas-only job: every rank steps its own copy; the job's time is the max over ranks
    (all_reduce MAX on whatever backend the group has) and value = world * points * steps / time."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms_local], dtype=torch.float64)
    if world > 1:
        if dist.get_backend(group) == "nccl":
            t = t.cuda()
        dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    ms = float(t.item())
    return world * points * steps / (ms * 1e-3), ms


def run_reference(args, wname):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    spec = WORKLOADS[wname]
    import oracle as orc
    import workloads as wl
    threads = orc.max_threads()
    full = wl.CONFIGS[spec["cfg"]]["n"]
    total = args.steps + args.warmup
    # pick the largest proxy grid whose whole run fits ~150 s
    n = 64
    while n < full:
        w = wl.make_workload(spec["cfg"], n=n, dtype=spec["dtype"])
        p = orc.params_of(w)
        cnt, dt, imag = w.schedule[0]
        t0 = time.perf_counter()
        orc.step(w.psi0, w.V, w.Omega, w.delta, p, 1, dt, imag)
        sec = time.perf_counter() - t0
        if 4.2 * sec * total > 150.0:
            break
        n *= 2
    w = wl.make_workload(spec["cfg"], n=n, dtype=spec["dtype"])
    p = orc.params_of(w)
    cnt, dt, imag = w.schedule[0]
    psi = orc.step(w.psi0, w.V, w.Omega, w.delta, p, args.warmup, dt, imag)
    t0 = time.perf_counter()
    orc.step(psi, w.V, w.Omega, w.delta, p, args.steps, dt, imag)
    el = time.perf_counter() - t0
    value = n * n * args.steps / el
    sample = (f"each step = one oracle Strang step of config {spec['cfg']}'s recipe on a {n}x{n} proxy grid "
              f"(full size {full}x{full}); fp64, own radix-2 FFT, OpenMP over lines")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * el / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"config {spec['cfg']} recipe, {n}x{n} proxy of {full}x{full}, "
                               f"{spec['dtype']} inputs, oracle on host cores"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_ours(args, wname):
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: libspgpe has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    import paper_2010_15069_b200 as sp
    import workloads as wl
    sp.lib()  # fails loudly when libspgpe.so is missing

    spec = WORKLOADS[wname]
    w = wl.make_workload(spec["cfg"], dtype=spec["dtype"])
    cnt, dt, imag = w.schedule[0]
    K, W = args.steps, args.warmup
    P = w.points
    stream = torch.cuda.Stream()
    h = sp.from_workload(w, stream=stream.cuda_stream)
    cdt, rdt = h._np_dtypes
    esz = np.dtype(cdt).itemsize
    rsz = np.dtype(rdt).itemsize
    nfields = sum(f is not None for f in (w.V, w.Omega, w.delta))
    psi_bytes = 2 * P * esz

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed_region(fn):
        """One region of exactly K steps: barrier + synchronize, CUDA events on the handle's stream, barrier +
        synchronize; returns the max over ranks in ms."""
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(stream):
            e0.record(stream)
            fn()
            e1.record(stream)
        barrier()
        return whole_job_value(P, K, e0.elapsed_time(e1), world)[1]

    sampler = ClockSampler(local)
    # ---- device-resident throughput --------------------------------------------------------------------
    sp.spgpe_step(h, W, dt, imag)
    sp.spgpe_synchronize(h)
    sampler.start()
    l0 = sp.spgpe_launch_count(h)
    # the paper's statistic: REPEATS regions of exactly K steps each, median and
    # median absolute deviation; `value` and `ms_per_step` are the median region's
    region_ms = [timed_region(lambda: sp.spgpe_step(h, K, dt, imag)) for _ in range(args.repeats)]
    launches = (sp.spgpe_launch_count(h) - l0) // args.repeats
    ms = float(np.median(region_ms))
    mad_ms = float(np.median(np.abs(np.array(region_ms) - ms)))
    # ---- optional: the same K steps replayed from a CUDA graph of one captured spgpe_step(K) call -----------
    graph_leg = None
    if args.graph:
        g = torch.cuda.CUDAGraph()
        with torch.cuda.stream(stream):
            with torch.cuda.graph(g, stream=stream):
                sp.spgpe_step(h, K, dt, imag)
        g_ms = [timed_region(lambda: g.replay()) for _ in range(args.repeats)]
        gm = float(np.median(g_ms))
        graph_leg = {"ms_per_step": gm / K, "ms_per_step_mad": float(np.median(np.abs(np.array(g_ms) - gm))) / K,
                     "ms_per_step_all": [m / K for m in g_ms],
                     "note": "the caller captured one spgpe_step(K) call (stream capture) and replays it; "
                             "context, `value` is the plain call's"}
        del g
    # ---- per-launch durations of the two pass kernels (second region of K steps) -----------------------
    sp.spgpe_profile(h, True)
    sp.spgpe_step(h, K, dt, imag)
    kms, kcnt = sp.spgpe_profile_read(h)
    sp.spgpe_profile(h, False)
    clocks = sampler.stop()
    # ---- end to end through the host-buffer calls --------------------------------------------------------
    pin = torch.from_numpy(np.ascontiguousarray(w.psi0, dtype=cdt)).pin_memory()
    pout = torch.empty_like(pin).pin_memory()
    fields = [None if f is None else torch.from_numpy(np.ascontiguousarray(f, dtype=rdt)).pin_memory()
              for f in (w.V, w.Omega, w.delta)]
    L = sp.lib()

    def e2e_job():
        for name, f in zip(("potential", "raman", "zeeman"), fields):
            sp._check(getattr(L, f"spgpe_set_{name}_host")(h.ptr, None if f is None else f.data_ptr()))
        sp._check(L.spgpe_set_psi_host(h.ptr, pin.data_ptr()))
        sp._check(L.spgpe_step(h.ptr, K, dt, imag))
        sp._check(L.spgpe_get_psi_host(h.ptr, pout.data_ptr()))

    e2e_job()  # warm-up (page-locks, first-touch)
    barrier()
    t0 = time.perf_counter()
    e2e_job()  # ends with a stream synchronise inside get_psi_host
    barrier()
    e2e_s = torch.tensor([time.perf_counter() - t0], device="cuda", dtype=torch.float64)
    if world > 1:
        dist.all_reduce(e2e_s, op=dist.ReduceOp.MAX)
    e2e_s = float(e2e_s.item())
    finite = bool(np.isfinite(pout.numpy().view(rdt)).all())
    norms = sp.spgpe_norm(h)

    if rank == 0:
        peak, peak_src = read_peaks()
        # dominant kernel = the pass with the longer average launch
        avg = [kms[i] / max(1, kcnt[i]) for i in range(2)]
        dom = 0 if avg[0] >= avg[1] else 1
        bytes_pt = [2 * 2 * esz + nfields * rsz, 2 * 2 * esz]  # row pass: psi r+w + fields; column pass: psi r+w
        achieved = bytes_pt[dom] * P / (avg[dom] * 1e-3) / 1e9
        step_bytes = (bytes_pt[0] + bytes_pt[1]) * P
        flops_pt = 20.0 * np.log2(float(P)) + 360.0
        dfma_tf = sp.spgpe_probe_dfma(stream.cuda_stream)
        ffma_tf = sp.spgpe_probe_ffma(stream.cuda_stream)
        traffic, traffic_src = read_traffic(w.name, ["pass_x_kernel", "pass_y_kernel"][dom])
        line = {
            "metric": METRIC, "value": world * P * K / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": K,
            "warmup": W, "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64" if spec["dtype"] == "c128" else "f32", "data": "synthetic",
            "config": {"workload": w.name, "grid": [w.nx, w.ny], "storage": spec["dtype"],
                       "arithmetic": "fp64 throughout" if spec["dtype"] == "c128" else
                                     "fp32 transforms with two-float twiddles and phase factors, fp64 per-point "
                                     "2x2 exponential and reductions (DESIGN.md R-14)",
                       "time": "imaginary" if imag else "real", "dt": dt, "parallelism": "replicas only",
                       "l2": f"state {psi_bytes >> 20} MiB + fields {(nfields * P * rsz) >> 20} MiB per replica; "
                             + ("larger than the 126 MB L2, no flush" if psi_bytes > 126e6 else
                                "fits L2: the HBM roofline is not the binding bound")},
            "repeats": {"regions": args.repeats, "steps_per_region": K, "ms_per_step_median": ms / K,
                        "ms_per_step_mad": mad_ms / K, "ms_per_step_all": [r / K for r in region_ms]},
            "steps_per_s": world * K / (ms * 1e-3),
            "step_hbm_gbs": step_bytes / (ms / K * 1e-3) / 1e9,
            "step_roofline_frac": step_bytes / (ms / K * 1e-3) / 1e9 / peak,
            "roofline": {"bound": "hbm", "kernel": ["row pass (pass_x_kernel / row32_kernel)",
                                                    "column pass (pass_y_db_kernel / col32_kernel)"][dom],
                         "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": traffic, "traffic_source": traffic_src,
                         "algorithmic_bytes": bytes_pt[dom] * P, "peak_source": peak_src,
                         "avg_launch_us": {"row_pass": 1e3 * avg[0], "column_pass": 1e3 * avg[1]},
                         "launches_timed": kcnt, "bytes_per_point": bytes_pt},
            # second bound of BASELINE.json's roofline definition: nominal flops (20 log2(P) + 360 per point and step,
            # SURVEY.md 8(d)) against the FP64 FMA peak measured on this device by spgpe_probe_dfma
            "roofline_fp64": {"bound": "alu", "achieved": flops_pt * P / (ms / K * 1e-3) / 1e12, "peak": dfma_tf,
                              "unit": "TFLOP/s", "frac": flops_pt * P / (ms / K * 1e-3) / 1e12 / dfma_tf,
                              "flops_per_point_step": flops_pt,
                              "peak_source": "measured in this run (DFMA loop, 2 flops per FMA)"},
            **({} if spec["dtype"] == "c128" else {
                # complex64: the transforms' flops (20 log2 P per point and step) against the measured fp32 FMA peak
                "roofline_fp32": {"bound": "alu", "achieved": 20.0 * np.log2(float(P)) * P / (ms / K * 1e-3) / 1e12,
                                  "peak": ffma_tf, "unit": "TFLOP/s",
                                  "frac": 20.0 * np.log2(float(P)) * P / (ms / K * 1e-3) / 1e12 / ffma_tf,
                                  "peak_source": "measured in this run (FFMA loop, 2 flops per FMA)"}}),
            "e2e": {"value": world * P * K / e2e_s, "unit": UNIT,
                    "h2d_bytes_per_step": (psi_bytes + nfields * P * rsz) / K, "d2h_bytes_per_step": psi_bytes / K,
                    "job": f"fields + psi host->device, spgpe_step({K}), psi device->host; {e2e_s:.4f} s"},
            "gpu_launches": int(launches), "clocks": clocks, "finite": finite, "norms": list(map(float, norms)),
        }
        if graph_leg is not None:
            line["graph_replay"] = graph_leg
        if world == 1 and not args.no_cufft and psi_bytes <= (1 << 28):
            # context: the paper's formulation (torch.fft + elementwise torch operations) on this GPU, and a cross-check
            # of the library against it after the same number of steps from the same initial state
            n_cmp = min(K, 20)
            h2 = sp.from_workload(w, stream=stream.cuda_stream)
            sp.spgpe_step(h2, n_cmp, dt, imag)
            ours_cmp = sp.spgpe_get_psi_host(h2)
            sp.spgpe_destroy(h2)
            line["cufft_comparison"] = cufft_comparison(w, spec, n_cmp, 3, ours_cmp)
            line["cufft_comparison"]["ours_speedup"] = line["cufft_comparison"]["ms_per_step"] / (ms / K)
        if world == 1 and not args.no_cpu:
            v, cores, what, sec = oracle_sample(spec["cfg"], spec["dtype"], budget_s=20.0, steps=3)
            v1, _, what1, sec1 = oracle_sample(spec["cfg"], spec["dtype"], budget_s=10.0, steps=3, threads=1)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what,
                                    "s_per_step": sec,
                                    "single_thread": {"value": v1, "unit": UNIT, "cores": 1, "sample": what1,
                                                      "s_per_step": sec1}}
        print(json.dumps(line), flush=True)
    sp.spgpe_destroy(h)
    if world > 1:
        dist.destroy_process_group()


def run_sweep(args):
    """The paper's own benchmark (Figure 2): evaluation time of the stepping function against the
    grid size N = Nx Ny = 2^eta (N = points of one component), complex128, median and median absolute deviation over
    repeated timings, and the linear fit t(N) = theta N + xi the paper reports for its GPUs (theta = 9.7e-8 s per point).
    Config 4's recipe (all terms on, real time) on nx = 2^ceil(eta/2), ny = 2^floor(eta/2): square grids for even eta,
    2:1 grids for odd eta.  Two times per size: one spgpe_step(1) call (what the paper's timeit measures: a whole
    call, opening + column + closing pass) and the per-step time inside one spgpe_step(K) call (steady state)."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: libspgpe has no CPU fallback")
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import paper_2010_15069_b200 as sp
    import workloads as wl
    sp.lib()
    stream = torch.cuda.Stream()
    rows = []

    def region(fn):
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(stream):
            e0.record(stream)
            fn()
            e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e-3

    def med_mad(v):
        m = float(np.median(v))
        return m, float(np.median(np.abs(np.array(v) - m)))

    for eta in range(args.eta_min, args.eta_max + 1):
        nx, ny = 1 << ((eta + 1) // 2), 1 << (eta // 2)
        w = wl.make_workload(4, dtype="c128", nx=nx, ny=ny)
        _, dt, imag = w.schedule[0]
        h = sp.from_workload(w, stream=stream.cuda_stream)
        sp.spgpe_step(h, max(3, args.warmup), dt, imag)
        sp.spgpe_synchronize(h)
        sampler = ClockSampler(0)  # per size: the host-side generation of the next grid leaves the GPU idle
        sampler.start()
        t10 = region(lambda: sp.spgpe_step(h, 10, dt, imag)) / 10
        K = int(min(2000, max(10, 0.05 / t10)))  # regions of about 50 ms
        one, one_mad = med_mad([region(lambda: sp.spgpe_step(h, 1, dt, imag)) for _ in range(max(args.repeats, 21))])
        many, many_mad = med_mad([region(lambda: sp.spgpe_step(h, K, dt, imag)) / K for _ in range(args.repeats)])
        clocks = sampler.stop()
        # per-launch durations of the two pass kernels between events (serialised: no overlap of successive kernels)
        sp.spgpe_profile(h, True)
        sp.spgpe_step(h, min(K, 100), dt, imag)
        kms, kcnt = sp.spgpe_profile_read(h)
        sp.spgpe_profile(h, False)
        norms = sp.spgpe_norm(h)
        rows.append({"eta": eta, "grid": [nx, ny], "points": nx * ny, "one_step_call_s": one, "one_step_call_mad_s": one_mad,
                     "steps_per_region": K, "s_per_step": many, "s_per_step_mad": many_mad,
                     "serialised_launch_s": {"row_pass": kms[0] / max(kcnt[0], 1) * 1e-3,
                                             "column_pass": kms[1] / max(kcnt[1], 1) * 1e-3},
                     "finite": bool(np.isfinite(norms).all()), "clocks": clocks})
        sp.spgpe_destroy(h)
        del w
    N = np.array([r["points"] for r in rows], dtype=np.float64)
    A = np.stack([N, np.ones_like(N)], axis=1)

    def fit(key):
        th, xi = np.linalg.lstsq(A, np.array([r[key] for r in rows]), rcond=None)[0]
        return {"theta_s_per_point": float(th), "xi_s": float(xi)}

    print(json.dumps({
        "metric": "step evaluation time against grid size, t(N) = theta N + xi", "unit": "s", "dtype": "f64",
        "data": "synthetic", "n_gpus": 1, "higher_is_better": False,
        "config": {"workload": "config 4 recipe (complex128, real time, all terms on) at N = 2^eta points per component, "
                               "nx = 2^ceil(eta/2), ny = 2^floor(eta/2)", "eta": [args.eta_min, args.eta_max],
                   "repeats": args.repeats, "l2": "sizes up to eta = 21 fit the 126 MB L2, larger ones do not; no flush"},
        "sweep": rows, "fit_one_step_call": fit("one_step_call_s"), "fit_steady_state": fit("s_per_step"),
        "paper": {"theta_s_per_point": 9.7e-8, "where": "PAPER.md L189 (Figure 2): the paper's GPUs (MX150, GTX 980 Ti, "
                  "Titan V), PyTorch + cuFFT, complex128; another machine's number: context, not the target"}}),
          flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--repeats", type=int, default=5, help="timed regions of --steps steps each (median reported)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="4", choices=sorted(WORKLOADS))
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--graph", action="store_true",
                    help="also time replays of a CUDA graph of one captured spgpe_step(K) call (graph_replay)")
    ap.add_argument("--no-cufft", action="store_true", help="skip the torch.fft / elementwise comparison leg")
    ap.add_argument("--sweep", action="store_true",
                    help="the paper's Figure 2 instead of the headline line: step time against N = 2^eta (complex128)")
    ap.add_argument("--eta-min", type=int, default=12)
    ap.add_argument("--eta-max", type=int, default=24)
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    args.repeats = max(1, args.repeats)
    if args.sweep:
        if not (12 <= args.eta_min <= args.eta_max <= 26):
            ap.error("--eta-min / --eta-max: 12 <= eta <= 26 (line lengths 64 ... 8192)")
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args, args.workload)
    else:
        run_ours(args, args.workload)


if __name__ == "__main__":
    main()
