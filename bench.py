#!/usr/bin/env python
"""bench.py -- throughput of the spherical-harmonics hot path on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C2] [--no-sweep]
    python bench.py --impl reference ...        # the CPU oracle, as it stands, on the host cores
    python bench.py --lmax-sweep                # the full l_max table (profiles/lmax_sweep_r2.json)
    python bench.py --kernels-only --workload custom --dtype f32 --deriv 1 --l-max 24   # the command ncu wraps

A "step" is one pass of the hot path over one batch of the named workload: one
``sphericart_cuda_compute`` call and, for C5, the ``sphericart_cuda_vjp``
call that follows it (a10).  The headline workload is BASELINE.json ``configs[1]`` (C2: N=100000
f32 l_max=8 normalised values+gradients).  ``value`` is points/s with inputs resident in HBM;
``e2e`` is the same metric through the host-buffer entry point (pinned host memory, H2D of xyz and
D2H of every output inside the timed region).  The remaining configurations are parity-test cases;
at N=1 they are also timed briefly and reported under ``sweep`` (the metric is "points/s and output
GB/s vs l_max, f32/f64, +-grads") but the JSON line's headline keys are C2's.

Multi-GPU: the path shards over points with no communication; every rank
runs the same per-GPU batch ("scaling": "weak"), a barrier + synchronize brackets the timed region
and the time is the max over ranks.  `--gpus N` with no WORLD_SIZE in the environment starts its own
N ranks (torch.distributed.run on 127.0.0.1); under torchrun it is one of them.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

from paper_2302_08381_b200 import workloads as W  # noqa: E402

METRIC = "points/s"
N_SETS = 4          # output buffer sets the timed loop rotates over (C2: 4 x 129.6 MB > 126 MB L2)


def measured_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write, burst)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic_bytes(name):
    """ncu --set full: dram__bytes_read.sum + dram__bytes_write.sum per launch of the configuration's
    forward kernel, from the capture summarised in profiles/ncu_traffic.json (which names the capture
    and its command); None when there is no capture of the kernel as it stands."""
    p = ROOT / "profiles" / "ncu_traffic.json"
    if not p.exists():
        return None
    ent = json.loads(p.read_text()).get(name)
    return None if ent is None else float(ent["dram_bytes_per_launch"])


# -------------------------------------------------------------------------------------------------
# clocks during the timed region
# -------------------------------------------------------------------------------------------------
class ClockSampler:
    """Polls SM clock and throttle reasons through NVML while the timed region runs."""

    BAD = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20}
    NOTE = {"sw_power_cap": 0x4}

    def __init__(self, index: int, period_s: float = 0.02):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self.period = period_s
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml

            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:  # NVML missing: the JSON line then carries null clocks
            self.nv = None

    def sample(self):
        if self.nv is None:
            return
        try:
            self.samples.append(float(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
            mask = int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
            for name, bit in {**self.BAD, **self.NOTE}.items():
                if mask & bit:
                    self.reasons.add(name)
        except Exception:
            pass

    def _run(self):
        while not self._stop.is_set():
            self.sample()
            self._stop.wait(self.period)

    def start(self):
        self._thread = threading.Thread(target=self._run, daemon=True)
        self._thread.start()

    def stop(self):
        self._stop.set()
        if self._thread:
            self._thread.join()

    def summary(self):
        return {"sm_mhz": statistics.median(self.samples) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


# -------------------------------------------------------------------------------------------------
# the CUDA arm
# -------------------------------------------------------------------------------------------------
def algorithmic_bytes_per_point(cfg, with_vjp: bool):
    """forward = in + out; VJP = dsph + grad_sph read, grad_xyz written."""
    fwd = cfg.in_bytes_per_point + cfg.out_bytes_per_point
    vjp = (4 * cfg.n_sph + 3) * cfg.itemsize if with_vjp else 0
    return fwd, vjp


class DeviceWorkload:
    """Inputs resident in HBM + N_SETS output buffer sets for one configuration."""

    def __init__(self, cfg, torch, pkg, device, n_sets, seed=0):
        self.cfg, self.torch, self.pkg = cfg, torch, pkg
        dt = torch.float32 if cfg.dtype == "f32" else torch.float64
        self.dcode = pkg.F32 if cfg.dtype == "f32" else pkg.F64
        self.xyz = torch.from_numpy(W.make_xyz(cfg, seed=seed)).to(device)
        n, L = cfg.n, cfg.n_sph
        self.sets = []
        for _ in range(n_sets):
            sph = torch.empty((n, L), dtype=dt, device=device)
            dsph = torch.empty((n, 3, L), dtype=dt, device=device) if cfg.gradients else None
            ddsph = torch.empty((n, 3, 3, L), dtype=dt, device=device) if cfg.hessians else None
            self.sets.append((sph, dsph, ddsph))
        self.grad_sph = self.grad_xyz = None
        if cfg.vjp:
            self.grad_sph = torch.from_numpy(W.make_grad_sph(cfg, seed=seed)).to(device)
            self.grad_xyz = torch.empty((n, 3), dtype=dt, device=device)
        self.stream = torch.cuda.current_stream().cuda_stream

    def forward(self, i):
        c = self.cfg
        sph, dsph, ddsph = self.sets[i % len(self.sets)]
        self.pkg.sphericart_cuda_compute(self.xyz, c.n, c.l_max, c.normalized, self.dcode, sph, dsph, ddsph,
                                         self.stream)

    def backward(self, i):
        c = self.cfg
        _, dsph, _ = self.sets[i % len(self.sets)]
        self.pkg.sphericart_cuda_vjp(None, dsph, self.grad_sph, self.grad_xyz, c.n, c.l_max, self.dcode,
                                     self.stream)

    def forward_values_only(self, i):
        c = self.cfg
        sph, _, _ = self.sets[i % len(self.sets)]
        self.pkg.sphericart_cuda_compute(self.xyz, c.n, c.l_max, c.normalized, self.dcode, sph, None, None,
                                         self.stream)

    def backward_recompute(self, i):
        c = self.cfg
        self.pkg.sphericart_cuda_vjp_recompute(self.xyz, self.grad_sph, self.grad_xyz, c.n, c.l_max, c.normalized,
                                               self.dcode, self.stream)

    def step(self, i):
        self.forward(i)
        if self.cfg.vjp:
            self.backward(i)


class OpWorkload:
    """`--workload custom --op vjp_recompute | vjp2 | expand`: one of the other entry points as the step
    (the command ncu wraps for their kernels); same interface as DeviceWorkload."""

    def __init__(self, cfg, op, torch, pkg, device):
        self.cfg, self.op, self.pkg = cfg, op, pkg
        dt = torch.float32 if cfg.dtype == "f32" else torch.float64
        self.dcode = pkg.F32 if cfg.dtype == "f32" else pkg.F64
        self.sets = [None]
        self.stream = torch.cuda.current_stream().cuda_stream
        n, L = cfg.n, cfg.n_sph
        if op == "expand":
            n_rad, n_seg = 8, max(1, cfg.n // 32)
            xyz, rad, seg = W.make_expand_inputs(n_seg, cfg.l_max, n_rad, cfg.dtype, 32.0)
            self.x, self.rad, self.seg = (torch.from_numpy(a).to(device) for a in (xyz, rad, seg))
            self.n_seg, self.n_rad = n_seg, n_rad
            self.out = [torch.empty((n_seg, n_rad, L), dtype=dt, device=device) for _ in range(2)]
            self.points = xyz.shape[0]
            self.bytes = self.points * (3 + n_rad * (cfg.l_max + 1)) * cfg.itemsize + n_seg * (8 + n_rad * L * cfg.itemsize)
        else:
            self.x = torch.randn(n, 3, device=device, dtype=dt)
            self.w = torch.randn(n, L, device=device, dtype=dt)
            self.v = torch.randn(n, 3, device=device, dtype=dt)
            self.gx = torch.empty((n, 3), device=device, dtype=dt)
            self.ggs = torch.empty((n, L), device=device, dtype=dt)
            self.points = n
            # xyz + grad_sph read, grad_xyz written (+ v read, grad_grad_sph written for vjp2)
            self.bytes = n * ((L + 6) * cfg.itemsize + ((L + 3) * cfg.itemsize if op == "vjp2" else 0))

    def step(self, i):
        c, p = self.cfg, self.pkg
        if self.op == "expand":
            p.sphericart_cuda_expand(self.x, self.rad, self.seg, self.n_seg, c.l_max, self.n_rad, self.dcode,
                                     self.out[i % 2], self.stream)
        elif self.op == "vjp2":
            p.sphericart_cuda_vjp2(self.x, self.w, self.v, self.gx, self.ggs, c.n, c.l_max, c.normalized, self.dcode,
                                   self.stream)
        else:
            p.sphericart_cuda_vjp_recompute(self.x, self.w, self.gx, c.n, c.l_max, c.normalized, self.dcode, self.stream)

    forward = step


def time_loop(torch, fn, steps):
    """CUDA events on torch's current stream (the stream the library launches on) around `steps` calls."""
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(steps):
        fn(i)
    e1.record()
    return e0, e1


def capture_steps(torch, wl, steps):
    """The `steps` calls of the timed region captured ONCE into a CUDA graph (on a side stream, the
    workload's launches pointed at it for the capture).  Replaying it inside the timed region submits
    exactly the same kernels in the same order with no host launch latency between the timing events
    and the first kernel -- with K host launches that gap and the first launches' ramp are ~25 us of a
    460 us region at C2 (23.0 us per step at K = 20, 21.6 at K = 160).  Returns (graph, kernels in it)."""
    pkg = wl.pkg
    graph = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    saved = wl.stream
    before = pkg.sphericart_cuda_launch_count()
    try:
        with torch.cuda.stream(side):
            wl.stream = side.cuda_stream
            with torch.cuda.graph(graph, stream=side):
                for i in range(steps):
                    wl.step(i)
    finally:
        wl.stream = saved
    torch.cuda.current_stream().wait_stream(side)
    return graph, pkg.sphericart_cuda_launch_count() - before


def n_sets_for(cfg, free_bytes):
    per_set = cfg.n * cfg.out_bytes_per_point
    want = N_SETS if per_set < (2 << 30) else 2
    while want > 1 and want * per_set > 0.8 * free_bytes:
        want -= 1
    return want


def store_ceiling_gbs(torch, nbytes, device):
    """Write-only ceiling measured in the same run: cudaMemsetAsync over the same byte count,
    rotating over buffers larger than L2 (torch's fill kernel if libcudart cannot be reached)."""
    import ctypes

    nbytes = int(min(max(nbytes, 1 << 20), 8 << 30))
    n_bufs = max(2, int(600e6 // nbytes) + 1)
    bufs = [torch.empty(nbytes, dtype=torch.uint8, device=device) for _ in range(n_bufs)]
    fill = lambda i: bufs[i % n_bufs].zero_()
    try:
        rt = ctypes.CDLL("libcudart.so.12")
        rt.cudaMemsetAsync.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t, ctypes.c_void_p]
        stream = torch.cuda.current_stream().cuda_stream
        fill = lambda i: rt.cudaMemsetAsync(bufs[i % n_bufs].data_ptr(), 0, nbytes, stream)
    except OSError:
        pass
    for i in range(3):
        fill(i)
    torch.cuda.synchronize()
    reps = int(max(10, min(200, 4e9 // nbytes)))
    e0, e1 = time_loop(torch, fill, reps)
    torch.cuda.synchronize()
    return nbytes * reps / (e0.elapsed_time(e1) * 1e-3) / 1e9


def sweep_one(cfg, torch, pkg, device, peak):
    """Brief timing of one configuration (N=1 only): forward and VJP kernels timed separately."""
    free, _ = torch.cuda.mem_get_info()
    wl = DeviceWorkload(cfg, torch, pkg, device, n_sets_for(cfg, free))
    out_bytes = cfg.n * cfg.out_bytes_per_point
    reps = int(max(5, min(200, 2e9 // max(out_bytes, 1) * 10)))
    for i in range(3):
        wl.step(i)
    torch.cuda.synchronize()
    e0, e1 = time_loop(torch, wl.forward, reps)
    torch.cuda.synchronize()
    ms_f = e0.elapsed_time(e1) / reps
    fwd_b, vjp_b = algorithmic_bytes_per_point(cfg, cfg.vjp)
    res = {"workload": cfg.what, "dtype": cfg.dtype, "l_max": cfg.l_max, "n": cfg.n, "launches_timed": reps,
           "buffer_sets": len(wl.sets), "fwd_us": round(ms_f * 1e3, 2), "fwd_points_per_s": cfg.n / (ms_f * 1e-3),
           "fwd_gbs": cfg.n * fwd_b / (ms_f * 1e-3) / 1e9}
    res["fwd_frac_of_measured_peak"] = res["fwd_gbs"] / peak
    res["kernel"] = pkg.sphericart_cuda_last_kernel()
    res["roofline"] = {"bound": "hbm", "kernel": "forward (" + res["kernel"] + ")", "achieved": res["fwd_gbs"],
                       "peak": peak, "unit": "GB/s", "frac": res["fwd_gbs"] / peak,
                       "traffic": ncu_traffic_bytes(cfg.name), "algorithmic_bytes_per_launch": cfg.n * fwd_b,
                       "avg_launch_us": ms_f * 1e3}
    if cfg.vjp:
        e0, e1 = time_loop(torch, wl.backward, reps)
        torch.cuda.synchronize()
        ms_b = e0.elapsed_time(e1) / reps
        res.update({"vjp_us": round(ms_b * 1e3, 2), "vjp_gbs": cfg.n * vjp_b / (ms_b * 1e-3) / 1e9})
        res["vjp_frac_of_measured_peak"] = res["vjp_gbs"] / peak
        res["vjp_roofline"] = {"bound": "hbm", "kernel": "vjp (" + pkg.sphericart_cuda_last_kernel() + ")",
                               "achieved": res["vjp_gbs"], "peak": peak, "unit": "GB/s", "frac": res["vjp_gbs"] / peak,
                               "traffic": ncu_traffic_bytes(cfg.name + "_vjp"),
                               "algorithmic_bytes_per_launch": cfg.n * vjp_b, "avg_launch_us": ms_b * 1e3}
        # the same backward without stored derivatives (reads xyz + grad_sph only), and
        # the values-only forward it pairs with
        esize = 4 if cfg.dtype == "f32" else 8
        for key, fn, bytes_pt in (("vjp_recompute", wl.backward_recompute, (cfg.n_sph + 6) * esize),
                                  ("fwd_values_only", wl.forward_values_only, (cfg.n_sph + 3) * esize)):
            for i in range(3):
                fn(i)
            e0, e1 = time_loop(torch, fn, reps)
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / reps
            gbs = cfg.n * bytes_pt / (ms * 1e-3) / 1e9
            res.update({key + "_us": round(ms * 1e3, 2), key + "_gbs": gbs})
            res[key + "_roofline"] = {"bound": "hbm", "kernel": key + " (" + pkg.sphericart_cuda_last_kernel() + ")",
                                      "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak,
                                      "traffic": ncu_traffic_bytes(cfg.name + "_" + key),
                                      "algorithmic_bytes_per_launch": cfg.n * bytes_pt, "avg_launch_us": ms * 1e3}
    del wl
    torch.cuda.empty_cache()
    return res


def sweep_expand(torch, pkg, device, peak):
    """the fused density expansion of Eq. 1 on a neighbour-list-shaped input
    (32768 centres x Poisson(32) neighbours, l_max = 8, n_rad = 8, f32), and the values-only forward
    over the same points as context (what an unfused consumer would have to run first)."""
    l_max, n_rad, n_seg = 8, 8, 32768
    xyz, rad, seg = W.make_expand_inputs(n_seg, l_max, n_rad, "f32", 32.0)
    n = xyz.shape[0]
    x_d, r_d, s_d = (torch.from_numpy(a).to(device) for a in (xyz, rad, seg))
    L = (l_max + 1) ** 2
    outs = [torch.empty((n_seg, n_rad, L), dtype=torch.float32, device=device) for _ in range(4)]
    sphs = [torch.empty((n, L), dtype=torch.float32, device=device) for _ in range(2)]
    stream = torch.cuda.current_stream().cuda_stream
    fused = lambda i: pkg.sphericart_cuda_expand(x_d, r_d, s_d, n_seg, l_max, n_rad, pkg.F32, outs[i % 4], stream)
    fwd = lambda i: pkg.sphericart_cuda_compute(x_d, n, l_max, 1, pkg.F32, sphs[i % 2], None, None, stream)
    res = {"workload": f"Eq. 1: {n_seg} segments, {n} points (Poisson(32) per segment), l_max={l_max}, n_rad={n_rad}, f32",
           "n_points": n}
    for key, fn in (("expand", fused), ("fwd_values_only", fwd)):
        for i in range(3):
            fn(i)
        torch.cuda.synchronize()
        e0, e1 = time_loop(torch, fn, 50)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / 50
        res[key + "_us"] = round(ms * 1e3, 2)
        res[key + "_points_per_s"] = n / (ms * 1e-3)
    in_bytes = n * (12 + n_rad * (l_max + 1) * 4) + n_seg * (8 + n_rad * L * 4)
    res["expand_algorithmic_gbs"] = in_bytes / (res["expand_us"] * 1e-6) / 1e9
    res["roofline"] = {"bound": "hbm", "kernel": "expand", "achieved": res["expand_algorithmic_gbs"], "peak": peak,
                       "unit": "GB/s", "frac": res["expand_algorithmic_gbs"] / peak,
                       "traffic": ncu_traffic_bytes("N2_expand"), "algorithmic_bytes_per_launch": in_bytes,
                       "avg_launch_us": res["expand_us"]}
    return res


def sweep_backward(torch, pkg, device, peak):
    """SURVEY 8(f) N1 / N4 against l_max (f32 and f64, normalised, xyz ~ N(0,1), grad_sph ~ N(0,1)): the
    training step with stored derivatives (forward V+G, then sphericart_cuda_vjp) beside the one without
    (forward V, then sphericart_cuda_vjp_recompute), the second-order VJP, and the forward pass in the e3nn
    'component' convention; us per call and the kernel family that served each."""
    st = torch.cuda.current_stream().cuda_stream
    out = {}
    for dtype, tdt, es in (("f32", torch.float32, 4), ("f64", torch.float64, 8)):
        dc = pkg.F32 if dtype == "f32" else pkg.F64
        for l_max in (4, 8, 12, 16, 24, 32):
            L = (l_max + 1) ** 2
            n = max(148 * 64, int(min(2_000_000, 0.8e9 // (4 * L * es))) // 256 * 256)
            x = torch.randn(n, 3, device=device, dtype=tdt)
            w = torch.randn(n, L, device=device, dtype=tdt)
            v = torch.randn(n, 3, device=device, dtype=tdt)
            sph = torch.empty((n, L), device=device, dtype=tdt)
            dsph = torch.empty((n, 3, L), device=device, dtype=tdt)
            gx = torch.empty((n, 3), device=device, dtype=tdt)
            ggs = torch.empty((n, L), device=device, dtype=tdt)
            calls = {
                "fwd_vg": lambda i: pkg.sphericart_cuda_compute(x, n, l_max, 1, dc, sph, dsph, None, st),
                "vjp_stored": lambda i: pkg.sphericart_cuda_vjp(None, dsph, w, gx, n, l_max, dc, st),
                "fwd_v": lambda i: pkg.sphericart_cuda_compute(x, n, l_max, 1, dc, sph, None, None, st),
                "vjp_recompute": lambda i: pkg.sphericart_cuda_vjp_recompute(x, w, gx, n, l_max, 1, dc, st),
                "vjp2": lambda i: pkg.sphericart_cuda_vjp2(x, w, v, gx, ggs, n, l_max, 1, dc, st),
                "fwd_vg_e3nn_component": lambda i: pkg.sphericart_cuda_compute_ex(x, n, l_max, 1, dc, pkg.AXES_E3NN,
                                                                                 pkg.SCALE_COMPONENT, sph, dsph, None, st),
            }
            row = {"n": n}
            for key, fn in calls.items():
                for i in range(2):
                    fn(i)
                torch.cuda.synchronize()
                e0, e1 = time_loop(torch, fn, 5)
                torch.cuda.synchronize()
                row[key + "_us"] = round(e0.elapsed_time(e1) / 5 * 1e3, 1)
                row[key + "_kernel"] = pkg.sphericart_cuda_last_kernel()
            row["step_stored_us"] = round(row["fwd_vg_us"] + row["vjp_stored_us"], 1)
            row["step_recompute_us"] = round(row["fwd_v_us"] + row["vjp_recompute_us"], 1)
            # algorithmic bytes of the recompute VJP: xyz + grad_sph read, grad_xyz written
            row["vjp_recompute_gbs"] = round(n * (L + 6) * es / (row["vjp_recompute_us"] * 1e-6) / 1e9, 1)
            row["vjp_stored_gbs"] = round(n * (4 * L + 3) * es / (row["vjp_stored_us"] * 1e-6) / 1e9, 1)
            out[f"{dtype}_l{l_max}"] = row
            del x, w, v, sph, dsph, gx, ggs
    return out


LMAX_FULL = (1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11, 12, 13, 14, 15, 16, 20, 24, 28, 32)
LMAX_BRIEF = (8, 12, 16, 20, 24, 28, 32)       # the cells of the default run (the >= 70 % clause: l_max >= 8)


def lmax_cell_points(bytes_per_point):
    """Points of one cell of the l_max axis: ~1.5 GB of output per call, at most 4 M points, at least 256
    per SM.  (The floor was 64 per SM at first: the long rows then ran calls of a few CTAs per SM whose
    ramp and tail cost them 5-30 % -- f64 Hessians at l_max = 32: 4.2 TB/s at 13 k points, 5.8 at 38 k,
    6.0 at 76 k; C4, the configuration with such rows, has 262 k.  Sizing EVERY cell for ~3.2 GB instead
    was measured too: the sweep then runs power-capped, median SM clock 1826 MHz instead of 1935-1965,
    and the compute-heavy f64 cells lose 7-15 %.)"""
    n = int(min(4_000_000, 1.5e9 // bytes_per_point)) // 256 * 256
    return max(n, 148 * 256)


def lmax_cell(torch, pkg, device, peak, dtype, deriv, l_max, normalized=1, n=None, reps=None):
    """One cell of the metric's axis: xyz ~ N(0,1) on the device, n from lmax_cell_points, two rotating
    output sets where they fit; CUDA events."""
    st = torch.cuda.current_stream().cuda_stream
    tdt, es = (torch.float32, 4) if dtype == "f32" else (torch.float64, 8)
    mult = (1, 4, 13)[deriv]
    L = (l_max + 1) ** 2
    per_pt = L * es * mult
    if n is None:
        n = lmax_cell_points(per_pt)
    x = torch.randn(n, 3, device=device, dtype=tdt)
    n_sets = 2 if n * per_pt < 3e9 else 1
    outs = [(torch.empty((n, L), device=device, dtype=tdt),
             torch.empty((n, 3, L), device=device, dtype=tdt) if deriv >= 1 else None,
             torch.empty((n, 3, 3, L), device=device, dtype=tdt) if deriv >= 2 else None)
            for _ in range(n_sets)]
    fn = lambda i: pkg.sphericart_cuda_compute(x, n, l_max, normalized, pkg.F32 if dtype == "f32" else pkg.F64,
                                               *outs[i % n_sets], st)
    for i in range(3):
        fn(i)
    torch.cuda.synchronize()
    if reps is None:
        reps = 10 if n * per_pt < 3e9 else 4
    e0, e1 = time_loop(torch, fn, reps)
    torch.cuda.synchronize()
    sec = e0.elapsed_time(e1) / reps * 1e-3
    gbs = n * per_pt / sec / 1e9
    del outs, x
    return {"n": n, "us": round(sec * 1e6, 1), "points_per_s": n / sec, "out_gbs": round(gbs, 1),
            "frac": round(gbs / peak, 3), "kernel": pkg.sphericart_cuda_last_kernel()}


def lmax_sweep(torch, pkg, device, peak, l_values=LMAX_FULL):
    """The metric's own axis -- output GB/s and points/s against l_max, f32 / f64, values / + gradients
    / + Hessians (normalised harmonics), with the kernel family that served each cell and the fraction
    of the measured HBM peak.  `--lmax-sweep` prints every l_max of LMAX_FULL as one JSON object; the
    default run carries LMAX_BRIEF under sweep.lmax."""
    rows = {}
    for dtype in ("f32", "f64"):
        for deriv, tag in ((0, "values"), (1, "grads"), (2, "hessians")):
            rows[f"{dtype}_{tag}"] = {str(l): lmax_cell(torch, pkg, device, peak, dtype, deriv, l) for l in l_values}
    cells = [c for r in rows.values() for l, c in r.items() if int(l) >= 8]
    rows["summary"] = {"cells_lmax_ge_8": len(cells),
                       "cells_at_or_above_0.70_of_measured_peak": sum(c["frac"] >= 0.70 for c in cells),
                       "min_out_gbs_lmax_ge_8": min(c["out_gbs"] for c in cells) if cells else None,
                       "frac_is": "out_gbs / measured copy peak (MEASURED_PEAKS.json hbm_gbs)"}
    return rows


def render_lmax_table(path):
    """`--render-lmax-table FILE`: the markdown table of DESIGN.md / BASELINE.md from a stored `--lmax-sweep`
    JSON (profiles/lmax_sweep_r2.json): output GB/s and the kernel family per cell."""
    d = json.loads(Path(path).read_text())
    rows, peak = d["lmax_sweep"], d["peak_gbs"]
    names = {"f32_values": "f32 values", "f32_grads": "f32 grads", "f32_hessians": "f32 hessians",
             "f64_values": "f64 values", "f64_grads": "f64 grads", "f64_hessians": "f64 hessians"}
    ls = list(rows["f32_values"].keys())
    out = ["| variant \\ l_max | " + " | ".join(ls) + " |", "|---" * (len(ls) + 1) + "|"]
    for key, name in names.items():
        out.append(f"| {name} | " + " | ".join(f"{rows[key][l]['out_gbs']:.0f} {rows[key][l]['kernel']}" for l in ls) + " |")
    sm = rows["summary"]
    out.append("")
    out.append(f"Measured copy peak {peak:.0f} GB/s; cells with l_max >= 8: {sm['cells_lmax_ge_8']}, of which at or above 0.70 of "
               f"that peak ({0.7 * peak:.0f} GB/s): {sm['cells_at_or_above_0.70_of_measured_peak']}; slowest: "
               f"{sm['min_out_gbs_lmax_ge_8']:.0f} GB/s.")
    print("\n".join(out))


def time_e2e(cfg, torch, pkg, steps):
    """The same metric through the host-buffer C-ABI call: pinned host arrays in, pinned host arrays
    out, H2D + kernels + D2H inside the timed region (wall clock around a synchronous call)."""
    dt = torch.float32 if cfg.dtype == "f32" else torch.float64
    dcode = pkg.F32 if cfg.dtype == "f32" else pkg.F64
    n, L = cfg.n, cfg.n_sph
    xyz = torch.from_numpy(W.make_xyz(cfg)).pin_memory()
    sph = torch.empty((n, L), dtype=dt).pin_memory()
    dsph = torch.empty((n, 3, L), dtype=dt).pin_memory() if cfg.gradients else None
    ddsph = torch.empty((n, 3, 3, L), dtype=dt).pin_memory() if cfg.hessians else None
    gs = gx = None
    if cfg.vjp:
        gs = torch.from_numpy(W.make_grad_sph(cfg)).pin_memory()
        gx = torch.empty((n, 3), dtype=dt).pin_memory()

    def one():
        pkg.sphericart_cuda_compute_host(xyz, n, cfg.l_max, cfg.normalized, dcode, sph, dsph, ddsph)
        if cfg.vjp:
            pkg.sphericart_cuda_vjp_host(None, dsph, gs, gx, n, cfg.l_max, dcode)

    for _ in range(2):
        one()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(steps):
        one()
    torch.cuda.synchronize()
    dt_s = (time.perf_counter() - t0) / steps
    h2d = n * cfg.in_bytes_per_point + (n * 4 * L * cfg.itemsize if cfg.vjp else 0)
    d2h = n * cfg.out_bytes_per_point + (n * 3 * cfg.itemsize if cfg.vjp else 0)
    return {"value": n / dt_s, "unit": METRIC, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
            "ms_per_step": dt_s * 1e3, "steps": steps,
            "how": "sphericart_cuda_compute_host on pinned host buffers, wall clock around the synchronous call"}


def oracle_baseline(cfg, budget_s=12.0):
    """The oracle's double build, as it stands, on the host cores, on a bounded sample of cfg."""
    import oracle

    oracle.build()
    cores = oracle.num_threads("f64")
    per_point_guess = 40e-9 * cfg.n_sph * (1 + 3 * cfg.gradients + 9 * cfg.hessians)   # seconds, 1 core
    n = int(min(cfg.n, max(2048, budget_s * cores / 5 / per_point_guess)))
    xyz = W.make_xyz(cfg, n)
    L = cfg.n_sph
    out = (np.empty((n, L)), np.empty((n, 3, L)) if cfg.gradients else None,
           np.empty((n, 3, 3, L)) if cfg.hessians else None)
    g = W.make_grad_sph(cfg, n).astype(np.float64) if cfg.vjp else None

    def one():
        oracle.compute(xyz, cfg.l_max, cfg.normalized, cfg.gradients, cfg.hessians, kind="f64", out=out)
        if cfg.vjp:
            oracle.vjp(out[1], g, cfg.l_max, kind="f64")

    one()
    times, t_all = [], time.perf_counter()
    while len(times) < 5 or (time.perf_counter() - t_all < budget_s / 2 and len(times) < 200):
        t0 = time.perf_counter()
        one()
        times.append(time.perf_counter() - t0)
    med = statistics.median(times)
    return {"value": n / med, "unit": METRIC, "cores": cores, "kind": "oracle",
            "sample": f"{cfg.name}: first {n} of {cfg.n} points, oracle f64 build (gcc -O2 -fopenmp), "
                      f"median of {len(times)} passes, {med * 1e3:.2f} ms per pass"}, n, med


def workload_config(args):
    """One of BASELINE.json's configurations, or `--workload custom`: any (dtype, l_max, outputs) cell
    on xyz ~ N(0,1), n sized as in the l_max sweep -- the command ncu wraps for the kernels that serve
    cells outside the five configurations."""
    if args.workload != "custom":
        return W.CONFIGS[args.workload]
    es = 4 if args.dtype == "f32" else 8
    per_pt = (args.l_max + 1) ** 2 * es * (1, 4, 13)[args.deriv]
    n = args.n or lmax_cell_points(per_pt)
    what = (f"custom: N={n} {args.dtype} l_max={args.l_max} {'solid' if args.solid else 'normalized'} "
            f"{('Y', 'Y+grad', 'Y+grad+Hessian')[args.deriv]}, xyz~N(0,1)")
    return W.Config("C9", n, args.dtype, args.l_max, not args.solid, args.deriv >= 1, args.deriv >= 2, False, what)


def spawn_ranks(n_ranks, argv, extra_env=None):
    """`--gpus N` without a launcher: start N ranks of this script under torch.distributed.run on
    127.0.0.1 (free port), one per GPU, and pass their output through (rank 0 prints the JSON line).
    NCCL's own communicator lines stay on (NCCL_DEBUG=INFO goes to stderr)."""
    import socket
    import subprocess

    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")
    env.setdefault("OMP_NUM_THREADS", "1")
    env.update(extra_env or {})
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n_ranks}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), str(Path(__file__).resolve()), *argv]
    return subprocess.run(cmd, env=env).returncode


def run_stub(args):
    """--impl stub (tests only, no GPU): the rank plumbing of run_cuda -- process group, barrier,
    max-over-ranks time, one JSON line from rank 0 -- on the gloo backend with a sleep as the step."""
    import torch
    import torch.distributed as dist

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:
        dist.init_process_group("gloo")
        dist.barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        time.sleep(0.001 * (1 + rank))
    ms = torch.tensor([(time.perf_counter() - t0) * 1e3], dtype=torch.float64)
    if world > 1:
        dist.barrier()
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps({"impl": "stub", "n_gpus": world, "steps": args.steps, "ms_per_step": float(ms) / args.steps,
                          "value": world * 1000 / (float(ms) / args.steps * 1e-3), "scaling": "weak"}))


def run_cuda(args):
    import torch

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; --impl reference times the oracle)")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=device)

    import paper_2302_08381_b200 as pkg

    pkg.load()                                   # raises if the CUDA library is missing
    for kv in args.option:
        k, _, v = kv.partition("=")
        pkg.sphericart_cuda_set_option(k, v)
    cfg = workload_config(args)
    peak, peak_src = measured_peaks()
    if args.lmax_sweep:
        if rank == 0:
            sampler = ClockSampler(local_rank)     # the SM clock the cells were timed at (boxes differ by several %)
            sampler.start()
            rows = lmax_sweep(torch, pkg, device, peak)
            sampler.stop()
            print(json.dumps({"lmax_sweep": rows, "peak_gbs": peak, "peak_source": peak_src,
                              "clocks": sampler.summary()}))
        return
    free, _ = torch.cuda.mem_get_info()
    if args.op != "forward":
        if args.workload != "custom" or not args.kernels_only:
            raise SystemExit("--op needs --workload custom --kernels-only")
        wl = OpWorkload(cfg, args.op, torch, pkg, device)
    else:
        wl = DeviceWorkload(cfg, torch, pkg, device, n_sets_for(cfg, free), seed=rank)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for i in range(max(args.warmup, 3)):
        wl.step(i)
    barrier()
    # the K steps of the timed region: one CUDA graph replay (default), or K host launches (--submit eager)
    graph, eager_ms_step, graph_note = None, None, None
    if args.submit == "graph" and not args.kernels_only:     # (profiling runs keep plain launches)
        e0, e1 = time_loop(torch, wl.step, args.steps)      # the eager number, reported beside the graph's
        barrier()
        eager_ms_step = e0.elapsed_time(e1) / args.steps
        try:
            graph, graph_kernels = capture_steps(torch, wl, args.steps)
            graph.replay()                                   # (untimed: instantiation and upload of the graph)
        except Exception as exc:                             # capture refused: time the host launches instead
            graph, graph_note = None, f"graph capture failed ({type(exc).__name__}): K host launches timed"
        barrier()
    clocks = ClockSampler(local_rank)
    clocks.start()
    launches0 = pkg.sphericart_cuda_launch_count()
    if graph is not None:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        graph.replay()
        e1.record()
    else:
        e0, e1 = time_loop(torch, wl.step, args.steps)
    clocks.sample()                              # the GPU is still draining the queue here
    barrier()
    clocks.stop()
    launches = graph_kernels if graph is not None else pkg.sphericart_cuda_launch_count() - launches0
    ms_total = e0.elapsed_time(e1)
    if dist is not None:
        t = torch.tensor([ms_total], device=device, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    ms_step = ms_total / args.steps
    value = world * cfg.n / (ms_step * 1e-3)

    # dominant kernel: the forward kernel.  One launch per step for forward-only workloads, so its
    # average duration IS the step time; for C5 the forward launches are timed in a pass of their own.
    fwd_b, vjp_b = algorithmic_bytes_per_point(cfg, cfg.vjp)
    if args.op != "forward":
        fwd_b = wl.bytes / cfg.n
    if cfg.vjp:
        f0, f1 = time_loop(torch, wl.forward, args.steps)
        torch.cuda.synchronize()
        ms_fwd = f0.elapsed_time(f1) / args.steps
    else:
        ms_fwd = ms_step
    achieved = cfg.n * fwd_b / (ms_fwd * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": "forward (" + pkg.sphericart_cuda_last_kernel() + ")", "achieved": achieved,
                "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": ncu_traffic_bytes(cfg.name),
                "peak_source": peak_src, "algorithmic_bytes_per_launch": cfg.n * fwd_b,
                "avg_launch_us": ms_fwd * 1e3, "output_gbs": cfg.n * cfg.out_bytes_per_point / (ms_fwd * 1e-3) / 1e9,
                "frac_of_nominal_8tbs": achieved / 8000.0}

    line = {"metric": METRIC, "value": value, "unit": METRIC, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": cfg.dtype, "data": "synthetic",
            "config": {"workload": f"{cfg.name}: {cfg.what}",
                       "why_this_workload": "BASELINE.json configs[1], the configuration the metric is quoted on; the "
                                            "larger single-GPU configurations (C3, C4, C5) and the l_max axis carry "
                                            "their own roofline blocks under sweep",
                       "n_points_per_gpu": cfg.n, "l_max": cfg.l_max,
                       "normalized": cfg.normalized, "gradients": cfg.gradients, "hessians": cfg.hessians,
                       "vjp": cfg.vjp, "parallelism": f"points sharded over {world} GPU(s), no collective",
                       "l2": f"outputs rotate over {len(wl.sets)} buffer sets "
                             f"({len(wl.sets) * cfg.n * cfg.out_bytes_per_point / 1e6:.0f} MB written before reuse "
                             "> 126 MB L2)",
                       "submission": ("the K steps are captured once into a CUDA graph and replayed inside the timed "
                                      "region (same kernels, same order, no host launch latency between the events); "
                                      f"K host launches instead: {eager_ms_step * 1e3:.2f} us per step (--submit eager)")
                                     if graph is not None else (graph_note or "K host launches inside the timed region")},
            "clocks": clocks.summary(), "gpu_launches": int(launches), "roofline": roofline}
    if rank == 0 and not args.kernels_only:
        line["roofline"]["store_ceiling_gbs"] = store_ceiling_gbs(torch, cfg.n * cfg.out_bytes_per_point, device)
    del wl
    torch.cuda.empty_cache()
    if args.kernels_only:                        # profiling runs (ncu): the timed kernels and nothing else
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        if rank == 0:
            print(json.dumps(line))
        return

    e2e = time_e2e(cfg, torch, pkg, max(3, min(args.steps, args.e2e_steps)))
    if dist is not None:
        t = torch.tensor([e2e["ms_per_step"]], device=device, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e["ms_per_step"] = float(t.item())
        e2e["value"] = world * cfg.n / (e2e["ms_per_step"] * 1e-3)
    line["e2e"] = e2e

    if rank == 0 and world == 1:
        base, _, _ = oracle_baseline(cfg)
        line["cpu_baseline"] = base
        if not args.no_sweep:
            line["sweep"] = {}
            # the l_max axis first: it follows the oracle's seconds on the host, i.e. a GPU that is not yet
            # power-capped by the large configurations below (their cells are HBM-bound and do not care)
            lmax_rows = lmax_sweep(torch, pkg, device, peak, LMAX_BRIEF)
            for name in ("C1", "C2", "C3", "C4", "C5"):
                c = W.CONFIGS[name]
                free, _ = torch.cuda.mem_get_info()
                if c.n * (c.out_bytes_per_point + c.in_bytes_per_point) * 1.05 > free:
                    line["sweep"][name] = {"skipped": "does not fit in free HBM"}
                    continue
                line["sweep"][name] = sweep_one(c, torch, pkg, device, peak)
            line["sweep"]["N2_expand"] = sweep_expand(torch, pkg, device, peak)
            line["sweep"]["lmax"] = lmax_rows
            line["sweep"]["backward"] = sweep_backward(torch, pkg, device, peak)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line))


def run_reference(args):
    """--impl reference: the oracle (f64 build, OpenMP) on the host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle

    oracle.build()
    cfg = workload_config(args)
    cores = oracle.num_threads("f64")
    # one step = one oracle pass over a bounded sample, sized so the whole run ends within minutes
    per_point = 60e-9 * cfg.n_sph * (1 + 3 * cfg.gradients + 9 * cfg.hessians) / cores
    total = max(args.steps + max(args.warmup, 1), 1)
    n = int(min(cfg.n, max(1024, 120.0 / total / per_point)))
    xyz = W.make_xyz(cfg, n)
    L = cfg.n_sph
    out = (np.empty((n, L)), np.empty((n, 3, L)) if cfg.gradients else None,
           np.empty((n, 3, 3, L)) if cfg.hessians else None)
    g = W.make_grad_sph(cfg, n).astype(np.float64) if cfg.vjp else None

    def one():
        oracle.compute(xyz, cfg.l_max, cfg.normalized, cfg.gradients, cfg.hessians, kind="f64", out=out)
        if cfg.vjp:
            oracle.vjp(out[1], g, cfg.l_max, kind="f64")

    for _ in range(max(args.warmup, 1)):
        one()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        one()
    ms_step = (time.perf_counter() - t0) / args.steps * 1e3
    value = n / (ms_step * 1e-3)
    sample = f"{cfg.name}: first {n} of {cfg.n} points per step, oracle f64 build (gcc -O2 -fopenmp)"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": METRIC, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": max(args.warmup, 1), "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{cfg.name}: {cfg.what}", "l_max": cfg.l_max, "sample_points_per_step": n},
            "cpu_baseline": {"value": value, "unit": METRIC, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": METRIC, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", choices=["cuda", "reference", "stub"], default="cuda")
    ap.add_argument("--workload", choices=sorted(W.CONFIGS) + ["custom"], default="C2")
    ap.add_argument("--dtype", choices=["f32", "f64"], default="f32", help="--workload custom")
    ap.add_argument("--l-max", type=int, default=8, help="--workload custom")
    ap.add_argument("--deriv", type=int, choices=[0, 1, 2], default=1, help="--workload custom: 0 Y, 1 +grad, 2 +Hessian")
    ap.add_argument("--solid", action="store_true", help="--workload custom: solid harmonics instead of normalised")
    ap.add_argument("--n", type=int, default=0, help="--workload custom: points (default: as the l_max sweep, ~1.5 GB of output)")
    ap.add_argument("--op", choices=["forward", "vjp_recompute", "vjp2", "expand"], default="forward",
                    help="--workload custom --kernels-only: the entry point the step calls")
    ap.add_argument("--option", action="append", default=[], metavar="NAME=VALUE",
                    help="sphericart_cuda_set_option(NAME, VALUE) before anything runs (experiments)")
    ap.add_argument("--e2e-steps", type=int, default=20)
    ap.add_argument("--no-sweep", action="store_true", help="skip the brief timing of the other configurations")
    ap.add_argument("--submit", choices=("graph", "eager"), default="graph",
                    help="the K timed steps as one CUDA graph replay (default) or as K host launches")
    ap.add_argument("--lmax-sweep", action="store_true",
                    help="print output GB/s against l_max (f32/f64, +-gradients) as one JSON object and exit")
    ap.add_argument("--render-lmax-table", metavar="FILE", default=None,
                    help="print the markdown table of a stored --lmax-sweep JSON (no GPU needed) and exit")
    ap.add_argument("--kernels-only", action="store_true",
                    help="time the device-resident step only (no e2e, no oracle, no sweep): the command ncu wraps")
    args = ap.parse_args()
    if args.render_lmax_table:
        return render_lmax_table(args.render_lmax_table)
    if args.impl == "reference":
        args.steps = 20 if args.steps is None else args.steps
        args.warmup = 1 if args.warmup is None else args.warmup
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:      # no launcher: start the ranks ourselves
        raise SystemExit(spawn_ranks(args.gpus, sys.argv[1:]))
    if args.impl == "stub":
        args.steps = 5 if args.steps is None else args.steps
        return run_stub(args)
    args.steps = 2000 if args.steps is None else args.steps
    args.warmup = 20 if args.warmup is None else args.warmup
    run_cuda(args)


if __name__ == "__main__":
    main()
