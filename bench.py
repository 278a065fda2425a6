#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200-native NSFRB search (contract: task prompt, section 4).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c2|c3|c4|c5|c1] [--no-extra] [--impl reference]

A step is one pass of the whole hot path over one batch of synthetic input:
  c2 (default; BASELINE.json configs[1], the real-time config the chunk-latency metric is quoted on):
       one nsfrb_stream_push of a 25-sample chunk into the full 1536-sample ring (steady state);
  c3/c4/c5/c1: one nsfrb_search of the whole cube.
metric = Gcells/s, a cell being one (pixel, DM, width, start-sample) S/N evaluation, counted exactly.
The default line (c2, one GPU) also carries a `workloads` object: c3, c4 and c5 timed in the same run (3 steps each), with
their per-kernel split and both roofline fractions (BASELINE.json's contract formula and the full FP32 count), against
on-chip peaks measured in the same run (nsfrb_measure_peaks).  --no-extra skips them.
N > 1 (torchrun): the path does not shard below a pixel and BASELINE.json fixes the build at one GPU,
so every rank runs an independent replica of the same workload ("replicas only", weak scaling).
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
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2510_18136_b200 import workloads as W  # noqa: E402

CHUNK_DURATION_MS = 25 * W.TSAMP_S * 1e3  # 3355 ms (25 samples x 134 ms)
# dram__bytes_read.sum + dram__bytes_write.sum of one launch of the dominant kernel, from the committed `ncu --set full`
# capture named beside it (a constant of that capture, not measured in this run)
NCU_TRAFFIC = {"c2": (2.668e9, "profiles/r02_k_stream_c2_details.csv / r02.md (dram__bytes_read 2.493 GB + write 0.174 GB, round-2 capture of the history-mode kernel)")}


# ---------------------------------------------------------------------------- helpers
def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            d = json.load(open(path))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)", d
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)", {}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([v.strip() for v in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for nm, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def dist_setup(n_gpus):
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl" if torch.cuda.is_available() else "gloo")
    return rank, world, local


def max_over_ranks(value: float, world: int) -> float:
    """max over ranks of a device-measured time (the contract's multi-GPU timing rule)."""
    if world <= 1:
        return value
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device="cuda" if dist.get_backend() == "nccl" else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def barrier(world):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


# ---------------------------------------------------------------------------- workloads on the device
class StreamBench:
    """C2: ring filled to steady state, then timed pushes."""

    def __init__(self, wl, plan_mod, cubes=False, running=False):
        self.wl = wl
        self.plan = plan_mod.Plan.for_workload(wl, cand_capacity=4096)
        self.delays = self.plan.delays()
        self.info = self.plan.info()
        if cubes:  # NEXT 3: also write the per-(dm, width, pixel) S/N and TOA cubes every push
            shape = (len(wl.dm_list), len(wl.width_list), wl.npix)
            self.cubes = (torch.empty(shape, device="cuda"), torch.empty(shape, dtype=torch.int32, device="cuda"))
            self.plan.stream_set_cubes(*self.cubes)
        if running:  # NEXT 1: also the maps normalised by the running standard deviation
            self.run = (torch.empty(wl.npix, device="cuda"), torch.empty((3, wl.npix), dtype=torch.int32, device="cuda"))
            self.plan.stream_set_running_sigma(0.05, *self.run)
        n_fill = -(-wl.nt // wl.chunk_nt) + 1
        self.src = W.ChunkSource(wl, self.delays, n_fill + 600, "cuda")
        self.out = self.plan.alloc_outputs()
        # a pool of distinct chunks (> L2 when cycled together with the 6.4 GB ring)
        self.pool = [self.src.next().clone() for _ in range(8)]
        for i in range(n_fill):
            self.plan.stream_push(self.pool[i % len(self.pool)], self.out)
        torch.cuda.synchronize()
        self.i = 0
        self.host_pool = [c.cpu().pin_memory() for c in self.pool[:4]]
        self.host_out = self.plan._host_out()
        self.host_outs = [self.plan._host_out(), self.plan._host_out()]   # two pushes in flight
        # steady state: exactly chunk_nt windows per (pixel, dm, width) (S5)
        self.cells_per_step = wl.npix * len(wl.dm_list) * len(wl.width_list) * wl.chunk_nt
        self.ring_bytes = wl.nchan * wl.nt * wl.npix * 4
        self.chunk_bytes = wl.nchan * wl.chunk_nt * wl.npix * 4

    def step(self):
        self.plan.stream_push(self.pool[self.i % len(self.pool)], self.out)
        self.i += 1

    def step_host(self):
        # pipelined host-buffer push: the H2D copy of this chunk overlaps the search of the previous one
        self.plan.stream_push_host_async(self.host_pool[self.i % len(self.host_pool)], self.host_outs[self.i & 1])
        self.i += 1

    def finish_host(self):
        self.plan.stream_wait()

    def step_host_sync(self):
        self.plan.stream_push_host(self.host_pool[self.i % len(self.host_pool)], self.host_out)
        self.i += 1

    def h2d_bytes(self):
        return self.chunk_bytes

    def d2h_bytes(self):
        return self.wl.npix * 16 + 4 + 4096 * 20     # maps, count, all cand_capacity records

    def algorithmic_bytes(self):
        # the whole ring is read once per push (mu/sigma span it) + the chunk is written into it
        return self.ring_bytes + self.chunk_bytes

    def kernel_bytes(self):
        # k_stream alone: the ring read once (per unit: 4 B per (channel, ring sample, pixel))
        return self.ring_bytes


class OfflineBench:
    def __init__(self, wl, plan_mod):
        self.wl = wl
        self.plan = plan_mod.Plan.for_workload(wl, cand_capacity=4096)
        self.delays = self.plan.delays()
        self.info = self.plan.info()
        self.cube = W.make_cube(wl, "cuda")
        extra = None
        if wl.name == "c1":
            with plan_mod.Plan(wl.nx, wl.ny, wl.nchan, wl.nt, wl.freqs_GHz, wl.tsamp_s, [500.0], [1], 6.0) as p5:
                extra = p5.delays()[0]
        self.pulses = W.injection_table(wl, self.delays)
        W.inject(self.cube, self.pulses, self.delays, extra_delays=extra)
        self.out = self.plan.alloc_outputs()
        torch.cuda.synchronize()
        self.cells_per_step = self.info["cells_per_pixel"] * wl.npix
        self.cube_bytes = wl.nchan * wl.nt * wl.npix * 4
        self.host_cube = None
        self.host_out = None

    def step(self):
        self.plan.search(self.cube, self.out)

    def step_host(self):
        """nsfrb_search_host from pinned host memory: the library stages the cube pixel batch by pixel batch.
        False when the host cannot hold (or pin) a copy of the cube."""
        if self.host_cube is None:
            try:
                import psutil
                if psutil.virtual_memory().available < self.cube_bytes + (8 << 30):
                    return False
                self.host_cube = torch.empty(self.cube.shape, dtype=torch.float32, pin_memory=True)
                self.host_cube.copy_(self.cube)
                torch.cuda.synchronize()
            except Exception:
                self.host_cube = None
                return False
            self.host_out = self.plan._host_out()
        self.plan.search_host(self.host_cube, self.host_out)
        return True

    def h2d_bytes(self):
        return self.cube_bytes

    def d2h_bytes(self):
        return self.wl.npix * 16 + 4

    def algorithmic_bytes(self):
        return self.cube_bytes

    def kernel_bytes(self):
        return self.cube_bytes


def time_steps(fn, steps, warmup, flush=None):
    """CUDA events on the current stream around exactly `steps` calls (after `warmup`)."""
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for a, b in ev:
        if flush is not None:
            flush()
        a.record()
        fn()
        b.record()
    torch.cuda.synchronize()
    return [a.elapsed_time(b) for a, b in ev]


def offline_roofline(wl, bench, search_ms, ms_per_step, hbm_peak, peak_src, onchip, sm_max_mhz):
    """BASELINE.json's contract roofline -- the slower of (cube bytes once / HBM) and (shift-adds + prefix adds) / FP32 issue
    rate -- and, beside it, the full FP32 count of SURVEY.md 8(d) (nchan + 3 + 2 nW lane-ops per (pixel, DM, sample)).
    The FP32 issue rate is the FADD rate nsfrb_measure_peaks achieved in this run; the theoretical 148 x 128 x clock is
    reported next to it."""
    info = bench.info
    alu_theory = 148 * 128 * sm_max_mhz * 1e6 / 1e12          # T lane-ops/s
    alu_peak = onchip["fadd"]["per_s"] / 1e12 if onchip else alu_theory
    alu_src = "measured FADD issue rate (nsfrb_measure_peaks, this run)" if onchip else "148 SMs x 128 lanes x sm_max_mhz (not measured)"
    T_sum = sum(wl.nt - int(x) for x in bench.delays.max(axis=1))        # valid samples over all DM trials
    contract_ops = (info["shift_adds_per_pixel"] + T_sum) * wl.npix
    full_ops = (wl.nchan + 3 + 2 * len(wl.width_list)) * T_sum * wl.npix
    t_hbm = bench.kernel_bytes() / (hbm_peak * 1e9)
    t_alu = contract_ops / (alu_peak * 1e12)
    t_full = full_ops / (alu_peak * 1e12)
    if t_alu > t_hbm:
        ach = contract_ops / (search_ms * 1e-3) / 1e12
        roof = {"bound": "alu", "achieved": ach, "peak": alu_peak, "unit": "T lane-ops/s", "frac": ach / alu_peak,
                "peak_source": alu_src, "algorithmic_ops": contract_ops}
    else:
        ach = bench.kernel_bytes() / (search_ms * 1e-3) / 1e9
        roof = {"bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak,
                "peak_source": peak_src}
    contract_ms = max(t_hbm, t_alu) * 1e3
    roof.update({"traffic": None, "kernel": "k_search4", "kernel_ms": search_ms, "share_of_step": search_ms / ms_per_step,
                 "algorithmic_bytes": bench.kernel_bytes(), "contract_roofline_ms": contract_ms,
                 "step_frac": contract_ms / ms_per_step,
                 "full_count_ops": full_ops, "full_count_roofline_ms": t_full * 1e3,
                 "full_count_frac": t_full * 1e3 / search_ms, "full_count_step_frac": t_full * 1e3 / ms_per_step,
                 "alu_peak_theoretical": alu_theory})
    return roof


def measure_offline_workload(name, nsfrb, hbm_peak, peak_src, onchip, sm_max_mhz, local, steps=3, warmup=3, e2e_ok=False):
    """One entry of the `workloads` object: c3 / c4 / c5 at BASELINE size, `steps` timed nsfrb_search calls."""
    wl = W.config(name)
    need = wl.nchan * wl.nt * wl.npix * 4 + (6 << 30)
    if torch.cuda.mem_get_info()[0] < need:
        return {"skipped": f"needs {need >> 30} GiB of free device memory"}
    bench = OfflineBench(wl, nsfrb)
    bench.plan.prepare()
    sampler = ClockSampler(local)
    sampler.start()
    t0 = time.perf_counter()
    per_step = time_steps(bench.step, steps, warmup)
    while time.perf_counter() - t0 < 1.0:            # keep the load up until nvidia-smi has sampled it
        bench.step()
        torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = float(np.mean(per_step))
    bench.plan.set_profiling(True)
    kms = []
    for _ in range(3):
        bench.step()
        kms.append(bench.plan.kernel_ms())
    bench.plan.set_profiling(False)
    kernel_ms = {k: float(np.mean([m[k] for m in kms])) for k in kms[0]}
    launches = bench.plan.last_launches()
    roof = offline_roofline(wl, bench, kernel_ms["search"], ms, hbm_peak, peak_src, onchip, sm_max_mhz)
    # end to end through nsfrb_search_host (pinned host cube -> maps and candidates in host memory); PCIe-bound
    e2e = {"value": None, "unit": "Gcells/s", "h2d_bytes_per_step": bench.h2d_bytes(), "d2h_bytes_per_step": bench.d2h_bytes(),
           "pcie_floor_ms_at_55GBs": bench.h2d_bytes() / 55e9 * 1e3}
    if e2e_ok and bench.step_host() is not False:
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(2):
            bench.step_host()
        torch.cuda.synchronize()
        e2e_ms = (time.perf_counter() - t0) * 1e3 / 2
        e2e.update({"value": bench.cells_per_step / (e2e_ms * 1e-3) / 1e9, "ms_per_step": e2e_ms,
                    "h2d_gbs": bench.h2d_bytes() / (e2e_ms * 1e-3) / 1e9, "call": "nsfrb_search_host, pixel batches staged from pinned memory"})
    else:
        e2e["note"] = "the host cannot hold a pinned copy of the cube" if e2e_ok else "not requested"
    bench.host_cube = None
    out = {"workload": f"{wl.name}: {wl.note}", "e2e": e2e, "nchan": wl.nchan, "nt": wl.nt, "nx": wl.nx, "ny": wl.ny, "ndm": len(wl.dm_list),
           "ndm_unique": bench.info["ndm_unique"], "nwidth": len(wl.width_list), "cells_per_step": bench.cells_per_step,
           "steps": steps, "warmup": warmup, "ms_per_step": ms, "ms_per_step_all": per_step,
           "value": bench.cells_per_step / (ms * 1e-3) / 1e9, "unit": "Gcells/s", "kernel_ms": kernel_ms,
           "gpu_launches_per_step": launches, "workspace_bytes": bench.plan.info()["workspace_bytes"],
           "contract_roofline_ms": roof["contract_roofline_ms"], "contract_frac": roof["step_frac"],
           "full_count_roofline_ms": roof["full_count_roofline_ms"], "full_count_frac": roof["full_count_step_frac"],
           "roofline": roof, "clocks": clocks, "l2": "inputs larger than L2"}
    del bench
    torch.cuda.empty_cache()
    return out


def run_cuda_arm(args, rank, world, local):
    from paper_2510_18136_b200 import nsfrb
    torch.cuda.set_device(local)
    hbm_peak, peak_src, peaks = measured_peaks()
    wl = W.config(args.workload)
    bench = StreamBench(wl, nsfrb, cubes=args.cubes, running=args.running) if wl.streaming else OfflineBench(wl, nsfrb)

    flusher = None
    if bench.algorithmic_bytes() < (256 << 20):
        fbuf = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")  # > 126 MB L2
        flusher = lambda: fbuf.zero_()  # noqa: E731

    sampler = ClockSampler(local)
    barrier(world)
    torch.cuda.synchronize()
    if rank == 0:
        sampler.start()
    t_all0 = time.perf_counter()
    per_step = time_steps(bench.step, args.steps, args.warmup, flusher)
    wall_s = time.perf_counter() - t_all0
    # the timed region of a 3 ms step is shorter than nvidia-smi's sampling period: keep the same load running
    # (untimed) until the sampler has seen about a second of it
    t_soak = time.perf_counter()
    while time.perf_counter() - t_soak < max(0.0, 1.2 - wall_s):
        for _ in range(8):
            bench.step()
        torch.cuda.synchronize()
    barrier(world)
    clocks = sampler.stop() if rank == 0 else None
    total_ms = max_over_ranks(float(np.sum(per_step)), world)
    ms_per_step = total_ms / args.steps
    launches = bench.plan.last_launches()

    value = world * bench.cells_per_step / (ms_per_step * 1e-3) / 1e9

    # device time of the dominant kernel (k_stream / k_search), measured live: the library records CUDA
    # events on the launching stream around each kernel it enqueues (nsfrb_plan_set_profiling)
    bench.plan.set_profiling(True)
    kms = []
    for _ in range(max(3, min(args.steps, 10))):
        if flusher is not None:
            flusher()
        bench.step()
        kms.append(bench.plan.kernel_ms())
    bench.plan.set_profiling(False)
    torch.cuda.synchronize()
    kernel_ms = {k: float(np.mean([m[k] for m in kms])) for k in kms[0]}
    dominant_ms = max_over_ranks(kernel_ms["search"], world)

    # end-to-end through the host-buffer entry points (pinned host memory, H2D + D2H inside)
    e2e = None
    e2e_steps = max(3, min(args.steps, 10))
    ok = True
    for _ in range(2):
        ok = bench.step_host() is not False
        if not ok:
            break
    if ok:
        torch.cuda.synchronize()
        barrier(world)
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            bench.step_host()
        if hasattr(bench, "finish_host"):
            bench.finish_host()          # every result of the timed pushes is in host memory before the clock stops
        torch.cuda.synchronize()
        e2e_ms = (time.perf_counter() - t0) * 1e3 / e2e_steps
        e2e_ms = max_over_ranks(e2e_ms, world)
        e2e = {"value": world * bench.cells_per_step / (e2e_ms * 1e-3) / 1e9, "unit": "Gcells/s",
               "ms_per_step": e2e_ms, "h2d_bytes_per_step": bench.h2d_bytes(), "d2h_bytes_per_step": bench.d2h_bytes()}
        if hasattr(bench, "step_host_sync"):   # the one-call-at-a-time entry point, for comparison
            e2e["call"] = "nsfrb_stream_push_host_async, two pushes in flight"
            bench.step_host_sync()
            torch.cuda.synchronize()
            barrier(world)
            t0 = time.perf_counter()
            for _ in range(e2e_steps):
                bench.step_host_sync()
            torch.cuda.synchronize()
            e2e["sync_call_ms_per_step"] = max_over_ranks((time.perf_counter() - t0) * 1e3 / e2e_steps, world)
    else:
        e2e = {"value": None, "unit": "Gcells/s", "h2d_bytes_per_step": bench.h2d_bytes(),
               "d2h_bytes_per_step": bench.d2h_bytes(), "note": "the host cannot hold a pinned copy of the cube"}

    if rank != 0:
        return
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    try:
        onchip = measure_onchip_peaks(nsfrb)
    except Exception as exc:  # the roofline then falls back to the theoretical issue rate, and says so
        onchip = None
        print(f"nsfrb_measure_peaks failed: {exc}", file=sys.stderr)
    alg_bytes = bench.algorithmic_bytes()
    kern_bytes = bench.kernel_bytes()
    info = bench.info
    if wl.streaming:
        achieved = kern_bytes / (dominant_ms * 1e-3) / 1e9
        mode = bench.plan.stream_mode()
        # dram__bytes_read.sum + dram__bytes_write.sum of one launch, from the committed ncu capture named in traffic_source
        # (taken in the default mode 3; no capture exists for the other modes)
        traffic, traffic_src = NCU_TRAFFIC.get(wl.name, (None, None)) if mode == 3 else (None, None)
        read_bytes, read_note = stream_read_bytes(wl, info, mode)
        roof = {"bound": "hbm", "achieved": achieved, "peak": hbm_peak, "unit": "GB/s", "frac": achieved / hbm_peak,
                "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src, "kernel": "k_stream",
                "kernel_ms": dominant_ms, "share_of_step": dominant_ms / ms_per_step, "algorithmic_bytes": kern_bytes,
                "step_frac": alg_bytes / (ms_per_step * 1e-3) / 1e9 / hbm_peak,
                "stream_mode": mode,
                "note": "achieved/frac use the contract numerator (the ring once per push, SURVEY.md 8(d): work-avoiding levers raise it); "
                        "what the kernel itself moves is read_bytes (derived) and traffic (ncu): a frac above 1 means the path avoids "
                        "re-reading the ring, not that the kernel beats HBM -- frac_read is its own DRAM rate over the peak",
                "read_bytes": read_bytes, "read_bytes_note": read_note,
                "achieved_read": read_bytes / (dominant_ms * 1e-3) / 1e9,
                "frac_read": read_bytes / (dominant_ms * 1e-3) / 1e9 / hbm_peak,
                # the capture's DRAM bytes over this run's kernel time: how close the kernel is to the bandwidth roofline of what it moves
                "frac_traffic": (traffic / (dominant_ms * 1e-3) / 1e9 / hbm_peak) if traffic else None}
    else:
        roof = offline_roofline(wl, bench, dominant_ms, ms_per_step, hbm_peak, peak_src, onchip, sm_max)
    line = {
        "metric": "Gcells/s (pixel*DM*width*sample)", "value": value, "unit": "Gcells/s", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{wl.name}: {wl.note}", "nchan": wl.nchan, "nt": wl.nt, "nx": wl.nx, "ny": wl.ny,
                   "ndm": len(wl.dm_list), "ndm_unique": info["ndm_unique"], "nwidth": len(wl.width_list),
                   "cells_per_step": bench.cells_per_step,
                   "l2": "inputs larger than L2 (ring 6.4 GB + rotating chunks)" if flusher is None else "L2 flushed between steps",
                   "parallelism": "replicas only" if world > 1 else "1 GPU", "cubes": bool(args.cubes and wl.streaming),
                   "running_sigma": bool(args.running and wl.streaming)},
        "e2e": e2e, "gpu_launches": launches * args.steps, "gpu_launches_per_step": launches,
        "clocks": clocks,
        "roofline": roof,
        "kernel_ms": kernel_ms,
        "ms_per_step_p50": float(np.median(per_step)), "ms_per_step_max": float(np.max(per_step)),
        "wall_s": wall_s,
    }
    if wl.streaming:
        line["chunk_latency_ms"] = ms_per_step
        line["chunk_duration_ms"] = CHUNK_DURATION_MS
        line["chunk_latency_frac"] = ms_per_step / CHUNK_DURATION_MS
    line["onchip_peaks"] = onchip
    line["cpu_baseline"] = cpu_baseline(wl, bench, budget_s=args.cpu_budget) if world == 1 and not args.no_cpu else None
    if wl.name == "c2" and world == 1 and not args.no_extra and not args.cubes and not args.running:
        # the three offline configs in the same run (BASELINE.json: "on all five configs"); c2 stays the headline value
        del bench
        torch.cuda.empty_cache()
        line["workloads"] = {}
        for name in ("c3", "c4", "c5"):
            try:
                line["workloads"][name] = measure_offline_workload(name, nsfrb, hbm_peak, peak_src, onchip, sm_max, local,
                                                                   e2e_ok=True)
            except Exception as exc:
                line["workloads"][name] = {"error": f"{type(exc).__name__}: {exc}"}
                torch.cuda.empty_cache()
    print(json.dumps(line))


# ---------------------------------------------------------------------------- the oracle, timed
def cpu_baseline(wl, bench, budget_s=15.0):
    """The oracle as it stands on the host cores, on a bounded pixel sample of the same workload."""
    from oracle import oracle
    cores = os.cpu_count() or 1
    d = bench.delays
    per_pixel_cells = bench.cells_per_step / wl.npix
    # cost model only to size the sample: ~1 ns per shift-add + ~1.2 ns per cell per core
    if wl.streaming:
        shift_adds = wl.nchan * wl.nt * len(wl.dm_list)
        cells_eval = per_pixel_cells
    else:
        shift_adds = bench.info["shift_adds_per_pixel"]
        cells_eval = per_pixel_cells
    est_s = (shift_adds * 1.0e-9 + cells_eval * 1.2e-9 + wl.nt * len(wl.dm_list) * 6e-9)
    n_pix = int(max(cores, min(wl.npix, budget_s * cores / max(est_s, 1e-9))))
    rng = np.random.default_rng(99)
    pix = np.sort(rng.choice(wl.npix, n_pix, replace=False))
    if wl.streaming:
        # chronological ring contents as the plan holds them is not visible from outside: rebuild the same
        # shape of problem from fresh chunks (timing only)
        ring = torch.randn((wl.nchan, wl.nt, n_pix), generator=torch.Generator().manual_seed(1)).numpy()
        t0 = time.perf_counter()
        oracle.search(ring, d, wl.width_list, raw_end_min=wl.nt - wl.chunk_nt, t_offset=0, nthreads=cores)
        dt = time.perf_counter() - t0
    else:
        sub = bench.cube[:, :, torch.as_tensor(pix, device="cuda")].cpu().numpy()
        t0 = time.perf_counter()
        oracle.search(sub, d, wl.width_list, nthreads=cores)
        dt = time.perf_counter() - t0
    return {"value": n_pix * per_pixel_cells / dt / 1e9, "unit": "Gcells/s", "cores": cores, "kind": "oracle",
            "sample": f"{n_pix} of {wl.npix} pixels of {wl.name}, all DMs/widths, {dt:.1f} s on {cores} threads"}


def run_reference_arm(args, rank, world):
    """--impl reference: the oracle timed on the host cores on the same config/metric."""
    if rank != 0:
        return
    from oracle import oracle
    wl = W.config(args.workload)
    cores = os.cpu_count() or 1
    d = oracle.delays(wl.freqs_GHz, wl.tsamp_s, wl.dm_list)
    if wl.streaming:
        per_pixel_cells = len(wl.dm_list) * len(wl.width_list) * wl.chunk_nt
        est = wl.nchan * wl.nt * len(wl.dm_list) * 1e-9 * 1.5
    else:
        per_pixel_cells = oracle.cells_per_pixel(d, wl.width_list, wl.nt)
        est = per_pixel_cells * 1.2e-9 + wl.nchan * wl.nt * len(wl.dm_list) * 1e-9
    kw = dict(raw_end_min=wl.nt - wl.chunk_nt) if wl.streaming else {}
    # bounded sample: calibrate on a few pixels, then size the per-step sample so that the whole
    # --steps/--warmup run takes about two minutes
    g = torch.Generator().manual_seed(wl.seed)
    n0 = max(cores, 8)
    probe = torch.randn((wl.nchan, wl.nt, n0), generator=g).numpy()
    t0 = time.perf_counter()
    oracle.search(probe, d, wl.width_list, nthreads=cores, **kw)
    dt0 = max(time.perf_counter() - t0, 1e-4)
    per_step_budget = 120.0 / max(args.steps + args.warmup, 1)
    n_pix = int(max(cores, min(wl.npix, n0 * per_step_budget / dt0)))
    del est
    data = torch.randn((wl.nchan, wl.nt, n_pix), generator=g).numpy()
    times = []
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        oracle.search(data, d, wl.width_list, nthreads=cores, **kw)
        if i >= args.warmup:
            times.append(time.perf_counter() - t0)
    s_per_step = float(np.mean(times))
    value = n_pix * per_pixel_cells / s_per_step / 1e9
    sample = f"{n_pix} of {wl.npix} pixels of {wl.name} per step, all DMs/widths"
    print(json.dumps({
        "impl": "reference", "metric": "Gcells/s (pixel*DM*width*sample)", "value": value, "unit": "Gcells/s",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": s_per_step * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{wl.name}: {wl.note}", "nchan": wl.nchan, "nt": wl.nt, "nx": wl.nx, "ny": wl.ny,
                   "ndm": len(wl.dm_list), "nwidth": len(wl.width_list),
                   "cells_per_step": int(wl.npix * per_pixel_cells), "sample": sample},
        "cpu_baseline": {"value": value, "unit": "Gcells/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "Gcells/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def run_bin_arm(args):
    """--op bin: NEXT 2's binning kernel on the C3-shaped cube (x5, the paper's 0.67 s timescale): HBM-bound,
    algorithmic bytes = cube read once + binned cube written once."""
    from paper_2510_18136_b200 import nsfrb
    torch.cuda.set_device(0)
    hbm_peak, peak_src, _ = measured_peaks()
    wl = W.config(args.workload if args.workload != "c2" else "c3")
    factor = args.bin_factor
    cube = torch.randn((wl.nchan, wl.nt, wl.npix), device="cuda", generator=torch.Generator(device="cuda").manual_seed(wl.seed))
    out = torch.empty((wl.nchan, wl.nt // factor, wl.npix), device="cuda")
    per_step = time_steps(lambda: nsfrb.bin_time(cube, factor, out), args.steps, args.warmup)
    ms = float(np.mean(per_step))
    nbytes = cube.numel() * 4 + out.numel() * 4
    print(json.dumps({"metric": "GB/s (time binning, NEXT 2)", "value": nbytes / (ms * 1e-3) / 1e9, "unit": "GB/s", "n_gpus": 1,
                      "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
                      "dtype": "f32", "data": "synthetic",
                      "config": {"workload": f"{wl.name}-shaped cube binned x{factor}", "nchan": wl.nchan, "nt": wl.nt,
                                 "npix": wl.npix, "l2": "inputs larger than L2"},
                      "gpu_launches": args.steps,
                      "roofline": {"bound": "hbm", "achieved": nbytes / (ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                                   "frac": nbytes / (ms * 1e-3) / 1e9 / hbm_peak, "traffic": None, "peak_source": peak_src,
                                   "kernel": "k_bin", "algorithmic_bytes": nbytes}}))


def run_median_arm(args):
    """--op median: NEXT 1's per-(channel, pixel) median subtraction.  HBM-bound by contract: algorithmic bytes =
    cube read once + written once (+ the medians).  Default: 40 chunk-shaped cubes of C2 (16 x 25 x 65 536, the
    paper's 3.35 s chunk) back to back so the inputs exceed L2; --workload c3: the 2048-sample offline cube."""
    from paper_2510_18136_b200 import nsfrb
    torch.cuda.set_device(0)
    hbm_peak, peak_src, _ = measured_peaks()
    wl = W.config(args.workload)
    g = torch.Generator(device="cuda").manual_seed(wl.seed)
    if wl.name == "c2":
        nt, ncubes = wl.chunk_nt, 40
    else:
        nt, ncubes = wl.nt, 1
    cubes = [torch.randn((wl.nchan, nt, wl.npix), device="cuda", generator=g) for _ in range(ncubes)]
    outs = [torch.empty_like(c) for c in cubes[:2]]
    meds = torch.empty((wl.nchan, wl.npix), device="cuda")
    L = nsfrb.lib()
    s = int(torch.cuda.current_stream().cuda_stream)

    def step():
        for i, c in enumerate(cubes):
            rc = L.nsfrb_median_subtract(c.data_ptr(), wl.nchan, nt, wl.npix, outs[i & 1].data_ptr(), meds.data_ptr(), s)
            assert rc == 0, nsfrb.last_error()

    per_step = time_steps(step, args.steps, args.warmup)
    ms = float(np.mean(per_step)) / ncubes
    nbytes = cubes[0].numel() * 8 + meds.numel() * 4
    kern = f"k_median_reg<{nt}>" if nt <= 32 else "k_median_stream"
    print(json.dumps({"metric": "GB/s (median subtraction, NEXT 1)", "value": nbytes / (ms * 1e-3) / 1e9, "unit": "GB/s", "n_gpus": 1,
                      "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
                      "dtype": "f32", "data": "synthetic",
                      "config": {"workload": f"{wl.name}: {wl.nchan} ch x {nt} samples x {wl.npix} pixels", "cubes_per_step": ncubes,
                                 "l2": "inputs larger than L2"},
                      "gpu_launches": args.steps * ncubes,
                      "roofline": {"bound": "hbm", "achieved": nbytes / (ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                                   "frac": nbytes / (ms * 1e-3) / 1e9 / hbm_peak, "traffic": None, "peak_source": peak_src,
                                   "kernel": kern, "algorithmic_bytes": nbytes}}))


def run_cluster_arm(args):
    """--op cluster: NEXT 3's candidate selection (top-10 + PSF-mask clustering, one launch of k_cluster) on a
    map of the workload's image size.  Algorithmic bytes = the S/N map read once (the ten selection rounds re-read
    each CTA's 8 KB slice from L1/L2); at these sizes the launch is latency-bound, which the fraction shows."""
    from paper_2510_18136_b200 import nsfrb
    torch.cuda.set_device(0)
    hbm_peak, peak_src, _ = measured_peaks()
    wl = W.config(args.workload)
    psf = W.synthetic_psf(301, 0)
    m, _ = W.synthetic_snr_map(wl.nx, wl.ny, psf, 0)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    with nsfrb.Plan(wl.nx, wl.ny, 2, 64, [1.3, 1.5], W.TSAMP_S, [0.0], [1], wl.threshold) as plan:
        dm = torch.from_numpy(m.ravel().copy()).cuda()
        arg = torch.zeros((3, wl.npix), dtype=torch.int32, device="cuda")
        dpsf = torch.from_numpy(psf).cuda()
        dmask, _ = nsfrb.psf_mask(dpsf, 90.0)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        for i in range(args.warmup + args.steps):
            flush.zero_()                                  # L2 flush between iterations
            j = i - args.warmup
            if j >= 0:
                ev[j][0].record()
            res = plan.cluster(dm, arg, dpsf, dmask, 10)
            if j >= 0:
                ev[j][1].record()
        torch.cuda.synchronize()
        ms = float(np.mean([a.elapsed_time(b) for a, b in ev]))
        got = res.to_host()
    nbytes = wl.npix * 4
    print(json.dumps({"metric": "maps/s (top-10 + PSF clustering, NEXT 3)", "value": 1e3 / ms, "unit": "maps/s", "n_gpus": 1,
                      "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
                      "dtype": "f32 keys, f64 means", "data": "synthetic",
                      "config": {"workload": f"{wl.nx}x{wl.ny} S/N map, 301x301 PSF, top 10", "l2": "flushed between steps",
                                 "n_found": len(got["pixels"]), "best_pixel": got["pixels"][got["best"]] if got["pixels"] else -1},
                      "gpu_launches": args.steps,
                      "roofline": {"bound": "hbm", "achieved": nbytes / (ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                                   "frac": nbytes / (ms * 1e-3) / 1e9 / hbm_peak, "traffic": None, "peak_source": peak_src,
                                   "kernel": "k_cluster", "algorithmic_bytes": nbytes,
                                   "note": "latency-bound: one launch, three dependent phases"}}))


def run_image_arm(args):
    """--op image: NEXT 4, the paper's imaging block (25 samples x 8 channels x 4656 baselines x 2 pols = 14.9 MB -> 25 images
    of 175 x 175) for 16 sub-bands back to back = one 3.35 s chunk of the array.  ALU-bound by its own count: 4 FMA per
    (gridded visibility, image column) in the row transform + 2 per (row, pixel) in the column transform."""
    from paper_2510_18136_b200 import nsfrb
    torch.cuda.set_device(0)
    hbm_peak, peak_src, _ = measured_peaks()
    onchip = measure_onchip_peaks(nsfrb)
    uv = W.imaging_array(0)
    n, nt, nsub = W.IMG_N, 25, 16
    imagers = [nsfrb.Imager(n, W.IMG_PIXEL_RAD, uv, W.imaging_freqs(sb)) for sb in range(nsub)]
    g = torch.Generator(device="cuda").manual_seed(7)
    vis = [torch.view_as_complex(torch.randn((nt, 8, len(uv), 2, 2), device="cuda", generator=g)) for _ in range(nsub)]
    chunk = torch.empty((nsub, nt, n * n), device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    # the 16 sub-bands are independent (one correlator node each in the paper, L48): each imager is one launch of ~150 CTAs, so
    # they go out on four streams and share the GPU; the timed stream waits for all of them
    side = [torch.cuda.Stream() for _ in range(int(os.environ.get("NSFRB_BENCH_IMAGE_STREAMS", "4")))]
    ev0 = torch.cuda.Event()
    evs = [torch.cuda.Event() for _ in side]

    def step():
        cur = torch.cuda.current_stream()
        ev0.record(cur)
        for st in side:
            st.wait_event(ev0)
        for sb in range(nsub):
            imagers[sb].image(vis[sb], out=chunk[sb], stream=side[sb % len(side)])
        for st, ev in zip(side, evs):
            ev.record(st)
            cur.wait_event(ev)

    per_step = time_steps(step, args.steps, args.warmup, lambda: flush.zero_())
    ms = float(np.mean(per_step))
    nent = sum(int((im.table()[1] > 0).sum()) for im in imagers)
    ops = (nent * n * 4 + nsub * (n // 2 + 1) * n * n * 2) * nt          # FMA lane-ops per chunk
    peak = onchip["ffma"]["per_s"] / 1e12
    nbytes = sum(v.numel() * 8 for v in vis) + chunk.numel() * 4
    # the oracle on one time sample of one sub-band, scaled
    from oracle import imaging as OI
    v1 = vis[0][:1].cpu().numpy()
    t0 = time.perf_counter()
    OI.image(v1, uv, W.imaging_freqs(0))
    cpu_s = time.perf_counter() - t0
    for im in imagers:
        im.close()
    print(json.dumps({"metric": "images/s (NEXT 4: grid + inverse DFT, 175 x 175, 8 channels summed)", "value": nsub * nt / (ms * 1e-3),
                      "unit": "images/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
                      "higher_is_better": True, "dtype": "f32", "data": "synthetic",
                      "config": {"workload": "one 3.35 s chunk of the array: 16 sub-bands x 25 samples x 8 channels x 4656 baselines x 2 pols",
                                 "l2": "flushed between steps", "chunk_latency_frac": ms / CHUNK_DURATION_MS,
                                 "streams": len(side)},
                      "gpu_launches": nsub * args.steps,
                      "roofline": {"bound": "alu", "achieved": ops / (ms * 1e-3) / 1e12, "peak": peak, "unit": "T lane-ops/s",
                                   "frac": ops / (ms * 1e-3) / 1e12 / peak, "traffic": None,
                                   "peak_source": "measured FFMA issue rate (nsfrb_measure_peaks, this run)", "kernel": "k_image",
                                   "algorithmic_ops": ops, "algorithmic_bytes": nbytes,
                                   "hbm_frac": nbytes / (ms * 1e-3) / 1e9 / hbm_peak},
                      "cpu_baseline": {"value": 1.0 / cpu_s, "unit": "images/s", "cores": 1, "kind": "oracle",
                                       "sample": "one time sample of one sub-band (numpy ifft2 route)"}}))


def stream_read_bytes(wl, info, mode):
    """Bytes one k_stream launch has to read, derived from the plan: mode 1 marches over raw rows up to the widest
    window; modes 2/3 read one history value per (unique trial, step) in the start ranges of the widths and, in the plain runs
    between them, every row (mode 2) or one 8-row block sum per 8 rows plus the ragged ends (mode 3)."""
    C = wl.chunk_nt
    steps = min(wl.nt, int(info["wmax"]) + C)
    if mode <= 1:
        return steps * wl.nchan * wl.npix * 4, "raw rows up to the widest window, every channel"
    tt = 6
    cell = [False] * (steps + tt + 1)
    for w in sorted(set(int(x) for x in wl.width_list)):
        for r in range(max(0, w // tt * tt), min(steps, (w + C - 1) // tt * tt + tt)):
            cell[r] = True
    for r in range(0, min(steps, C + tt)):
        cell[r] = True
    rows, r = 0.0, 0
    while r < steps:
        if cell[r]:
            rows += 1
            r += 1
            continue
        r0 = r
        while r < steps and not cell[r]:
            r += 1
        n = r - r0
        rows += n if mode == 2 else min(n, tt + 7 + max(0, n - tt - 14) / 8.0 + 7)
    return int(rows * int(info["ndm_unique"]) * wl.npix * 4), "history rows: start ranges row by row, plain runs by 8-row blocks (estimate from the width list)"


def measure_onchip_peaks(nsfrb_mod, iters=2000):
    """The achieved on-chip ceilings of this GPU (nsfrb_measure_peaks: FADD/FMNMX/FMNMX3 issue, the search's
    2 FADD + 1 FMNMX3 cell pair, conflict-free shared-memory streams), with the SM clock derived from the two timings."""
    pk = nsfrb_mod.measure_peaks(iters)
    out = {}
    for name, (per_s, per_clk_sm) in pk.items():
        out[name] = {"per_s": per_s, "per_clk_per_sm": per_clk_sm,
                     "implied_sm_mhz": per_s / per_clk_sm / 148 / 1e6 if per_clk_sm > 0 else None}
    return out


def run_peaks_arm(args):
    """--op peaks: the measured denominators of the offline (alu) roofline."""
    from paper_2510_18136_b200 import nsfrb
    torch.cuda.set_device(0)
    sampler = ClockSampler(0)
    sampler.start()
    pk = None
    t0 = time.perf_counter()
    while pk is None or time.perf_counter() - t0 < 1.0:   # keep the load up long enough for nvidia-smi to see it
        pk = measure_onchip_peaks(nsfrb, 4000)
    clocks = sampler.stop()
    print(json.dumps({"metric": "T lane-ops/s (FADD issue) and T words/s (shared memory), measured", "unit": "T/s",
                      "value": pk["fadd"]["per_s"] / 1e12, "n_gpus": 1, "higher_is_better": True, "data": "synthetic",
                      "config": {"workload": "on-chip peaks: 2 CTAs x 1024 threads per SM, 8 independent chains per thread"},
                      "peaks": pk, "clocks": clocks}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c2")
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--cpu-budget", type=float, default=15.0)
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="c2: do not also time c3, c4, c5 (the `workloads` object)")
    ap.add_argument("--cubes", action="store_true", help="c2: also write the S/N and TOA cubes every push (NEXT 3)")
    ap.add_argument("--running", action="store_true", help="c2: also the running-sigma maps every push (NEXT 1)")
    ap.add_argument("--op", default="search", choices=["search", "bin", "cluster", "median", "peaks", "image"],
                    help="bin: time the binning kernel (NEXT 2); cluster: top-10 + PSF clustering (NEXT 3); "
                         "median: per-pixel median subtraction (NEXT 1)")
    ap.add_argument("--bin-factor", type=int, default=5)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "cuda" else args.warmup
    rank, world, local = dist_setup(args.gpus)
    if args.op == "bin" and args.impl == "cuda":
        if rank == 0:
            run_bin_arm(args)
    elif args.op == "median" and args.impl == "cuda":
        if rank == 0:
            run_median_arm(args)
    elif args.op == "image" and args.impl == "cuda":
        if rank == 0:
            run_image_arm(args)
    elif args.op == "peaks" and args.impl == "cuda":
        if rank == 0:
            run_peaks_arm(args)
    elif args.op == "cluster" and args.impl == "cuda":
        if rank == 0:
            run_cluster_arm(args)
    elif args.impl == "reference":
        run_reference_arm(args, rank, world)
    else:
        run_cuda_arm(args, rank, world, local)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
