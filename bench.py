#!/usr/bin/env python
"""bench.py -- throughput of the MUSER dirty-imaging hot path (BASELINE.json: "gridded visibilities/s and dirty
images/s (MUSER-II frame), % of roofline").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

Workload: BASELINE.json configs[2], the MUSER-II full frame (60 antennas -> 1770 baselines x 16 channels x 2
polarisations = 56,640 visibilities -> 113,280 gridded samples, 1024^2 grid, PSWF support 7, oversample 128).
One STEP = one pass of the whole hot path (reset -> bin -> grid -> cuFFT rows -> column FFT + correction: dirty image + beam)
over a batch of FRAMES_PER_STEP = 80 distinct seeded synthetic frames (145 MB of inputs, larger than the 126 MB
L2, so every frame's inputs come from HBM).  value = input visibilities gridded per second over all ranks, inputs
resident in HBM; e2e = the same through muser_frame_host with pinned HOST buffers (H2D + D2H inside the timing).
Multi-GPU: frames are independent, so ranks process disjoint frames with no data-path collective (weak scaling).
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

CFG = 3
FRAMES_PER_STEP = 80
# dram__bytes_read.sum + dram__bytes_write.sum of one k_grid_owner_s7 launch of this workload, from the committed
# `ncu --set full` capture (profiles/); None until that capture exists
TRAFFIC_NCU = 1.859e9   # profiles/r01f_final.md: k_grid_owner_s7 226 MB read + 1,633 MB written (includes the 671 MB FFT input H)
WORKLOAD = ("configs[2] MUSER-II full frame: 56,640 vis (113,280 samples) -> 1024^2 grid, PSWF S=7 Q=128 "
            "-> dirty image + beam")
METRIC = "gridded_visibilities_per_s"
UNIT = "vis/s"


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def make_frames(nframes, seed0=0):
    """nframes distinct frames of the cfg-3 shape: the array geometry and sky are those of synth.make_frame(3); every
    frame gets its own noise realisation (so buffers differ and nothing is cached between frames)."""
    from paper_1712_06913_b200 import synth
    base = synth.make_frame(CFG)
    frames = []
    for k in range(nframes):
        rng = np.random.default_rng([synth.SEED0, 1000 + CFG, seed0 + k])
        noise = (rng.standard_normal((base.nvis, 2)) * 0.05).astype(np.float32)
        vis = (base.vis + (noise[:, 0] + 1j * noise[:, 1]).astype(np.complex64)).astype(np.complex64)
        frames.append((base.uvw_m.copy(), base.freq_hz.copy(), vis, base.weight.copy()))
    return base.params, frames


class ClockSampler(threading.Thread):
    """Samples SM clock and clock-event reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.sm, self.reasons, self.max_mhz = index, False, [], set(), None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def sample(self):
        if not self.nv:
            return
        nv = self.nv
        try:
            self.sm.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
            r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
            names = {"hw_slowdown": nv.nvmlClocksEventReasonHwSlowdown,
                     "hw_thermal_slowdown": nv.nvmlClocksEventReasonHwThermalSlowdown,
                     "sw_thermal_slowdown": nv.nvmlClocksEventReasonSwThermalSlowdown,
                     "sw_power_cap": nv.nvmlClocksEventReasonSwPowerCap}
            for k, bit in names.items():
                if r & bit:
                    self.reasons.add(k)
        except Exception:
            pass

    def run(self):
        while not self.stop_flag:
            self.sample()
            time.sleep(0.002)

    def result(self):
        return {"sm_mhz": float(np.median(self.sm)) if self.sm else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.sm)}


def cpu_oracle_frame(params, frame, T, cx):
    """One frame through the oracle as it stands: plain-C fp64 gridder + numpy fp64 centred inverse FFT + correction
    (dirty image and beam)."""
    from oracle import muser_oracle as mo
    from oracle import oracle_c as oc
    uvw, freq, vis, wt = frame
    G, Gw, st = oc.grid(uvw, freq, vis, wt, params.n, params.n, params.cell_arcsec, params.oversample, params.support, T)
    d, _ = mo.dirty_image(G[0], cx, cx)
    p, _ = mo.dirty_image(Gw[0].astype(np.complex128), cx, cx)
    return d, p, st


def run_reference(args):
    """--impl reference: the oracle timed on the host cores; each step = ORACLE_FRAMES_PER_STEP frames of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import muser_oracle as mo
    params, frames = make_frames(4)
    T = mo.table_pswf(params.support, params.oversample)
    cx = mo.corrector(T, params.support, params.oversample, params.n)
    nvis = frames[0][2].shape[0]
    per_step = 2
    for w in range(args.warmup):
        cpu_oracle_frame(params, frames[w % 4], T, cx)
    t0 = time.perf_counter()
    for k in range(args.steps):
        for j in range(per_step):
            cpu_oracle_frame(params, frames[(k * per_step + j) % 4], T, cx)
    dt = time.perf_counter() - t0
    value = args.steps * per_step * nvis / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "frames_per_step": per_step, "nvis_per_frame": nvis,
                   "sample": "each step = 2 whole frames of the workload through the oracle on one host core"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle",
                         "sample": f"{args.steps * per_step} whole frames (oracle_c gridder + numpy fp64 FFT + correction)"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "images_per_s": args.steps * per_step / dt,
    }
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="muser")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    from paper_1712_06913_b200 import binding, build, shard
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        build.build()
    if dist:
        dist.barrier()
    W = max(args.warmup, 3)

    params, frames = make_frames(FRAMES_PER_STEP, seed0=shard.frame_seeds(rank, FRAMES_PER_STEP)[0])
    n, nvis = params.n, frames[0][2].shape[0]
    B = FRAMES_PER_STEP
    # one batch = B frames back to back in memory, frame b -> grid b (muser_grid_batched)
    host = [np.ascontiguousarray(np.concatenate([fr[i] for fr in frames])) for i in range(4)]
    host.append(np.repeat(np.arange(B, dtype=np.int32), nvis))
    dev = [torch.from_numpy(a).cuda() for a in host]
    im = binding.Imager(n, n, params.cell_arcsec, params.support, params.oversample)
    im.set_batch(B)
    dirty = torch.empty((B, n, n), device="cuda")
    psf = torch.empty((B, n, n), device="cuda")
    stream = torch.cuda.current_stream()

    def step():
        im.reset()
        im.grid_batched(*dev)
        im.dirty_psf(dirty, psf)

    def barrier():
        torch.cuda.synchronize()
        if dist:
            dist.barrier()
            torch.cuda.synchronize()

    def max_over_ranks(ms):
        return shard.max_over_ranks(ms, dist, device="cuda")

    for _ in range(W):
        step()
    barrier()
    sampler = ClockSampler(local)
    sampler.sample()
    sampler.start()
    l0 = im.get_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    barrier()
    sampler.stop_flag = True
    sampler.join()
    sampler.sample()
    launches = im.get_launch_count() - l0
    ms = max_over_ranks(e0.elapsed_time(e1))
    frames_total = args.steps * B * world
    value = shard.aggregate_rate(args.steps * B * nvis, world, ms)

    # ---- per-stage device time, live, with CUDA events on the launching stream (second timed pass)
    im.set_profiling(True)
    for _ in range(max(3, min(args.steps, 10))):
        step()
    prof = im.get_profile()
    im.set_profiling(False)
    stage_us = {k: (1e3 * v[0] / v[1] if v[1] else None) for k, v in prof.items()}
    grid_us = stage_us["grid"]
    # algorithmic bytes of one gridding launch: per frame 32 B per input visibility + every
    # cell of G (8 B) and Gw (4 B) written once; one launch grids B frames
    alg_bytes = B * (32.0 * nvis + 12.0 * n * n)
    peak, peak_src = _peaks()
    achieved = alg_bytes / (grid_us * 1e-6) / 1e9
    roofline = {"bound": "hbm", "kernel": "k_grid_owner_s7 (gridding stage; zero-fill units of empty tiles included)", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": TRAFFIC_NCU, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": alg_bytes, "kernel_us": grid_us,
                "kernel_us_per_frame": grid_us / B, "stage_us_per_launch": stage_us,
                "stage_us_per_frame": {k: (v / B if v else None) for k, v in stage_us.items()}}

    # ---- latency of ONE frame through the un-batched calls (reset -> grid -> dirty_psf on one 1024^2 grid)
    im1 = binding.Imager(n, n, params.cell_arcsec, params.support, params.oversample)
    dev1 = [[torch.from_numpy(a).cuda() for a in fr] for fr in frames[:16]]
    d1 = torch.empty((n, n), device="cuda")
    p1 = torch.empty((n, n), device="cuda")
    for fr in dev1[:4]:
        im1.reset(); im1.grid(*fr); im1.dirty_psf(d1, p1)
    barrier()
    e0.record(stream)
    for fr in dev1:
        im1.reset(); im1.grid(*fr); im1.dirty_psf(d1, p1)
    e1.record(stream)
    barrier()
    single_us = 1e3 * e0.elapsed_time(e1) / len(dev1)
    im1.destroy()
    del dev1

    # ---- end to end through the host-buffer entry point (pinned host memory; H2D + D2H inside the timed region)
    pin = [torch.from_numpy(a).pin_memory() for a in host]
    d_host = torch.empty((B, n, n), dtype=torch.float32).pin_memory()
    p_host = torch.empty((B, n, n), dtype=torch.float32).pin_memory()
    for _ in range(2):
        im.frame_host(pin[0], pin[1], pin[2], pin[3], pin[4], d_host, p_host)
    barrier()
    e2e_steps = max(2, min(args.steps, 5))
    e0.record(stream)
    for k in range(e2e_steps):
        im.frame_host(pin[0], pin[1], pin[2], pin[3], pin[4], d_host, p_host)
    e1.record(stream)
    barrier()
    e2e_ms = max_over_ranks(e0.elapsed_time(e1))
    e2e_value = e2e_steps * B * world * nvis / (e2e_ms * 1e-3)
    h2d = sum(int(a.nbytes) for a in host)
    d2h = 2 * B * n * n * 4

    cpu = None
    if rank == 0 and not args.no_cpu_baseline:
        from oracle import muser_oracle as mo
        T = mo.table_pswf(params.support, params.oversample)
        cx = mo.corrector(T, params.support, params.oversample, n)
        cpu_oracle_frame(params, frames[0], T, cx)
        t0 = time.perf_counter()
        done = 0
        while done < 3 or (time.perf_counter() - t0 < 10.0 and done < FRAMES_PER_STEP):
            cpu_oracle_frame(params, frames[done % len(frames)], T, cx)
            done += 1
        dt = time.perf_counter() - t0
        cpu = {"value": done * nvis / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"{done} whole frames of the workload (oracle_c fp64 gridder + numpy fp64 FFT + correction), "
                         f"{dt:.1f} s on {os.cpu_count()} available cores, 1 used",
               "images_per_s": done / dt}

    limits = binding.microbench() if rank == 0 else None

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": W,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": WORKLOAD, "batching": "one step = 80 distinct frames, each onto its own grid, in one "
                                   "muser_grid_batched + muser_dirty_psf call", "frames_per_step": FRAMES_PER_STEP,
                       "nvis_per_frame": nvis,
                       "l2_policy": "per step 145 MB of inputs and 1.0 GB of grids stream through a 126 MB L2",
                       "launch": "stream", "parallelism": f"frames x{world}" if world > 1 else "single"},
            "images_per_s": frames_total / (ms * 1e-3), "dirty_and_beam_pairs_per_s": frames_total / (ms * 1e-3),
            "us_per_frame": 1e3 * ms / (args.steps * FRAMES_PER_STEP), "single_frame_latency_us": single_us,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps_timed": e2e_steps, "us_per_frame": 1e3 * e2e_ms / (e2e_steps * B)},
            "gpu_launches": int(launches), "clocks": sampler.result(), "roofline": roofline, "cpu_baseline": cpu,
            "device_limits": limits,
        }
        print(json.dumps(line))
    im.destroy()
    if dist:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
