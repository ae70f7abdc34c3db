#!/usr/bin/env python
"""bench.py -- throughput of the MUSER dirty-imaging hot path (BASELINE.json: "gridded visibilities/s and dirty
images/s (MUSER-II frame), % of roofline").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config {1,2,3,4,5}] [--impl reference]

Default workload: BASELINE.json configs[2] (cfg 3), the MUSER-II full frame (60 antennas -> 1770 baselines x 16
channels x 2 polarisations = 56,640 visibilities -> 113,280 gridded samples, 1024^2 grid, PSWF support 7, oversample
128).  One STEP = one pass of the whole hot path (reset -> bin -> grid -> row FFT -> column FFT + correction: dirty
image + beam) over a batch of 80 distinct seeded synthetic frames, each onto its own grid (145 MB of inputs per step,
larger than the 126 MB L2).  value = input visibilities gridded per second over all ranks through the flat call
muser_grid_batched (32 B per visibility), inputs resident in HBM; e2e = the same through the host-buffer
entry point with pinned HOST buffers (H2D + D2H inside the timing).  The line also carries the channelised entry
muser_grid_rows ("rows"), the un-batched single-frame numbers (stream-launched and CUDA-graph-replayed), three roofline
fractions and the oracle timed on the host.  --config N benches another BASELINE.json config
(its line names the workload); those lines are kept under profiles/.
Multi-GPU: frames are independent, so ranks process disjoint frames with no data-path collective (weak scaling).
"""
from __future__ import annotations

import argparse
import json
import os
import re
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "gridded_visibilities_per_s"
UNIT = "vis/s"
WORKLOADS = {
    1: "configs[0] MUSER-I snapshot: 780 vis -> 256^2 grid, Gaussian S=7 Q=8 -> dirty image + beam",
    2: "configs[1] MUSER-I full frame: 24,960 vis -> 512^2 grid, PSWF S=7 Q=128 -> dirty image + beam",
    3: "configs[2] MUSER-II full frame: 56,640 vis (113,280 samples) -> 1024^2 grid, PSWF S=7 Q=128 -> dirty image + beam",
    4: "configs[3] MUSER-II per-frame/channel/polarisation imaging: chunk of 64 frames = 2048 grids of 512^2, 1770 vis each",
    5: "configs[4] MUSER-II 300 snapshots, 16,992,000 vis -> one 4096^2 grid, 32 w-planes (supports 7..31), Q=64",
}
FRAMES_PER_STEP = {1: 256, 2: 128, 3: 80}


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def _committed_traffic(kernel):
    """dram bytes per launch of `kernel` from the newest committed ncu summary (profiles/r02*_final.md), or (None, None)."""
    best = None
    pdir = os.path.join(ROOT, "profiles")
    for fn in sorted(os.listdir(pdir)) if os.path.isdir(pdir) else []:
        if not re.match(r"r\d+.*final\.md$", fn):
            continue
        for line in open(os.path.join(pdir, fn)):
            m = re.match(r"\|\s*traffic_bytes_per_launch\s+" + re.escape(kernel) + r"\s*\|\s*([0-9.eE+]+)\s*\|", line)
            if m:
                best = (float(m.group(1)), "profiles/" + fn)
    return best if best else (None, None)


def make_frames(nframes, seed0=0, cfg=3):
    """nframes distinct frames of the config's shape: the array geometry and sky are those of synth.make_frame(cfg); every
    frame gets its own noise realisation (so buffers differ and nothing is cached between frames)."""
    from inputs import synth
    base = synth.make_frame(cfg)
    frames = []
    for k in range(nframes):
        rng = np.random.default_rng([synth.SEED0, 1000 + cfg, seed0 + k])
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


# ------------------------------------------------------------------------------------------------- oracle on the host
_ORACLE_CTX = {}


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


def _oracle_worker(k):
    c = _ORACLE_CTX
    cpu_oracle_frame(c["params"], c["frames"][k % len(c["frames"])], c["T"], c["cx"])
    return k


def _oracle_tables(params):
    from oracle import muser_oracle as mo
    T = mo.table_pswf(params.support, params.oversample) if params.kernel == "pswf" else mo.table_gauss(params.support, params.oversample)
    return T, mo.corrector(T, params.support, params.oversample, params.n)


def cpu_baseline(params, frames, nvis, budget_s=10.0):
    """The oracle on the box's host cores: one core, then all cores (independent frames on a process pool)."""
    import multiprocessing as mp
    T, cx = _oracle_tables(params)
    cpu_oracle_frame(params, frames[0], T, cx)
    t0 = time.perf_counter()
    done = 0
    while done < 3 or (time.perf_counter() - t0 < budget_s and done < len(frames)):
        cpu_oracle_frame(params, frames[done % len(frames)], T, cx)
        done += 1
    dt = time.perf_counter() - t0
    out = {"value": done * nvis / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
           "sample": f"{done} whole frames of the workload (oracle_c fp64 gridder + numpy fp64 FFT + correction), {dt:.1f} s",
           "images_per_s": done / dt}
    ncores = os.cpu_count() or 1
    try:
        _ORACLE_CTX.update(params=params, frames=frames[:8], T=T, cx=cx)
        njobs = max(2 * ncores, 8)
        with mp.get_context("fork").Pool(ncores) as pool:
            pool.map(_oracle_worker, range(ncores))                      # warm the workers
            t0 = time.perf_counter()
            pool.map(_oracle_worker, range(njobs))
            dta = time.perf_counter() - t0
        out["all_cores"] = {"value": njobs * nvis / dta, "unit": UNIT, "cores": ncores, "images_per_s": njobs / dta,
                            "sample": f"{njobs} whole frames on a pool of {ncores} processes, {dta:.1f} s"}
    except Exception as ex:                                              # a box without fork / enough memory
        out["all_cores"] = {"unavailable": str(ex)[:100]}
    return out


def cpu_direct_dft_cfg1():
    """the direct-DFT imager (definition (I)) on cfg 1, every pixel (1,560 samples x 65,536 pixels)."""
    from oracle import muser_oracle as mo
    from oracle import oracle_c as oc
    from inputs import synth
    fr = synth.make_frame(1)
    p = fr.params
    smp = mo.coordinates(fr.uvw_m, fr.freq_hz, fr.vis, fr.weight, p.n, p.n, p.cell_arcsec, p.oversample, p.support)
    xs, ys = np.meshgrid(np.arange(p.n), np.arange(p.n))
    cell = p.cell_arcsec * mo.ARCSEC
    l, m = (xs.ravel() - p.n / 2) * cell, (ys.ravel() - p.n / 2) * cell
    t0 = time.perf_counter()
    oc.dft(smp["u"], smp["v"], smp["w"], smp["val"], l, m)
    dt = time.perf_counter() - t0
    return {"seconds": dt, "samples": int(smp["val"].shape[0]), "pixels": int(l.shape[0]), "cores": 1,
            "images_per_s": 1.0 / dt}


def run_reference(args):
    """--impl reference: the oracle timed on the host cores; each step = 2 frames of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = args.config if args.config in (1, 2, 3) else 3
    params, frames = make_frames(4, cfg=cfg)
    T, cx = _oracle_tables(params)
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
        "config": {"workload": WORKLOADS[cfg], "frames_per_step": per_step, "nvis_per_frame": nvis,
                   "sample": "each step = 2 whole frames of the workload through the oracle on one host core"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle",
                         "sample": f"{args.steps * per_step} whole frames (oracle_c gridder + numpy fp64 FFT + correction)"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "images_per_s": args.steps * per_step / dt,
    }
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------- GPU arm
def _stage_us(im, step, reps):
    im.set_profiling(True)
    for _ in range(reps):
        step()
    prof = im.get_profile()
    im.set_profiling(False)
    # per STEP (a stage may be several launches per step: the transform runs rows -> columns over sub-batches of grids)
    return {k: (1e3 * v[0] / reps if v[1] else None) for k, v in prof.items()}


def _timed(torch, stream, fn, steps, barrier):
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for _ in range(steps):
        fn()
    e1.record(stream)
    barrier()
    return e0.elapsed_time(e1)


def bench_frames(args, cfg, torch, binding, shard, dist, rank, world, local):
    """cfgs 1-3: batches of whole frames, one grid per frame."""
    W = max(args.warmup, 3)
    B = FRAMES_PER_STEP[cfg]
    params, frames = make_frames(B, seed0=shard.frame_seeds(rank, B)[0], cfg=cfg)
    n, nvis = params.n, frames[0][2].shape[0]
    host = [np.ascontiguousarray(np.concatenate([fr[i] for fr in frames])) for i in range(4)]
    host.append(np.repeat(np.arange(B, dtype=np.int32), nvis))
    dev = [torch.from_numpy(a).cuda() for a in host]

    def new_imager(ngrids):
        im_ = binding.Imager(n, n, params.cell_arcsec, params.support, params.oversample)
        if params.kernel == "gauss":
            im_.set_kernel(binding.MUSER_KERNEL_GAUSS, 0.0)
        if ngrids > 1:
            im_.set_batch(ngrids)
        return im_

    im = new_imager(B)
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

    for _ in range(W):
        step()
    sampler = ClockSampler(local)
    sampler.sample()
    sampler.start()
    l0 = im.get_launch_count()
    ms = shard.max_over_ranks(_timed(torch, stream, step, args.steps, barrier), dist, device="cuda")
    sampler.stop_flag = True
    sampler.join()
    sampler.sample()
    launches = im.get_launch_count() - l0
    value = shard.aggregate_rate(args.steps * B * nvis, world, ms)

    # ---- per-stage device time, live, with CUDA events on the launching stream (second timed pass)
    stage_us = _stage_us(im, step, max(3, min(args.steps, 10)))
    peak, peak_src = _peaks()
    bin_us, grid_us = stage_us["bin"], stage_us["grid"]
    # algorithmic bytes: 32 B per input visibility (read by the BINNING kernels) + every cell of G (8 B)
    # and Gw (4 B) written once (by the GRIDDING kernel); one launch handles B frames
    in_bytes, grid_bytes = B * 32.0 * nvis, B * 12.0 * n * n
    # the committed ncu capture is of cfg 3 with 80 frames per launch: it says nothing about any other workload
    traffic, traffic_src = _committed_traffic("k_grid_owner_s7") if (cfg == 3 and B == 80) else (None, None)
    frac_a1a2 = (in_bytes + grid_bytes) / ((bin_us + grid_us) * 1e-6) / 1e9 / peak
    # beside the algorithmic figure, the DRAM bytes the A1+A2 kernels really move (ncu dram__bytes_read + write of the
    # committed capture of this same workload) over the live bin + grid time: what fraction of the HBM bandwidth is in use
    a1a2_kernels = ("k_owner_count", "k_owner_scan_write", "k_owner_scatter", "k_grid_owner_s7")
    moved = [_committed_traffic(k)[0] for k in a1a2_kernels] if (cfg == 3 and B == 80) else [None]
    moved_bytes = sum(moved) if all(m is not None for m in moved) else None
    frac_moved = moved_bytes / ((bin_us + grid_us) * 1e-6) / 1e9 / peak if moved_bytes else None
    roofline = {
        "bound": "hbm", "kernel": "A1 + A2: k_owner_count, k_owner_scan_*, k_owner_scatter (binning) + k_grid_owner_s7 (gridding; "
                                  "tiles without samples are flagged, not zero-filled)",
        "achieved": (in_bytes + grid_bytes) / ((bin_us + grid_us) * 1e-6) / 1e9, "peak": peak, "unit": "GB/s", "frac": frac_a1a2,
        "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
        "algorithmic_bytes_per_launch": in_bytes + grid_bytes,
        "fractions": {
            "a1_a2_over_bin_plus_grid_time": frac_a1a2,
            "k4_alone_all_bytes_over_grid_time": (in_bytes + grid_bytes) / (grid_us * 1e-6) / 1e9 / peak,
            "k4_alone_grid_bytes_over_grid_time": grid_bytes / (grid_us * 1e-6) / 1e9 / peak,
            "k4_half_plane_bytes_written_over_grid_time": 0.5 * grid_bytes / (grid_us * 1e-6) / 1e9 / peak,
            "a1_a2_dram_bytes_moved_over_bin_plus_grid_time": frac_moved,
        },
        "dram_bytes_moved_a1_a2": moved_bytes,
        "note": "frac = A1+A2 ALGORITHMIC bytes (SURVEY 8(d): 32 B/vis + 12 B/cell) over binning + gridding time: the figure the "
                ">= 0.50 target of north_star is judged against (DESIGN.md section 6).  It is not bandwidth in use: the gridder "
                "stores the non-empty tiles of the Hermitian half-plane only (at most 6 B/cell), so the DRAM bytes the four A1+A2 "
                "kernels really move (`dram_bytes_moved_a1_a2`, ncu, committed capture of this workload) are fewer; that fraction "
                "of the HBM peak is `a1_a2_dram_bytes_moved_over_bin_plus_grid_time`.  `traffic` is k_grid_owner_s7's alone",
        "kernel_us": bin_us + grid_us, "stage_us_per_launch": stage_us,
        "stage_us_per_frame": {k: (v / B if v else None) for k, v in stage_us.items()}}

    # ---- the channelised entry point on the same frames (12.4 B per visibility; polarisations summed before gridding)
    nchan, npol = 16, 2 if cfg > 1 else 1
    rows = None
    if cfg > 1:
        nrow = nvis // (nchan * npol)
        r_uvw = torch.from_numpy(np.stack([fr[0].reshape(npol, nchan, nrow, 3)[0, 0] for fr in frames])).cuda()
        r_freq = torch.from_numpy(frames[0][1].reshape(npol, nchan, nrow)[0, :, 0].copy()).cuda()
        r_vis = torch.from_numpy(np.stack([fr[2].reshape(npol, nchan, nrow) for fr in frames])).cuda()
        r_wt = torch.from_numpy(np.stack([fr[3].reshape(npol, nchan, nrow) for fr in frames])).cuda()
        r_gid = torch.from_numpy(np.repeat(np.arange(B, dtype=np.int32)[:, None], nchan, 1).copy()).cuda()

        def step_rows():
            im.reset()
            im.grid_rows(r_uvw, r_freq, r_vis, r_wt, r_gid, binding.MUSER_POLS_SUM)
            im.dirty_psf(dirty, psf)

        for _ in range(W):
            step_rows()
        ms_r = shard.max_over_ranks(_timed(torch, stream, step_rows, args.steps, barrier), dist, device="cuda")
        su = _stage_us(im, step_rows, max(3, min(args.steps, 10)))
        r_in = B * (8.0 + 4.0) * nvis + B * 12.0 * nrow + 8.0 * nchan
        rows = {"entry": "muser_grid_rows, MUSER_POLS_SUM, grid = frame", "value": shard.aggregate_rate(args.steps * B * nvis, world, ms_r),
                "unit": UNIT, "ms_per_step": ms_r / args.steps, "bytes_per_vis": r_in / (B * nvis),
                "stage_us_per_frame": {k: (v / B if v else None) for k, v in su.items()},
                "roofline_frac_a1_a2": (r_in + grid_bytes) / ((su["bin"] + su["grid"]) * 1e-6) / 1e9 / peak,
                "images_per_s": args.steps * B * world / (ms_r * 1e-3)}
        del r_uvw, r_vis, r_wt

    # ---- ONE frame at a time through the un-batched calls (reset -> grid -> dirty_psf on one grid): stream-launched, and
    # the same sequence replayed as a CUDA graph (the calls only enqueue, so they capture)
    im1 = new_imager(1)
    nf1 = min(16, B)
    dev1 = [[torch.from_numpy(a).cuda() for a in fr] for fr in frames[:nf1]]
    d1 = torch.empty((n, n), device="cuda")
    p1 = torch.empty((n, n), device="cuda")

    def one(fr):
        im1.reset(); im1.grid(*fr); im1.dirty_psf(d1, p1)

    for fr in dev1[:4]:
        one(fr)
    single_ms = _timed(torch, stream, lambda: [one(fr) for fr in dev1], 1, barrier)
    single_us = 1e3 * single_ms / nf1
    graph_us = None
    try:
        side = torch.cuda.Stream()
        with torch.cuda.stream(side):
            one(dev1[0])
        side.synchronize()
        graphs = []
        for fr in dev1:
            gph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(gph, stream=side):
                one(fr)
            graphs.append(gph)
        for gph in graphs[:4]:
            gph.replay()
        graph_ms = _timed(torch, stream, lambda: [gph.replay() for gph in graphs], 4, barrier)
        graph_us = 1e3 * graph_ms / (4 * nf1)
        del graphs
    except Exception as ex:
        graph_us = {"unavailable": str(ex)[:120]}
    im1.destroy()
    del dev1

    # ---- end to end through the host-buffer entry point (pinned host memory; H2D + D2H inside the timed region): two
    # handles of B/2 grids on two streams, so that one half's copy back overlaps the other half's upload and imaging
    half = B // 2
    ims = [new_imager(half), new_imager(B - half)]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    cut = half * nvis
    pins, outs = [], []
    for k, (a, b) in enumerate(((0, cut), (cut, B * nvis))):
        gidk = (host[4][a:b] - (0 if k == 0 else half)).astype(np.int32)
        pins.append([torch.from_numpy(np.ascontiguousarray(x[a:b])).pin_memory() for x in host[:4]] + [torch.from_numpy(gidk).pin_memory()])
        ng = half if k == 0 else B - half
        outs.append((torch.empty((ng, n, n), dtype=torch.float32).pin_memory(), torch.empty((ng, n, n), dtype=torch.float32).pin_memory()))

    def e2e_step():
        for k in range(2):
            ims[k].frame_host_async(*pins[k], outs[k][0], outs[k][1], stream=streams[k].cuda_stream)

    def e2e_wait():
        for s_ in streams:
            s_.synchronize()

    for _ in range(2):
        e2e_step(); e2e_wait()
    e2e_steps = max(2, min(args.steps, 5))
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    e2e_wait()
    e2e_ms = shard.max_over_ranks(1e3 * (time.perf_counter() - t0), dist, device="cuda")
    e2e_value = e2e_steps * B * world * nvis / (e2e_ms * 1e-3)
    h2d = sum(int(a.nbytes) for a in host)
    d2h = 2 * B * n * n * 4
    # the same with beam_out = NULL: every frame of a step shares its uvw and weights, so its 80 beams are identical and a
    # monitoring caller fetches the beam once per geometry: dirty images only come back
    def e2e_step_dirty():
        for k in range(2):
            ims[k].frame_host_async(*pins[k], outs[k][0], None, stream=streams[k].cuda_stream)

    e2e_step_dirty(); e2e_wait()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step_dirty()
    e2e_wait()
    e2e_dirty_ms = shard.max_over_ranks(1e3 * (time.perf_counter() - t0), dist, device="cuda")
    e2e_dirty_value = e2e_steps * B * world * nvis / (e2e_dirty_ms * 1e-3)
    for x in ims:
        x.destroy()

    cpu = None
    if rank == 0 and not args.no_cpu_baseline:
        cpu = cpu_baseline(params, frames, nvis)
        if cfg in (1, 3):
            cpu["direct_dft_cfg1"] = cpu_direct_dft_cfg1()
    limits = binding.microbench() if rank == 0 else None
    line = None
    if rank == 0:
        frames_total = args.steps * B * world
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": W,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": WORKLOADS[cfg], "entry": "muser_grid_batched (flat, 32 B per visibility)",
                       "batching": f"one step = {B} distinct frames, each onto its own grid, in one muser_grid_batched + "
                                   "muser_dirty_psf call", "frames_per_step": B, "nvis_per_frame": nvis,
                       "l2_policy": f"per step {h2d / 1e6:.0f} MB of inputs and {12e-6 * B * n * n:.0f} MB of grids stream through a 126 MB L2",
                       "launch": "stream", "parallelism": f"frames x{world}" if world > 1 else "single"},
            "images_per_s": frames_total / (ms * 1e-3), "dirty_and_beam_pairs_per_s": frames_total / (ms * 1e-3),
            "us_per_frame": 1e3 * ms / (args.steps * B),
            "single_frame": {"stream_launched_us": single_us, "cuda_graph_replayed_us": graph_us,
                             "note": "reset -> grid -> dirty_psf of ONE frame on one grid, frames one after another"},
            "single_frame_latency_us": single_us,
            "rows": rows,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps_timed": e2e_steps, "us_per_frame": 1e3 * e2e_ms / (e2e_steps * B),
                    "how": "muser_frame_host_async, two handles of B/2 grids on two streams, pinned host buffers, wall clock "
                           "around the stream synchronisations",
                    "dirty_only": {"value": e2e_dirty_value, "unit": UNIT, "d2h_bytes_per_step": d2h // 2,
                                   "us_per_frame": 1e3 * e2e_dirty_ms / (e2e_steps * B),
                                   "note": "beam_out = NULL (the beam depends on uvw and weights only: fetched once per geometry)"}},
            "gpu_launches": int(launches), "clocks": sampler.result(), "roofline": roofline, "cpu_baseline": cpu,
            "device_limits": limits,
        }
    im.destroy()
    return line


def bench_cfg4(args, torch, binding, shard, dist, rank, world, local):
    """cfg 4: a chunk of 64 frames = 2048 independent 512^2 grids of 1770 visibilities (the full config is 500 such chunks)."""
    from inputs import synth
    W = max(args.warmup, 3)
    fr = synth.make_frame(4, nframes=64)
    p = fr.params
    n, nvis, ng = p.n, fr.nvis, p.ngrids
    dev = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (fr.uvw_m, fr.freq_hz, fr.vis, fr.weight, fr.grid_id)]
    im = binding.Imager(n, n, p.cell_arcsec, p.support, p.oversample)
    im.set_batch(ng)
    dirty = torch.empty((ng, n, n), device="cuda")
    psf = torch.empty((ng, n, n), device="cuda")
    stream = torch.cuda.current_stream()

    def step():
        im.reset(); im.grid_batched(*dev); im.dirty_psf(dirty, psf)

    def barrier():
        torch.cuda.synchronize()
        if dist:
            dist.barrier(); torch.cuda.synchronize()

    for _ in range(W):
        step()
    sampler = ClockSampler(local); sampler.sample(); sampler.start()
    l0 = im.get_launch_count()
    ms = shard.max_over_ranks(_timed(torch, stream, step, args.steps, barrier), dist, device="cuda")
    sampler.stop_flag = True; sampler.join(); sampler.sample()
    launches = im.get_launch_count() - l0
    su = _stage_us(im, step, 3)
    # the channelised call: 64 frames x 2 pol x 16 chan, one grid per (frame, pol, chan)
    nchan, npol, nt = 16, 2, 64
    nrow = nvis // (nt * nchan * npol)
    r_uvw = torch.from_numpy(np.ascontiguousarray(fr.uvw_m.reshape(nt, npol, nchan, nrow, 3)[:, 0, 0])).cuda()
    r_freq = torch.from_numpy(fr.freq_hz.reshape(nt, npol, nchan, nrow)[0, 0, :, 0].copy()).cuda()
    r_vis = torch.from_numpy(np.ascontiguousarray(fr.vis.reshape(nt, npol, nchan, nrow))).cuda()
    r_wt = torch.from_numpy(np.ascontiguousarray(fr.weight.reshape(nt, npol, nchan, nrow))).cuda()
    r_gid = torch.from_numpy(np.ascontiguousarray(fr.grid_id.reshape(nt, npol, nchan, nrow)[..., 0])).cuda()

    def step_rows():
        im.reset(); im.grid_rows(r_uvw, r_freq, r_vis, r_wt, r_gid, binding.MUSER_POLS_SPLIT); im.dirty_psf(dirty, psf)

    for _ in range(W):
        step_rows()
    ms_r = _timed(torch, stream, step_rows, args.steps, barrier)
    su_r = _stage_us(im, step_rows, 3)
    peak, peak_src = _peaks()
    alg = 32.0 * nvis + 12.0 * ng * n * n
    line = None
    if rank == 0:
        line = {"metric": METRIC, "value": shard.aggregate_rate(args.steps * nvis, world, ms), "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": W, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": WORKLOADS[4], "entry": "muser_grid_batched", "grids_per_step": ng, "nvis_per_step": nvis,
                           "l2_policy": "6.4 GB of grids per step stream through a 126 MB L2", "launch": "stream"},
                "images_per_s": args.steps * ng * world / (ms * 1e-3), "gpu_launches": int(launches), "clocks": sampler.result(),
                "rows": {"entry": "muser_grid_rows, MUSER_POLS_SPLIT", "value": args.steps * nvis / (ms_r * 1e-3),
                         "ms_per_step": ms_r / args.steps, "stage_us_per_step": su_r,
                         "images_per_s": args.steps * ng / (ms_r * 1e-3)},
                "roofline": {"bound": "hbm", "kernel": "A1 + A2 (binning + k_grid_owner_s7)", "achieved": alg / ((su["bin"] + su["grid"]) * 1e-6) / 1e9,
                             "peak": peak, "unit": "GB/s", "frac": alg / ((su["bin"] + su["grid"]) * 1e-6) / 1e9 / peak, "traffic": None,
                             "peak_source": peak_src, "algorithmic_bytes_per_launch": alg, "stage_us_per_launch": su},
                "e2e": None, "cpu_baseline": None}
    im.destroy()
    return line


def bench_cfg5(args, torch, binding, shard, dist, rank, world, local):
    """cfg 5: the whole configuration per step, 17 M visibilities onto one 4096^2 grid through 32 w-planes."""
    from inputs import synth
    W = max(args.warmup, 3)
    fr = synth.make_frame(5)
    p = fr.params
    n, nvis, P = p.n, fr.nvis, p.nplanes
    # plane layout of reading R15 (plain numpy; bench accounting, not the method): centres linear in |w|, supports 7..31
    w_max = 19900.0
    fov = n * p.cell_arcsec * np.pi / 648000.0
    wc = np.arange(P) * (w_max / (P - 1))
    sup = (7 + 2 * np.floor(wc * fov * fov / 4.0 + 0.5)).astype(np.int32)
    wl = np.abs(fr.uvw_m[:, 2].astype(np.float64) * fr.freq_hz / 299792458.0)
    plane = np.clip(np.floor(wl / (w_max / (P - 1)) + 0.5).astype(np.int64), 0, P - 1)      # nearest centre of a linear ladder
    hist = np.bincount(plane, minlength=P)
    flop = 8.0 * float((2.0 * hist * sup.astype(np.float64) ** 2).sum())                    # 8 S_p^2 per gridded sample, 2 samples per visibility
    dev = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (fr.uvw_m, fr.freq_hz, fr.vis, fr.weight)]
    im = binding.Imager(n, n, p.cell_arcsec, 7, p.oversample)
    im.set_wplanes(wc, sup, None)
    dirty = torch.empty((1, n, n), device="cuda")
    psf = torch.empty((1, n, n), device="cuda")
    stream = torch.cuda.current_stream()

    def step():
        im.reset(); im.grid(*dev); im.dirty_psf(dirty, psf)

    def barrier():
        torch.cuda.synchronize()

    for _ in range(W):
        step()
    sampler = ClockSampler(local); sampler.sample(); sampler.start()
    l0 = im.get_launch_count()
    ms = _timed(torch, stream, step, args.steps, barrier)
    sampler.stop_flag = True; sampler.join(); sampler.sample()
    launches = im.get_launch_count() - l0
    su = _stage_us(im, step, 3)
    # ---- the channelised entry point on the same data: 300 snapshots x 2 polarisations x 16 channels x 1770 baselines,
    # polarisations summed before gridding (half as many records)
    nchan, npol, nrow = 16, 2, 1770
    ntime = nvis // (nchan * npol * nrow)
    r_uvw = torch.from_numpy(np.ascontiguousarray(fr.uvw_m.reshape(ntime, npol, nchan, nrow, 3)[:, 0, 0])).cuda()
    r_freq = torch.from_numpy(fr.freq_hz.reshape(ntime, npol, nchan, nrow)[0, 0, :, 0].copy()).cuda()
    r_vis, r_wt = dev[2].view(ntime, npol, nchan, nrow), dev[3].view(ntime, npol, nchan, nrow)

    def step_rows():
        im.reset(); im.grid_rows(r_uvw, r_freq, r_vis, r_wt, None, binding.MUSER_POLS_SUM); im.dirty_psf(dirty, psf)

    for _ in range(W):
        step_rows()
    ms_r = _timed(torch, stream, step_rows, args.steps, barrier)
    su_r = _stage_us(im, step_rows, 3)
    rows = {"entry": "muser_grid_rows, MUSER_POLS_SUM (k_coords<ROWS> + k_wgrid)", "value": args.steps * nvis / (ms_r * 1e-3), "unit": UNIT,
            "ms_per_step": ms_r / args.steps, "stage_us_per_launch": su_r, "images_per_s": args.steps / (ms_r * 1e-3)}
    limits = binding.microbench()
    fpeak = limits["fp32_fma_flops"]
    line = {"metric": METRIC, "value": args.steps * nvis / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": W,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic", "rows": rows,
            "config": {"workload": WORKLOADS[5], "entry": "muser_grid (w-planes: MUSER_STRATEGY_WPLANE, window gridder k_wgrid<shape>)", "nvis_per_step": nvis,
                       "l2_policy": "544 MB of inputs per step stream through a 126 MB L2", "launch": "stream",
                       "plane_histogram_visibilities": hist.tolist(), "plane_supports": sup.tolist(),
                       "gridding_flop_8_sum_Np_Sp2": flop},
            "images_per_s": args.steps / (ms * 1e-3), "gpu_launches": int(launches), "clocks": sampler.result(),
            "roofline": {"bound": "alu", "kernel": "k_wgrid<0..7> (A3: one kernel per window shape, overlapped on side streams; flop = 8 S_p^2 per sample of the full plane, the stored half-plane needs half of them)", "achieved": flop / (su["grid"] * 1e-6) / 1e12,
                         "peak": fpeak / 1e12, "unit": "TFLOP/s", "frac": flop / (su["grid"] * 1e-6) / fpeak, "traffic": None,
                         "peak_source": "measured in this run (muser_microbench fp32_fma_flops)", "stage_us_per_launch": su},
            "e2e": None, "cpu_baseline": None, "device_limits": limits}
    im.destroy()
    return line


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="muser")
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5])
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
    if args.config in (1, 2, 3):
        line = bench_frames(args, args.config, torch, binding, shard, dist, rank, world, local)
    elif args.config == 4:
        line = bench_cfg4(args, torch, binding, shard, dist, rank, world, local)
    else:
        line = bench_cfg5(args, torch, binding, shard, dist, rank, world, local)
    if rank == 0 and line is not None:
        print(json.dumps(line))
    if dist:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
