"""-m gpu parity at BASELINE.json's FULL sizes, in the launch configurations that are actually used:

  * cfg 3 as bench.py times it: 80 distinct MUSER-II frames, one muser_grid_batched + muser_dirty_psf call (owner-tile
    gridder: the first call after a reset stores the non-empty tiles of the half-plane and flags them); three of the 80 grids are compared cell by cell and pixel by
    pixel with the oracle, the counters over all of them.
  * cfg 3 through the channelised entry (muser_grid_rows, MUSER_POLS_SUM) and through the host-buffer entry on two handles /
    two streams, exactly as bench.py's `rows` and `e2e` legs run them, against the oracle.
  * cfg 4: a 64-frame chunk = 2048 independent 512x512 grids of 1770 visibilities (the full config is 500 such chunks;
    one chunk is what fits comfortably beside its images); sampled grids against the oracle, counters over all.
  * cfg 5 in full: 16,992,000 visibilities, 300 snapshots, 32 w-planes with supports 7..31, one 4096x4096 grid, against
    the plain-C oracle run on everything (about 90 s of CPU).
"""
import numpy as np
import pytest

from oracle import muser_oracle as mo
from oracle import oracle_c as oc
from paper_1712_06913_b200 import binding
from inputs import synth

import gpu_util as gu

pytestmark = pytest.mark.gpu


def _images_of(im, gi_list, G_or, Gw_or, T, S, Q):
    """R9 gates on selected grids of a batched imager (dirty + beam, corrected and un-corrected)."""
    import torch
    ng, ny, nx = im.ngrids, im.ny, im.nx
    d = torch.empty((ng, ny, nx), dtype=torch.float32, device="cuda")
    p = torch.empty((ng, ny, nx), dtype=torch.float32, device="cuda")
    out = {}
    for corr in (False, True):
        im.set_grid_correction(corr)
        im.dirty_psf(d, p)
        torch.cuda.synchronize()
        out[corr] = (d[gi_list].cpu().numpy().astype(np.float64), p[gi_list].cpu().numpy().astype(np.float64))
    im.set_grid_correction(True)
    cx, cy = mo.corrector(T, S, Q, nx), mo.corrector(T, S, Q, ny)
    box = gu.inner_box(ny, cy)[:, None] & gu.inner_box(nx, cx)[None, :]
    for k in range(len(gi_list)):
        raw_d, cor_d, raw_p, cor_p, _ = gu.oracle_images(G_or[k][None], Gw_or[k][None], T, S, Q)
        for name, o_raw, o_cor, g_raw, g_cor in (("dirty", raw_d[0], cor_d[0], out[False][0][k], out[True][0][k]),
                                                 ("beam", raw_p[0], cor_p[0], out[False][1][k], out[True][1][k])):
            e_raw = np.abs(g_raw - o_raw).max() / np.abs(o_raw).max()
            e_box = np.abs(g_cor - o_cor)[box].max() / np.abs(o_cor[box]).max()
            assert e_raw <= gu.IMG_TOL, f"{name} grid {gi_list[k]}: un-corrected error {e_raw:.2e} of peak"
            assert e_box <= gu.IMG_TOL, f"{name} grid {gi_list[k]}: corrected inner-75% error {e_box:.2e} of peak"


def test_cfg3_batch_of_80_frames_as_benched():
    import torch
    import bench
    params, frames = bench.make_frames(bench.FRAMES_PER_STEP[3])
    B, n, nvis = len(frames), params.n, frames[0][2].shape[0]
    host = [np.ascontiguousarray(np.concatenate([fr[i] for fr in frames])) for i in range(4)]
    gid = np.repeat(np.arange(B, dtype=np.int32), nvis)
    im = binding.Imager(n, n, params.cell_arcsec, params.support, params.oversample)
    try:
        im.set_batch(B)
        dev = [gu.to_dev(a) for a in host] + [gu.to_dev(gid)]
        for _ in range(2):                                   # the second pass re-uses every scratch buffer
            im.reset()
            im.grid_batched(*dev)
        st = im.get_stats()
        T = mo.table_pswf(params.support, params.oversample)
        pick = [0, 37, B - 1]
        G = torch.empty((B, n, n, 2), dtype=torch.float32, device="cuda")
        Gw = torch.empty((B, n, n), dtype=torch.float32, device="cuda")
        im.get_grid(G, Gw)
        torch.cuda.synchronize()
        G_or, Gw_or, n_gridded, sum_w = [], [], 0, 0.0
        for b in range(B):
            if b in pick:
                g_or, w_or, s_or = oc.grid(*frames[b], n, n, params.cell_arcsec, params.oversample, params.support, T)
                G_or.append(g_or[0]); Gw_or.append(w_or[0])
                g = G[b].cpu().numpy().astype(np.float64)
                eg = gu.rel_l2(g[..., 0] + 1j * g[..., 1], g_or[0])
                ew = gu.rel_l2(Gw[b].cpu().numpy().astype(np.float64), w_or[0])
                assert eg <= gu.GRID_TOL and ew <= gu.GRID_TOL, f"grid {b}: rel-L2 {eg:.2e} / {ew:.2e}"
                per_frame = s_or
        # every frame shares the geometry, so the counters of one frame times 80 are the batch's
        assert st["n_gridded"] == per_frame["n_gridded"] * B and st["n_dropped"] == per_frame["n_dropped"] * B
        assert abs(st["sum_weights"] - per_frame["sum_weights"] * B) <= 1e-9 * per_frame["sum_weights"] * B
        _images_of(im, pick, G_or, Gw_or, T, params.support, params.oversample)
    finally:
        im.destroy()


def _oracle_images_of_frame(fr, params, T):
    """(dirty un-corrected, dirty corrected, beam un-corrected, beam corrected, box) of one frame by the oracle."""
    n = params.n
    g_or, w_or, s_or = oc.grid(*fr, n, n, params.cell_arcsec, params.oversample, params.support, T)
    raw_d, cor_d, raw_p, cor_p, _ = gu.oracle_images(g_or, w_or, T, params.support, params.oversample)
    c = mo.corrector(T, params.support, params.oversample, n)
    box = gu.inner_box(n, c)[:, None] & gu.inner_box(n, c)[None, :]
    return g_or[0], w_or[0], cor_d[0], cor_p[0], box, s_or


def test_cfg3_rows_entry_80_frames_as_benched():
    """The bench's `rows` leg at full size: 80 cfg-3 frames in the instrument's layout [time][pol][chan][baseline] through
    muser_grid_rows with MUSER_POLS_SUM and one grid per frame (grid id per [time][chan]); sampled grids and images against
    the oracle run on the FLAT frame (the channelised call must give the flat call's result), counters over everything."""
    import torch
    import bench
    params, frames = bench.make_frames(bench.FRAMES_PER_STEP[3])
    B, n, nvis = len(frames), params.n, frames[0][2].shape[0]
    nchan, npol = 16, 2
    nrow = nvis // (nchan * npol)
    r_uvw = torch.from_numpy(np.stack([fr[0].reshape(npol, nchan, nrow, 3)[0, 0] for fr in frames])).cuda()
    r_freq = torch.from_numpy(frames[0][1].reshape(npol, nchan, nrow)[0, :, 0].copy()).cuda()
    r_vis = torch.from_numpy(np.stack([fr[2].reshape(npol, nchan, nrow) for fr in frames])).cuda()
    r_wt = torch.from_numpy(np.stack([fr[3].reshape(npol, nchan, nrow) for fr in frames])).cuda()
    r_gid = torch.from_numpy(np.repeat(np.arange(B, dtype=np.int32)[:, None], nchan, 1).copy()).cuda()
    # the flat frames really are the broadcast of these arrays (else the comparison below would be of different inputs)
    f0 = frames[3]
    assert np.array_equal(np.broadcast_to(f0[0].reshape(npol, nchan, nrow, 3)[0, 0], (npol, nchan, nrow, 3)).reshape(-1, 3), f0[0])
    assert np.array_equal(np.broadcast_to(frames[0][1].reshape(npol, nchan, nrow)[0, :, :1], (npol, nchan, nrow)).reshape(-1), f0[1])
    im = binding.Imager(n, n, params.cell_arcsec, params.support, params.oversample)
    try:
        im.set_batch(B)
        for _ in range(2):
            im.reset()
            im.grid_rows(r_uvw, r_freq, r_vis, r_wt, r_gid, binding.MUSER_POLS_SUM)
        st = im.get_stats()
        T = mo.table_pswf(params.support, params.oversample)
        pick = [1, 40, B - 1]
        G = torch.empty((B, n, n, 2), dtype=torch.float32, device="cuda")
        Gw = torch.empty((B, n, n), dtype=torch.float32, device="cuda")
        im.get_grid(G, Gw)
        torch.cuda.synchronize()
        G_or, Gw_or = [], []
        for b in pick:
            g_or, w_or, s_or = oc.grid(*frames[b], n, n, params.cell_arcsec, params.oversample, params.support, T)
            G_or.append(g_or[0]); Gw_or.append(w_or[0])
            g = G[b].cpu().numpy().astype(np.float64)
            eg = gu.rel_l2(g[..., 0] + 1j * g[..., 1], g_or[0])
            ew = gu.rel_l2(Gw[b].cpu().numpy().astype(np.float64), w_or[0])
            assert eg <= gu.GRID_TOL and ew <= gu.GRID_TOL, f"grid {b}: rel-L2 {eg:.2e} / {ew:.2e}"
        assert st["n_gridded"] == s_or["n_gridded"] * B and st["n_dropped"] == s_or["n_dropped"] * B and st["n_flagged"] == 0
        assert abs(st["sum_weights"] - s_or["sum_weights"] * B) <= 1e-9 * s_or["sum_weights"] * B
        _images_of(im, pick, G_or, Gw_or, T, params.support, params.oversample)
    finally:
        im.destroy()


def test_cfg3_end_to_end_leg_as_benched_against_the_oracle():
    """The bench's `e2e` leg: two handles of 40 grids on two streams, pinned host buffers, muser_frame_host_async twice in a
    row (the second call re-uses the staging buffers and only enqueues); sampled dirty images and beams of both halves
    against the ORACLE's (corrected, inner 75 % box, 1e-4 of the peak)."""
    import torch
    import bench
    params, frames = bench.make_frames(bench.FRAMES_PER_STEP[3])
    B, n, nvis = len(frames), params.n, frames[0][2].shape[0]
    host = [np.ascontiguousarray(np.concatenate([fr[i] for fr in frames])) for i in range(4)]
    gid = np.repeat(np.arange(B, dtype=np.int32), nvis)
    half = B // 2
    ims, streams, pins, outs = [], [torch.cuda.Stream(), torch.cuda.Stream()], [], []
    try:
        for k, (a, b) in enumerate(((0, half * nvis), (half * nvis, B * nvis))):
            im = binding.Imager(n, n, params.cell_arcsec, params.support, params.oversample)
            ims.append(im)
            im.set_batch(half)
            gk = (gid[a:b] - k * half).astype(np.int32)
            pins.append([torch.from_numpy(np.ascontiguousarray(x[a:b])).pin_memory() for x in host] + [torch.from_numpy(gk).pin_memory()])
            outs.append((torch.zeros((half, n, n), dtype=torch.float32).pin_memory(), torch.zeros((half, n, n), dtype=torch.float32).pin_memory()))
        for _ in range(2):
            for k in range(2):
                ims[k].frame_host_async(*pins[k], outs[k][0], outs[k][1], stream=streams[k].cuda_stream)
        for s_ in streams:
            s_.synchronize()
        T = mo.table_pswf(params.support, params.oversample)
        for b in (0, half - 1, half, B - 1):
            _, _, cor_d, cor_p, box, _ = _oracle_images_of_frame(frames[b], params, T)
            k, j = divmod(b, half)
            for name, got, want in (("dirty", outs[k][0][j].numpy().astype(np.float64), cor_d),
                                    ("beam", outs[k][1][j].numpy().astype(np.float64), cor_p)):
                e = np.abs(got - want)[box].max() / np.abs(want[box]).max()
                assert e <= gu.IMG_TOL, f"{name} of frame {b}: {e:.2e} of the peak"
    finally:
        for im in ims:
            im.destroy()


def test_cfg4_chunk_of_2048_grids():
    import torch
    fr = synth.make_frame(4, nframes=64)
    p = fr.params
    assert p.ngrids == 2048 and fr.nvis == 64 * 56640
    im = binding.Imager(p.n, p.n, p.cell_arcsec, p.support, p.oversample)
    try:
        im.set_batch(p.ngrids)
        im.reset()
        im.grid_batched(gu.to_dev(fr.uvw_m), gu.to_dev(fr.freq_hz), gu.to_dev(fr.vis), gu.to_dev(fr.weight),
                        gu.to_dev(fr.grid_id))
        st = im.get_stats()
        T = mo.table_pswf(p.support, p.oversample)
        # counters: keep/drop does not depend on the grid id, so the oracle runs once over everything on one grid
        _, _, s_all = oc.grid(fr.uvw_m, fr.freq_hz, fr.vis, fr.weight, p.n, p.n, p.cell_arcsec, p.oversample, p.support, T)
        assert st["n_gridded"] == s_all["n_gridded"] and st["n_dropped"] == s_all["n_dropped"]
        assert s_all["n_dropped"] > 0                          # cfg 4's longest baselines leave the 512^2 grid (R5)
        pick = [0, 1, 31, 32, 777, 1024, 2046, 2047]
        G = torch.empty((p.ngrids, p.n, p.n, 2), dtype=torch.float32, device="cuda")
        Gw = torch.empty((p.ngrids, p.n, p.n), dtype=torch.float32, device="cuda")
        im.get_grid(G, Gw)
        torch.cuda.synchronize()
        G_or, Gw_or = [], []
        for b in pick:
            sel = fr.grid_id == b
            g_or, w_or, _ = oc.grid(fr.uvw_m[sel], fr.freq_hz[sel], fr.vis[sel], fr.weight[sel], p.n, p.n, p.cell_arcsec,
                                    p.oversample, p.support, T)
            G_or.append(g_or[0]); Gw_or.append(w_or[0])
            g = G[b].cpu().numpy().astype(np.float64)
            eg = gu.rel_l2(g[..., 0] + 1j * g[..., 1], g_or[0])
            ew = gu.rel_l2(Gw[b].cpu().numpy().astype(np.float64), w_or[0])
            assert eg <= gu.GRID_TOL and ew <= gu.GRID_TOL, f"grid {b}: rel-L2 {eg:.2e} / {ew:.2e}"
        del G, Gw
        _images_of(im, pick, G_or, Gw_or, T, p.support, p.oversample)
    finally:
        im.destroy()


def test_cfg5_full_wprojection_17M_visibilities():
    fr = synth.make_frame(5)
    p = fr.params
    assert fr.nvis == 16_992_000 and p.n == 4096 and p.nplanes == 32
    wc, sup = mo.wplane_layout(p.n, p.cell_arcsec, p.nplanes, 19900.0)
    assert sup.min() == 7 and sup.max() == 31
    fov = p.n * p.cell_arcsec * mo.ARCSEC
    tabs = [mo.table_wkernel(int(S), p.oversample, float(w), fov) for S, w in zip(sup, wc)]
    im = binding.Imager(p.n, p.n, p.cell_arcsec, 7, p.oversample)
    try:
        im.set_wplanes(wc, sup, [t.astype(np.complex64) for t in tabs])
        im.reset()
        im.grid(gu.to_dev(fr.uvw_m), gu.to_dev(fr.freq_hz), gu.to_dev(fr.vis), gu.to_dev(fr.weight))
        st = im.get_stats()
        G, Gw = gu.gpu_grids(im)
        G_or, Gw_or, st_or = oc.grid(fr.uvw_m, fr.freq_hz, fr.vis, fr.weight, p.n, p.n, p.cell_arcsec, p.oversample,
                                     sup, tabs, wc=wc)
        assert st["n_gridded"] == st_or["n_gridded"] and st["n_dropped"] == st_or["n_dropped"]
        assert abs(st["sum_weights"] - st_or["sum_weights"]) <= 1e-9 * st_or["sum_weights"]
        eg, ew = gu.rel_l2(G, G_or), gu.rel_l2(Gw, Gw_or)
        assert eg <= gu.GRID_TOL and ew <= gu.GRID_TOL, f"rel-L2 {eg:.2e} / {ew:.2e}"
        gu.check_images(im, G_or, Gw_or, tabs[0].real, 7, p.oversample)
    finally:
        im.destroy()
