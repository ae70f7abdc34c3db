"""-m gpu parity tests of SURVEY.md 8(f)'s NEXT rows against the oracle: phase correction fused into A1 (NEXT-3), uniform
weighting as the paper prints it + the 2x beam (NEXT-2), peak search and histogram fused into / after A6 and Table 2's
non-power-of-two image sizes (NEXT-4).  Integer results (hit counts, peak position, histogram) must be equal; grids
rel-L2 <= 1e-5; images <= 1e-4 of the peak (gates of DESIGN.md R9)."""
import numpy as np
import pytest

from oracle import muser_oracle as mo
from oracle import oracle_c as oc
from paper_1712_06913_b200 import binding
from inputs import synth

import gpu_util as gu

pytestmark = pytest.mark.gpu

TILED, OWNER = binding.MUSER_STRATEGY_TILED, binding.MUSER_STRATEGY_OWNER


def _bright(vis):
    return (vis * 0.05 + 1.0).astype(np.complex64)          # a point-like component keeps the image peak above the noise


@pytest.mark.parametrize("strategy", [OWNER, TILED])
def test_phase_offset_is_applied_before_gridding(strategy):
    fr = synth.make_frame(2)
    p = fr.params
    off = (2.4e-4, -1.1e-4)                                  # ~50", ~23": inside the field
    im = gu.make_imager(p.n, p.cell_arcsec, p.support, p.oversample, strategy=strategy)
    try:
        im.set_phase_offset(*off)
        im.reset()
        im.grid(gu.to_dev(fr.uvw_m), gu.to_dev(fr.freq_hz), gu.to_dev(fr.vis), gu.to_dev(fr.weight))
        G, Gw = gu.gpu_grids(im)
        T = mo.table_pswf(p.support, p.oversample)
        G_or, Gw_or, st = oc.grid(fr.uvw_m, fr.freq_hz, fr.vis, fr.weight, p.n, p.n, p.cell_arcsec, p.oversample, p.support, T,
                                  offset=off)
        assert im.get_stats()["n_gridded"] == st["n_gridded"]
        assert gu.rel_l2(G, G_or) <= gu.GRID_TOL and gu.rel_l2(Gw, Gw_or) <= gu.GRID_TOL
        G0, _, _ = oc.grid(fr.uvw_m, fr.freq_hz, fr.vis, fr.weight, p.n, p.n, p.cell_arcsec, p.oversample, p.support, T)
        assert gu.rel_l2(G, G0) > 1e-2                       # and it is not a no-op
        gu.check_images(im, G_or, Gw_or, T, p.support, p.oversample)
        im.set_phase_offset(0.0, 0.0)                        # switching it off again
        im.reset()
        im.grid(gu.to_dev(fr.uvw_m), gu.to_dev(fr.freq_hz), gu.to_dev(fr.vis), gu.to_dev(fr.weight))
        G, _ = gu.gpu_grids(im)
        assert gu.rel_l2(G, G0) <= gu.GRID_TOL
    finally:
        im.destroy()


def test_phase_offset_centres_an_off_centre_source():
    """P7 backwards on the GPU: a unit source at pixel (x0, y0), corrected by its own offset, peaks at the phase centre."""
    n, cell, Q = 256, 20.0, 32
    uvw, freq, _, wt = synth.random_visibilities(17, 4000, n, cell, margin_cells=6.0)
    x0, y0 = 170, 101
    l0, m0 = (x0 - n / 2) * cell * mo.ARCSEC, (y0 - n / 2) * cell * mo.ARCSEC
    il = freq / mo.C_M_S
    u, v = uvw[:, 0].astype(np.float64) * il, uvw[:, 1].astype(np.float64) * il
    vis = np.exp(-2j * np.pi * (u * l0 + v * m0)).astype(np.complex64)
    im = gu.make_imager(n, cell, 7, Q)
    try:
        im.set_peak_search(True)
        for off, want in (((0.0, 0.0), (x0, y0)), ((l0, m0), (n // 2, n // 2))):
            im.set_phase_offset(*off)
            im.reset()
            im.grid(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt))
            d, _ = gu.gpu_images(im)
            val, x, y, _ = im.get_peak()[0]
            assert (x, y) == want
            assert abs(val / im.get_stats()["sum_weights"] - 1) < 5e-3
    finally:
        im.destroy()


@pytest.mark.parametrize("strategy", [OWNER, TILED])
@pytest.mark.parametrize("ngrids", [1, 3])
def test_uniform_weighting_counts_grids_and_images(strategy, ngrids):
    import torch
    fr = synth.make_frame(2)
    p = fr.params
    gid = (np.arange(fr.nvis) % ngrids).astype(np.int32)
    im = gu.make_imager(p.n, p.cell_arcsec, p.support, p.oversample, ngrids=ngrids, strategy=strategy)
    try:
        im.set_weighting(binding.MUSER_WEIGHT_UNIFORM)
        d = [gu.to_dev(a) for a in (fr.uvw_m, fr.freq_hz, _bright(fr.vis), fr.weight, gid)]
        h = fr.nvis // 2
        im.reset()
        im.grid_batched(*[a[:h] for a in d])                 # two accumulating calls: counts accumulate too
        im.grid_batched(*[a[h:] for a in d])
        T = mo.table_pswf(p.support, p.oversample)
        G_or, Gw_or, st = oc.grid(fr.uvw_m, fr.freq_hz, _bright(fr.vis), fr.weight, p.n, p.n, p.cell_arcsec, p.oversample,
                                  p.support, T, grid_id=gid, ngrids=ngrids, counts=True)
        cnt = torch.empty((ngrids, p.n, p.n), dtype=torch.int32, device="cuda")
        im.get_counts(cnt)
        Gu = torch.empty((ngrids, p.n, p.n, 2), device="cuda"); Gwu = torch.empty((ngrids, p.n, p.n), device="cuda")
        im.get_weighted_grid(Gu, Gwu)
        torch.cuda.synchronize()
        assert np.array_equal(cnt.cpu().numpy().astype(np.int64), st["cnt"])          # integers: exact
        assert st["cnt"].sum() == 2 * st["n_gridded"] and st["cnt"].max() > 1
        U_or, Uw_or = mo.wgt_grid(G_or, st["cnt"], 1), mo.wgt_grid(Gw_or, st["cnt"], 1)
        g = Gu.cpu().numpy().astype(np.float64)
        assert gu.rel_l2(g[..., 0] + 1j * g[..., 1], U_or) <= gu.GRID_TOL
        assert gu.rel_l2(Gwu.cpu().numpy().astype(np.float64), Uw_or) <= gu.GRID_TOL
        G, Gw = gu.gpu_grids(im)                             # the accumulated grids themselves are not modified
        assert gu.rel_l2(G, G_or) <= gu.GRID_TOL and gu.rel_l2(Gw, Gw_or) <= gu.GRID_TOL
        gu.check_images(im, U_or, Uw_or, T, p.support, p.oversample)
        im.reset()                                           # reset clears the counts
        im.get_counts(cnt)
        torch.cuda.synchronize()
        assert not cnt.any()
    finally:
        im.destroy()


def test_uniform_weighting_on_the_library_fft_path_and_natural_mode_identity():
    """96 x 160 takes cuFFT 2-D + k_pack (the weighting is applied in the pack kernel); natural mode: weighted == plain."""
    import torch
    n, ny, cell, Q = 96, 160, 40.0, 16
    uvw, freq, vis, wt = synth.random_visibilities(23, 3000, n, cell, margin_cells=6.0)
    uvw[:, :2] *= 0.3                                         # crowd the cells: counts well above 1
    vis = _bright(vis)
    im = gu.make_imager(n, cell, 7, Q, ny=ny)
    try:
        T = gu.oracle_table("pswf", 7, Q)
        im.reset()
        im.grid(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt))
        Gn = torch.empty((1, ny, n, 2), device="cuda"); Gp = torch.empty_like(Gn)
        im.get_weighted_grid(Gn, None); im.get_grid(Gp, None)
        torch.cuda.synchronize()
        assert torch.equal(Gn, Gp)
        im.set_weighting(binding.MUSER_WEIGHT_UNIFORM)
        im.reset()
        im.grid(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt))
        G_or, Gw_or, st = oc.grid(uvw, freq, vis, wt, n, ny, cell, Q, 7, T, counts=True)
        assert st["cnt"].max() >= 3
        gu.check_images(im, mo.wgt_grid(G_or, st["cnt"], 1), mo.wgt_grid(Gw_or, st["cnt"], 1), T, 7, Q)
    finally:
        im.destroy()


@pytest.mark.parametrize("strategy", [OWNER, TILED])
def test_beam_on_twice_the_field(strategy):
    import torch
    fr = synth.make_frame(1)
    p = fr.params
    im = gu.make_imager(p.n, p.cell_arcsec, p.support, p.oversample, kernel="gauss", strategy=strategy)
    try:
        im.set_psf2x(True)
        im.reset()
        im.grid(gu.to_dev(fr.uvw_m), gu.to_dev(fr.freq_hz), gu.to_dev(fr.vis), gu.to_dev(fr.weight))
        b2 = torch.empty((1, 2 * p.n, 2 * p.n), device="cuda")
        im.psf2x(b2)
        b1 = torch.empty((1, p.n, p.n), device="cuda")
        im.psf(b1)
        torch.cuda.synchronize()
        T = mo.table_gauss(p.support, p.oversample)
        n2 = 2 * p.n
        _, Gw2, st2 = oc.grid(fr.uvw_m, fr.freq_hz, fr.vis, fr.weight, n2, n2, p.cell_arcsec, p.oversample, p.support, T)
        assert st2["n_gridded"] == im.get_stats()["n_gridded"]  # same uv extent (half the uv cell, twice the cells): same drops
        raw, cor, *_ = gu.oracle_images(Gw2.astype(np.complex128), Gw2, T, p.support, p.oversample)
        c2 = mo.corrector(T, p.support, p.oversample, n2)
        box = gu.inner_box(n2, c2)[:, None] & gu.inner_box(n2, c2)[None, :]
        got = b2.cpu().numpy().astype(np.float64)[0]
        assert np.abs(got - cor[0])[box].max() <= gu.IMG_TOL * np.abs(cor[0][box]).max()
        # the 1x beam is still the ordinary one
        _, Gw1, _ = oc.grid(fr.uvw_m, fr.freq_hz, fr.vis, fr.weight, p.n, p.n, p.cell_arcsec, p.oversample, p.support, T)
        _, cor1, *_ = gu.oracle_images(Gw1.astype(np.complex128), Gw1, T, p.support, p.oversample)
        c1 = mo.corrector(T, p.support, p.oversample, p.n)
        box1 = gu.inner_box(p.n, c1)[:, None] & gu.inner_box(p.n, c1)[None, :]
        assert np.abs(b1.cpu().numpy()[0] - cor1[0])[box1].max() <= gu.IMG_TOL * np.abs(cor1[0][box1]).max()
    finally:
        im.destroy()


@pytest.mark.parametrize("nx,ny,ngrids", [(512, 512, 1), (256, 1024, 3), (96, 160, 2)])
def test_peak_search_and_histogram_equal_the_oracle_on_the_same_image(nx, ny, ngrids):
    """Fused column epilogue (first two) and cuFFT 2-D + k_correct (last).  The oracle is applied to the GPU's own fp32
    image: peak value, position and minimum must be equal, the histogram bin by bin."""
    import torch
    cell, Q = 30.0, 16
    n = min(nx, ny)
    nvis = 3000
    uvw, freq, vis, wt = synth.random_visibilities(61 + nx, nvis, n, cell * max(nx, ny) / n, margin_cells=6.0)
    gid = (np.arange(nvis) % ngrids).astype(np.int32)
    im = gu.make_imager(nx, cell, 7, Q, ngrids=ngrids, ny=ny)
    try:
        im.set_peak_search(True)
        im.reset()
        im.grid_batched(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(_bright(vis)), gu.to_dev(wt), gu.to_dev(gid))
        d = torch.empty((ngrids, ny, nx), device="cuda")
        im.dirty(d)
        hist = torch.empty((ngrids, 2000), dtype=torch.int32, device="cuda")
        im.histogram(d, 2000, 0.0, 0.0, hist)                 # lo >= hi: each image's own minimum and maximum
        hist2 = torch.empty((ngrids, 64), dtype=torch.int32, device="cuda")
        im.histogram(d, 64, -5.0, 40.0, hist2)
        torch.cuda.synchronize()
        peaks = im.get_peak()
        img = d.cpu().numpy()
        for g in range(ngrids):
            val, y, x, lo = mo.image_peak(img[g])
            assert peaks[g] == (np.float32(val), x, y, np.float32(lo))
            assert np.array_equal(hist[g].cpu().numpy().astype(np.int64), mo.image_histogram(img[g], 2000, lo, val))
            assert np.array_equal(hist2[g].cpu().numpy().astype(np.int64), mo.image_histogram(img[g], 64, -5.0, 40.0))
            assert int(hist[g].sum()) == nx * ny
    finally:
        im.destroy()


@pytest.mark.parametrize("n", [1280, 2560])
def test_table2_non_power_of_two_image_size(n):
    """PAPER.md:114-116 (Table 2): 1280^2 (2560^2 and 5120^2 take the same code path: cuFFT 2-D + k_correct)."""
    cell, Q = 8.0, 32
    uvw, freq, vis, wt = synth.random_visibilities(5, 20000, n, cell, margin_cells=6.0)
    vis = _bright(vis)
    im = gu.make_imager(n, cell, 7, Q)
    try:
        im.reset()
        im.grid(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt))
        T = gu.oracle_table("pswf", 7, Q)
        G_or, Gw_or, st = oc.grid(uvw, freq, vis, wt, n, n, cell, Q, 7, T)
        G, Gw = gu.gpu_grids(im)
        assert im.get_stats()["n_gridded"] == st["n_gridded"]
        assert gu.rel_l2(G, G_or) <= gu.GRID_TOL and gu.rel_l2(Gw, Gw_or) <= gu.GRID_TOL
        gu.check_images(im, G_or, Gw_or, T, 7, Q)
    finally:
        im.destroy()


def _rows_inputs(cfg, ntime, seed=0):
    """Channelised inputs with the shape of a MUSER frame: baselines of synth's array at `ntime` hour angles."""
    fr = synth.make_frame(cfg)
    p = fr.params
    nchan, npol = 16, 2
    nrow = fr.nvis // (nchan * npol)
    uvw1 = fr.uvw_m.reshape(npol, nchan, nrow, 3)[0, 0]
    freq = fr.freq_hz.reshape(npol, nchan, nrow)[0, :, 0].copy()
    rng = np.random.default_rng(100 + seed)
    uvw = np.stack([uvw1 * (1.0 - 0.01 * t) for t in range(ntime)]).astype(np.float32)
    vis = np.stack([fr.vis.reshape(npol, nchan, nrow)] * ntime).copy()
    vis += (0.05 * (rng.standard_normal(vis.shape) + 1j * rng.standard_normal(vis.shape))).astype(np.complex64)
    wt = rng.uniform(0.5, 1.5, vis.shape).astype(np.float32)
    return p, uvw, freq, vis.astype(np.complex64), wt


@pytest.mark.parametrize("strategy", [binding.MUSER_STRATEGY_AUTO, TILED])
@pytest.mark.parametrize("mode", ["sum_one_grid", "sum_per_time_channel", "split"])
def test_channelised_rows_call_equals_the_oracle_on_the_flattened_arrays(mode, strategy):
    import torch
    ntime = 2
    p, uvw, freq, vis, wt = _rows_inputs(2, ntime)
    _, npol, nchan, nrow = vis.shape
    # flags in single polarisations and an off-grid baseline: per-visibility counters
    wt[0, 1, 3, 5] = 0.0
    wt[1, 0, 7, 11] = np.nan
    vis[1, 1, 2, 9] = complex(np.inf, 0.0)
    uvw[0, 17, 0] = 1.0e7
    if mode == "sum_one_grid":
        gid, split, ngrids = None, False, 1
    elif mode == "sum_per_time_channel":
        gid, split = (np.arange(ntime * nchan) % 5).reshape(ntime, nchan).astype(np.int32), False
        ngrids = 5
    else:
        gid, split = (np.arange(ntime * npol * nchan) % 6).reshape(ntime, npol, nchan).astype(np.int32), True
        ngrids = 6
    im = gu.make_imager(p.n, p.cell_arcsec, p.support, p.oversample, ngrids=ngrids, strategy=strategy)
    try:
        im.set_weighting(binding.MUSER_WEIGHT_UNIFORM)       # the hit counts check the per-visibility bookkeeping too
        im.reset()
        im.grid_rows(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt), None if gid is None else gu.to_dev(gid),
                     binding.MUSER_POLS_SPLIT if split else binding.MUSER_POLS_SUM)
        fu, ff, fv, fw = mo.grid_rows_inputs(uvw, freq, vis, wt)
        fg = mo.rows_grid_ids(gid, ntime, npol, nchan, nrow, split)
        T = mo.table_pswf(p.support, p.oversample)
        G_or, Gw_or, st = oc.grid(fu, ff, fv, fw, p.n, p.n, p.cell_arcsec, p.oversample, p.support, T, grid_id=fg, ngrids=ngrids,
                                  counts=True)
        got = im.get_stats()
        assert (got["n_gridded"], got["n_dropped"], got["n_flagged"]) == (st["n_gridded"], st["n_dropped"], st["n_flagged"])
        assert st["n_flagged"] == 3 and st["n_dropped"] >= npol * nchan
        assert abs(got["sum_weights"] - st["sum_weights"]) <= 1e-9 * st["sum_weights"]
        G, Gw = gu.gpu_grids(im)
        assert gu.rel_l2(G, G_or) <= gu.GRID_TOL and gu.rel_l2(Gw, Gw_or) <= gu.GRID_TOL
        cnt = torch.empty((ngrids, p.n, p.n), dtype=torch.int32, device="cuda")
        im.get_counts(cnt)
        torch.cuda.synchronize()
        assert np.array_equal(cnt.cpu().numpy().astype(np.int64), st["cnt"])
        im.set_weighting(binding.MUSER_WEIGHT_NATURAL)
        im.reset()
        im.grid_rows(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt), None if gid is None else gu.to_dev(gid),
                     binding.MUSER_POLS_SPLIT if split else binding.MUSER_POLS_SUM)
        gu.check_images(im, G_or, Gw_or, T, p.support, p.oversample)
    finally:
        im.destroy()


@pytest.mark.parametrize("split", [False, True])
def test_channelised_rows_call_with_w_planes(split):
    """muser_grid_rows in w mode (generic binning kernel k_coords<ROWS> + the w-plane window gridder): polarisations summed
    before gridding or split over grids, flags in single polarisations, against the oracle on the flattened arrays."""
    n, cell, P, Q, w_max = 256, 60.0, 6, 16, 4000.0
    wc, sup = mo.wplane_layout(n, cell, P, w_max)
    fov = n * cell * mo.ARCSEC
    tabs = [mo.table_wkernel(int(S), Q, float(w), fov) for S, w in zip(sup, wc)]
    ntime, npol, nchan, nrow = 2, 2, 4, 700
    rng = np.random.default_rng(77)
    uvw = np.stack([synth.random_visibilities(40 + t, nrow, n, cell, margin_cells=sup.max() / 2 + 2, w_max_lambda=w_max)[0]
                    for t in range(ntime)]).astype(np.float32)
    freq = 1.0e9 * (1.0 + 0.01 * np.arange(nchan))
    vis = (1.0 + 0.2 * (rng.standard_normal((ntime, npol, nchan, nrow)) + 1j * rng.standard_normal((ntime, npol, nchan, nrow)))).astype(np.complex64)
    wt = rng.uniform(0.5, 1.5, vis.shape).astype(np.float32)
    wt[0, 1, 2, 5] = 0.0
    vis[1, 0, 3, 9] = complex(np.nan, 0.0)
    if split:
        gid, ngrids = (np.arange(ntime * npol * nchan) % 3).reshape(ntime, npol, nchan).astype(np.int32), 3
    else:
        gid, ngrids = None, 1
    im = gu.make_imager(n, cell, 7, Q, ngrids=ngrids)
    try:
        im.set_wplanes(wc, sup, [t.astype(np.complex64) for t in tabs])
        im.grid_rows(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt), None if gid is None else gu.to_dev(gid),
                     binding.MUSER_POLS_SPLIT if split else binding.MUSER_POLS_SUM)
        fu, ff, fv, fw = mo.grid_rows_inputs(uvw, freq, vis, wt)
        fg = mo.rows_grid_ids(gid, ntime, npol, nchan, nrow, split)
        G_or, Gw_or, st = oc.grid(fu, ff, fv, fw, n, n, cell, Q, sup, tabs, wc=wc, grid_id=fg, ngrids=ngrids)
        got = im.get_stats()
        assert (got["n_gridded"], got["n_dropped"], got["n_flagged"]) == (st["n_gridded"], st["n_dropped"], st["n_flagged"])
        assert st["n_flagged"] == 2
        assert abs(got["sum_weights"] - st["sum_weights"]) <= 1e-9 * st["sum_weights"]
        G, Gw = gu.gpu_grids(im)
        assert gu.rel_l2(G, G_or) <= gu.GRID_TOL and gu.rel_l2(Gw, Gw_or) <= gu.GRID_TOL
        if not split:
            gu.check_images(im, G_or, Gw_or, tabs[0].real, int(sup[0]), Q)
    finally:
        im.destroy()


def test_channelised_rows_call_with_phase_offset_and_accumulation():
    ntime = 3
    p, uvw, freq, vis, wt = _rows_inputs(2, ntime, seed=1)
    off = (1.3e-4, 0.9e-4)
    im = gu.make_imager(p.n, p.cell_arcsec, p.support, p.oversample)
    try:
        im.set_phase_offset(*off)
        im.reset()
        for t in range(ntime):                               # one call per time step, accumulating
            im.grid_rows(gu.to_dev(uvw[t:t + 1]), gu.to_dev(freq), gu.to_dev(vis[t:t + 1]), gu.to_dev(wt[t:t + 1]))
        fu, ff, fv, fw = mo.grid_rows_inputs(uvw, freq, vis, wt)
        T = mo.table_pswf(p.support, p.oversample)
        G_or, Gw_or, st = oc.grid(fu, ff, fv, fw, p.n, p.n, p.cell_arcsec, p.oversample, p.support, T, offset=off)
        assert im.get_stats()["n_gridded"] == st["n_gridded"]
        G, Gw = gu.gpu_grids(im)
        assert gu.rel_l2(G, G_or) <= gu.GRID_TOL and gu.rel_l2(Gw, Gw_or) <= gu.GRID_TOL
    finally:
        im.destroy()
