"""-m gpu parity tests: the CUDA path (through the C ABI / binding) against the fp64 oracle, element by element,
on the same seeded inputs.  Tolerances are BASELINE.json's: grid relative L2 <= 1e-5, images max-abs <= 1e-4 of
the peak (gates of DESIGN.md R9).  Integer results (counters) must be equal."""
import numpy as np
import pytest

from oracle import muser_oracle as mo
from oracle import oracle_c as oc
from paper_1712_06913_b200 import binding
from inputs import synth

import gpu_util as gu

pytestmark = pytest.mark.gpu

TILED, OWNER, WPLANE = binding.MUSER_STRATEGY_TILED, binding.MUSER_STRATEGY_OWNER, binding.MUSER_STRATEGY_WPLANE


@pytest.mark.parametrize("strategy", [OWNER, TILED])
@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_single_grid_configs_match_oracle(cfg, strategy):
    fr = synth.make_frame(cfg)
    p = fr.params
    res = gu.run_case(fr.uvw_m, fr.freq_hz, fr.vis, fr.weight, p.n, p.cell_arcsec, p.support, p.oversample,
                      kernel=p.kernel, strategy=strategy)
    assert res["stats"]["n_gridded"] > 0.9 * fr.nvis


@pytest.mark.parametrize("strategy", [TILED, WPLANE])
@pytest.mark.parametrize("S,Q,nvis", [(7, 128, 1), (7, 16, 31), (7, 128, 5000), (3, 8, 777), (5, 32, 1000), (9, 64, 1500),
                                      (1, 2, 100), (15, 16, 300), (9, 16, 30000), (21, 8, 4000), (31, 4, 2000)])
def test_random_visibilities_any_support(S, Q, nvis, strategy):
    n, cell = 128, 40.0
    uvw, freq, vis, wt = synth.random_visibilities(7 + S, nvis, n, cell, margin_cells=S / 2 + 2)
    gu.run_case(uvw, freq, vis, wt, n, cell, S, Q, strategy=strategy)


@pytest.mark.parametrize("strategy", [OWNER, TILED])
def test_accumulation_over_calls_equals_one_call(strategy):
    fr = synth.make_frame(2)
    p = fr.params
    gu.run_case(fr.uvw_m, fr.freq_hz, fr.vis, fr.weight, p.n, p.cell_arcsec, p.support, p.oversample,
                strategy=strategy, splits=5, images=False)


def test_owner_tiles_never_written_stand_for_zeros_until_a_later_call_or_a_dense_consumer():
    """The owner gridder does not zero-fill empty tiles: a tile keeps flag 0 ("zeros", whatever its memory holds) until a
    later accumulating call stores into it or a consumer of the dense grids fills it.  The grids are pre-filled with
    rubbish (a first dense cycle), reset, then gridded in two calls that touch different tiles; images straight from
    the flagged half-plane after each call, then the dense grids."""
    import torch
    n, cell, S, Q = 512, 20.0, 7, 32
    uvw, freq, vis, wt = synth.random_visibilities(61, 6000, n, cell, margin_cells=6.0)
    vis = (1.0 + 0.1 * vis).astype(np.complex64)
    r = np.hypot(uvw[:, 0], uvw[:, 1])
    inner, outer = r < np.median(r) * 0.5, r >= np.median(r) * 0.5
    im = gu.make_imager(n, cell, S, Q, strategy=OWNER)
    T = gu.oracle_table("pswf", S, Q)
    try:
        big = [gu.to_dev(a) for a in (uvw, freq, (vis * 1e3).astype(np.complex64), wt)]
        im.grid(*big)                                        # every tile that will matter now holds large stale values
        gu.gpu_grids(im)                                     # (dense consumer: fills the rest)
        im.reset()
        sel = [gu.to_dev(np.ascontiguousarray(a[inner])) for a in (uvw, freq, vis, wt)]
        im.grid(*sel)
        G1, W1, _ = oc.grid(uvw[inner], freq[inner], vis[inner], wt[inner], n, n, cell, Q, S, T)
        gu.check_images(im, G1, W1, T, S, Q)                 # row transform on the flagged half-plane
        sel = [gu.to_dev(np.ascontiguousarray(a[outer])) for a in (uvw, freq, vis, wt)]
        im.grid(*sel)                                        # accumulating call: stores into tiles still at flag 0
        G2, W2, st = oc.grid(uvw, freq, vis, wt, n, n, cell, Q, S, T)
        gu.check_images(im, G2, W2, T, S, Q)
        G, Gw = gu.gpu_grids(im)                             # dense grids: unwritten tiles read back as exact zeros
        assert gu.rel_l2(G, G2) <= gu.GRID_TOL and gu.rel_l2(Gw, W2) <= gu.GRID_TOL
        assert np.all(G[0][np.abs(G2[0]) == 0] == 0)
        assert im.get_stats()["n_gridded"] == st["n_gridded"]
    finally:
        im.destroy()


@pytest.mark.parametrize("seed", [0, 1, 2, 3, 4])
def test_random_call_sequences_keep_the_lazy_state_consistent(seed):
    """reset / grid (pieces of the data, by the owner or the generic gridder) / images / dense read-backs in random order: after
    every step that produces something, it equals the oracle on the pieces gridded since the last reset.  Exercises the
    deferred reset, the tile flags, the lower half-plane mirror and the cached row transform together."""
    import torch
    rng = np.random.default_rng(1000 + seed)
    n, cell, S, Q = 256, 20.0, 7, 16
    uvw, freq, vis, wt = synth.random_visibilities(70 + seed, 4000, n, cell, margin_cells=6.0)
    vis = (1.0 + 0.2 * vis).astype(np.complex64)
    r = np.hypot(uvw[:, 0], uvw[:, 1])
    order = np.argsort(r)                                    # pieces are rings in uv: different calls touch different tiles
    pieces = np.array_split(order, 8)
    T = gu.oracle_table("pswf", S, Q)
    im = gu.make_imager(n, cell, S, Q)
    since = []                                               # pieces gridded since the last reset
    def expected():
        if not since:
            return np.zeros((1, n, n), np.complex128), np.zeros((1, n, n)), 0
        idx = np.concatenate(since)
        G, W, st = oc.grid(uvw[idx], freq[idx], vis[idx], wt[idx], n, n, cell, Q, S, T)
        return G, W, st["n_gridded"]
    try:
        for step in range(24):
            op = rng.choice(["reset", "grid", "grid", "grid_tiled", "images", "dense", "dirty_only"])
            if op == "reset":
                im.reset(); since = []
            elif op in ("grid", "grid_tiled"):
                im.set_strategy(TILED if op == "grid_tiled" else binding.MUSER_STRATEGY_AUTO)
                idx = pieces[rng.integers(len(pieces))]
                im.grid(*[gu.to_dev(np.ascontiguousarray(a[idx])) for a in (uvw, freq, vis, wt)])
                since.append(idx)
            elif op == "dense":
                G, Gw = gu.gpu_grids(im)
                G_or, W_or, ng = expected()
                assert im.get_stats()["n_gridded"] == ng
                if ng:
                    assert gu.rel_l2(G, G_or) <= gu.GRID_TOL and gu.rel_l2(Gw, W_or) <= gu.GRID_TOL, (step, op)
                else:
                    assert not G.any() and not Gw.any(), (step, op)
            else:
                d = torch.full((1, n, n), 7.0, device="cuda"); b = torch.full((1, n, n), 7.0, device="cuda")
                if op == "images":
                    im.dirty_psf(d, b)
                else:
                    im.dirty(d); im.psf(b)
                torch.cuda.synchronize()
                G_or, W_or, ng = expected()
                if ng:
                    _, cor_d, _, cor_p, _ = gu.oracle_images(G_or, W_or, T, S, Q)
                    q = n // 8
                    for got, ref in ((d.cpu().numpy(), cor_d), (b.cpu().numpy(), cor_p)):
                        err = np.abs(got - ref)[:, q:-q, q:-q].max() / np.abs(ref[:, q:-q, q:-q]).max()
                        assert err <= gu.IMG_TOL, (step, op, err)
                else:
                    assert not d.cpu().numpy().any() and not b.cpu().numpy().any(), (step, op)
    finally:
        im.destroy()


@pytest.mark.parametrize("strategy", [OWNER, TILED])
def test_flagged_and_off_grid_visibilities_are_skipped_and_counted(strategy):
    n, cell = 256, 20.0
    uvw, freq, vis, wt = synth.random_visibilities(3, 4000, n, cell, margin_cells=0.0)   # some fall off the grid
    rng = np.random.default_rng(5)
    bad = rng.choice(4000, 400, replace=False)
    wt[bad[:100]] = 0.0
    wt[bad[100:150]] = -1.0
    wt[bad[150:180]] = np.nan
    vis[bad[180:230]] = np.nan + 0j
    vis[bad[230:260]] = complex(0.0, np.inf)
    uvw[bad[260:300], 0] = np.inf
    uvw[bad[300:340], 2] = np.nan
    freq[bad[340:370]] = np.nan
    uvw[bad[370:400], 1] = 1e30          # finite but absurdly far off the grid -> dropped, not flagged
    res = gu.run_case(uvw, freq, vis, wt, n, cell, 7, 32, strategy=strategy)
    assert res["stats"]["n_flagged"] == 370
    assert res["stats"]["n_dropped"] >= 30


@pytest.mark.parametrize("Q,nvis,n,ny", [(128, 1, 128, None), (16, 31, 128, None), (128, 5000, 128, None), (2, 3000, 64, None),
                                          (256, 20000, 256, None), (64, 4000, 96, 160)])
def test_owner_strategy_random_visibilities(Q, nvis, n, ny):
    """Owner-tile gridder (support 7): ragged tile edges (n = 96, 160 are not multiples of 32), one sample, the
    largest oversampling, non-square grids."""
    cell = 40.0
    uvw, freq, vis, wt = synth.random_visibilities(11 + Q, nvis, n if ny is None else min(n, ny), cell, margin_cells=5.5)
    if ny is None:
        gu.run_case(uvw, freq, vis, wt, n, cell, 7, Q, strategy=OWNER)
    else:
        im = gu.make_imager(n, cell, 7, Q, strategy=OWNER, ny=ny)
        try:
            im.reset()
            im.grid(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt))
            G, Gw = gu.gpu_grids(im)
            T = gu.oracle_table("pswf", 7, Q)
            G_or, Gw_or, st = oc.grid(uvw, freq, vis, wt, n, ny, cell, Q, 7, T)
            assert im.get_stats()["n_gridded"] == st["n_gridded"]
            assert gu.rel_l2(G[0], G_or[0]) <= gu.GRID_TOL and gu.rel_l2(Gw[0], Gw_or[0]) <= gu.GRID_TOL
        finally:
            im.destroy()


@pytest.mark.parametrize("item_size", [0, 10000, 1 << 20])
def test_owner_heavy_tile_is_split_into_chunks_and_summed(item_size):
    """40,000 visibilities inside +-6 cells of the uv origin: the centre tile holds ~80,000 samples = 20 chunk items
    whose partial tiles the last chunk adds up; the second call exercises accumulate mode on a heavy tile.
    item_size 10000: chunks of several sort units (kOwUnit = 4096) with a ragged last unit; 2^20: the whole tile is one
    item of ~10 units (the multi-unit path of k_grid_owner_s7, no partial-tile sum)."""
    n, cell, Q = 256, 20.0, 64
    rng = np.random.default_rng(99)
    nvis = 40000
    fov = n * cell * mo.ARCSEC
    uv_l = rng.uniform(-6.0, 6.0, (nvis, 2)) / fov                        # wavelengths
    freq = np.full(nvis, 1.0e9)
    uvw = np.zeros((nvis, 3), np.float32)
    uvw[:, :2] = (uv_l * mo.C_M_S / 1.0e9).astype(np.float32)
    vis = (rng.standard_normal(nvis) + 1j * rng.standard_normal(nvis)).astype(np.complex64)
    wt = rng.uniform(0.5, 1.5, nvis).astype(np.float32)
    # images=False: with all the power inside +-6 cells of the origin the image is smooth and small against the fp32
    # FFT noise that 1/(cx*cy) amplifies towards the edge of the 75% box; the grid gates are what this case is about
    res = gu.run_case(uvw, freq, vis, wt, n, cell, 7, Q, strategy=OWNER, splits=2, images=False, item_size=item_size)
    assert res["stats"]["n_gridded"] == nvis


def test_owner_strategy_is_refused_where_it_does_not_apply():
    im = gu.make_imager(128, 40.0, 5, 8, strategy=OWNER)
    try:
        uvw, freq, vis, wt = synth.random_visibilities(1, 10, 128, 40.0)
        with pytest.raises(binding.MuserError) as e:
            im.grid(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt))
        assert e.value.code == binding.MUSER_EUNSUPPORTED
    finally:
        im.destroy()


def test_reset_then_read_back_is_zero_with_lazy_zeroing():
    """muser_reset defers the memset when the owner-tile gridder follows; every other consumer must still see zeros."""
    im = gu.make_imager(128, 40.0, 7, 8)
    try:
        uvw, freq, vis, wt = synth.random_visibilities(2, 300, 128, 40.0)
        im.grid(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt))
        im.reset()
        G, Gw = gu.gpu_grids(im)
        assert not G.any() and not Gw.any()
        im.grid(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt))
        im.reset()
        d, p = gu.gpu_images(im)
        assert not d.any() and not p.any()
        im.reset()
        im.set_strategy(TILED)                                   # a deferred reset must survive a strategy change
        im.grid(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt))
        G1, _ = gu.gpu_grids(im)
        im.set_strategy(OWNER)
        im.reset()
        im.grid(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt))
        G2, _ = gu.gpu_grids(im)
        assert gu.rel_l2(G2, G1) <= 1e-6
    finally:
        im.destroy()


@pytest.mark.parametrize("strategy", [OWNER, TILED])
def test_side_stream_first_call_and_scratch_growth(strategy):
    """Every call on a non-blocking side stream (torch.cuda.Stream()), starting with a fresh handle: the library's own
    zero-initialisations (histograms, tickets, grids after set_batch) must be ordered before the kernels that read
    them on that stream, on the first call and again when the scratch buffers grow."""
    import torch
    n, cell, Q = 256, 20.0, 32
    side = torch.cuda.Stream()
    T = gu.oracle_table("pswf", 7, Q)
    with torch.cuda.stream(side):
        im = gu.make_imager(n, cell, 7, Q, strategy=strategy)
        try:
            for ngrids, nvis in ((1, 500), (3, 40000)):          # the second round re-allocates grids and grows every scratch
                if ngrids != 1:
                    im.set_batch(ngrids)
                uvw, freq, vis, wt = synth.random_visibilities(40 + ngrids, nvis, n, cell, margin_cells=5.5)
                vis = (vis * 0.05 + 1.0).astype(np.complex64)  # a bright point-like component: image peak well above the noise
                if nvis > 1000:                                  # crowd the centre tile: heavy-tile chunks and tickets
                    uvw[: nvis // 2, :2] *= 0.02
                gid = (np.arange(nvis) % ngrids).astype(np.int32)
                d = [gu.to_dev(a) for a in (uvw, freq, vis, wt, gid)]
                im.reset()
                im.grid_batched(*d)
                G, Gw = gu.gpu_grids(im)
                st = im.get_stats()
                G_or, Gw_or, st_or = oc.grid(uvw, freq, vis, wt, n, n, cell, Q, 7, T, grid_id=gid, ngrids=ngrids)
                assert st["n_gridded"] == st_or["n_gridded"]
                assert gu.rel_l2(G, G_or) <= gu.GRID_TOL and gu.rel_l2(Gw, Gw_or) <= gu.GRID_TOL
                gu.check_images(im, G_or, Gw_or, T, 7, Q)
        finally:
            im.destroy()
    side.synchronize()


def test_empty_input_and_reset():
    import torch
    im = gu.make_imager(128, 40.0, 7, 8)
    try:
        z = torch.zeros(0, device="cuda")
        im.grid(z.reshape(0, 3), z.double(), z.reshape(0, 2), z)            # nvis = 0: no-op
        uvw, freq, vis, wt = synth.random_visibilities(0, 100, 128, 40.0)
        im.grid(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt))
        assert im.get_stats()["n_gridded"] == 100
        im.reset()
        G, Gw = gu.gpu_grids(im)
        assert not G.any() and not Gw.any()
        st = im.get_stats()
        assert st == dict(sum_weights=0.0, n_gridded=0, n_dropped=0, n_flagged=0)
        d, p = gu.gpu_images(im)
        assert not d.any() and not p.any()
    finally:
        im.destroy()


def test_dirty_and_psf_separately_equal_the_fused_call():
    import torch
    fr = synth.make_frame(1)
    p = fr.params
    im = gu.make_imager(p.n, p.cell_arcsec, p.support, p.oversample, kernel=p.kernel)
    try:
        im.grid(gu.to_dev(fr.uvw_m), gu.to_dev(fr.freq_hz), gu.to_dev(fr.vis), gu.to_dev(fr.weight))
        a = torch.empty((p.n, p.n), device="cuda"); b = torch.empty_like(a); c = torch.empty_like(a); d = torch.empty_like(a)
        im.psf(b); im.dirty(a)                # either order; the transform is shared
        im.dirty_psf(c, d)
        torch.cuda.synchronize()
        assert torch.equal(a, c) and torch.equal(b, d)
        # gridding more afterwards still works (the grids are not consumed by imaging)
        im.grid(gu.to_dev(fr.uvw_m), gu.to_dev(fr.freq_hz), gu.to_dev(fr.vis), gu.to_dev(fr.weight))
        im.dirty(c)
        torch.cuda.synchronize()
        q = p.n // 4                                   # central half: away from the corrector's noise amplification
        ci, ai = c[q:-q, q:-q], a[q:-q, q:-q]
        assert float((ci - 2 * ai).abs().max()) <= 1e-4 * float(ai.abs().max())
    finally:
        im.destroy()


def test_point_source_peak_is_sum_of_weights_P1():
    fr = synth.make_frame(2)
    p = fr.params
    vis = np.ones_like(fr.vis)
    im = gu.make_imager(p.n, p.cell_arcsec, p.support, p.oversample)
    try:
        im.grid(gu.to_dev(fr.uvw_m), gu.to_dev(fr.freq_hz), gu.to_dev(vis), gu.to_dev(fr.weight))
        d, b = gu.gpu_images(im)
        sw = im.get_stats()["sum_weights"]
        assert abs(d[0, p.n // 2, p.n // 2] / sw - 1) < 2e-3
        assert np.unravel_index(np.argmax(d[0]), d[0].shape) == (p.n // 2, p.n // 2)
        q = p.n // 4
        assert np.abs(d - b)[0, q:-q, q:-q].max() <= 1e-4 * sw          # V = 1: dirty image == beam
    finally:
        im.destroy()


def test_device_table_matches_oracle_table():
    for kernel, S, Q in (("pswf", 7, 128), ("gauss", 7, 8)):
        im = gu.make_imager(64, 60.0, S, Q, kernel=kernel)
        try:
            assert np.abs(im.get_table(0) - gu.oracle_table(kernel, S, Q)).max() <= 1e-7
        finally:
            im.destroy()


def _wplane_case(n, cell, P, Q, nvis, w_max, seed, library_tables):
    wc, sup = mo.wplane_layout(n, cell, P, w_max)
    fov = n * cell * mo.ARCSEC
    tabs = [mo.table_wkernel(int(S), Q, float(w), fov) for S, w in zip(sup, wc)]
    uvw, freq, vis, wt = synth.random_visibilities(seed, nvis, n, cell, margin_cells=sup.max() / 2 + 2, w_max_lambda=w_max)
    return wc, sup, tabs, (uvw, freq, vis, wt)


@pytest.mark.parametrize("strategy", [TILED, WPLANE])
@pytest.mark.parametrize("library_tables", [False, True])
def test_wprojection_planes_match_oracle(strategy, library_tables):
    n, cell, P, Q, w_max = 256, 60.0, 6, 16, 4000.0          # fov 4.3 deg: supports 7..17
    wc, sup, tabs, (uvw, freq, vis, wt) = _wplane_case(n, cell, P, Q, 3000, w_max, 11, library_tables)
    assert sup.max() >= 13
    im = gu.make_imager(n, cell, 7, Q, strategy=strategy)
    try:
        im.set_wplanes(wc, sup, None if library_tables else [t.astype(np.complex64) for t in tabs])
        im.grid(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt))
        G, Gw = gu.gpu_grids(im)
        G_or, Gw_or, st_or = oc.grid(uvw, freq, vis, wt, n, n, cell, Q, sup, tabs, wc=wc)
        st = im.get_stats()
        assert (st["n_gridded"], st["n_dropped"], st["n_flagged"]) == (st_or["n_gridded"], st_or["n_dropped"], st_or["n_flagged"])
        assert gu.rel_l2(G, G_or) <= gu.GRID_TOL
        assert gu.rel_l2(Gw, Gw_or) <= gu.GRID_TOL
        gu.check_images(im, G_or, Gw_or, tabs[0].real, int(sup[0]), Q)
        for p_ in range(P):
            assert np.abs(im.get_table(p_).view(np.complex64) - tabs[p_]).max() <= 2e-7
    finally:
        im.destroy()


def test_wprojection_unevenly_spaced_planes_take_the_full_plane_scan():
    """Plane centres that are not a ladder p * step: K1 scans all planes (the O(1) search only applies to ladders)."""
    n, cell, P, Q, w_max = 256, 60.0, 6, 16, 4000.0
    wc, sup = mo.wplane_layout(n, cell, P, w_max)
    wc = wc * (1.0 + 0.35 * np.arange(P) / P)                 # stretched: uneven spacing, still increasing
    fov = n * cell * mo.ARCSEC
    sup = (7 + 2 * np.floor(wc * fov * fov / 4.0 + 0.5)).astype(np.int64)
    tabs = [mo.table_wkernel(int(S), Q, float(w), fov) for S, w in zip(sup, wc)]
    uvw, freq, vis, wt = synth.random_visibilities(29, 3000, n, cell, margin_cells=sup.max() / 2 + 2, w_max_lambda=w_max)
    im = gu.make_imager(n, cell, 7, Q)
    try:
        im.set_wplanes(wc, sup, [t.astype(np.complex64) for t in tabs])
        im.grid(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt))
        G, Gw = gu.gpu_grids(im)
        G_or, Gw_or, st_or = oc.grid(uvw, freq, vis, wt, n, n, cell, Q, sup, tabs, wc=wc)
        st = im.get_stats()
        assert (st["n_gridded"], st["n_dropped"], st["n_flagged"]) == (st_or["n_gridded"], st_or["n_dropped"], st_or["n_flagged"])
        assert gu.rel_l2(G, G_or) <= gu.GRID_TOL
        assert gu.rel_l2(Gw, Gw_or) <= gu.GRID_TOL
    finally:
        im.destroy()


def test_wprojection_calls_capture_into_a_cuda_graph():
    """reset -> grid -> dirty_psf in w mode only enqueue work (the per-shape kernels fork onto side streams and join the
    caller's stream with events), so the sequence captures into a CUDA graph; the replay equals the plain calls."""
    import torch
    n, cell, P, Q, w_max = 256, 60.0, 6, 16, 4000.0
    wc, sup = mo.wplane_layout(n, cell, P, w_max)
    uvw, freq, vis, wt = synth.random_visibilities(11, 20000, n, cell, margin_cells=sup.max() / 2 + 2, w_max_lambda=w_max)
    vis = (1.0 + 0.2 * vis).astype(np.complex64)
    im = gu.make_imager(n, cell, 7, Q)
    try:
        im.set_wplanes(wc, sup, None)
        dev = [gu.to_dev(a) for a in (uvw, freq, vis, wt)]
        d = torch.empty((1, n, n), device="cuda"); b = torch.empty_like(d)

        def step(s=None):
            im.reset(s); im.grid(*dev, stream=s); im.dirty_psf(d, b, s)

        step()
        torch.cuda.synchronize()
        ref_d, ref_b = d.clone(), b.clone()
        side = torch.cuda.Stream()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.stream(side):
            step(side.cuda_stream)                           # allocations happen outside the capture
            torch.cuda.synchronize()
            with torch.cuda.graph(graph, stream=side):
                step(side.cuda_stream)
        d.zero_(); b.zero_()
        for _ in range(3):
            graph.replay()
        torch.cuda.synchronize()
        q = n // 4                                           # (the corrected corners amplify fp32 reordering noise)
        for got, ref in ((d, ref_d), (b, ref_b)):
            assert float((got - ref)[:, q:-q, q:-q].abs().max()) <= 1e-5 * float(ref[:, q:-q, q:-q].abs().max())
    finally:
        im.destroy()


@pytest.mark.parametrize("strategy", [TILED, WPLANE])
def test_wprojection_small_supports_and_arbitrary_caller_tables(strategy):
    """Supports 1, 3, 5 (windows smaller than their register layout), 7 and 9 with arbitrary complex tables supplied by the
    caller (parity does not depend on what the tables mean), uniform weighting on (hit counts through the generic binning)."""
    import torch
    n, cell, Q = 128, 60.0, 4
    sup = np.array([1, 3, 5, 7, 9], np.int64)
    wc = np.array([0.0, 300.0, 700.0, 1200.0, 2000.0])
    rng = np.random.default_rng(314)
    tabs = [(rng.uniform(0.2, 1.0, S * Q + 1) + 1j * rng.uniform(-0.5, 0.5, S * Q + 1)) for S in sup]
    tabs = [0.5 * (t + t[::-1]) for t in tabs]                # even, as every gridding kernel is (the half-plane design needs it)
    tabs[0] = tabs[0].real.astype(np.complex128)              # plane 0's real part defines the grid correction
    uvw, freq, vis, wt = synth.random_visibilities(19, 20000, n, cell, margin_cells=7.0, w_max_lambda=2200.0)
    uvw = uvw.copy(); uvw[::3, :2] *= 0.1                     # a dense patch: runs of several records per window
    im = gu.make_imager(n, cell, 7, Q, strategy=strategy)
    try:
        im.set_weighting(binding.MUSER_WEIGHT_UNIFORM)
        bad = [t.astype(np.complex64) for t in tabs]
        bad[2] = bad[2].copy(); bad[2][1] += 0.3              # an odd component: refused
        with pytest.raises(binding.MuserError):
            im.set_wplanes(wc, sup, bad)
        im.set_wplanes(wc, sup, [t.astype(np.complex64) for t in tabs])
        im.grid(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt))
        G, Gw = gu.gpu_grids(im)
        tabs32 = [t.astype(np.complex64).astype(np.complex128) for t in tabs]
        G_or, Gw_or, st_or = oc.grid(uvw, freq, vis, wt, n, n, cell, Q, sup, tabs32, wc=wc, counts=True)
        st = im.get_stats()
        assert (st["n_gridded"], st["n_dropped"], st["n_flagged"]) == (st_or["n_gridded"], st_or["n_dropped"], st_or["n_flagged"])
        assert gu.rel_l2(G, G_or) <= gu.GRID_TOL
        assert gu.rel_l2(Gw, Gw_or) <= gu.GRID_TOL
        cnt = torch.empty((1, n, n), dtype=torch.int32, device="cuda")
        im.get_counts(cnt)
        torch.cuda.synchronize()
        assert np.array_equal(cnt.cpu().numpy().astype(np.int64), st_or["cnt"])
    finally:
        im.destroy()


@pytest.mark.parametrize("strategy", [TILED, WPLANE])
@pytest.mark.parametrize("ngrids", [1, 3])
def test_wprojection_every_support_class_dense_runs_and_batches(strategy, ngrids):
    """Supports 7..31 (all three classes of the window gridder), dense uv coverage near the origin (long runs of records
    per window, items of 4096 records split across CTAs), positive and negative w, several grids."""
    n, cell, P, Q, w_max = 256, 60.0, 14, 8, 9000.0
    wc, sup, tabs, (uvw, freq, vis, wt) = _wplane_case(n, cell, P, Q, 40000, w_max, 23, False)
    assert sup.min() == 7 and sup.max() == 31 and len(set(sup.tolist())) >= 10
    uvw = uvw.copy()
    uvw[::2, :2] *= 0.12                                      # half of the visibilities crowd a few tiles around the origin
    vis = (1.0 + 0.2 * vis).astype(np.complex64)              # a source at the phase centre (no w phase there) + noise: the
                                                              # image has a real peak for the 1e-4-of-peak gate to refer to
    gid = (np.arange(uvw.shape[0]) % ngrids).astype(np.int32) if ngrids > 1 else None
    im = gu.make_imager(n, cell, 7, Q, strategy=strategy, ngrids=ngrids)
    try:
        im.set_wplanes(wc, sup, [t.astype(np.complex64) for t in tabs])
        if gid is None:
            im.grid(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt))
        else:
            im.grid_batched(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt), gu.to_dev(gid))
        G, Gw = gu.gpu_grids(im)
        G_or, Gw_or, st_or = oc.grid(uvw, freq, vis, wt, n, n, cell, Q, sup, tabs, wc=wc, grid_id=gid, ngrids=ngrids)
        st = im.get_stats()
        assert (st["n_gridded"], st["n_dropped"], st["n_flagged"]) == (st_or["n_gridded"], st_or["n_dropped"], st_or["n_flagged"])
        assert gu.rel_l2(G, G_or) <= gu.GRID_TOL
        assert gu.rel_l2(Gw, Gw_or) <= gu.GRID_TOL
        if ngrids == 1:
            gu.check_images(im, G_or, Gw_or, tabs[0].real, int(sup[0]), Q)
    finally:
        im.destroy()


@pytest.mark.parametrize("strategy", [OWNER, TILED])
def test_batched_grids_cfg4_slice(strategy):
    fr = synth.make_frame(4, nframes=1)                       # 32 grids of 512x512, 1770 visibilities each
    p = fr.params
    assert p.ngrids == 32
    gu.run_case(fr.uvw_m, fr.freq_hz, fr.vis, fr.weight, p.n, p.cell_arcsec, p.support, p.oversample,
                strategy=strategy, grid_id=fr.grid_id, ngrids=p.ngrids)


def test_batched_rejects_out_of_range_grid_ids_as_flagged():
    n, cell = 128, 40.0
    uvw, freq, vis, wt = synth.random_visibilities(1, 500, n, cell)
    gid = (np.arange(500) % 5 - 1).astype(np.int32)           # -1 and 3 are outside [0, 3)
    res = gu.run_case(uvw, freq, vis, wt, n, cell, 7, 8, grid_id=np.clip(gid, 0, 2), ngrids=3, images=False)
    im = gu.make_imager(n, cell, 7, 8, ngrids=3)
    try:
        im.grid_batched(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt), gu.to_dev(gid))
        st = im.get_stats()
        assert st["n_flagged"] == int(((gid < 0) | (gid >= 3)).sum())
        assert st["n_gridded"] + st["n_dropped"] + st["n_flagged"] == 500
    finally:
        im.destroy()
    assert res["stats"]["n_flagged"] == 0


def test_cfg5_reduced_wprojection_4096():
    fr = synth.make_frame(5, nsnap=2)                         # 113,280 visibilities, 4096^2 grid, 32 planes
    p = fr.params
    wc, sup = mo.wplane_layout(p.n, p.cell_arcsec, p.nplanes, 19900.0)     # |w| beyond the last centre -> last plane
    assert sup.min() == 7 and sup.max() == 31
    fov = p.n * p.cell_arcsec * mo.ARCSEC
    tabs = [mo.table_wkernel(int(S), p.oversample, float(w), fov) for S, w in zip(sup, wc)]
    im = gu.make_imager(p.n, p.cell_arcsec, 7, p.oversample)
    try:
        im.set_wplanes(wc, sup, [t.astype(np.complex64) for t in tabs])
        im.grid(gu.to_dev(fr.uvw_m), gu.to_dev(fr.freq_hz), gu.to_dev(fr.vis), gu.to_dev(fr.weight))
        G, Gw = gu.gpu_grids(im)
        G_or, Gw_or, st_or = oc.grid(fr.uvw_m, fr.freq_hz, fr.vis, fr.weight, p.n, p.n, p.cell_arcsec, p.oversample,
                                     sup, tabs, wc=wc)
        assert im.get_stats()["n_gridded"] == st_or["n_gridded"]
        assert gu.rel_l2(G, G_or) <= gu.GRID_TOL
        assert gu.rel_l2(Gw, Gw_or) <= gu.GRID_TOL
        gu.check_images(im, G_or, Gw_or, tabs[0].real, 7, p.oversample)
    finally:
        im.destroy()


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_column_pass_staged_by_tma_equals_per_lane_loads(cfg):
    """MUSER_TUNE_COLS_TMA: the strip of the fused column transform fetched by cp.async.bulk.tensor or by per-lane loads
    (ny = 256, 512, 1024; two grids)."""
    import torch
    fr = synth.make_frame(cfg)
    p = fr.params
    im = gu.make_imager(p.n, p.cell_arcsec, p.support, p.oversample, kernel=p.kernel, ngrids=2)
    try:
        gid = (np.arange(fr.nvis) % 2).astype(np.int32)
        im.grid_batched(gu.to_dev(fr.uvw_m), gu.to_dev(fr.freq_hz), gu.to_dev(fr.vis), gu.to_dev(fr.weight), gu.to_dev(gid))
        out = {}
        for mode in (1, 2):
            im.set_tuning(binding.MUSER_TUNE_COLS_TMA, mode)
            d = torch.zeros((2, p.n, p.n), device="cuda"); b = torch.zeros_like(d)
            im.dirty_psf(d, b)
            torch.cuda.synchronize()
            out[mode] = (d.cpu().numpy(), b.cpu().numpy())
        assert np.abs(out[1][0]).max() > 0
        if p.n == 256:                                       # same arithmetic after the staging: identical images
            assert np.array_equal(out[1][0], out[2][0]) and np.array_equal(out[1][1], out[2][1])
        else:                                                # ny = 512, 1024: the TMA path also runs two radix-8 stages instead of
            for a, b in zip(out[1], out[2]):                 # three radix-4 ones: same transform, fp32 rounding differs
                q = p.n // 8
                assert np.abs(a - b)[:, q:-q, q:-q].max() <= 1e-5 * np.abs(a[:, q:-q, q:-q]).max()   # (corrected: x900 at the box corners)
    finally:
        im.destroy()


def test_frame_host_end_to_end_equals_device_path():
    import torch
    fr = synth.make_frame(2)
    p = fr.params
    im = gu.make_imager(p.n, p.cell_arcsec, p.support, p.oversample)
    try:
        d_host = np.empty((p.n, p.n), np.float32); b_host = np.empty((p.n, p.n), np.float32)
        im.frame_host(fr.uvw_m, fr.freq_hz, fr.vis, fr.weight, None, d_host, b_host)
        im.frame_host(fr.uvw_m, fr.freq_hz, fr.vis, fr.weight, None, d_host, b_host)   # resets: no accumulation
        d = torch.empty((p.n, p.n), device="cuda"); b = torch.empty_like(d)
        im.reset()
        im.grid(gu.to_dev(fr.uvw_m), gu.to_dev(fr.freq_hz), gu.to_dev(fr.vis), gu.to_dev(fr.weight))
        im.dirty_psf(d, b)
        torch.cuda.synchronize()
        q = p.n // 4
        dd, bb = d.cpu().numpy()[q:-q, q:-q], b.cpu().numpy()[q:-q, q:-q]
        assert np.abs(d_host[q:-q, q:-q] - dd).max() <= 1e-5 * np.abs(dd).max()
        assert np.abs(b_host[q:-q, q:-q] - bb).max() <= 1e-5 * np.abs(bb).max()
    finally:
        im.destroy()


def test_abi_argument_errors_on_device():
    L = binding.lib()
    im = gu.make_imager(128, 40.0, 7, 8)
    try:
        h = im._h
        assert L.muser_grid(h, None, None, None, None, 5, None) == binding.MUSER_EINVAL
        assert L.muser_grid(h, None, None, None, None, -1, None) == binding.MUSER_EINVAL
        assert L.muser_grid(h, None, None, None, None, 0, None) == binding.MUSER_OK
        assert L.muser_dirty(h, None, None) == binding.MUSER_EINVAL
        assert L.muser_set_batch(h, 0) == binding.MUSER_EINVAL
        assert L.muser_set_kernel(h, 9, 0.0) == binding.MUSER_EINVAL
        assert L.muser_set_strategy(h, 17) == binding.MUSER_EINVAL
        assert b"strategy" in L.muser_last_error(h)
        assert L.muser_set_wplanes(h, 2, None, None, None) == binding.MUSER_EINVAL
    finally:
        im.destroy()


def test_microbenchmarks_report_plausible_device_limits():
    mb = binding.microbench()
    assert set(mb) == set(binding.MICROBENCH)
    assert 1e13 < mb["fp32_fma_flops"] < 1.2e14                  # B200: 148 SMs x 128 lanes x 2 x <= 1.965 GHz = 74.5e12
    assert mb["shared_int_adds"] > 1.5 * mb["shared_f32_cas_adds"] > 0   # why the owner gridder merges in fixed point
    assert mb["global_f32_red_adds"] > 1e11


@pytest.mark.parametrize("nx,ny", [(512, 256), (256, 512), (1024, 1024), (272, 1024), (512, 2048), (2048, 512), (256, 4096)])
def test_images_on_fused_and_library_fft_paths(nx, ny):
    """ny = 256 ... 4096 (a power of two) with nx a multiple of 16 takes the fused column pass (8 columns per CTA up to 1024,
    4 above), with the own row pass when nx is a power of two too, else cuFFT rows; non-square grids; dirty image and beam
    against the oracle's O4 + O5."""
    import torch
    cell, Q = 30.0, 32
    n = min(nx, ny)
    uvw, freq, vis, wt = synth.random_visibilities(5 + nx + ny, 3000, n, cell * max(nx, ny) / n, margin_cells=6.0)
    # a bright point-like component keeps the image peak well above the noise of the random visibilities
    vis = (vis * 0.05 + 1.0).astype(np.complex64)
    im = gu.make_imager(nx, cell, 7, Q, ny=ny)
    try:
        im.reset()
        im.grid(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt))
        T = gu.oracle_table("pswf", 7, Q)
        G_or, Gw_or, st = oc.grid(uvw, freq, vis, wt, nx, ny, cell, Q, 7, T)
        assert im.get_stats()["n_gridded"] == st["n_gridded"] > 2000
        gu.check_images(im, G_or, Gw_or, T, 7, Q)
        d = torch.empty((1, ny, nx), device="cuda"); p = torch.empty_like(d); d2 = torch.empty_like(d); p2 = torch.empty_like(d)
        im.dirty_psf(d, p)
        im.dirty(d2); im.psf(p2)                             # separate calls re-use the row transform
        torch.cuda.synchronize()
        assert torch.equal(d, d2) and torch.equal(p, p2)
    finally:
        im.destroy()


def test_owner_fixed_point_merge_bound_per_cell_with_a_1e6_outlier():
    """The owner gridder merges register sums into a 32-bit fixed-point tile whose unit is 2^-31 / 0.98 of the work unit's
    L1 bound B = max(sum |wt Re V|, sum |wt Im V|) (sum wt for the weight grid).  Guarantee: every merge rounds to the
    nearest unit, so a cell that received m merges is off by at most m * 2^-32 * B / 0.98, plus the fp32 rounding of
    the register sums (a few 1e-7 of the cell's own magnitude).  One visibility 1e6 times brighter than 300 unit ones
    in the same tile: the global rel-L2 is trivially fine, the per-cell bound is what is checked -- and it shows the
    dynamic-range limit: cells 1e6 times fainter than the tile's bound keep ~3 significant digits."""
    n, cell, Q = 256, 20.0, 32
    rng = np.random.default_rng(77)
    nvis = 301
    fov = n * cell * mo.ARCSEC
    # all samples inside the tile x in [96, 160), y in [128, 160) (cells relative to the centre (128, 128): u in [-28, 28), v in [4, 28))
    cu = rng.uniform(-26.0, 26.0, nvis); cv = rng.uniform(6.0, 26.0, nvis)
    cu[0], cv[0] = 20.3, 20.4                                 # the outlier
    far = np.hypot(cu - cu[0], cv - cv[0]) > 9.0              # unit samples whose footprint does not overlap the outlier's
    far[0] = True
    cu, cv = cu[far], cv[far]
    nvis = cu.size
    freq = np.full(nvis, 1.0e9)
    uvw = np.zeros((nvis, 3), np.float32)
    uvw[:, 0] = (cu / fov * mo.C_M_S / 1.0e9).astype(np.float32)
    uvw[:, 1] = (cv / fov * mo.C_M_S / 1.0e9).astype(np.float32)
    vis = (rng.standard_normal(nvis) + 1j * rng.standard_normal(nvis)).astype(np.complex64)
    vis[0] = 1.0e6 * (0.6 + 0.8j)
    wt = np.ones(nvis, np.float32)
    res = gu.run_case(uvw, freq, vis, wt, n, cell, 7, Q, strategy=OWNER, images=False)
    G, G_or = res["G"][0], res["G_or"][0]
    up = slice(n // 2, n)                                     # the tile sits in the stored half-plane; the rest is its mirror
    B = max(np.abs(vis.real).sum(), np.abs(vis.imag).sum())
    unit = B / (0.98 * 2.0 ** 31)
    m_max = 2 * nvis                                          # at most one merge per record
    err = np.abs(G[up] - G_or[up])
    bound = m_max * 0.5 * unit * np.sqrt(2.0) + 2e-6 * np.abs(G_or[up])
    assert (err <= bound).all(), f"worst excess {np.max(err - bound):.3e}"
    # away from the outlier the cells are O(1): the absolute error there really is of the order of the unit, not of 1e-7
    faint = (np.abs(G_or[up]) > 0.05) & (np.abs(G_or[up]) < 50.0)
    assert faint.sum() > 500 and err[faint].max() <= m_max * 0.5 * unit * np.sqrt(2.0)
    assert err[faint].max() < 20 * unit                       # in practice a handful of merges per cell


def _edge_visibilities(n, cell, h, seed, w_max=0.0, with_ties=True):
    """Visibilities whose nearest cell is h, h + 1, n - 1 - h or n - h on one axis or on both (the keep / drop boundary of R5,
    oracle pin P13), at random sub-cell offsets, plus exact half-cell ties at the boundary (frequency scanned ulp by ulp so
    that O1's own operation order lands on the tie exactly)."""
    rng = np.random.default_rng([7, seed])
    su = n * cell * mo.ARCSEC
    edge = np.array([h, h + 1, n - 1 - h, n - h], np.float64)
    m = 600
    pu = rng.choice(edge, m) + rng.uniform(-0.49, 0.49, m)
    pv = rng.uniform(h + 2, n - h - 2, m)
    pu[m // 3:2 * m // 3], pv[m // 3:2 * m // 3] = pv[m // 3:2 * m // 3].copy(), (rng.choice(edge, m) + rng.uniform(-0.49, 0.49, m))[m // 3:2 * m // 3]
    pv[2 * m // 3:] = rng.choice(edge, m - 2 * m // 3) + rng.uniform(-0.49, 0.49, m - 2 * m // 3)      # corners: both axes at the edge
    freq = np.full(m, 1.0e9)
    lam = mo.C_M_S / 1.0e9
    uvw = np.zeros((m, 3), np.float32)
    uvw[:, 0] = ((pu - n / 2) / su * lam).astype(np.float32)
    uvw[:, 1] = ((pv - n / 2) / su * lam).astype(np.float32)
    ties = []
    for off in (n / 2 - h - 0.5, -(n / 2 - h - 0.5), n / 2 - h - 1.5, -(n / 2 - h - 1.5)):
        um = np.float32(off / su * lam)
        f = off / (float(um) * su) * mo.C_M_S
        for _ in range(4000):
            f = np.nextafter(f, -np.inf)
        for _ in range(8000):
            if float(um) * (f / mo.C_M_S) * su == off:
                ties.append((um, float(f)))
                break
            f = np.nextafter(f, np.inf)
    assert len(ties) == 4
    if not with_ties:
        ties = []
    tu = np.zeros((2 * len(ties), 3), np.float32)
    tf = np.empty(2 * len(ties))
    for i, (um, f) in enumerate(ties):
        tu[2 * i, 0] = um; tu[2 * i + 1, 1] = um                      # the tie on the u axis, then on the v axis
        tf[2 * i] = tf[2 * i + 1] = f
    uvw = np.concatenate([uvw, tu]); freq = np.concatenate([freq, tf])
    nv = uvw.shape[0]
    if w_max > 0:
        uvw[:, 2] = (rng.uniform(-w_max, w_max, nv) * lam).astype(np.float32)
    vis = (rng.standard_normal(nv) + 1j * rng.standard_normal(nv)).astype(np.complex64)
    wt = rng.uniform(0.5, 1.5, nv).astype(np.float32)
    return uvw, freq, vis, wt


def _check_stored_halfplane_and_mirror(G, G_or):
    """Exact half-cell ties (R4): both samples of a visibility round UP, so the full-grid oracle's two footprints are
    not mirror images of each other (one edge cell each) and its grid is Hermitian only up to that.  The CUDA path computes
    the rows >= ny/2 with the oracle's rule and completes the rest as the Hermitian mirror.  What is unique: the stored
    half-plane equals the oracle's; what must be valid: the other half is the conjugate mirror of it."""
    ny, nx = G.shape[-2:]
    up = slice(ny // 2, ny)
    assert gu.rel_l2(G[..., up, :], G_or[..., up, :]) <= gu.GRID_TOL
    low, mir = G[..., 1:ny // 2, 1:], np.conj(G[..., ny - 1:ny // 2:-1, :0:-1])
    assert gu.rel_l2(low, mir) <= 1e-6


@pytest.mark.parametrize("strategy", [OWNER, TILED])
def test_keep_drop_boundary_cells_2d(strategy):
    """Samples on cells h, h+1, n-1-h, n-h: kept / dropped counts and grids equal the oracle's (P13 pins the oracle's rule by
    hand); nothing is written to row / column 0.  Then the same with exact half-cell ties at the boundary added."""
    n, cell, Q = 256, 20.0, 16
    uvw, freq, vis, wt = _edge_visibilities(n, cell, 3, 1, with_ties=False)
    res = gu.run_case(uvw, freq, vis, wt, n, cell, 7, Q, strategy=strategy, images=False)
    assert res["stats"]["n_dropped"] > 100 and res["stats"]["n_gridded"] > 100
    assert not res["G"][0][0, :].any() and not res["G"][0][:, 0].any()
    assert res["G"][0][:, 1].any() and res["G"][0][:, n - 1].any()
    uvw, freq, vis, wt = _edge_visibilities(n, cell, 3, 1)
    im = gu.make_imager(n, cell, 7, Q, strategy=strategy)
    try:
        im.reset()
        im.grid(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt))
        G, Gw = gu.gpu_grids(im)
        G_or, Gw_or, st_or = oc.grid(uvw, freq, vis, wt, n, n, cell, Q, 7, gu.oracle_table("pswf", 7, Q, 0.0))
        st = im.get_stats()
        assert (st["n_gridded"], st["n_dropped"], st["n_flagged"]) == (st_or["n_gridded"], st_or["n_dropped"], st_or["n_flagged"])
        assert st["n_gridded"] == res["stats"]["n_gridded"] + 4 and st["n_dropped"] == res["stats"]["n_dropped"] + 4   # by hand: P13
        _check_stored_halfplane_and_mirror(G, G_or)
        _check_stored_halfplane_and_mirror(Gw, Gw_or)
        assert not G[0][0, :].any() and not G[0][:, 0].any()
    finally:
        im.destroy()


@pytest.mark.parametrize("strategy", [TILED, WPLANE])
def test_keep_drop_boundary_cells_wplanes(strategy):
    """The same with two w planes of supports 7 and 9: the boundary depends on the plane a visibility falls into."""
    n, cell, Q = 256, 20.0, 16
    wc, sup = np.array([0.0, 400.0]), np.array([7, 9])
    fov = n * cell * mo.ARCSEC
    tabs = [mo.table_wkernel(int(s_), Q, float(w_), fov) for s_, w_ in zip(sup, wc)]
    uvw3, freq3, vis3, wt3 = _edge_visibilities(n, cell, 3, 2, w_max=400.0)
    uvw4, freq4, vis4, wt4 = _edge_visibilities(n, cell, 4, 3, w_max=400.0)
    uvw, freq, vis, wt = (np.concatenate(a) for a in ((uvw3, uvw4), (freq3, freq4), (vis3, vis4), (wt3, wt4)))
    im = gu.make_imager(n, cell, 7, Q, strategy=strategy)
    try:
        im.set_wplanes(wc, sup, [t.astype(np.complex64) for t in tabs])
        im.grid(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt))
        G, Gw = gu.gpu_grids(im)
        G_or, Gw_or, st_or = oc.grid(uvw, freq, vis, wt, n, n, cell, Q, sup, tabs, wc=wc)
        st = im.get_stats()
        assert (st["n_gridded"], st["n_dropped"], st["n_flagged"]) == (st_or["n_gridded"], st_or["n_dropped"], st_or["n_flagged"])
        assert st["n_dropped"] > 200 and st["n_gridded"] > 200
        _check_stored_halfplane_and_mirror(G, G_or)              # the input holds exact ties
        _check_stored_halfplane_and_mirror(Gw, Gw_or)
        assert not G[0][0, :].any() and not G[0][:, 0].any()
    finally:
        im.destroy()
