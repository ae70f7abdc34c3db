"""The plain-C oracle (oracle/oracle_c.c) against the numpy transcription (oracle/muser_oracle.py) and against
closed forms -- two independent transcriptions of O1/O3/O6 and of (I) must agree to fp64 rounding."""
import numpy as np
import pytest

from oracle import muser_oracle as mo
from oracle import oracle_c as oc
from inputs import synth

ARCSEC = np.pi / 648000.0


def test_c_gridder_equals_numpy_gridder_cfg1_and_counters():
    fr = synth.make_frame(1)
    p = fr.params
    uvw = fr.uvw_m.copy(); wt = fr.weight.copy(); vis = fr.vis.copy()
    wt[5] = 0.0; wt[6] = -1.0; vis[7] = np.nan; uvw[8, 0] = np.inf        # flagged data: skipped and counted
    im = mo.Imager(p.n, p.n, p.cell_arcsec, p.support, p.oversample, p.kernel)
    im.grid(uvw, fr.freq_hz, vis, wt)
    G, Gw, st = oc.grid(uvw, fr.freq_hz, vis, wt, p.n, p.n, p.cell_arcsec, p.oversample, p.support, im.T)
    assert st == im.stats
    assert st["n_flagged"] == 4 and st["n_dropped"] > 0
    assert st["n_gridded"] + st["n_dropped"] + st["n_flagged"] == fr.nvis
    np.testing.assert_allclose(G, im.G, atol=1e-13 * np.abs(im.G).max())
    np.testing.assert_allclose(Gw, im.Gw, atol=1e-13 * im.Gw.max())


def test_c_gridder_equals_numpy_gridder_wmode_and_batched():
    n, cell, Q, P, w_max = 128, 80.0, 16, 8, 19900.0
    uvw, f, vis, wt = synth.random_visibilities(21, 200, n, cell, margin_cells=20, w_max_lambda=w_max)
    im = mo.Imager(n, n, cell, 7, Q, "pswf")
    im.set_wplanes(P, w_max)
    smp = im.grid(uvw, f, vis, wt)
    assert len(set(smp["plane"].tolist())) >= 6 and smp["conj_kernel"].sum() == smp["conj_kernel"].size // 2
    G, Gw, st = oc.grid(uvw, f, vis, wt, n, n, cell, Q, im.supports, im.tables, wc=im.wc)
    assert st == im.stats
    np.testing.assert_allclose(G, im.G, atol=1e-13 * np.abs(im.G).max())
    np.testing.assert_allclose(Gw, im.Gw, atol=1e-13 * np.abs(im.Gw).max())
    # batched: grid_id routes each visibility to its own grid
    gid = (np.arange(200) % 3).astype(np.int32)
    b = mo.Imager(n, n, cell, 7, Q, "pswf", ngrids=3)
    b.grid(uvw, f, vis, wt, grid_id=gid)
    G3, Gw3, _ = oc.grid(uvw, f, vis, wt, n, n, cell, Q, 7, b.T, grid_id=gid, ngrids=3)
    np.testing.assert_allclose(G3, b.G, atol=1e-13 * np.abs(b.G).max())
    for g in range(3):
        one = mo.Imager(n, n, cell, 7, Q, "pswf"); one.grid(uvw[gid == g], f[gid == g], vis[gid == g], wt[gid == g])
        np.testing.assert_allclose(G3[g], one.G[0], atol=1e-13 * np.abs(b.G).max())


def test_c_dft_equals_numpy_dft_and_plane_wave_closed_form():
    rng = np.random.default_rng(5)
    ns = 300
    u, v, w = rng.uniform(-500, 500, ns), rng.uniform(-500, 500, ns), rng.uniform(-3000, 3000, ns)
    val = rng.standard_normal(ns) + 1j * rng.standard_normal(ns)
    n, cell = 64, 60.0
    xs, ys = rng.integers(0, n, 20), rng.integers(0, n, 20)
    l, m = (xs - n / 2) * cell * ARCSEC, (ys - n / 2) * cell * ARCSEC
    for use_w in (False, True):
        a = mo.direct_dft(u, v, w, val, xs, ys, n, n, cell, use_w)
        b = oc.dft(u, v, w, val, l, m, use_w)
        np.testing.assert_allclose(b, a, atol=1e-10 * np.abs(a).max())
    # one sample: a pure plane wave
    out = oc.dft([100.0], [-50.0], [0.0], [2.0 + 0j], l, m)
    np.testing.assert_allclose(out, 2.0 * np.exp(2j * np.pi * (100.0 * l - 50.0 * m)), atol=1e-12)


def test_synth_shapes_counts_and_determinism():
    for cfg, nvis, nbl in ((1, 780, 780), (2, 24960, 780), (3, 56640, 1770)):
        fr = synth.make_frame(cfg)
        assert fr.nvis == nvis and fr.uvw_m.dtype == np.float32 and fr.freq_hz.dtype == np.float64
        assert fr.vis.dtype == np.complex64 and fr.weight.dtype == np.float32 and fr.uvw_m.shape == (nvis, 3)
        again = synth.make_frame(cfg)
        assert np.array_equal(fr.vis, again.vis) and np.array_equal(fr.uvw_m, again.uvw_m)
        b = np.linalg.norm(fr.uvw_m[:nbl].astype(np.float64), axis=1)
        assert 1.0 < b.min() < 30.0 and 2000.0 < b.max() < 6500.0        # metres ... ~3 km arms
    fr4 = synth.make_frame(4, nframes=2)
    assert fr4.nvis == 2 * 32 * 1770 and fr4.params.ngrids == 64 and fr4.grid_id.max() == 63
    assert np.all(np.bincount(fr4.grid_id) == 1770)
    fr5 = synth.make_frame(5, nsnap=3)
    assert fr5.nvis == 3 * 32 * 1770
    wl = np.abs(fr5.uvw_m[:, 2].astype(np.float64) * fr5.freq_hz / 299792458.0)
    assert 5000.0 < wl.max() < 25000.0


def test_cfg3_uv_coverage_is_centrally_condensed():
    """The statistic that drives the kernel design (SURVEY.md hard part 3): few 32x32 tiles hold most samples."""
    fr = synth.make_frame(3)
    p = fr.params
    smp = mo.coordinates(fr.uvw_m, fr.freq_hz, fr.vis, fr.weight, p.n, p.n, p.cell_arcsec, p.oversample, p.support)
    tile = (smp["iv0"] // 32) * 32 + smp["iu0"] // 32
    cnt = np.sort(np.bincount(tile, minlength=1024))[::-1]
    assert (cnt > 0).sum() < 600
    assert cnt[:4].sum() > 0.3 * cnt.sum()


def test_oracle_c_counts_and_phase_offset_equal_the_numpy_oracle():
    """NEXT-2 / NEXT-3 in the plain-C transcription: hit counts equal mo.hit_counts exactly; a phase offset equals
    mo.phase_correct applied first (fp64 on both sides)."""
    from inputs import synth
    fr = synth.make_frame(1)
    p = fr.params
    T = mo.table_gauss(p.support, p.oversample)
    off = (3.1e-4, -1.7e-4)
    G, Gw, st = oc.grid(fr.uvw_m, fr.freq_hz, fr.vis, fr.weight, p.n, p.n, p.cell_arcsec, p.oversample, p.support, T,
                        offset=off, counts=True)
    smp = mo.coordinates(fr.uvw_m, fr.freq_hz, mo.phase_correct(fr.uvw_m, fr.freq_hz, fr.vis, *off), fr.weight, p.n, p.n,
                         p.cell_arcsec, p.oversample, p.support)
    G_np, Gw_np = mo.grid(smp, T, p.support, p.oversample, p.n, p.n)
    assert np.array_equal(st["cnt"], mo.hit_counts(smp, p.n, p.n))
    assert np.abs(G - G_np).max() <= 1e-12 * np.abs(G_np).max()
    assert np.abs(Gw - Gw_np).max() <= 1e-13 * np.abs(Gw_np).max()
