"""Pins of the oracle functions for SURVEY.md 8(f)'s NEXT rows (all CPU, `-m "not gpu"`): each function is checked
against something other than itself -- an independently built input, a textbook identity written out by brute
force, a hand-worked tiny case, a closed form, or numpy's own routine on inputs where the two must agree exactly."""
import numpy as np
import pytest

from oracle import muser_oracle as mo
from inputs import synth


def _small_rows(seed=3, ntime=2, npol=2, nchan=3, nrow=25, n=64, cell=60.0):
    rng = np.random.default_rng(seed)
    half = (n / 2 - 6) / (n * cell * mo.ARCSEC)
    freq = 1.0e9 + 25e6 * np.arange(nchan)
    uvw = np.zeros((ntime, nrow, 3), np.float32)
    uvw[..., :2] = (rng.uniform(-half, half, (ntime, nrow, 2)) * mo.C_M_S / freq[-1]).astype(np.float32)
    vis = (rng.standard_normal((ntime, npol, nchan, nrow)) + 1j * rng.standard_normal((ntime, npol, nchan, nrow))).astype(np.complex64)
    wt = rng.uniform(0.5, 1.5, (ntime, npol, nchan, nrow)).astype(np.float32)
    return uvw, freq, vis, wt


# ------------------------------------------------------------------------------------------------- N1: channelised input
def test_N1_rows_layout_is_the_flat_path_on_broadcast_arrays():
    n, cell, S, Q = 64, 60.0, 7, 8
    uvw, freq, vis, wt = _small_rows()
    ntime, npol, nchan, nrow = vis.shape
    fu, ff, fv, fw = mo.grid_rows_inputs(uvw, freq, vis, wt)
    # independent construction by broadcasting (no loops)
    bu = np.broadcast_to(uvw[:, None, None, :, :], (ntime, npol, nchan, nrow, 3)).reshape(-1, 3)
    bf = np.broadcast_to(freq[None, None, :, None], (ntime, npol, nchan, nrow)).reshape(-1)
    assert np.array_equal(fu, bu) and np.array_equal(ff, bf) and np.array_equal(fv, vis.reshape(-1)) and np.array_equal(fw, wt.reshape(-1))
    # the grid of the whole call equals, bit for bit, the grids of the (t, p, c) slices accumulated in loop order
    T = mo.table_gauss(S, Q)
    smp = mo.coordinates(fu, ff, fv, fw, n, n, cell, Q, S)
    G, Gw = mo.grid(smp, T, S, Q, n, n)
    G2 = np.zeros_like(G); Gw2 = np.zeros_like(Gw)
    for t in range(ntime):
        for p in range(npol):
            for c in range(nchan):
                f1 = np.full(nrow, freq[c])
                s1 = mo.coordinates(uvw[t], f1, vis[t, p, c], wt[t, p, c], n, n, cell, Q, S)
                for k in range(s1["val"].shape[0]):              # same sample order, same sequential sums
                    one = {key: (val[k:k + 1] if isinstance(val, np.ndarray) else val) for key, val in s1.items()}
                    g1, w1 = mo.grid(one, T, S, Q, n, n)
                    nzr = np.nonzero(np.abs(g1[0]).sum(1))[0]
                    G2[0, nzr] += g1[0, nzr]
                    Gw2[0, nzr] += w1[0, nzr]
    assert np.array_equal(G, G2) and np.array_equal(Gw, Gw2)


def test_N1_grid_ids_of_summed_and_split_polarisations():
    gid_sum = np.arange(2 * 3).reshape(2, 3)
    g = mo.rows_grid_ids(gid_sum, 2, 2, 3, 4, pols_split=False).reshape(2, 2, 3, 4)
    assert (g[:, 0] == g[:, 1]).all() and (g[1, 0, 2] == 5).all()
    gid_split = np.arange(2 * 2 * 3).reshape(2, 2, 3)
    g = mo.rows_grid_ids(gid_split, 2, 2, 3, 4, pols_split=True).reshape(2, 2, 3, 4)
    assert (g[1, 1, 0] == 9).all() and (g[0, 1, 2] == 5).all()
    assert mo.rows_grid_ids(None, 2, 2, 3, 4, False) is None


# ------------------------------------------------------------------------------------------------- N1b: half-plane
def test_N1b_halfplane_completion_is_the_full_grid_P3():
    fr = synth.make_frame(1)
    p = fr.params
    T = mo.table_gauss(p.support, p.oversample)
    smp = mo.coordinates(fr.uvw_m, fr.freq_hz, fr.vis, fr.weight, p.n, p.n, p.cell_arcsec, p.oversample, p.support)
    G, Gw = mo.grid(smp, T, p.support, p.oversample, p.n, p.n)
    H, Hw = mo.grid_halfplane(smp, T, p.support, p.oversample, p.n, p.n)
    assert not H[:, :p.n // 2].any() and np.array_equal(H[:, p.n // 2:], G[:, p.n // 2:])
    # Hermitian identity (P3): the completed half-plane is the full grid to fp64 rounding of the sums
    assert np.abs(mo.full_from_halfplane(H) - G).max() <= 1e-13 * np.abs(G).max()
    assert np.abs(mo.full_from_halfplane(Hw) - Gw).max() <= 1e-13 * np.abs(Gw).max()
    assert np.abs(mo.image_from_halfplane(H[0]) - mo.transform(G[0]).real).max() <= 1e-12 * np.abs(mo.transform(G[0])).max()


def test_N1b_image_from_halfplane_is_the_textbook_real_transform():
    """I(y, x) = sum_{iv = ny/2} H e^{...} + 2 Re sum_{iv > ny/2} H e^{...}, written out by brute force on a tiny grid."""
    rng = np.random.default_rng(8)
    ny, nx = 12, 16
    H = np.zeros((ny, nx), np.complex128)
    H[ny // 2 + 1:, 1:] = rng.standard_normal((ny // 2 - 1, nx - 1)) + 1j * rng.standard_normal((ny // 2 - 1, nx - 1))
    row = rng.standard_normal(nx // 2 - 1) + 1j * rng.standard_normal(nx // 2 - 1)      # row ny/2 is Hermitian in itself
    H[ny // 2, nx // 2 + 1:] = row
    H[ny // 2, 1:nx // 2] = np.conj(row[::-1])
    H[ny // 2, nx // 2] = 3.0
    img = mo.image_from_halfplane(H)
    xs, ys = np.arange(nx) - nx // 2, np.arange(ny) - ny // 2
    ref = np.zeros((ny, nx))
    for y in range(ny):
        for x in range(nx):
            ph = np.exp(2j * np.pi * (np.outer(ys, np.full(nx, ys[y])) / ny + np.outer(np.full(ny, xs[x]), xs) / nx))
            term = H * ph
            ref[y, x] = term[ny // 2].sum().real + 2.0 * term[ny // 2 + 1:].sum().real
    assert np.abs(img - ref).max() <= 1e-12 * np.abs(ref).max()


# ------------------------------------------------------------------------------------------------- N2: uniform weighting
def _lattice_visibilities(cells, n, cell, freq=1.0e9):
    """Visibilities exactly on grid cells (iu, iv) (phase 0): u_m chosen so that u_lambda * n * cell is an integer."""
    fov = n * cell * mo.ARCSEC
    cells = np.asarray(cells, np.float64)
    uvw = np.zeros((cells.shape[0], 3), np.float64)
    uvw[:, 0] = (cells[:, 0] - n / 2) / fov * mo.C_M_S / freq
    uvw[:, 1] = (cells[:, 1] - n / 2) / fov * mo.C_M_S / freq
    return uvw


def test_N2_hit_counts_by_hand_and_invariants():
    n, cell, S, Q = 64, 60.0, 7, 8
    # f32 metres cannot hit a lattice point exactly; +0.2 of a cell keeps the nearest cell unambiguous
    uvw = _lattice_visibilities([(40.2, 45.2), (40.2, 45.2), (20.2, 50.2)], n, cell).astype(np.float32)
    freq = np.full(3, 1.0e9)
    vis = np.array([1 + 1j, 3 - 1j, 2.0], np.complex64)
    wt = np.ones(3, np.float32)
    smp = mo.coordinates(uvw, freq, vis, wt, n, n, cell, Q, S)
    cnt = mo.hit_counts(smp, n, n)[0]
    assert cnt.sum() == 6 and cnt[45, 40] == 2 and cnt[50, 20] == 1
    assert cnt[n - 45, n - 40] == 2 and cnt[n - 50, n - 20] == 1          # the conjugates
    fr = synth.make_frame(1)
    p = fr.params
    smp = mo.coordinates(fr.uvw_m, fr.freq_hz, fr.vis, fr.weight, p.n, p.n, p.cell_arcsec, p.oversample, p.support)
    cnt = mo.hit_counts(smp, p.n, p.n)[0]
    assert cnt.sum() == smp["val"].shape[0]
    assert np.array_equal(cnt[1:, 1:], cnt[1:, 1:][::-1, ::-1])           # Hermitian: cnt[ny-y][nx-x] = cnt[y][x]


def test_N2_wgt_grid_as_printed():
    """Alg. 1 l.1-16: cell * (1/cnt) where cnt != 0 in uniform mode; untouched where cnt == 0; identity in natural mode.
    Isolated visibilities on (almost) one cell: the uniformly weighted centre cell is their kernel-weighted mean."""
    n, cell, S, Q = 64, 60.0, 7, 8
    uvw = _lattice_visibilities([(40.0, 45.0)] * 4, n, cell).astype(np.float32)
    vis = np.array([1 + 1j, 3 - 1j, 2.0, -2 + 4j], np.complex64)
    freq, wt = np.full(4, 1.0e9), np.ones(4, np.float32)
    T = mo.table_gauss(S, Q)
    smp = mo.coordinates(uvw, freq, vis, wt, n, n, cell, Q, S)
    G, Gw = mo.grid(smp, T, S, Q, n, n)
    cnt = mo.hit_counts(smp, n, n)
    assert np.array_equal(mo.wgt_grid(G, cnt, 0), G)
    U = mo.wgt_grid(G, cnt, 1)
    cu, cv = int(smp["iu0"][0]), int(smp["iv0"][0])
    assert cnt[0, cv, cu] == 4
    assert np.abs(U[0, cv, cu] - G[0, cv, cu] / 4).max() <= 1e-15 * abs(G[0, cv, cu])
    k00 = T[S * Q // 2 - int(smp["ru"][0])] * T[S * Q // 2 - int(smp["rv"][0])]       # kernel value at the nearest cell
    assert abs(U[0, cv, cu] - k00 * vis.astype(np.complex128).mean()) <= 1e-12
    zero = cnt == 0
    assert np.array_equal(U[zero], G[zero]) and np.abs(G[zero]).max() > 0  # the kernel's spill-over cells are left alone
    Uw = mo.wgt_grid(Gw, cnt, 1)
    assert abs(Uw[0, cv, cu] - k00) <= 1e-12                                # 4 unit weights / 4


def test_N2_imager_uniform_mode_and_2x_beam():
    fr = synth.make_frame(1)
    p = fr.params
    im = mo.Imager(p.n, p.n, p.cell_arcsec, p.support, p.oversample, kernel="gauss")
    im.grid(fr.uvw_m, fr.freq_hz, fr.vis, fr.weight)
    nat, _ = im.dirty()
    im.weighting = 1
    uni, _ = im.dirty()
    assert np.abs(uni - nat).max() > 1e-3 * np.abs(nat).max()               # the weighting does something
    # uniform weighting flattens the sampling density: the beam's peak is the number of occupied cells (their
    # kernel-weighted, count-divided sums) rather than the number of samples
    beam, _ = im.psf()
    occupied = (im.cnt[0] > 0).sum()
    assert 0.5 * occupied < beam[0, p.n // 2, p.n // 2] < 1.5 * occupied
    # NEXT-2b, the beam on twice the field: an imager of 2n x 2n pixels with the same cell; (I) pins it:
    # at the phase centre the direct-DFT beam is the sum of weights, and gridding + FFT reaches it (P1)
    im2 = mo.Imager(2 * p.n, 2 * p.n, p.cell_arcsec, p.support, p.oversample, kernel="gauss")
    smp = im2.grid(fr.uvw_m, fr.freq_hz, np.ones_like(fr.vis), fr.weight)
    b2, _ = im2.psf()
    sw = im2.stats["sum_weights"]
    assert abs(b2[0, p.n, p.n] / sw - 1) < 1e-2
    xs = np.array([p.n, p.n + 40, p.n - 140, p.n + 150]); ys = np.array([p.n, p.n - 17, p.n + 135, p.n - 150])   # beyond the 1x field (|offset| > n/2 = 128)
    dd = mo.direct_dft(smp["u"], smp["v"], smp["w"], smp["wt"].astype(np.complex128), xs, ys, 2 * p.n, 2 * p.n, p.cell_arcsec).real
    assert abs(dd[0] - sw) <= 1e-9 * sw
    assert np.abs(b2[0, ys, xs] - dd).max() <= 3e-2 * sw                    # Gaussian kernel, Q = 8: snap + aliasing level (P4)


# ------------------------------------------------------------------------------------------------- N3: phase correction
def test_N3_phase_correction_moves_a_source_to_the_phase_centre_P7_backwards():
    n, cell = 64, 60.0
    rng = np.random.default_rng(4)
    nvis = 60
    half = (n / 2 - 6) / (n * cell * mo.ARCSEC)
    freq = np.full(nvis, 1.4e9)
    uvw = np.zeros((nvis, 3), np.float32)
    uvw[:, :2] = (rng.uniform(-half, half, (nvis, 2)) * mo.C_M_S / 1.4e9).astype(np.float32)
    x0, y0 = 41, 23
    l0, m0 = (x0 - n / 2) * cell * mo.ARCSEC, (y0 - n / 2) * cell * mo.ARCSEC
    il = freq / mo.C_M_S
    u, v = uvw[:, 0].astype(np.float64) * il, uvw[:, 1].astype(np.float64) * il
    wt = rng.uniform(0.5, 1.5, nvis)
    vis = np.exp(-2j * np.pi * (u * l0 + v * m0))                          # a unit source at pixel (x0, y0) (P7)
    vc = mo.phase_correct(uvw, freq, vis, l0, m0)
    assert np.abs(vc - 1.0).max() <= 1e-9                                   # it now sits at the phase centre
    U, V_, VAL = np.concatenate([u, -u]), np.concatenate([v, -v]), np.concatenate([wt * vc, wt * np.conj(vc)])
    xs, ys = np.meshgrid(np.arange(n), np.arange(n))
    img = mo.direct_dft(U, V_, np.zeros_like(U), VAL, xs.ravel(), ys.ravel(), n, n, cell).real.reshape(n, n)
    assert np.unravel_index(np.argmax(img), img.shape) == (n // 2, n // 2)
    assert abs(img[n // 2, n // 2] - 2 * wt.sum()) <= 1e-9 * wt.sum()
    # and the imager applies it to what it grids
    a = mo.Imager(n, n, cell, 7, 8)
    a.offset = (l0, m0)
    a.grid(uvw, freq, vis.astype(np.complex64), wt.astype(np.float32))
    b = mo.Imager(n, n, cell, 7, 8)
    b.grid(uvw, freq, np.ones(nvis, np.complex64), wt.astype(np.float32))
    assert np.abs(a.G - b.G).max() <= 1e-6 * np.abs(b.G).max()              # complex64 rounding of the input visibilities


# ------------------------------------------------------------------------------------------------- N4: peak, histogram
def test_N4_peak_by_hand_and_ties():
    img = np.array([[0.0, 1.0, -3.0], [5.0, 2.0, 5.0]], np.float32)
    assert mo.image_peak(img) == (5.0, 1, 0, -3.0)                          # first of the two equal maxima
    rng = np.random.default_rng(1)
    a = rng.standard_normal((37, 53)).astype(np.float32)
    v, y, x, lo = mo.image_peak(a)
    assert v == a.max() and a[y, x] == v and lo == a.min()


def test_N4_histogram_by_hand_and_against_numpy_on_exact_inputs():
    assert mo.image_histogram(np.array([0.0, 0.5, 1.0, 1.5, -0.1], np.float32), 2, 0.0, 1.0).tolist() == [1, 2]
    rng = np.random.default_rng(2)
    k = rng.integers(0, 1025, 5000)
    v = (k / 1024.0).astype(np.float32)                                     # dyadic values: every product below is exact
    h = mo.image_histogram(v, 256, 0.0, 1.0)
    ref, _ = np.histogram(v.astype(np.float64), bins=256, range=(0.0, 1.0))
    assert np.array_equal(h, ref) and h.sum() == 5000
    # 2000 ranges between the image's own minimum and maximum: everything is counted, both ends included
    img = rng.standard_normal((64, 64)).astype(np.float32)
    h = mo.image_histogram(img, 2000, img.min(), img.max())
    assert h.sum() == img.size and h[0] >= 1 and h[-1] >= 1
