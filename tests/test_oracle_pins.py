"""Pins P1..P12 (DESIGN.md / SURVEY.md §8(c)) for the CPU oracle.  The paper prints no worked numerical
example of gridding (PAPER.md has none), so every pin is mathematical: closed forms, invariants, library
special functions, brute force on tiny inputs.  None of these tests touches the CUDA path."""
import numpy as np
import pytest
from scipy import special as sp

from oracle import muser_oracle as mo
from oracle import oracle_c as oc
from inputs import synth

ARCSEC = np.pi / 648000.0
C = 299792458.0


def _tiny(seed=0, nvis=40, n=64, cell=60.0, **kw):
    return synth.random_visibilities(seed, nvis, n, cell, **kw)


def _inner(n, frac):
    c = np.arange(n) - n // 2
    m = np.abs(c) < frac * n / 2
    return np.ix_(m, m)


# ------------------------------------------------------------------ P1: point source at phase centre
@pytest.mark.parametrize("kernel,Q,tol", [("pswf", 128, 1e-3), ("gauss", 8, 1e-2)])
def test_P1_point_source_peak_is_sum_of_weights(kernel, Q, tol):
    n, cell = 64, 60.0
    uvw, f, _, wt = _tiny(1, 60, n, cell)
    vis = np.ones(60, np.complex64)
    im = mo.Imager(n, n, cell, 7, Q, kernel)
    smp = im.grid(uvw, f, vis, wt)
    sw = im.stats["sum_weights"]
    assert sw == pytest.approx(2.0 * wt.astype(np.float64).sum(), rel=1e-15)
    # (I): exactly the sum of weights at pixel (n/2, n/2)
    peak = mo.direct_dft(smp["u"], smp["v"], smp["w"], smp["val"], [n // 2], [n // 2], n, n, cell)[0]
    assert abs(peak - sw) <= 1e-12 * sw
    # (II): up to aliasing; dirty image == PSF when V == 1
    d, _ = im.dirty()
    p, _ = im.psf()
    assert abs(d[0, n // 2, n // 2] - sw) <= tol * sw
    np.testing.assert_allclose(d, p, rtol=0, atol=1e-9 * sw)
    assert np.unravel_index(np.argmax(d[0]), d[0].shape) == (n // 2, n // 2)


# ------------------------------------------------------------------ P2: uniform disk closed form
def test_P2_disk_visibility_closed_form_vs_pixelated_disk():
    """Forward DFT of a finely pixelated unit-flux disk of radius 16' reproduces 2 J1(x)/x, x = 2 pi R q,
    and the first null sits at q = 1.21967/theta (theta = 32' -> 131.0 lambda)."""
    R = 16.0 * 60.0 * ARCSEC
    pix = 4.0 * ARCSEC
    g = (np.arange(-260, 261) + 0.0) * pix
    L, M = np.meshgrid(g, g)
    inside = (L ** 2 + M ** 2) <= R ** 2
    l, m = L[inside], M[inside]
    flux = np.full(l.size, 1.0 / l.size)
    q = np.array([0.0, 30.0, 80.0, 131.0, 200.0, 350.0])
    for ang in (0.0, 0.7):
        u, v = q * np.cos(ang), q * np.sin(ang)
        vis_px = np.array([np.sum(flux * np.exp(-2j * np.pi * (uu * l + vv * m))) for uu, vv in zip(u, v)])
        vis_cf = synth.sky_visibilities(u, v, 0 * u, [], False)
        np.testing.assert_allclose(vis_px.real, vis_cf.real, atol=2e-3)
        np.testing.assert_allclose(vis_px.imag, 0.0, atol=1e-9)
    null = 1.21967 / (2 * R)
    assert abs(null - 131.0) < 0.1
    assert abs(synth.sky_visibilities(np.array([null]), np.array([0.0]), np.array([0.0]), [], False)[0]) < 1e-4


def test_P2_direct_dft_of_disk_visibilities_is_a_flat_disk():
    """(I) applied to closed-form disk visibilities on a dense uv lattice returns brightness 1/(pi R^2) inside
    radius R and ~0 outside: pins the units of `direct_dft` (cell, lambda) and of the generator's disk model."""
    R = 16.0 * 60.0 * ARCSEC
    du = 12.0                                   # lambda; field 1/du = 4.8 deg >> disk
    k = np.arange(-160, 161) * du
    U, V = np.meshgrid(k, k)
    u, v = U.ravel(), V.ravel()
    taper = np.exp(-(u ** 2 + v ** 2) / (2 * 900.0 ** 2))          # mild apodisation against Gibbs ripple
    vis = synth.sky_visibilities(u, v, 0 * u, [], False) * taper
    n, cell = 256, 10.0
    rad_px = R / (cell * ARCSEC)                 # 96 px
    xs = np.array([128, 128 + 40, 128, 128 + 70, 128 + 120, 128, 10])
    ys = np.array([128, 128, 128 - 60, 128 + 30, 128, 128 + 125, 128])
    img = mo.direct_dft(u, v, 0 * u, vis, xs, ys, n, n, cell).real * du * du
    r = np.hypot(xs - 128, ys - 128)
    level = 1.0 / (np.pi * R * R)
    assert np.all(np.abs(img[r < 0.85 * rad_px] / level - 1.0) < 0.03)
    assert np.all(np.abs(img[r > 1.15 * rad_px] / level) < 0.03)


# ------------------------------------------------------------------ P3: Hermitian symmetry
def test_P3_hermitian_grid_and_real_image():
    n, cell = 64, 60.0
    uvw, f, vis, wt = _tiny(3, 80, n, cell)
    im = mo.Imager(n, n, cell, 7, 128, "pswf")
    im.grid(uvw, f, vis, wt)
    G, Gw = im.G[0], im.Gw[0]
    scale = np.abs(G).max()
    mirror = np.conj(G[1:, 1:][::-1, ::-1])
    assert np.abs(G[1:, 1:] - mirror).max() <= 1e-13 * scale
    assert np.abs(Gw[1:, 1:] - Gw[1:, 1:][::-1, ::-1]).max() <= 1e-13 * Gw.max()
    assert np.all(G[0, :] == 0) and np.all(G[:, 0] == 0)          # row/col 0 have no mirror: kept empty (R5)
    F = mo.transform(G)
    assert np.abs(F.imag).max() <= 1e-12 * np.abs(F.real).max()


# ------------------------------------------------------------------ P4: (II) vs (I) on a tiny case
@pytest.mark.parametrize("kernel,Q,gate50,gate75", [("pswf", 128, 2e-4, 3e-3), ("gauss", 8, 1.2e-2, 5e-2)])
def test_P4_gridded_fft_image_matches_direct_dft_at_snapped_positions(kernel, Q, gate50, gate75):
    n, cell = 64, 60.0
    uvw, f, vis, wt = _tiny(4, 40, n, cell)
    im = mo.Imager(n, n, cell, 7, Q, kernel)
    smp = im.grid(uvw, f, vis, wt)
    su = n * cell * ARCSEC
    us = (smp["iu0"] + smp["ru"] / Q - n / 2) / su            # snapped positions the table actually serves
    vs = (smp["iv0"] + smp["rv"] / Q - n / 2) / su
    ys, xs = np.mgrid[0:n, 0:n]
    for val, img in ((smp["val"], im.dirty()[0][0]), (smp["wt"].astype(complex), im.psf()[0][0])):
        ref = mo.direct_dft(us, vs, 0 * us, val, xs.ravel(), ys.ravel(), n, n, cell).reshape(n, n)
        assert np.abs(ref.imag).max() < 1e-9 * np.abs(ref.real).max()
        peak = np.abs(ref.real).max()
        err = np.abs(img - ref.real) / peak
        assert err[_inner(n, 0.5)].max() < gate50
        assert err[_inner(n, 0.75)].max() < gate75
    # against the TRUE positions the table's 1/Q snap shows (expected, not a bug) -- but stays small at Q=128
    if Q == 128:
        ref = mo.direct_dft(smp["u"], smp["v"], 0 * us, smp["val"], xs.ravel(), ys.ravel(), n, n, cell).reshape(n, n)
        err = np.abs(im.dirty()[0][0] - ref.real) / np.abs(ref.real).max()
        assert err[_inner(n, 0.5)].max() < 2e-2


# ------------------------------------------------------------------ P5: PSWF table
@pytest.mark.parametrize("S", [5, 6, 7, 9])
def test_P5_pswf_satisfies_its_integral_eigen_equation(S):
    """psi is an eigenfunction of the finite Fourier transform: Int_{-1}^{1} psi(t) e^{i c x t} dt = mu psi(x)."""
    c = np.pi * S / 2
    xg, wg = np.polynomial.legendre.leggauss(200)
    psi_t = mo.pswf(xg, c)
    x = np.linspace(0.0, 1.0, 41)
    lhs = (np.exp(1j * c * x[:, None] * xg[None, :]) * psi_t[None, :]) @ wg
    assert np.abs(lhs.imag).max() < 1e-12
    mu = lhs.real[0]                                  # psi(0) = 1
    np.testing.assert_allclose(lhs.real / mu, mo.pswf(x, c), atol=2e-9)


def test_P5_pswf_matches_eigenvector_of_discretised_sinc_operator():
    """Independent construction: psi_0 is the top eigenfunction of the sinc kernel sin(c(x-t))/(pi(x-t)) on [-1,1]."""
    c = 3.5 * np.pi
    xg, wg = np.polynomial.legendre.leggauss(120)
    d = xg[:, None] - xg[None, :]
    with np.errstate(invalid="ignore", divide="ignore"):
        K = np.where(d == 0, c / np.pi, np.sin(c * d) / (np.pi * d))
    sw = np.sqrt(wg)
    lam, vec = np.linalg.eigh(sw[:, None] * K * sw[None, :])
    psi = vec[:, -1] / sw
    i0 = np.argmin(np.abs(xg))
    # normalise through interpolation-free ratio: compare shape psi(x)/psi(x_i0)
    ref = mo.pswf(xg, c) / mo.pswf(xg[i0], c)
    np.testing.assert_allclose(psi / psi[i0], ref, atol=1e-8)


def test_P5_table_shape_symmetry_monotone_and_corrector_self_transform():
    S, Q, n = 7, 128, 512
    T = mo.table_pswf(S, Q)
    assert T.shape == (S * Q + 1,)
    assert T[S * Q // 2] == pytest.approx(1.0, abs=1e-14)
    np.testing.assert_allclose(T, T[::-1], atol=1e-14)
    assert np.all(np.diff(T[S * Q // 2:]) < 0)
    assert 1.5e-4 < T[0] < 2.5e-4                         # C(S/2) = psi(1)/psi(0), small but non-zero
    # table entries at integer cell offsets equal psi(2 D / 7)
    for D in (1, 2, 3):
        assert T[S * Q // 2 + D * Q] == pytest.approx(float(mo.pswf(2 * D / 7, 3.5 * np.pi)), abs=1e-14)
    # O5 corrector of the PSWF table is the PSWF itself: cx(l)/cx(0) = psi(2 l)  (self-transform, R8)
    cx = mo.corrector(T, S, Q, n)
    ell = (np.arange(n) - n / 2) / n
    np.testing.assert_allclose(cx / cx[n // 2], mo.pswf(2 * ell, 3.5 * np.pi), atol=2e-6)


def test_P5_gauss_table_and_corrector_closed_form():
    S, Q, n, a = 7, 8, 256, 1.55
    T = mo.table_gauss(S, Q, a)
    x = (np.arange(S * Q + 1) - S * Q / 2) / Q
    np.testing.assert_allclose(T, np.exp(-x * x / (a * a)), rtol=1e-15)
    # FT of exp(-(x/a)^2) is a sqrt(pi) exp(-(pi a l)^2); truncation at +-3.5 (C = 6e-3 there) costs ~4e-3 of 2.75
    cx = mo.corrector(T, S, Q, n)
    ell = (np.arange(n) - n / 2) / n
    np.testing.assert_allclose(cx, a * np.sqrt(np.pi) * np.exp(-(np.pi * a * ell) ** 2), atol=6e-3)


# ------------------------------------------------------------------ P6: indexing
def test_P6_single_visibility_on_lattice_point_and_half_cell_tie():
    n, cell, S, Q = 64, 60.0, 7, 8
    su = n * cell * ARCSEC
    f = np.array([1.0e9])
    lam = C / f[0]
    T = mo.table_gauss(S, Q)
    # exactly on a lattice point (up = 32 + 5) and exactly on a half-cell tie (up = 32 + 5.5); f64 metres are
    # searched ulp by ulp so that O1's own arithmetic lands exactly on the target (O1 accepts any float input)
    for du, exp_iu, exp_ru in ((5.0, 37, 0), (5.5, 38, -Q // 2)):
        um = du / su * lam
        for _ in range(64):
            if um * (f[0] / C) * su + n / 2 == n / 2 + du:
                break
            um = np.nextafter(um, np.inf if um * (f[0] / C) * su + n / 2 < n / 2 + du else -np.inf)
        assert um * (f[0] / C) * su + n / 2 == n / 2 + du
        uvw = np.array([[um, 0.0, 0.0]], np.float64)
        smp = mo.coordinates(uvw, f, np.array([2 + 1j]), np.array([1.5]), n, n, cell, Q, S)
        assert smp["iu0"][0] == exp_iu and smp["ru"][0] == exp_ru      # tie -> phase -Q/2 of the NEXT cell (R4)
    # footprint of the on-lattice sample = outer product of integer-offset kernel values, nowhere else
    im = mo.Imager(n, n, cell, S, Q, "gauss")
    smp = mo.coordinates(np.zeros((1, 3), np.float32), f, np.array([2 + 1j]), np.array([1.5]), n, n, cell, Q, S)
    assert smp["iu0"][0] == 32 and smp["ru"][0] == 0 and smp["iv0"][1] == 32
    G, Gw = mo.grid(smp, T, S, Q, n, n)
    k1 = np.exp(-(np.arange(-3, 4) / 1.55) ** 2)
    foot = np.outer(k1, k1)
    exp = np.zeros((n, n), complex)
    exp[29:36, 29:36] = foot * 1.5 * ((2 + 1j) + (2 - 1j))          # primary + conjugate both at the centre
    np.testing.assert_allclose(G[0], exp, atol=1e-15)
    expw = np.zeros((n, n)); expw[29:36, 29:36] = foot * 3.0
    np.testing.assert_allclose(Gw[0], expw, atol=1e-15)


def test_P6_table_index_is_cell_minus_sample_distance():
    """T[jx*Q - ru + S*Q/2] is the kernel at (cell - sample) = jx - ru/Q; check with a sample shifted by +3/8 cell."""
    n, cell, S, Q = 64, 60.0, 7, 8
    su = n * cell * ARCSEC
    f = np.array([1.0e9]); lam = C / f[0]
    uvw = np.array([[(4 + 3 / 8) / su * lam, 0.0, 0.0]], np.float32)
    smp = mo.coordinates(uvw, f, np.array([1 + 0j]), np.array([1.0]), n, n, cell, Q, S)
    assert smp["iu0"][0] == 36 and smp["ru"][0] == 3
    assert smp["iu0"][1] == 28 and smp["ru"][1] == -3
    G, _ = mo.grid({k: (v[:1] if isinstance(v, np.ndarray) else v) for k, v in smp.items()}, mo.table_gauss(S, Q), S, Q, n, n)
    row = G[0, 32, 33:40].real
    np.testing.assert_allclose(row, np.exp(-((np.arange(33, 40) - (36 + 3 / 8)) / 1.55) ** 2), atol=1e-15)


# ------------------------------------------------------------------ P7: sign and axis conventions
def test_P7_offcentre_point_source_lands_on_its_pixel_not_its_mirror():
    n, cell = 64, 60.0
    uvw, f, _, wt = _tiny(7, 80, n, cell)
    x0, y0 = 41, 25
    l0, m0 = (x0 - n / 2) * cell * ARCSEC, (y0 - n / 2) * cell * ARCSEC
    il = f / C
    u, v = uvw[:, 0].astype(np.float64) * il, uvw[:, 1].astype(np.float64) * il
    vis = np.exp(-2j * np.pi * (u * l0 + v * m0))
    im = mo.Imager(n, n, cell, 7, 128, "pswf")
    smp = im.grid(uvw, f, vis, wt)           # complex128 vis: no fp32 rounding of V
    ys, xs = np.mgrid[0:n, 0:n]
    ref = mo.direct_dft(smp["u"], smp["v"], smp["w"], smp["val"], xs.ravel(), ys.ravel(), n, n, cell).real.reshape(n, n)
    sw = im.stats["sum_weights"]
    assert ref[y0, x0] == pytest.approx(sw, rel=1e-12)
    assert np.unravel_index(np.argmax(ref), ref.shape) == (y0, x0)
    assert ref[n - y0, n - x0] < 0.9 * sw
    d = im.dirty()[0][0]
    assert np.unravel_index(np.argmax(d), d.shape) == (y0, x0)
    assert d[y0, x0] == pytest.approx(sw, rel=5e-3)


# ------------------------------------------------------------------ P8: linearity / accumulation
def test_P8_accumulation_linearity_permutation():
    n, cell = 64, 60.0
    uvw, f, vis, wt = _tiny(8, 50, n, cell)
    a = mo.Imager(n, n, cell, 7, 128); a.grid(uvw, f, vis, wt)
    b = mo.Imager(n, n, cell, 7, 128); b.grid(uvw[:20], f[:20], vis[:20], wt[:20]); b.grid(uvw[20:], f[20:], vis[20:], wt[20:])
    np.testing.assert_allclose(a.G, b.G, atol=1e-13 * np.abs(a.G).max())
    assert a.stats == pytest.approx(b.stats)
    c = mo.Imager(n, n, cell, 7, 128); c.grid(uvw, f, vis, 2.0 * wt)        # power of two: exact in the fp32 weight
    np.testing.assert_allclose(c.G, 2.0 * a.G, rtol=1e-12, atol=1e-13 * np.abs(a.G).max())
    perm = np.random.default_rng(0).permutation(50)
    d = mo.Imager(n, n, cell, 7, 128); d.grid(uvw[perm], f[perm], vis[perm], wt[perm])
    np.testing.assert_allclose(a.G, d.G, atol=1e-13 * np.abs(a.G).max())


# ------------------------------------------------------------------ P9: conservation
def test_P9_sum_of_grid_equals_sum_of_sample_row_sums():
    fr = synth.make_frame(1)
    p = fr.params
    im = mo.Imager(p.n, p.n, p.cell_arcsec, p.support, p.oversample, p.kernel)
    smp = im.grid(fr.uvw_m, fr.freq_hz, fr.vis, fr.weight)
    S, Q, T = p.support, p.oversample, im.T
    j = np.arange(-3, 4)
    rsx = T[j[None, :] * Q - smp["ru"][:, None] + S * Q // 2].sum(axis=1)
    rsy = T[j[None, :] * Q - smp["rv"][:, None] + S * Q // 2].sum(axis=1)
    assert im.G.sum() == pytest.approx((smp["val"] * rsx * rsy).sum(), rel=1e-12)
    assert im.Gw.sum() == pytest.approx((smp["wt"] * rsx * rsy).sum(), rel=1e-12)


# ------------------------------------------------------------------ P10: O4 conventions
@pytest.mark.parametrize("ny,nx", [(8, 8), (12, 8), (16, 20)])
def test_P10_transform_is_the_centred_unnormalised_inverse_dft(ny, nx):
    rng = np.random.default_rng(10)
    G = rng.standard_normal((ny, nx)) + 1j * rng.standard_normal((ny, nx))
    np.testing.assert_allclose(mo.transform(G), mo.transform_bruteforce(G), atol=1e-12 * nx * ny)
    # a single unit cell at (iv, iu) gives the plane wave exp(+2 pi i [(iu-nx/2)(x-nx/2)/nx + ...])
    G = np.zeros((ny, nx), complex); G[ny // 2 + 1, nx // 2 + 2] = 1.0
    y, x = np.mgrid[0:ny, 0:nx]
    np.testing.assert_allclose(mo.transform(G), np.exp(2j * np.pi * (2 * (x - nx // 2) / nx + 1 * (y - ny // 2) / ny)), atol=1e-12)


# ------------------------------------------------------------------ P11: w-mode
def _wsetup(n=128, cell=80.0, P=8, w_max=19900.0, Q=16):
    im = mo.Imager(n, n, cell, 7, Q, "pswf")
    im.set_wplanes(P, w_max)
    return im


def test_P11_plane0_kernel_is_the_pswf_table_and_zero_w_reduces_to_2d():
    n, cell, Q = 128, 80.0, 16
    fov = n * cell * ARCSEC
    k0 = mo.table_wkernel(7, Q, 0.0, fov)
    np.testing.assert_allclose(k0.imag, 0.0, atol=1e-13)
    np.testing.assert_allclose(k0.real, mo.table_pswf(7, Q), atol=2e-9)      # k_0(D) = psi(2D/7)/psi(0)
    np.testing.assert_allclose(mo.table_wkernel(9, Q, -800.0, fov), np.conj(mo.table_wkernel(9, Q, 800.0, fov)), atol=1e-15)
    uvw, f, vis, wt = synth.random_visibilities(11, 60, n, cell, margin_cells=20)
    a = mo.Imager(n, n, cell, 7, Q, "pswf"); a.grid(uvw, f, vis, wt)
    b = _wsetup(n, cell, 8, 19900.0, Q); b.grid(uvw, f, vis, wt)
    np.testing.assert_allclose(b.G, a.G, atol=1e-8 * np.abs(a.G).max())
    np.testing.assert_allclose(b.Gw.real, a.Gw, atol=1e-8 * a.Gw.max())
    np.testing.assert_allclose(b.Gw.imag, 0.0, atol=1e-13 * a.Gw.max())


def test_P11_wplane_layout_supports_span_7_to_31_for_cfg5():
    wc, S = mo.wplane_layout(4096, 2.5, 32, 19900.0)
    assert S[0] == 7 and S[-1] == 31 and np.all(np.diff(S) >= 0) and np.all(S % 2 == 1)
    assert wc[0] == 0 and wc[-1] == pytest.approx(19900.0)


def test_P11_offcentre_point_source_with_w_phases():
    """(I)-with-w returns sum_weights at the source pixel; w-projection (II) recovers it inside the solar-disk
    region up to plane quantisation + Fresnel + truncation error, while the 2-D path visibly fails."""
    n, cell, Q, P, w_max = 128, 80.0, 16, 16, 19900.0
    uvw, f, _, wt = synth.random_visibilities(12, 150, n, cell, margin_cells=20, w_max_lambda=w_max)
    x0, y0 = 64 + 9, 64 - 7                                   # ~15' from the centre: inside the 16' solar disk
    l0, m0 = (x0 - n / 2) * cell * ARCSEC, (y0 - n / 2) * cell * ARCSEC
    il = f / C
    u, v, w = (uvw[:, k].astype(np.float64) * il for k in range(3))
    vis = np.exp(-2j * np.pi * (u * l0 + v * m0 + w * (np.sqrt(1 - l0 * l0 - m0 * m0) - 1)))
    im = _wsetup(n, cell, P, w_max, Q)
    smp = im.grid(uvw, f, vis, wt)
    sw = im.stats["sum_weights"]
    exact = mo.direct_dft(smp["u"], smp["v"], smp["w"], smp["val"], [x0], [y0], n, n, cell, use_w=True)[0]
    assert exact.real == pytest.approx(sw, rel=1e-12) and abs(exact.imag) < 1e-9 * sw
    d = im.dirty()[0][0]
    assert np.abs(im.dirty()[1][0].imag).max() < 1e-10 * sw          # Hermitian also in w-mode -> real image
    assert d[y0, x0] == pytest.approx(sw, rel=3e-2)
    flat = mo.Imager(n, n, cell, 7, Q, "pswf"); flat.grid(uvw, f, vis, wt)
    assert flat.dirty()[0][0][y0, x0] < 0.8 * sw                      # ignoring w smears the source


def test_P12_small_w_2d_and_w_paths_agree_within_phase_bound():
    """|pi (l^2+m^2) w| < 0.1: with w <= 1.5 k-lambda the two paths agree over the disk to that phase error."""
    n, cell, Q = 128, 80.0, 16
    uvw, f, _, wt = synth.random_visibilities(13, 100, n, cell, margin_cells=20, w_max_lambda=1500.0)
    x0, y0 = 64 + 8, 64 + 6
    l0, m0 = (x0 - 64) * cell * ARCSEC, (y0 - 64) * cell * ARCSEC
    il = f / C
    u, v, w = (uvw[:, k].astype(np.float64) * il for k in range(3))
    vis = np.exp(-2j * np.pi * (u * l0 + v * m0 + w * (np.sqrt(1 - l0 * l0 - m0 * m0) - 1)))
    flat = mo.Imager(n, n, cell, 7, Q, "pswf"); flat.grid(uvw, f, vis, wt)
    sw = flat.stats["sum_weights"]
    phase = np.pi * (l0 * l0 + m0 * m0) * 1500.0
    assert phase < 0.1
    assert flat.dirty()[0][0][y0, x0] == pytest.approx(sw, rel=phase ** 2 / 2 + 2e-3)
