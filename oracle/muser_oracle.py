"""CPU fp64 ORACLE for the MUSER dirty-imaging hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs may
import this module.  It shares no code, header, table generator or constant with the CUDA path under
`paper_1712_06913_b200/`; it never imports that package.  Everything is numpy/scipy fp64, written in the
order and notation of SURVEY.md §8(c) so that it can be checked against the paper by eye.

What the paper fixes (PAPER.md = /root/reference/PAPER.md, arXiv 1712.06913):
  * "Gridding is the convolution of the visibilities with a particular function, which resamples the
    visibilities to lie on a regular rectangular grid"                       PAPER.md:78  (sec. 2)
  * the GCF is a truncated spheroidal function (Schwab 1984)                  PAPER.md:136-138 (sec. 3.2.3)
  * "Inverse FFT is performed after gridding for generating dirty image"
  * dirty image "with the sun disk at the center"; outputs dirty image + dirty beam
                                                                              PAPER.md:254-256 (Alg. 1 l.19-21)
  * the grid is complex, row-major `iv*nu+iu`, Hermitian                      PAPER.md:216-228 (Alg. 1 l.1-6)
  * natural weighting multiplies by 1                                         PAPER.md:240-243 (Alg. 1 l.12-13)
  * the 2-D transform is the small-field limit of the 3-D (u,v,w) transform; phase error |pi(l^2+m^2)w|
                                                                              PAPER.md:74-76,126,204,328
  * w-projection is used when that error is not small                         PAPER.md:126 (sec. 3.2.2)
Everything the paper leaves open is read as DESIGN.md "Readings" R1..R21 (= SURVEY.md §8(c) Q1..Q21) says.

Two layers:
  (I)  the plain definition: direct-DFT dirty image / beam   -> `direct_dft`
  (II) the algorithm step by step: O1 coordinates -> O2 table -> O3 gridding -> O4 transform -> O5 correction
       (+ O6 w-projection planes)                            -> `coordinates`, `table_*`, `grid`, `transform`,
                                                                `corrector`, `dirty_image`
Pins (tests/test_oracle_*.py, all `-m "not gpu"`): P1..P16 of DESIGN.md for the path (P13..P16, tests/test_oracle_pins2.py:
keep / drop boundary, plane selection, flag rule and the fp32 bin decision, each by hand), N1..N4 (tests/test_oracle_next.py)
for the NEXT rows at the end of this file (channelised input, Hermitian half-plane, uniform weighting as the paper
prints it, phase correction, peak / histogram).  No function here is unpinned; what stays unpinned *by the paper* is
the identity of its own GCF coefficients and w-kernels (R2, R15).
"""
from __future__ import annotations

import numpy as np
from scipy import special as _sp

C_M_S = 299792458.0                 # speed of light, m/s
ARCSEC = np.pi / 648000.0           # rad per arcsec


# --------------------------------------------------------------------------- O2: tables
def pswf(eta, c):
    """Order-0, degree-0 angular prolate spheroidal function of the first kind, psi(eta), |eta|<=1,
    bandwidth parameter c, normalised psi(0)=1.  Library special function (scipy.special.pro_ang1);
    at |eta| = 1 the library returns NaN, so the limit eta -> 1-2^-53 is used (R2)."""
    eta = np.abs(np.asarray(eta, dtype=np.float64))
    eta = np.minimum(eta, 1.0 - 2.0 ** -53)
    val = _sp.pro_ang1(0, 0, c, eta)[0]
    return val / _sp.pro_ang1(0, 0, c, 0.0)[0]


def table_pswf(S: int, Q: int) -> np.ndarray:
    """O2, PSWF: T[t] = psi(2 x_t / S)/psi(0), x_t = (t - S*Q/2)/Q, t = 0..S*Q, c_psi = pi*S/2 (R2)."""
    t = np.arange(S * Q + 1, dtype=np.float64)
    x = (t - S * Q / 2.0) / Q
    return pswf(2.0 * x / S, np.pi * S / 2.0)


def table_gauss(S: int, Q: int, a: float = 1.55) -> np.ndarray:
    """O2, Gaussian: T[t] = exp(-(x_t/a)^2), a in cells (R3)."""
    t = np.arange(S * Q + 1, dtype=np.float64)
    x = (t - S * Q / 2.0) / Q
    return np.exp(-(x / a) ** 2)


def wplane_layout(n: int, cell_arcsec: float, nplanes: int, w_max: float):
    """O6 / R15: plane centres linear in |w|, wc[p] = p*w_max/(P-1); supports S_p = 7 + 2*round(wc*FOV^2/4)."""
    fov = n * cell_arcsec * ARCSEC
    wc = np.arange(nplanes, dtype=np.float64) * (w_max / (nplanes - 1) if nplanes > 1 else 0.0)
    supports = (7 + 2 * np.floor(wc * fov * fov / 4.0 + 0.5)).astype(np.int64)
    return wc, supports


_TAPER_CACHE = {}


def _taper_quadrature(nquad):
    """Gauss-Legendre nodes/weights on [-1/2, 1/2] and the taper A(l) = psi(2 l), c = 3.5 pi (memoised: the
    library PSWF routine is slow per point)."""
    if nquad not in _TAPER_CACHE:
        xg, wg = np.polynomial.legendre.leggauss(nquad)
        _TAPER_CACHE[nquad] = (0.5 * xg, 0.5 * wg, pswf(xg, 3.5 * np.pi))
    return _TAPER_CACHE[nquad]


def table_wkernel(S: int, Q: int, w: float, fov: float, nquad: int = 4096) -> np.ndarray:
    """O6 / R15: Fresnel-separable w-kernel, one axis, complex table of S*Q+1 entries:
        k_w(D) = Int_{-1/2}^{1/2} A(l) exp(-i pi w (l*FOV)^2) exp(-2 pi i D l) dl / Int A,   A(l) = psi(2 l), c = 3.5 pi
    evaluated with an nquad-point Gauss-Legendre rule on [-1/2, 1/2]."""
    ell, wq, A = _taper_quadrature(nquad)
    norm = np.sum(wq * A)
    chirp = A * np.exp(-1j * np.pi * w * (ell * fov) ** 2) * wq
    t = np.arange(S * Q + 1, dtype=np.float64)
    D = (t - S * Q / 2.0) / Q
    out = np.empty(S * Q + 1, dtype=np.complex128)
    for k0 in range(0, D.size, 256):
        d = D[k0:k0 + 256]
        out[k0:k0 + 256] = np.exp(-2j * np.pi * d[:, None] * ell[None, :]) @ chirp
    return out / norm


# --------------------------------------------------------------------------- O1: coordinates
def coordinates(uvw_m, freq_hz, vis, weight, nx, ny, cell_arcsec, Q, supports, wc=None, grid_id=None):
    """O1 (+ plane selection of O6).  Operation order is normative (R4).

    supports: int S (2-D mode) or array S_p per plane (w-mode, with wc = plane centres).
    Returns dict of per-SAMPLE arrays for kept samples (primary and conjugate interleaved: 2k, 2k+1)
    and the counters of muser_get_stats."""
    uvw_m = np.asarray(uvw_m)
    nvis = uvw_m.shape[0]
    f = np.asarray(freq_hz, dtype=np.float64)
    wt = np.asarray(weight).astype(np.float64)
    V = np.asarray(vis).astype(np.complex128)
    cell = cell_arcsec * ARCSEC
    su = nx * cell
    sv = ny * cell
    il = f / C_M_S
    ul = uvw_m[:, 0].astype(np.float64) * il
    vl = uvw_m[:, 1].astype(np.float64) * il
    wl = uvw_m[:, 2].astype(np.float64) * il
    with np.errstate(invalid="ignore"):
        finite = (np.isfinite(ul) & np.isfinite(vl) & np.isfinite(wl) & np.isfinite(wt)
                  & np.isfinite(V.real) & np.isfinite(V.imag) & np.isfinite(f))
        flagged = ~(finite & (wt > 0))
    wmode = wc is not None
    if wmode:
        wc = np.asarray(wc, np.float64)
        supports = np.asarray(supports, np.int64)
        aw = np.where(flagged, 0.0, np.abs(wl))
        plane = np.argmin(np.abs(aw[:, None] - wc[None, :]), axis=1)     # tie -> lower p (argmin picks first)
        h = (supports[plane] - 1) // 2
    else:
        plane = np.zeros(nvis, np.int64)
        h = np.full(nvis, (int(supports) - 1) // 2, np.int64)

    def cell_and_phase(c_lambda, scale, n):
        with np.errstate(invalid="ignore"):
            p = c_lambda * scale + n / 2
            i0 = np.floor(p + 0.5)
            fr = p - i0
            r = np.floor(fr * Q + 0.5)
        return i0, r

    ok = ~flagged
    samples = []
    for sgn in (1.0, -1.0):
        iu0, ru = cell_and_phase(np.where(ok, sgn * ul, 0.0), su, nx)
        iv0, rv = cell_and_phase(np.where(ok, sgn * vl, 0.0), sv, ny)
        inside = (iu0 >= h + 1) & (iu0 <= nx - 1 - h) & (iv0 >= h + 1) & (iv0 <= ny - 1 - h)
        samples.append((iu0, ru, iv0, rv, inside))
    kept = ok & samples[0][4] & samples[1][4]
    idx = np.nonzero(kept)[0]
    ns = 2 * idx.size
    out = {k: np.empty(ns, np.int64) for k in ("iu0", "iv0", "ru", "rv", "plane", "grid")}
    out["conj_kernel"] = np.empty(ns, bool)
    out["val"] = np.empty(ns, np.complex128)
    out["wt"] = np.empty(ns, np.float64)
    out["u"] = np.empty(ns, np.float64); out["v"] = np.empty(ns, np.float64); out["w"] = np.empty(ns, np.float64)
    gid = np.zeros(nvis, np.int64) if grid_id is None else np.asarray(grid_id, np.int64)
    for s, sgn in enumerate((1.0, -1.0)):
        iu0, ru, iv0, rv, _ = samples[s]
        sl = slice(s, ns, 2)
        out["iu0"][sl] = iu0[idx]; out["iv0"][sl] = iv0[idx]
        out["ru"][sl] = ru[idx]; out["rv"][sl] = rv[idx]
        out["plane"][sl] = plane[idx]; out["grid"][sl] = gid[idx]
        out["conj_kernel"][sl] = (sgn * wl[idx]) < 0
        out["val"][sl] = wt[idx] * (V[idx] if sgn > 0 else np.conj(V[idx]))
        out["wt"][sl] = wt[idx]
        out["u"][sl] = sgn * ul[idx]; out["v"][sl] = sgn * vl[idx]; out["w"][sl] = sgn * wl[idx]
    out["stats"] = dict(sum_weights=float(2.0 * wt[idx].sum()), n_gridded=int(idx.size),
                        n_dropped=int((ok & ~kept).sum()), n_flagged=int(flagged.sum()))
    return out


# --------------------------------------------------------------------------- O3 / O6: gridding
def grid(samples, tables, supports, Q, nx, ny, ngrids=1, wmode=False):
    """O3 (2-D: one real table) / O6 (w-mode: per-plane complex tables).  Sequential fp64 sums.
    Returns G [ngrids,ny,nx] complex128 and Gw ([ngrids,ny,nx] float64, complex128 in w-mode)."""
    G = np.zeros((ngrids, ny, nx), np.complex128)
    Gw = np.zeros((ngrids, ny, nx), np.complex128 if wmode else np.float64)
    if not wmode:
        tables = [np.asarray(tables, np.float64)]
        supports = [int(supports)]
    for s in range(samples["val"].shape[0]):
        p = int(samples["plane"][s])
        S = int(supports[p]); h = (S - 1) // 2
        T = tables[p]
        j = np.arange(-h, h + 1)
        kx = T[j * Q - int(samples["ru"][s]) + S * Q // 2]
        ky = T[j * Q - int(samples["rv"][s]) + S * Q // 2]
        if wmode and samples["conj_kernel"][s]:
            kx = np.conj(kx); ky = np.conj(ky)
        k2 = ky[:, None] * kx[None, :]
        iu0 = int(samples["iu0"][s]); iv0 = int(samples["iv0"][s]); g = int(samples["grid"][s])
        G[g, iv0 - h:iv0 + h + 1, iu0 - h:iu0 + h + 1] += k2 * samples["val"][s]
        Gw[g, iv0 - h:iv0 + h + 1, iu0 - h:iu0 + h + 1] += k2 * samples["wt"][s]
    return G, Gw


# --------------------------------------------------------------------------- O4: transform
def transform(G):
    """O4: F[y][x] = sum G[iv][iu] exp(+2 pi i[(iu-nx/2)(x-nx/2)/nx + (iv-ny/2)(y-ny/2)/ny]), unnormalised."""
    ny, nx = G.shape[-2:]
    return np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(G, axes=(-2, -1)), axes=(-2, -1)), axes=(-2, -1)) * (nx * ny)


def transform_bruteforce(G):
    """O4 written out as the double sum (tiny grids only) -- pins the fftshift conventions of `transform`."""
    ny, nx = G.shape
    x = np.arange(nx) - nx // 2
    y = np.arange(ny) - ny // 2
    Ex = np.exp(2j * np.pi * np.outer(x, x) / nx)     # [x, iu]
    Ey = np.exp(2j * np.pi * np.outer(y, y) / ny)     # [y, iv]
    return Ey @ G @ Ex.T


# --------------------------------------------------------------------------- O5: correction
def corrector(T, S, Q, n):
    """O5: c[x] = (1/Q) sum_t om_t T[t] cos(2 pi l_x x_t), l_x = (x-n/2)/n, trapezoid weights om_0=om_SQ=1/2.
    For a complex table the real part is used (plane-0 tables are real)."""
    T = np.real(np.asarray(T))
    t = np.arange(S * Q + 1, dtype=np.float64)
    xt = (t - S * Q / 2.0) / Q
    om = np.ones_like(t); om[0] = om[-1] = 0.5
    ell = (np.arange(n) - n / 2) / n
    return (np.cos(2.0 * np.pi * ell[:, None] * xt[None, :]) @ (om * T)) / Q


def dirty_image(G, cx, cy):
    """O4 + O5: dirty[y][x] = Re F[y][x] / (cx[x] cy[y]).  Also returns the un-corrected F."""
    F = transform(G)
    return F.real / (cy[:, None] * cx[None, :]), F


# --------------------------------------------------------------------------- (I): direct DFT
def direct_dft(u, v, w, val, xs, ys, nx, ny, cell_arcsec, use_w=False):
    """(I): I(l,m) = sum_s val_s exp(+2 pi i (u_s l + v_s m [+ w_s (sqrt(1-l^2-m^2) - 1)])) at pixels (xs, ys),
    l = (x-nx/2) cell, m = (y-ny/2) cell.  val_s = wt_s V_s (dirty) or wt_s (beam)."""
    cell = cell_arcsec * ARCSEC
    l = (np.asarray(xs, np.float64) - nx / 2) * cell
    m = (np.asarray(ys, np.float64) - ny / 2) * cell
    out = np.empty(l.shape[0], np.complex128)
    for k in range(l.shape[0]):
        ph = u * l[k] + v * m[k]
        if use_w:
            ph = ph + w * (np.sqrt(1.0 - l[k] ** 2 - m[k] ** 2) - 1.0)
        out[k] = np.sum(val * np.exp(2j * np.pi * ph))
    return out


# --------------------------------------------------------------------------- whole path (II)
class Imager:
    """Algorithm (II) end to end, mirroring the C-ABI call sequence (create / set_kernel / set_wplanes /
    grid / dirty / psf) so tests can drive both sides with the same inputs."""

    def __init__(self, nx, ny, cell_arcsec, support, oversample, kernel="pswf", gauss_a=1.55, ngrids=1):
        self.nx, self.ny, self.cell, self.S, self.Q, self.ngrids = nx, ny, cell_arcsec, support, oversample, ngrids
        self.T = table_pswf(support, oversample) if kernel == "pswf" else table_gauss(support, oversample, gauss_a)
        self.wc = None
        self.tables = None
        self.supports = None
        self.weighting = 0                       # 0 natural, 1 uniform (wgt_grid)
        self.offset = (0.0, 0.0)                 # phase-centre offset (dl, dm), NEXT-3
        self.reset()

    def set_wplanes(self, nplanes, w_max, tables=None, supports=None, wc=None):
        fov = self.nx * self.cell * ARCSEC
        if wc is None:
            self.wc, self.supports = wplane_layout(self.nx, self.cell, nplanes, w_max)
        else:
            self.wc, self.supports = np.asarray(wc, np.float64), np.asarray(supports, np.int64)
        if tables is None:
            tables = [table_wkernel(int(S), self.Q, float(w), fov) for S, w in zip(self.supports, self.wc)]
        self.tables = [np.asarray(t, np.complex128) for t in tables]
        self.reset()

    def reset(self):
        wmode = self.wc is not None
        self.G = np.zeros((self.ngrids, self.ny, self.nx), np.complex128)
        self.Gw = np.zeros((self.ngrids, self.ny, self.nx), np.complex128 if wmode else np.float64)
        self.cnt = np.zeros((self.ngrids, self.ny, self.nx), np.int64)
        self.stats = dict(sum_weights=0.0, n_gridded=0, n_dropped=0, n_flagged=0)

    def grid(self, uvw_m, freq_hz, vis, weight, grid_id=None, gridder=None):
        wmode = self.wc is not None
        if self.offset != (0.0, 0.0):
            vis = phase_correct(uvw_m, freq_hz, vis, *self.offset)
        smp = coordinates(uvw_m, freq_hz, vis, weight, self.nx, self.ny, self.cell, self.Q,
                          self.supports if wmode else self.S, self.wc, grid_id)
        gfun = grid if gridder is None else gridder
        G, Gw = gfun(smp, self.tables if wmode else self.T, self.supports if wmode else self.S, self.Q,
                     self.nx, self.ny, self.ngrids, wmode)
        self.G += G
        self.Gw += Gw
        self.cnt += hit_counts(smp, self.nx, self.ny, self.ngrids)
        for k, val in smp["stats"].items():
            self.stats[k] += val
        return smp

    def correctors(self):
        T0 = self.tables[0] if self.wc is not None else self.T
        S0 = int(self.supports[0]) if self.wc is not None else self.S
        return corrector(T0, S0, self.Q, self.nx), corrector(T0, S0, self.Q, self.ny)

    def weighted(self):
        """The grids after wgtGrid_kernel (identity in natural mode)."""
        return wgt_grid(self.G, self.cnt, self.weighting), wgt_grid(self.Gw, self.cnt, self.weighting)

    def dirty(self):
        cx, cy = self.correctors()
        Gv, _ = self.weighted()
        out = [dirty_image(Gv[g], cx, cy) for g in range(self.ngrids)]
        return np.stack([o[0] for o in out]), np.stack([o[1] for o in out])

    def psf(self):
        cx, cy = self.correctors()
        _, Gwv = self.weighted()
        out = [dirty_image(Gwv[g].astype(np.complex128), cx, cy) for g in range(self.ngrids)]
        return np.stack([o[0] for o in out]), np.stack([o[1] for o in out])


# =========================================================================== NEXT rows of SURVEY.md 8(f)
# --------------------------------------------------------------------------- NEXT-1: channelised input
def grid_rows_inputs(uvw_m, freq_hz, vis, weight):
    """NEXT-1 (a 3 ms frame is 16 channels x 2 polarisations of the SAME baselines).  Channelised layout:
    uvw_m [ntime][nrow][3] f32, freq_hz [nchan] f64, vis / weight [ntime][npol][nchan][nrow].  The method is unchanged:
    visibility (t, p, c, r) has coordinates uvw_m[t][r] * freq_hz[c] / c0, so this writes the loop out, in the order
    t, p, c, r, as the flat per-visibility arrays of O1 -- the result is DEFINED as the flat path's on these arrays."""
    uvw_m = np.asarray(uvw_m, np.float32)
    vis = np.asarray(vis)
    ntime, npol, nchan, nrow = vis.shape
    assert uvw_m.shape == (ntime, nrow, 3) and np.asarray(freq_hz).shape == (nchan,)
    uvw = np.empty((ntime, npol, nchan, nrow, 3), np.float32)
    f = np.empty((ntime, npol, nchan, nrow), np.float64)
    for t in range(ntime):
        for p in range(npol):
            for c in range(nchan):
                uvw[t, p, c] = uvw_m[t]
                f[t, p, c] = freq_hz[c]
    return (uvw.reshape(-1, 3), f.reshape(-1), np.ascontiguousarray(vis).reshape(-1),
            np.ascontiguousarray(np.asarray(weight, np.float32)).reshape(-1))


def rows_grid_ids(grid_id, ntime, npol, nchan, nrow, pols_split):
    """Per-visibility grid ids of the channelised call: grid_id is [ntime][nchan] (polarisations summed onto one grid)
    or [ntime][npol][nchan] (one grid per polarisation); None = everything onto grid 0."""
    if grid_id is None:
        return None
    g = np.asarray(grid_id, np.int64)
    g = g.reshape(ntime, npol, nchan) if pols_split else np.broadcast_to(g.reshape(ntime, 1, nchan), (ntime, npol, nchan))
    return np.ascontiguousarray(np.broadcast_to(g[..., None], (ntime, npol, nchan, nrow))).reshape(-1)


# --------------------------------------------------------------------------- NEXT-1b: Hermitian half-plane
def grid_halfplane(samples, tables, supports, Q, nx, ny, ngrids=1, wmode=False):
    """"half the grid (as the data is Hermitian)": O3/O6 restricted to grid rows iv >= ny/2.  Every sample
    (each visibility AND its conjugate, each with its own O1 coordinates) contributes the cells of its footprint that
    lie in those rows; rows below ny/2 stay zero.  `full_from_halfplane` rebuilds the rest."""
    G, Gw = grid(samples, tables, supports, Q, nx, ny, ngrids, wmode)
    G[:, :ny // 2, :] = 0
    Gw[:, :ny // 2, :] = 0
    return G, Gw


def full_from_halfplane(H):
    """Hermitian completion about the centre cell [ny/2][nx/2]: H[ny-y][nx-x] = conj H[y][x] for y in (ny/2, ny-1],
    x in [1, nx-1]; row 0 and column 0 have no mirror and are empty (drop rule R5)."""
    H = np.array(H)
    ny, nx = H.shape[-2:]
    y = np.arange(1, ny // 2)
    x = np.arange(1, nx)
    H[..., y[:, None], x[None, :]] = np.conj(H[..., (ny - y)[:, None], (nx - x)[None, :]])
    H[..., 0, :] = 0
    H[..., :ny // 2, 0] = 0
    return H


def image_from_halfplane(H):
    """Real image of a Hermitian grid given by its rows >= ny/2 only: O4 applied to the completed grid.  (A complex-
    to-real transform; written through the completion so that it can be checked by eye.)"""
    return transform(full_from_halfplane(H)).real


# --------------------------------------------------------------------------- NEXT-2: uniform weighting as printed
def hit_counts(samples, nx, ny, ngrids=1):
    """Integer hit-count grid `cnt` of Alg. 1 l.1: cnt[g][iv0][iu0] += 1 for every gridded sample (each
    visibility and its conjugate) at its NEAREST cell (reading R22: the paper does not print where cnt is filled)."""
    cnt = np.zeros((ngrids, ny, nx), np.int64)
    for s in range(samples["val"].shape[0]):
        cnt[int(samples["grid"][s]), int(samples["iv0"][s]), int(samples["iu0"][s])] += 1
    return cnt


def wgt_grid(Grd, cnt, mode):
    """wgtGrid_kernel of Alg. 1 l.1-16 over the whole grid: where cnt != 0 the cell is multiplied
    by wgt = 1/cnt (mode 1, uniform) or 1 (natural); cells with cnt == 0 are left alone.  The paper runs it on half
    the grid because the data are Hermitian; cnt is Hermitian too, so running it on every cell is the same thing.
    Applied to the visibility grid and, for a consistent beam, to the weight grid (R22)."""
    out = np.array(Grd)
    if mode == 1:
        nz = cnt != 0
        out[nz] = out[nz] * (1.0 / cnt[nz])
    return out


# --------------------------------------------------------------------------- NEXT-3: phase correction of visibilities
def phase_correct(uvw_m, freq_hz, vis, dl, dm):
    """Phase correction by a (RA, DEC) offset (PAPER.md:174 step 3, :286 Alg. 1 IMPROVED_CLEAN): the visibility of
    baseline (u, v) in wavelengths is multiplied by exp(+2 pi i (u dl + v dm)), which moves a source at direction
    cosines (dl, dm) to the phase centre (sign convention R7: the image is sum V exp(+2 pi i (u l + v m)))."""
    il = np.asarray(freq_hz, np.float64) / C_M_S
    ul = np.asarray(uvw_m)[:, 0].astype(np.float64) * il
    vl = np.asarray(uvw_m)[:, 1].astype(np.float64) * il
    return np.asarray(vis).astype(np.complex128) * np.exp(2j * np.pi * (ul * dl + vl * dm))


# --------------------------------------------------------------------------- NEXT-4: consumers of the dirty image
def image_peak(img):
    """Strength and position of the peak of the dirty map (Alg. 1 l.33/36): maximum value and its
    (y, x); on equal values the lowest flat index.  Also the minimum (the histogram's lower edge)."""
    img = np.asarray(img)
    k = int(np.argmax(img))
    return float(img.reshape(-1)[k]), k // img.shape[1], k % img.shape[1], float(img.min())


def image_histogram(img, nbins, lo, hi):
    """"the data from a dirty image is divided into 2000 ranges": nbins equal ranges of [lo, hi]
    (reading R23: lo, hi = the image's minimum and maximum unless the caller fixes them), bin = floor((v - lo) * (nbins /
    (hi - lo))), the value hi itself in the last bin, values outside [lo, hi] not counted.  The decision is taken in
    fp32, the precision of the image (both sides take it in the same precision)."""
    v = np.asarray(img, np.float32).reshape(-1)
    lo32, hi32 = np.float32(lo), np.float32(hi)
    scale = np.float32(nbins) / (hi32 - lo32)
    t = (v - lo32) * scale
    b = np.floor(t).astype(np.int64)
    ok = (v >= lo32) & (v <= hi32)
    b = np.minimum(b, nbins - 1)
    return np.bincount(b[ok], minlength=nbins).astype(np.int64)
