"""Seeded synthetic MUSER-shaped inputs.

This module is the ONLY code shared by the CUDA path's tests/bench and the oracle's tests.
It holds none of the imaging method's arithmetic (no coordinates-to-grid mapping, no kernel
tables, no gridding, no FFT, no correction): it only fabricates *inputs* -- antenna layouts,
baseline uvw in metres, per-visibility frequencies, sky-model visibilities, weights -- with the
shapes and statistics of the instrument PAPER.md describes:

  * 40 / 60 antennas -> 780 / 1770 baselines              PAPER.md:53 (Table 1)
  * 16 channels x 25 MHz per 3 ms frame, dual polarisation PAPER.md:43,56,60
  * baselines ~4-8 m ... ~3 km
  * site latitude 42.211833333 deg                         PAPER.md:122 (sec. 3.2.2)
  * Sun ~32 arcmin across                                  PAPER.md:328 (units garbled there)
  * spiral-arm, centrally condensed uv coverage            PAPER.md:132 (Fig. 2 caption)

The paper's own observations are not available; these frames stand in for them.
Every constant below is a choice fixed for reproducibility.
"""
from __future__ import annotations

import dataclasses

import numpy as np
from scipy.special import j1

C_M_S = 299792458.0
ARCSEC = np.pi / 648000.0
ARCMIN = 60.0 * ARCSEC
LAT_DEG = 42.211833333
DEC_DEG = 20.0                  # BASELINE.json configs[0]
SIDEREAL_DAY_S = 86164.0905
SEED0 = 171206913


@dataclasses.dataclass
class ImagingParams:
    """Imaging parameters of a BASELINE.json config (cells for cfgs 2,4,5: SURVEY.md §8(c) Q11)."""
    n: int
    cell_arcsec: float
    support: int
    oversample: int
    kernel: str          # "gauss" | "pswf"
    nplanes: int = 0     # >0: w-projection (cfg 5)
    ngrids: int = 1


@dataclasses.dataclass
class Frame:
    cfg: int
    params: ImagingParams
    uvw_m: np.ndarray      # f32 [nvis,3] metres
    freq_hz: np.ndarray    # f64 [nvis]
    vis: np.ndarray        # c64 [nvis]
    weight: np.ndarray     # f32 [nvis]
    grid_id: np.ndarray | None = None   # i32 [nvis] (cfg 4)
    sources: list | None = None         # [(flux, l0, m0)], Gaussian components

    @property
    def nvis(self) -> int:
        return int(self.vis.shape[0])


PARAMS = {
    1: ImagingParams(256, 10.0, 7, 8, "gauss"),
    2: ImagingParams(512, 10.0, 7, 128, "pswf"),
    3: ImagingParams(1024, 2.5, 7, 128, "pswf"),
    4: ImagingParams(512, 5.0, 7, 128, "pswf"),
    5: ImagingParams(4096, 2.5, 7, 64, "pswf", nplanes=32),
}


def _streams(cfg: int):
    ss = np.random.SeedSequence([SEED0, cfg])
    return [np.random.default_rng(s) for s in ss.spawn(3)]   # layout, sources, noise


def antenna_layout(array: str, rng: np.random.Generator) -> np.ndarray:
    """Three-arm log spiral, local East/North/Up with Up = 0.  Returns [nant,3] f64 metres."""
    if array == "muser1":
        m, r_min, r_max, centre = 13, 10.0, 1500.0, True
    elif array == "muser2":
        m, r_min, r_max, centre = 20, 5.0, 3000.0, False
    else:
        raise ValueError(array)
    pos = []
    if centre:
        pos.append((0.0, 0.0, 0.0))
    jit = rng.standard_normal((3, m))
    for a in range(3):
        for i in range(m):
            r = r_min * (r_max / r_min) ** (i / (m - 1)) * (1.0 + 0.02 * jit[a, i])
            phi = 2.0 * np.pi * a / 3.0 + 1.5 * np.pi * i / (m - 1)
            pos.append((r * np.cos(phi), r * np.sin(phi), 0.0))
    return np.asarray(pos, dtype=np.float64)


def baselines(pos: np.ndarray) -> np.ndarray:
    i, j = np.triu_indices(pos.shape[0], k=1)
    return pos[i] - pos[j]


def enu_to_uvw(b_enu: np.ndarray, hour_angle_rad: float, dec_rad: float, lat_rad: float) -> np.ndarray:
    """Textbook ENU -> equatorial XYZ -> uvw rotation (metres)."""
    e, n, u = b_enu[:, 0], b_enu[:, 1], b_enu[:, 2]
    x = -np.sin(lat_rad) * n + np.cos(lat_rad) * u
    y = e
    z = np.cos(lat_rad) * n + np.sin(lat_rad) * u
    sh, ch = np.sin(hour_angle_rad), np.cos(hour_angle_rad)
    sd, cd = np.sin(dec_rad), np.cos(dec_rad)
    uu = sh * x + ch * y
    vv = -sd * ch * x + sd * sh * y + cd * z
    ww = cd * ch * x - cd * sh * y + sd * z
    return np.stack([uu, vv, ww], axis=1)


def draw_sources(rng: np.random.Generator, nsrc: int = 2):
    src = []
    for _ in range(nsrc):
        flux = rng.uniform(0.1, 1.0)
        r = 14.0 * ARCMIN * np.sqrt(rng.uniform())
        th = rng.uniform(0.0, 2.0 * np.pi)
        src.append((float(flux), float(r * np.cos(th)), float(r * np.sin(th))))
    return src


def sky_visibilities(u, v, w, sources, with_w: bool) -> np.ndarray:
    """Unit-flux uniform disk (radius 16') + Gaussian components (FWHM 1').  u,v,w in wavelengths (f64)."""
    q = np.hypot(u, v)
    x = 2.0 * np.pi * (16.0 * ARCMIN) * q
    with np.errstate(invalid="ignore", divide="ignore"):
        disk = np.where(x > 1e-12, 2.0 * j1(x) / x, 1.0)
    vis = disk.astype(np.complex128)
    fwhm = 1.0 * ARCMIN
    for flux, l0, m0 in sources:
        amp = flux * np.exp(-(np.pi ** 2) * fwhm ** 2 * q ** 2 / (4.0 * np.log(2.0)))
        ph = u * l0 + v * m0
        if with_w:
            ph = ph + w * (np.sqrt(1.0 - l0 * l0 - m0 * m0) - 1.0)
        vis = vis + amp * np.exp(-2j * np.pi * ph)
    return vis


def _assemble(cfg, array, hour_angles, freqs, npol, with_w, per_image_grid, noise_sigma=0.05):
    rng_layout, rng_src, rng_noise = _streams(cfg)
    pos = antenna_layout(array, rng_layout)
    b = baselines(pos)
    nbl = b.shape[0]
    sources = draw_sources(rng_src)
    lat, dec = np.deg2rad(LAT_DEG), np.deg2rad(DEC_DEG)
    nt, nch = len(hour_angles), len(freqs)
    uvw = np.empty((nt, npol, nch, nbl, 3), dtype=np.float32)
    for t, h in enumerate(hour_angles):
        uvw[t] = enu_to_uvw(b, h, dec, lat).astype(np.float32)[None, None]
    freq = np.broadcast_to(np.asarray(freqs, np.float64)[None, None, :, None], (nt, npol, nch, nbl))
    uvw = uvw.reshape(-1, 3)
    freq = np.ascontiguousarray(freq).reshape(-1)
    il = freq / C_M_S
    ul, vl, wl = (uvw[:, k].astype(np.float64) * il for k in range(3))
    vis = sky_visibilities(ul, vl, wl, sources, with_w)
    nvis = vis.shape[0]
    noise = rng_noise.standard_normal((nvis, 2)) * noise_sigma
    vis = (vis + noise[:, 0] + 1j * noise[:, 1]).astype(np.complex64)
    weight = np.ones(nvis, dtype=np.float32)
    grid_id = None
    if per_image_grid:
        g = np.arange(nt * npol * nch, dtype=np.int32)
        grid_id = np.ascontiguousarray(np.broadcast_to(g[:, None], (nt * npol * nch, nbl))).reshape(-1)
    return uvw, freq, vis, weight, grid_id, sources


def make_frame(cfg: int, *, nframes: int | None = None, nsnap: int | None = None) -> Frame:
    """Build the synthetic input of BASELINE.json configs[cfg-1].

    nframes (cfg 4) / nsnap (cfg 5) shrink the time axis for tests; None = the full config.
    """
    p = dataclasses.replace(PARAMS[cfg])
    if cfg == 1:
        out = _assemble(1, "muser1", [0.0], [1.7e9], 1, False, False)
    elif cfg == 2:
        out = _assemble(2, "muser1", [0.0], 0.4e9 + 25e6 * np.arange(16), 2, False, False)
    elif cfg == 3:
        out = _assemble(3, "muser2", [0.0], 2.0e9 + 25e6 * np.arange(16), 2, False, False)
    elif cfg == 4:
        nf = 1000 if nframes is None else int(nframes)
        hs = np.arange(nf) * 0.003 * 2.0 * np.pi / SIDEREAL_DAY_S
        out = _assemble(4, "muser2", hs, 2.0e9 + 25e6 * np.arange(16), 2, False, True)
        p.ngrids = nf * 32
    elif cfg == 5:
        ns = 300 if nsnap is None else int(nsnap)
        hs = np.deg2rad(np.linspace(-30.0, 30.0, ns)) if ns > 1 else np.array([np.deg2rad(-30.0)])
        out = _assemble(5, "muser2", hs, 2.0e9 + 25e6 * np.arange(16), 2, True, False)
    else:
        raise ValueError(f"cfg must be 1..5, got {cfg}")
    uvw, freq, vis, weight, grid_id, sources = out
    return Frame(cfg, p, uvw, freq, vis, weight, grid_id, sources)


def random_visibilities(seed: int, nvis: int, n: int, cell_arcsec: float, freq_hz: float = 1.0e9,
                        margin_cells: float = 6.0, w_max_lambda: float = 0.0):
    """Small generic test input: uniformly scattered uv points inside the grid, random complex V, weights in (0.5,1.5)."""
    rng = np.random.default_rng([SEED0, 99, seed])
    half = (n / 2 - margin_cells) / (n * cell_arcsec * ARCSEC)     # wavelengths
    lam = C_M_S / freq_hz
    uvw = np.zeros((nvis, 3), np.float32)
    uvw[:, 0] = (rng.uniform(-half, half, nvis) * lam).astype(np.float32)
    uvw[:, 1] = (rng.uniform(-half, half, nvis) * lam).astype(np.float32)
    if w_max_lambda > 0:
        uvw[:, 2] = (rng.uniform(-w_max_lambda, w_max_lambda, nvis) * lam).astype(np.float32)
    freq = np.full(nvis, freq_hz, np.float64)
    vis = (rng.standard_normal(nvis) + 1j * rng.standard_normal(nvis)).astype(np.complex64)
    weight = rng.uniform(0.5, 1.5, nvis).astype(np.float32)
    return uvw, freq, vis, weight
