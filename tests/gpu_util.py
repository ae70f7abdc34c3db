"""Helpers shared by the -m gpu parity tests: drive the CUDA library through the binding and the oracle through
its own modules on the same seeded inputs, and compare with the tolerances of BASELINE.json's north_star
(grid relative L2 <= 1e-5; images max-abs <= 1e-4 of the peak, gated as DESIGN.md R9 says)."""
import numpy as np

from oracle import muser_oracle as mo
from oracle import oracle_c as oc
from paper_1712_06913_b200 import binding

GRID_TOL = 1e-5
IMG_TOL = 1e-4


def to_dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def make_imager(n, cell, S, Q, kernel="pswf", gauss_a=0.0, ngrids=1, strategy=binding.MUSER_STRATEGY_AUTO, ny=None):
    im = binding.Imager(n, n if ny is None else ny, cell, S, Q)
    if kernel == "gauss":
        im.set_kernel(binding.MUSER_KERNEL_GAUSS, gauss_a)
    if ngrids != 1:
        im.set_batch(ngrids)
    im.set_strategy(strategy)
    return im


def gpu_grids(im):
    import torch
    ng, ny, nx = im.ngrids, im.ny, im.nx
    G = torch.empty((ng, ny, nx, 2), dtype=torch.float32, device="cuda")
    Gw = torch.empty((ng, ny, nx, 2) if im.nplanes else (ng, ny, nx), dtype=torch.float32, device="cuda")
    im.get_grid(G, Gw)
    torch.cuda.synchronize()
    G = G.cpu().numpy().astype(np.float64)
    Gw = Gw.cpu().numpy().astype(np.float64)
    Gc = G[..., 0] + 1j * G[..., 1]
    Gwc = Gw[..., 0] + 1j * Gw[..., 1] if im.nplanes else Gw
    return Gc, Gwc


def gpu_images(im, correction=True):
    import torch
    ng, ny, nx = im.ngrids, im.ny, im.nx
    d = torch.empty((ng, ny, nx), dtype=torch.float32, device="cuda")
    p = torch.empty((ng, ny, nx), dtype=torch.float32, device="cuda")
    im.set_grid_correction(correction)
    im.dirty_psf(d, p)
    im.set_grid_correction(True)
    torch.cuda.synchronize()
    return d.cpu().numpy().astype(np.float64), p.cpu().numpy().astype(np.float64)


def rel_l2(a, b):
    den = np.sqrt(np.sum(np.abs(b) ** 2))
    num = np.sqrt(np.sum(np.abs(a - b) ** 2))
    return num / den if den > 0 else num


def oracle_table(kernel, S, Q, gauss_a=1.55):
    return mo.table_pswf(S, Q) if kernel == "pswf" else mo.table_gauss(S, Q, gauss_a if gauss_a > 0 else 1.55)


def oracle_images(G, Gw, T, S, Q):
    """O4 + O5 on [ng, ny, nx] grids: returns (uncorrected Re F, corrected) for the dirty image and the beam."""
    ny, nx = G.shape[-2:]
    cx, cy = mo.corrector(T, S, Q, nx), mo.corrector(T, S, Q, ny)
    Fd = mo.transform(G)
    Fp = mo.transform(Gw.astype(np.complex128))
    corr = cy[:, None] * cx[None, :]
    return Fd.real, Fd.real / corr, Fp.real, Fp.real / corr, max(np.abs(Fd.imag).max(), np.abs(Fp.imag).max())


# R9 gate region: the central 75% of each axis, further limited (for kernels wider than the S = 7 PSWF of the
# configs) to where the per-axis corrector has not fallen below its S = 7 value at the 75% edge, c(0.375)/c(0) =
# 0.0329 -- beyond that 1/(cx*cy) amplifies fp32 rounding past any fixed fraction of the peak.
CORR_FLOOR = 0.0329


def inner_box(n, corr=None, frac=0.75):
    c = np.arange(n) - n // 2
    box = np.abs(c) < frac * n / 2
    if corr is not None:
        box &= corr / corr[n // 2] >= CORR_FLOOR * (1 - 1e-6)
    return box


def check_images(im, G_or, Gw_or, T, S, Q, tol=IMG_TOL):
    """R9 gates: (i) un-corrected Re F over the full frame, (ii) corrected image over the central 75% box."""
    raw_d, cor_d, raw_p, cor_p, _ = oracle_images(G_or, Gw_or, T, S, Q)
    g_raw_d, g_raw_p = gpu_images(im, correction=False)
    g_cor_d, g_cor_p = gpu_images(im, correction=True)
    ny, nx = raw_d.shape[-2:]
    by, bx = inner_box(ny, mo.corrector(T, S, Q, ny)), inner_box(nx, mo.corrector(T, S, Q, nx))
    box = by[:, None] & bx[None, :]
    out = {}
    for name, o_raw, o_cor, g_raw, g_cor in (("dirty", raw_d, cor_d, g_raw_d, g_cor_d), ("psf", raw_p, cor_p, g_raw_p, g_cor_p)):
        for gi in range(o_raw.shape[0]):
            peak_raw = np.abs(o_raw[gi]).max()
            peak_box = np.abs(o_cor[gi][box]).max()
            e_raw = np.abs(g_raw[gi] - o_raw[gi]).max() / peak_raw if peak_raw > 0 else np.abs(g_raw[gi]).max()
            e_box = np.abs(g_cor[gi] - o_cor[gi])[box].max() / peak_box if peak_box > 0 else np.abs(g_cor[gi][box]).max()
            assert e_raw <= tol, f"{name}[{gi}] un-corrected full-frame error {e_raw:.3e} of peak"
            assert e_box <= tol, f"{name}[{gi}] corrected inner-75% error {e_box:.3e} of peak"
            out[(name, gi)] = (e_raw, e_box)
    return out


def run_case(uvw, freq, vis, wt, n, cell, S, Q, kernel="pswf", gauss_a=0.0, strategy=binding.MUSER_STRATEGY_AUTO,
             grid_id=None, ngrids=1, splits=1, images=True, item_size=0):
    """Grid on the GPU (optionally in `splits` accumulating calls) and in the oracle; assert parity; return both."""
    im = make_imager(n, cell, S, Q, kernel, gauss_a, ngrids, strategy)
    try:
        if item_size:
            im.set_tuning(binding.MUSER_TUNE_ITEM_SIZE, item_size)
        d = [to_dev(uvw), to_dev(freq), to_dev(vis), to_dev(wt)]
        dg = to_dev(np.asarray(grid_id, np.int32)) if grid_id is not None else None
        nvis = vis.shape[0]
        edges = np.linspace(0, nvis, splits + 1).astype(int)
        im.reset()
        for a, b in zip(edges[:-1], edges[1:]):
            if grid_id is None:
                im.grid(d[0][a:b], d[1][a:b], d[2][a:b], d[3][a:b])
            else:
                im.grid_batched(d[0][a:b], d[1][a:b], d[2][a:b], d[3][a:b], dg[a:b])
        G, Gw = gpu_grids(im)
        stats = im.get_stats()
        T = oracle_table(kernel, S, Q, gauss_a)
        G_or, Gw_or, st_or = oc.grid(uvw, freq, vis, wt, n, n, cell, Q, S, T, grid_id=grid_id, ngrids=ngrids)
        assert stats["n_gridded"] == st_or["n_gridded"]
        assert stats["n_dropped"] == st_or["n_dropped"]
        assert stats["n_flagged"] == st_or["n_flagged"]
        assert abs(stats["sum_weights"] - st_or["sum_weights"]) <= 1e-9 * max(1.0, st_or["sum_weights"])
        eg, ew = rel_l2(G, G_or), rel_l2(Gw, Gw_or)
        assert eg <= GRID_TOL, f"grid rel-L2 {eg:.3e}"
        assert ew <= GRID_TOL, f"weight-grid rel-L2 {ew:.3e}"
        res = dict(G=G, Gw=Gw, G_or=G_or, Gw_or=Gw_or, stats=stats, eg=eg, ew=ew)
        if images:
            res["img"] = check_images(im, G_or, Gw_or, T, S, Q)
        return res
    finally:
        im.destroy()
