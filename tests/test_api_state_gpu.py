"""-m gpu tests of handle state that earlier suites did not pin: the 2x-beam child follows later set_* calls on its parent and
is gridded by the host-buffer entry point, w mode is refused while it is on, and the own-range histogram refuses to run
before a dirty image exists.  Expected values come from the oracle (gates of DESIGN.md R9)."""
import numpy as np
import pytest

from oracle import muser_oracle as mo
from oracle import oracle_c as oc
from paper_1712_06913_b200 import binding
from inputs import synth

import gpu_util as gu

pytestmark = pytest.mark.gpu


def _oracle_beam2x(fr, T):
    p = fr.params
    n2 = 2 * p.n
    _, Gw2, st2 = oc.grid(fr.uvw_m, fr.freq_hz, fr.vis, fr.weight, n2, n2, p.cell_arcsec, p.oversample, p.support, T)
    _, cor, *_ = gu.oracle_images(Gw2.astype(np.complex128), Gw2, T, p.support, p.oversample)
    c2 = mo.corrector(T, p.support, p.oversample, n2)
    box = gu.inner_box(n2, c2)[:, None] & gu.inner_box(n2, c2)[None, :]
    return cor[0], box


@pytest.mark.parametrize("strategy", [binding.MUSER_STRATEGY_OWNER, binding.MUSER_STRATEGY_TILED])
def test_beam2x_follows_set_kernel_and_set_strategy_and_is_gridded_by_frame_host(strategy):
    import torch
    fr = synth.make_frame(1)
    p = fr.params
    im = binding.Imager(p.n, p.n, p.cell_arcsec, p.support, p.oversample)       # PSWF, AUTO
    try:
        im.set_psf2x(True)
        im.set_kernel(binding.MUSER_KERNEL_GAUSS, 0.0)          # after the child exists: must reach it
        im.set_strategy(strategy)
        T = mo.table_gauss(p.support, p.oversample)
        want, box = _oracle_beam2x(fr, T)
        tol = gu.IMG_TOL * np.abs(want[box]).max()
        b2 = torch.empty((1, 2 * p.n, 2 * p.n), device="cuda")
        # device-pointer path
        im.reset()
        im.grid(gu.to_dev(fr.uvw_m), gu.to_dev(fr.freq_hz), gu.to_dev(fr.vis), gu.to_dev(fr.weight))
        im.psf2x(b2)
        torch.cuda.synchronize()
        assert np.abs(b2.cpu().numpy().astype(np.float64)[0] - want)[box].max() <= tol
        # host-buffer path: resets and grids the child too
        b2.zero_()
        img = np.empty((1, p.n, p.n), np.float32)
        beam = np.empty((1, p.n, p.n), np.float32)
        im.frame_host(fr.uvw_m, fr.freq_hz, fr.vis, fr.weight, None, img, beam)
        im.psf2x(b2)
        torch.cuda.synchronize()
        got = b2.cpu().numpy().astype(np.float64)[0]
        assert np.abs(got).max() > 0
        assert np.abs(got - want)[box].max() <= tol
        # w mode is 2-D-beam-less: refused while the 2x beam is on, accepted after it is switched off
        with pytest.raises(binding.MuserError) as e:
            im.set_wplanes(np.array([0.0, 50.0]), np.array([7, 9]))
        assert e.value.code == binding.MUSER_EUNSUPPORTED
        im.set_psf2x(False)
        im.set_wplanes(np.array([0.0, 50.0]), np.array([7, 9]))
    finally:
        im.destroy()


def test_own_range_histogram_needs_a_dirty_image_first():
    import torch
    n = 256
    uvw, freq, vis, wt = synth.random_visibilities(5, 500, n, 30.0, margin_cells=6.0)
    im = gu.make_imager(n, 30.0, 7, 16)
    try:
        d = torch.zeros((1, n, n), device="cuda")
        hist = torch.empty((1, 100), dtype=torch.int32, device="cuda")
        with pytest.raises(binding.MuserError) as e:
            im.histogram(d, 100, 0.0, 0.0, hist)                # peak search off
        assert e.value.code == binding.MUSER_ESTATE
        im.set_peak_search(True)
        with pytest.raises(binding.MuserError) as e:
            im.histogram(d, 100, 0.0, 0.0, hist)                # on, but no dirty image yet
        assert e.value.code == binding.MUSER_ESTATE
        im.histogram(d, 100, -1.0, 1.0, hist)                   # a fixed range needs neither
        im.reset()
        im.grid(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt))
        im.dirty(d)
        im.histogram(d, 100, 0.0, 0.0, hist)
        torch.cuda.synchronize()
        assert int(hist.sum()) == n * n
        im.set_batch(2)                                         # new grids, new slots: invalid again
        with pytest.raises(binding.MuserError):
            im.histogram(torch.zeros((2, n, n), device="cuda"), 100, 0.0, 0.0, torch.empty((2, 100), dtype=torch.int32, device="cuda"))
    finally:
        im.destroy()


@pytest.mark.parametrize("sub", [1, 3, 100])
def test_fft_subbatches_give_the_same_images(sub):
    """MUSER_TUNE_FFT_SUBBATCH runs rows -> columns over sub-batches of grids: the same kernels on the same grids.  The grids
    are re-gridded between the two runs (the only way to invalidate the cached row transform), and the order of the fp32 sums
    inside the gridder differs from run to run, so the images are compared un-corrected to 1e-5 of the peak (a wrong grid offset
    in a sub-batch would be an O(1) error); 7 grids, so 3 leaves a ragged tail.  The beam taken again from the cached row
    transform (column passes only, still per sub-batch) must be bit-identical."""
    import torch
    ngrids, n = 7, 256
    uvw, freq, vis, wt = synth.random_visibilities(31, 4000, n, 30.0, margin_cells=6.0)
    gid = (np.arange(4000) % ngrids).astype(np.int32)
    im = gu.make_imager(n, 30.0, 7, 16, ngrids=ngrids)
    try:
        im.set_peak_search(True)
        im.set_grid_correction(False)
        im.reset()
        im.grid_batched(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt), gu.to_dev(gid))
        d0, p0 = (torch.empty((ngrids, n, n), device="cuda") for _ in range(2))
        im.dirty_psf(d0, p0)
        torch.cuda.synchronize()
        peaks0 = im.get_peak()
        im.set_tuning(binding.MUSER_TUNE_FFT_SUBBATCH, sub)
        im.reset()
        im.grid_batched(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt), gu.to_dev(gid))
        d1, p1 = (torch.zeros((ngrids, n, n), device="cuda") for _ in range(2))
        im.dirty_psf(d1, p1)
        torch.cuda.synchronize()
        for g in range(ngrids):
            assert float((d0[g] - d1[g]).abs().max()) <= 1e-5 * float(d0[g].abs().max())
            assert float((p0[g] - p1[g]).abs().max()) <= 1e-5 * float(p0[g].abs().max())
        peaks1 = im.get_peak()
        for a, b in zip(peaks0, peaks1):
            assert a[1:3] == b[1:3] and abs(a[0] - b[0]) <= 1e-5 * abs(a[0])
        p2 = torch.zeros_like(p1)
        im.psf(p2)
        torch.cuda.synchronize()
        assert torch.equal(p2, p1)
    finally:
        im.destroy()
