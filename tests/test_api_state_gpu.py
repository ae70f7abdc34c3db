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
