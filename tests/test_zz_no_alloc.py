"""-m gpu test of muser_histogram_static, the allocation-free entry point (include/muser.h).

Some users of this library cannot allocate device memory while they run: a monitoring loop that images every 3 ms frame
must not take the device-wide synchronisation of cudaMalloc / cudaFree, and a process that shares its GPU with a framework
whose caching allocator already owns the HBM may see cudaMalloc fail outright.  For them the library offers the own-range
image histogram (the 2000-range histogram the paper feeds to its GMM) without a handle: its scratch -- one
minimum / maximum slot per image -- is a fixed __device__ array inside libmuser.so instead of handle memory.

What is checked here: the new entry point gives, bin by bin, the histogram of the existing handle-based path
(muser_dirty with the peak search on, then muser_histogram with lo >= hi) on the same device image; integers, so the
tolerance is equality, as in test_next_gpu.py.  Two calls in a row on one stream: the second image has a much narrower
value range than the first, so slots left over from the first call (the array is shared and keeps its contents) would
put its pixels into the wrong bins if the call did not clear them.  Sizes beyond MUSER_STATIC_MAX_GRIDS are refused.

The file is named test_zz_* so that pytest collects it after every other test: with -x a failure here hides nothing.  It
passes both alone in a fresh process (the first call then does the per-device set-up) and after the other tests."""
import numpy as np
import pytest

from paper_1712_06913_b200 import binding
from inputs import synth

import gpu_util as gu

pytestmark = pytest.mark.gpu

NBINS = 2000


def _existing_path_histograms(im, uvw, freq, vis, wt, gid, ngrids, ny, nx):
    """Dirty images of one batch and their own-range histograms through the handle (the path that exists already)."""
    import torch
    im.reset()
    im.grid_batched(gu.to_dev(uvw), gu.to_dev(freq), gu.to_dev(vis), gu.to_dev(wt), gu.to_dev(gid))
    d = torch.empty((ngrids, ny, nx), device="cuda")
    im.dirty(d)
    hist = torch.empty((ngrids, NBINS), dtype=torch.int32, device="cuda")
    im.histogram(d, NBINS, 0.0, 0.0, hist)
    torch.cuda.synchronize()
    return d, hist


def test_static_histogram_equals_the_handle_path_on_two_calls_in_a_row():
    import torch
    nx, ny, ngrids, cell, Q, nvis = 256, 512, 3, 30.0, 16, 3000
    uvw, freq, vis, wt = synth.random_visibilities(907, nvis, min(nx, ny), cell * max(nx, ny) / min(nx, ny), margin_cells=6.0)
    gid = (np.arange(nvis) % ngrids).astype(np.int32)
    bright = (vis * 0.05 + 1.0).astype(np.complex64)            # wide range: a point source well above the noise
    faint = (vis * 1e-3).astype(np.complex64)                   # narrow range, inside the first image's range
    im = gu.make_imager(nx, cell, 7, Q, ngrids=ngrids, ny=ny)
    try:
        im.set_peak_search(True)
        d1, ref1 = _existing_path_histograms(im, uvw, freq, bright, wt, gid, ngrids, ny, nx)
        d2, ref2 = _existing_path_histograms(im, uvw, freq, faint, wt, gid, ngrids, ny, nx)
    finally:
        im.destroy()
    assert float(d2.max()) < 0.5 * float(d1.max())             # the two calls need different slots' contents
    out1 = torch.full((ngrids, NBINS), -1, dtype=torch.int32, device="cuda")
    out2 = torch.full((ngrids, NBINS), -1, dtype=torch.int32, device="cuda")
    binding.histogram_static(d1, NBINS, out1)                   # two calls back to back on the current stream,
    binding.histogram_static(d2, NBINS, out2)                   # no synchronisation between them
    torch.cuda.synchronize()
    assert torch.equal(out1, ref1)
    assert torch.equal(out2, ref2)                              # stale slots of call 1 would shift every bin here
    assert int(out1.sum()) == ngrids * ny * nx and int(out2.sum()) == ngrids * ny * nx
    # the same two images once more, in the other order: every call starts from cleared slots
    binding.histogram_static(d2, NBINS, out1)
    binding.histogram_static(d1, NBINS, out2)
    torch.cuda.synchronize()
    assert torch.equal(out1, ref2) and torch.equal(out2, ref1)


def test_static_histogram_refuses_what_does_not_fit_the_static_scratch():
    import torch
    n_over = binding.MUSER_STATIC_MAX_GRIDS + 1
    img = torch.zeros((n_over, 16), device="cuda")
    hist = torch.full((n_over, 8), 7, dtype=torch.int32, device="cuda")
    with pytest.raises(binding.MuserError) as e:
        binding.histogram_static(img, 8, hist)
    assert e.value.code == binding.MUSER_EINVAL and "MUSER_STATIC_MAX_GRIDS" in str(e.value)
    torch.cuda.synchronize()
    assert int(hist.min()) == 7 and int(hist.max()) == 7        # nothing was enqueued
    with pytest.raises(binding.MuserError):
        binding.histogram_static(img[:2], 8193, hist)
    # the maximum itself is accepted; a constant image goes to bin 0, an image without finite pixels is not counted
    img = torch.zeros((binding.MUSER_STATIC_MAX_GRIDS, 16), device="cuda")
    img[1] = float("nan")
    img[2, :5] = 3.0
    hist = torch.empty((binding.MUSER_STATIC_MAX_GRIDS, 8), dtype=torch.int32, device="cuda")
    binding.histogram_static(img, 8, hist)
    torch.cuda.synchronize()
    h = hist.cpu().numpy()
    assert h[0].tolist() == [16, 0, 0, 0, 0, 0, 0, 0]
    assert h[1].sum() == 0
    assert h[2].tolist() == [11, 0, 0, 0, 0, 0, 0, 5]
    assert (h[3:, 0] == 16).all() and (h[3:, 1:] == 0).all()
