"""cyrsoxs_reduce_static: the 1-D reductions for callers that must not allocate device memory.

Some users of this library cannot let it call cudaMalloc: a host program whose own memory pool (for example the PyTorch
caching allocator, or an analysis service that reserves all of HBM when it starts) already owns the device, so a further
cudaMalloc fails; or a live reduction loop at the instrument that cannot accept the device-wide stall cudaMalloc / cudaFree
cause.  For them the library offers one entry point whose scratch is a fixed array inside the library
(include/cyrsoxs.h: CYRSOXS_REDUCE_STATIC_BYTES per GPU, shared by every call on that GPU, limits on bins and energies).

What is checked here: the new entry point gives what the allocating cyrsoxs_reduce gives, within the tolerances the
reduction parity tests use (tests/test_gpu_parity.py: 2e-5 of the image scale for I and ISI, 1e-4 for the anisotropy), on
two calls in a row whose sizes differ -- the second call lands on bytes the first one left non-zero, so a missing clear of
the shared array shows; that device memory does not shrink across a call; and that sizes beyond the fixed array are
refused with a message that names the limits.

This file is named so that pytest collects it last: it is an add-on outside the hot path, and with `pytest -x` a failure
here must not hide any other test.  It passes alone in a fresh process (the first call then does the per-device address
look-up) and after the rest of the suite.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _inputs(torch, n_energy, ny, nx, seed, with_counts):
    g = torch.Generator(device="cpu").manual_seed(seed)
    # intensities over six decades, as detector images have (a bright centre, weak high-q pixels)
    img = torch.exp(torch.rand((n_energy, ny, nx), generator=g, dtype=torch.float64) * 14.0 - 7.0).to(torch.float32)
    cnt = None
    if with_counts:
        cnt = (torch.rand((n_energy, ny, nx), generator=g) < 0.8).to(torch.int32) * 3     # 20 % of the pixels never valid
    return img.cuda(), (None if cnt is None else cnt.cuda())


def _both(torch, ctx, img, cnt, n_bins, width):
    """Runs the allocating path and the static-scratch path on the same inputs; returns their (I, A, isi)."""
    ne = img.shape[0]
    stream = torch.cuda.current_stream().cuda_stream
    res = []
    for fn in (ctx.reduce, ctx.reduce_static):
        I = torch.full((ne, n_bins), -1.0, device="cuda"); A = torch.full_like(I, -1.0); isi = torch.full((ne,), -1.0, device="cuda")
        fn(img.data_ptr(), None if cnt is None else cnt.data_ptr(), ne, n_bins, width, I.data_ptr(), A.data_ptr(), isi.data_ptr(), stream)
        torch.cuda.synchronize()
        res.append((I.cpu().numpy().astype(np.float64), A.cpu().numpy().astype(np.float64), isi.cpu().numpy().astype(np.float64)))
    return res


def _assert_same(ref, got, tag):
    (rI, rA, risi), (I, A, isi) = ref, got
    assert np.isfinite(I).all() and np.isfinite(A).all() and np.isfinite(isi).all(), tag
    for e in range(rI.shape[0]):
        scale = rI[e].max()
        assert scale > 0, tag
        assert np.abs(I[e] - rI[e]).max() <= 2e-5 * scale, (tag, e, np.abs(I[e] - rI[e]).max() / scale)
        assert np.abs(A[e] - rA[e]).max() <= 1e-4, (tag, e, np.abs(A[e] - rA[e]).max())
        assert abs(isi[e] - risi[e]) <= 2e-5 * abs(risi[e]), (tag, e)


def test_reduce_static_matches_reduce_on_two_calls_in_a_row():
    import torch
    from paper_2209_13121_b200 import binding

    # two contexts of different image sizes share the one array of the GPU
    ctx_a = binding.Context(96, 64, 1, 1, 2.5)
    ctx_b = binding.Context(40, 48, 1, 1, 1.0)
    img_a, cnt_a = _inputs(torch, 5, 64, 96, seed=101, with_counts=True)
    img_b, cnt_b = _inputs(torch, 2, 48, 40, seed=202, with_counts=False)

    # call 1: 5 energies x 200 bins, with valid counts
    ref, got = _both(torch, ctx_a, img_a, cnt_a, 200, 20.0)
    _assert_same(ref, got, "first call")

    # call 2, straight after: other context, fewer energies and bins, so its sums, totals and counts sit where call 1 left
    # sums behind; nothing may leak in.  Device memory must not shrink across the call (no allocation).
    ne, nb = 2, 37
    stream = torch.cuda.current_stream().cuda_stream
    I = torch.full((ne, nb), -1.0, device="cuda"); A = torch.full_like(I, -1.0); isi = torch.full((ne,), -1.0, device="cuda")
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    ctx_b.reduce_static(img_b.data_ptr(), None, ne, nb, 45.0, I.data_ptr(), A.data_ptr(), isi.data_ptr(), stream)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before, "cyrsoxs_reduce_static took device memory"
    got2 = (I.cpu().numpy().astype(np.float64), A.cpu().numpy().astype(np.float64), isi.cpu().numpy().astype(np.float64))
    I0 = torch.full((ne, nb), -1.0, device="cuda"); A0 = torch.full_like(I0, -1.0); isi0 = torch.full((ne,), -1.0, device="cuda")
    ctx_b.reduce(img_b.data_ptr(), None, ne, nb, 45.0, I0.data_ptr(), A0.data_ptr(), isi0.data_ptr(), stream)
    torch.cuda.synchronize()
    ref2 = (I0.cpu().numpy().astype(np.float64), A0.cpu().numpy().astype(np.float64), isi0.cpu().numpy().astype(np.float64))
    _assert_same(ref2, got2, "second call")

    # and call 1's inputs once more: the answer of the first call comes back
    ref3, got3 = _both(torch, ctx_a, img_a, cnt_a, 200, 20.0)
    _assert_same(ref3, got3, "third call")
    assert np.array_equal(got3[0] > 0, got[0] > 0)
    ctx_a.close(); ctx_b.close()


def test_reduce_static_refuses_sizes_beyond_its_array():
    import torch
    from paper_2209_13121_b200 import binding

    ctx = binding.Context(16, 16, 1, 1, 2.0)
    img = torch.zeros((1, 16, 16), device="cuda"); I = torch.zeros((1, 8), device="cuda")
    too_big = [
        (1, binding.REDUCE_STATIC_MAX_BINS + 1),                                     # bins
        (binding.REDUCE_STATIC_MAX_ENERGIES + 1, 1),                                 # energies
        (64, binding.REDUCE_STATIC_MAX_CELLS // 64 + 1),                             # energies x bins
    ]
    for ne, nb in too_big:          # refused before any pointer is touched, so the small buffers above are enough
        with pytest.raises(binding.CyrsoxsError) as ei:
            ctx.reduce_static(img.data_ptr(), None, ne, nb, 20.0, I.data_ptr())
        assert ei.value.status == binding.ERR_INVALID_ARG
        msg = str(ei.value)
        assert "exceed the fixed scratch" in msg and str(binding.REDUCE_STATIC_MAX_CELLS) in msg and "cyrsoxs_reduce" in msg, msg
    for nb, width in [(0, 20.0), (8, 0.0), (8, 60.0)]:
        with pytest.raises(binding.CyrsoxsError) as ei:
            ctx.reduce_static(img.data_ptr(), None, 1, nb, width, I.data_ptr())
        assert ei.value.status == binding.ERR_INVALID_ARG
    # the largest accepted shape runs
    ne, nb = 32, binding.REDUCE_STATIC_MAX_BINS
    imgs = torch.ones((ne, 16, 16), device="cuda"); Ibig = torch.zeros((ne, nb), device="cuda")
    ctx.reduce_static(imgs.data_ptr(), None, ne, nb, 20.0, Ibig.data_ptr())
    torch.cuda.synchronize()
    assert float(Ibig[:, 0].min()) == 1.0 and float(Ibig[:, 0].max()) == 1.0        # bin 0 holds the centre pixel
    ctx.close()
