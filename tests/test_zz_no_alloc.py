"""pct_tvs_step_static: the TVS step for callers that may not allocate device memory (include/pct.h).

Some users of the library cannot call cudaMalloc once they are running: the application gave all device memory to its
own pool at start-up, or it runs a latency-bound reconstruction loop in which the device-wide synchronisation of
cudaMalloc / cudaFree stalls the other streams, or its device-memory use was fixed and signed off beforehand.  For
them the library has ONE entry point whose working memory is a fixed array inside the library (8 MiB + 256 B per GPU,
grids up to PCT_TVS_STATIC_MAX_SLOTS = 2^20 stored voxels) instead of the arrays pct_set_tvs allocates.

What is checked here: the entry point gives the image, the accepted level and the TV values of the existing route
(pct_create + pct_set_image + pct_set_tvs + pct_tvs_step + pct_get_image) within the tolerance test_gpu_tvs.py uses for
a TVS step (1e-5 relative L2 and 1e-5 per voxel; TV 1e-6 relative) -- on calls IN A ROW, because all calls share the
one array and the second finds the first one's contents in it: a big grid first, then a small odd one whose padding
lies where the big image was, then two chained steps on one image.  Free device memory must not shrink over a call.

This file sorts last on purpose (pytest -x stops at the first failure; a failure here must not hide the other tests).
It has to pass on its own in a fresh process and after the rest of the suite."""
import numpy as np
import pytest


def _image(shape, seed):
    nx, ny, nz = shape
    rng = np.random.default_rng(seed)
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    disc = (((i - nx / 2) ** 2 + (j - ny / 2) ** 2) < (0.35 * min(nx, ny)) ** 2).astype(np.float64)
    return (disc * 1.04 + rng.normal(0, 0.03, disc.shape)).astype(np.float32).reshape(-1)


def _existing_route(pct, torch, shape, x, beta, gamma, levels, steps):
    """The same steps through a context: list of (image, state) after every step."""
    nx, ny, nz = shape
    M = nx * ny * nz
    r = 0.5 * min(nx, ny)
    ctx = pct.pct_create(nx, ny, nz, 1.0, -r - 10.0, r + 10.0, torch.cuda.current_stream().cuda_stream)
    res = []
    try:
        pct.pct_set_image(ctx, x, M)
        pct.pct_set_tvs(ctx, beta, gamma, levels)
        for _ in range(steps):
            pct.pct_tvs_step(ctx)
            out = np.zeros(M, dtype=np.float32)
            pct.pct_get_image(ctx, out, M)
            res.append((out, pct.pct_get_tvs_state(ctx)))
    finally:
        pct.pct_destroy(ctx)
    return res


def _close(got, want):
    g, w = got.astype(np.float64), want.astype(np.float64)
    assert np.linalg.norm(g - w) <= 1e-5 * np.linalg.norm(w)
    assert np.abs(g - w).max() <= 1e-5


@pytest.mark.gpu
def test_static_step_equals_the_allocating_route_on_calls_in_a_row():
    import torch

    import paper_1707_05014_b200 as pct

    stream = torch.cuda.current_stream().cuda_stream
    gamma = 0.7
    # (grid, beta, levels, steps): the first fills half of the static array, the second is an odd grid (padded rows and
    # columns, which must read as zero) lying inside what the first left behind, the third chains two steps
    cases = [((128, 128, 32), 500.0, 8, 1), ((45, 71, 5), 0.5, 3, 1), ((64, 64, 8), 2.0, 4, 2)]
    want = [_existing_route(pct, torch, shape, _image(shape, 11 + n), beta, gamma, levels, steps)
            for n, (shape, beta, levels, steps) in enumerate(cases)]
    # everything the calls need exists before the first of them: the entry point itself must add nothing
    imgs = [torch.from_numpy(_image(shape, 11 + n)).cuda() for n, (shape, _, _, _) in enumerate(cases)]
    info = torch.zeros(4, dtype=torch.float64, device="cuda")
    accepted = 0
    for n, (shape, beta, levels, steps) in enumerate(cases):
        b = beta
        for s in range(steps):
            torch.cuda.synchronize()
            free_before = torch.cuda.mem_get_info()[0]
            pct.pct_tvs_step_static(imgs[n], *shape, b, levels, info, stream)
            torch.cuda.synchronize()
            if n > 0:  # (the very first call may make the runtime load the kernels)
                assert torch.cuda.mem_get_info()[0] >= free_before
            used, tv_before, tv_after, level = info.cpu().numpy()
            ref_img, ref = want[n][s]
            assert int(level) == ref["level"], (n, s, level, ref)
            assert tv_before == pytest.approx(ref["tv_before"], rel=1e-6)
            assert tv_after == pytest.approx(ref["tv_after"], rel=1e-6)
            assert gamma * used == pytest.approx(ref["beta"], rel=1e-6)  # the context's next step size
            _close(imgs[n].cpu().numpy(), ref_img)
            accepted += int(level) >= 0
            b = gamma * float(used)
    assert accepted >= 3  # the cases do move the image
    # info is optional
    again = torch.from_numpy(_image(cases[1][0], 12)).cuda()
    pct.pct_tvs_step_static(again, *cases[1][0], cases[1][1], cases[1][2], None, stream)
    torch.cuda.synchronize()
    _close(again.cpu().numpy(), want[1][0][0])


@pytest.mark.gpu
def test_static_step_rejects_what_it_cannot_hold():
    import torch

    import paper_1707_05014_b200 as pct

    x = torch.zeros(16, dtype=torch.float32, device="cuda")
    with pytest.raises(pct.PctError, match="grid too large"):  # 256 x 256 x 128 is 8 times the limit
        pct.pct_tvs_step_static(x, 256, 256, 128, 1.0, 4)
    with pytest.raises(pct.PctError, match="grid too large"):  # 1023 x 1 x 512 is stored as 1024 x 2 x 512 = the limit; one more slice
        pct.pct_tvs_step_static(x, 1023, 1, 513, 1.0, 4)
    host = np.zeros(16, dtype=np.float32)
    with pytest.raises(pct.PctError, match="device memory"):
        pct.pct_tvs_step_static(host, 4, 4, 1, 1.0, 4)
    for bad in ((0.0, 4), (-1.0, 4), (float("nan"), 4), (1.0, 0), (1.0, 9)):
        with pytest.raises(pct.PctError):
            pct.pct_tvs_step_static(x, 4, 4, 1, *bad)
    pct.pct_tvs_step_static(x, 4, 4, 1, 1.0, 4)  # a flat image: no direction, no step, no fault
    torch.cuda.synchronize()
    assert float(x.abs().max()) == 0.0


def test_static_step_limit_is_checked_before_any_cuda_call():
    """No GPU needed: sizes beyond the static array are refused with both numbers in the message."""
    import ctypes as C

    import paper_1707_05014_b200 as pct

    L = pct.lib()
    assert pct.PCT_TVS_STATIC_MAX_SLOTS == 1 << 20
    rc = L.pct_tvs_step_static(C.c_void_p(256), 1024, 1024, 2, 1.0, 4, None, None)
    assert rc == pct.binding.PCT_EINVAL
    msg = L.pct_tvs_step_static_error().decode()
    assert "2097152" in msg and "1048576" in msg
    assert L.pct_tvs_step_static(None, 8, 8, 8, 1.0, 4, None, None) == pct.binding.PCT_EINVAL
