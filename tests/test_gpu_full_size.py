"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times: configs[3] (5e8 histories,
19 GB) and configs[4] (2e9 histories, 76 GB, history indices up to 2e9 - 1 < 2^31) resident on the GPU.

The oracle cannot run such a sweep, so it is asked for what it can compute one by one: the rows of histories
sampled over the whole index range (first, last, around block boundaries, random) -- voxel sequences bit-exact --
and one whole DROP block deep in the set against the image the full sweep left (hit counts exact, Delta within the
block tolerance).  Plus the properties that hold at any size: every history counted once, the image finite.
Inputs come from the seeded CUDA generator (synth/), copied to the host for the oracle."""
import numpy as np
import pytest

import synth
from helpers import oracle_geom

pytestmark = pytest.mark.gpu


def _host_slice(D, lo, hi):
    H = {}
    for k, v in D.items():
        if k in ("proj_cos", "proj_sin"):
            H[k] = v.cpu().numpy()
        elif k == "proj":
            H[k] = v[lo:hi].cpu().numpy().view(np.uint16)
        else:
            H[k] = v[lo:hi].cpu().numpy()
    return H


@pytest.mark.parametrize("index", [3, 4])
def test_full_size_rows_and_a_deep_block(oracle_mod, index):
    import torch

    import paper_1707_05014_b200 as pct
    import synth.cuda_gen as cuda_gen

    oracle = oracle_mod
    cfg = synth.config(index)
    n, B, M = cfg.n, cfg.block_size, cfg.n_voxels
    free, _ = torch.cuda.mem_get_info()
    if free < 46 * n + (8 << 30):
        pytest.skip("needs %.0f GB of device memory" % (46 * n / 1e9))
    D = cuda_gen.generate_cuda(cfg, n)  # synth names, on the device
    geom = oracle_geom(oracle, cfg)
    table = oracle.sigma1_table(geom.h, geom.nmin)
    n_blocks = (n + B - 1) // B
    ctx = pct.pct_create(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out, torch.cuda.current_stream().cuda_stream)
    try:
        pct.pct_set_histories(ctx, n, synth.to_pct_names(D))
        pct.pct_iterate(ctx, cfg.lam, B, 1)  # one whole sweep, as bench.py launches it
        img = torch.empty(M, dtype=torch.float32, device="cuda")
        pct.pct_get_image(ctx, img, M)
        st = pct.pct_get_stats(ctx)
        assert st["histories"] == n and 0.98 * n < st["rows"] <= n
        assert 150 * n < st["nnz"] <= st["segments"] < 260 * n
        assert bool(torch.isfinite(img).all().item())
        # rows of sampled histories, over the whole index range
        rng = np.random.default_rng(index)
        starts = [0, n - 8, B - 4, (n_blocks - 1) * B - 4, n // 2] + [int(s) for s in rng.integers(0, n - 8, 11)]
        ms = geom.nmin + 2
        checked = 0
        for first in starts:
            nseg = torch.zeros(8, dtype=torch.int32, device="cuda")
            nnz = torch.zeros(8, dtype=torch.int32, device="cuda")
            seg_idx = torch.full((8, ms), -7, dtype=torch.int32, device="cuda")
            pct.pct_debug_rows(ctx, first, 8, ms, nseg, nnz, seg_idx)
            pct.pct_synchronize(ctx)
            hs = oracle.Histories(_host_slice(D, first, first + 8))
            for i in range(8):
                r = oracle.row_f32(geom, hs.hist(i), table)
                assert int(nseg[i]) == r["nseg"] and int(nnz[i]) == r["nnz"], (first, i)
                assert np.array_equal(seg_idx[i, :r["nseg"]].cpu().numpy(), r["seg_idx"]), (first, i)
                checked += r["nseg"] > 0
        assert checked > 100
        # one whole block deep in the set, against the image the sweep left
        b = n_blocks - 3
        delta = torch.zeros(M, dtype=torch.float32, device="cuda")
        cnt = torch.zeros(M, dtype=torch.float32, device="cuda")
        pct.pct_debug_block(ctx, b * B, B, delta, cnt)
        pct.pct_synchronize(ctx)
        hs = oracle.Histories(_host_slice(D, b * B, (b + 1) * B))
        d_ref, c_ref, _ = oracle.block_accumulate(geom, hs, 0, B, img.cpu().numpy().astype(np.float64))
        assert np.array_equal(cnt.cpu().numpy(), c_ref.astype(np.float32))  # hit counts: exact
        d = delta.cpu().numpy().astype(np.float64)
        assert np.linalg.norm(d - d_ref) <= 2e-5 * np.linalg.norm(d_ref)
        assert np.abs(d - d_ref).max() <= 2e-4 * max(1.0, np.abs(d_ref).max())
    finally:
        pct.pct_destroy(ctx)
        del D
        torch.cuda.empty_cache()
