"""Grids wider than the two-histories-per-warp kernel serves (its two row buffers per warp outgrow shared memory from
min(nx,ny) of about 420): pct_create must configure only the kernel that will run (k_drop_block), up to the documented
limit min(nx,ny) <= 1318, and pct_set_step(ctx, 2) must work on a 512-wide grid (1024 nodes per path).  Rows bit-exact
and one DROP block against the oracle, as on the narrow grids; sizes beyond the limit are refused with PCT_EINVAL."""
import numpy as np
import pytest

import synth
from helpers import oracle_geom, to_device

pytestmark = pytest.mark.gpu


def _wide_cfg(nx, ny, nz, h, n):
    base = synth.config(0)  # the cylinder with three inserts, scaled to the hull of this grid
    scale = 0.5 * h * min(nx, ny) / 32.0
    return synth.Config(8, "wide", n, nx, ny, nz, h, 37, 500, 0.1, 1, base.shapes * scale, seed=2024)


def _histories(cfg, n):
    """Seeded histories of the scaled phantom, flattened into the thin slab these grids have (two slices: the paths must not
    leave through the top or bottom, or none would be long enough to need the wide row buffers)."""
    H = synth.generate_numpy(cfg, n)
    H = {k: np.array(v, copy=True) for k, v in H.items()}
    H["thv_in"][:] = 0.0
    H["thv_out"][:] = 0.0
    H["v_in"][:] = H["v_out"][:] = (0.4 * cfg.h * (np.arange(n) % 5 - 2) / 2).astype(np.float32)
    return H


def _rows(pct, torch, ctx, n, ms):
    nseg = torch.zeros(n, dtype=torch.int32, device="cuda")
    nnz = torch.zeros(n, dtype=torch.int32, device="cuda")
    seg_idx = torch.full((n, ms), -7, dtype=torch.int32, device="cuda")
    seg_len = torch.zeros((n, ms), dtype=torch.float32, device="cuda")
    pct.pct_debug_rows(ctx, 0, n, ms, nseg, nnz, seg_idx, seg_len, None, None)
    pct.pct_synchronize(ctx)
    return nseg.cpu().numpy(), nnz.cpu().numpy(), seg_idx.cpu().numpy(), seg_len.cpu().numpy()


def _compare_rows(oracle, geom, hs, rows, n):
    nseg, nnz, seg_idx, seg_len = rows
    longest = 0
    for i in range(n):
        r = oracle.row_f32(geom, hs.hist(i))
        assert nseg[i] == r["nseg"] and nnz[i] == r["nnz"], i
        assert np.array_equal(seg_idx[i, :r["nseg"]], r["seg_idx"]), i
        assert np.array_equal(seg_len[i, :r["nseg"]], r["seg_len"]), i
        longest = max(longest, r["nseg"])
    return longest


def test_a_1024_wide_grid_runs_the_one_history_kernel(oracle_mod):
    import torch

    import paper_1707_05014_b200 as pct

    oracle = oracle_mod
    n = 700
    cfg = _wide_cfg(1024, 1024, 2, 0.25, n)
    H = _histories(cfg, n)
    geom = oracle_geom(oracle, cfg)
    hs = oracle.Histories(H)
    D = to_device(H)
    M = cfg.n_voxels
    ctx = pct.pct_create(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out, torch.cuda.current_stream().cuda_stream)
    try:
        pct.pct_set_histories(ctx, n, D)
        assert _compare_rows(oracle, geom, hs, _rows(pct, torch, ctx, n, 1026), n) > 850
        with pytest.raises(pct.PctError, match="too wide"):  # 2048 nodes per path do not fit
            pct.pct_set_step(ctx, 2)
        x0 = (synth.rsp_volume(cfg) * 0.7).astype(np.float32)
        pct.pct_set_image(ctx, x0, M)
        delta = torch.zeros(M, dtype=torch.float32, device="cuda")
        cnt = torch.zeros(M, dtype=torch.float32, device="cuda")
        pct.pct_debug_block(ctx, 0, n, delta, cnt)
        pct.pct_synchronize(ctx)
        d_ref, c_ref, _ = oracle.block_accumulate(geom, hs, 0, n, x0.astype(np.float64))
        assert np.array_equal(cnt.cpu().numpy(), c_ref.astype(np.float32))
        d = delta.cpu().numpy().astype(np.float64)
        assert np.linalg.norm(d - d_ref) <= 2e-5 * np.linalg.norm(d_ref)
        # and a sweep through pct_iterate (blocks of 250: two full ones and a ragged one)
        out = np.zeros(M, dtype=np.float32)
        pct.pct_iterate(ctx, 0.5, 250, 1)
        pct.pct_get_image(ctx, out, M)
        x_ref, st = oracle.drop_iterate(geom, hs, 0.5, 250, 1, x0.astype(np.float64))
        assert np.linalg.norm(out - x_ref) <= 1e-4 * np.linalg.norm(x_ref)
        gs = pct.pct_get_stats(ctx)
        assert (gs["rows"], gs["nnz"]) == st
    finally:
        pct.pct_destroy(ctx)


def test_half_voxel_step_on_a_512_wide_grid(oracle_mod):
    import torch

    import paper_1707_05014_b200 as pct

    oracle = oracle_mod
    n = 500
    cfg = _wide_cfg(512, 512, 2, 0.5, n)
    H = _histories(cfg, n)
    geom = oracle_geom(oracle, cfg)
    hs = oracle.Histories(H)
    D = to_device(H)
    ctx = pct.pct_create(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out, torch.cuda.current_stream().cuda_stream)
    try:
        pct.pct_set_histories(ctx, n, D)
        assert _compare_rows(oracle, geom, hs, _rows(pct, torch, ctx, n, 514), n) > 420
        pct.pct_set_step(ctx, 2)
        oracle.set_substeps(2)
        try:
            assert _compare_rows(oracle, geom, hs, _rows(pct, torch, ctx, n, 1026), n) > 850
        finally:
            oracle.set_substeps(1)
    finally:
        pct.pct_destroy(ctx)


def test_the_documented_limit():
    import torch

    import paper_1707_05014_b200 as pct

    s = torch.cuda.current_stream().cuda_stream
    ctx = pct.pct_create(1318, 1400, 1, 0.2, -200.0, 200.0, s)  # the widest grid the header promises
    pct.pct_destroy(ctx)
    with pytest.raises(pct.PctError, match="too wide"):
        pct.pct_create(1319, 1400, 1, 0.2, -200.0, 200.0, s)
