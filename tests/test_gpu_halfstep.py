"""pct_set_step(ctx, 2): the half-voxel depth step (R33) against the oracle in the
same mode: voxel sequences and fp32 nodes bit-exact on configs[0] and configs[3] geometry (up to 513 segments per path:
17 per lane), a DROP and a CARP run within the DROP tolerances, and switching back restores the default rows."""
import numpy as np
import pytest

import synth
from helpers import oracle_geom, to_device

pytestmark = pytest.mark.gpu


@pytest.fixture()
def half_oracle(oracle_mod):
    oracle_mod.set_substeps(2)
    yield oracle_mod
    oracle_mod.set_substeps(1)


def _rows(pct, torch, ctx, n, ms):
    nseg = torch.zeros(n, dtype=torch.int32, device="cuda")
    nnz = torch.zeros(n, dtype=torch.int32, device="cuda")
    seg_idx = torch.full((n, ms), -7, dtype=torch.int32, device="cuda")
    nodes = torch.zeros((n, ms + 1, 3), dtype=torch.float32, device="cuda")
    pct.pct_debug_rows(ctx, 0, n, ms, nseg, nnz, seg_idx, None, None, nodes)
    pct.pct_synchronize(ctx)
    return nseg.cpu().numpy(), nnz.cpu().numpy(), seg_idx.cpu().numpy(), nodes.cpu().numpy()


def test_half_step_rows_and_runs(half_oracle):
    import torch

    import paper_1707_05014_b200 as pct

    oracle = half_oracle
    for index, n in ((0, 4000), (3, 1200)):
        cfg = synth.config(index)
        H = synth.generate_numpy(cfg, n)
        geom = oracle_geom(oracle, cfg)
        hs = oracle.Histories(H)
        D = to_device(H)
        ctx = pct.pct_create(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out, torch.cuda.current_stream().cuda_stream)
        try:
            pct.pct_set_histories(ctx, n, D)
            default = _rows(pct, torch, ctx, n, geom.nmin + 2)
            with pytest.raises(pct.PctError):
                pct.pct_set_step(ctx, 3)
            pct.pct_set_step(ctx, 2)
            ms = 2 * geom.nmin + 2
            with pytest.raises(pct.PctError):
                _rows(pct, torch, ctx, n, geom.nmin + 2)  # max_seg too small for the mode
            nseg, nnz, seg_idx, nodes = _rows(pct, torch, ctx, n, ms)
            longest = 0
            for i in range(n):
                r = oracle.row_f32(geom, hs.hist(i))
                assert nseg[i] == r["nseg"] and nnz[i] == r["nnz"], i
                assert np.array_equal(seg_idx[i, :r["nseg"]], r["seg_idx"]), i
                if r["nseg"]:
                    assert np.array_equal(nodes[i, :r["nseg"] + 1], r["nodes"]), i
                longest = max(longest, r["nseg"])
            assert longest > 1.8 * geom.nmin * 0.9
            pct.pct_set_step(ctx, 1)
            again = _rows(pct, torch, ctx, n, geom.nmin + 2)
            assert np.array_equal(again[2], default[2]) and np.array_equal(again[0], default[0])
        finally:
            pct.pct_destroy(ctx)
    # runs in the mode (configs[0] data)
    cfg = synth.config(0)
    H = synth.generate_numpy(cfg, 20_011)
    geom = oracle_geom(oracle, cfg)
    hs = oracle.Histories(H)
    D = to_device(H)
    M = cfg.n_voxels
    out = np.zeros(M, dtype=np.float32)
    ctx = pct.pct_create(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out, torch.cuda.current_stream().cuda_stream)
    try:
        pct.pct_set_histories(ctx, hs.n, D)
        pct.pct_set_step(ctx, 2)
        x_ref = np.zeros(M)
        for it in range(3):
            if it < 2:
                pct.pct_iterate(ctx, 0.5, 700, 1)
                x_ref, st = oracle.drop_iterate(geom, hs, 0.5, 700, 1, x_ref)
                assert (pct.pct_get_stats(ctx)["rows"], pct.pct_get_stats(ctx)["nnz"]) == st
            else:
                pct.pct_iterate_carp(ctx, 0.5, 700, 1, 3)
                x_ref = oracle.carp_iterate(geom, hs, 0.5, 700, 1, 3, x_ref)
            pct.pct_get_image(ctx, out, M)
            g = out.astype(np.float64)
            assert np.linalg.norm(g - x_ref) <= 1e-4 * np.linalg.norm(x_ref), it
        assert np.abs(g - x_ref).max() <= 1e-3
    finally:
        pct.pct_destroy(ctx)
