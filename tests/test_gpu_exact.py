"""pct_set_walk(ctx, PCT_WALK_EXACT): exact traversal of the path polyline (R34) against
the oracle in the same mode: the piece lists (voxel of every piece, in order) bit-exact and the piece lengths bitwise on
configs[0], an odd grid and configs[3] geometry, also with the half-voxel step; DROP and CARP runs within the DROP
tolerances; switching back restores the default rows."""
import numpy as np
import pytest

import synth
from helpers import oracle_geom, to_device

pytestmark = pytest.mark.gpu


@pytest.fixture()
def exact_oracle(oracle_mod):
    oracle_mod.set_walk_mode(1)
    yield oracle_mod
    oracle_mod.set_walk_mode(0)
    oracle_mod.set_substeps(1)


def _rows(pct, torch, ctx, n, ms):
    nseg = torch.zeros(n, dtype=torch.int32, device="cuda")
    nnz = torch.zeros(n, dtype=torch.int32, device="cuda")
    seg_idx = torch.full((n, ms), -7, dtype=torch.int32, device="cuda")
    seg_len = torch.zeros((n, ms), dtype=torch.float32, device="cuda")
    row_len = torch.zeros((n, ms), dtype=torch.float32, device="cuda")
    nodes = torch.zeros((n, ms + 1, 3), dtype=torch.float32, device="cuda")
    pct.pct_debug_rows(ctx, 0, n, ms, nseg, nnz, seg_idx, seg_len, row_len, nodes)
    pct.pct_synchronize(ctx)
    return [t.cpu().numpy() for t in (nseg, nnz, seg_idx, seg_len, row_len, nodes)]


def _check(oracle, pct, torch, cfg, H, substeps=1):
    geom = oracle_geom(oracle, cfg)
    hs = oracle.Histories(H)
    D = to_device(H)
    n = hs.n
    oracle.set_substeps(substeps)
    ctx = pct.pct_create(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out, torch.cuda.current_stream().cuda_stream)
    try:
        pct.pct_set_histories(ctx, n, D)
        default = _rows(pct, torch, ctx, n, geom.nmin + 2)
        pct.pct_set_step(ctx, substeps)
        pct.pct_set_walk(ctx, pct.PCT_WALK_EXACT)
        ms = 8 * (substeps * geom.nmin + 2)
        nseg, nnz, seg_idx, seg_len, row_len, nodes = _rows(pct, torch, ctx, n, ms)
        paths = 0
        for i in range(n):
            r = oracle.row_f32(geom, hs.hist(i))
            ns = r["nseg"]
            assert nseg[i] == ns and nnz[i] == r["nnz"], i
            if ns == 0:
                continue
            paths += 1
            assert np.array_equal(seg_idx[i, :ns], r["seg_idx"]), i   # voxel of every piece: bit-exact
            assert np.array_equal(seg_len[i, :ns], r["seg_len"]), i   # fixed fp32 operation order: bitwise
            nn = r["nodes"].shape[0]
            assert np.array_equal(nodes[i, :nn], r["nodes"]), i
            heads = row_len[i, :ns] > 0
            assert np.array_equal(seg_idx[i, :ns][heads], r["row_idx"]), i
            assert row_len[i, :ns][heads] == pytest.approx(r["row_len"], rel=1e-6)
        pct.pct_set_walk(ctx, pct.PCT_WALK_MIDPOINT)
        pct.pct_set_step(ctx, 1)
        again = _rows(pct, torch, ctx, n, geom.nmin + 2)
        assert np.array_equal(again[2], default[2]) and np.array_equal(again[0], default[0])
        with pytest.raises(pct.PctError):
            pct.pct_set_walk(ctx, 5)
    finally:
        pct.pct_destroy(ctx)
        oracle.set_substeps(1)
    return paths


def test_pieces_bit_exact(exact_oracle):
    import torch

    import paper_1707_05014_b200 as pct

    cfg = synth.config(0)
    assert _check(exact_oracle, pct, torch, cfg, synth.generate_numpy(cfg, 5000)) > 3500
    base = synth.config(0)
    odd = synth.Config(9, "odd", 3000, 45, 71, 5, 0.8, 37, 500, 0.1, 1, base.shapes * 0.5, seed=99)
    assert _check(exact_oracle, pct, torch, odd, synth.generate_numpy(odd, 3000)) > 700
    cfg3 = synth.config(3)
    assert _check(exact_oracle, pct, torch, cfg3, synth.generate_numpy(cfg3, 800)) > 400
    assert _check(exact_oracle, pct, torch, cfg, synth.generate_numpy(cfg, 1500), substeps=2) > 1000


def test_runs_in_the_exact_mode(exact_oracle):
    import torch

    import paper_1707_05014_b200 as pct

    oracle = exact_oracle
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
        pct.pct_set_walk(ctx, pct.PCT_WALK_EXACT)
        # one block against the oracle: hit counts exact, Delta within the block tolerance
        x0 = (synth.rsp_volume(cfg) * 0.9).astype(np.float32)
        pct.pct_set_image(ctx, x0, M)
        delta = torch.zeros(M, dtype=torch.float32, device="cuda")
        cnt = torch.zeros(M, dtype=torch.float32, device="cuda")
        pct.pct_debug_block(ctx, 100, 7000, delta, cnt)
        pct.pct_synchronize(ctx)
        d_ref, c_ref, _ = oracle.block_accumulate(geom, hs, 100, 7000, x0.astype(np.float64))
        assert np.array_equal(cnt.cpu().numpy(), c_ref.astype(np.float32))
        d = delta.cpu().numpy().astype(np.float64)
        assert np.linalg.norm(d - d_ref) <= 2e-5 * np.linalg.norm(d_ref)
        pct.pct_set_image(ctx, np.zeros(M, dtype=np.float32), M)
        x_ref = np.zeros(M)
        for it in range(3):
            if it < 2:
                pct.pct_iterate(ctx, 0.5, 700, 1)
                x_ref, st = oracle.drop_iterate(geom, hs, 0.5, 700, 1, x_ref)
                gs = pct.pct_get_stats(ctx)
                assert (gs["rows"], gs["nnz"]) == st
            else:
                pct.pct_iterate_carp(ctx, 0.5, 700, 1, 3)
                x_ref = oracle.carp_iterate(geom, hs, 0.5, 700, 1, 3, x_ref)
            pct.pct_get_image(ctx, out, M)
            g = out.astype(np.float64)
            assert np.linalg.norm(g - x_ref) <= 1e-4 * np.linalg.norm(x_ref), it
        assert np.abs(g - x_ref).max() <= 1e-3
    finally:
        pct.pct_destroy(ctx)


def test_a_row_that_outgrows_the_scratch_is_reported_not_dropped_silently():
    """A lane's part of the scratch holds 8 runs per segment of the longest chunk + 8 (16 on a 24-wide grid).  A history
    at a slope no tracker delivers (dt/du = 15 at 45 degrees to the grid: each of its two segments crosses 17 voxel faces)
    produces more.  Its row is left out of the block -- and every call that hands out results says so: pct_synchronize,
    pct_get_image and pct_get_stats return PCT_EINTERNAL; the sane histories alone give PCT_OK."""
    import torch

    import paper_1707_05014_b200 as pct

    base = synth.config(0)
    n = 64
    cfg = synth.Config(7, "small", n, 24, 24, 4, 1.0, 8, n, 0.1, 1, base.shapes * 0.375, seed=5)
    H = synth.generate_numpy(cfg, n)
    M = cfg.n_voxels
    out = torch.zeros(M, dtype=torch.float32, device="cuda")
    codes = []
    for steep in (True, False):
        Hs = {k: np.array(v, copy=True) for k, v in H.items()}
        if steep:  # one straight line through the centre of the object, fifteen voxels sideways per voxel of depth
            Hs["tht_in"][5] = Hs["tht_out"][5] = 15.0
            Hs["t_in"][5], Hs["t_out"][5] = 15.0 * cfg.u_in, 15.0 * cfg.u_out
            Hs["thv_in"][5] = Hs["thv_out"][5] = 0.0
            Hs["v_in"][5] = Hs["v_out"][5] = 0.3
            Hs["proj"][5] = 1  # 45 degrees (8 angles)
        ctx = pct.pct_create(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out, torch.cuda.current_stream().cuda_stream)
        try:
            pct.pct_set_histories(ctx, n, to_device(Hs))
            pct.pct_set_walk(ctx, pct.PCT_WALK_EXACT)
            pct.pct_iterate(ctx, 0.5, n, 1)
            got = []
            for call in (lambda: pct.pct_synchronize(ctx), lambda: pct.pct_get_image(ctx, out, M), lambda: pct.pct_get_stats(ctx)):
                try:
                    call()
                    got.append(0)
                except pct.PctError as e:
                    got.append(e.code)
                    assert "more runs" in str(e)
            codes.append(got)
        finally:
            pct.pct_destroy(ctx)
    assert codes == [[-5, -5, -5], [0, 0, 0]], codes
