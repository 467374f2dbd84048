"""Parity in DEPTH (SURVEY.md 8(d) "Parity at scale"): every config run for ITS OWN iteration count.

* configs[1] in full -- 1e7 histories, B = 1e4, lambda = 0.1, all 6 iterations -- against the oracle's DROP
  run: image relative L2 <= 1e-4 after every iteration, |x - x_oracle| <= 1e-3 per voxel at the end
  (BASELINE.json north_star).  ~6000 sequential block updates of the image.
* configs[2], [3], [4] in full for their n_iter (8 / 10 / 12 sweeps, up to 1.2e5 sequential block updates): the
  oracle cannot follow such a run, so the image is SNAPSHOT before one block in the first, a middle and the last
  iteration; that one block is run by the oracle from the snapshot (orc_block_accumulate: hit counts exact, Delta
  within the block tolerance) and its x-update x + lambda * Delta / max(1, c) in fp64 is compared per voxel with
  the image the library holds after that block.  The sweep is split around the snapshot block by handing the
  library sub-ranges of the same device arrays (block boundaries unchanged: PAPER.md:50, the image is the whole
  solver state between blocks).
Inputs: the seeded CUDA generator (synth/), ONE set of arrays for both sides."""
import numpy as np
import pytest

import synth
from helpers import oracle_geom

pytestmark = pytest.mark.gpu

REL_L2_PER_ITER = 1e-4
ABS_FINAL = 1e-3
TABLES = ("proj_cos", "proj_sin")


def _host(D, lo, hi):
    H = {}
    for k, v in D.items():
        if k in TABLES:
            H[k] = v.cpu().numpy()
        elif k == "proj":
            H[k] = v[lo:hi].cpu().numpy().view(np.uint16)
        else:
            H[k] = v[lo:hi].cpu().numpy()
    return H


def _sub(P, lo, hi):
    """Histories [lo, hi) of the device arrays (views: no copy), include/pct.h names."""
    return {k: (v if k in TABLES else v[lo:hi]) for k, v in P.items()}


def test_config1_in_full_all_six_iterations(oracle_mod):
    import torch

    import paper_1707_05014_b200 as pct
    import synth.cuda_gen as cuda_gen

    oracle = oracle_mod
    cfg = synth.config(1)
    n, B, M = cfg.n, cfg.block_size, cfg.n_voxels
    assert (n, B, cfg.n_iter) == (10_000_000, 10_000, 6)
    D = cuda_gen.generate_cuda(cfg, n)
    hs = oracle.Histories(_host(D, 0, n))
    geom = oracle_geom(oracle, cfg)
    ctx = pct.pct_create(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out, torch.cuda.current_stream().cuda_stream)
    out = torch.zeros(M, dtype=torch.float32, device="cuda")
    x_ref = np.zeros(M)
    try:
        pct.pct_set_histories(ctx, n, synth.to_pct_names(D))
        for it in range(cfg.n_iter):
            pct.pct_iterate(ctx, cfg.lam, B, 1)
            pct.pct_get_image(ctx, out, M)
            x_ref, stats = oracle.drop_iterate(geom, hs, cfg.lam, B, 1, x_ref)
            x = out.cpu().numpy().astype(np.float64)
            rel = np.linalg.norm(x - x_ref) / np.linalg.norm(x_ref)
            assert rel <= REL_L2_PER_ITER, "iteration %d: rel L2 %.3g" % (it, rel)
            gs = pct.pct_get_stats(ctx)
            assert (gs["rows"], gs["nnz"]) == stats
        assert np.abs(x - x_ref).max() <= ABS_FINAL
        # the run went somewhere: water cylinder near RSP 1 on the axis
        vol = x.reshape(cfg.nz, cfg.ny, cfg.nx)
        assert 0.9 < vol[cfg.nz // 2, cfg.ny // 2, cfg.nx // 2] < 1.1
    finally:
        pct.pct_destroy(ctx)


@pytest.mark.parametrize("index", [2, 3, 4])
def test_full_iteration_count_with_snapshot_blocks(oracle_mod, index):
    import torch

    import paper_1707_05014_b200 as pct
    import synth.cuda_gen as cuda_gen

    oracle = oracle_mod
    cfg = synth.config(index)
    n, B, M, lam = cfg.n, cfg.block_size, cfg.n_voxels, cfg.lam
    free, _ = torch.cuda.mem_get_info()
    if free < 46 * n + (8 << 30):
        pytest.skip("needs %.0f GB of device memory" % (46 * n / 1e9))
    D = cuda_gen.generate_cuda(cfg, n)
    P = synth.to_pct_names(D)
    geom = oracle_geom(oracle, cfg)
    n_blocks = (n + B - 1) // B
    # (iteration, block): first / middle / last iteration, blocks spread over the sweep (never the first block
    # of the first sweep: its snapshot would be x0 = 0)
    snaps = {0: n_blocks // 3, cfg.n_iter // 2: (2 * n_blocks) // 3 + 1, cfg.n_iter - 1: n_blocks - 2}
    assert len(snaps) == 3
    ctx = pct.pct_create(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out, torch.cuda.current_stream().cuda_stream)
    img = torch.empty(M, dtype=torch.float32, device="cuda")
    delta = torch.zeros(M, dtype=torch.float32, device="cuda")
    cnt = torch.zeros(M, dtype=torch.float32, device="cuda")
    full_set = False
    try:
        for it in range(cfg.n_iter):
            if it not in snaps:
                if not full_set:
                    pct.pct_set_histories(ctx, n, P)
                    full_set = True
                pct.pct_iterate(ctx, lam, B, 1)
                continue
            b = snaps[it]
            lo, hi = b * B, min(n, (b + 1) * B)
            full_set = False
            pct.pct_set_histories(ctx, lo, _sub(P, 0, lo))  # blocks 0 .. b-1 of this iteration
            pct.pct_iterate(ctx, lam, B, 1)
            pct.pct_get_image(ctx, img, M)
            x_snap = img.cpu().numpy().astype(np.float64)  # the image that enters block b (exact: fp32 -> fp64)
            pct.pct_set_histories(ctx, hi - lo, _sub(P, lo, hi))  # block b alone
            pct.pct_debug_block(ctx, 0, hi - lo, delta, cnt)  # leaves image and accumulator as they were
            pct.pct_iterate(ctx, lam, B, 1)
            pct.pct_get_image(ctx, img, M)
            x_after = img.cpu().numpy().astype(np.float64)
            hs = oracle.Histories(_host(D, lo, hi))
            d_ref, c_ref, st = oracle.block_accumulate(geom, hs, 0, hi - lo, x_snap)
            assert st[0] > 0.9 * (hi - lo)
            assert np.array_equal(cnt.cpu().numpy(), c_ref.astype(np.float32)), (it, b)  # hit counts: exact
            d = delta.cpu().numpy().astype(np.float64)
            assert np.linalg.norm(d - d_ref) <= 2e-5 * np.linalg.norm(d_ref), (it, b)
            assert np.abs(d - d_ref).max() <= 2e-4 * max(1.0, np.abs(d_ref).max()), (it, b)
            # the block's x-update in fp64 (R12), per voxel
            x_ref = x_snap + lam * d_ref / np.maximum(1.0, c_ref)
            moved = np.abs(x_ref - x_snap).max()
            assert moved > 1e-5  # the block did change the image
            assert np.abs(x_after - x_ref).max() <= max(2e-6, 2e-4 * moved), (it, b)
            assert np.linalg.norm(x_after - x_ref) <= 1e-6 * np.linalg.norm(x_ref), (it, b)
            if hi < n:
                pct.pct_set_histories(ctx, n - hi, _sub(P, hi, n))  # the rest of this iteration
                pct.pct_iterate(ctx, lam, B, 1)
        pct.pct_get_image(ctx, img, M)
        assert bool(torch.isfinite(img).all().item())
        # after the config's own n_iter sweeps the soft tissue at the centre is near its RSP (1.04; configs[3]/[4]
        # have random inserts, so only a loose band)
        vol = img.view(cfg.nz, cfg.ny, cfg.nx)
        c = float(vol[cfg.nz // 2 - 2:cfg.nz // 2 + 2, cfg.ny // 2 - 20:cfg.ny // 2 + 20, cfg.nx // 2 - 20:cfg.nx // 2 + 20].mean())
        assert 0.8 < c < 1.3, c
    finally:
        pct.pct_destroy(ctx)
        del D, P
        torch.cuda.empty_cache()
