"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Bars (BASELINE.json north_star): voxel-index sequences bit-exact; MLP node positions within
1e-4 mm of the fp64 definition; per-iteration image relative L2 error <= 1e-4; final RSP within
1e-3 absolute per voxel.  Hit counts are integers: exact."""
import numpy as np
import pytest

import synth
from helpers import oracle_geom, slice_hist, to_device

pytestmark = pytest.mark.gpu

REL_L2_PER_ITER = 1e-4
ABS_FINAL = 1e-3


@pytest.fixture(scope="module")
def torch_cuda():
    import torch

    assert torch.cuda.is_available(), "these tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def pct():
    import paper_1707_05014_b200 as p

    return p


def _ctx(pct, torch, cfg):
    return pct.pct_create(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out, torch.cuda.current_stream().cuda_stream)


def _gpu_rows(pct, torch, ctx, first, count, nmin):
    ms = nmin + 2
    dev = "cuda"
    nseg = torch.zeros(count, dtype=torch.int32, device=dev)
    nnz = torch.zeros(count, dtype=torch.int32, device=dev)
    seg_idx = torch.full((count, ms), -7, dtype=torch.int32, device=dev)
    seg_len = torch.zeros((count, ms), dtype=torch.float32, device=dev)
    row_len = torch.zeros((count, ms), dtype=torch.float32, device=dev)
    nodes = torch.zeros((count, ms + 1, 3), dtype=torch.float32, device=dev)
    pct.pct_debug_rows(ctx, first, count, ms, nseg, nnz, seg_idx, seg_len, row_len, nodes)
    pct.pct_synchronize(ctx)
    return [t.cpu().numpy() for t in (nseg, nnz, seg_idx, seg_len, row_len, nodes)]


def _check_rows(oracle, pct, torch, cfg, H, stride=1, t64_every=7):
    geom = oracle_geom(oracle, cfg)
    hs = oracle.Histories(H)
    D = to_device(H)
    ctx = _ctx(pct, torch, cfg)
    try:
        pct.pct_set_histories(ctx, hs.n, D)
        nseg, nnz, seg_idx, seg_len, row_len, nodes = _gpu_rows(pct, torch, ctx, 0, hs.n, geom.nmin)
    finally:
        pct.pct_destroy(ctx)
    table = oracle.sigma1_table(geom.h, geom.nmin)
    n_paths, worst64 = 0, 0.0
    for i in range(0, hs.n, stride):
        r = oracle.row_f32(geom, hs.hist(i), table)
        ns = r["nseg"]
        assert nseg[i] == ns, "history %d: segment count" % i
        assert nnz[i] == r["nnz"], "history %d: nnz" % i
        if ns == 0:
            continue
        n_paths += 1
        # bit-exact: voxel index of every raw segment (the decision floor(fp32 midpoint))
        assert np.array_equal(seg_idx[i, :ns], r["seg_idx"]), "history %d: voxel sequence" % i
        # the whole rule is IEEE fp32 with a fixed operation order: lengths and nodes agree bitwise too
        assert np.array_equal(seg_len[i, :ns], r["seg_len"]), "history %d: segment lengths" % i
        assert np.array_equal(nodes[i, :ns + 1], r["nodes"]), "history %d: node positions" % i
        # merged row: heads carry the merged length (fp32 sum in k order), others 0
        heads = row_len[i, :ns] > 0
        assert np.array_equal(seg_idx[i, :ns][heads], r["row_idx"])
        assert row_len[i, :ns][heads] == pytest.approx(r["row_len"], rel=1e-6)
        if (i // stride) % t64_every == 0:
            n64, _ = oracle.path_f64(geom, hs.hist(i))
            if n64 is not None and n64.shape[0] == ns + 1:
                worst64 = max(worst64, float(np.abs(nodes[i, :ns + 1].astype(np.float64) - n64).max()))
    assert worst64 < 1e-4  # MLP positions within 1e-4 mm of the fp64 matrix-form definition
    return n_paths


def test_rows_bit_exact_config0(oracle_mod, pct, torch_cuda):
    cfg = synth.config(0)
    H = synth.generate_numpy(cfg, 12000)
    assert _check_rows(oracle_mod, pct, torch_cuda, cfg, H) > 8000


@pytest.mark.parametrize("index,n,stride", [(1, 4000, 1), (2, 3000, 1), (3, 3000, 1), (4, 1500, 1)])
def test_rows_bit_exact_larger_grids(oracle_mod, pct, torch_cuda, index, n, stride):
    """Samples of the larger workloads: paths of 100-256 segments span 4-9 lane rounds and a ragged tail."""
    cfg = synth.config(index)
    H = synth.generate_numpy(cfg, n)
    assert _check_rows(oracle_mod, pct, torch_cuda, cfg, H, stride) > n // 2


def test_rows_bit_exact_odd_geometry(oracle_mod, pct, torch_cuda):
    """Non-square grid, non-unit voxel (h = 0.8 mm), odd sizes: nmin = 45 -> hull radius 18 mm."""
    base = synth.config(0)
    cfg = synth.Config(9, "odd", 6000, 45, 71, 5, 0.8, 37, 500, 0.1, 1, base.shapes * 0.5, seed=99)
    H = synth.generate_numpy(cfg, 6000)
    assert _check_rows(oracle_mod, pct, torch_cuda, cfg, H) > 1500


def test_projection_index_past_the_tables_is_the_last_angle(oracle_mod, pct, torch_cuda):
    """DESIGN.md R24 / include/pct.h pct_set_histories: "a proj[i] >= n_proj is clamped to n_proj-1".  Every third history
    carries an index past the angle tables (n_proj, n_proj + 5, 65535): rows bit-exact and a DROP block against the oracle,
    which reads the same rule (pinned on the CPU in test_oracle_drop.py)."""
    cfg = synth.config(0)
    H = synth.generate_numpy(cfg, 3000)
    n_proj = H["proj_cos"].shape[0]
    H["proj"] = H["proj"].copy()
    sel = np.arange(0, 3000, 3)
    H["proj"][sel] = np.array([n_proj, n_proj + 5, 65535], dtype=np.uint16)[np.arange(sel.size) % 3]
    assert _check_rows(oracle_mod, pct, torch_cuda, cfg, H) > 2000
    stats = _block_parity(oracle_mod, pct, torch_cuda, cfg, H, 0, 3000, synth.rsp_volume(cfg) * 0.9)
    assert stats[0] > 2000


def test_rule_reciprocal_and_square_root_are_ieee_on_every_argument_in_range(pct, torch_cuda):
    """Bit-exactness against the CPU side rests on the rule's 1/det and sqrt(squared length) -- hardware approximation +
    one FMA Newton step (pct_rule.cuh) -- being the correctly rounded IEEE results the oracle gets from gcc's division
    and sqrtf.  Swept in full, not sampled: every fp32 bit pattern of the ranges DESIGN.md states for the two arguments
    (det 1e-16 .. 1e19; squared segment length from 8e-7 mm^2 up, here to the largest finite float) and, beyond them, of
    [2^-100, 2^100] for the reciprocal: 1.0e9 + 1.2e9 + 1.7e9 arguments, zero mismatches."""
    bits = lambda v: int(np.float32(v).view(np.uint32))
    s = torch_cuda.cuda.current_stream().cuda_stream
    for which, lo, hi in ((0, 1e-16, 1e19), (1, 8e-7, np.finfo(np.float32).max), (0, 2.0 ** -100, 2.0 ** 100)):
        assert hi > lo and bits(hi) - bits(lo) > 5e8
        bad, first = pct.pct_debug_rule_sweep(which, bits(lo), bits(hi), s)
        assert bad == 0, (which, bad, hex(first))
    # the check can fail: outside the stated range the shortcut is NOT exact (the reciprocal of a huge argument is denormal, flushed to zero)
    bad, first = pct.pct_debug_rule_sweep(0, bits(2.0 ** 126), bits(2.0 ** 127), s)
    assert bad > 0 and first >= bits(2.0 ** 126)


def test_rows_handcrafted_edge_cases(oracle_mod, pct, torch_cuda):
    """Misses, grazing rays, NaN, paths leaving the grid in z (dropped segments break runs),
    exactly axis-aligned central rays, steep rays."""
    cfg = synth.config(0)
    cs, sn = synth.generate.angle_table(cfg.n_angles)
    rows = [
        # t_in v_in t_out v_out tht_in thv_in tht_out thv_out proj
        (0, 0, 0, 0, 0, 0, 0, 0, 0),            # central ray, axis aligned
        (0, 0, 0, 0, 0, 0, 0, 0, 22),           # central ray, 88 degrees
        (40, 0, 40, 0, 0, 0, 0, 0, 3),          # misses the hull
        (31.9999, 0, 31.9999, 0, 0, 0, 0, 0, 5),  # grazing: L tiny
        (32.0, 0, 32.0, 0, 0, 0, 0, 0, 5),      # tangent: disc == 0 -> skipped
        (0, 4.5, 0, 0, 0, 0, 0, 0, 1),          # enters above the grid
        (0, 3.9, 0, 3.9, 0, 0.02, 0, 0.02, 1),  # v rises: entry inside, exit hull point outside -> skipped
        (0, 3.99, 0, -3.99, 0, -0.0831, 0, -0.0831, 7),  # steep in v, stays inside
        (float("nan"), 0, 0, 0, 0, 0, 0, 0, 0),
        (0, 0, float("inf"), 0, 0, 0, 0, 0, 0),
        (5, 1, 9, -1, 0.05, -0.02, 0.03, -0.02, 11),  # large kink
        (-20, -3.5, -22, 3.5, -0.02, 0.07, -0.02, 0.07, 45),
        (10, 0, 10, 0, 0.3, 0, 0.3, 0, 17),     # 17 degree slope
        (0, 0, 0.5, 0, 0, 0, 0, 0, 89),
        (0, 3.19, 0, 3.19, 0, 0.05, 0, -0.05, 2),  # bulges above the grid: dropped segments split the row
        (0, 3.73, 0, 3.73, 0, 0.01, 0, -0.01, 2),  # only the middle of the path is above the grid
    ]
    a = np.array(rows, dtype=np.float64)
    H = dict(t_in=a[:, 0], v_in=a[:, 1], t_out=a[:, 2], v_out=a[:, 3], tht_in=a[:, 4], thv_in=a[:, 5],
             tht_out=a[:, 6], thv_out=a[:, 7], wepl=np.ones(len(rows)), proj=a[:, 8].astype(np.uint16),
             proj_cos=cs, proj_sin=sn)
    H = {k: (v.astype(np.float32) if v.dtype == np.float64 else v) for k, v in H.items()}
    n_paths = _check_rows(oracle_mod, pct, torch_cuda, cfg, H, t64_every=10 ** 9)
    assert n_paths == 10


def _block_parity(oracle, pct, torch, cfg, H, first, count, x0):
    geom = oracle_geom(oracle, cfg)
    hs = oracle.Histories(H)
    D = to_device(H)
    M = cfg.n_voxels
    ctx = _ctx(pct, torch, cfg)
    try:
        pct.pct_set_histories(ctx, hs.n, D)
        pct.pct_set_image(ctx, torch.from_numpy(x0.astype(np.float32)).cuda(), M)
        delta = torch.zeros(M, dtype=torch.float32, device="cuda")
        cnt = torch.zeros(M, dtype=torch.float32, device="cuda")
        pct.pct_debug_block(ctx, first, count, delta, cnt)
        pct.pct_synchronize(ctx)
        # the accumulator must be left zeroed: a second call gives the same answer
        delta2 = torch.zeros_like(delta)
        cnt2 = torch.zeros_like(cnt)
        pct.pct_debug_block(ctx, first, count, delta2, cnt2)
        pct.pct_synchronize(ctx)
    finally:
        pct.pct_destroy(ctx)
    d_ref, c_ref, stats = oracle.block_accumulate(geom, hs, first, count, x0.astype(np.float32).astype(np.float64))
    assert np.array_equal(cnt.cpu().numpy(), c_ref.astype(np.float32))  # integers: exact
    assert np.array_equal(cnt2.cpu().numpy(), c_ref.astype(np.float32))
    d = delta.cpu().numpy().astype(np.float64)
    scale = np.linalg.norm(d_ref)
    assert np.linalg.norm(d - d_ref) <= 2e-5 * scale
    assert np.abs(d - d_ref).max() <= 2e-4 * max(1.0, np.abs(d_ref).max())
    assert np.linalg.norm(delta2.cpu().numpy() - d_ref) <= 2e-5 * scale
    return stats


def test_block_accumulate_from_zero_and_from_an_image(oracle_mod, pct, torch_cuda):
    cfg = synth.config(0)
    H = synth.generate_numpy(cfg, 9000)
    st = _block_parity(oracle_mod, pct, torch_cuda, cfg, H, 0, 9000, np.zeros(cfg.n_voxels))
    assert st[0] > 6000
    x0 = synth.rsp_volume(cfg) * 0.9
    _block_parity(oracle_mod, pct, torch_cuda, cfg, H, 1234, 4321, x0)  # ragged range, non-zero residuals near 10 %


def test_block_accumulate_config2_sample(oracle_mod, pct, torch_cuda):
    cfg = synth.config(2)
    H = synth.generate_numpy(cfg, 20000)
    x0 = synth.rsp_volume(cfg) * 0.8
    _block_parity(oracle_mod, pct, torch_cuda, cfg, H, 0, 20000, x0)


def _run_parity(oracle, pct, torch, cfg, H, lam, block, n_iter, x0=None, per_call=1):
    """Full DROP run, image compared after every iteration."""
    geom = oracle_geom(oracle, cfg)
    hs = oracle.Histories(H)
    D = to_device(H)
    M = cfg.n_voxels
    x_ref = np.zeros(M) if x0 is None else x0.astype(np.float32).astype(np.float64)
    ctx = _ctx(pct, torch, cfg)
    out = torch.zeros(M, dtype=torch.float32, device="cuda")
    worst = 0.0
    try:
        pct.pct_set_histories(ctx, hs.n, D)
        if x0 is not None:
            pct.pct_set_image(ctx, x0.astype(np.float32), M)  # host pointer
        for it in range(0, n_iter, per_call):
            pct.pct_iterate(ctx, lam, block, per_call)
            pct.pct_get_image(ctx, out, M)
            x_ref, stats = oracle.drop_iterate(geom, hs, lam, block, per_call, x_ref)
            x = out.cpu().numpy().astype(np.float64)
            rel = np.linalg.norm(x - x_ref) / np.linalg.norm(x_ref)
            worst = max(worst, rel)
            assert rel <= REL_L2_PER_ITER, "iteration %d: rel L2 %.3g" % (it, rel)
            gs = pct.pct_get_stats(ctx)
            assert (gs["rows"], gs["nnz"]) == stats  # non-empty rows and non-zeros of the sweep: exact
        assert np.abs(x - x_ref).max() <= ABS_FINAL
    finally:
        pct.pct_destroy(ctx)
    return x, x_ref, worst


def test_full_run_config0(oracle_mod, pct, torch_cuda):
    """BASELINE.json configs[0] exactly: 1e5 protons, 64x64x8, B = 1e3, lambda = 0.1, 1 iteration."""
    cfg = synth.config(0)
    H = synth.generate_numpy(cfg)
    x, x_ref, _ = _run_parity(oracle_mod, pct, torch_cuda, cfg, H, cfg.lam, cfg.block_size, cfg.n_iter)
    assert np.linalg.norm(x_ref) > 1.0  # the image moved


def test_config0_several_iterations_and_ragged_blocks(oracle_mod, pct, torch_cuda):
    cfg = synth.config(0)
    H = synth.generate_numpy(cfg, 30011)  # prime-ish: last block short (30011 = 42*700 + 611)
    x, x_ref, _ = _run_parity(oracle_mod, pct, torch_cuda, cfg, H, 0.5, 700, 4)
    # sanity: after 4 sweeps the water cylinder is near RSP 1 in the central slice
    vol = x.reshape(cfg.nz, cfg.ny, cfg.nx)
    assert 0.7 < vol[4, 32, 40] < 1.3


def test_config1_sample(oracle_mod, pct, torch_cuda):
    """configs[1] geometry and parameters on its first 4e5 histories (40 blocks of 1e4), 2 iterations."""
    cfg = synth.config(1)
    H = synth.generate_numpy(cfg, 400_000)
    _run_parity(oracle_mod, pct, torch_cuda, cfg, H, cfg.lam, cfg.block_size, 2)


def _carp_parity(oracle, pct, torch, cfg, H, lam, block, n_iter, n_strings, x0=None, order=None):
    """CARP run (R27-R29), image compared with the oracle after every iteration."""
    geom = oracle_geom(oracle, cfg)
    hs = oracle.Histories(H)
    D = to_device(H)
    M = cfg.n_voxels
    x_ref = np.zeros(M) if x0 is None else x0.astype(np.float32).astype(np.float64)
    ctx = _ctx(pct, torch, cfg)
    out = torch.zeros(M, dtype=torch.float32, device="cuda")
    try:
        if order is not None:
            pct.pct_set_option(ctx, pct.PCT_OPT_ORDER, order)
        pct.pct_set_histories(ctx, hs.n, D)
        if x0 is not None:
            pct.pct_set_image(ctx, x0.astype(np.float32), M)
        for it in range(n_iter):
            pct.pct_iterate_carp(ctx, lam, block, 1, n_strings)
            pct.pct_get_image(ctx, out, M)
            x_ref = oracle.carp_iterate(geom, hs, lam, block, 1, n_strings, x_ref)
            x = out.cpu().numpy().astype(np.float64)
            rel = np.linalg.norm(x - x_ref) / np.linalg.norm(x_ref)
            assert rel <= REL_L2_PER_ITER, "iteration %d: rel L2 %.3g" % (it, rel)
        assert np.abs(x - x_ref).max() <= ABS_FINAL
        # the counters of the last iteration: the strings' sweeps added up = one sweep over all histories (rows and
        # non-zeros are properties of the paths, not of the image)
        _, st = oracle.drop_iterate(geom, hs, lam, block, 1, np.zeros(M))
        gs = pct.pct_get_stats(ctx)
        assert (gs["rows"], gs["nnz"]) == st
    finally:
        pct.pct_destroy(ctx)
    return x, x_ref


@pytest.mark.parametrize("n_strings", [1, 4, 7])
def test_carp_config0(oracle_mod, pct, torch_cuda, n_strings):
    """configs[0] data and parameters, CARP with 1 / 4 / 7 strings (ragged strings and last blocks), 3 iterations."""
    cfg = synth.config(0)
    H = synth.generate_numpy(cfg, 60_011)
    x, x_ref = _carp_parity(oracle_mod, pct, torch_cuda, cfg, H, 0.5, cfg.block_size, 3, n_strings)
    assert np.linalg.norm(x_ref) > 1.0


@pytest.mark.parametrize("n_strings", [2, 3])
def test_carp_strings_long_enough_for_the_graph_loop(oracle_mod, pct, torch_cuda, n_strings):
    """Strings of 150+ blocks: pct_iterate_carp replays every string's block loop from a CUDA graph of 64 (accumulate,
    update) pairs (from 128 blocks per string on) and launches the ragged rest one by one; the second call reuses the
    graphs.  Same comparison as the short strings."""
    cfg = synth.config(0)
    H = synth.generate_numpy(cfg, 60_011)
    block = 200 if n_strings == 2 else 130  # 151 / 154 blocks per string, the last one ragged
    x, x_ref = _carp_parity(oracle_mod, pct, torch_cuda, cfg, H, 0.5, block, 2, n_strings)
    assert np.linalg.norm(x_ref) > 1.0


@pytest.mark.parametrize("order", [1, 2])
def test_carp_config1_sample_from_an_image(oracle_mod, pct, torch_cuda, order):
    """configs[1] geometry and block size, 3 strings of 1e5 histories, two iterations from a non-trivial image;
    order = 2 (pct_set_option PCT_OPT_ORDER) forces the depth-slab ordering of every string's blocks."""
    cfg = synth.config(1)
    H = synth.generate_numpy(cfg, 300_000)
    _carp_parity(oracle_mod, pct, torch_cuda, cfg, H, cfg.lam, cfg.block_size, 2, 3, x0=synth.rsp_volume(cfg) * 0.8, order=order)


def test_carp_one_string_is_drop_and_arguments(pct, torch_cuda):
    torch = torch_cuda
    cfg = synth.config(0)
    H = synth.generate_numpy(cfg, 20_000)
    D = to_device(H)
    imgs = []
    for carp in (False, True):
        ctx = _ctx(pct, torch, cfg)
        try:
            if carp:
                with pytest.raises(pct.PctError):
                    pct.pct_iterate_carp(ctx, 0.5, 1000, 1, 2)  # no histories yet
            pct.pct_set_histories(ctx, 20_000, D)
            if carp:
                for bad in (0, 65, -1):
                    with pytest.raises(pct.PctError):
                        pct.pct_iterate_carp(ctx, 0.5, 1000, 1, bad)
                pct.pct_iterate_carp(ctx, 0.5, 1000, 2, 1)
                pct.pct_iterate_carp(ctx, 0.5, 1000, 0, 3)  # n_iter = 0: nothing happens
            else:
                pct.pct_iterate(ctx, 0.5, 1000, 2)
            out = torch.zeros(cfg.n_voxels, dtype=torch.float32, device="cuda")
            pct.pct_get_image(ctx, out, cfg.n_voxels)
            imgs.append(out.cpu().numpy())
        finally:
            pct.pct_destroy(ctx)
    assert np.linalg.norm(imgs[0] - imgs[1]) <= 1e-5 * np.linalg.norm(imgs[0])


def test_carp_distributed_on_one_rank_is_the_drop_sweeps(pct, torch_cuda):
    """replicas.carp_distributed_pct (one string per rank, all-reduce of the image per iteration) at world = 1:
    get / set of the device image around every sweep must leave n_iter DROP sweeps."""
    from paper_1707_05014_b200 import replicas

    torch = torch_cuda
    cfg = synth.config(0)
    D = to_device(synth.generate_numpy(cfg, 20_000))
    imgs = []
    for dist_form in (False, True):
        ctx = _ctx(pct, torch, cfg)
        try:
            pct.pct_set_histories(ctx, 20_000, D)
            if dist_form:
                replicas.carp_distributed_pct(pct, ctx, cfg.n_voxels, 0.5, 1000, 3, 1)
            else:
                pct.pct_iterate(ctx, 0.5, 1000, 3)
            out = torch.zeros(cfg.n_voxels, dtype=torch.float32, device="cuda")
            pct.pct_get_image(ctx, out, cfg.n_voxels)
            imgs.append(out.cpu().numpy())
        finally:
            pct.pct_destroy(ctx)
    assert np.abs(imgs[0]).max() > 0.1
    assert np.linalg.norm(imgs[0] - imgs[1]) <= 1e-5 * np.linalg.norm(imgs[0])


@pytest.fixture()
def spline_oracle(oracle_mod):
    oracle_mod.set_path_model(1)
    yield oracle_mod
    oracle_mod.set_path_model(0)


def test_spline_path_model_rows_and_run(spline_oracle, pct, torch_cuda):
    """PCT_PATH_SPLINE (NEXT-3, R30) against the oracle in the same mode: voxel sequences bit-exact on configs[0]
    and on configs[3] geometry, a full DROP run and a CARP run within the DROP tolerances; and switching back to
    the most-likely path gives the default rows again."""
    torch = torch_cuda
    oracle = spline_oracle
    for index, n in ((0, 4000), (3, 1500)):
        cfg = synth.config(index)
        H = synth.generate_numpy(cfg, n)
        geom = oracle_geom(oracle, cfg)
        hs = oracle.Histories(H)
        table = oracle.sigma1_table(geom.h, geom.nmin)
        ctx = _ctx(pct, torch, cfg)
        D = to_device(H)  # borrowed by the library: kept alive until pct_destroy
        try:
            pct.pct_set_histories(ctx, n, D)
            default = _gpu_rows(pct, torch, ctx, 0, n, geom.nmin)
            pct.pct_set_path_model(ctx, pct.PCT_PATH_SPLINE)
            nseg, nnz, seg_idx, seg_len, row_len, nodes = _gpu_rows(pct, torch, ctx, 0, n, geom.nmin)
            differ = 0
            for i in range(n):
                r = oracle.row_f32(geom, hs.hist(i), table)
                assert nseg[i] == r["nseg"] and nnz[i] == r["nnz"], i
                assert np.array_equal(seg_idx[i, :r["nseg"]], r["seg_idx"]), i
                if r["nseg"]:
                    assert np.array_equal(nodes[i, :r["nseg"] + 1], r["nodes"]), i  # fp32 node positions: bitwise
                differ += int(not np.array_equal(seg_idx[i], default[2][i]))
            assert differ > 0  # the two models do walk different voxels now and then
            pct.pct_set_path_model(ctx, pct.PCT_PATH_MLP)
            again = _gpu_rows(pct, torch, ctx, 0, n, geom.nmin)
            assert np.array_equal(again[2], default[2])
            with pytest.raises(pct.PctError):
                pct.pct_set_path_model(ctx, 7)
        finally:
            pct.pct_destroy(ctx)
    # full runs in spline mode
    cfg = synth.config(0)
    H = synth.generate_numpy(cfg, 30_011)
    geom = oracle_geom(oracle, cfg)
    hs = oracle.Histories(H)
    M = cfg.n_voxels
    ctx = _ctx(pct, torch, cfg)
    out = torch.zeros(M, dtype=torch.float32, device="cuda")
    D = to_device(H)
    try:
        pct.pct_set_histories(ctx, hs.n, D)
        pct.pct_set_path_model(ctx, pct.PCT_PATH_SPLINE)
        x_ref = np.zeros(M)
        for it in range(3):
            if it < 2:
                pct.pct_iterate(ctx, 0.5, 700, 1)
                x_ref, _ = oracle.drop_iterate(geom, hs, 0.5, 700, 1, x_ref)
            else:
                pct.pct_iterate_carp(ctx, 0.5, 700, 1, 3)
                x_ref = oracle.carp_iterate(geom, hs, 0.5, 700, 1, 3, x_ref)
            pct.pct_get_image(ctx, out, M)
            x = out.cpu().numpy().astype(np.float64)
            assert np.linalg.norm(x - x_ref) <= REL_L2_PER_ITER * np.linalg.norm(x_ref)
        assert np.abs(x - x_ref).max() <= ABS_FINAL
    finally:
        pct.pct_destroy(ctx)


@pytest.mark.parametrize("index,n", [(3, 250_000), (4, 260_000)])
def test_bench_launch_configuration_sample(oracle_mod, pct, torch_cuda, index, n):
    """configs[3] / configs[4] geometry with THEIR block sizes (1e5 / 2e5 histories per launch: the
    persistent grid, queue schedule and chunk sizes bench.py times), full blocks plus a ragged one,
    two sweeps from a non-trivial image; every voxel compared with the oracle."""
    import synth.cuda_gen as cuda_gen

    cfg = synth.config(index)
    D = cuda_gen.generate_cuda(cfg, n)  # the generator bench.py uses; ONE set of arrays feeds both sides
    H = {k: v.cpu().numpy() for k, v in D.items()}
    H["proj"] = H["proj"].view(np.uint16)
    del D
    x0 = synth.rsp_volume(cfg) * 0.8
    _run_parity(oracle_mod, pct, torch_cuda, cfg, H, cfg.lam, cfg.block_size, 2, x0=x0)


def test_graph_path_and_call_splitting(oracle_mod, pct, torch_cuda):
    """>= 128 (accumulate, update) pairs go through the replayed CUDA graph; one call with
    n_iter = 3 equals three calls with n_iter = 1 (the image is the whole solver state)."""
    cfg = synth.config(0)
    H = synth.generate_numpy(cfg, 20000)
    xa, ref_a, _ = _run_parity(oracle_mod, pct, torch_cuda, cfg, H, 0.3, 100, 3, per_call=3)   # 600 pairs in one call
    xb, ref_b, _ = _run_parity(oracle_mod, pct, torch_cuda, cfg, H, 0.3, 100, 3, per_call=1)   # 200 pairs per call
    assert np.array_equal(ref_a, ref_b)
    assert np.linalg.norm(xa - xb) <= 1e-5 * np.linalg.norm(xa)


def test_degenerate_inputs(oracle_mod, pct, torch_cuda):
    torch = torch_cuda
    cfg = synth.config(0)
    H = synth.generate_numpy(cfg, 500)
    # a single history, block larger than n
    _run_parity(oracle_mod, pct, torch, cfg, slice_hist(H, slice(7, 8)), 1.0, 1000, 2)
    # block size 1 (Kaczmarz order), lambda = 1
    _run_parity(oracle_mod, pct, torch, cfg, slice_hist(H, slice(0, 60)), 1.0, 1, 1)
    # every history misses the hull: the image stays at x0
    Hm = {k: v.copy() for k, v in H.items()}
    Hm["t_in"][:] = 45.0
    Hm["t_out"][:] = 45.0
    Hm["tht_in"][:] = 0
    Hm["tht_out"][:] = 0
    D = to_device(Hm)
    ctx = _ctx(pct, torch, cfg)
    try:
        x0 = np.random.default_rng(0).uniform(0, 1, cfg.n_voxels).astype(np.float32)
        pct.pct_set_histories(ctx, 500, D)
        pct.pct_set_image(ctx, x0, cfg.n_voxels)
        pct.pct_iterate(ctx, 0.5, 100, 2)
        out = np.zeros(cfg.n_voxels, dtype=np.float32)
        pct.pct_get_image(ctx, out, cfg.n_voxels)  # host destination
        assert np.array_equal(out, x0)
        assert pct.pct_get_stats(ctx)["rows"] == 0
    finally:
        pct.pct_destroy(ctx)


def test_host_entry_point_matches_device_entry_point(oracle_mod, pct, torch_cuda):
    from helpers import to_host_pct

    torch = torch_cuda
    cfg = synth.config(0)
    H = synth.generate_numpy(cfg, 5000)
    imgs = []
    for host in (False, True):
        ctx = _ctx(pct, torch, cfg)
        try:
            if host:
                pct.pct_set_histories_host(ctx, 5000, to_host_pct(H))
            else:
                D = to_device(H)
                pct.pct_set_histories(ctx, 5000, D)
            pct.pct_iterate(ctx, 0.2, 500, 2)
            out = np.zeros(cfg.n_voxels, dtype=np.float32)
            pct.pct_get_image(ctx, out, cfg.n_voxels)
            imgs.append(out)
        finally:
            pct.pct_destroy(ctx)
    assert np.linalg.norm(imgs[0] - imgs[1]) <= 1e-5 * np.linalg.norm(imgs[0])


@pytest.mark.parametrize("order", [1, 2])
def test_pipelined_host_upload_spans_several_chunks(pct, torch_cuda, order):
    """pct_set_histories_host uploads in chunks of 2^20 .. 2^24 histories on a copy stream and the first
    sweep starts before the upload has finished: 9.5e6 histories (five chunks, the last one ragged) from
    pinned host arrays must give the image the device entry point gives -- for the first sweep, after
    the host arrays are overwritten once pct_synchronize has returned, for the inspection entry point
    on the last chunk, and for a SECOND set of the same size, which reuses the device block.  order = 2
    (pct_set_option PCT_OPT_ORDER) forces the depth-slab ordering of the DROP blocks (by default only grids larger than the L2 get it), whose
    sort then runs batch by batch behind the upload."""
    import synth.cuda_gen as cuda_gen

    torch = torch_cuda
    cfg = synth.config(0)
    n, B = 9_500_000, 20_000
    tables = ("proj_cos", "proj_sin")
    D2 = synth.to_pct_names(cuda_gen.generate_cuda(cfg, 2 * n))
    sets = [{k: (v if k in tables else v[i * n:(i + 1) * n].contiguous()) for k, v in D2.items()} for i in range(2)]
    res = []
    for use_host in (False, True):
        ctx = _ctx(pct, torch, cfg)
        try:
            pct.pct_set_option(ctx, pct.PCT_OPT_ORDER, order)
            for D in sets:
                if use_host:
                    host = {k: torch.empty(v.shape, dtype=v.dtype, pin_memory=True).copy_(v) for k, v in D.items()}
                    torch.cuda.synchronize()
                    pct.pct_set_histories_host(ctx, n, host)
                else:
                    pct.pct_set_histories(ctx, n, D)
                pct.pct_iterate(ctx, cfg.lam, B, 1)
                if use_host:
                    pct.pct_synchronize(ctx)
                    host["wepl"].fill_(1.0e9)  # the library may not read the host arrays any more
                pct.pct_iterate(ctx, cfg.lam, B, 1)
                out = torch.empty(cfg.n_voxels, dtype=torch.float32, device="cuda")
                pct.pct_get_image(ctx, out, cfg.n_voxels)
                res.append(out.cpu().numpy())
                nseg, nnz = _gpu_rows(pct, torch, ctx, n - 64, 64, min(cfg.nx, cfg.ny))[:2]
                res.append(np.concatenate([nseg, nnz]))
        finally:
            pct.pct_destroy(ctx)
    dev, hst = res[:4], res[4:]
    assert np.isfinite(dev[0]).all() and np.abs(dev[0]).max() > 0.1
    assert not np.array_equal(dev[1], dev[3])  # the two sets differ
    for i in (0, 2):
        assert np.linalg.norm(dev[i] - hst[i]) <= 1e-5 * np.linalg.norm(dev[i])
        assert np.array_equal(dev[i + 1], hst[i + 1])


def test_error_reporting(pct, torch_cuda):
    torch = torch_cuda
    cfg = synth.config(0)
    ctx = _ctx(pct, torch, cfg)
    try:
        with pytest.raises(pct.PctError) as e:
            pct.pct_iterate(ctx, 0.1, 10, 1)
        assert e.value.code == -4  # PCT_ESTATE: no histories yet
        H = synth.generate_numpy(cfg, 100)
        D = to_device(H)
        with pytest.raises(pct.PctError) as e:
            pct.pct_set_histories(ctx, 0, D)
        assert e.value.code == -1
        from helpers import to_host_pct

        with pytest.raises(pct.PctError) as e:
            pct.pct_set_histories(ctx, 100, to_host_pct(H))  # host pointers where device is required
        assert e.value.code == -1
        pct.pct_set_histories(ctx, 100, D)
        for lam, b, it in [(0.0, 10, 1), (2.0, 10, 1), (0.1, 0, 1), (0.1, 10, -1), (0.1, 2 ** 24 + 1, 1), (float("nan"), 10, 1)]:
            with pytest.raises(pct.PctError) as e:
                pct.pct_iterate(ctx, lam, b, it)
            assert e.value.code == -1
        with pytest.raises(pct.PctError):
            pct.pct_get_image(ctx, torch.zeros(10, device="cuda"), 10)
        pct.pct_iterate(ctx, 0.1, 10, 0)  # zero iterations: a no-op
        pct.pct_iterate(ctx, 0.1, 10, 1)
        pct.pct_synchronize(ctx)
    finally:
        pct.pct_destroy(ctx)


def test_carp_across_two_contexts_averaged_in_place_is_carp_with_two_strings(oracle_mod, pct, torch_cuda):
    """The multi-GPU form of CARP (replicas.carp_distributed_pct: one string per rank, the average taken in place on the
    library's own image array) with the two ranks played by two contexts of ONE process, one after the other (their
    kernels never wait on one another): the all-reduce is written out as the sum of the two storage arrays / 2.
    Must equal pct_iterate_carp(P = 2) on one context and the oracle's CARP with two strings."""
    from paper_1707_05014_b200 import replicas

    torch = torch_cuda
    cfg = synth.config(0)
    n, B, lam, iters = 30_011, 700, 0.5, 3
    H = synth.generate_numpy(cfg, n)
    D = to_device(H)
    M = cfg.n_voxels
    tables = ("proj_cos", "proj_sin")
    ctxs, xs = [], []
    try:
        for r in range(2):
            lo, hi = replicas.string_range(r, 2, n)
            Dr = {k: (v if k in tables else v[lo:hi]) for k, v in D.items()}
            c = _ctx(pct, torch, cfg)
            ctxs.append((c, Dr))
            pct.pct_set_histories(c, hi - lo, Dr)
            addr, n_slots = pct.pct_image_storage(c)
            xs.append(torch.as_tensor(replicas._DeviceArray(addr, n_slots), device="cuda"))
        assert xs[0].numel() >= M and xs[0].numel() == xs[1].numel()
        for _ in range(iters):
            for c, _d in ctxs:
                pct.pct_iterate(c, lam, B, 1)
            mean = (xs[0] + xs[1]) / 2  # what all_reduce(sum) followed by /= world leaves on every rank
            xs[0].copy_(mean)
            xs[1].copy_(mean)
        out = torch.zeros(M, dtype=torch.float32, device="cuda")
        pct.pct_get_image(ctxs[1][0], out, M)
        got = out.cpu().numpy().astype(np.float64)
    finally:
        for c, _d in ctxs:
            pct.pct_destroy(c)
    geom = oracle_geom(oracle_mod, cfg)
    x_ref = oracle_mod.carp_iterate(geom, oracle_mod.Histories(H), lam, B, iters, 2, np.zeros(M))
    assert np.linalg.norm(got - x_ref) <= REL_L2_PER_ITER * np.linalg.norm(x_ref)
    assert np.abs(got - x_ref).max() <= ABS_FINAL


def test_carp_across_contexts_with_tvs_takes_one_step_per_iteration(oracle_mod, pct, torch_cuda):
    """TVS in the one-string-per-rank form of CARP (replicas.carp_distributed_pct(tvs=True)): PAPER.md:113 puts the step
    "just once to the initial solution at the start of each iteration", so every rank takes ONE step on the common image
    and then sweeps its string without further steps -- pct_iterate_carp with one string.  At world = 1 through
    carp_distributed_pct itself, and with two ranks played by two contexts of this process (as in the test above), against
    the oracle's CARP with a TVS step per iteration and P = 1 / 2 strings."""
    from oracle import tvs

    from paper_1707_05014_b200 import replicas

    torch = torch_cuda
    cfg = synth.config(0)
    n, B, lam, iters = 24_000, 1000, 0.5, 3
    beta0, gamma, levels = 0.4, 0.9, 4
    H = synth.generate_numpy(cfg, n)
    D = to_device(H)
    M = cfg.n_voxels
    geom = oracle_geom(oracle_mod, cfg)
    hs = oracle_mod.Histories(H)
    tables = ("proj_cos", "proj_sin")
    out = torch.zeros(M, dtype=torch.float32, device="cuda")
    for world in (1, 2):
        ctxs, xs = [], []
        try:
            for r in range(world):
                lo, hi = replicas.string_range(r, world, n)
                Dr = {k: (v if k in tables else v[lo:hi]) for k, v in D.items()}
                c = _ctx(pct, torch, cfg)
                ctxs.append((c, Dr))
                pct.pct_set_histories(c, hi - lo, Dr)
                pct.pct_set_tvs(c, beta0, gamma, levels)
                addr, n_slots = pct.pct_image_storage(c)
                xs.append(torch.as_tensor(replicas._DeviceArray(addr, n_slots), device="cuda"))
            if world == 1:
                replicas.carp_distributed_pct(pct, ctxs[0][0], M, lam, B, iters, 1, tvs=True)
            else:
                for _ in range(iters):
                    for c, _d in ctxs:
                        pct.pct_iterate_carp(c, lam, B, 1, 1)  # the sweep carp_distributed_pct(tvs=True) runs on a rank
                    mean = (xs[0] + xs[1]) / 2
                    xs[0].copy_(mean)
                    xs[1].copy_(mean)
            pct.pct_get_image(ctxs[-1][0], out, M)
            got = out.cpu().numpy().astype(np.float64)
            states = [pct.pct_get_tvs_state(c) for c, _d in ctxs]
        finally:
            for c, _d in ctxs:
                pct.pct_destroy(c)
        x_ref, beta, infos = tvs.carp_iterate_tvs(oracle_mod, geom, hs, lam, B, iters, world, np.zeros(M), beta0, gamma, levels)
        assert np.linalg.norm(got - x_ref) <= REL_L2_PER_ITER * np.linalg.norm(x_ref), world
        for st in states:  # one step per iteration on every rank, the same one
            assert st["steps"] == iters and st["level"] == infos[-1]["level"]
            assert st["beta"] == pytest.approx(beta, rel=1e-5)


@pytest.mark.parametrize("n_strings", [2, 3])
def test_carp_on_an_odd_grid(oracle_mod, pct, torch_cuda, n_strings):
    """CARP with several strings on the 45 x 71 x 5 grid (15975 voxels: not a multiple of four; the strings' images and
    accumulators must each start on a 16-byte boundary, and the stored slices are padded to even sides)."""
    base = synth.config(0)
    cfg = synth.Config(9, "odd", 9000, 45, 71, 5, 0.8, 37, 500, 0.1, 1, base.shapes * 0.5, seed=99)
    H = synth.generate_numpy(cfg, 9000)
    x, x_ref = _carp_parity(oracle_mod, pct, torch_cuda, cfg, H, 0.5, 500, 2, n_strings)
    assert np.linalg.norm(x_ref) > 0.5


@pytest.mark.parametrize("index,n", [(0, 6001), (3, 2500), (4, 1001)])
def test_rows_of_the_pair_walk_bit_exact(oracle_mod, pct, torch_cuda, index, n):
    """The walk of the throughput kernel (k_drop_pair: two histories per warp, sixteen lanes each, one chunk size per
    pair) inspected directly: pct_set_option(PCT_OPT_ROWS_PAIR, 1) makes pct_debug_rows walk histories (2w, 2w+1) side by side with that code.
    Voxel sequences, segment lengths (bitwise) and merged rows against the oracle; odd counts leave a lone last history."""
    torch = torch_cuda
    cfg = synth.config(index)
    H = synth.generate_numpy(cfg, n)
    geom = oracle_geom(oracle_mod, cfg)
    hs = oracle_mod.Histories(H)
    D = to_device(H)
    ms = geom.nmin + 2
    ctx = _ctx(pct, torch, cfg)
    try:
        pct.pct_set_option(ctx, pct.PCT_OPT_ROWS_PAIR, 1)
        with pytest.raises(pct.PctError):
            pct.pct_set_option(ctx, 7, 1)
        with pytest.raises(pct.PctError):
            pct.pct_set_option(ctx, pct.PCT_OPT_ORDER, 3)
        pct.pct_set_histories(ctx, n, D)
        nseg = torch.zeros(n, dtype=torch.int32, device="cuda")
        nnz = torch.zeros(n, dtype=torch.int32, device="cuda")
        seg_idx = torch.full((n, ms), -7, dtype=torch.int32, device="cuda")
        seg_len = torch.zeros((n, ms), dtype=torch.float32, device="cuda")
        row_len = torch.zeros((n, ms), dtype=torch.float32, device="cuda")
        pct.pct_debug_rows(ctx, 0, n, ms, nseg, nnz, seg_idx, seg_len, row_len, None)  # (no nodes: the pair walk is used)
        pct.pct_synchronize(ctx)
        nseg, nnz, seg_idx, seg_len, row_len = (t.cpu().numpy() for t in (nseg, nnz, seg_idx, seg_len, row_len))
    finally:
        pct.pct_destroy(ctx)
    table = oracle_mod.sigma1_table(geom.h, geom.nmin)
    paths = 0
    for i in range(n):
        r = oracle_mod.row_f32(geom, hs.hist(i), table)
        ns = r["nseg"]
        assert nseg[i] == ns and nnz[i] == r["nnz"], i
        if ns == 0:
            continue
        paths += 1
        assert np.array_equal(seg_idx[i, :ns], r["seg_idx"]), i
        inside = r["seg_idx"] >= 0  # (the row buffer of the hot path keeps no length for a segment outside the grid)
        assert np.array_equal(seg_len[i, :ns][inside], r["seg_len"][inside]), i
        heads = row_len[i, :ns] > 0
        assert np.array_equal(seg_idx[i, :ns][heads], r["row_idx"]), i
        assert row_len[i, :ns][heads] == pytest.approx(r["row_len"], rel=1e-6)
    assert paths > n // 2
