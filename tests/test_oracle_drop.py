"""Pins for the oracle's DROP loop (R12-R18; Fig. 1).  CPU only.

The rows come from the oracle's own T32 walk (pinned in test_oracle_walk.py); here the block
update is pinned by a dense numpy re-statement, the Kaczmarz identity, hit-count identities, the
block structure the paper states, and convergence to a dense least-squares solve."""
import numpy as np
import pytest

import synth


def _tiny_problem(oracle_mod, n=3000, n_angles=12, seed=11, grid=(6, 6, 4)):
    """Histories through a 6x6x4 grid of 1 mm voxels: straight-ish tracks with small kinks."""
    nx, ny, nz = grid
    geom = oracle_mod.Geometry(nx, ny, nz, 1.0, -6.0, 6.0)
    rng = np.random.default_rng(seed)
    proj = (np.arange(n) % n_angles).astype(np.uint16)
    phi = 2 * np.pi * np.arange(n_angles) / n_angles
    t_in = rng.uniform(-3, 3, n)
    v_in = rng.uniform(-1.9, 1.9, n)
    tht_in = rng.normal(0, 0.02, n)
    thv_in = rng.normal(0, 0.02, n)
    tht_out = tht_in + rng.normal(0, 0.03, n)
    thv_out = thv_in + rng.normal(0, 0.03, n)
    t_out = t_in + 12 * 0.5 * (tht_in + tht_out) + rng.normal(0, 0.05, n)
    v_out = v_in + 12 * 0.5 * (thv_in + thv_out) + rng.normal(0, 0.02, n)
    H = dict(t_in=t_in, v_in=v_in, t_out=t_out, v_out=v_out, tht_in=tht_in, thv_in=thv_in, tht_out=tht_out,
             thv_out=thv_out, wepl=np.zeros(n), proj=proj, proj_cos=np.cos(phi), proj_sin=np.sin(phi))
    return geom, H


def _dense_rows(oracle_mod, geom, hs):
    A = np.zeros((hs.n, geom.n_voxels))
    table = oracle_mod.sigma1_table(geom.h, geom.nmin)
    for i in range(hs.n):
        r = oracle_mod.row_f32(geom, hs.hist(i), table)
        # merged row, lengths merged in double from the raw segments
        last = -1
        for idx, ln in zip(r["seg_idx"], r["seg_len"]):
            if idx >= 0:
                A[i, idx] += float(ln)
                assert not (idx != last and A[i, idx] != float(ln)), "non-consecutive repeat"
            last = idx
    return A


@pytest.fixture(scope="module")
def tiny(oracle_mod):
    geom, H = _tiny_problem(oracle_mod)
    hs = oracle_mod.Histories(H)
    A = _dense_rows(oracle_mod, geom, hs)
    rng = np.random.default_rng(5)
    x_true = rng.uniform(0.5, 1.5, geom.n_voxels)
    H["wepl"] = (A @ x_true).astype(np.float32)
    hs = oracle_mod.Histories(H)
    return geom, H, hs, A, x_true


def test_block_update_equals_dense_formula(oracle_mod, tiny):
    """x <- x + lam * U * sum_i ((b_i - a_i.x)/||a_i||^2) a_i,  U = diag(1/max(1,c_j)) -- dense numpy."""
    geom, H, hs, A, _ = tiny
    rng = np.random.default_rng(0)
    x0 = rng.uniform(0, 1, geom.n_voxels)
    first, count, lam = 100, 250, 0.7
    Ab = A[first:first + count]
    b = hs.a["wepl"][first:first + count].astype(np.float64)
    nz = (Ab != 0).any(axis=1)
    r = np.zeros(count)
    r[nz] = (b[nz] - Ab[nz] @ x0) / (Ab[nz] ** 2).sum(axis=1)
    delta_ref = Ab.T @ r
    c_ref = (Ab != 0).sum(axis=0)
    delta, cnt, stats = oracle_mod.block_accumulate(geom, hs, first, count, x0)
    assert cnt.tolist() == c_ref.tolist()
    assert delta == pytest.approx(delta_ref, abs=1e-12)
    assert stats[0] == int(nz.sum()) and stats[1] == int((Ab != 0).sum())
    # one-block sweep through the public loop
    Hb = {k: (v[first:first + count] if k in synth.FIELDS or k == "proj" else v) for k, v in H.items()}
    x1, _ = oracle_mod.drop_iterate(geom, oracle_mod.Histories(Hb), lam, count, 1, x0.copy())
    assert x1 == pytest.approx(x0 + lam * delta_ref / np.maximum(1, c_ref), abs=1e-12)


def test_p8_single_row_is_kaczmarz(oracle_mod, tiny):
    """B = 1, lam = 1: right after row i the row equation holds exactly, a_i.x = b_i."""
    geom, H, hs, A, _ = tiny
    x = np.zeros(geom.n_voxels)
    for i in range(40):
        Hi = {k: (v[i:i + 1] if k in synth.FIELDS or k == "proj" else v) for k, v in H.items()}
        x, _ = oracle_mod.drop_iterate(geom, oracle_mod.Histories(Hi), 1.0, 1, 1, x)
        if A[i].any():
            assert A[i] @ x == pytest.approx(float(hs.a["wepl"][i]), abs=1e-10)


def test_p9_hit_counts_and_linearity(oracle_mod, tiny):
    geom, H, hs, A, _ = tiny
    x0 = np.zeros(geom.n_voxels)
    delta, cnt, stats = oracle_mod.block_accumulate(geom, hs, 0, 500, x0)
    assert cnt.sum() == stats[1] == int((A[:500] != 0).sum())
    assert cnt.max() <= 500
    assert stats[2] >= stats[1]  # raw segments >= merged non-zeros
    xa, _ = oracle_mod.drop_iterate(geom, hs, 0.2, hs.n, 1, x0.copy())
    xb, _ = oracle_mod.drop_iterate(geom, hs, 0.4, hs.n, 1, x0.copy())
    assert xb == pytest.approx(2 * xa, abs=1e-13)  # first block from x0 = 0 is linear in lambda


def test_p10_block_structure(oracle_mod, tiny):
    """x1 from block 0, then block 1 starts from x1; a new iteration starts from the
    last solution.  One call with B = N/2 == two calls on the halves with the image carried over,
    and 2 iterations in one call == two 1-iteration calls."""
    geom, H, hs, _, _ = tiny
    half = hs.n // 2
    x_one, _ = oracle_mod.drop_iterate(geom, hs, 0.5, half, 1, np.zeros(geom.n_voxels))
    parts = [{k: (v[s] if k in synth.FIELDS or k == "proj" else v) for k, v in H.items()}
             for s in (slice(0, half), slice(half, None))]
    x_two = np.zeros(geom.n_voxels)
    for p in parts:
        x_two, _ = oracle_mod.drop_iterate(geom, oracle_mod.Histories(p), 0.5, half, 1, x_two)
    assert x_one == pytest.approx(x_two, abs=1e-14)
    # order matters (block-sequential, not simultaneous): reversed halves give another iterate
    x_rev = np.zeros(geom.n_voxels)
    for p in parts[::-1]:
        x_rev, _ = oracle_mod.drop_iterate(geom, oracle_mod.Histories(p), 0.5, half, 1, x_rev)
    assert np.abs(x_rev - x_one).max() > 1e-6
    xa, _ = oracle_mod.drop_iterate(geom, hs, 0.5, 700, 2, np.zeros(geom.n_voxels))
    xb, _ = oracle_mod.drop_iterate(geom, hs, 0.5, 700, 1, np.zeros(geom.n_voxels))
    xb, _ = oracle_mod.drop_iterate(geom, hs, 0.5, 700, 1, xb)
    assert xa == pytest.approx(xb, abs=1e-14)
    # ragged last block (3000 = 4*700 + 200) is processed: every history is used once per sweep
    _, st = oracle_mod.drop_iterate(geom, hs, 0.5, 700, 1, np.zeros(geom.n_voxels))
    _, st_all = oracle_mod.drop_iterate(geom, hs, 0.5, hs.n, 1, np.zeros(geom.n_voxels))
    assert st == st_all


def test_p7_converges_to_dense_least_squares(oracle_mod, tiny):
    """Noise-free consistent data on a 6x6x4 grid: the DROP iterate converges to the dense
    least-squares solution on the hit columns (brute force: numpy lstsq on the dense A)."""
    geom, H, hs, A, x_true = tiny
    hit = (A != 0).any(axis=0)
    b = hs.a["wepl"].astype(np.float64)
    x_ls, *_ = np.linalg.lstsq(A[:, hit], b, rcond=None)
    assert np.linalg.matrix_rank(A[:, hit]) == hit.sum()  # unique solution on the hit columns
    x, _ = oracle_mod.drop_iterate(geom, hs, 1.9, 50, 600, np.zeros(geom.n_voxels))
    err = np.abs(x[hit] - x_ls)
    col = np.linalg.norm(A[:, hit], axis=0)
    # Columns of the corner slivers of the inscribed hull are hit once with a ~0.01 mm chord
    # (sigma_min/sigma_max ~ 5e-4): they converge last.  Everything else is there after 600 sweeps.
    assert (col > 1.0).sum() >= 120 and err[col > 1.0].max() < 5e-4
    assert err[col > 0.1].max() < 5e-3
    assert np.abs(x[hit] - x_true[hit])[col > 1.0].max() < 1e-3  # fp32 WEPL quantisation ~1e-7 relative
    assert (x[~hit] == 0).all()  # voxels never hit keep x0 (R16)
    # the row equations hold (x is the unique LS solution of consistent data), except in the rows
    # that touch a sliver column (chord ~0.01 mm, hit once), which are still converging
    res = np.abs(A @ x - b)
    sliver_rows = (A[:, hit][:, col <= 0.1] != 0).any(axis=1)
    assert sliver_rows.sum() <= 3 and res[~sliver_rows].max() < 1e-3 and res.max() < 2e-2
    # in the singular basis the error lives only in the weakly determined directions
    _, S, Vt = np.linalg.svd(A[:, hit], full_matrices=False)
    e = Vt @ (x[hit] - x_ls)
    assert np.abs(e[S > 0.02 * S[0]]).max() < 5e-4
    # and the error keeps shrinking monotonically sweep after sweep
    x2, _ = oracle_mod.drop_iterate(geom, hs, 1.9, 50, 200, x.copy())
    assert np.linalg.norm(x2[hit] - x_ls) < np.linalg.norm(x[hit] - x_ls)


def test_r24_projection_index_past_the_tables_means_the_last_angle(oracle_mod):
    """DESIGN.md R24 (the library's pct_set_histories promises it): proj[i] >= n_proj is read as n_proj - 1, never out of
    bounds.  Pinned by substitution: histories whose index was pushed past the tables give, row by row and in a DROP
    block, exactly what the same histories with the index written as n_proj - 1 give -- and NOT what angle 0 gives."""
    geom, H = _tiny_problem(oracle_mod, n=600)
    n_proj = H["proj_cos"].shape[0]
    H["wepl"] = np.full(600, 5.0, dtype=np.float32)
    bad = dict(H)
    bad["proj"] = H["proj"].copy()
    sel = np.arange(0, 600, 3)
    bad["proj"][sel] = np.array([n_proj, n_proj + 5, 65535], dtype=np.uint16)[np.arange(sel.size) % 3]
    want = dict(H)
    want["proj"] = H["proj"].copy()
    want["proj"][sel] = n_proj - 1
    wrong = dict(H)
    wrong["proj"] = H["proj"].copy()
    wrong["proj"][sel] = 0
    hb, hw, h0 = oracle_mod.Histories(bad), oracle_mod.Histories(want), oracle_mod.Histories(wrong)
    differs = 0
    for i in sel:
        rb, rw, r0 = (oracle_mod.row_f32(geom, h.hist(int(i))) for h in (hb, hw, h0))
        assert rb["nseg"] == rw["nseg"] and np.array_equal(rb["seg_idx"], rw["seg_idx"]) and np.array_equal(rb["seg_len"], rw["seg_len"])
        differs += rb["nseg"] != r0["nseg"] or not np.array_equal(rb["seg_idx"], r0["seg_idx"])
    assert differs > sel.size // 2  # the pin can tell the last angle from the first
    x0 = np.linspace(0.5, 1.5, geom.n_voxels)
    db, cb, _ = oracle_mod.block_accumulate(geom, hb, 0, 600, x0)   # the C loader (load_hist)
    dw, cw, _ = oracle_mod.block_accumulate(geom, hw, 0, 600, x0)
    d0, c0, _ = oracle_mod.block_accumulate(geom, h0, 0, 600, x0)
    assert np.array_equal(db, dw) and np.array_equal(cb, cw)
    assert not np.array_equal(cb, c0)
