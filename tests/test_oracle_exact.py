"""Pins of the oracle's exact voxel traversal (orc_set_walk_mode(1), R34).  CPU only.

The row must be the list of the polyline's chord lengths per voxel.  Pinned against a brute-force restatement typed
here (every polyline segment sampled at 4000 points, each sample's length credited to the voxel it falls in), by the
exact sum (pieces add up to the polyline), by adjacency (no voxel is skipped at a corner cut: consecutive voxels of a row
share a face), and by an axis-aligned ray whose chords are known by hand."""
import numpy as np
import pytest

import synth
from helpers import oracle_geom


@pytest.fixture()
def exact(oracle_mod):
    oracle_mod.set_walk_mode(1)
    yield oracle_mod
    oracle_mod.set_walk_mode(0)


def _brute_force_chords(cfg, nodes, samples=4000):
    """Chord length per voxel of the polyline through `nodes` (float64 object-frame mm), by dense sampling."""
    out = {}
    half = np.array([cfg.nx, cfg.ny, cfg.nz]) * 0.5
    dims = np.array([cfg.nx, cfg.ny, cfg.nz])
    t = (np.arange(samples) + 0.5) / samples
    for a, b in zip(nodes[:-1], nodes[1:]):
        seg = np.linalg.norm(b - a)
        pts = a[None, :] + t[:, None] * (b - a)[None, :]
        ijk = np.floor(pts / cfg.h + half).astype(np.int64)
        ok = np.all((ijk >= 0) & (ijk < dims), axis=1)
        lin = ijk[:, 0] + cfg.nx * (ijk[:, 1] + cfg.ny * ijk[:, 2])
        for v, c in zip(*np.unique(lin[ok], return_counts=True)):
            out[int(v)] = out.get(int(v), 0.0) + seg * c / samples
    return out


def test_rows_are_the_chord_lengths_of_the_polyline(exact):
    o = exact
    cfg = synth.config(0)
    H = synth.generate_numpy(cfg, 400)
    geom = oracle_geom(o, cfg)
    hs = o.Histories(H)
    checked = 0
    for i in range(0, 400, 3):
        r = o.row_f32(geom, hs.hist(i))
        if r["nseg"] == 0:
            continue
        checked += 1
        nodes = r["nodes"].astype(np.float64)
        poly = np.linalg.norm(np.diff(nodes, axis=0), axis=1).sum()
        # (1) the pieces add up to the polyline (inside the grid: these phantoms keep the path inside in z)
        assert r["seg_len"].astype(np.float64).sum() == pytest.approx(poly, rel=2e-6)
        inside = r["seg_idx"] >= 0
        assert r["row_len"].astype(np.float64).sum() == pytest.approx(r["seg_len"][inside].astype(np.float64).sum(), rel=1e-6)
        # (2) per voxel, the brute-force chord
        ref = _brute_force_chords(cfg, nodes)
        got = {}
        for v, l in zip(r["row_idx"], r["row_len"]):
            got[int(v)] = got.get(int(v), 0.0) + float(l)
        assert set(got) >= {v for v, l in ref.items() if l > 2e-3}  # nothing longer than a sampling step is missed
        for v, l in got.items():
            assert l == pytest.approx(ref.get(v, 0.0), abs=3e-3), (i, v)
        # (3) no voxel skipped: consecutive voxels of the row share a face (one index differs by one)
        idx = r["row_idx"]
        ii, jj, kk = idx % cfg.nx, (idx // cfg.nx) % cfg.ny, idx // (cfg.nx * cfg.ny)
        step = np.abs(np.diff(ii)) + np.abs(np.diff(jj)) + np.abs(np.diff(kk))
        if inside.all():
            # (an exact passage through an edge or a corner may change two indices at once: at most a handful)
            assert (step >= 1).all() and (step <= 3).all() and (step == 1).mean() > 0.97
        # (4) more voxels than the midpoint rule finds, never fewer
    assert checked > 100


def test_midpoint_rule_finds_a_subset_of_the_voxels(exact):
    o = exact
    cfg = synth.config(1)
    H = synth.generate_numpy(cfg, 200)
    geom = oracle_geom(o, cfg)
    hs = o.Histories(H)
    more = 0
    for i in range(200):
        o.set_walk_mode(1)
        e = o.row_f32(geom, hs.hist(i))
        o.set_walk_mode(0)
        m = o.row_f32(geom, hs.hist(i))
        if m["nseg"] == 0:
            assert e["nseg"] == 0
            continue
        assert np.array_equal(e["nodes"], m["nodes"])  # the same polyline
        # the midpoint of a segment lies on the polyline: its voxel is one the exact traversal visits
        assert set(m["row_idx"].tolist()) <= set(e["row_idx"].tolist())
        assert e["row_len"].astype(np.float64).sum() == pytest.approx(m["row_len"].astype(np.float64).sum(), rel=1e-5)
        more += len(e["row_idx"]) > len(m["row_idx"])
    assert more > 100


def test_axis_aligned_ray_by_hand(exact):
    """phi = 0, a straight ray along +y at t = 0.3, v = 0.2 through the 64 x 64 x 8 grid of 1 mm voxels: the hull chord
    runs from y = -sqrt(32^2 - 0.09) to +sqrt(...); every voxel of column i = 32, slice k = 4 in between gets 1 mm, the two
    end voxels the remainder."""
    o = exact
    cfg = synth.config(0)
    geom = oracle_geom(o, cfg)
    cs, sn = np.array([1.0], np.float32), np.array([0.0], np.float32)
    H = dict(t_in=[0.3], v_in=[0.2], t_out=[0.3], v_out=[0.2], tht_in=[0.0], thv_in=[0.0], tht_out=[0.0], thv_out=[0.0],
             wepl=[1.0], proj=np.array([0], np.uint16), proj_cos=cs, proj_sin=sn)
    H = {k: (np.asarray(v, np.float32) if k not in ("proj",) else v) for k, v in H.items()}
    r = o.row_f32(geom, o.Histories(H).hist(0))
    half = np.sqrt(32.0 ** 2 - 0.3 ** 2)
    assert r["row_len"].astype(np.float64).sum() == pytest.approx(2 * half, abs=1e-4)
    idx = r["row_idx"]
    assert np.all(idx % 64 == 32) and np.all(idx // (64 * 64) == 4)
    jj = (idx // 64) % 64
    assert np.array_equal(jj, np.arange(jj[0], jj[0] + len(jj)))  # every voxel of the column once, in order
    assert len(jj) == 64 and jj[0] == 0
    assert r["row_len"][1:-1] == pytest.approx(1.0, abs=2e-5)
    assert r["row_len"][0] == pytest.approx(half - 31.0, abs=1e-4) and r["row_len"][-1] == pytest.approx(half - 31.0, abs=1e-4)


def test_drop_block_identities_hold_in_the_exact_mode(exact):
    o = exact
    cfg = synth.config(0)
    H = synth.generate_numpy(cfg, 1500)
    geom = oracle_geom(o, cfg)
    hs = o.Histories(H)
    d, c, st = o.block_accumulate(geom, hs, 0, 1500, synth.rsp_volume(cfg) * 0.9)
    assert c.sum() == st[1] and st[1] > 1.2 * 1500 * 0.9 * 40  # about 1.3 voxels per mm of path
    x, _ = o.drop_iterate(geom, hs, 1.0, 1, 1, np.zeros(cfg.n_voxels), n=40)  # Kaczmarz: after row i, a_i.x = b_i
    assert np.isfinite(x).all() and np.abs(x).max() > 0
