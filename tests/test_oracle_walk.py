"""Pins for the oracle's hull -> MLP -> voxel walk (fp32 rule mirror T32 vs fp64 definition T64,
SURVEY.md Appendix A worked example, geometric invariants).  CPU only."""
import json
import os

import numpy as np
import pytest

import synth

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "survey_appendix_a.json")))["full_rule"]


def _gold_case(oracle_mod, key):
    g = GOLD
    geom = oracle_mod.Geometry(*g["grid"], g["h"], g["u_in"], g["u_out"])
    hh = g["history"]
    hist = oracle_mod.binding._Hist(hh["t_in"], hh["v_in"], hh["t_out"], hh["v_out"], hh["tht_in"], hh["thv_in"],
                                    hh["tht_out"], hh["thv_out"], g[key]["cs"], g[key]["sn"])
    return geom, hist, g[key]


def test_p12_worked_example_phi0(oracle_mod):
    geom, hist, ref = _gold_case(oracle_mod, "phi0")
    nodes, hull = oracle_mod.path_f64(geom, hist)
    for name, val in zip(("u0", "t0", "v0", "u2", "t2", "v2", "L"), hull):
        assert val == pytest.approx(ref[name], abs=2e-7)  # the history is fp32-quantised (0.010 -> float)
    assert nodes.shape[0] == ref["K"] + 2
    # cs=1, sn=0: object frame (x,y,z) == beam frame (t,u,v)
    for k, tuv in ref["nodes_tuv"].items():
        assert nodes[int(k)] == pytest.approx(tuv, abs=2e-7)
    poly = np.linalg.norm(np.diff(nodes, axis=0), axis=1).sum()
    assert poly == pytest.approx(ref["polyline"], abs=2e-7)
    r = oracle_mod.row_f32(geom, hist)
    assert r["nnz"] == ref["nnz"] and r["nseg"] == ref["K"] + 1
    assert list(r["row_idx"][:3]) == ref["first_idx"] and r["row_idx"][-1] == ref["last_idx"]
    assert r["row_len"][0] == pytest.approx(ref["first_len"], abs=2e-7)
    assert np.abs(r["nodes"].astype(np.float64) - nodes).max() < 2e-5  # "T32 to ~1e-5 in position"
    assert float(r["row_len"].astype(np.float64).sum()) == pytest.approx(ref["polyline"], abs=2e-5)


def test_p12_worked_example_phi45(oracle_mod):
    geom, hist, ref = _gold_case(oracle_mod, "phi45")
    nodes, _ = oracle_mod.path_f64(geom, hist)
    assert np.linalg.norm(np.diff(nodes, axis=0), axis=1).sum() == pytest.approx(ref["polyline"], abs=2e-7)
    r = oracle_mod.row_f32(geom, hist)
    assert r["nnz"] == ref["nnz"]
    assert list(r["row_idx"][:6]) == ref["first_idx"]


@pytest.fixture(scope="module")
def cfg0_sample(oracle_mod):
    cfg = synth.config(0)
    H = synth.generate_numpy(cfg, 3000)
    geom = oracle_mod.Geometry(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out)
    return cfg, geom, oracle_mod.Histories(H)


def test_t32_nodes_within_1e4_mm_of_definition(oracle_mod, cfg0_sample):
    """north_star: MLP positions within 1e-4 mm.  Here: fp32 rule vs fp64 matrix form, and the
    voxel index may differ only where the fp64 midpoint is within 1e-3 mm of a voxel face."""
    cfg, geom, hs = cfg0_sample
    table = oracle_mod.sigma1_table(geom.h, geom.nmin)
    worst, face_flips, nseg_total, skipped = 0.0, 0, 0, 0
    for i in range(0, hs.n, 3):
        h = hs.hist(i)
        r = oracle_mod.row_f32(geom, h, table)
        nodes, _ = oracle_mod.path_f64(geom, h)
        if nodes is None:
            assert r["nseg"] == 0
            skipped += 1
            continue
        if nodes.shape[0] != r["nseg"] + 1:
            continue  # L - eps within rounding of a multiple of h (counted as a non-event)
        worst = max(worst, np.abs(r["nodes"].astype(np.float64) - nodes).max())
        mid = 0.5 * (nodes[1:] + nodes[:-1]) / geom.h + 0.5 * np.array([geom.nx, geom.ny, geom.nz])
        ijk = np.floor(mid).astype(np.int64)
        ok = np.all((ijk >= 0) & (ijk < [geom.nx, geom.ny, geom.nz]), axis=1)
        lin = np.where(ok, ijk[:, 0] + geom.nx * (ijk[:, 1] + geom.ny * ijk[:, 2]), -1)
        diff = lin != r["seg_idx"]
        nseg_total += lin.size
        if diff.any():
            dist = np.abs(mid - np.round(mid)).min(axis=1)
            assert (dist[diff] < 1e-3).all()
            face_flips += int(diff.sum())
    assert worst < 1e-4
    assert nseg_total > 20000 and face_flips < 1e-3 * nseg_total
    assert 0 < skipped < hs.n // 3  # some histories miss the hull, most do not


def test_p2_p3_p4_row_invariants(oracle_mod, cfg0_sample):
    cfg, geom, hs = cfg0_sample
    table = oracle_mod.sigma1_table(geom.h, geom.nmin)
    R = 0.5 * geom.h * geom.nmin
    n_rows = 0
    for i in range(0, hs.n, 5):
        h = hs.hist(i)
        r = oracle_mod.row_f32(geom, h, table)
        if r["nseg"] == 0:
            continue
        n_rows += 1
        nd = r["nodes"].astype(np.float64)
        # P3: first and last node are the hull points: on the hull cylinder, inside the z range
        for p in (nd[0], nd[-1]):
            assert np.hypot(p[0], p[1]) == pytest.approx(R, abs=2e-4)
            assert abs(p[2]) <= 0.5 * geom.nz * geom.h + 1e-6
        # P4: chord lengths sum to the polyline length recomputed from the node list ...
        seg = np.linalg.norm(np.diff(nd, axis=0), axis=1)
        assert r["seg_len"].astype(np.float64) == pytest.approx(seg, abs=1e-6)
        if (r["seg_idx"] >= 0).all():
            assert float(r["row_len"].astype(np.float64).sum()) == pytest.approx(seg.sum(), abs=2e-5)
        # ... which is at least the straight distance between the hull points
        assert seg.sum() >= np.linalg.norm(nd[-1] - nd[0]) - 1e-5
        # merged row: no two consecutive equal indices, all in range, lengths positive
        assert (np.diff(r["row_idx"]) != 0).all()
        assert (r["row_idx"] >= 0).all() and (r["row_idx"] < geom.n_voxels).all()
        assert (r["row_len"] > 0).all()
        assert r["nnz"] == int(np.count_nonzero(np.diff(np.concatenate([[-2], r["seg_idx"]]))[r["seg_idx"] >= 0]))
    assert n_rows > 300


def test_p2_collinear_history_walks_the_chord(oracle_mod):
    geom = oracle_mod.Geometry(64, 64, 8, 1.0, -48.0, 48.0)
    th, ph = 0.013, -0.004
    t_in, v_in = 5.0, 1.0
    hist = oracle_mod.binding._Hist(t_in, v_in, t_in + th * 96.0, v_in + ph * 96.0, th, ph, th, ph, 0.8, 0.6)
    r = oracle_mod.row_f32(geom, hist)
    nd = r["nodes"].astype(np.float64)
    chord = nd[-1] - nd[0]
    # every node on the straight line between the hull points; length sum == straight distance
    for p in nd:
        w = p - nd[0]
        assert np.linalg.norm(np.cross(w, chord)) / np.linalg.norm(chord) < 2e-5
    assert float(r["seg_len"].astype(np.float64).sum()) == pytest.approx(np.linalg.norm(chord), abs=3e-5)
    n64, _ = oracle_mod.path_f64(geom, hist)
    w = n64 - n64[0]
    # (the fp32-quantised exit point is collinear only to ~1e-7 mm)
    assert np.abs(np.cross(w, n64[-1] - n64[0])).max() / np.linalg.norm(n64[-1] - n64[0]) < 1e-6


def test_skip_rules(oracle_mod):
    geom = oracle_mod.Geometry(64, 64, 8, 1.0, -48.0, 48.0)
    mk = oracle_mod.binding._Hist
    assert oracle_mod.row_f32(geom, mk(40.0, 0, 40.0, 0, 0, 0, 0, 0, 1, 0))["nseg"] == 0  # misses the hull
    assert oracle_mod.row_f32(geom, mk(0.0, 4.5, 0.0, 0, 0, 0, 0, 0, 1, 0))["nseg"] == 0  # enters above the grid
    assert oracle_mod.row_f32(geom, mk(0.0, 0, 0.0, -4.5, 0, 0, 0, 0, 1, 0))["nseg"] == 0  # leaves below
    assert oracle_mod.row_f32(geom, mk(float("nan"), 0, 0.0, 0, 0, 0, 0, 0, 1, 0))["nseg"] == 0
    assert oracle_mod.path_f64(geom, mk(40.0, 0, 40.0, 0, 0, 0, 0, 0, 1, 0))[0] is None
    r = oracle_mod.row_f32(geom, mk(0.0, 0, 0.0, 0, 0, 0, 0, 0, 1, 0))  # central ray: 64 unit segments
    assert r["nseg"] == 64 and r["nnz"] == 64
    assert r["row_len"] == pytest.approx(np.ones(64), abs=1e-6)
    assert list(r["row_idx"]) == [32 + 64 * (j + 64 * 4) for j in range(64)]


def test_p11_sparsity_a_few_hundred_of_millions(oracle_mod):
    """'a few hundred out of about one or two million voxels' per proton."""
    cfg = synth.config(3)
    geom = oracle_mod.Geometry(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out)
    rng = np.random.default_rng(3)
    table = oracle_mod.sigma1_table(geom.h, geom.nmin)
    nnz = []
    for _ in range(150):
        t = rng.uniform(-128, 128)
        v = rng.uniform(-60, 60)
        ph = rng.integers(0, 360) * 2 * np.pi / 360
        h = oracle_mod.binding._Hist(t, v, t + rng.normal(0, 1.5), v + rng.normal(0, 1.5), rng.normal(0, 2e-3),
                                     rng.normal(0, 2e-3), rng.normal(0, 1e-2), rng.normal(0, 1e-2),
                                     np.float32(np.cos(ph)), np.float32(np.sin(ph)))
        r = oracle_mod.row_f32(geom, h, table)
        if r["nseg"]:
            nnz.append(r["nnz"])
    assert 150 < np.mean(nnz) < 260 and max(nnz) <= 256 + 1
