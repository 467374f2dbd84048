"""Pins of the oracle's half-voxel depth step (orc_set_substeps(2), R33).  CPU only.

The path is the same curve sampled twice as densely, so: every node of the full-step path is node 2k of the half-step
path (fp64 definition), the polyline can only get longer and by very little, the row still adds up to the polyline,
the fp32 rule stays within 1e-4 mm of the definition, and about half of the half-step segments fall into a voxel the
full-step row also has."""
import numpy as np
import pytest

import synth
from helpers import oracle_geom


@pytest.fixture()
def half(oracle_mod):
    yield oracle_mod
    oracle_mod.set_substeps(1)


def test_half_step_path_is_the_same_curve_sampled_twice_as_densely(half):
    o = half
    cfg = synth.config(1)
    H = synth.generate_numpy(cfg, 300)
    geom = oracle_geom(o, cfg)
    hs = o.Histories(H)
    checked = 0
    for i in range(300):
        o.set_substeps(1)
        n1, hull1 = o.path_f64(geom, hs.hist(i))
        r1 = o.row_f32(geom, hs.hist(i))
        o.set_substeps(2)
        n2, hull2 = o.path_f64(geom, hs.hist(i))
        r2 = o.row_f32(geom, hs.hist(i))
        if n1 is None:
            assert n2 is None and r2["nseg"] == 0
            continue
        checked += 1
        K1, K2 = n1.shape[0] - 2, n2.shape[0] - 2
        assert K2 in (2 * K1, 2 * K1 + 1)  # floor((L - eps) / (h/2))
        assert np.array_equal(hull1, hull2)
        # node k of the full-step path = node 2k of the half-step path; first and last are the hull points
        assert np.abs(n2[0:2 * K1 + 1:2] - n1[:K1 + 1]).max() < 1e-9
        assert np.array_equal(n2[-1], n1[-1])
        len1 = np.linalg.norm(np.diff(n1, axis=0), axis=1).sum()
        len2 = np.linalg.norm(np.diff(n2, axis=0), axis=1).sum()
        assert len1 - 1e-9 <= len2 <= len1 * (1 + 1e-4)
        # the fp32 rule in this mode: nodes within 1e-4 mm of the definition, row sums to its polyline
        assert r2["nseg"] == K2 + 1
        assert np.abs(r2["nodes"].astype(np.float64) - n2).max() < 1e-4
        inside = r2["seg_idx"] >= 0
        assert r2["row_len"].astype(np.float64).sum() == pytest.approx(r2["seg_len"][inside].astype(np.float64).sum(), rel=1e-6)
        # a finer walk finds at least as many voxels (corner cuts) and mostly the same ones
        s1, s2 = set(r1["row_idx"].tolist()), set(r2["row_idx"].tolist())
        assert len(s2) >= len(s1) and len(s1 & s2) >= 0.8 * len(s1)
    assert checked > 200


def test_half_step_table_and_block(half):
    """The Sigma1^-1 table of the mode is the full-step table of a grid with voxels half the size, and a DROP block
    in this mode still satisfies the block identities (hit counts sum to the non-zeros)."""
    o = half
    cfg = synth.config(0)
    geom = oracle_geom(o, cfg)
    t_half = o.sigma1_table(0.5 * geom.h, 2 * geom.nmin)
    t_full = o.sigma1_table(geom.h, geom.nmin)
    for a, b in zip(t_half, t_full):
        assert np.array_equal(a[2::2], b[1:])  # s = 2k * h/2 = k * h: the same depth, the same entry
    H = synth.generate_numpy(cfg, 2000)
    hs = o.Histories(H)
    o.set_substeps(2)
    d, c, st = o.block_accumulate(geom, hs, 0, 2000, synth.rsp_volume(cfg) * 0.9)
    assert c.sum() == st[1] and st[2] > 1.9 * 2000 * 0.9 * 40  # about twice the segments of the full step
    o.set_substeps(1)
    d1, c1, st1 = o.block_accumulate(geom, hs, 0, 2000, synth.rsp_volume(cfg) * 0.9)
    assert 1.9 * st1[2] < st[2] < 2.1 * st1[2] and st[1] >= st1[1]
    # the two walks see the same image: the accumulated corrections point the same way
    assert np.dot(d, d1) > 0.9 * np.linalg.norm(d) * np.linalg.norm(d1)
