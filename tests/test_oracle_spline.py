"""Pins for the oracle's cubic-spline path model (R30).  CPU only.

The spline through the hull entry and exit points with the measured directions is what the most-likely path
becomes for a constant scattering power (pin P1 in test_oracle_mlp.py); here the model itself is pinned: the
fp64 nodes against scipy's CubicHermiteSpline, the fp32 rule against the fp64 nodes, the row invariants, and
that the default model is untouched."""
import numpy as np
import pytest
from scipy.interpolate import CubicHermiteSpline

import synth


@pytest.fixture()
def spline(oracle_mod):
    oracle_mod.set_path_model(1)
    yield oracle_mod
    oracle_mod.set_path_model(0)


@pytest.fixture(scope="module")
def sample(oracle_mod):
    cfg = synth.config(0)
    H = synth.generate_numpy(cfg, 3000)
    geom = oracle_mod.Geometry(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out)
    return cfg, geom, H


def test_fp64_nodes_are_the_cubic_hermite_spline(spline, sample):
    """Projection angle 0 (object frame = beam frame): node k = the Hermite spline through (u0, t0, theta0) and
    (u2, t2, theta2) evaluated at u0 + k h, in both planes; the end nodes are the hull points."""
    cfg, geom, H = sample
    H0 = dict(H, proj=np.zeros_like(H["proj"]), proj_cos=np.ones(1, np.float32), proj_sin=np.zeros(1, np.float32))
    hs = spline.Histories(H0)
    checked = 0
    for i in range(0, 300):
        h = hs.hist(i)
        nodes, hull = spline.path_f64(geom, h)
        if nodes is None:
            continue
        u0, t0, v0, u2, t2, v2, L = hull
        K = nodes.shape[0] - 2
        u = np.concatenate([u0 + geom.h * np.arange(K + 1), [u2]])
        st = CubicHermiteSpline([u0, u2], [t0, t2], [float(H0["tht_in"][i]), float(H0["tht_out"][i])])
        sv = CubicHermiteSpline([u0, u2], [v0, v2], [float(H0["thv_in"][i]), float(H0["thv_out"][i])])
        assert nodes[:, 0] == pytest.approx(st(u), abs=1e-11)
        assert nodes[:, 1] == pytest.approx(u, abs=1e-11)
        assert nodes[:, 2] == pytest.approx(sv(u), abs=1e-11)
        checked += 1
    assert checked > 200


def test_fp32_rule_within_1e4_mm_and_rows_add_up(spline, sample):
    cfg, geom, H = sample
    hs = spline.Histories(H)
    table = spline.sigma1_table(geom.h, geom.nmin)
    worst, rows = 0.0, 0
    for i in range(0, hs.n, 5):
        h = hs.hist(i)
        r = spline.row_f32(geom, h, table)
        nodes, _ = spline.path_f64(geom, h)
        if nodes is None:
            assert r["nseg"] == 0
            continue
        if nodes.shape[0] != r["nseg"] + 1:
            continue
        worst = max(worst, np.abs(r["nodes"].astype(np.float64) - nodes).max())
        seg = np.linalg.norm(np.diff(r["nodes"].astype(np.float64), axis=0), axis=1)
        inside = r["seg_idx"] >= 0
        assert float(r["row_len"].sum()) == pytest.approx(seg[inside].sum(), rel=1e-6)  # chord lengths sum to the in-grid path length
        rows += 1
    assert worst < 1e-4 and rows > 400


def test_spline_is_close_to_the_mlp_and_the_default_is_untouched(oracle_mod, sample):
    cfg, geom, H = sample
    hs = oracle_mod.Histories(H)
    assert oracle_mod.get_path_model() == 0
    a = [oracle_mod.path_f64(geom, hs.hist(i))[0] for i in range(200)]
    oracle_mod.set_path_model(1)
    try:
        b = [oracle_mod.path_f64(geom, hs.hist(i))[0] for i in range(200)]
    finally:
        oracle_mod.set_path_model(0)
    c = [oracle_mod.path_f64(geom, hs.hist(i))[0] for i in range(200)]
    d = max(np.abs(x - y).max() for x, y in zip(a, b) if x is not None)
    assert 1e-6 < d < 0.05  # different models, a few hundredths of a millimetre apart at 64 mm depth
    assert all((x is None and z is None) or np.array_equal(x, z) for x, z in zip(a, c))
