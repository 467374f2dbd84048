"""Pins for the oracle's CARP loop (section 2.2 and Fig. 2; R27-R29).  CPU only.

"we proceed to get a new estimate x_n for each data subset n using the same initial guess x_0.  A new
solution is then computed from the average of the different string solutions."  The string estimate is the
DROP sweep pinned in test_oracle_drop.py; pinned here: the one-string case, the averaging (divisor, common
start), a dense numpy re-statement with one row per string (averaged Kaczmarz projections), the string
boundaries, and convergence on noise-free data."""
import numpy as np
import pytest

from test_oracle_drop import _dense_rows, _tiny_problem


@pytest.fixture(scope="module")
def tiny(oracle_mod):
    geom, H = _tiny_problem(oracle_mod)
    hs = oracle_mod.Histories(H)
    A = _dense_rows(oracle_mod, geom, hs)
    rng = np.random.default_rng(5)
    x_true = rng.uniform(0.5, 1.5, geom.n_voxels)
    H["wepl"] = (A @ x_true).astype(np.float32)
    return geom, H, oracle_mod.Histories(H), A, x_true


def _slice(H, sl):
    return {k: (v if k in ("proj_cos", "proj_sin") else v[sl]) for k, v in H.items()}


def test_one_string_is_drop(oracle_mod, tiny):
    geom, H, hs, A, _ = tiny
    x0 = np.linspace(0.2, 1.0, geom.n_voxels)
    xa = oracle_mod.carp_iterate(geom, hs, 0.7, 130, 3, 1, x0.copy())
    xb, _ = oracle_mod.drop_iterate(geom, hs, 0.7, 130, 3, x0.copy())
    assert np.array_equal(xa, xb)


def test_identical_strings_average_to_the_string_solution(oracle_mod, tiny):
    """Three copies of the same data as three strings: every string gives the same estimate from the common
    x0, and the mean of three equal vectors is that vector (a wrong divisor or a string that starts from
    the previous string's result shows up here)."""
    geom, H, hs, A, _ = tiny
    sub = _slice(H, slice(0, 900))
    tri = {k: (v if k in ("proj_cos", "proj_sin") else np.concatenate([v, v, v])) for k, v in sub.items()}
    x0 = np.full(geom.n_voxels, 0.3)
    xa = oracle_mod.carp_iterate(geom, oracle_mod.Histories(tri), 0.9, 250, 2, 3, x0.copy())
    xb, _ = oracle_mod.drop_iterate(geom, oracle_mod.Histories(sub), 0.9, 250, 2, x0.copy())
    assert xa == pytest.approx(xb, abs=1e-13)


def test_one_row_per_string_is_the_mean_of_kaczmarz_projections(oracle_mod, tiny):
    """P strings of one history each, blocks of one row: x = x0 + (1/P) sum_p lam (b_p - a_p.x0)/||a_p||^2 a_p
    (every hit count is 1), re-stated with the dense rows in numpy."""
    geom, H, hs, A, _ = tiny
    P = 40
    sub = _slice(H, slice(100, 100 + P))
    x0 = np.linspace(0.5, 1.5, geom.n_voxels)
    b = sub["wepl"].astype(np.float64)
    Ad = A[100:100 + P]
    nrm = (Ad * Ad).sum(axis=1)
    ok = nrm > 0  # a history that misses the hull has an empty row: its string returns x0 (R13)
    assert ok.sum() >= P - 4 and not ok.all()
    r = np.where(ok, (b - Ad @ x0) / np.where(ok, nrm, 1.0), 0.0)
    expect = x0 + (0.8 / P) * (r[:, None] * Ad).sum(axis=0)
    got = oracle_mod.carp_iterate(geom, oracle_mod.Histories(sub), 0.8, 1, 1, P, x0.copy())
    assert got == pytest.approx(expect, abs=1e-12)


def test_strings_are_contiguous_balanced_ranges_with_their_own_blocks(oracle_mod, tiny):
    """string p = [floor(p n / P), floor((p + 1) n / P)); its blocks count from its own first history."""
    geom, H, hs, A, _ = tiny
    n, P, B, lam = 1003, 4, 100, 0.6  # 1003 = 250 + 251 + 251 + 251: ragged strings, ragged last blocks
    sub = _slice(H, slice(0, n))
    x0 = np.full(geom.n_voxels, 0.4)
    parts = []
    for p in range(P):
        lo, hi = (p * n) // P, ((p + 1) * n) // P
        xs, _ = oracle_mod.drop_iterate(geom, oracle_mod.Histories(_slice(sub, slice(lo, hi))), lam, B, 1, x0.copy())
        parts.append(xs)
    got = oracle_mod.carp_iterate(geom, oracle_mod.Histories(sub), lam, B, 1, P, x0.copy())
    assert got == pytest.approx(np.mean(parts, axis=0), abs=1e-13)
    # second iteration starts every string from the average
    got2 = oracle_mod.carp_iterate(geom, oracle_mod.Histories(sub), lam, B, 2, P, x0.copy())
    again = oracle_mod.carp_iterate(geom, oracle_mod.Histories(sub), lam, B, 1, P, got.copy())
    assert got2 == pytest.approx(again, abs=1e-13)
    with pytest.raises(RuntimeError):
        oracle_mod.carp_iterate(geom, oracle_mod.Histories(_slice(sub, slice(0, 3))), lam, B, 1, 4, x0.copy())


def test_converges_on_consistent_data(oracle_mod, tiny):
    """Noise-free data: the CARP iterate approaches the dense least-squares solution on the well-determined
    columns (slower than DROP: the strings' steps are averaged), and the error keeps shrinking."""
    geom, H, hs, A, x_true = tiny
    hit = (A != 0).any(axis=0)
    b = hs.a["wepl"].astype(np.float64)
    x_ls, *_ = np.linalg.lstsq(A[:, hit], b, rcond=None)
    col = np.linalg.norm(A[:, hit], axis=0)
    x = oracle_mod.carp_iterate(geom, hs, 1.9, 50, 400, 4, np.zeros(geom.n_voxels))
    e1 = np.abs(x[hit] - x_ls)[col > 1.0].max()
    assert e1 < 5e-3
    x2 = oracle_mod.carp_iterate(geom, hs, 1.9, 50, 200, 4, x.copy())
    assert np.linalg.norm(x2[hit] - x_ls) < np.linalg.norm(x[hit] - x_ls)
    assert (x[~hit] == 0).all()
