"""Pins behind the block plan of the wavefront engine (csrc/pct_wave.cu, slab_range): the depth range a path can
reach is bounded from the hull points and the path's two shape functions, v(s) = chord(s) + c0(s) be0 + c2(s) be2
(DESIGN.md rule step 3c).  The library assumes |c0| <= 0.25 L for L <= 300 mm, <= 0.6 L beyond, and |c2| <= 0.16 L;
here those constants are checked against the fp64 matrix form of the most-likely path (oracle T64)
and against the cubic spline of the cheap path model (R30: 4/27 L).  CPU only."""
import numpy as np
import pytest


@pytest.mark.parametrize("L", [0.3, 1.0, 3.0, 10.0, 30.0, 64.0, 100.0, 128.0, 200.0, 256.0, 300.0])
def test_shape_functions_within_the_plan_bound_up_to_300mm(oracle_mod, L):
    ss = np.linspace(0.0, L, 301)[1:-1]
    c0 = np.array([oracle_mod.mlp_matrix_f64(s, L, [0, 1], [0, 0])[0] for s in ss])
    c2 = np.array([oracle_mod.mlp_matrix_f64(s, L, [0, 0], [0, 1])[0] for s in ss])
    assert np.abs(c0).max() <= 0.25 * L * 0.95  # 5 % to spare
    assert np.abs(c2).max() <= 0.16 * L * 0.95
    # a response to a unit slope never changes sign: the bound is on a one-signed bump
    assert c0.min() >= 0.0 and c2.max() <= 0.0


@pytest.mark.parametrize("L", [301.0, 400.0, 700.0, 1000.0, 2016.0, 4100.0])
def test_shape_functions_within_the_plan_bound_beyond_the_proton_range(oracle_mod, L):
    """Beyond the range of 200 MeV protons the scattering polynomial (R3) is extrapolated; the library accepts any
    hull chord up to min(nx, ny) = 2016 voxels, so the bound must hold there as well."""
    ss = np.linspace(0.0, L, 401)[1:-1]
    c0 = np.array([oracle_mod.mlp_matrix_f64(s, L, [0, 1], [0, 0])[0] for s in ss])
    c2 = np.array([oracle_mod.mlp_matrix_f64(s, L, [0, 0], [0, 1])[0] for s in ss])
    assert np.abs(c0).max() <= 0.6 * L * 0.95
    assert np.abs(c2).max() <= 0.16 * L * 0.95


def test_spline_shape_functions_are_bounded_by_four_twentyseventh():
    tau = np.linspace(0, 1, 10001)
    assert (tau * (1 - tau) ** 2).max() <= 4.0 / 27.0 + 1e-12 < 0.16
