"""Pins of the TVS oracle (oracle/tvs.py, reading R31 of DESIGN.md).  CPU only.

A plausible mistake -- a wrong sign of the direction, a difference taken backwards, a transposed axis, a missing
neighbour term of the gradient, a halving loop that accepts growth -- fails one of: the hand-computed spike, the
finite-difference check of the gradient, the axis-permutation check, the constant image, monotonicity."""
import numpy as np
import pytest

from oracle import tvs


def test_constant_image_is_a_fixed_point():
    shape = (5, 4, 3)
    x = np.full(60, 0.7)
    assert tvs.tv(x, shape) == pytest.approx(60 * tvs.EPS)
    assert np.abs(tvs.grad_tv(x, shape)).max() == 0.0
    z, info = tvs.tvs_step(x, shape, 1.0, 4)
    assert np.array_equal(z, x) and info["level"] == -1


def test_spike_on_a_line_by_hand():
    """x = (0, 1, 0, 0): TV = 2, grad = (-1, 2, -1, 0), v = (1, -2, 1, 0) / sqrt 6; with beta = 0.1 sqrt 6 the step
    gives (0.1, 0.8, 0.1, 0) and TV = 0.7 + 0.7 + 0.1 = 1.5."""
    shape = (4, 1, 1)
    x = np.array([0.0, 1.0, 0.0, 0.0])
    assert tvs.tv(x, shape) == pytest.approx(2.0, abs=1e-5)
    assert tvs.grad_tv(x, shape) == pytest.approx([-1.0, 2.0, -1.0, 0.0], abs=1e-5)
    z, info = tvs.tvs_step(x, shape, 0.1 * np.sqrt(6.0), 3)
    assert z == pytest.approx([0.1, 0.8, 0.1, 0.0], abs=1e-6)
    assert info["level"] == 0 and info["tv_after"] == pytest.approx(1.5, abs=1e-5)
    # the same spike along y and along z: the axes are treated alike
    for shp in ((1, 4, 1), (1, 1, 4)):
        z2, _ = tvs.tvs_step(x, shp, 0.1 * np.sqrt(6.0), 3)
        assert z2 == pytest.approx(z, abs=1e-12)


def test_too_long_a_step_is_halved_until_tv_does_not_grow():
    """Same spike, beta = 10 sqrt 6: z = (a, 1 - 2a, a, 0) with a = 10 / 2^l has TV = 2 |1 - 3a| + a, which exceeds 2
    for a = 10, 5, 2.5, 1.25, 0.625 and is 0.4375 for a = 0.3125: level 5."""
    shape = (4, 1, 1)
    x = np.array([0.0, 1.0, 0.0, 0.0])
    z, info = tvs.tvs_step(x, shape, 10.0 * np.sqrt(6.0), 8)
    assert info["level"] == 5
    assert info["tv_tried"] == pytest.approx([68.0, 33.0, 15.5, 6.75, 2.375, 0.4375], abs=1e-4)
    assert z == pytest.approx([0.3125, 0.375, 0.3125, 0.0], abs=1e-6)
    assert info["beta_used"] == pytest.approx(10.0 * np.sqrt(6.0) / 32.0)
    # with only five halvings nothing is accepted and the image stays
    z, info = tvs.tvs_step(x, shape, 10.0 * np.sqrt(6.0), 5)
    assert info["level"] == -1 and np.array_equal(z, x)
    assert info["beta_used"] == pytest.approx(10.0 * np.sqrt(6.0) / 32.0)


def test_gradient_against_central_differences():
    rng = np.random.default_rng(3)
    shape = (6, 5, 4)
    x = rng.uniform(0.0, 1.5, 120)
    g = tvs.grad_tv(x, shape)
    h = 1e-6
    for j in rng.choice(120, 25, replace=False):
        e = np.zeros(120)
        e[j] = h
        fd = (tvs.tv(x + e, shape) - tvs.tv(x - e, shape)) / (2 * h)
        assert g[j] == pytest.approx(fd, abs=2e-5)


def test_axes_are_in_the_order_of_the_voxel_index():
    """Voxel order i + nx (j + ny k): a ramp along x has the same TV as the same ramp laid along y or z of the
    transposed grid, and a ramp along x of a 5 x 3 x 2 grid contributes (nx - 1) * ny * nz unit differences."""
    nx, ny, nz = 5, 3, 2
    i = np.arange(nx * ny * nz) % nx
    assert tvs.tv(i.astype(float), (nx, ny, nz)) == pytest.approx((nx - 1) * ny * nz, abs=1e-3)
    j = (np.arange(nx * ny * nz) // nx) % ny
    assert tvs.tv(j.astype(float), (nx, ny, nz)) == pytest.approx(nx * (ny - 1) * nz, abs=1e-3)
    k = np.arange(nx * ny * nz) // (nx * ny)
    assert tvs.tv(k.astype(float), (nx, ny, nz)) == pytest.approx(nx * ny * (nz - 1), abs=1e-3)


def test_a_step_never_raises_the_total_variation_and_smooths_noise():
    rng = np.random.default_rng(5)
    shape = (16, 16, 4)
    base = np.zeros((4, 16, 16))
    base[:, 4:12, 4:12] = 1.0
    x = (base + rng.normal(0, 0.05, base.shape)).reshape(-1)
    beta, prev = 2.0, tvs.tv(x, shape)
    for _ in range(20):
        x, info = tvs.tvs_step(x, shape, beta, 6)
        assert info["tv_after"] <= info["tv_before"] == pytest.approx(prev)
        prev = info["tv_after"]
        beta = 0.9 * info["beta_used"]
    assert prev < 0.9 * tvs.tv((base + rng.normal(0, 0.05, base.shape)).reshape(-1), shape)
    # the step of a noisy flat region moves it towards its mean, not away
    assert np.abs(x.reshape(4, 16, 16)[:, 6:10, 6:10] - 1.0).std() < 0.05


def test_drop_with_tvs_reduces_to_drop_when_the_step_is_zero(oracle_mod):
    import synth
    from helpers import oracle_geom

    cfg = synth.config(0)
    H = synth.generate_numpy(cfg, 3000)
    geom = oracle_geom(oracle_mod, cfg)
    hs = oracle_mod.Histories(H)
    x0 = np.zeros(cfg.n_voxels)
    ref, _ = oracle_mod.drop_iterate(geom, hs, 0.5, 500, 1, x0.copy())  # (in place on its argument)
    got, beta, infos = tvs.drop_iterate_tvs(oracle_mod, geom, hs, 0.5, 500, 1, x0, 0.0, 0.9, 3)
    assert np.abs(got - ref).max() <= 1e-12 and len(infos) == 6
    got2, beta2, infos2 = tvs.drop_iterate_tvs(oracle_mod, geom, hs, 0.5, 500, 1, x0, 0.5, 0.9, 4)
    assert np.linalg.norm(got2 - ref) > 1e-6  # with a step it is another image
    assert tvs.tv(got2, (cfg.nx, cfg.ny, cfg.nz)) < tvs.tv(ref, (cfg.nx, cfg.ny, cfg.nz))
    assert 0 < beta2 <= 0.5 * 0.9 ** 6 + 1e-12
