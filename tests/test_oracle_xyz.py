"""Pins of the object-frame entry point of the oracle (orc_xyz_to_beam_*, R32).
CPU only.  The conversion is a rotation about z and a straight ray: pinned by special angles typed out by hand, by
the round trip through the rotation written the other way round (in the test), by the invariance under sliding the
hit along its ray, and fp32 against fp64."""
import numpy as np
import pytest


def test_special_angles_by_hand(oracle_mod):
    o = oracle_mod
    # phi = 0: x = t, y = u.  A hit at (3, -96, 2) with u_pl = -96 is already on the plane.
    assert o.xyz_to_beam_f64(-96.0, 3.0, -96.0, 2.0, 0.01, -0.02, 1.0, 0.0) == pytest.approx([3.0, 2.0])
    # phi = 90 deg: x = -u, y = t.  The plane u = -96 is x = +96; the hit (96, 5, 1) has t = 5.
    assert o.xyz_to_beam_f64(-96.0, 96.0, 5.0, 1.0, 0.0, 0.0, 0.0, 1.0) == pytest.approx([5.0, 1.0])
    # a hit 10 mm upstream of the plane (u = -106) with slopes 0.1, -0.05 arrives 1 mm / -0.5 mm further
    assert o.xyz_to_beam_f64(-96.0, 3.0, -106.0, 2.0, 0.1, -0.05, 1.0, 0.0) == pytest.approx([4.0, 1.5])


def test_round_trip_and_sliding_along_the_ray(oracle_mod):
    o = oracle_mod
    rng = np.random.default_rng(11)
    for _ in range(200):
        phi = rng.uniform(0, 2 * np.pi)
        cs, sn = np.cos(phi), np.sin(phi)
        t, v, tht, thv = rng.uniform(-90, 90), rng.uniform(-30, 30), rng.normal(0, 0.02), rng.normal(0, 0.02)
        u_pl = -96.0
        # beam frame -> object frame, written out here (x = t cos - u sin, y = t sin + u cos: pct.h conventions)
        for slide in (0.0, -7.5, 12.25):  # the same ray, hit recorded elsewhere along it
            u = u_pl + slide
            tt, vv = t + tht * slide, v + thv * slide
            x, y = tt * cs - u * sn, tt * sn + u * cs
            got = o.xyz_to_beam_f64(u_pl, x, y, vv, tht, thv, cs, sn)
            assert got == pytest.approx([t, v], abs=1e-10)


def test_fp32_rule_against_the_definition(oracle_mod):
    o = oracle_mod
    rng = np.random.default_rng(12)
    n, n_proj = 4000, 90
    phi = 2 * np.pi * np.arange(n_proj) / n_proj
    pc, ps = np.cos(phi).astype(np.float32), np.sin(phi).astype(np.float32)
    proj = rng.integers(0, n_proj, n).astype(np.uint16)
    x, y, z = (rng.uniform(-100, 100, n).astype(np.float32) for _ in range(3))
    tht, thv = (rng.normal(0, 0.03, n).astype(np.float32) for _ in range(2))
    t32, v32 = o.xyz_to_beam_f32(-96.0, x, y, z, tht, thv, proj, pc, ps)
    for i in range(0, n, 17):
        p = proj[i]
        ref = o.xyz_to_beam_f64(-96.0, x[i], y[i], z[i], tht[i], thv[i], pc[p], ps[p])
        assert abs(t32[i] - ref[0]) < 4e-5 and abs(v32[i] - ref[1]) < 4e-5  # a few ulp of 100 mm
    # an index beyond the table is clamped (R24)
    proj[:] = 65535
    t_c, _ = o.xyz_to_beam_f32(-96.0, x[:5], y[:5], z[:5], tht[:5], thv[:5], proj[:5], pc, ps)
    t_l, _ = o.xyz_to_beam_f32(-96.0, x[:5], y[:5], z[:5], tht[:5], thv[:5], np.full(5, n_proj - 1, np.uint16), pc, ps)
    assert np.array_equal(t_c, t_l)
