"""Analytic phantoms and the five workload configurations of BASELINE.json:configs.

A phantom is an ordered list of ellipsoids (cx, cy, cz, ax, ay, az, rsp) in the object frame
(mm); a cylinder about z is an ellipsoid with az = inf.  RSP at a point = rsp of the LAST shape
that contains it, else air (0.001).  Details BASELINE.json leaves open (insert positions, sinus
ellipsoids, sphere seeds) are fixed here and listed in DESIGN.md.
"""
from dataclasses import dataclass, field

import numpy as np

AIR = 0.001
INF = 1.0e30
BASE_SEED = 170705014


@dataclass
class Config:
    index: int
    name: str
    n: int
    nx: int
    ny: int
    nz: int
    h: float
    n_angles: int
    block_size: int
    lam: float
    n_iter: int
    shapes: np.ndarray = field(repr=False)  # (S, 7) float64
    seed: int = BASE_SEED
    wepl_noise: float = 0.01

    @property
    def u_in(self):
        return -0.75 * self.h * max(self.nx, self.ny)

    @property
    def u_out(self):
        return 0.75 * self.h * max(self.nx, self.ny)

    @property
    def n_voxels(self):
        return self.nx * self.ny * self.nz

    @property
    def workload(self):
        return "configs[%d]: %s" % (self.index, self.name)


def _cyl(cx, cy, r, rsp):
    return [cx, cy, 0.0, r, r, INF, rsp]


def _ell(cx, cy, cz, ax, ay, az, rsp):
    return [cx, cy, cz, ax, ay, az, rsp]


def _ring(radius, r_insert, rsps, phase_deg):
    out = []
    for i, rsp in enumerate(rsps):
        a = np.deg2rad(phase_deg + 360.0 * i / len(rsps))
        out.append(_cyl(radius * np.cos(a), radius * np.sin(a), r_insert, rsp))
    return out


def _head(ax, ay, az, seed, n_spheres):
    shapes = [_ell(0, 0, 0, ax, ay, az, 1.7), _ell(0, 0, 0, ax - 5, ay - 5, az - 5, 1.04)]
    rng = np.random.Generator(np.random.Philox(key=seed + 7919))
    k = 0
    while k < n_spheres:
        p = rng.uniform(-1, 1, 3)
        if p @ p > 1.0:
            continue
        c = 0.8 * p * np.array([ax, ay, az])
        r = rng.uniform(3.0, 12.0)
        rsp = rng.uniform(0.2, 1.8)
        shapes.append(_ell(c[0], c[1], c[2], r, r, r, rsp))
        k += 1
    return shapes


def config(index, n=None):
    """Workload k of BASELINE.json:configs (n overrides the history count, e.g. for samples)."""
    seed = BASE_SEED + index
    if index == 0:
        shapes = [_cyl(0, 0, 28.0, 1.0)] + _ring(15.0, 5.0, [0.0, 1.2, 1.6], 90.0)
        c = Config(0, "1e5 protons, 64x64x8, water cylinder + 3 inserts", 100_000, 64, 64, 8, 1.0, 90,
                   1_000, 0.1, 1, np.array(shapes), seed)
    elif index == 1:
        shapes = [_cyl(0, 0, 60.0, 1.0)] + _ring(35.0, 10.0, [0.25, 0.56, 0.87, 1.18, 1.49, 1.80], 0.0)
        c = Config(1, "1e7 protons, 128x128x32, cylinder + 6 inserts", 10_000_000, 128, 128, 32, 1.0,
                   180, 10_000, 0.1, 6, np.array(shapes), seed)
    elif index == 2:
        shapes = [_ell(0, 0, 0, 80, 95, 32, 1.7), _ell(0, 0, 0, 75, 90, 27, 1.04),
                  _ell(-20, 50, 0, 10, 15, 8, AIR), _ell(20, 50, 0, 10, 15, 8, AIR)]
        c = Config(2, "1e8 protons, 200x200x64, ellipsoid head + bone shell + air sinuses", 100_000_000,
                   200, 200, 64, 1.0, 360, 50_000, 0.05, 8, np.array(shapes), seed)
    elif index == 3:
        c = Config(3, "5e8 protons, 256x256x128, head ellipsoid + 20 random spheres", 500_000_000, 256,
                   256, 128, 1.0, 360, 100_000, 0.05, 10, np.array(_head(80, 95, 56, seed, 20)), seed)
    elif index == 4:
        c = Config(4, "2e9 protons, 256x256x160, head ellipsoid + 20 random spheres", 2_000_000_000, 256,
                   256, 160, 1.0, 720, 200_000, 0.03, 12, np.array(_head(80, 95, 70, seed, 20)), seed)
    else:
        raise ValueError("config index must be 0..4")
    if n is not None:
        c.n = int(n)
    return c


def rsp_at(shapes, x, y, z):
    """RSP of the phantom at object-frame points (numpy arrays, mm)."""
    x, y, z = np.broadcast_arrays(np.asarray(x, float), np.asarray(y, float), np.asarray(z, float))
    out = np.full(x.shape, AIR)
    for cx, cy, cz, ax, ay, az, rsp in np.asarray(shapes, float):
        inside = ((x - cx) / ax) ** 2 + ((y - cy) / ay) ** 2 + ((z - cz) / az) ** 2 <= 1.0
        out = np.where(inside, rsp, out)
    return out


def rsp_volume(cfg):
    """Voxel-centre sampling of the phantom, linear index i + nx*(j + ny*k)."""
    xs = (np.arange(cfg.nx) + 0.5 - cfg.nx / 2) * cfg.h
    ys = (np.arange(cfg.ny) + 0.5 - cfg.ny / 2) * cfg.h
    zs = (np.arange(cfg.nz) + 0.5 - cfg.nz / 2) * cfg.h
    Z, Y, X = np.meshgrid(zs, ys, xs, indexing="ij")
    return rsp_at(cfg.shapes, X, Y, Z).reshape(-1)
