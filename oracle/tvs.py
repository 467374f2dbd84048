"""CPU oracle of the total-variation superiorization (TVS) step -- TEST INFRASTRUCTURE, not the product.

PAPER.md:113 (section 4.2): "both algorithms incorporate total variation superiorization (TVS), which 'jiggles' the
solution to the imaging equation at some point in the reconstruction stream in order to find an optimal, feasible
solution.  A consequence of TVS is smoothing.  In CARP, TVS is applied just once to the initial solution at the start of
each iteration.  In DROP, however, TVS is applied to the initial solution that enters each block."  The paper prints no
formula; the step below is reading R31 of DESIGN.md (the perturbation step of the superiorization literature the
paper's group uses: a normalised non-ascending direction of the total variation, a step that is halved until the total
variation does not grow, and step sizes that shrink geometrically so that the perturbations are summable):

    TV(x)   = sum over voxels (i,j,k) of t_ijk,  t = sqrt(dx^2 + dy^2 + dz^2 + eps^2),
              dx = x[i+1,j,k] - x[i,j,k] (0 on the last column), dy, dz likewise        (isotropic, forward differences)
    g       = grad TV(x);   v = -g / ||g||_2   (no step if ||g|| = 0)
    for l = 0 .. n_half-1:   z = x + beta 2^-l v;   if TV(z) <= TV(x): x <- z, beta_used = beta 2^-l, stop
    (none accepted: x unchanged, beta_used = beta 2^-n_half)
    beta <- gamma * beta_used                                                            (for the next step)

Everything in float64 numpy, written out as the definition; no blocking, no fusion.  Shares no code with the CUDA path.
"""
import numpy as np

EPS = 1.0e-6


def _vol(x, shape):
    nx, ny, nz = shape
    return np.asarray(x, dtype=np.float64).reshape(nz, ny, nx)


def _diffs(v):
    """Forward differences along x, y, z (zero across the far faces)."""
    dx = np.zeros_like(v)
    dy = np.zeros_like(v)
    dz = np.zeros_like(v)
    dx[:, :, :-1] = v[:, :, 1:] - v[:, :, :-1]
    dy[:, :-1, :] = v[:, 1:, :] - v[:, :-1, :]
    dz[:-1, :, :] = v[1:, :, :] - v[:-1, :, :]
    return dx, dy, dz


def tv(x, shape, eps=EPS):
    """Total variation of the image x (flat, voxel order i + nx (j + ny k)); shape = (nx, ny, nz)."""
    dx, dy, dz = _diffs(_vol(x, shape))
    return float(np.sqrt(dx * dx + dy * dy + dz * dz + eps * eps).sum())


def grad_tv(x, shape, eps=EPS):
    """Gradient of tv() with respect to every voxel, flat."""
    v = _vol(x, shape)
    dx, dy, dz = _diffs(v)
    t = np.sqrt(dx * dx + dy * dy + dz * dz + eps * eps)
    px, py, pz = dx / t, dy / t, dz / t  # d t_ijk / d (the forward neighbour); minus their sum = d t_ijk / d x_ijk
    g = -(px + py + pz)
    g[:, :, 1:] += px[:, :, :-1]
    g[:, 1:, :] += py[:, :-1, :]
    g[1:, :, :] += pz[:-1, :, :]
    return g.reshape(-1)


def tvs_step(x, shape, beta, n_half, eps=EPS):
    """One perturbation step.  -> (x_new, info) with info = dict(tv_before, tv_after, level (-1: none accepted),
    beta_used, grad_norm, tv_tried=list of TV(z) for the levels tried)."""
    x = np.asarray(x, dtype=np.float64).reshape(-1)
    t0 = tv(x, shape, eps)
    g = grad_tv(x, shape, eps)
    gn = float(np.sqrt((g * g).sum()))
    info = dict(tv_before=t0, tv_after=t0, level=-1, beta_used=beta * 2.0 ** (-n_half), grad_norm=gn, tv_tried=[])
    if gn == 0.0:
        return x.copy(), info
    v = -g / gn
    for lev in range(n_half):
        b = beta * 2.0 ** (-lev)
        z = x + b * v
        tz = tv(z, shape, eps)
        info["tv_tried"].append(tz)
        if tz <= t0:
            info.update(tv_after=tz, level=lev, beta_used=b)
            return z, info
    return x.copy(), info


def drop_iterate_tvs(oracle, geom, hists, lam, block_size, n_iter, x, beta, gamma, n_half, n=None, eps=EPS):
    """DROP with a TVS step on the image that enters every block.  The block update itself is the
    oracle's (orc_block_accumulate + R12 in fp64).  -> (x, beta, infos)"""
    x = np.asarray(x, dtype=np.float64).copy()
    n = hists.n if n is None else n
    shape = (geom.nx, geom.ny, geom.nz)
    infos = []
    for _ in range(n_iter):
        for first in range(0, n, block_size):
            count = min(block_size, n - first)
            x, info = tvs_step(x, shape, beta, n_half, eps)
            beta = gamma * info["beta_used"]
            infos.append(info)
            d, c, _ = oracle.block_accumulate(geom, hists, first, count, x)
            x = x + lam * d / np.maximum(1.0, c)
    return x, beta, infos


def carp_iterate_tvs(oracle, geom, hists, lam, block_size, n_iter, n_strings, x, beta, gamma, n_half, eps=EPS):
    """CARP with one TVS step on the common start of every iteration.  -> (x, beta, infos)"""
    x = np.asarray(x, dtype=np.float64).copy()
    shape = (geom.nx, geom.ny, geom.nz)
    infos = []
    for _ in range(n_iter):
        x, info = tvs_step(x, shape, beta, n_half, eps)
        beta = gamma * info["beta_used"]
        infos.append(info)
        x = oracle.carp_iterate(geom, hists, lam, block_size, 1, n_strings, x)
    return x, beta, infos
