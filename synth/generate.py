"""numpy forward model: synthetic tracker histories for a phantom.

Per history i: projection p = i mod n_angles, entry uniform over the grid face at the entry tracker
plane with direction ~ N(0, 2 mrad); 1 mm depth steps through the analytic phantom with Gaussian
multiple scattering (Highland sigma without the log term per step), WEPL = sum RSP ds, residual
energy from the Bragg-Kleeman range; exit position/direction at the exit tracker plane; WEPL noise.
Deterministic in (seed, i): histories are drawn in fixed chunks of 65536, chunk c keyed (seed, c).
"""
import numpy as np

from .phantoms import rsp_at

FIELDS = ("t_in", "v_in", "t_out", "v_out", "tht_in", "thv_in", "tht_out", "thv_out", "wepl")
CHUNK = 65536
X0_MM = 361.0
MP = 938.272
E0 = 200.0
BK_A_MM, BK_P = 0.022, 1.77  # Bragg-Kleeman range R = 0.022 mm * E^1.77


def angle_table(n_angles):
    phi = 2.0 * np.pi * np.arange(n_angles) / n_angles
    return np.cos(phi).astype(np.float32), np.sin(phi).astype(np.float32)


def _chunk(cfg, c, noise):
    rng = np.random.Generator(np.random.Philox(key=[cfg.seed, c]))
    i = np.arange(c * CHUNK, (c + 1) * CHUNK, dtype=np.int64)
    proj = (i % cfg.n_angles).astype(np.uint16)
    phi = 2.0 * np.pi * proj / cfg.n_angles
    cs, sn = np.cos(phi), np.sin(phi)
    half_x, half_z = 0.5 * cfg.nx * cfg.h, 0.5 * cfg.nz * cfg.h
    t = rng.uniform(-half_x, half_x, CHUNK)
    v = rng.uniform(-half_z, half_z, CHUNK)
    tht = rng.normal(0.0, 2.0e-3, CHUNK)
    thv = rng.normal(0.0, 2.0e-3, CHUNK)
    out = dict(t_in=t.copy(), v_in=v.copy(), tht_in=tht.copy(), thv_in=thv.copy(), proj=proj)
    r0 = BK_A_MM * E0 ** BK_P
    wepl = np.zeros(CHUNK)
    u = cfg.u_in
    n_steps = int(round(cfg.u_out - cfg.u_in))
    for _ in range(n_steps):
        ds = np.sqrt(1.0 + tht * tht + thv * thv)
        tm, um, vm = t + 0.5 * tht, u + 0.5, v + 0.5 * thv
        rsp = rsp_at(cfg.shapes, tm * cs - um * sn, tm * sn + um * cs, vm)
        wepl += rsp * ds
        e = np.maximum((np.maximum(r0 - wepl, 0.0) / BK_A_MM) ** (1.0 / BK_P), 1.0)
        pv = (e * e + 2.0 * e * MP) / (e + MP)
        sig = 13.6 / pv * np.sqrt(rsp * ds / X0_MM)
        t += tht
        v += thv
        u += 1.0
        tht += sig * rng.standard_normal(CHUNK)
        thv += sig * rng.standard_normal(CHUNK)
    if noise:
        wepl += cfg.wepl_noise * wepl * rng.standard_normal(CHUNK)
    out.update(t_out=t, v_out=v, tht_out=tht, thv_out=thv, wepl=wepl)
    return out


def generate_numpy(cfg, n=None, noise=True):
    """First n histories of cfg as a dict of host arrays (float32 fields, uint16 proj, fp32 tables)."""
    n = cfg.n if n is None else int(n)
    parts = [_chunk(cfg, c, noise) for c in range((n + CHUNK - 1) // CHUNK)]
    out = {k: np.concatenate([p[k] for p in parts])[:n].astype(np.float32) for k in FIELDS}
    out["proj"] = np.concatenate([p["proj"] for p in parts])[:n]
    out["proj_cos"], out["proj_sin"] = angle_table(cfg.n_angles)
    return out
