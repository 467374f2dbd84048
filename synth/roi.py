"""Region-of-interest analysis of a reconstructed image of a synthetic phantom: mean, standard deviation
and per-cent error of the RSP inside every insert -- the synthetic counterpart of the paper's Table 2
("mean RSP value and standard deviation for a region of interest within each insert").
Analysis of the OUTPUT only; none of the method's arithmetic.

    python -m synth.roi --config 1 [--iterations 6] [--carp-strings 4] [--histories 1e7] [--tvs 0.5 0.9995 4]

runs the reconstruction on cuda:0 through the C ABI and prints the table (markdown)."""
import argparse
import json

import numpy as np

from .phantoms import AIR, config, rsp_volume


def roi_table(cfg, image, shrink=0.7, z_shrink=0.8):
    """One row per shape of the phantom: voxels whose centre lies inside the shape shrunk by `shrink` about its
    centre (cylinders: the central `z_shrink` of the grid's depth) and in no later shape's bounding region.
    -> list of dict(shape, true, voxels, mean, std, err_pct)."""
    img = np.asarray(image, dtype=np.float64).reshape(cfg.nz, cfg.ny, cfg.nx)
    xs = (np.arange(cfg.nx) + 0.5 - cfg.nx / 2) * cfg.h
    ys = (np.arange(cfg.ny) + 0.5 - cfg.ny / 2) * cfg.h
    zs = (np.arange(cfg.nz) + 0.5 - cfg.nz / 2) * cfg.h
    Z, Y, X = np.meshgrid(zs, ys, xs, indexing="ij")
    shapes = np.asarray(cfg.shapes, float)
    zlim = z_shrink * 0.5 * cfg.nz * cfg.h
    rows = []
    for k, (cx, cy, cz, ax, ay, az, rsp) in enumerate(shapes):
        inside = ((X - cx) / (shrink * ax)) ** 2 + ((Y - cy) / (shrink * ay)) ** 2 + ((Z - cz) / (shrink * az if az < 1e29 else az)) ** 2 <= 1.0
        inside &= np.abs(Z) <= zlim
        for (dx, dy, dz, bx, by, bz, _) in shapes[k + 1:]:  # keep clear of the shapes drawn on top of this one
            grow = 1.0 / shrink
            inside &= ((X - dx) / (grow * bx)) ** 2 + ((Y - dy) / (grow * by)) ** 2 + ((Z - dz) / (grow * bz if bz < 1e29 else bz)) ** 2 > 1.0
        v = img[inside]
        if v.size == 0:
            continue
        mean, std = float(v.mean()), float(v.std())
        rows.append(dict(shape=k, true=float(rsp), voxels=int(v.size), mean=mean, std=std,
                         err_pct=100.0 * (mean - rsp) / rsp if rsp > 10 * AIR else float("nan")))
    return rows


def markdown(rows):
    out = ["| shape | true RSP | voxels | mean | std | error % |", "|---|---|---|---|---|---|"]
    for r in rows:
        out.append("| %d | %.3f | %d | %.4f | %.4f | %s |" % (r["shape"], r["true"], r["voxels"], r["mean"], r["std"],
                                                             "%+.2f" % r["err_pct"] if r["err_pct"] == r["err_pct"] else "—"))
    return "\n".join(out)


def reconstruct(cfg, n, n_iter, carp_strings=0, spline=False, tvs=None):
    """The reconstruction of cfg's first n histories on cuda:0 through the C ABI -> image (numpy float32)."""
    import torch

    import paper_1707_05014_b200 as pct
    from . import to_pct_names
    from .cuda_gen import generate_cuda

    D = to_pct_names(generate_cuda(cfg, n))
    ctx = pct.pct_create(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out, torch.cuda.current_stream().cuda_stream)
    try:
        pct.pct_set_histories(ctx, n, D)
        pct.pct_set_path_model(ctx, pct.PCT_PATH_SPLINE if spline else pct.PCT_PATH_MLP)
        if tvs is not None:  # (beta0, gamma, n_halvings): total-variation superiorization
            pct.pct_set_tvs(ctx, *tvs)
        if carp_strings > 0:
            pct.pct_iterate_carp(ctx, cfg.lam, cfg.block_size, n_iter, carp_strings)
        else:
            pct.pct_iterate(ctx, cfg.lam, cfg.block_size, n_iter)
        out = torch.empty(cfg.n_voxels, dtype=torch.float32, device="cuda")
        pct.pct_get_image(ctx, out, cfg.n_voxels)
        return out.cpu().numpy()
    finally:
        pct.pct_destroy(ctx)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--histories", type=float, default=None)
    ap.add_argument("--iterations", type=int, default=None)
    ap.add_argument("--carp-strings", type=int, default=0)
    ap.add_argument("--spline", action="store_true", help="cubic-spline path model instead of the most-likely path")
    ap.add_argument("--tvs", type=float, nargs=3, default=None, metavar=("BETA0", "GAMMA", "HALVINGS"),
                    help="total-variation superiorization step before every DROP block / CARP iteration (PAPER.md:113)")
    ap.add_argument("--json", action="store_true")
    a = ap.parse_args()
    cfg = config(a.config)
    n = cfg.n if a.histories is None else int(a.histories)
    it = cfg.n_iter if a.iterations is None else a.iterations
    tvs = None if a.tvs is None else (a.tvs[0], a.tvs[1], int(a.tvs[2]))
    img = reconstruct(cfg, n, it, a.carp_strings, a.spline, tvs)
    rows = roi_table(cfg, img)
    truth = rsp_volume(cfg)
    hull = truth > 10 * AIR
    rms = float(np.sqrt(np.mean((img[hull] - truth[hull]) ** 2)))
    head = "%s, %d histories, %d iterations, %s, lambda %.3g, block %d; RMS error inside the object %.4f" % (
        cfg.workload, n, it, ("CARP with %d strings" % a.carp_strings if a.carp_strings else "DROP") + (", spline path" if a.spline else ", most-likely path"), cfg.lam, cfg.block_size, rms)
    if tvs is not None:
        head += "; TVS beta0 %g, gamma %g, %d halvings" % tvs
    if a.json:
        print(json.dumps(dict(run=head, rows=rows, rms=rms)))
    else:
        print(head + "\n\n" + markdown(rows))


if __name__ == "__main__":
    main()
