"""pct_set_histories_xyz (object-frame entry point, R32) against the oracle:
tracker hits given as object-frame points somewhere along the rays; the oracle converts them with its own fp32 rule
(orc_xyz_to_beam_f32) and walks / iterates on the result: voxel sequences bit-exact, DROP run within the tolerances."""
import numpy as np
import pytest

import synth
from helpers import oracle_geom

pytestmark = pytest.mark.gpu


def test_rows_and_a_run_from_object_frame_hits(oracle_mod):
    import torch

    import paper_1707_05014_b200 as pct

    oracle = oracle_mod
    cfg = synth.config(1)
    n = 6000
    H = synth.generate_numpy(cfg, n)
    rng = np.random.default_rng(21)
    cs, sn = H["proj_cos"].astype(np.float64)[H["proj"]], H["proj_sin"].astype(np.float64)[H["proj"]]
    X = {}
    for side, u_pl in (("in", cfg.u_in), ("out", cfg.u_out)):
        slide = rng.uniform(-6.0, 6.0, n)  # the hit is recorded up to 6 mm before or behind the plane
        u = u_pl + slide
        t = H["t_" + side].astype(np.float64) + H["tht_" + side].astype(np.float64) * slide
        v = H["v_" + side].astype(np.float64) + H["thv_" + side].astype(np.float64) * slide
        X[side] = ((t * cs - u * sn).astype(np.float32), (t * sn + u * cs).astype(np.float32), v.astype(np.float32))
    # oracle side: its own conversion, then the usual path
    Ho = dict(H)
    Ho["t_in"], Ho["v_in"] = oracle.xyz_to_beam_f32(cfg.u_in, *X["in"], H["tht_in"], H["thv_in"], H["proj"], H["proj_cos"], H["proj_sin"])
    Ho["t_out"], Ho["v_out"] = oracle.xyz_to_beam_f32(cfg.u_out, *X["out"], H["tht_out"], H["thv_out"], H["proj"], H["proj_cos"], H["proj_sin"])
    assert np.abs(Ho["t_in"] - H["t_in"]).max() < 2e-4  # the hits do come back to the planes
    hs = oracle.Histories(Ho)
    geom = oracle_geom(oracle, cfg)
    table = oracle.sigma1_table(geom.h, geom.nmin)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    D = dict(entry_x=dev(X["in"][0]), entry_y=dev(X["in"][1]), entry_z=dev(X["in"][2]),
             exit_x=dev(X["out"][0]), exit_y=dev(X["out"][1]), exit_z=dev(X["out"][2]),
             entry_dt=dev(H["tht_in"]), entry_dv=dev(H["thv_in"]), exit_dt=dev(H["tht_out"]), exit_dv=dev(H["thv_out"]),
             wepl=dev(H["wepl"]), proj=dev(H["proj"].view(np.int16)), proj_cos=dev(H["proj_cos"]), proj_sin=dev(H["proj_sin"]))
    M = cfg.n_voxels
    ctx = pct.pct_create(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out, torch.cuda.current_stream().cuda_stream)
    try:
        with pytest.raises(pct.PctError):
            pct.pct_set_histories_xyz(ctx, n, {k: (v.cpu() if k == "entry_x" else v) for k, v in D.items()})  # a host pointer
        pct.pct_set_histories_xyz(ctx, n, D)
        ms = geom.nmin + 2
        nseg = torch.zeros(n, dtype=torch.int32, device="cuda")
        nnz = torch.zeros(n, dtype=torch.int32, device="cuda")
        seg_idx = torch.full((n, ms), -7, dtype=torch.int32, device="cuda")
        pct.pct_debug_rows(ctx, 0, n, ms, nseg, nnz, seg_idx)
        pct.pct_synchronize(ctx)
        nseg, nnz, seg_idx = nseg.cpu().numpy(), nnz.cpu().numpy(), seg_idx.cpu().numpy()
        paths = 0
        for i in range(0, n, 3):
            r = oracle.row_f32(geom, hs.hist(i), table)
            assert nseg[i] == r["nseg"] and nnz[i] == r["nnz"], i
            assert np.array_equal(seg_idx[i, :r["nseg"]], r["seg_idx"]), i
            paths += r["nseg"] > 0
        assert paths > 1500
        pct.pct_iterate(ctx, 0.3, 1000, 2)
        out = np.zeros(M, dtype=np.float32)
        pct.pct_get_image(ctx, out, M)
        x_ref, _ = oracle.drop_iterate(geom, hs, 0.3, 1000, 2, np.zeros(M))
        g = out.astype(np.float64)
        assert np.linalg.norm(g - x_ref) <= 1e-4 * np.linalg.norm(x_ref)
        assert np.abs(g - x_ref).max() <= 1e-3
    finally:
        pct.pct_destroy(ctx)
