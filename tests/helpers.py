"""Shared test helpers: map the seeded synthetic histories (synth/) onto the two sides.

synth names its arrays after the beam frame (t_in, tht_in, ...); include/pct.h names them
entry_t, entry_dt, ...  Nothing here computes anything of the method."""
import numpy as np

SYNTH_TO_PCT = dict(t_in="entry_t", v_in="entry_v", t_out="exit_t", v_out="exit_v", tht_in="entry_dt",
                    thv_in="entry_dv", tht_out="exit_dt", thv_out="exit_dv", wepl="wepl", proj="proj",
                    proj_cos="proj_cos", proj_sin="proj_sin")


def to_device(H, device="cuda"):
    """synth dict of numpy arrays -> dict of CUDA tensors keyed as include/pct.h."""
    import torch

    out = {}
    for k, v in H.items():
        a = np.ascontiguousarray(v)
        if a.dtype == np.uint16:
            t = torch.from_numpy(a.view(np.int16)).to(device)
        else:
            t = torch.from_numpy(a.astype(np.float32)).to(device)
        out[SYNTH_TO_PCT[k]] = t
    return out


def to_host_pct(H):
    """synth dict -> dict of contiguous numpy arrays keyed as include/pct.h (for pct_set_histories_host)."""
    out = {}
    for k, v in H.items():
        a = np.ascontiguousarray(v)
        out[SYNTH_TO_PCT[k]] = a if a.dtype == np.uint16 else a.astype(np.float32)
    return out


def slice_hist(H, sl):
    return {k: (v[sl] if k not in ("proj_cos", "proj_sin") else v) for k, v in H.items()}


def oracle_geom(oracle, cfg):
    return oracle.Geometry(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out)
