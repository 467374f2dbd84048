"""Synthetic counterpart of the paper's Table 2 (RSP of every insert of a cylindrical
phantom within about 1 % of the true value): configs[1] reconstructed in full on the GPU -- 1e7 histories,
128 x 128 x 32, the config's own block size, lambda and 6 iterations -- and the mean RSP of the body and of
the six inserts compared with the phantom.  Not a parity test: it checks that the path as a whole (hull, MLP,
walk, DROP / CARP) reconstructs the object the histories were generated from."""
import numpy as np
import pytest

import synth
from synth.roi import reconstruct, roi_table

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("carp_strings", [0, 4])
def test_config1_inserts_within_one_and_a_half_per_cent(carp_strings):
    import torch

    assert torch.cuda.is_available()
    cfg = synth.config(1)
    img = reconstruct(cfg, cfg.n, cfg.n_iter, carp_strings)
    assert np.isfinite(img).all()
    rows = roi_table(cfg, img)
    assert [r["shape"] for r in rows] == list(range(7))  # the body and the six inserts
    for r in rows:
        assert abs(r["err_pct"]) < 1.5, r
        assert r["std"] < 0.08, r
    # air outside the cylinder stays near zero, the body near 1
    vol = img.reshape(cfg.nz, cfg.ny, cfg.nx)
    assert abs(vol[cfg.nz // 2, 2, 2]) < 0.05
    assert rows[0]["voxels"] > 50_000 and abs(rows[0]["mean"] - 1.0) < 0.01
