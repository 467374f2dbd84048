"""synth.roi.roi_table (the analysis behind BASELINE.md section 4 and tests/test_gpu_roi.py) on images whose answer is
known: the phantom's own RSP volume must come back with zero error and zero spread in every region, and a constant
offset must come back as that offset.  CPU only; none of the method's arithmetic is involved."""
import numpy as np
import pytest

import synth
from synth.roi import markdown, roi_table


@pytest.mark.parametrize("index", [0, 1])
def test_truth_volume_has_zero_error_everywhere(index):
    cfg = synth.config(index)
    truth = synth.rsp_volume(cfg)
    rows = roi_table(cfg, truth)
    assert len(rows) == len(cfg.shapes)  # every shape has a region
    for r in rows:
        assert r["voxels"] > 20
        assert r["mean"] == pytest.approx(r["true"], abs=1e-12) and r["std"] == pytest.approx(0.0, abs=1e-12)
        if r["true"] > 0.01:
            assert r["err_pct"] == pytest.approx(0.0, abs=1e-9)
    # an image that is 2 % high everywhere reads 2 % high in every region, noise shows up as the spread
    rows = roi_table(cfg, truth * 1.02)
    assert all(r["err_pct"] == pytest.approx(2.0, abs=1e-9) for r in rows if r["true"] > 0.01)
    noisy = truth + np.random.default_rng(0).normal(0, 0.03, truth.shape)
    rows = roi_table(cfg, noisy)
    assert all(0.02 < r["std"] < 0.04 for r in rows)
    assert "| shape | true RSP |" in markdown(rows)
