"""pct_measure_peaks (the micro-benchmarks behind bench.py's roofline): sanity of what it returns on the
GPU of the run -- rates positive and ordered the way the hardware orders them, argument checks."""
import pytest

pytestmark = pytest.mark.gpu


def test_peaks_are_sane():
    import torch

    import paper_1707_05014_b200 as pct

    torch.zeros(1, device="cuda")
    r = pct.pct_measure_peaks(32 << 20)
    assert r["footprint_bytes"] == 32 << 20
    g = 1e9
    # an L2-resident footprint: tens to hundreds of G accesses per second, never above one per lane and clock
    for k in ("gather_random_per_s", "gather_path_per_s", "gather_path_tiled_per_s", "red_v2_random_per_s", "red_v2_path_per_s",
              "red_v2_path_tiled_per_s"):
        assert 20 * g < r[k] < 5000 * g, (k, r[k])
    # shaping the accesses like a path shares sectors between lanes; the tiled order shares more
    assert r["gather_path_per_s"] > r["gather_random_per_s"]
    assert r["gather_path_tiled_per_s"] > r["gather_path_per_s"]
    assert r["red_v2_path_tiled_per_s"] > r["red_v2_path_per_s"] > 0.9 * r["red_v2_random_per_s"]
    assert 0.5e12 < r["stream_read_bytes_per_s"] < 30e12
    # a packed FMA does two: the same flops at half the instructions
    assert 5e12 < r["ffma_inst_per_s"] < 60e12
    assert r["ffma2_inst_per_s"] == pytest.approx(0.5 * r["ffma_inst_per_s"], rel=0.15)
    # a footprint far beyond the L2 is slower
    big = pct.pct_measure_peaks(512 << 20)
    assert big["gather_random_per_s"] < 0.5 * r["gather_random_per_s"]
    for bad in (1000, 1 << 40):
        with pytest.raises(pct.PctError):
            pct.pct_measure_peaks(bad)
