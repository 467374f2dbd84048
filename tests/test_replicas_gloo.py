"""N > 1 host logic (replicas only), world_size 2 over gloo on CPU.

The path has no data-path collective: what N > 1 adds is the slice of the seeded stream each rank
draws, the barrier, the max-over-ranks of the device time and the whole-job rate -- and, for the
reference arm, that rank 0 alone runs and prints.
"""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    import synth
    from paper_1707_05014_b200 import replicas

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n, steps = 70000, 3  # not a multiple of the generator's chunk: the slices straddle one
        first = replicas.shard_first(rank, n)
        cfg = synth.config(0)
        H = synth.generate_numpy(cfg, first + n)  # the stream is deterministic in (seed, index)
        np.save(os.path.join(out_dir, "t_in_%d.npy" % rank), H["t_in"][first:first + n])
        replicas.barrier(world)
        ms_local = 100.0 + 50.0 * rank  # rank 1 is the slow one
        ms, rate = replicas.whole_job_rate(ms_local, n, steps, world)
        with open(os.path.join(out_dir, "r%d.json" % rank), "w") as f:
            json.dump({"first": first, "ms": ms, "rate": rate}, f)
    finally:
        dist.destroy_process_group()


def test_two_replicas_draw_disjoint_slices_and_report_the_slowest(tmp_path):
    import synth

    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    res = [json.load(open(tmp_path / ("r%d.json" % r))) for r in range(world)]
    n, steps = 70000, 3
    assert [r["first"] for r in res] == [0, n]
    for r in res:  # every rank holds the max over ranks, and the whole-job rate over that time
        assert r["ms"] == 150.0
        assert r["rate"] == pytest.approx(world * n * steps / 0.150)
    # the two slices, side by side, are the first 2n histories of the one seeded stream
    whole = synth.generate_numpy(synth.config(0), world * n)["t_in"]
    got = np.concatenate([np.load(tmp_path / ("t_in_%d.npy" % r)) for r in range(world)])
    assert np.array_equal(got, whole)
    assert not np.array_equal(got[:n], got[n:])


def test_world_one_needs_no_process_group():
    sys.path.insert(0, ROOT)
    from paper_1707_05014_b200 import replicas

    assert replicas.max_over_ranks(12.5, 1) == 12.5
    assert replicas.whole_job_rate(200.0, 1000, 2, 1) == (200.0, 1000 * 2 / 0.2)
    with pytest.raises(ValueError):
        replicas.shard_first(-1, 10)


def _carp_worker(rank, world, port, out_dir, alias=False):
    import torch
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    import oracle
    import synth
    from paper_1707_05014_b200 import replicas

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = synth.config(0)
        n, lam, B, n_iter = 6001, 0.5, 700, 2
        H = synth.generate_numpy(cfg, n)
        lo, hi = replicas.string_range(rank, world, n)
        mine = {k: (v if k in ("proj_cos", "proj_sin") else v[lo:hi]) for k, v in H.items()}
        geom = oracle.Geometry(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out)
        hs = oracle.Histories(mine)
        state = {"x": np.zeros(cfg.n_voxels)}

        def sweep():  # the rank's local solver stands in for libpct on a GPU: one DROP sweep over its string
            state["x"], _ = oracle.drop_iterate(geom, hs, lam, B, 1, state["x"])

        if alias:
            # the form carp_distributed_pct uses on a GPU: get_image hands out the LIVE buffer the solver works on (the
            # library's own image array), the all-reduce and the division happen in place on it, set_image has nothing to do
            live = torch.zeros(cfg.n_voxels, dtype=torch.float64)

            def sweep_live():
                x, _ = oracle.drop_iterate(geom, hs, lam, B, 1, live.numpy())
                live.copy_(torch.from_numpy(x))

            replicas.carp_distributed(sweep_live, lambda: live, lambda t: None, n_iter, world)
            state["x"] = live.numpy().copy()
        else:
            replicas.carp_distributed(sweep, lambda: torch.from_numpy(state["x"].copy()),
                                      lambda t: state.update(x=t.numpy().copy()), n_iter, world)
        np.save(os.path.join(out_dir, "carp_%d.npy" % rank), state["x"])
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("alias", [False, True])
def test_carp_one_string_per_rank_equals_the_single_process_definition(tmp_path, alias):
    """CARP with one string per rank and an all-reduce of the image per iteration (the paper's cluster form,
    PAPER.md:52-56) gives, on every rank, what the oracle's single-process CARP gives for P = world strings -- in the copy
    form (get_image / set_image move copies) and in the in-place alias form replicas.carp_distributed_pct uses (get_image
    returns the live buffer, the collective works on it, set_image is a no-op)."""
    sys.path.insert(0, ROOT)
    import oracle
    import synth

    world, port = 2, _free_port()
    mp.spawn(_carp_worker, args=(world, port, str(tmp_path), alias), nprocs=world, join=True)
    cfg = synth.config(0)
    H = synth.generate_numpy(cfg, 6001)
    geom = oracle.Geometry(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out)
    want = oracle.carp_iterate(geom, oracle.Histories(H), 0.5, 700, 2, world, np.zeros(cfg.n_voxels))
    got = [np.load(tmp_path / ("carp_%d.npy" % r)) for r in range(world)]
    assert np.array_equal(got[0], got[1])  # every rank ends with the same image
    assert np.abs(want).max() > 0.1
    assert got[0] == pytest.approx(want, abs=1e-12)


def test_string_range_is_balanced_and_contiguous():
    sys.path.insert(0, ROOT)
    from paper_1707_05014_b200 import replicas

    n, world = 1003, 4
    r = [replicas.string_range(k, world, n) for k in range(world)]
    assert r[0][0] == 0 and r[-1][1] == n
    assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))
    assert max(b - a for a, b in r) - min(b - a for a, b in r) <= 1
    with pytest.raises(ValueError):
        replicas.string_range(4, 4, n)


def test_reference_arm_under_torchrun_prints_once():
    """`bench.py --impl reference` launched as the driver launches N = 2: rank 0 runs the oracle on its
    bounded sample and prints ONE JSON line, rank 1 exits 0 without work."""
    env = dict(os.environ, OMP_NUM_THREADS="4")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
           "--config", "0", "--steps", "1", "--warmup", "0"]
    r = subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
