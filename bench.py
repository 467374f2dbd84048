#!/usr/bin/env python
"""bench.py -- protons*iterations/s of the pCT hot path (MLP + voxel walk + DROP projection) on B200.

Contract (driver): ``python bench.py --gpus N --steps K --warmup W`` prints ONE JSON line on rank 0.
  * workload: BASELINE.json configs[3] (5e8 synthetic protons, 256x256x128 grid, B = 1e5, lambda = 0.05),
    the configuration the metric is quoted on; it fits one GPU (19 GB of histories).
  * a "step" = ONE DROP sweep over all N histories (rows a0-a6 of SURVEY.md section 8(a): history
    stream, hull, MLP, voxel walk, row projection, scatter, block update; 5000 blocks), i.e. one
    iteration of the paper's solver; `value` = N / step time = protons*iterations/s.
  * `value`: histories resident in HBM; `e2e`: the same step through the C ABI from pinned HOST
    arrays (pct_set_histories_host -> pct_iterate -> pct_get_image to host), copies inside the timing.
  * `roofline`: the fused accumulate kernel, timed with CUDA events around every launch (pct_profile_sweep), against the
    L2 rate measured in this run for its own access mix (pct_measure_peaks: 4 B gathers + 8 B vector reductions shaped like
    the row passes, L2-resident footprint) -- the metric's "HBM/L2 roofline"; the fp32-issue and HBM figures are reported
    beside it (`roofline.alu`, `roofline.hbm`), `roofline.traffic` comes from the ncu captures named in profiles/traffic.csv;
    `cpu_baseline`: the oracle timed on this box's host cores on a bounded sample.
  * ``--impl reference``: the oracle as it stands on the host cores (there is no reference code).
  * N > 1 (torchrun): replicas only -- every rank runs the same workload on its own histories, no
    data-path collective; value = sum of histories / max time.
  * side measurements (short JSON lines, not the driver's contract): --peaks, --carp (CARP, one string per rank under
    torchrun), --carp-strings P, --time-ordered, --path-model spline.
Inputs are seeded synthetic histories (synth/), generated on the GPU; nothing reads /root/reference.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "protons*iterations/s (MLP+projection)"
UNIT = "protons*iterations/s"

# Algorithmic work per unit, derived in DESIGN.md "Roofline": per raw path segment the rule
# prescribes 106 fp32/int operations (70 MLP node + 30 segment/voxel + 6 projection, FMA = 1);
# per history 38 B of HBM; per segment one 4 B gather, per non-zero one 8 B (Delta, c) reduction.
OPS_PER_SEGMENT = 106
HBM_BYTES_PER_HISTORY = 38
SM_COUNT_B200 = 148  # only the fallback: the run asks the device (multi_processor_count)
LANES_PER_SM = 128
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the fused accumulate kernel come from the committed ncu
# captures of THIS build, recorded in profiles/traffic.csv (file, commit, bytes per launch with ncu's cache flush and with
# --cache-control none), keyed by "config:block_size".
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "traffic.csv")


def ncu_traffic(config, block_size):
    try:
        import csv

        with open(TRAFFIC_CSV) as f:
            for row in csv.DictReader(f):
                if row["config:block_size"] == "%d:%d" % (config, block_size):
                    t = {"cold_bytes": float(row["cold_bytes"]), "warm_bytes": float(row["warm_bytes"]), "commit": row["commit"],
                         "file": row["file"], "kernel": row["kernel"]}
                    # hardware counters of the same capture (optional columns): what the kernel is limited by as ncu sees it
                    for k in ("warp_inst_per_launch", "issue_active", "warps_active_pct", "lts_throughput_pct", "l1_data_pipe_pct",
                              "dram_throughput_pct", "fma_pipe_pct", "registers"):
                        if row.get(k) not in (None, ""):
                            t[k] = float(row[k])
                    return t
    except (OSError, ValueError, KeyError):
        pass
    return None


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json configs index (default 3, the metric's)")
    ap.add_argument("--histories", type=float, default=None, help="override N (debugging only; reported)")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-full", dest="full", action="store_false",
                    help="skip the whole reconstruction (the config's own iteration count from x0 = 0, `full_reconstruction` in the line)")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--carp", action="store_true",
                    help="CARP across the ranks (the paper's own multi-processor scheme, PAPER.md:52-56): one string per rank, one "
                         "all-reduce of the image per iteration; a step = one CARP iteration.  Under torchrun with --gpus N; at N = 1 "
                         "it is one string = the DROP sweep.  A side measurement: `scaling` is strong (the N strings split one set)")
    ap.add_argument("--no-peaks", action="store_true", help="skip the L2 / fp32 micro-benchmarks behind roofline.l2")
    ap.add_argument("--peaks", action="store_true", help="only run the micro-benchmarks (pct_measure_peaks) and print them")
    ap.add_argument("--time-ordered", action="store_true",
                    help="histories in acquisition order (a block is nearly single-angle: the scanner rotates continuously, "
                         "PAPER.md:78) instead of interleaved angles; a sensitivity measurement (SURVEY.md 8(d))")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU time of the oracle sample")
    ap.add_argument("--path-model", default="mlp", choices=["mlp", "spline"],
                    help="spline: the cubic-spline path model (SURVEY.md 8(f) NEXT-3), a side measurement; the metric's is mlp")
    ap.add_argument("--tvs", type=float, default=0.0, metavar="BETA",
                    help="BETA > 0: a total-variation superiorization step (pct_set_tvs(BETA, 1.0, 4)) on the image that enters every "
                         "block (PAPER.md:113; SURVEY.md 8(f) NEXT-2), a side measurement: four more launches per block")
    ap.add_argument("--carp-strings", type=int, default=0,
                    help="P > 0: time pct_iterate_carp with P strings instead of the metric's DROP sweep (SURVEY.md 8(f) NEXT-1; "
                         "a side measurement: one short JSON line, not the driver's contract)")
    return ap.parse_args()


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            p = json.load(f)
        return dict(hbm_gbs=float(p["hbm_gbs"]), sm_max_mhz=float(p.get("sm_max_mhz", 1965.0)), source="measured")
    except (OSError, KeyError, ValueError):
        return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled every 200 ms while the timed region runs."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.lines = []
        self.proc = None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def __exit__(self, *exc):
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.proc.kill()
            self.thread.join(timeout=2)

    def summary(self):
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [s.strip() for s in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "power_w_max": max(pw), "reasons": sorted(reasons),
                "samples": len(sm)}


def cpu_oracle_rate(cfg, H, target_seconds, max_blocks=64):
    """The oracle as it stands (oracle/, OpenMP over the histories of a block) on the host cores:
    DROP sweep from x0 = 0 over the first blocks of the workload.  -> (rate, cores, blocks, seconds)."""
    import numpy as np

    import oracle

    oracle.build()
    geom = oracle.Geometry(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out)
    hs = oracle.Histories(H)
    B = cfg.block_size
    avail = hs.n // B
    t0 = time.perf_counter()
    oracle.drop_iterate(geom, hs, cfg.lam, B, 1, np.zeros(cfg.n_voxels), n=B)
    t1 = time.perf_counter() - t0
    nb = int(max(1, min(avail, max_blocks, round(target_seconds / max(t1, 1e-3)))))
    t0 = time.perf_counter()
    oracle.drop_iterate(geom, hs, cfg.lam, B, 1, np.zeros(cfg.n_voxels), n=nb * B)
    dt = time.perf_counter() - t0
    return nb * B / dt, oracle.num_threads(), nb, dt


def run_reference(args):
    """--impl reference: there is no reference code (the paper ships none); the arm is the oracle,
    unmodified, on the host cores.  A step = one DROP sweep over a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import numpy as np

    import oracle
    import synth

    cfg = synth.config(args.config)
    B = cfg.block_size
    nb = 4  # blocks per step: 4e5 histories of configs[3]
    H = synth.generate_numpy(cfg, nb * B)
    oracle.build()
    geom = oracle.Geometry(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out)
    hs = oracle.Histories(H)
    x = np.zeros(cfg.n_voxels)
    for _ in range(args.warmup):
        oracle.drop_iterate(geom, hs, cfg.lam, B, 1, x)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.drop_iterate(geom, hs, cfg.lam, B, 1, x)
    dt = time.perf_counter() - t0
    rate = nb * B * args.steps / dt
    cores = oracle.num_threads()
    sample = "%d blocks of %d histories of %s per step (generated by synth.generate_numpy)" % (nb, B, cfg.workload)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.workload, "grid": [cfg.nx, cfg.ny, cfg.nz], "block_size": B, "lambda": cfg.lam,
                   "histories_per_step": nb * B, "note": "CPU oracle (fp64 accumulation, fp32 rule rows); bounded sample"},
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    import paper_1707_05014_b200 as pct  # fails loudly if libpct.so cannot be built/loaded: no CPU path
    import synth
    import synth.cuda_gen as cuda_gen

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device: the path has no CPU fallback"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    from paper_1707_05014_b200 import replicas

    def barrier():
        replicas.barrier(world)

    def max_over_ranks(v):
        return replicas.max_over_ranks(v, world, "cuda")

    cfg = synth.config(args.config)
    n = cfg.n if args.histories is None else int(args.histories)
    B, lam, M = cfg.block_size, cfg.lam, cfg.n_voxels
    n_blocks = (n + B - 1) // B

    if args.time_ordered:
        n -= n % cfg.n_angles
        n_blocks = (n + B - 1) // B
    # replicas only: rank r draws histories [r*n, (r+1)*n) of the same seeded stream
    D = cuda_gen.generate_cuda(cfg, n, first=replicas.shard_first(rank, n))
    if args.time_ordered:
        # the generator interleaves the angles (history i belongs to projection i mod n_angles); acquisition order is
        # projection after projection: a transpose of the (n / n_angles, n_angles) view of every field
        for k in list(D):
            if k not in ("proj_cos", "proj_sin"):
                D[k] = D[k].view(n // cfg.n_angles, cfg.n_angles).t().contiguous().view(-1)
    P = synth.to_pct_names(D)
    stream = torch.cuda.Stream()
    out = {}
    if rank == 0 and not args.no_peaks:
        # the L2 / fp32 denominators of the roofline, measured on THIS GPU before the timed region (a second or two):
        # on an L2-resident footprint (32 MB) and on the footprint of image + accumulator of the workload
        torch.cuda.synchronize()
        out["peaks_l2"] = pct.pct_measure_peaks(32 << 20)
        out["peaks_ws"] = pct.pct_measure_peaks(max(1 << 20, 12 * M))
    with torch.cuda.stream(stream):  # torch.cuda.Event records on this stream, the one the kernels run on
        ctx = pct.pct_create(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out, stream.cuda_stream)
        try:
            pct.pct_set_path_model(ctx, pct.PCT_PATH_SPLINE if args.path_model == "spline" else pct.PCT_PATH_MLP)
            if args.tvs > 0:
                pct.pct_set_tvs(ctx, args.tvs, 1.0, 4)
            pct.pct_set_histories(ctx, n, P)
            for _ in range(args.warmup):
                pct.pct_iterate(ctx, lam, B, 1)
            pct.pct_synchronize(ctx)
            barrier()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            with ClockSampler(local) as clk:
                e0.record()
                for _ in range(args.steps):
                    pct.pct_iterate(ctx, lam, B, 1)
                e1.record()
                torch.cuda.synchronize()
                barrier()
            ms, out["value"] = replicas.whole_job_rate(e0.elapsed_time(e1), n, args.steps, world, "cuda")
            out["ms_per_step"] = ms / args.steps
            out["clocks"] = clk.summary()
            out["stats"] = pct.pct_get_stats(ctx)
            if args.tvs > 0:
                out["tvs_state"] = pct.pct_get_tvs_state(ctx)
            # the dominant kernel, CUDA events around every launch, one more sweep of the same workload
            prof = pct.pct_profile_sweep(ctx, lam, B)
            out["prof"] = prof
            img = torch.empty(M, dtype=torch.float32, device="cuda")
            pct.pct_get_image(ctx, img, M)
            out["image_finite"] = bool(torch.isfinite(img).all().item())
            out["image_mean_central"] = float(img.view(cfg.nz, cfg.ny, cfg.nx)[cfg.nz // 2, cfg.ny // 2 - 8:cfg.ny // 2 + 8,
                                                                           cfg.nx // 2 - 8:cfg.nx // 2 + 8].mean().item())
            out["sm_count"] = torch.cuda.get_device_properties(local).multi_processor_count
            if args.full and rank == 0:
                # the reconstruction north_star names: the config's own iteration count from x0 = 0, histories resident
                pct.pct_set_image(ctx, torch.zeros(M, dtype=torch.float32, device="cuda"), M)
                pct.pct_synchronize(ctx)
                e0.record()
                pct.pct_iterate(ctx, lam, B, cfg.n_iter)
                e1.record()
                pct.pct_get_image(ctx, img, M)
                out["full"] = {"iterations": cfg.n_iter, "seconds": e0.elapsed_time(e1) * 1e-3,
                               "image_finite": bool(torch.isfinite(img).all().item())}
        finally:
            pct.pct_destroy(ctx)

        # ---- end to end through the C ABI from pinned host memory ----
        if not args.no_e2e:
            host = {}
            for k, v in P.items():
                h = torch.empty(v.shape, dtype=v.dtype, pin_memory=True)
                h.copy_(v)
                host[k] = h
            torch.cuda.synchronize()
            h2d = sum(host[k].numel() * host[k].element_size() for k in host)
            img_host = torch.empty(M, dtype=torch.float32, pin_memory=True)
            ctx = pct.pct_create(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out, stream.cuda_stream)
            try:
                pct.pct_set_path_model(ctx, pct.PCT_PATH_SPLINE if args.path_model == "spline" else pct.PCT_PATH_MLP)
                if args.tvs > 0:
                    pct.pct_set_tvs(ctx, args.tvs, 1.0, 4)
                host_ms = [0.0, 0.0, 0.0]  # host clock: upload enqueue (+ device allocation), sweep enqueue, wait + D2H

                def e2e_step():
                    t0 = time.perf_counter()
                    pct.pct_set_histories_host(ctx, n, host)  # pipelined upload on the library's copy stream
                    t1 = time.perf_counter()
                    pct.pct_iterate(ctx, lam, B, 1)  # the first blocks start while the rest is on its way
                    t2 = time.perf_counter()
                    pct.pct_get_image(ctx, img_host, M)  # synchronises
                    t3 = time.perf_counter()
                    for i, d in enumerate((t1 - t0, t2 - t1, t3 - t2)):
                        host_ms[i] += d * 1e3

                e2e_step()  # warm-up (allocations, graph instantiation)
                barrier()
                torch.cuda.synchronize()
                host_ms[:] = [0.0, 0.0, 0.0]
                e0.record()
                for _ in range(args.e2e_steps):
                    e2e_step()
                e1.record()
                torch.cuda.synchronize()
                barrier()
                ms = max_over_ranks(e0.elapsed_time(e1))
                if "full" in out:  # the same reconstruction end to end: pinned host histories in, host image out
                    pct.pct_set_image(ctx, torch.zeros(M, dtype=torch.float32, device="cuda"), M)
                    pct.pct_synchronize(ctx)
                    t0 = time.perf_counter()
                    pct.pct_set_histories_host(ctx, n, host)
                    pct.pct_iterate(ctx, lam, B, cfg.n_iter)
                    pct.pct_get_image(ctx, img_host, M)
                    out["full"]["e2e_seconds"] = time.perf_counter() - t0
                out["e2e"] = {"value": world * n * args.e2e_steps / (ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                              "d2h_bytes_per_step": 4 * M, "steps": args.e2e_steps, "ms_per_step": ms / args.e2e_steps,
                              "host_ms_per_step": {"set_histories_host": host_ms[0] / args.e2e_steps,
                                                   "iterate_enqueue": host_ms[1] / args.e2e_steps,
                                                   "get_image_wait": host_ms[2] / args.e2e_steps},
                              "path": "pct_set_histories_host (pinned host SoA, upload pipelined with the first sweep) -> "
                                      "pct_iterate(1 sweep) -> pct_get_image (pinned host)"}
            finally:
                pct.pct_destroy(ctx)
            del host

    # ---- CPU baseline: the oracle on this box's host cores, rank 0, N = 1 only ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        n_s = min(n, 64 * B)
        Hs = {k: v[:n_s].cpu().numpy() for k, v in D.items() if k not in ("proj_cos", "proj_sin")}
        Hs["proj"] = Hs["proj"].view(np.uint16)
        Hs["proj_cos"], Hs["proj_sin"] = D["proj_cos"].cpu().numpy(), D["proj_sin"].cpu().numpy()
        rate, cores, nb, dt = cpu_oracle_rate(cfg, Hs, args.cpu_seconds)
        cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": dt,
               "sample": "first %d DROP blocks (%d histories) of the same workload, one sweep from x0 = 0" % (nb, nb * B)}

    if world > 1:
        dist.destroy_process_group()
    if rank != 0:
        return

    peaks = measured_peaks()
    st, prof = out["stats"], out["prof"]
    seg_per_hist = st["segments"] / max(1, st["histories"])
    nnz_per_hist = st["nnz"] / max(1, st["histories"])
    k_ms = prof["accumulate_ms"] / prof["blocks"]  # average device time of one launch
    hist_per_launch = n / prof["blocks"]
    ops = OPS_PER_SEGMENT * seg_per_hist * hist_per_launch
    sm_count = out.get("sm_count", SM_COUNT_B200)
    alu_peak = sm_count * LANES_PER_SM * peaks["sm_max_mhz"] * 1e6 / 1e12  # T thread-instructions/s
    alu_ach = ops / (k_ms * 1e-3) / 1e12
    hbm_ach = HBM_BYTES_PER_HISTORY * hist_per_launch / (k_ms * 1e-3) / 1e9
    l2_bytes = (4.0 * seg_per_hist + 8.0 * nnz_per_hist) * hist_per_launch
    traffic = ncu_traffic(args.config, B) or {}
    t_kernel = k_ms * 1e-3
    alu = {"achieved": alu_ach, "peak": alu_peak, "unit": "Tinst/s", "frac": alu_ach / alu_peak,
           "peak_source": "%d SM (asked of the device) x 128 fp32 lanes x %.0f MHz (MEASURED_PEAKS.json sm_max_mhz, %s)" % (sm_count, peaks["sm_max_mhz"], peaks["source"]),
           "algorithmic": "%d fp32/int ops per path segment (DESIGN.md Roofline) x %.1f segments/history x %d histories/launch" % (
               OPS_PER_SEGMENT, seg_per_hist, hist_per_launch),
           "time_at_peak_us": ops / (alu_peak * 1e12) * 1e6}
    hbm = {"achieved": hbm_ach, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": hbm_ach / peaks["hbm_gbs"],
           "peak_source": "MEASURED_PEAKS.json hbm_gbs (%s)" % peaks["source"], "algorithmic": "38 B/history",
           "time_at_peak_us": HBM_BYTES_PER_HISTORY * hist_per_launch / (peaks["hbm_gbs"] * 1e9) * 1e6}
    common = {
        "kernel": "pct::k_drop_pair (fused hull+MLP+walk+projection+scatter, two histories per warp; k_drop_block for blocks under four histories per warp)",
        "kernel_ms": k_ms, "launches_timed": prof["blocks"],
        "kernel_share_of_step": prof["accumulate_ms"] / prof["sweep_ms"],
        "update_kernel_ms": prof["update_ms"] / prof["blocks"],
        "timing": "CUDA events around every launch on the kernels' stream (pct_profile_sweep), one sweep of the timed workload",
        "traffic": traffic.get("cold_bytes"), "traffic_warm": traffic.get("warm_bytes"),
        "traffic_source": "%s (commit %s): dram__bytes_read.sum + dram__bytes_write.sum of one launch, ncu --set full (caches flushed) / "
                          "--cache-control none (warm)" % (traffic.get("file"), traffic.get("commit")) if traffic else None,
        "alu": alu, "hbm": hbm,
    }
    issue = None
    if "issue_active" in traffic:
        issue = {"warp_inst_per_history": traffic["warp_inst_per_launch"] / hist_per_launch if "warp_inst_per_launch" in traffic else None,
                 "issue_active": traffic["issue_active"], "warps_active_pct": traffic.get("warps_active_pct"),
                 "lts_throughput_pct": traffic.get("lts_throughput_pct"), "l1_data_pipe_pct": traffic.get("l1_data_pipe_pct"),
                 "dram_throughput_pct": traffic.get("dram_throughput_pct"), "fma_pipe_pct": traffic.get("fma_pipe_pct"),
                 "registers_per_thread": traffic.get("registers"),
                 "source": "%s (commit %s): one launch under ncu --set full" % (traffic.get("file"), traffic.get("commit"))}
        # what binds, as the hardware counters see it: a memory level counts as the limiter from 60 % of its peak throughput
        levels = {"l2": traffic.get("lts_throughput_pct", 0.0), "hbm": traffic.get("dram_throughput_pct", 0.0),
                  "l1 data pipe": traffic.get("l1_data_pipe_pct", 0.0)}
        top = max(levels, key=levels.get)
        issue["binds"] = top if levels[top] >= 60.0 else (
            "instruction issue and latency (issue slots %.0f %% busy at %.0f %% of the warp slots; no memory level above 60 %% of its "
            "peak: %s %.0f %%)" % (100 * traffic["issue_active"], traffic.get("warps_active_pct", 0.0), top, levels[top]))
    if "peaks_l2" in out:
        pk, pw = out["peaks_l2"], out["peaks_ws"]
        rg, rr, rm = pk["gather_path_tiled_per_s"], pk["red_v2_path_tiled_per_s"], pk["mixed_pairs_tiled_per_s"]
        # seconds per history at the measured L2 rates: the kernel's own mix (a gather and a reduction at the same voxel,
        # measured together) for the non-zeros, plain gathers for the segments that continue a run; and, beside it, the
        # two accesses at their separately measured rates, added up
        t_peak_hist = nnz_per_hist / rm + (seg_per_hist - nnz_per_hist) / rg
        t_peak_sum = seg_per_hist / rg + nnz_per_hist / rr
        l2_peak = l2_bytes / hist_per_launch / t_peak_hist / 1e9
        l2_ach = l2_bytes / t_kernel / 1e9
        alu_meas = pk["ffma_inst_per_s"] / 1e12
        alu["peak_measured_ffma"] = alu_meas
        alu["frac_of_measured_ffma"] = alu_ach / alu_meas
        times = {"l2": t_peak_hist * hist_per_launch * 1e6, "alu": alu["time_at_peak_us"], "hbm": hbm["time_at_peak_us"]}
        roofline = dict(common)
        roofline.update({
            "bound": "l2", "achieved": l2_ach, "peak": l2_peak, "unit": "GB/s", "frac": l2_ach / l2_peak,
            "algorithmic": "4 B gather per path segment + 8 B (Delta, c) reduction per non-zero: %.1f segments, %.1f non-zeros per "
                           "history = %.0f B/history x %d histories/launch" % (seg_per_hist, nnz_per_hist, l2_bytes / hist_per_launch,
                                                                                hist_per_launch),
            "peak_source": "measured in this run, before the timed region (pct_measure_peaks, 32 MiB = L2-resident, accesses shaped like "
                           "the row passes, voxels in the library's 2x2 tiles): %.0f G (gather + reduction) pairs/s measured "
                           "together, %.0f G gathers/s, %.0f G reductions/s alone; peak = the same bytes at the pair rate" % (
                               rm / 1e9, rg / 1e9, rr / 1e9),
            "frac_with_rates_added_up": (t_peak_sum * hist_per_launch) / t_kernel,
            "binds": issue["binds"] if issue else "unknown (no ncu counters recorded for this config in profiles/traffic.csv); "
                                                  "longest time-at-peak: " + max(times, key=times.get),
            "time_at_peak_us": times, "issue": issue,
            "l2_rates_on_working_set": {"footprint_bytes": pw["footprint_bytes"],
                                        "gather_path_tiled_per_s": pw["gather_path_tiled_per_s"],
                                        "red_v2_path_tiled_per_s": pw["red_v2_path_tiled_per_s"],
                                        "note": "the same micro-benchmarks on image + accumulator of this workload (not L2-resident "
                                                "when above ~64 MB): context, not the peak"},
            "peaks_measured": pk,
        })
    else:
        roofline = dict(common)
        roofline.update({"bound": "alu", "achieved": alu_ach, "peak": alu_peak, "unit": "Tinst/s", "frac": alu_ach / alu_peak,
                         "peak_source": alu["peak_source"], "algorithmic": alu["algorithmic"]})
    line = {
        "metric": METRIC, "value": out["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": out["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": cfg.workload, "histories": n, "grid": [cfg.nx, cfg.ny, cfg.nz], "voxel_mm": cfg.h,
                   "angles": cfg.n_angles, "block_size": B, "blocks_per_step": n_blocks, "lambda": lam,
                   "step": "one DROP sweep (iteration) over all histories",
                   "l2": "inputs larger than L2 (histories %.1f GB, image+accumulator %.0f MB vs 126 MB L2)" % (
                       38.0 * n / 1e9, 12.0 * M / 1e6),
                   "multi_gpu": "replicas only", "histories_override": args.histories is not None,
                   "history_order": "acquisition order, projection after projection (sensitivity run)" if args.time_ordered
                   else "angles interleaved (every block sees every angle)",
                   "path_model": "most-likely path (the metric's)" if args.path_model == "mlp"
                   else "cubic spline (side measurement, SURVEY.md 8(f) NEXT-3; the roofline's op count is the MLP's)"},
        "clocks": out["clocks"], "gpu_launches": (6 if args.tvs > 0 else 2) * n_blocks * args.steps,
        "segments_per_history": seg_per_hist, "nonzeros_per_history": nnz_per_hist,
        "skipped_fraction": 1.0 - st["rows"] / max(1, st["histories"]),
        "image_finite": out["image_finite"], "image_mean_central": out["image_mean_central"],
        "roofline": roofline,
    }
    if args.tvs > 0:
        line["config"]["tvs"] = "a TVS step before every block (side measurement): beta0 %g, gamma 1, 4 halvings" % args.tvs
        line["tvs"] = {"us_per_step": 1e3 * out["prof"]["tvs_ms"] / max(1, out["prof"]["blocks"]), "state": out["tvs_state"]}
    if "full" in out:
        line["full_reconstruction"] = dict(out["full"], workload=cfg.workload,
                                           note="DROP, %d iterations from x0 = 0 on one B200; e2e_seconds = host clock from pinned host "
                                                "histories to the host image.  Context only: PAPER.md:94 reports 91:43 for 0.527e9 histories "
                                                "on 1 core + 1 Tesla (CARP, whole program, iteration count unstated)" % cfg.n_iter)
    if "e2e" in out:
        line["e2e"] = out["e2e"]
    if cpu is not None:
        line["cpu_baseline"] = cpu
    print(json.dumps(line))


def run_carp(args):
    """Side measurement: one CARP iteration (P strings, each a DROP sweep over its histories, then the mean)."""
    import torch

    import paper_1707_05014_b200 as pct
    import synth
    import synth.cuda_gen as cuda_gen

    cfg = synth.config(args.config)
    n = cfg.n if args.histories is None else int(args.histories)
    P = args.carp_strings
    D = synth.to_pct_names(cuda_gen.generate_cuda(cfg, n))
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        ctx = pct.pct_create(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out, stream.cuda_stream)
        try:
            pct.pct_set_histories(ctx, n, D)
            for _ in range(args.warmup):
                pct.pct_iterate_carp(ctx, cfg.lam, cfg.block_size, 1, P)
            pct.pct_synchronize(ctx)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            with ClockSampler(0) as clk:
                e0.record()
                for _ in range(args.steps):
                    pct.pct_iterate_carp(ctx, cfg.lam, cfg.block_size, 1, P)
                e1.record()
                torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
        finally:
            pct.pct_destroy(ctx)
    print(json.dumps({"metric": METRIC, "value": n * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
                      "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "dtype": "f32",
                      "data": "synthetic", "clocks": clk.summary(),
                      "config": {"workload": cfg.workload, "algorithm": "CARP (PAPER.md:52-56)", "strings": P, "histories": n,
                                 "block_size": cfg.block_size, "lambda": cfg.lam,
                                 "step": "one CARP iteration: every string one DROP sweep over its histories, then the mean"}}))


def run_carp_ranks(args):
    """CARP with one string per rank (replicas.carp_distributed_pct): every rank sweeps its own string of the one seeded
    history set from the common image, then the all-reduce (sum, / world) of the image, in place on the library's array."""
    import torch
    import torch.distributed as dist

    import paper_1707_05014_b200 as pct
    import synth
    import synth.cuda_gen as cuda_gen
    from paper_1707_05014_b200 import replicas

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device: the path has no CPU fallback"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    cfg = synth.config(args.config)
    n = cfg.n if args.histories is None else int(args.histories)
    lo, hi = replicas.string_range(rank, world, n)  # R27: contiguous balanced strings of the caller's order
    D = synth.to_pct_names(cuda_gen.generate_cuda(cfg, hi - lo, first=lo))
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        ctx = pct.pct_create(cfg.nx, cfg.ny, cfg.nz, cfg.h, cfg.u_in, cfg.u_out, stream.cuda_stream)
        try:
            pct.pct_set_histories(ctx, hi - lo, D)
            _, n_slots = pct.pct_image_storage(ctx)
            tvs = args.tvs > 0  # one step per iteration on the common image, the placement of pct_iterate_carp
            if tvs:
                pct.pct_set_tvs(ctx, args.tvs, 1.0, 4)
            replicas.carp_distributed_pct(pct, ctx, cfg.n_voxels, cfg.lam, cfg.block_size, args.warmup, world, stream.cuda_stream, tvs=tvs)
            pct.pct_synchronize(ctx)
            replicas.barrier(world)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            with ClockSampler(local) as clk:
                e0.record()
                replicas.carp_distributed_pct(pct, ctx, cfg.n_voxels, cfg.lam, cfg.block_size, args.steps, world, stream.cuda_stream, tvs=tvs)
                e1.record()
                torch.cuda.synchronize()
                replicas.barrier(world)
            ms = replicas.max_over_ranks(e0.elapsed_time(e1), world, "cuda")
            img = torch.empty(cfg.n_voxels, dtype=torch.float32, device="cuda")
            pct.pct_get_image(ctx, img, cfg.n_voxels)
            finite = bool(torch.isfinite(img).all().item())
        finally:
            pct.pct_destroy(ctx)
    if world > 1:
        dist.destroy_process_group()
    if rank != 0:
        return
    n_blocks = ((hi - lo) + cfg.block_size - 1) // cfg.block_size
    print(json.dumps({
        "metric": METRIC, "value": n * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic", "clocks": clk.summary(), "gpu_launches": 2 * n_blocks * args.steps, "image_finite": finite,
        "comm": {"collective": "all-reduce (sum) of the image, in place on the library's array" if world > 1 else "none (one string)",
                 "bytes_per_rank_per_step": 4 * n_slots if world > 1 else 0},
        "config": {"workload": cfg.workload, "algorithm": "CARP, one string per rank (PAPER.md:52-56; DESIGN.md R27-R29)",
                   "strings": world, "histories": n, "histories_per_rank": hi - lo, "block_size": cfg.block_size, "lambda": cfg.lam,
                   "step": "one CARP iteration: every rank one DROP sweep over its string from the common image, then the average",
                   "note": "side measurement, not the driver's contract; unmeasured on N > 1 in this repository's runs (one GPU per run)"}}))


def run_peaks(args):
    """Only the micro-benchmarks behind roofline.l2 (pct_measure_peaks), on an L2-resident footprint and on the
    footprint of image + accumulator of the config."""
    import torch

    import paper_1707_05014_b200 as pct
    import synth

    cfg = synth.config(args.config)
    torch.cuda.set_device(0)
    torch.zeros(1, device="cuda")
    res = {"config": cfg.workload}
    for name, fp in (("l2_resident_32MiB", 32 << 20), ("image_plus_accumulator", max(1 << 20, 12 * cfg.n_voxels))):
        res[name] = pct.pct_measure_peaks(fp)
    print(json.dumps(res))


def main():
    args = parse_args()
    if args.peaks:
        run_peaks(args)
    elif args.carp and args.impl != "reference":
        run_carp_ranks(args)
    elif args.carp_strings > 0 and args.impl != "reference":
        run_carp(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
