#!/usr/bin/env python
"""bench.py -- throughput of the RadiusFPS hot path on B200 (one JSON line on stdout).

A "step" is one pass of the WHOLE hot path over one batch of synthetic clouds: fps_index_build
(a1-a6: bbox, voxel keys, radix sort, SoA gather, segments, spheres) + fps_sample (a7-a13: the
persistent fused kernel, all M-1 iterations), inputs already resident in HBM.  Default workload:
BASELINE.json configs[1] ("C2": B=16 indoor-room-like clouds, N=24000, M=6000).  `e2e` is the same
metric through fps_sample_host with HOST buffers (H2D + build + sample + D2H inside the timed
region).  `roofline` is for the dominant kernel (k_fps_batched, exact batched picking): algorithmic
bytes per launch (from the kernel's own counters in a separate,
untimed stats run) divided by its average launch duration measured with CUDA events on the
launching stream.  The same run also times the per-pick persistent kernel (the paper's iteration
structure, FPS_FLAG_PER_PICK) once as an ablation.
`cpu_baseline` is the CPU oracle timed on this box's host cores (rank 0, N=1 only).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C1..C5] [--impl reference]
  python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...
Multi-GPU: replicas only: every rank runs its own batch (seeds disjoint),
no data-path collective; time = max over ranks; value = all ranks' samples / that time ("weak").
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2606_06255_b200 import inputs, sharding  # noqa: E402

METRIC = "fps_samples_per_s"
UNIT = "samples/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C2", choices=sorted(inputs.WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra-configs", action="store_true", help="skip the per-config summary (C1..C5)")
    ap.add_argument("--n-vox", type=int, default=0)
    ap.add_argument("--tile-points", type=int, default=0)
    ap.add_argument("--cluster-size", type=int, default=0)
    ap.add_argument("--block-threads", type=int, default=0)
    ap.add_argument("--local-warps", type=int, default=0)
    ap.add_argument("--cand-per-thread", type=int, default=0)
    ap.add_argument("--per-pick", action="store_true", help="time the per-pick persistent kernel instead (ablation)")
    return ap.parse_args()


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ---------------------------------------------------------------------------------------------
# clocks sampler (nvidia-smi during the timed region)
# ---------------------------------------------------------------------------------------------
class Clocks:
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.rows, self.proc, self.gpu = [], None, gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self) -> dict:
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.12)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            f = [c.strip() for c in r.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ---------------------------------------------------------------------------------------------
# algorithmic bytes (DESIGN.md / SURVEY.md 8(d)) from the kernel's counters
# ---------------------------------------------------------------------------------------------
def algorithmic_bytes(st: dict) -> int:
    """SURVEY.md 8(d) / DESIGN.md "Algorithmic bytes", evaluated with the counters of the schedule
    that ran.  20 B per radius-prune test (centre 12, radius 4, Dist_v 4; group tests and voxel
    tests alike) + 16 B per (visited point, pick) pair (x, y, z, Dist_p) + 8 B key write-back per
    voxel visit + 4 B per effective Dist_p store + 8 B per voxel key per argmax (one argmax per
    pick in the per-pick kernel, one per round in the batched kernel) + 20 B per pick (s_j,
    out_idx, out_mindist) + batched kernel only: 4 B per point scanned by the candidate extraction
    and 20 B per candidate moved (x, y, z, Dist_p, index)."""
    argmaxes = st["rounds"] if st.get("rounds", 0) else st["iterations"]
    per_cloud_K = st["K_total"] / max(1, st["B"])
    return int(20 * (st["voxel_tests"] + st.get("group_tests", 0)) + 16 * st["points_visited"] + 8 * st["voxels_visited"]
               + 4 * st["effective"] + 8 * per_cloud_K * argmaxes + 20 * st["iterations"]
               + 4 * st.get("extract_points", 0) + 20 * st.get("candidates", 0))


def ncu_traffic(workload: str, per_pick: bool):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed
    `ncu --set full` capture of this workload (profiles/r01_traffic.csv: workload,kernel,bytes), else None."""
    path = os.path.join(ROOT, "profiles", "r01_traffic.csv")
    want = "k_fps_sample" if per_pick else "k_fps_batched"
    try:
        for row in open(path).read().splitlines()[1:]:
            f = [c.strip() for c in row.split(",")]
            if len(f) >= 3 and f[0] == workload and f[1] == want:
                return float(f[2])
    except OSError:
        pass
    return None


def latency_report(rf, kern_s, w, sm_mhz) -> dict:
    """The bound that binds: the M-1 picks of a cloud are sequentially dependent, so `fps_sample` cannot be
    faster than (M-1) x the dependent chain of one pick.  The floor is MEASURED live: the bare chain on one
    warp with 1 candidate per lane (fps_pick_chain_cycles; the kernel's pick warp holds 2 per lane).  The
    clouds of a batch run in parallel, so the achieved figure is kernel time / (M-1) per cloud."""
    ghz = (sm_mhz or GHZ_FALLBACK * 1e3) * 1e-3
    floor1 = rf.fps_pick_chain_cycles(1, 8192)
    floor2 = rf.fps_pick_chain_cycles(2, 8192)
    achieved = kern_s * ghz * 1e9 / max(1, w.M - 1)
    return {"bound": "latency", "unit": "SM cycles per pick", "floor": floor1, "floor_2_candidates_per_lane": floor2,
            "achieved": achieved, "frac": floor1 / achieved,
            "note": "floor = bare chain update -> lane max -> redux(max D) -> redux(slot id) -> 3 shared loads on one warp, "
                    "no tie handling, no candidate selection, no global rounds"}


def opts_from(args) -> dict:
    return dict(n_vox=args.n_vox, tile_points=args.tile_points, cluster_size=args.cluster_size,
                block_threads=args.block_threads, local_warps=args.local_warps, cand_per_thread=args.cand_per_thread,
                flags=(16 if args.per_pick else 0))


GHZ_FALLBACK = 1.965


def phase_ms(st: dict, sm_mhz) -> dict:
    """Per-phase time of the batched kernel (SM cycles seen by thread 0 of each cloud's first CTA,
    averaged over clouds, converted with the SM clock sampled during the run)."""
    ghz = (sm_mhz or GHZ_FALLBACK * 1e3) * 1e-3
    f = lambda k: st.get(k, 0) / max(1, st["B"]) / ghz / 1e6  # noqa: E731
    workers = max(1, st["B"] * max(1, st["cluster_size"] - 1))
    g = lambda k: st.get(k, 0) / workers / ghz / 1e6  # noqa: E731
    return {"picker_cta": {"argmax": f("cycles_max"), "extract": f("cycles_extract"),
                           "local_incl_wait_for_workers": f("cycles_local"), "apply_if_single_cta": f("cycles_apply")},
            "worker_cta_avg": {"prune_tests": g("cycles_prune_sum"), "point_visits": g("cycles_visit_sum")},
            "note": "with cluster_size > 1 the workers apply the picks while the picker CTA is still producing them"}


def time_config(rf, torch, w, P_host, steps, warmup, opts, flush):
    """Returns dict with per-step ms (whole path), sample-kernel ms, build ms, stats."""
    Pd = torch.from_numpy(P_host).cuda()
    out_idx = torch.empty((w.B, w.M), dtype=torch.int32, device="cuda")
    out_mind = torch.empty((w.B, w.M), dtype=torch.float32, device="cuda")
    ev = lambda: torch.cuda.Event(enable_timing=True)  # noqa: E731
    step_ms, kern_ms, build_ms = [], [], []
    st = None
    for it in range(warmup + steps):
        if flush is not None:
            flush.fill_(it)                       # evict L2 between iterations (not timed)
        e0, e1, e2 = ev(), ev(), ev()
        e0.record()
        ix = rf.fps_index_build(Pd, **opts)
        e1.record()
        rf.fps_sample(ix, w.M, w.start_idx, out_idx, out_mind)
        e2.record()
        e2.synchronize()
        if st is None:
            st = rf.fps_get_stats(ix)
        rf.fps_index_destroy(ix)
        if it >= warmup:
            step_ms.append(e0.elapsed_time(e2)); build_ms.append(e0.elapsed_time(e1)); kern_ms.append(e1.elapsed_time(e2))
    return dict(step_ms=step_ms, kern_ms=kern_ms, build_ms=build_ms, stats=st, out_idx=out_idx, out_mind=out_mind)


def stats_run(rf, torch, w, P_host, opts):
    Pd = torch.from_numpy(P_host).cuda()
    opts = dict(opts)
    opts["flags"] = opts.get("flags", 0) | rf.FPS_FLAG_STATS
    ix = rf.fps_index_build(Pd, **opts)
    rf.fps_sample(ix, w.M, w.start_idx)
    torch.cuda.synchronize()
    st = rf.fps_get_stats(ix)
    rf.fps_index_destroy(ix)
    return st


def cpu_oracle_sample(w, P_host, budget_s=15.0):
    """Times oracle/fps_oracle.c as it stands on a bounded sample of the workload: the first
    `nb` clouds (one thread per cloud) and the first `m` samples of each, sized from a calibration
    so that the run takes roughly `budget_s` seconds of wall time.  The oracle's cost per sample is
    N point updates whatever the iteration, so samples/s on a prefix is unbiased."""
    import oracle
    cores = os.cpu_count() or 1
    nb = min(w.B, cores)
    t = time.perf_counter()
    oracle.fps(P_host[:1], min(w.M, 65), w.start_idx, threads=1)          # calibration: 64 iterations, 1 cloud
    per_it = (time.perf_counter() - t) / 64
    m = int(max(2, min(w.M, budget_s / max(per_it, 1e-9))))
    t = time.perf_counter()
    oracle.fps(P_host[:nb], m, w.start_idx, threads=nb)
    dt = time.perf_counter() - t
    out = {"value": nb * m / dt, "unit": UNIT, "cores": int(oracle.fps.threads_used), "kind": "oracle",
           "sample": f"first {nb} of {w.B} clouds x first {m} of {w.M} samples, {dt:.1f} s wall, "
                     f"oracle/fps_oracle.c -O2 one thread per cloud", "ms_per_cloud_extrapolated": dt / m * w.M * 1e3}
    # SURVEY 8(d) CPU baseline (2): the plain CPU pruned variant (oracle/fps_pruned_cpu.c, the paper's section 3
    # algorithm, untuned), same clouds and threading, all M samples (its cost per sample falls as the prune bites,
    # so a prefix would be biased); its ratio to the oracle is the analogue of the paper's CPU speedups (`:697-705`).
    t = time.perf_counter()
    oracle.pruned_fps(P_host[:nb], w.M, w.start_idx, n_vox=16, threads=nb)
    dtp = time.perf_counter() - t
    out["pruned_cpu_variant"] = {"value": nb * w.M / dtp, "unit": UNIT, "cores": int(oracle.pruned_fps.threads_used),
                                 "n_vox": 16, "ms_per_cloud": dtp * 1e3,
                                 "speedup_over_oracle": (nb * w.M / dtp) / (nb * m / dt),
                                 "sample": f"first {nb} of {w.B} clouds x all {w.M} samples, {dtp:.2f} s wall, "
                                           f"oracle/fps_pruned_cpu.c one thread per cloud"}
    return out


def reference_arm(args, rank, world):
    """--impl reference: the CPU oracle on the host cores, same metric/config; rank 0 only."""
    if rank != 0:
        return
    w = inputs.WORKLOADS[args.workload]
    P = inputs.make_batch(w)
    import oracle
    cores = os.cpu_count() or 1
    nb = min(w.B, cores)
    t = time.perf_counter()
    oracle.fps(P[:1], min(w.M, 65), w.start_idx, threads=1)
    per_it = (time.perf_counter() - t) / 64
    total_steps = args.steps + args.warmup
    m = int(max(2, min(w.M, (120.0 / total_steps) / max(per_it, 1e-9))))   # whole run within ~2 minutes
    times = []
    for it in range(total_steps):
        t = time.perf_counter()
        oracle.fps(P[:nb], m, w.start_idx, threads=nb)
        if it >= args.warmup:
            times.append(time.perf_counter() - t)
    tot = sum(times)
    value = nb * m * args.steps / tot
    sample = f"each step = first {nb} of {w.B} clouds x first {m} of {w.M} samples (oracle/fps_oracle.c, one thread per cloud)"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": tot / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"{w.name}: {w.note}", "B": w.B, "N": w.N, "M": w.M, "start_idx": w.start_idx},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": int(oracle.fps.threads_used), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    args = parse()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        reference_arm(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    from paper_2606_06255_b200 import binding as rf
    rf.load()                                     # fails loudly if the CUDA library is missing
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    w = inputs.WORKLOADS[args.workload]
    seed = sharding.rank_seed(inputs.BASE_SEED, rank, w.B)      # weak scaling: disjoint clouds per rank
    P = inputs.make_batch(w, seed)
    opts = opts_from(args)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")    # 256 MiB > 126 MB L2

    # untimed: counters for the algorithmic bytes (identical outputs, separate stats build)
    st_counts = stats_run(rf, torch, w, P, opts)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    clocks = Clocks(local_rank)
    barrier()
    clocks.start()
    r = time_config(rf, torch, w, P, args.steps, args.warmup, opts, flush)
    barrier()
    clk = clocks.stop()
    total_ms = sharding.max_over_ranks(float(sum(r["step_ms"])), dist if world > 1 else None)
    value = world * w.B * w.M * args.steps / (total_ms * 1e-3)

    # end to end through the host entry point: pinned host buffers, copies inside the timed region
    Ph = torch.from_numpy(P).pin_memory()
    oi = torch.empty((w.B, w.M), dtype=torch.int32).pin_memory()
    om = torch.empty((w.B, w.M), dtype=torch.float32).pin_memory()
    for _ in range(args.warmup):
        rf.fps_sample_host(Ph, w.M, w.start_idx, out_idx=oi, out_mindist=om, **opts)
    barrier()
    t0 = time.perf_counter()
    for i in range(args.steps):
        rf.fps_sample_host(Ph, w.M, w.start_idx, out_idx=oi, out_mindist=om, **opts)
    torch.cuda.synchronize()
    e2e_s = sharding.max_over_ranks(time.perf_counter() - t0, dist if world > 1 else None)
    e2e_ok = bool(np.array_equal(oi.numpy(), r["out_idx"].cpu().numpy()))

    if rank == 0:
        peak, peak_src = measured_peak()
        kern_s = float(np.mean(r["kern_ms"])) * 1e-3
        alg = algorithmic_bytes(st_counts)
        achieved = alg / kern_s / 1e9
        st = r["stats"]
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"{w.name}: {w.note}", "B": w.B, "N": w.N, "M": w.M, "start_idx": w.start_idx,
                       "step": "fps_index_build + fps_sample (a1-a13)", "l2": "flushed between iterations (256 MiB fill)",
                       "n_vox": st["n_vox"], "K_max": st["K_max"], "cluster_size": st["cluster_size"],
                       "block_threads": st["block_threads"], "local_warps": st["local_warps"],
                       "cand_per_thread": st["cand_per_thread"],
                       "kernel": "per-pick persistent (ablation)" if args.per_pick else "exact batched picking",
                       "parallelism": f"replicas x{world}"},
            "ms_per_cloud": total_ms / args.steps / w.B,
            "sample_kernel_ms": float(np.mean(r["kern_ms"])), "index_build_ms": float(np.mean(r["build_ms"])),
            "sample_only_samples_per_s": w.B * w.M / kern_s, "us_per_iteration": kern_s * 1e6 / max(1, w.M - 1),
            "roofline": {"bound": "hbm", "kernel": "k_fps_sample" if args.per_pick else "k_fps_batched",
                         "achieved": achieved, "peak": peak, "unit": "GB/s",
                         "frac": achieved / peak, "frac_of_8000_nominal": achieved / 8000.0, "peak_source": peak_src,
                         "algorithmic_bytes_per_launch": alg, "traffic": ncu_traffic(w.name, args.per_pick),
                         "note": "BASELINE.json asks for the HBM roofline; it is NOT what binds this path: the working "
                                 "set is L1/L2 resident (see traffic) and the M-1 picks are sequentially dependent, so "
                                 "the kernel is bound by the latency of its pick chain (DESIGN.md section 8)",
                         "dense_equivalent_GBps": w.B * w.N * 16.0 * (w.M - 1) / kern_s / 1e9,
                         "us_per_pick": kern_s * 1e6 / max(1, w.M - 1)},
            "latency": latency_report(rf, kern_s, w, clk.get("sm_mhz")),
            "phases_ms_per_cloud": None if args.per_pick else phase_ms(st_counts, clk.get("sm_mhz")),
            "counters": {k: st_counts[k] for k in ("iterations", "group_tests", "voxel_tests", "voxels_visited",
                                                   "points_visited", "points_computed", "effective", "rounds",
                                                   "extract_retries", "single_picks", "candidates", "extract_points",
                                                   "sub_batches", "local_subrounds", "local_fallbacks")},
            "e2e": {"value": world * w.B * w.M * args.steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(P.nbytes),
                    "d2h_bytes_per_step": int(oi.numel() * 4 + om.numel() * 4), "ms_per_step": e2e_s / args.steps * 1e3,
                    "api": "fps_sample_host (pinned host buffers)", "matches_device_path": e2e_ok},
            "gpu_launches": (st["build_launches"] + 1) * args.steps,
            "clocks": clk,
        }
        if world == 1 and not args.per_pick and not args.no_extra_configs:
            o2 = dict(opts, flags=16, local_warps=0, cand_per_thread=0)
            r2 = time_config(rf, torch, w, P, 3, 3, o2, flush)
            line["ablation_per_pick_kernel"] = {
                "what": "the paper's iteration structure (one cluster-wide argmax exchange per sample) as ONE persistent "
                        "kernel, FPS_FLAG_PER_PICK; same index, same outputs",
                "sample_kernel_ms": float(np.median(r2["kern_ms"])),
                "outputs_identical": bool(torch.equal(r2["out_idx"], r["out_idx"]) and torch.equal(r2["out_mind"], r["out_mind"]))}
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_oracle_sample(w, P)
        if world == 1 and not args.no_extra_configs:
            line["all_configs"] = per_config_summary(rf, torch, flush, opts, peak)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def per_config_summary(rf, torch, flush, opts, peak):
    """north_star asks for ms/cloud + roofline fraction on each of the five configs: short runs
    (3 warm-up + 5 timed), same protocol, reported inside the one JSON line."""
    out = {}
    for name in ("C1", "C2", "C3", "C4", "C5"):
        w = inputs.WORKLOADS[name]
        P = inputs.make_batch(w)
        stc = stats_run(rf, torch, w, P, opts)
        r = time_config(rf, torch, w, P, 5, 3, opts, flush)
        k = float(np.median(r["kern_ms"])) * 1e-3
        alg = algorithmic_bytes(stc)
        out[name] = {"B": w.B, "N": w.N, "M": w.M, "sample_ms": k * 1e3, "sample_ms_per_cloud": k * 1e3 / w.B,
                     "rounds_per_cloud": stc["rounds"] / w.B, "picks_per_round": stc["iterations"] / max(1, stc["rounds"]),
                     "build_plus_sample_ms_per_cloud": float(np.median(r["step_ms"])) / w.B,
                     "samples_per_s": w.B * w.M / k, "us_per_iteration": k * 1e6 / (w.M - 1),
                     "hbm_roofline_frac_measured_peak": alg / k / 1e9 / peak, "hbm_roofline_frac_8000": alg / k / 1e9 / 8000.0,
                     "n_vox": stc["n_vox"], "K_max": stc["K_max"], "cluster_size": stc["cluster_size"],
                     "points_visited_per_iter": stc["points_visited"] / stc["iterations"],
                     "voxels_visited_per_iter": stc["voxels_visited"] / stc["iterations"]}
    return out


if __name__ == "__main__":
    main()
