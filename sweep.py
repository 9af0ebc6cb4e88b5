"""Sweeps on the synthetic scenes, mirroring the paper's scalability study (Fig. 14: latency vs sample
size) and its voxel-resolution study (Fig. 15).

    python sweep.py [--workloads C1,C2,C3,C4,C5] [--reps 3]

prints one markdown table per study: for M = N/64 .. N/2 at the automatic n_vox the three panels of Fig. 14 --
latency (`fps_sample`, CUDA events, best of `reps`; and index build + sampling), memory (device bytes owned by the
handle) and throughput (samples/s and input points/s of build + sample) -- and for n_vox = 8 .. 256 at the config's M
the latency, memory and voxel count, for the batched kernel and the per-pick kernel.  Results never depend on either
parameter (tests/test_gpu_parity.py); only time and memory do.  A third table times batches of small clouds (the
sampling layers of a point-cloud network) on the small-cloud kernel and on the general one.  Needs a CUDA device; there
is no CPU fallback.
"""
from __future__ import annotations

import argparse

import numpy as np
import torch

from paper_2606_06255_b200 import binding as rf
from paper_2606_06255_b200 import inputs


def time_sample(Pd, M, start, reps, **opts):
    """(best fps_sample ms, stats incl. device_bytes, best index-build ms)"""
    best_build = float("inf")
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        ix = rf.fps_index_build(Pd, **opts)
        e1.record()
        e1.synchronize()
        best_build = min(best_build, e0.elapsed_time(e1))
        rf.fps_index_destroy(ix)
    ix = rf.fps_index_build(Pd, **opts)
    best = float("inf")
    try:
        for _ in range(reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            rf.fps_sample(ix, M, start)
            e1.record()
            e1.synchronize()
            best = min(best, e0.elapsed_time(e1))
        st = rf.fps_get_stats(ix)
    finally:
        rf.fps_index_destroy(ix)
    st["build_ms"] = best_build
    return best, st


def small_cloud_table(reps):
    """Batches shaped like the sampling layers of a point-cloud network (B clouds of 1 024 .. 16 384 points, M = N/4): the
    small-cloud kernel (one CTA per cloud, the default up to 8 192 points) beside the general kernel (an explicit
    cluster size selects it), and the index build."""
    print("\n### Small-cloud batches: B x N -> N/4 (uniform cube), fps_sample and index build\n")
    print("| B | N | M | default kernel | fps_sample ms | us per pick | general kernel ms (cluster of 4) | index build ms | M samples/s (build + sample) |")
    print("|---|---|---|---|---|---|---|---|---|")
    for B in (1, 32, 128):
        for N in (1024, 2048, 4096, 8192, 16384):
            if B * N > 1 << 21:
                continue
            M = N // 4
            Pd = torch.from_numpy(np.stack([inputs.uniform_cube(N, 7000 + b) for b in range(B)])).cuda()
            t, st = time_sample(Pd, M, 0, reps)
            tg, _ = time_sample(Pd, M, 0, reps, cluster_size=4)
            kern = "small-cloud" if st["whole_cloud_kernel"] else (f"general, grid {st['grid_ctas']}" if st["grid_ctas"] else f"general, cluster {st['cluster_size']}")
            tot = t + st["build_ms"]
            print(f"| {B} | {N} | {M} | {kern} | {t:.3f} | {t * 1e3 / max(1, M - 1):.3f} | {tg:.3f} | {st['build_ms']:.3f} | {B * M / tot / 1e3:.2f} |", flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workloads", default="C1,C2,C3,C4,C5")
    ap.add_argument("--reps", type=int, default=3)
    ap.add_argument("--no-small", action="store_true", help="skip the small-cloud batch table")
    args = ap.parse_args()
    if not args.no_small:
        small_cloud_table(args.reps)
    for name in args.workloads.split(","):
        w = inputs.WORKLOADS[name]
        Pd = torch.from_numpy(np.ascontiguousarray(inputs.make_batch(w))).cuda()
        print(f"\n### {name}: B={w.B} N={w.N} -- latency, memory and throughput vs sample size M (automatic n_vox; Fig. 14)\n")
        print("| M | fps_sample ms | us per pick per cloud | build + sample ms | index memory MB | M samples/s (build + sample) | M input points/s | per-pick kernel ms |")
        print("|---|---|---|---|---|---|---|---|")
        for div in (64, 32, 16, 8, 4, 2):
            M = w.N // div
            tb, st = time_sample(Pd, M, w.start_idx, args.reps)
            tp, _ = time_sample(Pd, M, w.start_idx, 1, flags=rf.FPS_FLAG_PER_PICK) if M <= 70000 else (float("nan"), None)
            tot = tb + st["build_ms"]
            print(f"| N/{div} = {M} | {tb:.3f} | {tb * 1e3 / max(1, M - 1):.3f} | {tot:.3f} | {st['device_bytes'] / 1e6:.2f} | "
                  f"{w.B * M / tot / 1e3:.2f} | {w.B * w.N / tot / 1e3:.1f} | {tp:.3f} |", flush=True)
        print(f"\n### {name}: time of fps_sample (M={w.M}) vs voxel resolution n_vox\n")
        print("| n_vox | K_max (tiles of <= 64 points) | CTAs per cloud | index memory MB | build ms | batched kernel ms | per-pick kernel ms |")
        print("|---|---|---|---|---|---|---|")
        for nv in (8, 16, 32, 64, 128, 256):
            try:
                tb, st = time_sample(Pd, w.M, w.start_idx, args.reps, n_vox=nv)
                try:
                    tp, _ = time_sample(Pd, w.M, w.start_idx, 1, n_vox=nv, flags=rf.FPS_FLAG_PER_PICK)
                except rf.FpsError:
                    tp = float("nan")
                print(f"| {nv} | {st['K_max']} | {st['cluster_size']}{' (grid)' if st['grid_ctas'] else ''} | {st['device_bytes'] / 1e6:.2f} | "
                      f"{st['build_ms']:.3f} | {tb:.3f} | {tp:.3f} |", flush=True)
            except rf.FpsError as e:
                print(f"| {nv} | refused: {str(e)[:60]} | | | | | |", flush=True)


if __name__ == "__main__":
    main()
