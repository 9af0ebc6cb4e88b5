"""Sweeps on the synthetic scenes, mirroring the paper's scalability study (Fig. 14: latency vs sample
size) and its voxel-resolution study (Fig. 15).

    python -m paper_2606_06255_b200.sweep [--workloads C2,C3,C4,C5] [--reps 3]

prints one markdown table per study: `fps_sample` time (CUDA events, best of `reps`) for
M = N/64 .. N/2 at the automatic n_vox, and for n_vox = 8 .. 256 at the config's M, for the batched
kernel and the per-pick kernel.  Results never depend on either parameter (tests/test_gpu_parity.py);
only the time does.  Needs a CUDA device; there is no CPU fallback.
"""
from __future__ import annotations

import argparse

import numpy as np
import torch

from . import binding as rf
from . import inputs


def time_sample(Pd, M, start, reps, **opts):
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
    return best, st


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workloads", default="C2,C3,C4,C5")
    ap.add_argument("--reps", type=int, default=3)
    args = ap.parse_args()
    for name in args.workloads.split(","):
        w = inputs.WORKLOADS[name]
        Pd = torch.from_numpy(np.ascontiguousarray(inputs.make_batch(w))).cuda()
        print(f"\n### {name}: B={w.B} N={w.N} -- time of fps_sample vs sample size M (automatic n_vox)\n")
        print("| M | batched kernel ms | us per pick per cloud | per-pick kernel ms |")
        print("|---|---|---|---|")
        for div in (64, 32, 16, 8, 4, 2):
            M = w.N // div
            tb, _ = time_sample(Pd, M, w.start_idx, args.reps)
            tp, _ = time_sample(Pd, M, w.start_idx, 1, flags=rf.FPS_FLAG_PER_PICK) if M <= 70000 else (float("nan"), None)
            print(f"| N/{div} = {M} | {tb:.3f} | {tb * 1e3 / max(1, M - 1):.3f} | {tp:.3f} |", flush=True)
        print(f"\n### {name}: time of fps_sample (M={w.M}) vs voxel resolution n_vox\n")
        print("| n_vox | K_max (tiles of <= 64 points) | cluster | batched kernel ms | per-pick kernel ms |")
        print("|---|---|---|---|---|")
        for nv in (8, 16, 32, 64, 128, 256):
            try:
                tb, st = time_sample(Pd, w.M, w.start_idx, args.reps, n_vox=nv)
                try:
                    tp, _ = time_sample(Pd, w.M, w.start_idx, 1, n_vox=nv, flags=rf.FPS_FLAG_PER_PICK)
                except rf.FpsError:
                    tp = float("nan")
                print(f"| {nv} | {st['K_max']} | {st['cluster_size']} | {tb:.3f} | {tp:.3f} |", flush=True)
            except rf.FpsError as e:
                print(f"| {nv} | refused: {str(e)[:60]} | | | |", flush=True)


if __name__ == "__main__":
    main()
