"""GPU parity: the CUDA path (through the C-ABI) against the CPU oracle, element by element.

Bar (BASELINE.json north_star): indices with 0 mismatches, out_mindist with 0 ULP difference --
both are compared as raw bits.  Small cases span several voxels/tiles, ragged tails and the
degenerate inputs of the method; the five full-size configurations run in the launch configuration
bench.py times (library defaults) and are compared with the live oracle (C1-C4) and with the
stored oracle hashes of tests/golden/full_size.json (all five; written by
tests/golden/make_golden.py from the oracle alone).
"""
import hashlib
import json
import os

import numpy as np
import pytest
import torch

import oracle
from paper_2606_06255_b200 import inputs

pytestmark = pytest.mark.gpu
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "full_size.json")


@pytest.fixture(scope="module")
def rf():
    from paper_2606_06255_b200 import binding
    binding.load()            # raises if the CUDA library is missing: no fallback
    assert torch.cuda.is_available()
    return binding


def run_gpu(rf, P, M, start=0, **opts):
    Pd = torch.from_numpy(np.ascontiguousarray(P)).cuda()
    ix = rf.fps_index_build(Pd, **opts)
    try:
        idx, mind = rf.fps_sample(ix, M, start)
        torch.cuda.synchronize()
        st = rf.fps_get_stats(ix)
    finally:
        rf.fps_index_destroy(ix)
    return idx.cpu().numpy(), mind.cpu().numpy(), st


def sha(a):
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()


def assert_same(got_idx, got_mind, ref_idx, ref_mind):
    got_idx = got_idx.reshape(ref_idx.shape)
    got_mind = got_mind.reshape(ref_mind.shape)
    bad = np.nonzero((got_idx != ref_idx).reshape(-1))[0]
    assert bad.size == 0, f"{bad.size} index mismatches, first at flat position {bad[0]}"
    badm = np.nonzero((got_mind.view(np.uint32) != ref_mind.view(np.uint32)).reshape(-1))[0]
    assert badm.size == 0, f"{badm.size} min-distance bit mismatches, first at {badm[0]}"


SMALL = {
    "uniform4096": lambda: (inputs.uniform_cube(4096, 1234), 1024),
    "room": lambda: (inputs.room(6000, 11), 1500),
    "room_dense": lambda: (inputs.room(5000, 12, size=(20.0, 15.0, 3.0), n_boxes=60, dense_half=True), 1250),
    "lidar": lambda: (inputs.lidar(6000, 13, n_azimuth=94), 1500),
    "clustered": lambda: (inputs.clustered(5000, 14), 1250),
    "lattice": lambda: (inputs.shuffled_lattice(16, 15), 1024),
    "dups": lambda: (inputs.with_duplicates(3000, 16, 700), 1000),
    "line": lambda: (inputs.integer_line(513), 513),
    "ragged_tail": lambda: (inputs.uniform_cube(4099, 5), 1031),
}


# the two sampling kernels: exact batched picking (default) and the per-pick persistent kernel
KERNELS = {"batched": 0, "per_pick": 16}


@pytest.mark.parametrize("kernel", sorted(KERNELS))
@pytest.mark.parametrize("name", sorted(SMALL))
def test_small_clouds_default_config(rf, name, kernel):
    P, M = SMALL[name]()
    ref = oracle.fps(P, M, 0)
    gi, gm, _ = run_gpu(rf, P, M, flags=KERNELS[kernel])
    assert_same(gi, gm, *ref)


@pytest.mark.parametrize("kernel", sorted(KERNELS))
@pytest.mark.parametrize("cluster", [1, 2, 3, 4, 6, 7, 8, 13, 16])
@pytest.mark.parametrize("name", ["room", "lattice", "lidar"])
def test_every_cluster_size(rf, name, cluster, kernel):
    if kernel == "per_pick" and cluster not in (1, 2, 4, 8, 16):
        pytest.skip("the per-pick kernel takes power-of-two clusters")
    P, M = SMALL[name]()
    ref = oracle.fps(P, M, 0)
    gi, gm, st = run_gpu(rf, P, M, cluster_size=cluster, flags=KERNELS[kernel])
    assert st["cluster_size"] == cluster
    assert_same(gi, gm, *ref)


@pytest.mark.parametrize("ctas", [2, 3, 5, 9, 40, 148])
@pytest.mark.parametrize("name", ["room", "lattice", "lidar", "dups"])
def test_grid_mode_ctas_per_cloud(rf, name, ctas):
    # one picker CTA + (ctas - 1) worker CTAs per cloud spread over the grid (cooperative launch), exchanging picks,
    # commands and candidates through global memory with release / acquire at gpu scope
    P, M = SMALL[name]()
    ref = oracle.fps(P, M, 0)
    gi, gm, st = run_gpu(rf, P, M, cluster_size=-ctas)
    assert st["grid_ctas"] == ctas
    assert_same(gi, gm, *ref)


def test_grid_mode_batch_and_repeat_calls(rf):
    w = inputs.scaled("C2", 4000, 1000, B=16)
    P = inputs.make_batch(w)
    ref = oracle.fps(P, w.M, 0)
    Pd = torch.from_numpy(P).cuda()
    ix = rf.fps_index_build(Pd, cluster_size=-9)
    try:
        for _ in range(10):
            idx, mind = rf.fps_sample(ix, w.M, 0)
            torch.cuda.synchronize()
            assert_same(idx.cpu().numpy(), mind.cpu().numpy(), *ref)
    finally:
        rf.fps_index_destroy(ix)
    with pytest.raises(rf.FpsError):                        # 16 clouds x 10 CTAs cannot be resident on 148 SMs
        rf.fps_index_build(Pd, cluster_size=-10)


@pytest.mark.parametrize("name,ctas", [("C2", 9), ("C3", 100), ("C4", 37), ("C5", 148)])
def test_grid_mode_full_size(rf, name, ctas):
    gold = json.load(open(GOLDEN))[name]
    w = inputs.WORKLOADS[name]
    P = inputs.make_batch(w)
    gi, gm, st = run_gpu(rf, P, w.M, w.start_idx, cluster_size=-ctas)
    assert st["grid_ctas"] == ctas
    assert sha(gi.astype(np.int32)) == gold["idx_sha256"]
    assert sha(gm.astype(np.float32)) == gold["mindist_sha256"]


LOCAL_SHAPES = [(32, 2), (32, 4), (32, 8), (16, 2), (16, 4), (16, 8), (4, 8), (1, 8), (8, 16)]


@pytest.mark.parametrize("lw,cpt", LOCAL_SHAPES)
@pytest.mark.parametrize("name", ["room", "lattice", "dups", "clustered", "line"])
def test_every_local_phase_shape(rf, name, lw, cpt):
    # local_warps = 32: parallel resolution (default); 16: hierarchical (one sequential pick warp); 1..8: flat.
    # Candidate capacity from 256 to 4096: different thresholds, batches and tie paths (lattice / line: exact
    # ties inside a lane, between lanes and between warps, first histogram bin overflowing; dups: Dist reaches +0)
    P, M = SMALL[name]()
    ref = oracle.fps(P, M, 0)
    gi, gm, st = run_gpu(rf, P, M, local_warps=lw, cand_per_thread=cpt, flags=rf.FPS_FLAG_STATS)
    assert (st["local_warps"], st["cand_per_thread"]) == (lw, cpt)
    assert_same(gi, gm, *ref)
    assert st["rounds"] >= 1 and st["rounds"] <= M
    if name == "room":
        assert st["rounds"] < M // 8            # batching really happens on ordinary data
        if lw >= 16:
            assert 0 < st["local_subrounds"] < M // 4 and st["local_fallbacks"] < st["local_subrounds"]
    if name == "lattice" and lw >= 16:
        assert st["local_fallbacks"] > 0        # many exactly equal distances: the block-wide argmax path ran


def test_batched_kernel_degenerates_to_per_pick_rounds_without_batching(rf):
    P, M = SMALL["room"]()
    ref = oracle.fps(P, M, 0)
    gi, gm, st = run_gpu(rf, P, M, flags=rf.FPS_FLAG_NO_BATCH | rf.FPS_FLAG_STATS)
    assert_same(gi, gm, *ref)
    assert st["rounds"] == M - 1 and st["single_picks"] == M - 1 and st["candidates"] == 0


@pytest.mark.parametrize("n_vox", [1, 2, 7, 16, 24, 64, 128])
@pytest.mark.parametrize("name", ["room", "lattice", "clustered"])
def test_result_independent_of_n_vox(rf, name, n_vox):
    # PAPER.md:695 "largely insensitive" is about speed; the RESULT must be identical for every n_vox
    P, M = SMALL[name]()
    ref = oracle.fps(P, M, 0)
    gi, gm, st = run_gpu(rf, P, M, n_vox=n_vox)
    assert st["n_vox"] == n_vox
    assert_same(gi, gm, *ref)


@pytest.mark.parametrize("tile", [-1, 8, 32, 200])
@pytest.mark.parametrize("name", ["lidar", "clustered", "dups"])
def test_result_independent_of_tiling(rf, name, tile):
    P, M = SMALL[name]()
    ref = oracle.fps(P, M, 0)
    gi, gm, st = run_gpu(rf, P, M, tile_points=tile, n_vox=8)
    if tile > 0:
        assert st["max_voxel_points"] <= tile
    assert_same(gi, gm, *ref)


@pytest.mark.parametrize("name", sorted(SMALL))
def test_single_launch_build_equals_the_kernel_chain(rf, name):
    # clouds of <= 8 192 points are indexed by ONE kernel launch (one CTA per cloud); FPS_FLAG_CHAIN_BUILD forces the
    # chain of ~22 kernels that large clouds take: same voxels, same tiles, same samples
    P, M = SMALL[name]()
    ref = oracle.fps(P, M, 0)
    a = run_gpu(rf, P, M, n_vox=8)
    b = run_gpu(rf, P, M, n_vox=8, flags=rf.FPS_FLAG_CHAIN_BUILD)
    assert a[2]["build_launches"] == 1 and b[2]["build_launches"] > 10
    for key in ("K_total", "K_max", "max_voxel_points", "n_vox"):
        assert a[2][key] == b[2][key], key
    assert_same(a[0], a[1], *ref)
    assert_same(b[0], b[1], *ref)


@pytest.mark.parametrize("gen,B,N", [("room", 3, 24000), ("cube", 2, 8193), ("lidar", 2, 32768), ("clustered", 1, 20011),
                                     ("room", 1, 65536), ("lidar", 2, 120000)])
def test_cluster_build_equals_the_kernel_chain(rf, gen, B, N):
    # clouds of 8 193 .. ~130 000 points (one cloud: .. 65 536): one launch, one thread-block cluster of 2-16 CTAs per
    # cloud, radix passes over distributed shared memory; same voxels, tiles and samples as the chain
    mk = {"room": inputs.room, "cube": inputs.uniform_cube, "clustered": inputs.clustered,
          "lidar": lambda n, s: inputs.lidar(n, s, n_azimuth=512)}[gen]
    P = np.stack([mk(N, 900 + b) for b in range(B)])
    M = 257
    ref = oracle.fps(P, M, 5)
    a = run_gpu(rf, P, M, 5, flags=rf.FPS_FLAG_STATS)
    b = run_gpu(rf, P, M, 5, flags=rf.FPS_FLAG_STATS | rf.FPS_FLAG_CHAIN_BUILD)
    assert a[2]["build_launches"] == 1 and b[2]["build_launches"] > 10
    for key in ("K_total", "K_max", "max_voxel_points", "n_vox", "voxel_tests", "voxels_visited", "points_visited", "effective"):
        assert a[2][key] == b[2][key], key
    assert_same(a[0], a[1], *ref)
    assert_same(b[0], b[1], *ref)


def test_cluster_build_ragged_batch_and_bad_input(rf):
    clouds = [inputs.room(20000, 31), inputs.uniform_cube(7, 32), inputs.lidar(9001, 33, n_azimuth=140), inputs.uniform_cube(1, 34),
              inputs.clustered(30000, 35)]
    Ms = [300, 7, 400, 1, 350]
    off = np.concatenate([[0], np.cumsum([c.shape[0] for c in clouds])]).astype(np.int64)
    P = torch.from_numpy(np.ascontiguousarray(np.concatenate(clouds, axis=0))).cuda()
    ix = rf.fps_index_build_ragged(P, off.tolist())
    try:
        assert rf.fps_get_stats(ix)["build_launches"] == 1
        idx, mind, ooff = rf.fps_sample_ragged(ix, Ms)
        torch.cuda.synchronize()
        idx, mind = idx.cpu().numpy(), mind.cpu().numpy()
        for b, c in enumerate(clouds):
            ref_i, ref_m = oracle.fps(c, Ms[b], 0)
            assert_same(idx[ooff[b]:ooff[b + 1]], mind[ooff[b]:ooff[b + 1]], ref_i.reshape(-1), ref_m.reshape(-1))
    finally:
        rf.fps_index_destroy(ix)
    bad = inputs.room(12000, 36).copy()
    bad[11999, 1] = np.nan
    with pytest.raises(rf.FpsError) as e:
        rf.fps_index_build(torch.from_numpy(bad).cuda())
    assert e.value.status == rf.FPS_ERR_NONFINITE


def test_single_launch_build_ragged_batch(rf):
    clouds = [inputs.room(5000, 21), inputs.uniform_cube(1, 22), inputs.lidar(7001, 23, n_azimuth=110),
              inputs.shuffled_lattice(8, 24), inputs.uniform_cube(33, 25), inputs.clustered(2500, 26)]
    Ms = [1250, 1, 1800, 512, 33, 600]
    off = np.concatenate([[0], np.cumsum([c.shape[0] for c in clouds])]).astype(np.int64)
    P = torch.from_numpy(np.ascontiguousarray(np.concatenate(clouds, axis=0))).cuda()
    for flags in (0, rf.FPS_FLAG_CHAIN_BUILD):
        ix = rf.fps_index_build_ragged(P, off.tolist(), flags=flags)
        try:
            idx, mind, ooff = rf.fps_sample_ragged(ix, Ms)
            torch.cuda.synchronize()
            idx, mind = idx.cpu().numpy(), mind.cpu().numpy()
            for b, c in enumerate(clouds):
                ref_i, ref_m = oracle.fps(c, Ms[b], 0)
                assert_same(idx[ooff[b]:ooff[b + 1]], mind[ooff[b]:ooff[b + 1]], ref_i.reshape(-1), ref_m.reshape(-1))
        finally:
            rf.fps_index_destroy(ix)


@pytest.mark.parametrize("threads", [64, 128, 256, 1024])
def test_block_sizes(rf, threads):
    P, M = SMALL["room"]()
    ref = oracle.fps(P, M, 0)
    gi, gm, st = run_gpu(rf, P, M, block_threads=threads, cluster_size=2, flags=rf.FPS_FLAG_PER_PICK)
    assert st["block_threads"] == threads
    assert_same(gi, gm, *ref)


@pytest.mark.parametrize("kernel", sorted(KERNELS))
@pytest.mark.parametrize("flags", [1, 2, 3, 4, 7])
def test_ablations_and_stats_are_bit_identical(rf, flags, kernel):
    # Table 4 structure: prune off / skip off / both off must not change a bit
    # (cluster_size = 2: the general batched kernel; by default a cloud of this size runs the small-cloud kernel, whose
    # flags and counters test_whole_cloud_kernel_flags covers)
    P, M = SMALL["room"]()
    ref = oracle.fps(P, M, 0)
    gi, gm, st = run_gpu(rf, P, M, flags=flags | KERNELS[kernel], cluster_size=2)
    assert_same(gi, gm, *ref)
    assert st["whole_cloud_kernel"] == 0
    if flags & rf.FPS_FLAG_STATS:
        assert st["iterations"] == M - 1
        if kernel == "per_pick":
            applied = M - 1                                      # every voxel is tested against every pick
            assert st["voxel_tests"] == st["K_total"] * applied
        else:
            # the picks of the last batch need not be applied (nothing needs them): a worker CTA that sees the end of
            # the sampling stops, so the CTAs may have applied different prefixes of that batch; the prune runs on
            # groups of 32 voxels first, voxels are only tested where their group survived
            if flags & rf.FPS_FLAG_NO_PRUNE:
                applied = st["voxel_tests"] / st["K_total"]
                assert st["group_tests"] == 0
            else:
                G = (st["K_total"] + 31) // 32
                applied = st["group_tests"] / G
                assert 0 < st["voxel_tests"] < st["K_total"] * applied
            assert M - 1 - 1024 <= applied <= M - 1
        if flags & rf.FPS_FLAG_NO_PRUNE:
            if kernel == "per_pick":
                assert st["voxels_visited"] == st["K_total"] * applied
            assert abs(st["points_visited"] - P.shape[0] * applied) <= 0.02 * st["points_visited"]
        if flags & rf.FPS_FLAG_NO_SKIP:
            assert st["points_computed"] == st["points_visited"]


def test_stats_match_cpu_pruned_variant_effective_updates(rf):
    # the number of EFFECTIVE updates (Eq. 2) is a property of the data, not of the index
    P, M = SMALL["room"]()
    _, _, cpu = oracle.pruned_fps(P, M, 0, n_vox=16)
    for kernel, kflag in KERNELS.items():
        _, _, st = run_gpu(rf, P, M, flags=rf.FPS_FLAG_STATS | kflag, cluster_size=2)
        assert st["whole_cloud_kernel"] == 0
        if kernel == "per_pick":
            assert st["effective"] == cpu["effective"]
        else:                       # the picks of the last batch are never applied (nothing needs them)
            assert 0.8 * cpu["effective"] <= st["effective"] <= cpu["effective"]
        assert st["points_visited"] < 0.2 * P.shape[0] * (M - 1)
    # the small-cloud kernel (the default for this size) applies every pick to every point it can still lower
    _, _, st = run_gpu(rf, P, M, flags=rf.FPS_FLAG_STATS)
    assert st["whole_cloud_kernel"] == 1
    assert 0.98 * cpu["effective"] <= st["effective"] <= cpu["effective"] + P.shape[0]      # (+ the last pick's updates)
    assert st["points_visited"] < 0.35 * P.shape[0] * (M - 1)


@pytest.mark.parametrize("kernel", sorted(KERNELS))
@pytest.mark.parametrize("N,M,start", [(1, 1, 0), (2, 2, 1), (3, 1, 2), (33, 33, 32), (64, 64, 7), (1000, 1000, 999)])
def test_degenerate_sizes_and_starts(rf, N, M, start, kernel):
    P = inputs.uniform_cube(N, 3)
    ref = oracle.fps(P, M, start)
    gi, gm, _ = run_gpu(rf, P, M, start, flags=KERNELS[kernel])
    assert_same(gi, gm, *ref)


@pytest.mark.parametrize("kernel", sorted(KERNELS))
def test_identical_points(rf, kernel):
    P = np.full((100, 3), 0.25, dtype=np.float32)
    ref = oracle.fps(P, 10, 3)
    gi, gm, _ = run_gpu(rf, P, 10, 3, flags=KERNELS[kernel])
    assert_same(gi, gm, *ref)
    assert gi.reshape(-1).tolist() == [3] + [0] * 9


@pytest.mark.parametrize("kernel", sorted(KERNELS))
def test_closed_form_line_and_corners(rf, kernel):
    gi, gm, _ = run_gpu(rf, inputs.integer_line(9), 9, flags=KERNELS[kernel])
    assert gi.reshape(-1).tolist() == [0, 8, 4, 2, 6, 1, 3, 5, 7]
    assert gm.reshape(-1).tolist() == [np.inf, 64, 16, 4, 4, 1, 1, 1, 1]
    gi, gm, _ = run_gpu(rf, inputs.cube_corners(), 8, flags=KERNELS[kernel])
    assert gi.reshape(-1).tolist() == [0, 7, 1, 2, 3, 4, 5, 6]


def test_large_coordinates_and_tiny_extent(rf):
    base = inputs.uniform_cube(3000, 8)
    for P in ((base * np.float32(1e6)).astype(np.float32), (base * np.float32(1e-6)).astype(np.float32),
              (base + np.float32(1000.0)).astype(np.float32)):
        ref = oracle.fps(P, 600, 0)
        gi, gm, _ = run_gpu(rf, P, 600)
        assert_same(gi, gm, *ref)


def test_batch_of_clouds_and_repeat_calls(rf):
    w = inputs.scaled("C2", 3000, 700, B=5)
    P = inputs.make_batch(w)
    ref = oracle.fps(P, w.M, 0)
    Pd = torch.from_numpy(P).cuda()
    ix = rf.fps_index_build(Pd)
    try:
        for _ in range(2):                                   # a handle is reusable: state resets per call
            idx, mind = rf.fps_sample(ix, w.M, 0)
            torch.cuda.synchronize()
            assert_same(idx.cpu().numpy(), mind.cpu().numpy(), *ref)
        idx, mind = rf.fps_sample(ix, 100, 17)               # other M / start on the same handle
        torch.cuda.synchronize()
        assert_same(idx.cpu().numpy(), mind.cpu().numpy(), *oracle.fps(P, 100, 17))
    finally:
        rf.fps_index_destroy(ix)


@pytest.mark.parametrize("kernel", sorted(KERNELS))
def test_ragged_batch_matches_the_oracle_cloud_by_cloud(rf, kernel):
    # clouds of different sizes, per-cloud M and start point, one index, one launch
    clouds = [inputs.room(5000, 21), inputs.uniform_cube(1, 22), inputs.lidar(7001, 23, n_azimuth=110),
              inputs.shuffled_lattice(8, 24), inputs.uniform_cube(33, 25), inputs.clustered(2500, 26),
              inputs.with_duplicates(900, 27, 200), inputs.uniform_cube(4099, 28)]
    Ms = [1250, 1, 1800, 512, 33, 600, 450, 1031]
    starts = [0, 0, 7000, 5, 32, 17, 899, 4098]
    off = np.concatenate([[0], np.cumsum([c.shape[0] for c in clouds])]).astype(np.int64)
    P = torch.from_numpy(np.ascontiguousarray(np.concatenate(clouds, axis=0))).cuda()
    ix = rf.fps_index_build_ragged(P, off.tolist(), flags=KERNELS[kernel])
    try:
        for ms, ss in ((Ms, starts), ([min(m, 7) for m in Ms], None)):       # the handle is reusable
            idx, mind, ooff = rf.fps_sample_ragged(ix, ms, ss)
            torch.cuda.synchronize()
            idx, mind = idx.cpu().numpy(), mind.cpu().numpy()
            for b, c in enumerate(clouds):
                ref_i, ref_m = oracle.fps(c, ms[b], ss[b] if ss else 0)
                assert_same(idx[ooff[b]:ooff[b + 1]], mind[ooff[b]:ooff[b + 1]], ref_i.reshape(-1), ref_m.reshape(-1))
        # one M / one start for all clouds also works on a ragged index when they fit ...
        idx, mind = rf.fps_sample(ix, 1, 0)
        torch.cuda.synchronize()
        assert idx.cpu().numpy().reshape(-1).tolist() == [0] * len(clouds)
        # ... and is refused when they do not (cloud 1 holds a single point)
        with pytest.raises(rf.FpsError) as e:
            rf.fps_sample(ix, 2, 0)
        assert e.value.status == rf.FPS_ERR_INVALID
        with pytest.raises(rf.FpsError):
            rf.fps_sample_ragged(ix, [m + 100000 for m in Ms])
    finally:
        rf.fps_index_destroy(ix)


def test_ragged_index_of_equal_clouds_equals_the_uniform_one(rf):
    w = inputs.scaled("C2", 3000, 700, B=4)
    P = inputs.make_batch(w)
    ref = oracle.fps(P, w.M, 0)
    Pd = torch.from_numpy(P.reshape(-1, 3)).cuda()
    ix = rf.fps_index_build_ragged(Pd, [b * w.N for b in range(w.B + 1)])
    try:
        idx, mind, _ = rf.fps_sample_ragged(ix, [w.M] * w.B)
        torch.cuda.synchronize()
        assert_same(idx.cpu().numpy(), mind.cpu().numpy(), *ref)
    finally:
        rf.fps_index_destroy(ix)


@pytest.mark.parametrize("chunk", [0, 1, 3, 8, 100])
def test_one_shot_ragged_chunks_match_the_oracle(rf, chunk):
    # SURVEY 8(f) NEXT-2, second half: build + sample + release in one call, the batch cut into chunks whose
    # index builds overlap the sampling of the chunk before; the chunking must never change a result
    clouds = [inputs.room(5000, 21), inputs.uniform_cube(1, 22), inputs.lidar(7001, 23, n_azimuth=110),
              inputs.shuffled_lattice(8, 24), inputs.uniform_cube(33, 25), inputs.clustered(2500, 26),
              inputs.with_duplicates(900, 27, 200), inputs.uniform_cube(4099, 28)]
    Ms = [1250, 1, 1800, 512, 33, 600, 450, 1031]
    starts = [0, 0, 7000, 5, 32, 17, 899, 4098]
    off = np.concatenate([[0], np.cumsum([c.shape[0] for c in clouds])]).astype(np.int64)
    P = torch.from_numpy(np.ascontiguousarray(np.concatenate(clouds, axis=0))).cuda()
    for ms, ss in ((Ms, starts), (Ms, None)):
        idx, mind, ooff = rf.fps_build_and_sample(P, ms, offsets=off.tolist(), start_idx=ss, chunk_clouds=chunk)
        torch.cuda.synchronize()
        idx, mind = idx.cpu().numpy(), mind.cpu().numpy()
        for b, c in enumerate(clouds):
            ref_i, ref_m = oracle.fps(c, ms[b], ss[b] if ss else 0)
            assert_same(idx[ooff[b]:ooff[b + 1]], mind[ooff[b]:ooff[b + 1]], ref_i.reshape(-1), ref_m.reshape(-1))
    with pytest.raises(rf.FpsError) as e:                    # cloud 1 holds one point: M = 2 cannot fit
        rf.fps_build_and_sample(P, 2, offsets=off.tolist(), chunk_clouds=chunk)
    assert e.value.status == rf.FPS_ERR_INVALID


@pytest.mark.parametrize("chunk", [0, 5, 16])
def test_one_shot_uniform_batch_pipelined_on_a_side_stream(rf, chunk):
    # 40 clouds in one chunk, eight chunks of 5 and chunks of 16 + 16 + 8, inputs produced on a side stream right before the call: the internal
    # build stream must wait for them, and the results must be ordered on that same stream
    w = inputs.scaled("C2", 3000, 700, B=40)
    P = inputs.make_batch(w)
    ref = oracle.fps(P, w.M, 0)
    Ph = torch.from_numpy(P).pin_memory()
    side = torch.cuda.Stream()
    for _ in range(3):
        with torch.cuda.stream(side):
            Pd = torch.empty_like(Ph, device="cuda")
            Pd.copy_(Ph, non_blocking=True)
            idx, mind = rf.fps_build_and_sample(Pd, w.M, chunk_clouds=chunk, stream=side)
            hi = idx.to("cpu", non_blocking=True)
            hm = mind.to("cpu", non_blocking=True)
        side.synchronize()
        assert_same(hi.numpy(), hm.numpy(), *ref)


def test_one_shot_rejects_bad_arguments(rf):
    P = torch.from_numpy(inputs.uniform_cube(100, 1)).cuda()
    for kw in (dict(M=0), dict(M=101), dict(M=5, chunk_clouds=-1), dict(M=[5, 5]), dict(M=5, start_idx=[100])):
        with pytest.raises((rf.FpsError, ValueError)):
            rf.fps_build_and_sample(P, kw.pop("M"), **kw)
    bad = P.clone()
    bad[7, 1] = float("nan")
    with pytest.raises(rf.FpsError) as e:
        rf.fps_build_and_sample(bad, 5)
    assert e.value.status == rf.FPS_ERR_NONFINITE


@pytest.mark.parametrize("cluster", [0, 2, 5])
def test_repeated_launches_under_load_are_identical(rf, cluster):
    # the batched kernel passes data between CTAs with release/acquire flags, DSMEM atomics and dynamic work
    # queues; compute-sanitizer is not available on the GPU pool, so races are hunted by repetition: 16
    # clouds in flight, 25 launches, every one must equal the oracle bit for bit
    w = inputs.scaled("C2", 4000, 1000, B=16)
    P = inputs.make_batch(w)
    ref = oracle.fps(P, w.M, 0)
    Pd = torch.from_numpy(P).cuda()
    ix = rf.fps_index_build(Pd, cluster_size=cluster)
    try:
        for _ in range(25):
            idx, mind = rf.fps_sample(ix, w.M, 0)
            torch.cuda.synchronize()
            assert_same(idx.cpu().numpy(), mind.cpu().numpy(), *ref)
    finally:
        rf.fps_index_destroy(ix)


@pytest.mark.parametrize("B,N,M,gen", [(100, 2048, 512, "cube"), (300, 1500, 300, "room")])
def test_many_clouds_more_than_resident_clusters(rf, B, N, M, gen):
    # B = 300 exceeds the clusters that can be resident at once: the clouds run in waves
    P = np.stack([(inputs.uniform_cube(N, 100 + b) if gen == "cube" else inputs.room(N, 500 + b)) for b in range(B)])
    ref = oracle.fps(P, M, 0)
    gi, gm, _ = run_gpu(rf, P, M)
    assert_same(gi, gm, *ref)


def test_sampling_every_point_of_a_cloud(rf):
    P = inputs.room(5000, 7)
    ref = oracle.fps(P, 5000, 3)
    for kflag in KERNELS.values():
        gi, gm, _ = run_gpu(rf, P, 5000, 3, flags=kflag)
        assert_same(gi, gm, *ref)
        assert sorted(gi.reshape(-1).tolist()) == list(range(5000))


def test_three_million_points_tile_size_grows(rf):
    """Beyond ~1.5 M points the automatic tile size grows so that the voxel state still fits the workers'
    shared memory.  Element by element against the oracle through the stored hashes of its outputs
    (tests/golden/full_size.json "L3M", written by make_golden.py from oracle/fps_oracle.c alone; 60 G point
    updates, minutes on one core), plus properties that hold at any size."""
    gold = json.load(open(GOLDEN))["L3M"]
    w = inputs.EXTRA_WORKLOADS["L3M"]
    P = inputs.make_batch(w)
    assert sha(P) == gold["input_sha256"], "input generator drifted from the one the golden was made with"
    gi, gm, st = run_gpu(rf, P, w.M)
    assert st["max_voxel_points"] > 64 and (st["cluster_size"] == 16 or st["grid_ctas"] > 16)
    gi, gm, P = gi.reshape(-1), gm.reshape(-1), P[0]
    assert gi[0] == 0 and np.isinf(gm[0]) and np.all(gm[1:] <= gm[:-1]) and np.unique(gi).size == w.M
    assert gi[:8].tolist() == gold["idx_head"]
    assert sha(gi.astype(np.int32)) == gold["idx_sha256"]
    assert sha(gm.astype(np.float32)) == gold["mindist_sha256"]


def test_gather_xyz_uniform_and_ragged(rf):
    w = inputs.scaled("C2", 3000, 700, B=3)
    P = inputs.make_batch(w)
    ix = rf.fps_index_build(torch.from_numpy(P).cuda())
    try:
        idx, _ = rf.fps_sample(ix, w.M, 0)
        xyz = rf.fps_gather_xyz(ix, idx)
        torch.cuda.synchronize()
        gi = idx.cpu().numpy()
        assert np.array_equal(xyz.cpu().numpy(), np.stack([P[b][gi[b]] for b in range(w.B)]))
    finally:
        rf.fps_index_destroy(ix)
    clouds = [inputs.room(2000, 31), inputs.uniform_cube(17, 32), inputs.lidar(3001, 33, n_azimuth=60)]
    off = np.concatenate([[0], np.cumsum([c.shape[0] for c in clouds])])
    ix = rf.fps_index_build_ragged(torch.from_numpy(np.concatenate(clouds)).cuda(), off.tolist())
    try:
        idx, _, ooff = rf.fps_sample_ragged(ix, [500, 17, 64], [3, 16, 0])
        xyz = rf.fps_gather_xyz(ix, idx, 0)
        torch.cuda.synchronize()
        gi, gx = idx.cpu().numpy(), xyz.cpu().numpy()
        for b, c in enumerate(clouds):
            assert np.array_equal(gx[ooff[b]:ooff[b + 1]], c[gi[ooff[b]:ooff[b + 1]]])
    finally:
        rf.fps_index_destroy(ix)


def test_pick_chain_floor_is_measurable(rf):
    c1, c4 = rf.fps_pick_chain_cycles(1, 4096), rf.fps_pick_chain_cycles(4, 4096)
    assert 40.0 < c1 < 1000.0 and c1 < c4 < 2000.0


# ---------------------------------------------------------------------------------------------
# Euclidean mode: the paper's literal distance, against its own oracle
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cluster", [0, 1, 5])
@pytest.mark.parametrize("name", sorted(SMALL))
def test_euclidean_mode_small_clouds(rf, name, cluster):
    P, M = SMALL[name]()
    ref = oracle.fps_euclid(P, M, 0)
    gi, gm, _ = run_gpu(rf, P, M, flags=rf.FPS_FLAG_EUCLIDEAN, cluster_size=cluster)
    assert_same(gi, gm, *ref)


@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C4"])
def test_euclidean_mode_full_size(rf, name):
    w = inputs.WORKLOADS[name]
    P = inputs.make_batch(w)
    ref = oracle.fps_euclid(P, w.M, w.start_idx)
    gi, gm, _ = run_gpu(rf, P, w.M, w.start_idx, flags=rf.FPS_FLAG_EUCLIDEAN)
    assert_same(gi, gm, *ref)


@pytest.mark.parametrize("name", ["C4", "C5"])
def test_euclidean_mode_full_size_against_stored_oracle_hashes(rf, name):
    # C5 is minutes of oracle time: its outputs' hashes are stored (make_golden.py --euclid, oracle.fps_euclid only)
    gold = json.load(open(GOLDEN))[name + ":euclid"]
    w = inputs.WORKLOADS[name]
    P = inputs.make_batch(w)
    assert sha(P) == gold["input_sha256"], "input generator drifted from the one the golden was made with"
    gi, gm, _ = run_gpu(rf, P, w.M, w.start_idx, flags=rf.FPS_FLAG_EUCLIDEAN)
    assert gi.reshape(w.B, w.M)[0, :8].tolist() == gold["idx_head"]
    assert sha(gi.astype(np.int32)) == gold["idx_sha256"]
    assert sha(gm.astype(np.float32)) == gold["mindist_sha256"]


def test_euclidean_mode_is_a_different_function_where_sqrt_collapses(rf):
    # two maxima one ulp apart in d2 with the same correctly rounded square root (found by search, as in
    # tests/test_oracle_pins.py): the squared mode takes the larger, the Euclidean mode ties -> lower index
    rng = np.random.default_rng(5)
    F = np.float32
    found = None
    for _ in range(200):
        Q = np.zeros((4000, 3), dtype=F)
        Q[:, :2] = rng.random((4000, 2), dtype=F) + F(0.5)
        d2 = ((Q[:, 0] * Q[:, 0]).astype(F) + (Q[:, 1] * Q[:, 1]).astype(F)).astype(F)
        order = np.argsort(d2, kind="stable")
        sd, r = d2[order], np.sqrt(d2[order]).astype(F)
        hit = np.nonzero((sd[1:] > sd[:-1]) & (r[1:] == r[:-1]))[0]
        if hit.size:
            found = (Q[order[hit[0]]], Q[order[hit[0] + 1]])
            break
    assert found is not None
    P = np.stack([np.zeros(3, dtype=F), found[0], found[1]])
    gi, _, _ = run_gpu(rf, P, 2)
    assert gi.reshape(-1).tolist() == [0, 2]
    gi, gm, _ = run_gpu(rf, P, 2, flags=rf.FPS_FLAG_EUCLIDEAN)
    assert gi.reshape(-1).tolist() == [0, 1]
    assert_same(gi, gm, *oracle.fps_euclid(P, 2, 0))


def test_euclidean_mode_refuses_the_per_pick_kernel(rf):
    P = torch.from_numpy(inputs.uniform_cube(100, 1)).cuda()
    with pytest.raises(rf.FpsError) as e:
        rf.fps_index_build(P, flags=rf.FPS_FLAG_EUCLIDEAN | rf.FPS_FLAG_PER_PICK)
    assert e.value.status == rf.FPS_ERR_INVALID
    with pytest.raises(rf.FpsError):
        rf.fps_index_build(P, flags=rf.FPS_FLAG_EUCLIDEAN, local_warps=4, cand_per_thread=8)


def test_integer_grid_overflowing_ties(rf):
    # an exact integer grid: thousands of points tie at the maximum, more than the candidate buffer holds, so
    # extraction attempts overflow, fall back to single global argmax picks, and the local phase takes its
    # block-wide tie-break path; all of it must still follow the oracle bit for bit
    g = np.arange(120, dtype=np.float32)
    P = np.stack(np.meshgrid(g, g, np.zeros(1, dtype=np.float32)), -1).reshape(-1, 3).astype(np.float32)
    P = np.ascontiguousarray(P[np.random.default_rng(3).permutation(P.shape[0])])
    ref = oracle.fps(P, 1500, 0)
    gi, gm, st = run_gpu(rf, P, 1500, flags=rf.FPS_FLAG_STATS)
    assert_same(gi, gm, *ref)
    assert st["extract_retries"] > 0 and st["single_picks"] > 0 and st["local_fallbacks"] > 0


# ---- the small-cloud kernel (k_fps_whole: every cloud <= 8 192 points, one CTA per cloud, the whole cloud in
# registers, radius prune on runs of 64 sorted points).  It is the default for such an index; an explicit
# cluster_size, local_warps = 16 / 8 / 4 / 1 or FPS_FLAG_NO_BATCH select the general kernel (tests above). ----

WHOLE_SIZES = [(1, 1, 0), (2, 2, 1), (63, 63, 5), (64, 20, 63), (65, 65, 64), (127, 40, 0), (129, 129, 128), (1023, 400, 7),
               (1024, 1024, 1023), (1025, 300, 0), (2047, 2047, 3), (2048, 512, 2047), (2049, 600, 11), (4095, 1024, 4094),
               (4096, 4096, 0), (4097, 1000, 4096), (6000, 1500, 17), (8191, 2000, 0), (8192, 8192, 8191)]


@pytest.mark.parametrize("N,M,start", WHOLE_SIZES)
def test_whole_cloud_kernel_sizes_around_blob_and_register_boundaries(rf, N, M, start):
    # 64 points per blob, 1 024 points per register position, 512 x {2, 4, 8, 16} capacity (with 16 most coordinates
    # live in shared memory); M up to N (beyond the 1 024 picks of the general kernel's batch buffer)
    P = inputs.uniform_cube(N, 1000 + N)
    ref = oracle.fps(P, M, start)
    gi, gm, st = run_gpu(rf, P, M, start)
    assert st["whole_cloud_kernel"] == 1 and st["cluster_size"] == 1
    assert st["cand_per_thread"] == (2 if N <= 1024 else 4 if N <= 2048 else 8 if N <= 4096 else 16)
    assert_same(gi, gm, *ref)


@pytest.mark.parametrize("name", ["uniform4096", "lattice", "dups", "line", "room", "lidar"])
@pytest.mark.parametrize("flags", [0, 1, 4, 5, 32, 36])
def test_whole_cloud_kernel_flags(rf, name, flags):
    # prune off (every pick applied to every blob), STATS build, Euclidean distances: same picks, bit for bit
    P, M = SMALL[name]()
    ref = oracle.fps_euclid(P, M, 0) if flags & rf.FPS_FLAG_EUCLIDEAN else oracle.fps(P, M, 0)
    gi, gm, st = run_gpu(rf, P, M, flags=flags)
    assert st["whole_cloud_kernel"] == 1
    assert_same(gi, gm, *ref)
    if flags & rf.FPS_FLAG_STATS:
        assert st["iterations"] == M - 1 and st["rounds"] == 1 and st["group_tests"] == 0
        assert st["voxel_tests"] > 0 and 0 < st["voxels_visited"] <= st["voxel_tests"]
        if flags & rf.FPS_FLAG_NO_PRUNE:
            assert st["voxels_visited"] * 2 > st["voxel_tests"]          # only blobs whose distances are all 0 are left out
        elif name == "uniform4096":
            assert st["voxels_visited"] * 4 < st["voxel_tests"]          # the prune does remove most (blob, pick) pairs


def test_whole_cloud_kernel_tie_heavy_inputs(rf):
    # exact ties everywhere: the first bin of the selection histogram overflows, the kernel falls back to runs of
    # single block-wide argmax picks with the lowest-index tie-break; duplicates run out of positive distances
    g = np.arange(64, dtype=np.float32)
    grid = np.stack(np.meshgrid(g, g, np.zeros(1, dtype=np.float32)), -1).reshape(-1, 3).astype(np.float32)
    grid = np.ascontiguousarray(grid[np.random.default_rng(5).permutation(grid.shape[0])])
    same = np.full((777, 3), -3.5, dtype=np.float32)
    few = inputs.with_duplicates(4000, 31, 50)
    for P, M, start in ((grid, 2000, 17), (same, 50, 776), (few, 300, 3999), (inputs.cube_corners(), 8, 0)):
        ref = oracle.fps(P, M, start)
        gi, gm, st = run_gpu(rf, P, M, start, flags=rf.FPS_FLAG_STATS)
        assert st["whole_cloud_kernel"] == 1
        assert_same(gi, gm, *ref)
    assert st["single_picks"] > 0


def test_whole_cloud_kernel_batches_uniform_and_ragged(rf):
    # more clouds than SMs; a ragged index with per-cloud M and start; repeat calls on one handle
    P = np.stack([inputs.uniform_cube(1500, 300 + b) if b % 2 else inputs.room(1500, 300 + b) for b in range(170)])
    ref = oracle.fps(P, 400, 3)
    Pd = torch.from_numpy(P).cuda()
    ix = rf.fps_index_build(Pd)
    try:
        assert rf.fps_get_stats(ix)["whole_cloud_kernel"] == 1
        for _ in range(2):
            idx, mind = rf.fps_sample(ix, 400, 3)
            torch.cuda.synchronize()
            assert_same(idx.cpu().numpy(), mind.cpu().numpy(), *ref)
    finally:
        rf.fps_index_destroy(ix)
    clouds = [inputs.room(4096, 41), inputs.uniform_cube(1, 42), inputs.lidar(3001, 43, n_azimuth=60), inputs.shuffled_lattice(8, 44),
              inputs.uniform_cube(33, 45), inputs.clustered(2500, 46), inputs.with_duplicates(900, 47, 200)]
    Ms = [4096, 1, 1800, 512, 33, 600, 450]
    starts = [0, 0, 3000, 5, 32, 17, 899]
    off = np.concatenate([[0], np.cumsum([c.shape[0] for c in clouds])]).astype(np.int64)
    Pr = torch.from_numpy(np.ascontiguousarray(np.concatenate(clouds, axis=0))).cuda()
    ix = rf.fps_index_build_ragged(Pr, off.tolist())
    try:
        assert rf.fps_get_stats(ix)["whole_cloud_kernel"] == 1
        for ms, ss in ((Ms, starts), ([min(m, 9) for m in Ms], None)):
            idx, mind, ooff = rf.fps_sample_ragged(ix, ms, ss)
            torch.cuda.synchronize()
            idx, mind = idx.cpu().numpy(), mind.cpu().numpy()
            for b, c in enumerate(clouds):
                ref_i, ref_m = oracle.fps(c, ms[b], ss[b] if ss else 0)
                assert_same(idx[ooff[b]:ooff[b + 1]], mind[ooff[b]:ooff[b + 1]], ref_i.reshape(-1), ref_m.reshape(-1))
    finally:
        rf.fps_index_destroy(ix)


def test_whole_cloud_kernel_overflowing_distances_and_scales(rf):
    # d2 overflows to +inf for the first picks (coordinates ~1e19..1e20): single picks until every distance is finite
    base = inputs.uniform_cube(2000, 51)
    big = (base * np.float32(2e19)).astype(np.float32)
    for P in (big, (base * np.float32(1e-12)).astype(np.float32), (base + np.float32(4096.0)).astype(np.float32)):
        ref = oracle.fps(P, 500, 0)
        gi, gm, st = run_gpu(rf, P, 500)
        assert st["whole_cloud_kernel"] == 1
        assert_same(gi, gm, *ref)
    assert np.isinf(oracle.fps(big, 3, 0)[1].reshape(-1)[1])       # the case does overflow


def test_small_clouds_general_kernel_still_selectable(rf):
    P, M = SMALL["uniform4096"]()
    ref = oracle.fps(P, M, 0)
    for opts in (dict(cluster_size=4), dict(local_warps=16), dict(flags=rf.FPS_FLAG_NO_BATCH), dict(cluster_size=1),
                 dict(cand_per_thread=2)):
        gi, gm, st = run_gpu(rf, P, M, **opts)
        assert st["whole_cloud_kernel"] == 0
        assert_same(gi, gm, *ref)


def test_host_entry_point(rf):
    w = inputs.scaled("C4", 4000, 900, B=2)
    P = inputs.make_batch(w)
    ref = oracle.fps(P, w.M, 0)
    idx, mind = rf.fps_sample_host(torch.from_numpy(P), w.M, 0)
    assert_same(idx.numpy(), mind.numpy(), *ref)


def test_errors(rf):
    P = torch.from_numpy(inputs.uniform_cube(100, 1)).cuda()
    ix = rf.fps_index_build(P)
    for M, start in [(0, 0), (101, 0), (10, -1), (10, 100)]:
        with pytest.raises(rf.FpsError) as e:
            rf.fps_sample(ix, M, start)
        assert e.value.status == rf.FPS_ERR_INVALID
    rf.fps_index_destroy(ix)
    bad = P.clone()
    bad[5, 1] = float("nan")
    with pytest.raises(rf.FpsError) as e:
        rf.fps_index_build(bad)
    assert e.value.status == rf.FPS_ERR_NONFINITE
    with pytest.raises(rf.FpsError):
        rf.fps_index_build(P, cluster_size=17)
    with pytest.raises(rf.FpsError):
        rf.fps_index_build(P, cluster_size=3, flags=rf.FPS_FLAG_PER_PICK)


# ---------------------------------------------------------------------------------------------
# full-size configurations, library-default launch configuration (= what bench.py times)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C4"])
def test_full_size_against_live_oracle(rf, name):
    w = inputs.WORKLOADS[name]
    P = inputs.make_batch(w)
    ref = oracle.fps(P, w.M, w.start_idx)
    gi, gm, _ = run_gpu(rf, P, w.M, w.start_idx)
    assert_same(gi, gm, *ref)
    gi, gm, _ = run_gpu(rf, P, w.M, w.start_idx, flags=rf.FPS_FLAG_PER_PICK)
    assert_same(gi, gm, *ref)


@pytest.mark.parametrize("kernel", sorted(KERNELS))
@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C4", "C5"])
def test_full_size_against_stored_oracle_hashes(rf, name, kernel):
    gold = json.load(open(GOLDEN))[name]
    w = inputs.WORKLOADS[name]
    P = inputs.make_batch(w)
    assert sha(P) == gold["input_sha256"], "input generator drifted from the one the golden was made with"
    gi, gm, _ = run_gpu(rf, P, w.M, w.start_idx, flags=KERNELS[kernel])
    assert gi.reshape(w.B, w.M)[0, :8].tolist() == gold["idx_head"]
    assert sha(gi.astype(np.int32)) == gold["idx_sha256"]
    assert sha(gm.astype(np.float32)) == gold["mindist_sha256"]


def test_C5_properties_and_sampled_recomputation(rf):
    """N = 10^6: properties that hold at any size + min-distances recomputed for sampled outputs."""
    w = inputs.WORKLOADS["C5"]
    P = inputs.make_batch(w)
    gi, gm, _ = run_gpu(rf, P, w.M, w.start_idx)
    gi, gm, P = gi.reshape(-1), gm.reshape(-1), P[0]
    assert gi[0] == w.start_idx and np.isinf(gm[0])
    assert np.all(gm[1:] <= gm[:-1])
    assert np.unique(gi).size == w.M
    S = P[gi]
    rng = np.random.default_rng(0)
    for j in [1, 2, 3, w.M - 1] + rng.integers(4, w.M, size=60).tolist():
        d = (S[:j] - S[j]).astype(np.float32)
        d2 = ((d[:, 0] * d[:, 0] + d[:, 1] * d[:, 1]).astype(np.float32) + d[:, 2] * d[:, 2]).astype(np.float32)
        assert d2.min().view(np.uint32) == gm[j].view(np.uint32), j
    # the second pick is one library argmax over all 10^6 points
    d = (P - P[w.start_idx]).astype(np.float32)
    d2 = ((d[:, 0] * d[:, 0] + d[:, 1] * d[:, 1]).astype(np.float32) + d[:, 2] * d[:, 2]).astype(np.float32)
    assert gi[1] == int(np.argmax(d2)) and gm[1].view(np.uint32) == d2.max().view(np.uint32)


def test_two_host_threads_pipelined_one_shot_calls(rf):
    """Two host threads call the chunked (pipelined) one-shot entry point at the same time, each on its own
    stream with its own inputs: every call owns its internal build stream and event, so neither can see the
    other's ordering.  Each result must equal the oracle."""
    import threading
    w = inputs.scaled("C2", 3000, 700, B=12)
    Ps = [inputs.make_batch(w, seed=4000 + 100 * t) for t in range(2)]
    refs = [oracle.fps(P, w.M, 0) for P in Ps]
    errs = []

    def work(t):
        try:
            torch.cuda.set_device(0)
            side = torch.cuda.Stream()
            Ph = torch.from_numpy(Ps[t]).pin_memory()
            for _ in range(6):
                with torch.cuda.stream(side):
                    Pd = torch.empty_like(Ph, device="cuda")
                    Pd.copy_(Ph, non_blocking=True)
                    idx, mind = rf.fps_build_and_sample(Pd, w.M, chunk_clouds=3 + t, stream=side)
                    hi, hm = idx.to("cpu", non_blocking=True), mind.to("cpu", non_blocking=True)
                side.synchronize()
                assert_same(hi.numpy(), hm.numpy(), *refs[t])
        except BaseException as e:          # noqa: BLE001 -- reported by the main thread
            errs.append((t, repr(e)))

    th = [threading.Thread(target=work, args=(t,)) for t in range(2)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    assert not errs, errs


def test_trim_and_rebuild(rf):
    P = torch.from_numpy(inputs.room(5000, 77)).cuda()
    ref = oracle.fps(P.cpu().numpy(), 500, 0)
    for _ in range(2):
        ix = rf.fps_index_build(P)
        idx, mind = rf.fps_sample(ix, 500, 0)
        torch.cuda.synchronize()
        rf.fps_index_destroy(ix)
        rf.fps_trim()
        assert_same(idx.cpu().numpy(), mind.cpu().numpy(), *ref)


def test_bench_replicas_on_two_gpus():
    """bench.py's world > 1 branch (NCCL init, per-rank seeds, max over ranks of CUDA-event times) on real GPUs.
    Needs >= 2 devices; the boxes this suite normally runs on have one, so it then SKIPS LOUDLY."""
    import subprocess
    import sys
    if torch.cuda.device_count() < 2:
        pytest.skip(f"needs >= 2 CUDA devices for torchrun --nproc-per-node 2, found {torch.cuda.device_count()}: "
                    "the multi-GPU replica path is covered on CPU by tests/test_sharding_gloo.py only")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", "29533", os.path.join(root, "bench.py"),
                          "--gpus", "2", "--steps", "3", "--warmup", "3", "--workload", "C1", "--quick"],
                         capture_output=True, text=True, timeout=600, cwd=root)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads([ln for ln in out.stdout.splitlines() if ln.startswith("{")][-1])
    assert line["n_gpus"] == 2 and line["value"] > 0 and line["scaling"] == "weak"
