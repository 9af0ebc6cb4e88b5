"""The tuned CPU RadiusFPS baseline (baselines/cpu_radiusfps) must return exactly what
classical FPS returns: compared bit for bit with the CPU oracle, on CPU only.  It is a baseline
program for bench.py, not the oracle and not product code."""
import os
import re

import numpy as np
import pytest

import oracle
from baselines import cpu_radiusfps as cr
from paper_2606_06255_b200 import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CLOUDS = {
    "uniform": lambda: (inputs.uniform_cube(4096, 1234), 1024),
    "room": lambda: (inputs.room(6000, 11), 1500),
    "room_dense": lambda: (inputs.room(5000, 12, size=(20.0, 15.0, 3.0), n_boxes=60, dense_half=True), 1250),
    "lidar": lambda: (inputs.lidar(6000, 13, n_azimuth=94), 1500),
    "clustered": lambda: (inputs.clustered(5000, 14), 1250),
    "lattice": lambda: (inputs.shuffled_lattice(16, 15), 1024),
    "dups": lambda: (inputs.with_duplicates(3000, 16, 700), 1000),
    "line": lambda: (inputs.integer_line(513), 513),
    "corners": lambda: (inputs.cube_corners(), 8),
    "one_point": lambda: (inputs.uniform_cube(1, 3), 1),
    "offset_tiny_extent": lambda: ((inputs.uniform_cube(3000, 8) * np.float32(1e-3) + np.float32(1000.0)).astype(np.float32), 600),
}


def same(a, b):
    return np.array_equal(a[0], b[0]) and np.array_equal(a[1].view(np.uint32), b[1].view(np.uint32))


@pytest.mark.parametrize("skip", [False, True])
@pytest.mark.parametrize("n_vox", [0, 1, 2, 7, 16, 33, 64])
@pytest.mark.parametrize("name", sorted(CLOUDS))
def test_equals_the_oracle_for_every_n_vox(name, n_vox, skip):
    P, M = CLOUDS[name]()
    ref = oracle.fps(P, M, 0)
    gi, gm, st = cr.fps(P, M, 0, n_vox, point_skip=skip)
    assert same((gi, gm), ref)
    if n_vox:
        assert st["n_vox"] == n_vox and 1 <= st["K"] <= min(P.shape[0], n_vox ** 3)


@pytest.mark.parametrize("start", [0, 17, 2999])
def test_start_points_and_sampling_every_point(start):
    P = inputs.room(3000, 21)
    assert same(cr.fps(P, 3000, start, 12)[:2], oracle.fps(P, 3000, start))


@pytest.mark.parametrize("threads", [1, 2, 0])
def test_batch_and_threads(threads):
    w = inputs.scaled("C2", 2000, 400, B=5)
    P = inputs.make_batch(w)
    gi, gm, st = cr.fps(P, w.M, 0, threads=threads)
    assert cr.fps.threads_used == (threads or min(5, os.cpu_count() or 1)) or threads == 0
    assert same((gi, gm), oracle.fps(P, w.M, 0))
    assert len(st) == 5 and all(s["voxels_visited"] > 0 for s in st)


def test_it_really_prunes():
    P, M = CLOUDS["room"]()
    _, _, st = cr.fps(P, M, 0, 16)
    assert st["points_visited"] < 0.1 * P.shape[0] * (M - 1)           # the oracle touches N (M-1) points
    assert st["voxel_tests"] < 0.5 * st["K"] * (M - 1)                 # the group level removes most voxel tests


def test_bad_arguments():
    P = inputs.uniform_cube(10, 1)
    for M, start in [(0, 0), (11, 0), (5, -1), (5, 10)]:
        with pytest.raises(ValueError):
            cr.fps(P, M, start)


def test_it_is_a_baseline_not_product_and_not_oracle():
    # nothing in the product or the oracle refers to it, and it refers to neither
    for folder in ("paper_2606_06255_b200", "oracle"):
        for dirpath, _, files in os.walk(os.path.join(ROOT, folder)):
            for f in files:
                if f.endswith((".py", ".cu", ".cuh", ".h", ".c")):
                    assert "baselines" not in open(os.path.join(dirpath, f)).read(), (folder, f)
    for f in os.listdir(os.path.join(ROOT, "baselines", "cpu_radiusfps")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "baselines", "cpu_radiusfps", f)).read()
            assert not re.search(r"^\s*(import|from)\s+(oracle|paper_2606_06255_b200)\b", src, flags=re.M), f
            assert "#include \"" not in src, f
