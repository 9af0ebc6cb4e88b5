"""The paper's section-3 CPU RadiusFPS (oracle/fps_pruned_cpu.c) against the classical oracle.

Three independent programs must agree bit for bit: the oracle, this CPU pruned variant and (in the
-m gpu tests) the CUDA path.  Also here: prune/skip ablations (Table 4 structure)
must not change a bit; the centroid-only prune of Fig. 5/6 must break exactness
on some input (the agreement test has teeth); Fig. 3's ">90% ineffective updates".
"""
import numpy as np
import pytest

import oracle
from paper_2606_06255_b200 import inputs

F = np.float32


def same(a, b):
    return np.array_equal(a[0], b[0]) and np.array_equal(a[1].view(np.uint32), b[1].view(np.uint32))


CLOUDS = {
    "uniform": lambda: inputs.uniform_cube(4096, 1234),
    "room": lambda: inputs.room(6000, 11),
    "room_dense": lambda: inputs.room(6000, 12, size=(20.0, 15.0, 3.0), n_boxes=60, dense_half=True),
    "lidar": lambda: inputs.lidar(6000, 13, n_azimuth=94),
    "clustered": lambda: inputs.clustered(5000, 14),
    "lattice": lambda: inputs.shuffled_lattice(16, 15),
    "dups": lambda: inputs.with_duplicates(3000, 16, 700),
    "line": lambda: inputs.integer_line(513),
}


@pytest.mark.parametrize("name", sorted(CLOUDS))
@pytest.mark.parametrize("n_vox", [1, 2, 7, 16, 24, 32])
def test_pruned_equals_oracle(name, n_vox):
    P = CLOUDS[name]()
    M = min(P.shape[0], 1024)
    ref = oracle.fps(P, M, 0)
    got = oracle.pruned_fps(P, M, 0, n_vox=n_vox)
    assert same(ref, got[:2])


@pytest.mark.parametrize("prune,skip", [(True, False), (False, True), (False, False)])
@pytest.mark.parametrize("name", ["room", "lattice", "lidar"])
def test_ablations_bit_identical(name, prune, skip):
    P = CLOUDS[name]()
    ref = oracle.fps(P, 800, 3)
    got = oracle.pruned_fps(P, 800, 3, n_vox=16, prune=prune, skip=skip)
    assert same(ref, got[:2])
    st = got[2]
    if not prune:
        assert st["voxels_visited"] == st["K"] * 799
    if not skip:
        assert st["points_computed"] == st["points_visited"]


def test_M_equals_N_and_other_starts():
    P = inputs.room(700, 5)
    for start in (0, 1, 699):
        assert same(oracle.fps(P, 700, start), oracle.pruned_fps(P, 700, start, n_vox=8)[:2])


def test_centroid_only_negative_control_breaks():
    """Fig. 5/6: pruning on the centre distance alone (r_k = 0) is unsafe.  It must change the
    result on at least one of these inputs, otherwise the agreement tests above prove nothing."""
    broken = 0
    for name in ("uniform", "room", "lattice", "clustered"):
        P = CLOUDS[name]()
        ref = oracle.fps(P, 512, 0)
        got = oracle.pruned_fps(P, 512, 0, n_vox=8, centroid_only=True)
        broken += not same(ref, got[:2])
    assert broken >= 1


def test_most_updates_are_ineffective():
    # Fig. 3: > 90 % of the classical method's N*(M-1) updates change nothing
    P = inputs.room(24000, inputs.BASE_SEED)
    M = 1500
    _, _, st = oracle.pruned_fps(P, M, 0, n_vox=32)
    dense = P.shape[0] * (M - 1)
    assert st["effective"] / dense < 0.01
    assert st["points_visited"] / dense < 0.10      # and the pruned method never looks at most of them


def test_batch_threads():
    w = inputs.scaled("C4", 3000, 300, B=3)
    P = inputs.make_batch(w)
    ref = oracle.fps(P, w.M, 0)
    got = oracle.pruned_fps(P, w.M, 0, n_vox=16, threads=2)
    assert oracle.pruned_fps.threads_used == 2
    assert same(ref, got[:2])
