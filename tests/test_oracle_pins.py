"""Pins for the CPU oracle (oracle/fps_oracle.c) -- CPU only, no GPU.

The paper prints no worked example, so nothing here is a paper-printed value.  The
oracle is pinned to things other than itself:

* the DEFINITION, Eq. 3: brute force that recomputes min over all earlier samples
  for every point at every step (no D array), in NumPy float32, on N <= 64;
* closed forms in exactly representable numbers (tests/golden/closed_forms.txt);
* M=2 reduces to one library argmax;
* the O(M^2) recomputation of out_mindist from the outputs alone;
* invariants and metamorphic relations;
* the arithmetic-sensitivity lattice: the stated fp32 expression (R1) and no other.
"""
import os

import numpy as np
import pytest

import oracle
from paper_2606_06255_b200 import inputs

F = np.float32
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ---------------------------------------------------------------------------------------------
# independent NumPy restatements used as pins (they share nothing with oracle/*.c)
# ---------------------------------------------------------------------------------------------
def d2_stated(P, s):
    """((dx*dx + dy*dy) + dz*dz) in float32, each op rounded (NumPy never fuses)."""
    d = (P - s[None, :]).astype(F)
    xx = (d[:, 0] * d[:, 0]).astype(F)
    yy = (d[:, 1] * d[:, 1]).astype(F)
    zz = (d[:, 2] * d[:, 2]).astype(F)
    return ((xx + yy).astype(F) + zz).astype(F)


def d2_reassoc(P, s):
    d = (P - s[None, :]).astype(F)
    xx = (d[:, 0] * d[:, 0]).astype(F)
    yy = (d[:, 1] * d[:, 1]).astype(F)
    zz = (d[:, 2] * d[:, 2]).astype(F)
    return (xx + (yy + zz).astype(F)).astype(F)


def d2_single_rounding(P, s):
    """What a fused / extended-precision evaluation would give: exact sum, rounded once."""
    d = (P - s[None, :]).astype(F).astype(np.float64)
    return (d[:, 0] * d[:, 0] + d[:, 1] * d[:, 1] + d[:, 2] * d[:, 2]).astype(F)


def d_sqrt(P, s):
    return np.sqrt(d2_stated(P, s)).astype(F)


def brute_force_fps(P, M, start, dist=d2_stated):
    """Eq. 3 literally: s_j = argmax_p min_{s in S_{j-1}} dist(p, s), ties to the lowest index
    (np.argmax returns the first maximum).  No cached distance array."""
    idx = [start]
    mind = [F(np.inf)]
    for _ in range(1, M):
        cols = np.stack([dist(P, P[s]) for s in idx], axis=1)       # [N, j]
        m = cols.min(axis=1)
        i = int(np.argmax(m))
        idx.append(i)
        mind.append(m[i])
    return np.array(idx, dtype=np.int32), np.array(mind, dtype=F)


def cached_fps(P, M, start, dist):
    """Alg. 1 with a D array, NumPy; used only to run the alternative-arithmetic variants."""
    D = np.full(P.shape[0], np.inf, dtype=F)
    idx, mind, cur = [start], [F(np.inf)], start
    for _ in range(1, M):
        D = np.minimum(D, dist(P, P[cur]))
        cur = int(np.argmax(D))
        idx.append(cur)
        mind.append(D[cur])
    return np.array(idx, dtype=np.int32), np.array(mind, dtype=F)


def same_bits(a, b):
    return np.array_equal(np.asarray(a, F).view(np.uint32), np.asarray(b, F).view(np.uint32))


# ---------------------------------------------------------------------------------------------
# 1. definition
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", range(6))
@pytest.mark.parametrize("N", [1, 2, 5, 33, 64])
def test_brute_force_definition_random(N, seed):
    P = inputs.uniform_cube(N, 100 + seed)
    start = seed % N
    idx, mind = oracle.fps(P, N, start)
    bidx, bmind = brute_force_fps(P, N, start)
    assert np.array_equal(idx, bidx)
    assert same_bits(mind, bmind)


@pytest.mark.parametrize("name", ["line", "corners", "lattice", "dups"])
def test_brute_force_definition_tie_heavy(name):
    P = {"line": inputs.integer_line(37), "corners": inputs.cube_corners(),
         "lattice": inputs.shuffled_lattice(4, 7), "dups": inputs.with_duplicates(48, 3, 40)}[name]
    N = P.shape[0]
    idx, mind = oracle.fps(P, N, 0)
    bidx, bmind = brute_force_fps(P, N, 0)
    assert np.array_equal(idx, bidx)
    assert same_bits(mind, bmind)


# ---------------------------------------------------------------------------------------------
# 2. closed forms
# ---------------------------------------------------------------------------------------------
def _closed_forms():
    rows = []
    with open(os.path.join(GOLDEN, "closed_forms.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            name, gen, start, idx, mind = [c.strip() for c in line.split("|")]
            rows.append((name, gen, int(start), [int(t) for t in idx.split()],
                         [float(t) for t in mind.split()]))
    return rows


@pytest.mark.parametrize("row", _closed_forms(), ids=lambda r: r[0])
def test_closed_forms(row):
    _, gen, start, want_idx, want_mind = row
    P = eval(gen, {"integer_line": inputs.integer_line, "cube_corners": inputs.cube_corners})
    idx, mind = oracle.fps(P, len(want_idx), start)
    assert idx.tolist() == want_idx
    assert mind.tolist() == want_mind


def test_identical_points_repeat_lowest_index():
    # reading A7: once max D = +0 every point ties and index 0 is returned again and again
    P = np.full((10, 3), 0.25, dtype=F)
    idx, mind = oracle.fps(P, 6, 3)
    assert idx.tolist() == [3, 0, 0, 0, 0, 0]
    assert mind.tolist() == [np.inf, 0, 0, 0, 0, 0]


def test_line_bisection_general():
    # N = 2^k + 1 points on a line: the pick order is the bisection order with ties to the lower
    # index; min-distances are (2^k)^2, then (2^(k-1))^2 once, (2^(k-2))^2 twice, ...
    k = 6
    N = (1 << k) + 1
    idx, mind = oracle.fps(inputs.integer_line(N), N, 0)
    want = [np.inf, float((N - 1) ** 2)]
    for level in range(1, k + 1):
        want += [float(((N - 1) >> level) ** 2)] * (1 << (level - 1))
    assert mind.tolist() == want
    assert sorted(idx.tolist()) == list(range(N))
    # within a level picks come in ascending index order
    pos = 2
    for level in range(1, k + 1):
        n = 1 << (level - 1)
        seg = idx[pos:pos + n].tolist()
        assert seg == sorted(seg)
        pos += n


# ---------------------------------------------------------------------------------------------
# 3. M = 2 is one library argmax
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", range(4))
def test_M2_is_argmax(seed):
    P = inputs.uniform_cube(5000, 50 + seed)
    start = 17 * seed
    idx, mind = oracle.fps(P, 2, start)
    d = d2_stated(P, P[start])
    assert idx.tolist() == [start, int(np.argmax(d))]
    assert same_bits(mind[1], d.max())


# ---------------------------------------------------------------------------------------------
# 4./5. min-distance recomputed from the outputs alone + invariants
# ---------------------------------------------------------------------------------------------
def check_outputs(P, idx, mind, start, full_max_check=False):
    M = len(idx)
    assert idx[0] == start and np.isinf(mind[0]) and mind[0] > 0
    S = P[idx]
    for j in range(1, M):
        d = d2_stated(S[:j], S[j])
        assert same_bits(mind[j], d.min()), j
    assert np.all(mind[1:] <= mind[:-1])                      # non-increasing, exactly
    pos = mind > 0
    assert len(set(idx[pos].tolist())) == int(pos.sum())       # distinct while mind > 0
    if M >= 2:
        assert same_bits(mind[1], d2_stated(P, P[start]).max())
    if full_max_check:
        D = np.full(P.shape[0], np.inf, dtype=F)
        for j in range(1, M):
            D = np.minimum(D, d2_stated(P, P[idx[j - 1]]))
            assert same_bits(D.max(), mind[j])
            assert idx[j] == int(np.argmax(D))


@pytest.mark.parametrize("gen", ["uniform", "room", "lidar", "clustered", "lattice"])
def test_outputs_recomputed(gen):
    P = {"uniform": lambda: inputs.uniform_cube(3000, 9),
         "room": lambda: inputs.room(3000, 9),
         "lidar": lambda: inputs.lidar(3000, 9, n_azimuth=47),
         "clustered": lambda: inputs.clustered(3000, 9),
         "lattice": lambda: inputs.shuffled_lattice(12, 9)}[gen]()
    M = 400
    idx, mind = oracle.fps(P, M, 5)
    check_outputs(P, idx, mind, 5, full_max_check=True)


# ---------------------------------------------------------------------------------------------
# 6. metamorphic
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("k", [-3, 1, 5])
def test_scaling_by_power_of_two(k):
    P = inputs.room(2000, 21)
    idx, mind = oracle.fps(P, 300, 0)
    idx2, mind2 = oracle.fps((P * F(2.0 ** k)).astype(F), 300, 0)
    assert np.array_equal(idx, idx2)
    assert same_bits(mind2, (mind * F(4.0 ** k)).astype(F))


def test_permutation_invariance_without_ties():
    P = inputs.uniform_cube(2000, 33)
    perm = np.random.default_rng(1).permutation(2000)
    idx, mind = oracle.fps(P, 300, 0)
    start2 = int(np.nonzero(perm == 0)[0][0])
    idx2, mind2 = oracle.fps(P[perm], 300, start2)
    assert len(np.unique(mind[1:])) == 299          # no ties among the picked values
    assert np.array_equal(perm[idx2], idx)
    assert same_bits(mind, mind2)


def test_batch_equals_singles_and_threads():
    w = inputs.scaled("C2", 1500, 200, B=5)
    P = inputs.make_batch(w)
    idx, mind = oracle.fps(P, w.M, 0, threads=3)
    assert oracle.fps.threads_used == 3
    for b in range(w.B):
        i1, m1 = oracle.fps(P[b], w.M, 0)
        assert np.array_equal(idx[b], i1) and same_bits(mind[b], m1)


def test_argument_errors():
    P = inputs.uniform_cube(10, 1)
    for M, start in [(0, 0), (11, 0), (5, -1), (5, 10)]:
        with pytest.raises(ValueError):
            oracle.fps(P, M, start)


# ---------------------------------------------------------------------------------------------
# 7. the stated arithmetic and no other
# ---------------------------------------------------------------------------------------------
def test_arithmetic_sensitivity_lattice():
    P = inputs.shuffled_lattice(16, 2024)           # 4096 points * 0.1f
    M = 256
    idx, mind = oracle.fps(P, M, 0)
    sidx, smind = cached_fps(P, M, 0, d2_stated)
    assert np.array_equal(idx, sidx) and same_bits(mind, smind)
    # the test has teeth: each alternative arithmetic gives a different answer on this input
    for alt in (d2_reassoc, d2_single_rounding, d_sqrt):
        aidx, amind = cached_fps(P, M, 0, alt)
        cmp_mind = amind if alt is not d_sqrt else (amind * amind).astype(F)
        assert (not np.array_equal(idx, aidx)) or (not same_bits(mind, cmp_mind)), alt.__name__


def test_arithmetic_sensitivity_random_bits():
    # on a random cloud the index sequence survives re-association / single rounding but the
    # min-distance BITS do not: the oracle must carry the stated expression's bits
    P = inputs.uniform_cube(4096, 77)
    idx, mind = oracle.fps(P, 512, 0)
    sidx, smind = cached_fps(P, 512, 0, d2_stated)
    assert np.array_equal(idx, sidx) and same_bits(mind, smind)
    _, rmind = cached_fps(P, 512, 0, d2_reassoc)
    _, fmind = cached_fps(P, 512, 0, d2_single_rounding)
    assert not same_bits(mind, rmind)
    assert not same_bits(mind, fmind)


# ---------------------------------------------------------------------------------------------
# 9. the Euclidean oracle (oracle.fps_euclid; the paper's literal Eq. 1 / Eq. 29)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", range(4))
@pytest.mark.parametrize("N", [1, 2, 5, 33, 64])
def test_euclid_brute_force_definition(N, seed):
    P = inputs.uniform_cube(N, 700 + seed)
    M = N
    bi, bm = brute_force_fps(P, M, seed % N, dist=d_sqrt)
    oi, om = oracle.fps_euclid(P, M, seed % N)
    assert np.array_equal(oi, bi) and same_bits(om, bm)


@pytest.mark.parametrize("name", ["lattice", "line", "corners", "dups"])
def test_euclid_brute_force_tie_heavy(name):
    P = {"lattice": inputs.shuffled_lattice(4, 3), "line": inputs.integer_line(33), "corners": inputs.cube_corners(),
         "dups": inputs.with_duplicates(40, 5, 9)}[name]
    M = min(P.shape[0], 40)
    bi, bm = brute_force_fps(P, M, 0, dist=d_sqrt)
    oi, om = oracle.fps_euclid(P, M, 0)
    assert np.array_equal(oi, bi) and same_bits(om, bm)


def test_euclid_closed_form_line():
    # integer line 0..8: same bisection as the squared case (PAPER.md:179 tie rule), distances not squared
    oi, om = oracle.fps_euclid(inputs.integer_line(9), 9, 0)
    assert oi.tolist() == [0, 8, 4, 2, 6, 1, 3, 5, 7]
    assert om.tolist() == [np.inf, 8, 4, 2, 2, 1, 1, 1, 1]


def test_euclid_equals_sqrt_of_squared_oracle_when_nothing_collapses():
    # sqrt is monotone, so the two oracles pick the same points unless two different squared maxima round
    # to the same square root; where the index sequences agree the distances must be sqrt of each other
    agree = 0
    for seed in range(6):
        P = inputs.room(1500, 800 + seed)
        si, sm = oracle.fps(P, 300, 0)
        ei, em = oracle.fps_euclid(P, 300, 0)
        n = 300 if np.array_equal(si, ei) else int(np.argmax(si != ei))
        assert n >= 2
        assert same_bits(em[:n], np.sqrt(sm[:n]).astype(F))
        agree += n == 300
    assert agree >= 1


def test_euclid_differs_from_squared_where_sqrt_collapses_two_maxima():
    # constructed: origin, A, B with fl(d2(B)) one ulp above fl(d2(A)) but the same correctly rounded
    # square root.  Squared FPS picks B (larger), Euclidean FPS sees a tie and takes the lower index A.
    rng = np.random.default_rng(5)
    found = None
    for _ in range(200):
        Q = np.zeros((4000, 3), dtype=F)
        Q[:, :2] = rng.random((4000, 2), dtype=F) + F(0.5)
        d2 = d2_stated(Q, np.zeros(3, dtype=F))
        order = np.argsort(d2, kind="stable")
        s = d2[order]
        r = np.sqrt(s).astype(F)
        hit = np.nonzero((s[1:] > s[:-1]) & (r[1:] == r[:-1]))[0]
        if hit.size:
            found = (Q[order[hit[0]]], Q[order[hit[0] + 1]])
            break
    assert found is not None
    P = np.stack([np.zeros(3, dtype=F), found[0], found[1]])
    si, _ = oracle.fps(P, 2, 0)
    ei, em = oracle.fps_euclid(P, 2, 0)
    assert si.tolist() == [0, 2] and ei.tolist() == [0, 1]
    assert same_bits(em[1:], d_sqrt(P[1:2], P[0]))


@pytest.mark.parametrize("threads", [1, 2, 0])
def test_euclid_batch_equals_singles_and_threads(threads):
    # the batch wrapper oracle_fps_euclid_batch (cloud stride 3N of the input, M of both outputs, OpenMP over
    # clouds) is pinned to the single-cloud function, which the brute-force tests above pin to Eq. 3; clouds of
    # three different generators so that a wrong stride cannot land on an identical neighbour
    N, M = 1500, 200
    P = np.stack([inputs.room(N, 901), inputs.uniform_cube(N, 902), inputs.clustered(N, 903),
                  inputs.room(N, 904, dense_half=True), inputs.lidar(N, 905, n_azimuth=24)])
    idx, mind = oracle.fps_euclid(P, M, 3, threads=threads)
    assert idx.shape == (5, M) and mind.shape == (5, M)
    for b in range(P.shape[0]):
        i1, m1 = oracle.fps_euclid(P[b], M, 3)
        assert np.array_equal(idx[b], i1) and same_bits(mind[b], m1)
        bi, bm = brute_force_fps(P[b][:48], 48, 3, dist=d_sqrt)         # and one step further down: Eq. 3 itself
        oi, om = oracle.fps_euclid(np.stack([P[b][:48]] * 2), 48, 3, threads=threads)
        assert np.array_equal(oi[1], bi) and same_bits(om[1], bm)
