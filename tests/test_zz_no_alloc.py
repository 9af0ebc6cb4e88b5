"""fps_sample_noalloc (include/radiusfps.h): the allocation-free entry point against the existing path.

The entry point keeps the voxel index of one cloud of <= FPS_NOALLOC_MAX_N points in a static device array instead of
an allocation.  Its outputs must equal those of fps_index_build + fps_sample bit for bit (the bar of
tests/test_gpu_parity.py: 0 index mismatches, 0 ULP), on calls IN A ROW that find the previous call's contents in the
shared array: a large cloud, then a smaller one of a different kind, then the first again.  The file is named so that
pytest collects it last; it passes alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest
import torch

from paper_2606_06255_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def rf():
    from paper_2606_06255_b200 import binding
    binding.load()            # raises if the CUDA library is missing: no fallback
    assert torch.cuda.is_available()
    return binding


def existing_path(rf, Pd, M, start, flags=0):
    ix = rf.fps_index_build(Pd, flags=flags)
    try:
        idx, mind = rf.fps_sample(ix, M, start)
        torch.cuda.synchronize()
    finally:
        rf.fps_index_destroy(ix)
    return idx.cpu().numpy().reshape(-1), mind.cpu().numpy().reshape(-1)


def no_alloc(rf, Pd, M, start, flags=0):
    out_idx = torch.full((M,), -7, dtype=torch.int32, device=Pd.device)
    out_mind = torch.full((M,), -1.0, dtype=torch.float32, device=Pd.device)
    rf.fps_sample_noalloc(Pd, M, out_idx, out_mind, start_idx=start, flags=flags)
    torch.cuda.synchronize()
    return out_idx.cpu().numpy(), out_mind.cpu().numpy()


def assert_bits_equal(got, ref):
    gi, gm = got
    ri, rm = ref
    bad = np.nonzero(gi != ri)[0]
    assert bad.size == 0, f"{bad.size} index mismatches, first at {bad[0]}"
    badm = np.nonzero(gm.view(np.uint32) != rm.view(np.uint32))[0]
    assert badm.size == 0, f"{badm.size} min-distance bit mismatches, first at {badm[0]}"


CASES = [
    # (cloud, M, start): the limit itself, then a smaller cloud of another kind, then a tiny one, then the first again
    (lambda: inputs.uniform_cube(8192, 77), 2048, 0),
    (lambda: inputs.room(3001, 5), 750, 17),
    (lambda: inputs.clustered(257, 3), 257, 256),
    (lambda: inputs.uniform_cube(8192, 77), 2048, 0),
    (lambda: inputs.with_duplicates(4096, 9, 300), 1024, 1),
]


def test_noalloc_equals_existing_path_on_calls_in_a_row(rf):
    clouds = [(torch.from_numpy(np.ascontiguousarray(f())).cuda(), M, s) for f, M, s in CASES]
    refs = [existing_path(rf, Pd, M, s) for Pd, M, s in clouds]
    # the calls follow one another with nothing in between that could reset the shared array
    for (Pd, M, s), ref in zip(clouds, refs):
        assert_bits_equal(no_alloc(rf, Pd, M, s), ref)
    # and back to back on the stream, outputs read only at the end
    outs = []
    for Pd, M, s in clouds:
        oi = torch.empty((M,), dtype=torch.int32, device=Pd.device)
        om = torch.empty((M,), dtype=torch.float32, device=Pd.device)
        rf.fps_sample_noalloc(Pd, M, oi, om, start_idx=s)
        outs.append((oi, om))
    torch.cuda.synchronize()
    for (oi, om), ref in zip(outs, refs):
        assert_bits_equal((oi.cpu().numpy(), om.cpu().numpy()), ref)


def test_noalloc_euclidean_mode(rf):
    Pd = torch.from_numpy(np.ascontiguousarray(inputs.room(6000, 11))).cuda()
    ref = existing_path(rf, Pd, 1500, 3, flags=rf.FPS_FLAG_EUCLIDEAN)
    for _ in range(2):
        assert_bits_equal(no_alloc(rf, Pd, 1500, 3, flags=rf.FPS_FLAG_EUCLIDEAN), ref)


def test_noalloc_takes_no_device_memory(rf):
    Pd = torch.from_numpy(np.ascontiguousarray(inputs.uniform_cube(8192, 78))).cuda()
    oi = torch.empty((2048,), dtype=torch.int32, device="cuda")
    om = torch.empty((2048,), dtype=torch.float32, device="cuda")
    rf.fps_sample_noalloc(Pd, 2048, oi, om)       # first call: kernels are loaded, the symbol's address is resolved
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        rf.fps_sample_noalloc(Pd, 2048, oi, om)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0, f"device memory in use grew by {free0 - free1} bytes over three calls"


def test_noalloc_rejects_sizes_beyond_the_maximum(rf):
    assert rf.FPS_NOALLOC_MAX_N == 8192
    Pd = torch.from_numpy(np.ascontiguousarray(inputs.uniform_cube(8193, 1))).cuda()
    oi = torch.full((16,), -7, dtype=torch.int32, device="cuda")
    om = torch.full((16,), -1.0, dtype=torch.float32, device="cuda")
    with pytest.raises(rf.FpsError) as e:
        rf.fps_sample_noalloc(Pd, 16, oi, om)
    assert e.value.status == rf.FPS_ERR_INVALID
    assert "FPS_NOALLOC_MAX_N" in str(e.value) and "8192" in str(e.value)
    torch.cuda.synchronize()
    assert (oi == -7).all() and (om == -1.0).all()          # nothing was launched
    # the other argument errors, and flags that the entry point does not take
    P2 = torch.from_numpy(np.ascontiguousarray(inputs.uniform_cube(100, 2))).cuda()
    for kw in (dict(M=0), dict(M=101), dict(M=10, start_idx=100), dict(M=10, flags=rf.FPS_FLAG_STATS)):
        M = kw.pop("M")
        o1 = torch.empty((max(M, 1),), dtype=torch.int32, device="cuda")
        o2 = torch.empty((max(M, 1),), dtype=torch.float32, device="cuda")
        with pytest.raises(rf.FpsError) as e:
            rf.fps_sample_noalloc(P2, M, o1, o2, **kw)
        assert e.value.status == rf.FPS_ERR_INVALID
    bad = inputs.uniform_cube(64, 3).copy()
    bad[5, 1] = np.nan
    with pytest.raises(rf.FpsError) as e:
        rf.fps_sample_noalloc(torch.from_numpy(bad).cuda(), 8, torch.empty(8, dtype=torch.int32, device="cuda"),
                              torch.empty(8, dtype=torch.float32, device="cuda"))
    assert e.value.status == rf.FPS_ERR_NONFINITE
    # and the entry point still works after the rejected calls
    ref = existing_path(rf, P2, 25, 0)
    assert_bits_equal(no_alloc(rf, P2, 25, 0), ref)
