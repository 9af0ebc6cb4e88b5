"""oracle -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

CPU reference programs for exact farthest point sampling (arxiv/paper_2606_06255):

* ``fps``         classical O(N*M) FPS, ``oracle/fps_oracle.c`` (Alg. 1; exactness
                  contract PAPER.md:179).  This is THE oracle.
* ``fps_euclid``  the same with the Euclidean (sqrt) distance of the paper's text, ``oracle/fps_oracle_euclid.c``
                  (Eq. 1 / Eq. 29): the oracle of the library's FPS_FLAG_EUCLIDEAN mode.
* ``pruned_fps``  the paper's section-3 CPU RadiusFPS, ``oracle/fps_pruned_cpu.c`` (Eq. 6-30,
                  PAPER.md:187-350); an independent program that must agree with ``fps`` bit for bit.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s CPU legs (``cpu_baseline``,
``--impl reference``) may import this package.  It imports nothing from the CUDA package
``paper_2606_06255_b200`` and that package imports nothing from here.

Parity pins: tests/test_oracle_pins.py (brute force from Eq. 3, closed forms, M=2 library argmax,
O(M^2) min-distance recomputation, invariants, metamorphic scaling, arithmetic-sensitivity lattice,
agreement of ``fps`` with ``pruned_fps``; section 9 of that file pins ``fps_euclid``).  Parity with the PAPER'S OWN implementation is unpinned
and unpinnable: the paper publishes no code and prints no worked example.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_BUILD = os.path.join(_HERE, "_build")
_CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared", "-fopenmp", "-Wall"]
_lock = threading.Lock()
_libs: dict[str, ctypes.CDLL] = {}


class PrunedStats(ctypes.Structure):
    _fields_ = [
        ("voxel_tests", ctypes.c_int64),
        ("voxels_visited", ctypes.c_int64),
        ("points_visited", ctypes.c_int64),
        ("points_computed", ctypes.c_int64),
        ("effective", ctypes.c_int64),
        ("K", ctypes.c_int32),
        ("n_vox", ctypes.c_int32),
    ]

    def as_dict(self) -> dict:
        return {name: int(getattr(self, name)) for name, _ in self._fields_}


def _compile(stem: str) -> str:
    src = os.path.join(_HERE, stem + ".c")
    out = os.path.join(_BUILD, "lib" + stem + ".so")
    if os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(src):
        return out
    os.makedirs(_BUILD, exist_ok=True)
    tmp = out + f".tmp{os.getpid()}"
    subprocess.run(["gcc", *_CFLAGS, src, "-o", tmp, "-lm"], check=True)
    os.replace(tmp, out)
    return out


def build() -> None:
    """Compile both C programs (called by __graft_entry__.build(); building is not using)."""
    for stem in ("fps_oracle", "fps_oracle_euclid", "fps_pruned_cpu"):
        _compile(stem)


def _lib(stem: str) -> ctypes.CDLL:
    with _lock:
        if stem not in _libs:
            _libs[stem] = ctypes.CDLL(_compile(stem))
        return _libs[stem]


def _as_batch(points) -> tuple[np.ndarray, bool]:
    p = np.ascontiguousarray(points, dtype=np.float32)
    if p.ndim == 2:
        if p.shape[1] != 3:
            raise ValueError("points must be [N,3] or [B,N,3]")
        return p[None], True
    if p.ndim != 3 or p.shape[2] != 3:
        raise ValueError("points must be [N,3] or [B,N,3]")
    return p, False


_f32p = ctypes.POINTER(ctypes.c_float)
_i32p = ctypes.POINTER(ctypes.c_int32)


def fps(points, M: int, start: int = 0, threads: int = 0):
    """Classical FPS.  points [N,3] or [B,N,3] float32 -> (idx int32, mindist float32) of shape
    [M] or [B,M].  ``threads``: OpenMP threads over clouds (0 = all).  Also returns nothing else;
    use ``fps_threads_used`` to learn the thread count of the last batch call."""
    p, single = _as_batch(points)
    B, N, _ = p.shape
    lib = _lib("fps_oracle")
    fn = lib.oracle_fps_batch
    fn.restype = ctypes.c_int
    fn.argtypes = [_f32p, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, _i32p, _f32p,
                   ctypes.c_int32]
    idx = np.empty((B, M), dtype=np.int32)
    mind = np.empty((B, M), dtype=np.float32)
    r = fn(p.ctypes.data_as(_f32p), B, N, M, start, idx.ctypes.data_as(_i32p), mind.ctypes.data_as(_f32p),
           threads)
    if r < 0:
        raise ValueError(f"oracle_fps_batch failed with code {r} (N={N}, M={M}, start={start})")
    fps.threads_used = r
    return (idx[0], mind[0]) if single else (idx, mind)


fps.threads_used = 1


def fps_euclid(points, M: int, start: int = 0, threads: int = 0):
    """Classical FPS with the Euclidean distance sqrtf(d2) (the paper's literal Eq. 1 / Eq. 29).  Same
    shapes as ``fps``; ``mindist`` holds distances, not squared distances."""
    p, single = _as_batch(points)
    B, N, _ = p.shape
    fn = _lib("fps_oracle_euclid").oracle_fps_euclid_batch
    fn.restype = ctypes.c_int
    fn.argtypes = [_f32p, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, _i32p, _f32p,
                   ctypes.c_int32]
    idx = np.empty((B, M), dtype=np.int32)
    mind = np.empty((B, M), dtype=np.float32)
    r = fn(p.ctypes.data_as(_f32p), B, N, M, start, idx.ctypes.data_as(_i32p), mind.ctypes.data_as(_f32p),
           threads)
    if r < 0:
        raise ValueError(f"oracle_fps_euclid_batch failed with code {r} (N={N}, M={M}, start={start})")
    return (idx[0], mind[0]) if single else (idx, mind)


def pruned_fps(points, M: int, start: int = 0, n_vox: int = 16, *, prune: bool = True, skip: bool = True,
               centroid_only: bool = False, threads: int = 0):
    """The paper's CPU RadiusFPS.  Returns (idx, mindist, stats) where stats is a dict (single
    cloud) or a list of dicts (batch).  ``centroid_only`` is the unsafe negative control of Fig. 5."""
    p, single = _as_batch(points)
    B, N, _ = p.shape
    lib = _lib("fps_pruned_cpu")
    fn = lib.pruned_fps_cpu_batch
    fn.restype = ctypes.c_int
    fn.argtypes = [_f32p, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32,
                   ctypes.c_int32, _i32p, _f32p, ctypes.POINTER(PrunedStats), ctypes.c_int32]
    flags = (0 if prune else 1) | (0 if skip else 2) | (4 if centroid_only else 0)
    idx = np.empty((B, M), dtype=np.int32)
    mind = np.empty((B, M), dtype=np.float32)
    stats = (PrunedStats * B)()
    r = fn(p.ctypes.data_as(_f32p), B, N, M, start, n_vox, flags, idx.ctypes.data_as(_i32p),
           mind.ctypes.data_as(_f32p), stats, threads)
    if r < 0:
        raise ValueError(f"pruned_fps_cpu_batch failed with code {r}")
    pruned_fps.threads_used = r
    sd = [s.as_dict() for s in stats]
    return (idx[0], mind[0], sd[0]) if single else (idx, mind, sd)


pruned_fps.threads_used = 1
