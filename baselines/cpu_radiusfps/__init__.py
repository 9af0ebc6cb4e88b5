"""baselines.cpu_radiusfps -- a tuned, multi-threaded CPU RadiusFPS (``radiusfps_cpu.c``): A BASELINE PROGRAM.

It is timed by bench.py's ``cpu_baseline`` leg beside the CPU oracle, as the analogue of the paper's own CPU
RadiusFPS (Fig. 15b).  It is not the oracle (``oracle/`` is: plain and slow on purpose), it is
not product code (nothing under ``paper_2606_06255_b200/`` imports it and the product has no CPU fallback), and it
shares no code with either.  tests/test_cpu_radiusfps.py requires its output to equal ``oracle.fps`` bit for bit.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_BUILD = os.path.join(_HERE, "_build")
# x86-64-v3 (AVX2) and not -march=native: the built .so travels from the build container to the GPU box
_CFLAGS = ["-O3", "-march=x86-64-v3", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared", "-fopenmp", "-Wall"]
_lock = threading.Lock()
_lib = None


class Stats(ctypes.Structure):
    _fields_ = [("group_tests", ctypes.c_int64), ("voxel_tests", ctypes.c_int64), ("voxels_visited", ctypes.c_int64),
                ("points_visited", ctypes.c_int64), ("K", ctypes.c_int32), ("n_vox", ctypes.c_int32)]


def build() -> str:
    src = os.path.join(_HERE, "radiusfps_cpu.c")
    out = os.path.join(_BUILD, "libradiusfps_cpu.so")
    if os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(src):
        return out
    os.makedirs(_BUILD, exist_ok=True)
    tmp = out + f".tmp{os.getpid()}"
    subprocess.run(["gcc", *_CFLAGS, src, "-o", tmp, "-lm"], check=True)
    os.replace(tmp, out)
    return out


def _load():
    global _lib
    with _lock:
        if _lib is None:
            _lib = ctypes.CDLL(build())
            f32p, i32p, i32 = ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_int32), ctypes.c_int32
            _lib.radiusfps_cpu_batch.restype = ctypes.c_int
            _lib.radiusfps_cpu_batch.argtypes = [f32p, i32, i32, i32, i32, i32, i32, i32p, f32p, ctypes.POINTER(Stats), i32]
        return _lib


def fps(points, M: int, start: int = 0, n_vox: int = 0, *, point_skip: bool = False, threads: int = 0):
    """points [N,3] or [B,N,3] float32 -> (idx int32, mindist float32, stats list).  n_vox 0 = choose from N."""
    p = np.ascontiguousarray(points, dtype=np.float32)
    single = p.ndim == 2
    if single:
        p = p[None]
    if p.ndim != 3 or p.shape[2] != 3:
        raise ValueError("points must be [N,3] or [B,N,3]")
    B, N, _ = p.shape
    idx = np.empty((B, M), dtype=np.int32)
    mind = np.empty((B, M), dtype=np.float32)
    st = (Stats * B)()
    f32p, i32p = ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_int32)
    r = _load().radiusfps_cpu_batch(p.ctypes.data_as(f32p), B, N, M, start, n_vox, 1 if point_skip else 0,
                                    idx.ctypes.data_as(i32p), mind.ctypes.data_as(f32p), st, threads)
    if r < 0:
        raise ValueError(f"radiusfps_cpu_batch failed with code {r}")
    fps.threads_used = r
    stats = [{n: int(getattr(s, n)) for n, _ in Stats._fields_} for s in st]
    return (idx[0], mind[0], stats[0]) if single else (idx, mind, stats)


fps.threads_used = 1
