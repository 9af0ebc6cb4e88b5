"""Thin ctypes binding of the C-ABI in include/radiusfps.h -- argument marshalling only.

Same names as the C entry points.  PyTorch is used for device memory and streams, nothing else:
every step of the path runs in the CUDA kernels of ``csrc/``.  There is no CPU fallback: if
``libradiusfps.so`` is missing this module raises at first use.
"""
from __future__ import annotations

import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
# RADIUSFPS_LIB: another build of the same library (kernel experiments); the default is the in-tree build
LIB_PATH = os.environ.get("RADIUSFPS_LIB") or os.path.join(_HERE, "libradiusfps.so")

FPS_OK, FPS_ERR_INVALID, FPS_ERR_CUDA, FPS_ERR_NONFINITE, FPS_ERR_NOMEM = 0, -1, -2, -3, -4
FPS_FLAG_NO_PRUNE, FPS_FLAG_NO_SKIP, FPS_FLAG_STATS, FPS_FLAG_NO_BATCH, FPS_FLAG_PER_PICK = 1, 2, 4, 8, 16
FPS_FLAG_EUCLIDEAN = 32
FPS_FLAG_CHAIN_BUILD = 64

EXPORTS = ["fps_index_build", "fps_index_build_ex", "fps_index_build_ragged", "fps_sample", "fps_sample_ragged", "fps_gather_xyz", "fps_pick_chain_cycles", "fps_index_destroy", "fps_get_stats",
           "fps_sample_host", "fps_build_and_sample", "fps_last_error", "fps_last_status", "fps_version", "fps_trim", "fps_sample_noalloc"]


class fps_build_opts(ctypes.Structure):
    _fields_ = [("n_vox", ctypes.c_int32), ("tile_points", ctypes.c_int32), ("cluster_size", ctypes.c_int32),
                ("block_threads", ctypes.c_int32), ("flags", ctypes.c_int32), ("stream", ctypes.c_void_p),
                ("local_warps", ctypes.c_int32), ("cand_per_thread", ctypes.c_int32)]


class fps_stats(ctypes.Structure):
    _fields_ = [("B", ctypes.c_int32), ("N", ctypes.c_int32), ("n_vox", ctypes.c_int32),
                ("cluster_size", ctypes.c_int32), ("block_threads", ctypes.c_int32),
                ("voxels_per_thread", ctypes.c_int32),
                ("K_total", ctypes.c_int64), ("K_max", ctypes.c_int32), ("max_voxel_points", ctypes.c_int32),
                ("device_bytes", ctypes.c_int64), ("build_launches", ctypes.c_int32), ("grid_ctas", ctypes.c_int32),
                ("iterations", ctypes.c_int64), ("voxel_tests", ctypes.c_int64),
                ("voxels_visited", ctypes.c_int64), ("points_visited", ctypes.c_int64),
                ("points_computed", ctypes.c_int64), ("effective", ctypes.c_int64),
                ("rounds", ctypes.c_int64), ("extract_retries", ctypes.c_int64), ("single_picks", ctypes.c_int64),
                ("candidates", ctypes.c_int64), ("extract_voxels", ctypes.c_int64), ("extract_points", ctypes.c_int64),
                ("cycles_apply", ctypes.c_int64), ("cycles_max", ctypes.c_int64), ("cycles_extract", ctypes.c_int64),
                ("cycles_local", ctypes.c_int64), ("group_tests", ctypes.c_int64),
                ("cycles_prune_sum", ctypes.c_int64), ("cycles_visit_sum", ctypes.c_int64),
                ("cycles_prune_max", ctypes.c_int64), ("cycles_visit_max", ctypes.c_int64), ("sub_batches", ctypes.c_int64),
                ("local_subrounds", ctypes.c_int64), ("local_fallbacks", ctypes.c_int64),
                ("local_warps", ctypes.c_int32), ("cand_per_thread", ctypes.c_int32),
                ("cycles_local_select", ctypes.c_int64), ("cycles_local_pick", ctypes.c_int64),
                ("cycles_local_update", ctypes.c_int64), ("cycles_local_pairs", ctypes.c_int64),
                ("cycles_local_publish", ctypes.c_int64), ("cycles_worker_tail", ctypes.c_int64),
                ("cycles_worker_extract", ctypes.c_int64), ("cycles_worker_idle", ctypes.c_int64),
                ("worker_pieces", ctypes.c_int64), ("whole_cloud_kernel", ctypes.c_int32), ("reserved0", ctypes.c_int32)]

    def as_dict(self) -> dict:
        return {n: int(getattr(self, n)) for n, _ in self._fields_}


class FpsError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"radiusfps status {status}: {message}")
        self.status = status


_lib = None


def load() -> ctypes.CDLL:
    """dlopen the in-tree library; raises (no fallback) when it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2606_06255_b200.build` "
            "(or __graft_entry__.build()); there is no CPU fallback")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i32 = ctypes.c_void_p, ctypes.c_int32
    lib.fps_index_build.restype = vp
    lib.fps_index_build.argtypes = [vp, i32, i32]
    lib.fps_index_build_ex.restype = vp
    lib.fps_index_build_ex.argtypes = [vp, i32, i32, ctypes.POINTER(fps_build_opts)]
    lib.fps_sample.restype = ctypes.c_int
    lib.fps_sample.argtypes = [vp, i32, i32, vp, vp, vp]
    lib.fps_index_build_ragged.restype = vp
    lib.fps_index_build_ragged.argtypes = [vp, ctypes.POINTER(i32), i32, ctypes.POINTER(fps_build_opts)]
    lib.fps_sample_ragged.restype = ctypes.c_int
    lib.fps_sample_ragged.argtypes = [vp, ctypes.POINTER(i32), ctypes.POINTER(i32), vp, vp, vp]
    lib.fps_gather_xyz.restype = ctypes.c_int
    lib.fps_gather_xyz.argtypes = [vp, vp, i32, vp, vp]
    lib.fps_pick_chain_cycles.restype = ctypes.c_int
    lib.fps_pick_chain_cycles.argtypes = [i32, i32, ctypes.POINTER(ctypes.c_float)]
    lib.fps_index_destroy.restype = None
    lib.fps_index_destroy.argtypes = [vp]
    lib.fps_get_stats.restype = ctypes.c_int
    lib.fps_get_stats.argtypes = [vp, ctypes.POINTER(fps_stats)]
    lib.fps_sample_host.restype = ctypes.c_int
    lib.fps_sample_host.argtypes = [vp, i32, i32, i32, i32, vp, vp, ctypes.POINTER(fps_build_opts)]
    lib.fps_build_and_sample.restype = ctypes.c_int
    lib.fps_build_and_sample.argtypes = [vp, ctypes.POINTER(i32), i32, i32, ctypes.POINTER(i32), i32, ctypes.POINTER(i32), vp, vp,
                                         ctypes.POINTER(fps_build_opts), i32]
    lib.fps_last_error.restype = ctypes.c_char_p
    lib.fps_last_error.argtypes = []
    lib.fps_version.restype = ctypes.c_char_p
    lib.fps_version.argtypes = []
    lib.fps_last_status.restype = ctypes.c_int
    lib.fps_last_status.argtypes = []
    lib.fps_trim.restype = None
    lib.fps_trim.argtypes = []
    lib.fps_sample_noalloc.restype = ctypes.c_int
    lib.fps_sample_noalloc.argtypes = [ctypes.c_void_p, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32,
                                       ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
    _lib = lib
    return lib


def fps_last_error() -> str:
    return load().fps_last_error().decode()


def fps_version() -> str:
    return load().fps_version().decode()


def fps_trim() -> None:
    load().fps_trim()


def _check_points(points: torch.Tensor) -> tuple[int, int]:
    if points.dtype != torch.float32 or not points.is_contiguous():
        raise ValueError("points must be a contiguous float32 tensor")
    if points.dim() == 2 and points.shape[1] == 3:
        return 1, points.shape[0]
    if points.dim() == 3 and points.shape[2] == 3:
        return points.shape[0], points.shape[1]
    raise ValueError("points must be [N,3] or [B,N,3]")


def _opts(n_vox=0, tile_points=0, cluster_size=0, block_threads=0, flags=0, stream=None, local_warps=0,
          cand_per_thread=0) -> fps_build_opts:
    return fps_build_opts(n_vox, tile_points, cluster_size, block_threads, flags, stream or 0, local_warps,
                          cand_per_thread)


class Index:
    """Owner of one ``fps_index_t*``.  ``points``: CUDA float32 [B,N,3] (or [N,3])."""

    def __init__(self, handle: int, B: int, N: int, device: torch.device, offsets: list[int] | None = None):
        self.handle, self.B, self.N, self.device = handle, B, N, device
        self.offsets = offsets          # ragged index: first point of every cloud (+ total), else None

    def sample(self, M: int, start_idx: int = 0, out_idx: torch.Tensor | None = None,
               out_mindist: torch.Tensor | None = None, stream: torch.cuda.Stream | None = None):
        return fps_sample(self, M, start_idx, out_idx, out_mindist, stream)

    def stats(self) -> dict:
        return fps_get_stats(self)

    def destroy(self) -> None:
        fps_index_destroy(self)

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def fps_index_build(points: torch.Tensor, *, n_vox: int = 0, tile_points: int = 0, cluster_size: int = 0,
                    block_threads: int = 0, flags: int = 0, stream: torch.cuda.Stream | None = None,
                    local_warps: int = 0, cand_per_thread: int = 0) -> Index:
    """fps_index_build / fps_index_build_ex.  The build is issued on ``stream`` (default: torch's
    current stream) and is complete when this returns."""
    lib = load()
    if not points.is_cuda:
        raise ValueError("points must live on a CUDA device (use fps_sample_host for host arrays)")
    B, N = _check_points(points)
    with torch.cuda.device(points.device):
        s = stream if stream is not None else torch.cuda.current_stream()
        o = _opts(n_vox, tile_points, cluster_size, block_threads, flags, s.cuda_stream, local_warps, cand_per_thread)
        h = lib.fps_index_build_ex(points.data_ptr(), N, B, ctypes.byref(o))
    if not h:
        raise FpsError(lib.fps_last_status(), fps_last_error())
    return Index(h, B, N, points.device)


def fps_sample(index: Index, M: int, start_idx: int = 0, out_idx: torch.Tensor | None = None,
               out_mindist: torch.Tensor | None = None, stream: torch.cuda.Stream | None = None):
    """fps_sample: enqueue on ``stream`` (default: torch's current stream); returns
    (out_idx int32 [B,M], out_mindist float32 [B,M]) without synchronising."""
    lib = load()
    if index.handle is None:
        raise ValueError("index was destroyed")
    M = int(M)
    with torch.cuda.device(index.device):
        if out_idx is None:
            out_idx = torch.empty((index.B, max(M, 0)), dtype=torch.int32, device=index.device)
        if out_mindist is None:
            out_mindist = torch.empty((index.B, max(M, 0)), dtype=torch.float32, device=index.device)
        if out_idx.dtype != torch.int32 or out_mindist.dtype != torch.float32 or not out_idx.is_contiguous() \
                or not out_mindist.is_contiguous() or out_idx.numel() < index.B * M or out_mindist.numel() < index.B * M:
            raise ValueError("out_idx must be contiguous int32 [B,M] and out_mindist contiguous float32 [B,M]")
        s = stream if stream is not None else torch.cuda.current_stream()
        rc = lib.fps_sample(index.handle, M, int(start_idx), out_idx.data_ptr(), out_mindist.data_ptr(), s.cuda_stream)
    if rc != FPS_OK:
        raise FpsError(rc, fps_last_error())
    return out_idx, out_mindist


FPS_NOALLOC_MAX_N = 8192


def fps_sample_noalloc(points: torch.Tensor, M: int, out_idx: torch.Tensor, out_mindist: torch.Tensor, start_idx: int = 0,
                       flags: int = 0, stream: torch.cuda.Stream | None = None):
    """fps_sample_noalloc: build + sample ONE cloud (``points`` CUDA float32 [N,3], N <= FPS_NOALLOC_MAX_N) with the index
    in the library's static device array -- no device allocation.  The caller passes the outputs (int32 [M], float32
    [M], CUDA); nothing is allocated here either.  Calls that overlap on the GPU race on the shared array."""
    lib = load()
    if not points.is_cuda or points.dtype != torch.float32 or not points.is_contiguous() or points.dim() != 2 or points.shape[1] != 3:
        raise ValueError("points must be a contiguous CUDA float32 tensor [N,3]")
    M = int(M)
    if out_idx.dtype != torch.int32 or out_mindist.dtype != torch.float32 or not out_idx.is_contiguous() or not out_mindist.is_contiguous() \
            or out_idx.device != points.device or out_mindist.device != points.device or out_idx.numel() < M or out_mindist.numel() < M:
        raise ValueError("out_idx must be contiguous CUDA int32 [M] and out_mindist contiguous CUDA float32 [M]")
    with torch.cuda.device(points.device):
        s = stream if stream is not None else torch.cuda.current_stream()
        rc = lib.fps_sample_noalloc(points.data_ptr(), points.shape[0], M, int(start_idx), int(flags), out_idx.data_ptr(),
                                    out_mindist.data_ptr(), s.cuda_stream)
    if rc != FPS_OK:
        raise FpsError(rc, fps_last_error())
    return out_idx, out_mindist


def fps_index_build_ragged(points: torch.Tensor, offsets, *, n_vox: int = 0, tile_points: int = 0, cluster_size: int = 0,
                           block_threads: int = 0, flags: int = 0, stream: torch.cuda.Stream | None = None,
                           local_warps: int = 0, cand_per_thread: int = 0) -> Index:
    """fps_index_build_ragged: ``points`` CUDA float32 [T,3] holds the clouds one after the other,
    ``offsets`` (B+1 ints, offsets[0] = 0, offsets[B] = T) says where each starts."""
    lib = load()
    if not points.is_cuda or points.dtype != torch.float32 or not points.is_contiguous() or points.dim() != 2 \
            or points.shape[1] != 3:
        raise ValueError("points must be a contiguous CUDA float32 tensor [T,3]")
    off = [int(v) for v in offsets]
    if len(off) < 2 or off[-1] != points.shape[0]:
        raise ValueError("offsets must hold B+1 entries and end at the number of points")
    B = len(off) - 1
    arr = (ctypes.c_int32 * (B + 1))(*off)
    with torch.cuda.device(points.device):
        s = stream if stream is not None else torch.cuda.current_stream()
        o = _opts(n_vox, tile_points, cluster_size, block_threads, flags, s.cuda_stream, local_warps, cand_per_thread)
        h = lib.fps_index_build_ragged(points.data_ptr(), arr, B, ctypes.byref(o))
    if not h:
        raise FpsError(lib.fps_last_status(), fps_last_error())
    return Index(h, B, max(off[b + 1] - off[b] for b in range(B)), points.device, off)


def fps_sample_ragged(index: Index, M, start_idx=None, out_idx: torch.Tensor | None = None,
                      out_mindist: torch.Tensor | None = None, stream: torch.cuda.Stream | None = None):
    """fps_sample_ragged: per-cloud sample counts ``M`` (B ints) and start points (B ints or None = 0).
    Returns (out_idx int32 [sum M], out_mindist float32 [sum M], out_offsets list of B+1 ints); cloud b's
    samples are out[out_offsets[b]:out_offsets[b+1]], indices relative to the cloud's first point."""
    lib = load()
    if index.handle is None:
        raise ValueError("index was destroyed")
    Ms = [int(v) for v in M]
    if len(Ms) != index.B:
        raise ValueError("M must hold one entry per cloud")
    total = sum(max(m, 0) for m in Ms)
    marr = (ctypes.c_int32 * index.B)(*Ms)
    sarr = None
    if start_idx is not None:
        ss = [int(v) for v in start_idx]
        if len(ss) != index.B:
            raise ValueError("start_idx must hold one entry per cloud")
        sarr = (ctypes.c_int32 * index.B)(*ss)
    with torch.cuda.device(index.device):
        if out_idx is None:
            out_idx = torch.empty((total,), dtype=torch.int32, device=index.device)
        if out_mindist is None:
            out_mindist = torch.empty((total,), dtype=torch.float32, device=index.device)
        if out_idx.dtype != torch.int32 or out_mindist.dtype != torch.float32 or not out_idx.is_contiguous() \
                or not out_mindist.is_contiguous() or out_idx.numel() < total or out_mindist.numel() < total:
            raise ValueError("out_idx must be contiguous int32 [sum M] and out_mindist contiguous float32 [sum M]")
        s = stream if stream is not None else torch.cuda.current_stream()
        rc = lib.fps_sample_ragged(index.handle, marr, sarr, out_idx.data_ptr(), out_mindist.data_ptr(), s.cuda_stream)
    if rc != FPS_OK:
        raise FpsError(rc, fps_last_error())
    offs = [0]
    for m in Ms:
        offs.append(offs[-1] + m)
    return out_idx, out_mindist, offs


def fps_gather_xyz(index: Index, idx: torch.Tensor, M: int | None = None, stream: torch.cuda.Stream | None = None):
    """fps_gather_xyz: coordinates of the sampled points.  ``idx`` int32 [B,M] from fps_sample (M taken from
    its shape) or the flat tensor of the last fps_sample_ragged call (pass M=0).  Returns float32 [...,3]."""
    lib = load()
    if idx.dtype != torch.int32 or not idx.is_cuda or not idx.is_contiguous():
        raise ValueError("idx must be a contiguous CUDA int32 tensor")
    if M is None:
        M = idx.shape[-1] if idx.dim() == 2 else 0
    with torch.cuda.device(index.device):
        out = torch.empty(tuple(idx.shape) + (3,), dtype=torch.float32, device=index.device)
        s = stream if stream is not None else torch.cuda.current_stream()
        rc = lib.fps_gather_xyz(index.handle, idx.data_ptr(), int(M), out.data_ptr(), s.cuda_stream)
    if rc != FPS_OK:
        raise FpsError(rc, fps_last_error())
    return out


def fps_pick_chain_cycles(cand_per_lane: int = 2, iters: int = 8192) -> float:
    """fps_pick_chain_cycles: SM cycles per pick of the bare one-warp pick chain (the latency floor)."""
    out = ctypes.c_float(0.0)
    rc = load().fps_pick_chain_cycles(int(cand_per_lane), int(iters), ctypes.byref(out))
    if rc != FPS_OK:
        raise FpsError(rc, fps_last_error())
    return float(out.value)


def fps_index_destroy(index: Index) -> None:
    if index.handle is not None:
        load().fps_index_destroy(index.handle)
        index.handle = None


def fps_get_stats(index: Index) -> dict:
    st = fps_stats()
    rc = load().fps_get_stats(index.handle, ctypes.byref(st))
    if rc != FPS_OK:
        raise FpsError(rc, fps_last_error())
    return st.as_dict()


def fps_sample_host(points_host: torch.Tensor, M: int, start_idx: int = 0, *, n_vox: int = 0, tile_points: int = 0,
                    cluster_size: int = 0, block_threads: int = 0, flags: int = 0, local_warps: int = 0,
                    cand_per_thread: int = 0,
                    out_idx: torch.Tensor | None = None, out_mindist: torch.Tensor | None = None):
    """fps_sample_host: HOST float32 [B,N,3] in, HOST int32/float32 [B,M] out; copies, index build and
    sampling all happen inside the C call (synchronous)."""
    lib = load()
    if points_host.is_cuda:
        raise ValueError("fps_sample_host takes host tensors")
    B, N = _check_points(points_host)
    if out_idx is None:
        out_idx = torch.empty((B, M), dtype=torch.int32, pin_memory=torch.cuda.is_available())
    if out_mindist is None:
        out_mindist = torch.empty((B, M), dtype=torch.float32, pin_memory=torch.cuda.is_available())
    o = _opts(n_vox, tile_points, cluster_size, block_threads, flags, None, local_warps, cand_per_thread)
    rc = lib.fps_sample_host(points_host.data_ptr(), N, B, int(M), int(start_idx), out_idx.data_ptr(),
                             out_mindist.data_ptr(), ctypes.byref(o))
    if rc != FPS_OK:
        raise FpsError(rc, fps_last_error())
    return out_idx, out_mindist


def fps_build_and_sample(points: torch.Tensor, M, *, offsets=None, start_idx=None, chunk_clouds: int = 0, n_vox: int = 0,
                         tile_points: int = 0, cluster_size: int = 0, block_threads: int = 0, flags: int = 0,
                         local_warps: int = 0, cand_per_thread: int = 0, out_idx: torch.Tensor | None = None,
                         out_mindist: torch.Tensor | None = None, stream: torch.cuda.Stream | None = None):
    """fps_build_and_sample: the one-shot call; the index of chunk k+1 is built while chunk k is sampled.
    ``points``: CUDA float32 [B,N,3], or [T,3] with ``offsets`` (B+1 ints).  ``M``: one int for all clouds or
    B ints; ``start_idx``: None (= 0) or B ints.  Returns (out_idx, out_mindist) shaped [B,M] when M is one
    int, else flat [sum M] plus the list of output offsets.  Results are ordered on ``stream``."""
    lib = load()
    if not points.is_cuda:
        raise ValueError("points must live on a CUDA device")
    if offsets is None:
        B, N = _check_points(points)
        oarr = None
    else:
        if points.dtype != torch.float32 or not points.is_contiguous() or points.dim() != 2 or points.shape[1] != 3:
            raise ValueError("points must be a contiguous CUDA float32 tensor [T,3]")
        off = [int(v) for v in offsets]
        if len(off) < 2 or off[-1] != points.shape[0]:
            raise ValueError("offsets must hold B+1 entries and end at the number of points")
        B, N = len(off) - 1, 0
        oarr = (ctypes.c_int32 * (B + 1))(*off)
    uniform = isinstance(M, int)
    Ms = [int(M)] * B if uniform else [int(v) for v in M]
    if len(Ms) != B:
        raise ValueError("M must be one int or hold one entry per cloud")
    marr = None if uniform else (ctypes.c_int32 * B)(*Ms)
    sarr = None
    if start_idx is not None:
        ss = [int(v) for v in start_idx]
        if len(ss) != B:
            raise ValueError("start_idx must hold one entry per cloud")
        sarr = (ctypes.c_int32 * B)(*ss)
    total = sum(max(m, 0) for m in Ms)
    shape = (B, max(Ms[0], 0)) if uniform else (total,)
    with torch.cuda.device(points.device):
        if out_idx is None:
            out_idx = torch.empty(shape, dtype=torch.int32, device=points.device)
        if out_mindist is None:
            out_mindist = torch.empty(shape, dtype=torch.float32, device=points.device)
        if out_idx.dtype != torch.int32 or out_mindist.dtype != torch.float32 or not out_idx.is_contiguous() \
                or not out_mindist.is_contiguous() or out_idx.numel() < total or out_mindist.numel() < total:
            raise ValueError("out_idx must be contiguous int32 and out_mindist contiguous float32, sum M entries each")
        s = stream if stream is not None else torch.cuda.current_stream()
        o = _opts(n_vox, tile_points, cluster_size, block_threads, flags, s.cuda_stream, local_warps, cand_per_thread)
        rc = lib.fps_build_and_sample(points.data_ptr(), oarr, N, B, marr, Ms[0] if uniform else 0, sarr,
                                      out_idx.data_ptr(), out_mindist.data_ptr(), ctypes.byref(o), int(chunk_clouds))
    if rc != FPS_OK:
        raise FpsError(rc, fps_last_error())
    if uniform:
        return out_idx, out_mindist
    offs = [0]
    for m in Ms:
        offs.append(offs[-1] + m)
    return out_idx, out_mindist, offs
