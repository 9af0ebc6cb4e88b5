"""Seeded synthetic point clouds shaped like the paper's workloads.

This module holds NO arithmetic of the sampling method (no distances between points, no voxel
grid, no argmax): it only draws inputs.  It is the one module both the CPU oracle's tests and the
CUDA path's tests/bench import, so that both sides see the same bytes.  It imports neither
``oracle`` nor the CUDA binding.

The paper measures on S3DIS, ScanNet, SemanticKITTI and the Stanford dragon;
none is available here, so the five configurations of BASELINE.json stand in for them
(recipe: DESIGN.md "Input recipe").  All maths is float64 NumPy with
``default_rng(seed)``; the result is cast to float32 at the end.  Cloud ``b`` of a batch uses
``seed + b``.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

BASE_SEED = 1234


@dataclass(frozen=True)
class Workload:
    name: str
    kind: str          # "uniform" | "room" | "lidar"
    B: int
    N: int
    M: int
    start_idx: int
    params: tuple      # generator parameters, see make_cloud
    note: str


# ----------------------------------------------------------------------------------------------
# generators
# ----------------------------------------------------------------------------------------------
def uniform_cube(N: int, seed: int) -> np.ndarray:
    """C1: N x 3 i.i.d. U[0,1) float32."""
    rng = np.random.default_rng(seed)
    return rng.random((N, 3), dtype=np.float32)


def _sample_rect(rng, n, origin, eu, ev):
    """n points uniform on the parallelogram origin + s*eu + t*ev, s,t in [0,1)."""
    s = rng.random(n)[:, None]
    t = rng.random(n)[:, None]
    return origin[None, :] + s * eu[None, :] + t * ev[None, :]


def room(N: int, seed: int, size=(10.0, 8.0, 3.0), n_boxes: int = 20, jitter: float = 0.005,
         dense_half: bool = False) -> np.ndarray:
    """Indoor-room-like cloud (C2, C3): floor, ceiling, 4 walls of a W x D x H box room plus
    ``n_boxes`` axis-aligned boxes (sides U[0.3, 2] m, 5 faces, standing on the floor, fully
    inside, may overlap), points uniform by area, Gaussian jitter ``jitter`` m per coordinate.
    ``dense_half``: half of the room (x < W/2) is sampled at 4x the rate of the other half
    (rejection: a candidate with x >= W/2 is kept with probability 1/4)."""
    rng = np.random.default_rng(seed)
    W, D, H = size
    rects = []  # (origin, eu, ev)
    z0 = np.zeros(3)
    ex, ey, ez = np.array([W, 0, 0.0]), np.array([0, D, 0.0]), np.array([0, 0, H])
    rects.append((z0, ex, ey))                         # floor
    rects.append((np.array([0, 0, H]), ex, ey))        # ceiling
    rects.append((z0, ex, ez))                         # wall y=0
    rects.append((np.array([0, D, 0.0]), ex, ez))      # wall y=D
    rects.append((z0, ey, ez))                         # wall x=0
    rects.append((np.array([W, 0, 0.0]), ey, ez))      # wall x=W
    for _ in range(n_boxes):
        sx, sy, sz = rng.uniform(0.3, 2.0, size=3)
        sz = min(sz, H)
        ox = rng.uniform(0.0, W - sx)
        oy = rng.uniform(0.0, D - sy)
        o = np.array([ox, oy, 0.0])
        bx, by, bz = np.array([sx, 0, 0.0]), np.array([0, sy, 0.0]), np.array([0, 0, sz])
        rects.append((o + bz, bx, by))                 # top
        rects.append((o, bx, bz))                      # side y=oy
        rects.append((o + by, bx, bz))                 # side y=oy+sy
        rects.append((o, by, bz))                      # side x=ox
        rects.append((o + bx, by, bz))                 # side x=ox+sx
    areas = np.array([np.linalg.norm(np.cross(eu, ev)) for _, eu, ev in rects])
    prob = areas / areas.sum()
    out = np.empty((0, 3))
    while out.shape[0] < N:
        want = int((N - out.shape[0]) * (1.8 if dense_half else 1.0)) + 64
        which = rng.choice(len(rects), size=want, p=prob)
        pts = np.empty((want, 3))
        for r, (o, eu, ev) in enumerate(rects):
            m = which == r
            c = int(m.sum())
            if c:
                pts[m] = _sample_rect(rng, c, o, eu, ev)
        if dense_half:
            keep = (pts[:, 0] < W / 2) | (rng.random(want) < 0.25)
            pts = pts[keep]
        out = np.concatenate([out, pts], axis=0)
    out = out[:N]
    out = out + rng.normal(0.0, jitter, size=out.shape)
    return out.astype(np.float32)


def _ray_hits(dirs, origin_z, boxes, cyls, max_range):
    """First-hit range of rays from (0,0,origin_z) along unit ``dirs`` [n,3] against the ground
    plane z=0, axis-aligned boxes (cx,cy,sx,sy,h) standing on the ground, and vertical cylinders
    (cx,cy,r,h) (side surface only).  inf where nothing is hit within max_range."""
    n = dirs.shape[0]
    dx, dy, dz = dirs[:, 0], dirs[:, 1], dirs[:, 2]
    t = np.full(n, np.inf)
    with np.errstate(divide="ignore", invalid="ignore"):
        tg = np.where(dz < 0, origin_z / -dz, np.inf)
        t = np.minimum(t, tg)
        inv = [1.0 / dx, 1.0 / dy, 1.0 / dz]
        o = (0.0, 0.0, origin_z)
        for (cx, cy, sx, sy, h) in boxes:
            lo = (cx - sx / 2, cy - sy / 2, 0.0)
            hi = (cx + sx / 2, cy + sy / 2, h)
            tmin = np.full(n, -np.inf)
            tmax = np.full(n, np.inf)
            for a in range(3):
                t1 = (lo[a] - o[a]) * inv[a]
                t2 = (hi[a] - o[a]) * inv[a]
                tmin = np.maximum(tmin, np.minimum(t1, t2))
                tmax = np.minimum(tmax, np.maximum(t1, t2))
            hit = (tmax >= tmin) & (tmin > 0)
            t = np.where(hit & (tmin < t), tmin, t)
        for (cx, cy, r, h) in cyls:
            a = dx * dx + dy * dy
            b = -2.0 * (dx * cx + dy * cy)
            c = cx * cx + cy * cy - r * r
            disc = b * b - 4 * a * c
            sq = np.sqrt(np.where(disc > 0, disc, np.nan))
            tc = (-b - sq) / (2 * a)
            zc = origin_z + tc * dz
            hit = np.isfinite(tc) & (tc > 0) & (zc >= 0) & (zc <= h)
            t = np.where(hit & (tc < t), tc, t)
    t = np.where(t <= max_range, t, np.inf)
    return t


def lidar(N: int, seed: int, n_beams: int = 64, elev_deg=(-25.0, 3.0), n_azimuth: int = 1875,
          n_objects: int = 40, max_range: float = 80.0, sensor_h: float = 1.73,
          range_sigma: float = 0.02) -> np.ndarray:
    """Outdoor spinning-LiDAR-like cloud (C4, C5).  ``n_beams`` elevations linearly spaced over
    ``elev_deg``, ``n_azimuth`` azimuth steps; rays from (0,0,sensor_h) hit the ground plane or
    ``n_objects`` objects (half boxes 1.5-5 x 1.5-2.5 x 1.2-2.5 m, half vertical cylinders r
    0.1-0.4 m, h 3-8 m; centres uniform in the disc of radius max_range, rejected unless the whole
    object is >= 4 m from the sensor axis); first hit kept, Gaussian range noise, returns beyond
    max_range dropped.  If the regular sweep yields fewer than N returns, rays with a random beam
    and a continuous random azimuth are added until N; if more, the first N of a random
    permutation are kept.  Final order is shuffled."""
    rng = np.random.default_rng(seed)
    boxes, cyls = [], []
    for k in range(n_objects):
        while True:
            rad = max_range * np.sqrt(rng.random())
            ang = rng.uniform(0, 2 * np.pi)
            cx, cy = rad * np.cos(ang), rad * np.sin(ang)
            if k % 2 == 0:
                sx, sy, h = rng.uniform(1.5, 5.0), rng.uniform(1.5, 2.5), rng.uniform(1.2, 2.5)
                reach = 0.5 * np.hypot(sx, sy)
                obj = (cx, cy, sx, sy, h)
            else:
                r, h = rng.uniform(0.1, 0.4), rng.uniform(3.0, 8.0)
                reach = r
                obj = (cx, cy, r, h)
            if rad - reach >= 4.0:
                (boxes if k % 2 == 0 else cyls).append(obj)
                break
    elev = np.deg2rad(np.linspace(elev_deg[0], elev_deg[1], n_beams))

    def cast(el, az):
        d = np.stack([np.cos(el) * np.cos(az), np.cos(el) * np.sin(az), np.sin(el)], axis=1)
        out = []
        for s in range(0, d.shape[0], 1 << 18):
            dd = d[s:s + (1 << 18)]
            t = _ray_hits(dd, sensor_h, boxes, cyls, max_range)
            ok = np.isfinite(t)
            tn = t[ok] + rng.normal(0.0, range_sigma, size=int(ok.sum()))
            p = dd[ok] * tn[:, None]
            p[:, 2] += sensor_h
            out.append(p)
        return np.concatenate(out, axis=0) if out else np.empty((0, 3))

    az_grid = np.arange(n_azimuth) * (2 * np.pi / n_azimuth)
    el_all = np.repeat(elev, n_azimuth)
    az_all = np.tile(az_grid, n_beams)
    pts = cast(el_all, az_all)
    if pts.shape[0] > N:
        pts = pts[rng.permutation(pts.shape[0])[:N]]
    while pts.shape[0] < N:
        want = int((N - pts.shape[0]) * 1.3) + 256
        el = elev[rng.integers(0, n_beams, size=want)]
        az = rng.uniform(0, 2 * np.pi, size=want)
        extra = cast(el, az)
        pts = np.concatenate([pts, extra[: N - pts.shape[0]]], axis=0)
    pts = pts[rng.permutation(N)]
    return pts.astype(np.float32)


# ----------------------------------------------------------------------------------------------
# tie-heavy / degenerate inputs used by the pins and the parity edge cases
# ----------------------------------------------------------------------------------------------
def integer_line(N: int) -> np.ndarray:
    """Points (i, 0, 0), i = 0..N-1 (exactly representable; many exact ties)."""
    p = np.zeros((N, 3), dtype=np.float32)
    p[:, 0] = np.arange(N, dtype=np.float32)
    return p


def cube_corners() -> np.ndarray:
    """The 8 corners of {0,1}^3, index = 4x + 2y + z."""
    return np.array([[(i >> 2) & 1, (i >> 1) & 1, i & 1] for i in range(8)], dtype=np.float32)


def shuffled_lattice(n: int, seed: int, step: float = 0.1) -> np.ndarray:
    """n^3 lattice points (i,j,k) * float32(step), in a seeded random order.  With step = 0.1f the
    coordinates are inexact in fp32, so squared distances carry rounding that differs between
    arithmetic variants (sqrt / FMA / re-association) while exact ties stay plentiful."""
    rng = np.random.default_rng(seed)
    g = np.arange(n, dtype=np.float32) * np.float32(step)
    p = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3).astype(np.float32)
    return p[rng.permutation(p.shape[0])]


def with_duplicates(N: int, seed: int, n_unique: int) -> np.ndarray:
    """N points drawn (with repetition) from n_unique distinct uniform points: exact duplicates."""
    rng = np.random.default_rng(seed)
    base = rng.random((n_unique, 3), dtype=np.float32)
    return base[rng.integers(0, n_unique, size=N)]


def clustered(N: int, seed: int, n_clusters: int = 8, sigma: float = 0.01) -> np.ndarray:
    """Gaussian blobs in the unit cube: strongly non-uniform density (voxel load imbalance)."""
    rng = np.random.default_rng(seed)
    c = rng.random((n_clusters, 3))
    which = rng.integers(0, n_clusters, size=N)
    return (c[which] + rng.normal(0, sigma, size=(N, 3))).astype(np.float32)


# ----------------------------------------------------------------------------------------------
# the five BASELINE.json configurations (+ reduced versions for CPU-time tests)
# ----------------------------------------------------------------------------------------------
WORKLOADS = {
    "C1": Workload("C1", "uniform", 1, 4096, 1024, 0, (),
                   "single cloud, N=4096 i.i.d. uniform in [0,1)^3, M=1024"),
    "C2": Workload("C2", "room", 16, 24000, 6000, 0, ((10.0, 8.0, 3.0), 20, False),
                   "indoor-room-like batch: B=16, N=24000, 10x8x3 m room + 20 boxes, jitter 5 mm, M=N/4"),
    "C3": Workload("C3", "room", 1, 150000, 37500, 0, ((20.0, 15.0, 3.0), 60, True),
                   "large indoor scene: N=150000, 20x15x3 m room + 60 boxes, 4x density in half the room, M=N/4"),
    "C4": Workload("C4", "lidar", 4, 120000, 30000, 0, (64, (-25.0, 3.0), 1875, 40, 80.0),
                   "outdoor LiDAR-like: B=4, N=120000, 64 beams x 1875 azimuths, 40 objects within 80 m, M=N/4"),
    "C5": Workload("C5", "lidar", 1, 1000000, 65536, 0, (128, (-25.0, 15.0), 7813, 200, 120.0),
                   "stress: N=1000000, 128 beams x 7813 azimuths, 200 objects within 120 m, M=65536"),
}

# not a BASELINE.json configuration: the parity case for clouds so large that the library's automatic tile size
# grows past 64 points per voxel (tests/test_gpu_parity.py, golden hash in tests/golden/full_size.json)
EXTRA_WORKLOADS = {
    "L3M": Workload("L3M", "lidar", 1, 3000000, 20000, 0, (128, (-25.0, 15.0), 23439, 200, 120.0),
                    "parity case: N=3000000, 128 beams x 23439 azimuths, 200 objects within 120 m, M=20000"),
}


def scaled(name: str, N: int, M: int, B: int | None = None) -> Workload:
    """The same generator as workload ``name`` at a reduced size (for CPU-time parity cases)."""
    w = WORKLOADS[name]
    params = w.params
    if w.kind == "lidar":
        # keep the beam count, shrink the azimuth count so the regular sweep still yields ~N rays
        beams, elev, _, nobj, rng_ = params
        params = (beams, elev, max(8, N // beams), nobj, rng_)
    return Workload(f"{name}@{N}", w.kind, w.B if B is None else B, N, M, w.start_idx, params,
                    f"reduced {name}: N={N}, M={M}")


def make_cloud(w: Workload, b: int = 0, seed: int = BASE_SEED) -> np.ndarray:
    s = seed + b
    if w.kind == "uniform":
        return uniform_cube(w.N, s)
    if w.kind == "room":
        size, n_boxes, dense = w.params
        return room(w.N, s, size=size, n_boxes=n_boxes, dense_half=dense)
    if w.kind == "lidar":
        beams, elev, n_az, nobj, max_range = w.params
        return lidar(w.N, s, n_beams=beams, elev_deg=elev, n_azimuth=n_az, n_objects=nobj,
                     max_range=max_range)
    raise ValueError(w.kind)


def make_batch(w: Workload | str, seed: int = BASE_SEED) -> np.ndarray:
    """[B][N][3] float32, C-contiguous."""
    if isinstance(w, str):
        w = WORKLOADS[w] if w in WORKLOADS else EXTRA_WORKLOADS[w]
    return np.ascontiguousarray(np.stack([make_cloud(w, b, seed) for b in range(w.B)], axis=0))
