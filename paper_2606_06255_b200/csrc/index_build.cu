// index_build.cu -- steps a1-a6 of the hot path: the on-device spherical-voxel index.
//
// Follows Alg. 2 Phases 1-3 of the paper and Eq. 6-10:
//   a1 bounding box           Eq. 6-7   (k_bbox)
//   a2 voxel id per point     Eq. 8, 31 (k_keys)
//   a3 radix sort by voxel id Alg. 2 l.11 (radix_sort_pairs: hand-written stable LSD radix sort)
//   a4 gather AoS -> SoA      Alg. 2 Phase 2 (k_gather)
//   a5 active-voxel segments  Alg. 2 Phase 3 (k_heads + scan + k_voxel_segments)
//   a6 per-voxel sphere       Eq. 10 / north_star "per-voxel center, radius" (k_sphere)
// What differs from the paper:
//   * the sort key carries a few Morton bits of the position INSIDE the voxel below V_id, so that
//     a voxel holding more than `tile_points` points can be cut into spatially compact tiles;
//     every tile is a "spherical voxel" of its own (own centre, own tight radius).  Any
//     partition with conservative spheres leaves the result unchanged (Eq. 20-26).
//   * c_k is the midpoint of the tile's own bounding box and r_k its tight radius rounded up,
//     instead of the cell centre and sqrt(3)/2 L (reading A10).
#include <cfloat>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <utility>
#include <vector>

#include "device_utils.cuh"
#include "internal.h"

namespace rfps {

// ---------------------------------------------------------------------------------------------
// small helpers
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned f2ord(float f)
{   // monotone map float -> uint (for atomicMin/Max on floats of either sign)
    unsigned u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float ord2f(unsigned u)
{
    return __uint_as_float((u & 0x80000000u) ? (u & 0x7fffffffu) : ~u);
}

// ---------------------------------------------------------------------------------------------
// Programmatic dependent launch: the build is a chain of ~20 short kernels, each depending on the one
// before it; every kernel lets its successor be scheduled at once (launch_dependents) and then waits for
// the complete predecessor grid and its memory (wait) before it touches anything, so the order of all
// memory operations is the stream order, and only the launch latency of the successor is overlapped.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void grid_dep_sync()
{
    asm volatile("griddepcontrol.launch_dependents;");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}
// Launch bookkeeping of ONE build (a local of build_index, passed down): kernels launched so far and the first
// launch error, checked once after the chain has been enqueued.
struct LaunchLog {
    int launches = 0;
    cudaError_t first_error = cudaSuccess;
};

template <typename... P, typename... A>
static void launch_pdl_smem(LaunchLog &log, size_t smem, void (*kern)(P...), dim3 grid, dim3 block, cudaStream_t st, A &&...args);

// the same with a thread-block cluster dimension (the single-launch build of mid-size clouds)
template <typename... P, typename... A>
static void launch_pdl_cluster(LaunchLog &log, size_t smem, int cluster, void (*kern)(P...), dim3 grid, dim3 block, cudaStream_t st, A &&...args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[2];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    at[1].id = cudaLaunchAttributeClusterDimension;
    at[1].val.clusterDim.x = (unsigned)cluster;
    at[1].val.clusterDim.y = 1;
    at[1].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 2;
    const cudaError_t e = cudaLaunchKernelEx(&cfg, kern, std::forward<A>(args)...);
    if (e != cudaSuccess && log.first_error == cudaSuccess) log.first_error = e;
    log.launches += 1;
}

template <typename... P, typename... A>
static void launch_pdl(LaunchLog &log, void (*kern)(P...), dim3 grid, dim3 block, cudaStream_t st, A &&...args)
{
    launch_pdl_smem(log, 0, kern, grid, block, st, std::forward<A>(args)...);
}

template <typename... P, typename... A>
static void launch_pdl_smem(LaunchLog &log, size_t smem, void (*kern)(P...), dim3 grid, dim3 block, cudaStream_t st, A &&...args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    const cudaError_t e = cudaLaunchKernelEx(&cfg, kern, std::forward<A>(args)...);
    if (e != cudaSuccess && log.first_error == cudaSuccess) log.first_error = e;
    log.launches += 1;
}

// ---------------------------------------------------------------------------------------------
// a1: bounding box (Eq. 6) + non-finite detection.  bbox[b] = {minx,miny,minz,maxx,maxy,maxz} as
// order-preserving uints; bbox[b][6] = non-finite flag.
// ---------------------------------------------------------------------------------------------
constexpr int BBOX_STRIDE = 8;

__global__ void k_bbox_init(unsigned *bbox, int B)
{
    grid_dep_sync();
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < B * BBOX_STRIDE) {
        int c = i % BBOX_STRIDE;
        bbox[i] = c < 3 ? 0xFFFFFFFFu : 0u;
    }
}

// Clouds may differ in size (ragged batches): cloud b holds the points [poff[b], poff[b+1]) of the
// concatenated arrays.  Every kernel below takes `poff`; grids are sized for the largest cloud.
__global__ void __launch_bounds__(256) k_bbox(const float *__restrict__ pts, const int *__restrict__ poff, unsigned *bbox)
{
    grid_dep_sync();
    const int b = blockIdx.y;
    const int base = poff[b], N = poff[b + 1] - base;
    const float *P = pts + (size_t)base * 3;
    float mn[3] = {FLT_MAX, FLT_MAX, FLT_MAX}, mx[3] = {-FLT_MAX, -FLT_MAX, -FLT_MAX};
    bool bad = false;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < N; i += gridDim.x * blockDim.x) {
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            float v = P[3 * (size_t)i + a];
            bad |= !(fabsf(v) <= FLT_MAX);   // NaN or inf
            mn[a] = fminf(mn[a], v);
            mx[a] = fmaxf(mx[a], v);
        }
    }
#pragma unroll
    for (int a = 0; a < 3; ++a)
        for (int o = 16; o > 0; o >>= 1) {
            mn[a] = fminf(mn[a], __shfl_xor_sync(0xffffffffu, mn[a], o));
            mx[a] = fmaxf(mx[a], __shfl_xor_sync(0xffffffffu, mx[a], o));
        }
    bad = __any_sync(0xffffffffu, bad);
    // block level through shared memory, then ONE set of atomics per block (the atomics on a handful of
    // addresses were most of this kernel's time when every warp issued them)
    __shared__ float smn[8][3], smx[8][3];
    __shared__ int sbad;
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) sbad = 0;
    __syncthreads();
    if (lane == 0) {
#pragma unroll
        for (int a = 0; a < 3; ++a) { smn[w][a] = mn[a]; smx[w][a] = mx[a]; }
        if (bad) sbad = 1;
    }
    __syncthreads();
    if (threadIdx.x < 3) {
        const int a = threadIdx.x;
        float lo = smn[0][a], hi = smx[0][a];
        for (int i = 1; i < 8; ++i) { lo = fminf(lo, smn[i][a]); hi = fmaxf(hi, smx[i][a]); }
        unsigned *bb = bbox + b * BBOX_STRIDE;
        if (lo <= hi) {
            atomicMin(bb + a, f2ord(lo));
            atomicMax(bb + 3 + a, f2ord(hi));
        }
        if (a == 0 && sbad) atomicOr(bb + 6, 1u);
    }
}

// ---------------------------------------------------------------------------------------------
// a2: sort key per point.  key = V_id << (3*sb) | morton(sub-cell); val = i.
// Voxel coordinates per Eq. 8 (floor, then clamp; reading A14); L per Eq. 7 with alpha = 1 + 1e-3.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned spread3(unsigned v)
{   // 0b abcd -> 0b a00b00c00d (up to 10 bits)
    v &= 0x3ffu;
    v = (v | (v << 16)) & 0x030000ffu;
    v = (v | (v << 8)) & 0x0300f00fu;
    v = (v | (v << 4)) & 0x030c30c3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}

// Hilbert index of a cell with `b` bits per axis (Skilling's transpose construction, "Programming the
// Hilbert curve", 2004): undo the excess work of the Gray-code walk, Gray-encode, interleave.
__device__ __forceinline__ unsigned hilbert3(unsigned x, unsigned y, unsigned z, int b)
{
    if (b <= 0) return 0u;
    unsigned X[3] = {x, y, z};
    const unsigned M = 1u << (b - 1);
    for (unsigned Q = M; Q > 1u; Q >>= 1) {
        const unsigned P = Q - 1u;
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            if (X[i] & Q) X[0] ^= P;
            else { const unsigned t = (X[0] ^ X[i]) & P; X[0] ^= t; X[i] ^= t; }
        }
    }
    X[1] ^= X[0];
    X[2] ^= X[1];
    unsigned t = 0u;
    for (unsigned Q = M; Q > 1u; Q >>= 1)
        if (X[2] & Q) t ^= Q - 1u;
    X[0] ^= t; X[1] ^= t; X[2] ^= t;
    return (spread3(X[0]) << 2) | (spread3(X[1]) << 1) | spread3(X[2]);
}

__global__ void __launch_bounds__(256) k_keys(const float *__restrict__ pts, const int *__restrict__ poff,
                                               const unsigned *__restrict__ bbox, int n_vox, int hb, int sb,
                                               unsigned *__restrict__ keys, int *__restrict__ vals)
{
    grid_dep_sync();
    const int b = blockIdx.y;
    const int base = poff[b], N = poff[b + 1] - base;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const unsigned *bb = bbox + b * BBOX_STRIDE;
    const float lo[3] = {ord2f(bb[0]), ord2f(bb[1]), ord2f(bb[2])};
    const float hi[3] = {ord2f(bb[3]), ord2f(bb[4]), ord2f(bb[5])};
    float E = fmaxf(fmaxf(hi[0] - lo[0], hi[1] - lo[1]), hi[2] - lo[2]);
    float L = (1.0f + 1e-3f) * E / (float)n_vox;
    if (!(L > 0.0f)) L = 1.0f;
    const float invsub = (float)(1 << sb);
    unsigned v[3], s[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        float t = (pts[((size_t)base + i) * 3 + a] - lo[a]) / L;
        float f = floorf(t);
        int c = (int)f;
        c = max(0, min(n_vox - 1, c));
        int sc = (int)floorf((t - (float)c) * invsub);
        sc = max(0, min((1 << sb) - 1, sc));
        v[a] = (unsigned)c;
        s[a] = (unsigned)sc;
    }
    // voxel id: the position of (v_x, v_y, v_z) on a 3-D Hilbert curve instead of the row-major id of
    // Eq. 31 -- any bijective id gives the same voxels.  Consecutive cells of the curve are face
    // neighbours (no seams as in Morton order), so 32 consecutive active voxels stay spatially compact,
    // which the sampling kernel's group-level prune relies on.
    unsigned vid = hilbert3(v[0], v[1], v[2], hb);
    unsigned sub = sb ? (spread3(s[0]) | (spread3(s[1]) << 1) | (spread3(s[2]) << 2)) : 0u;
    keys[(size_t)base + i] = (vid << (3 * sb)) | sub;
    vals[(size_t)base + i] = i;
}

// ---------------------------------------------------------------------------------------------
// batched exclusive scan of int32: three kernels (block sums, scan of block sums, apply)
// ---------------------------------------------------------------------------------------------
constexpr int SCAN_T = 256, SCAN_ITEMS = 8, SCAN_TILE = SCAN_T * SCAN_ITEMS;

__device__ __forceinline__ int block_excl_scan(int v, int *total, int *sm /*[33]*/)
{   // exclusive scan of one int per thread across a 256-thread block
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) sm[w] = inc;
    __syncthreads();
    if (w == 0) {
        int s = lane < (SCAN_T / 32) ? sm[lane] : 0;
        int si = s;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, si, o);
            if (lane >= o) si += t;
        }
        if (lane < (SCAN_T / 32)) sm[lane] = si - s;
        if (lane == 31) sm[32] = si;
    }
    __syncthreads();
    int r = inc - v + sm[w];
    *total = sm[32];
    __syncthreads();
    return r;
}

// `poff` != nullptr: array b is the ragged segment [poff[b], poff[b+1]) (n and stride are ignored)
__global__ void __launch_bounds__(SCAN_T) k_scan_blocksum(const int *__restrict__ in, int n, int stride, int nblk,
                                                           int *__restrict__ bsum, const int *__restrict__ poff)
{
    grid_dep_sync();
    __shared__ int sm[33];
    const int b = blockIdx.y;
    const int *src = in + (poff ? (size_t)poff[b] : (size_t)b * stride);
    if (poff) n = poff[b + 1] - poff[b];
    int base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
    int s = 0;
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i)
        if (base + i < n) s += src[base + i];
    int tot;
    block_excl_scan(s, &tot, sm);
    if (threadIdx.x == 0) bsum[(size_t)b * nblk + blockIdx.x] = tot;
}

__global__ void __launch_bounds__(SCAN_T) k_scan_bsums(int *bsum, int nblk, int *totals)
{
    grid_dep_sync();
    __shared__ int sm[33];
    const int b = blockIdx.x;
    int *s = bsum + (size_t)b * nblk;
    int carry = 0;
    for (int base = 0; base < nblk; base += SCAN_T) {
        int i = base + threadIdx.x;
        int v = i < nblk ? s[i] : 0;
        int tot;
        int e = block_excl_scan(v, &tot, sm);
        if (i < nblk) s[i] = e + carry;
        carry += tot;
    }
    if (threadIdx.x == 0 && totals) totals[b] = carry;
}

__global__ void __launch_bounds__(SCAN_T) k_scan_apply(const int *__restrict__ in, int *__restrict__ out, int n, int stride,
                                                        int nblk, const int *__restrict__ bsum, const int *__restrict__ poff)
{
    grid_dep_sync();
    __shared__ int sm[33];
    const int b = blockIdx.y;
    const size_t off = poff ? (size_t)poff[b] : (size_t)b * stride;
    if (poff) n = poff[b + 1] - poff[b];
    const int *src = in + off;
    int *dst = out + off;
    int base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
    int v[SCAN_ITEMS], s = 0;
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) {
        v[i] = base + i < n ? src[base + i] : 0;
        s += v[i];
    }
    int tot;
    int e = block_excl_scan(s, &tot, sm) + bsum[(size_t)b * nblk + blockIdx.x];
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) {
        if (base + i < n) dst[base + i] = e;
        e += v[i];
    }
}

// exclusive scan of B arrays of n ints (per-array stride `stride`); totals[b] (device, may be null)

// short arrays: the whole scan of one array in ONE block (1024 threads x 4 items per step, running carry);
// one launch instead of three, which is what a build of a small cloud is made of
constexpr int SCAN1_T = 1024, SCAN1_ITEMS = 4, SCAN1_TILE = SCAN1_T * SCAN1_ITEMS, SCAN1_MAX_N = 32768;

__global__ void __launch_bounds__(SCAN1_T) k_scan_single(const int *__restrict__ in, int *__restrict__ out, int n, int stride,
                                                         int *__restrict__ totals, const int *__restrict__ poff)
{
    grid_dep_sync();
    __shared__ int wsum[32];
    __shared__ int carry_s;
    const int b = blockIdx.x, lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const size_t off = poff ? (size_t)poff[b] : (size_t)b * stride;
    if (poff) n = poff[b + 1] - poff[b];
    const int *src = in + off;
    int *dst = out + off;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    // the steps are serially dependent through the carry: the next step's items are loaded before this
    // step's barriers so that their memory latency is not on that chain
    int nx[SCAN1_ITEMS];
#pragma unroll
    for (int i = 0; i < SCAN1_ITEMS; ++i) {
        const int q = threadIdx.x * SCAN1_ITEMS + i;
        nx[i] = q < n ? src[q] : 0;
    }
    for (int base = 0; base < n; base += SCAN1_TILE) {
        const int i0 = base + threadIdx.x * SCAN1_ITEMS;
        int v[SCAN1_ITEMS], s = 0;
#pragma unroll
        for (int i = 0; i < SCAN1_ITEMS; ++i) {
            v[i] = nx[i];
            s += v[i];
        }
#pragma unroll
        for (int i = 0; i < SCAN1_ITEMS; ++i) {
            const int q = i0 + SCAN1_TILE + i;
            nx[i] = q < n ? src[q] : 0;
        }
        int inc = s;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) wsum[w] = inc;
        __syncthreads();
        const int carry = carry_s;
        if (w == 0) {
            int ws = wsum[lane], wi = ws;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, wi, o);
                if (lane >= o) wi += t;
            }
            wsum[lane] = wi - ws;                      // exclusive warp offsets
            if (lane == 31) carry_s = carry + wi;      // running total for the next step
        }
        __syncthreads();
        int e = carry + wsum[w] + inc - s;
#pragma unroll
        for (int i = 0; i < SCAN1_ITEMS; ++i) {
            if (i0 + i < n) dst[i0 + i] = e;
            e += v[i];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0 && totals) totals[b] = carry_s;
}

// n = length of every array, or (poff given) of the longest one
static void scan_exclusive(LaunchLog &log, const int *in, int *out, int n, int stride, int B, int *totals, int *bsum_tmp,
                           cudaStream_t st, const int *poff = nullptr)
{
    if (n <= SCAN1_MAX_N) {
        launch_pdl(log, k_scan_single, dim3(B), dim3(SCAN1_T), st, in, out, n, stride, totals, poff);
        return;
    }
    const int nblk = (n + SCAN_TILE - 1) / SCAN_TILE;
    launch_pdl(log, k_scan_blocksum, dim3(dim3(nblk, B)), dim3(SCAN_T), st, in, n, stride, nblk, bsum_tmp, poff);
    launch_pdl(log, k_scan_bsums, dim3(B), dim3(SCAN_T), st, bsum_tmp, nblk, totals);
    launch_pdl(log, k_scan_apply, dim3(dim3(nblk, B)), dim3(SCAN_T), st, in, out, n, stride, nblk, bsum_tmp, poff);
}
static inline int scan_tmp_ints(int n, int B) { return ((n + SCAN_TILE - 1) / SCAN_TILE) * B + 1; }

// ---------------------------------------------------------------------------------------------
// a3: stable LSD radix sort of (key, val) pairs, 8 bits per pass, batched over clouds.
// One warp owns a chunk of RS_CHUNK consecutive keys; its 256 digit counters live in shared
// memory.  The counter table is digit-major ([digit][chunk]) so that one exclusive scan gives
// every (digit, chunk) its global output offset.  Stability: chunks are ordered by the table
// layout, rounds inside a chunk run in order, lanes inside a round are ranked by lane id
// (__match_any_sync + popc of lower lanes).
// ---------------------------------------------------------------------------------------------
constexpr int RS_CHUNK = 512, RS_WARPS = 4;

// the lanes of the warp that hold the same 8-bit digit as this one (valid lanes only): eight ballots, one per bit.
// (`__match_any_sync` does the same in one instruction, but measured several hundred cycles per call on B200: the
// ranking loop below is a chain of them.)
__device__ __forceinline__ unsigned same_digit_lanes(const unsigned d, const bool valid)
{
    unsigned peers = __ballot_sync(0xffffffffu, valid);
#pragma unroll
    for (int bit = 0; bit < 8; ++bit) {
        const bool one = (d >> bit) & 1u;
        const unsigned bal = __ballot_sync(0xffffffffu, one);
        peers &= one ? bal : ~bal;
    }
    return peers;
}    // short chunks: enough warps in flight on small clouds too

__global__ void __launch_bounds__(RS_WARPS * 32) k_radix_hist(const unsigned *__restrict__ keys, const int *__restrict__ poff,
                                                               int nchunk, int shift, int *__restrict__ table)
{
    grid_dep_sync();
    const int pbase = poff[blockIdx.y], N = poff[blockIdx.y + 1] - pbase;
    __shared__ int h[RS_WARPS][256];
    const int b = blockIdx.y, w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int c = blockIdx.x * RS_WARPS + w;
    for (int d = lane; d < 256; d += 32) h[w][d] = 0;
    __syncwarp();
    if (c < nchunk) {
        const unsigned *k = keys + (size_t)pbase;
        const int end = min(N, (c + 1) * RS_CHUNK);
        for (int p = c * RS_CHUNK + lane; p < end; p += 32) atomicAdd(&h[w][(k[p] >> shift) & 255u], 1);
        __syncwarp();
        int *t = table + (size_t)b * 256 * nchunk;
        for (int d = lane; d < 256; d += 32) t[(size_t)d * nchunk + c] = h[w][d];
    }
}

__global__ void __launch_bounds__(RS_WARPS * 32) k_radix_scatter(const unsigned *__restrict__ keys, const int *__restrict__ vals,
                                                                  const int *__restrict__ poff, int nchunk, int shift,
                                                                  const int *__restrict__ table,
                                                                  unsigned *__restrict__ okeys, int *__restrict__ ovals)
{
    grid_dep_sync();
    const int pbase = poff[blockIdx.y], N = poff[blockIdx.y + 1] - pbase;
    __shared__ int base[RS_WARPS][256];
    const int b = blockIdx.y, w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int c = blockIdx.x * RS_WARPS + w;
    if (c >= nchunk) return;
    const int *t = table + (size_t)b * 256 * nchunk;
    for (int d = lane; d < 256; d += 32) base[w][d] = t[(size_t)d * nchunk + c];
    __syncwarp();
    const unsigned *k = keys + (size_t)pbase;
    const int *v = vals + (size_t)pbase;
    unsigned *ok = okeys + (size_t)pbase;
    int *ov = ovals + (size_t)pbase;
    const int end = min(N, (c + 1) * RS_CHUNK);
    const unsigned lt = (1u << lane) - 1u;
    // the whole chunk is loaded before the ranking loop: its rounds are serially dependent through the
    // shared counters, and a global load inside each of them would put DRAM/L2 latency on that chain
    constexpr int R = RS_CHUNK / 32;
    unsigned key[R];
    int val[R];
    const int p0 = c * RS_CHUNK + lane;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int p = p0 + 32 * r;
        const bool valid = p < end;
        key[r] = valid ? k[p] : 0u;
        val[r] = valid ? v[p] : 0;
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const bool valid = p0 + 32 * r < end;
        if (c * RS_CHUNK + 32 * r >= end) break;          // warp-uniform
        const unsigned d = valid ? ((key[r] >> shift) & 255u) : 256u;
        const unsigned peers = same_digit_lanes(d, valid);
        const int rank = __popc(peers & lt);
        int dst = 0;
        if (valid) dst = base[w][d] + rank;
        __syncwarp();
        if (valid && rank == 0) base[w][d] += __popc(peers);
        __syncwarp();
        if (valid) { ok[dst] = key[r]; ov[dst] = val[r]; }
    }
}

// ---------------------------------------------------------------------------------------------
// a5: active voxels.  heads[p] = 1 where the grid-voxel id changes; scan -> voxel rank.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_heads(const unsigned *__restrict__ keys, const int *__restrict__ poff, int subbits,
                                                int *__restrict__ heads)
{
    grid_dep_sync();
    const int b = blockIdx.y;
    const int base = poff[b], N = poff[b + 1] - base;
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= N) return;
    const unsigned *k = keys + (size_t)base;
    heads[(size_t)base + p] = (p == 0 || (k[p] >> subbits) != (k[p - 1] >> subbits)) ? 1 : 0;
}

// voff[b][rank] = p for every head position p
__global__ void __launch_bounds__(256) k_voxel_offsets(const int *__restrict__ heads, const int *__restrict__ rank,
                                                        const int *__restrict__ poff, int *__restrict__ voff)
{
    grid_dep_sync();
    const int b = blockIdx.y;
    const int base = poff[b], N = poff[b + 1] - base;
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= N) return;
    if (heads[(size_t)base + p]) voff[(size_t)base + rank[(size_t)base + p]] = p;
}

// number of tiles of each grid voxel: ceil(cnt / tile_points) (1 if tiling is off)
__global__ void __launch_bounds__(256) k_ntiles(const int *__restrict__ voff, const int *__restrict__ Kv,
                                                 const int *__restrict__ poff, int tile_points, int *__restrict__ ntiles)
{
    grid_dep_sync();
    const int b = blockIdx.y;
    const int base = poff[b], N = poff[b + 1] - base;
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    const int kv = Kv[b];
    int nt = 0;
    if (k < kv) {
        const int off = voff[(size_t)base + k];
        const int cnt = (k + 1 < kv ? voff[(size_t)base + k + 1] : N) - off;
        nt = tile_points > 0 ? (cnt + tile_points - 1) / tile_points : 1;
    }
    ntiles[(size_t)base + k] = nt;
}

// vseg[b][tbase[k] + t] = {off + t*chunk, len}: equal-size tiles of the voxel run (Morton sub-cell order inside the voxel)
__global__ void __launch_bounds__(256) k_tiles(const int *__restrict__ voff, const int *__restrict__ Kv, const int *__restrict__ ntiles,
                                                const int *__restrict__ tbase, const int *__restrict__ poff, int K_cap,
                                                int2 *__restrict__ vseg)
{
    grid_dep_sync();
    const int b = blockIdx.y;
    const int base = poff[b], N = poff[b + 1] - base;
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int kv = Kv[b];
    if (k >= kv) return;
    const int off = voff[(size_t)base + k];
    const int cnt = (k + 1 < kv ? voff[(size_t)base + k + 1] : N) - off;
    const int nt = ntiles[(size_t)base + k];
    const int chunk = (cnt + nt - 1) / nt;
    int2 *dst = vseg + (size_t)b * K_cap + tbase[(size_t)base + k];
    for (int t = 0; t < nt; ++t) {
        const int s = t * chunk;
        dst[t] = make_int2(off + s, min(chunk, cnt - s));
    }
}

// ---------------------------------------------------------------------------------------------
// a4: gather AoS -> sorted SoA (+ permutation and its inverse)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_gather(const float *__restrict__ pts, const int *__restrict__ order,
                                                 const int *__restrict__ poff,
                                                 float *__restrict__ px, float *__restrict__ py, float *__restrict__ pz,
                                                 int *__restrict__ porig, int *__restrict__ pinv)
{
    grid_dep_sync();
    const int b = blockIdx.y;
    const size_t o = (size_t)poff[b];
    const int N = poff[b + 1] - poff[b];
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= N) return;
    const int i = order[o + p];
    const float *s = pts + (o + i) * 3;
    px[o + p] = s[0];
    py[o + p] = s[1];
    pz[o + p] = s[2];
    porig[o + p] = i;
    pinv[o + i] = p;
}

// ---------------------------------------------------------------------------------------------
// a6: per-voxel bounding sphere, one warp per voxel.
//   c_k = midpoint of the axis-aligned bounding box of the voxel's points (reading A10)
//   R_k = sqrt_rn(max_p d2(p, c_k)) * (1 + 2^-20)      (reading A9: rounded UP past every fp32
//         error of d2 and sqrt, so that ||p - c_k|| <= R_k holds over the reals)
// d2 is the library's one distance expression, ((dx*dx + dy*dy) + dz*dz) without FMA (d2_rn, device_utils.cuh).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_sphere(const float *__restrict__ px, const float *__restrict__ py,
                                                 const float *__restrict__ pz, const int2 *__restrict__ vseg,
                                                 const int *__restrict__ K, const int *__restrict__ poff, int K_cap,
                                                 float4 *__restrict__ vgeom, int *__restrict__ maxcnt)
{
    grid_dep_sync();
    const int b = blockIdx.y;
    const int lane = threadIdx.x & 31;
    const float *x = px + (size_t)poff[b], *y = py + (size_t)poff[b], *z = pz + (size_t)poff[b];
    const int Kb = K[b];
    int local_max = 0;
    for (int k = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); k < Kb; k += gridDim.x * (blockDim.x >> 5)) {
    const int2 sg = vseg[(size_t)b * K_cap + k];
    float mn[3] = {FLT_MAX, FLT_MAX, FLT_MAX}, mx[3] = {-FLT_MAX, -FLT_MAX, -FLT_MAX};
    for (int p = sg.x + lane; p < sg.x + sg.y; p += 32) {
        mn[0] = fminf(mn[0], x[p]); mx[0] = fmaxf(mx[0], x[p]);
        mn[1] = fminf(mn[1], y[p]); mx[1] = fmaxf(mx[1], y[p]);
        mn[2] = fminf(mn[2], z[p]); mx[2] = fmaxf(mx[2], z[p]);
    }
#pragma unroll
    for (int a = 0; a < 3; ++a)
        for (int o = 16; o > 0; o >>= 1) {
            mn[a] = fminf(mn[a], __shfl_xor_sync(0xffffffffu, mn[a], o));
            mx[a] = fmaxf(mx[a], __shfl_xor_sync(0xffffffffu, mx[a], o));
        }
    const float cx = __fadd_rn(__fmul_rn(0.5f, mn[0]), __fmul_rn(0.5f, mx[0]));
    const float cy = __fadd_rn(__fmul_rn(0.5f, mn[1]), __fmul_rn(0.5f, mx[1]));
    const float cz = __fadd_rn(__fmul_rn(0.5f, mn[2]), __fmul_rn(0.5f, mx[2]));
    float r2 = 0.0f;
    for (int p = sg.x + lane; p < sg.x + sg.y; p += 32) r2 = fmaxf(r2, d2_rn(x[p], y[p], z[p], cx, cy, cz));
    for (int o = 16; o > 0; o >>= 1) r2 = fmaxf(r2, __shfl_xor_sync(0xffffffffu, r2, o));
    if (lane == 0) {
        const float R = __fmul_rn(__fsqrt_rn(r2), 1.0f + 0x1p-20f);
        vgeom[(size_t)b * K_cap + k] = make_float4(cx, cy, cz, R);
        local_max = max(local_max, sg.y);
    }
    }
    if (lane == 0 && local_max > 0) atomicMax(maxcnt, local_max);
}

// ---------------------------------------------------------------------------------------------
// a6': group spheres.  32 consecutive (Hilbert-ordered) voxels form a group; its sphere encloses the
// member spheres:  c_g = midpoint of the box around the member spheres,
//   R_g = max_l ( sqrt_rn(d2(c_l, c_g)) * (1 + 2^-20) + R_l ) * (1 + 2^-20)     (rounded up, as A9)
// so every point p of a member voxel has ||p - c_g|| <= ||p - c_l|| + ||c_l - c_g|| <= R_g, and the
// prune test of Eq. 25 can be applied to the whole group with Dist_v := max over its voxels.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_group_sphere(const float4 *__restrict__ vgeom, const int *__restrict__ K, int K_cap,
                                                       int G_cap, float4 *__restrict__ ggeom, const unsigned *__restrict__ rb,
                                                       unsigned *host_rb, int rb_n)
{
    grid_dep_sync();
    // the last kernel of the chain also hands the build's read-back block (K per cloud, largest segment, bounding boxes
    // with the non-finite flags: complete once its predecessors are) to the host through mapped pinned memory, so that
    // the build's one host round trip needs no copy
    if (host_rb != nullptr && blockIdx.x == 0 && blockIdx.y == 0) {
        for (int i = threadIdx.x; i < rb_n; i += blockDim.x) host_rb[i] = rb[i];
        __threadfence_system();
    }
    const int b = blockIdx.y;
    const int lane = threadIdx.x & 31;
    const int Kb = K[b];
    const int G = (Kb + 31) / 32;
    for (int g = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); g < G; g += gridDim.x * (blockDim.x >> 5)) {
        const int k = g * 32 + lane;
        const bool in = k < Kb;
        const float4 v = in ? vgeom[(size_t)b * K_cap + k] : make_float4(0.f, 0.f, 0.f, 0.f);
        float mn[3] = {in ? v.x - v.w : FLT_MAX, in ? v.y - v.w : FLT_MAX, in ? v.z - v.w : FLT_MAX};
        float mx[3] = {in ? v.x + v.w : -FLT_MAX, in ? v.y + v.w : -FLT_MAX, in ? v.z + v.w : -FLT_MAX};
#pragma unroll
        for (int a = 0; a < 3; ++a)
            for (int o = 16; o > 0; o >>= 1) {
                mn[a] = fminf(mn[a], __shfl_xor_sync(0xffffffffu, mn[a], o));
                mx[a] = fmaxf(mx[a], __shfl_xor_sync(0xffffffffu, mx[a], o));
            }
        const float cx = __fadd_rn(__fmul_rn(0.5f, mn[0]), __fmul_rn(0.5f, mx[0]));
        const float cy = __fadd_rn(__fmul_rn(0.5f, mn[1]), __fmul_rn(0.5f, mx[1]));
        const float cz = __fadd_rn(__fmul_rn(0.5f, mn[2]), __fmul_rn(0.5f, mx[2]));
        float r = 0.0f;
        if (in) r = __fmul_rn(__fadd_rn(__fmul_rn(__fsqrt_rn(d2_rn(v.x, v.y, v.z, cx, cy, cz)), 1.0f + 0x1p-20f), v.w), 1.0f + 0x1p-20f);
        for (int o = 16; o > 0; o >>= 1) r = fmaxf(r, __shfl_xor_sync(0xffffffffu, r, o));
        if (lane == 0) ggeom[(size_t)b * G_cap + g] = make_float4(cx, cy, cz, r);
    }
}

// ---------------------------------------------------------------------------------------------
// Single-launch build for small clouds (N <= FUSED_MAX_N = 8 192): ONE CTA of 1 024 threads per cloud runs a1-a6 back
// to back -- bbox, keys, the LSD radix passes, segments, tiles, gather, spheres, group spheres -- with CTA barriers
// where the 22-kernel chain has kernel boundaries, and with every intermediate array (keys, values, digit table,
// ranks, offsets, tile counts: 16 B per point + 1 KB per chunk) in SHARED memory, so that a phase costs a barrier and
// a few hundred cycles instead of a kernel boundary (~4.7 us) or an L2 round trip.  Same arithmetic, same stable
// sort, same output arrays as the chain (the sampler cannot tell which path built an index).  Measured: a first
// version with the scratch in global memory took 63 us for 4 096 points and 264 us for 24 000 on its one SM -- slower
// than the chain for C2-sized clouds, which therefore keep the chain.
// ---------------------------------------------------------------------------------------------
constexpr int FUSED_T = 1024, FUSED_MAX_N = 8192;
constexpr int FUSED_CHUNK = 256;     // keys per warp and radix pass: 4 096 points keep 16 of the 32 warps busy, 8 192 all of them
static inline size_t fused_smem_bytes(int N) { return (size_t)16 * N + (size_t)1024 * (((N + FUSED_CHUNK - 1) / FUSED_CHUNK) | 1); }

struct FusedArgs {
    const float *pts;
    const int *poff;
    unsigned *bbox;                 // [B][8] (the non-finite flag is what the host reads)
    int n_vox, hb, sb, keybits, tile_points, K_cap, G_cap, Nmax;
    float *px, *py, *pz;
    int *porig, *pinv;
    int2 *vseg;
    float4 *vgeom, *ggeom;
    int *K_dev;
    int *maxcnt;                    // meta[0]
    // zero-copy read-back (build_index): a pinned, device-visible host block [3][B] = K, largest segment, non-finite
    // flag of every cloud, written by the kernel itself, so that the build's one host round trip needs no copy; and,
    // for a batch of equal-size clouds (uniform_N > 0), the cloud offsets are computed and written here instead of
    // being copied in.  Both null / 0 for fps_sample_noalloc
    int *host_rb = nullptr;
    int *poff_out = nullptr;
    int uniform_N = 0, B = 0;
};

// exclusive scan of n ints by the whole CTA: tiles of 4 096 with a running carry; returns the total
__device__ int cta_scan_excl(const int *in, int *out, const int n, int *sm /*[34]*/)
{
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    if (tid == 0) sm[33] = 0;
    __syncthreads();
    for (int base = 0; base < n; base += FUSED_T * 4) {
        const int i0 = base + tid * 4;
        int v[4], s = 0;
#pragma unroll
        for (int i = 0; i < 4; ++i) { v[i] = i0 + i < n ? in[i0 + i] : 0; s += v[i]; }
        int inc = s;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) sm[w] = inc;
        __syncthreads();
        const int carry = sm[33];
        if (w == 0) {
            const int ws = sm[lane];
            int wi = ws;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, wi, o);
                if (lane >= o) wi += t;
            }
            sm[lane] = wi - ws;
            if (lane == 31) sm[32] = carry + wi;
        }
        __syncthreads();
        int e = carry + sm[w] + inc - s;
#pragma unroll
        for (int i = 0; i < 4; ++i) { if (i0 + i < n) out[i0 + i] = e; e += v[i]; }
        __syncthreads();
        if (tid == 0) sm[33] = sm[32];
        __syncthreads();
    }
    return sm[33];
}

__global__ void __launch_bounds__(FUSED_T, 1) k_build_fused(const FusedArgs A)
{
    grid_dep_sync();
    extern __shared__ __align__(16) unsigned char fsm[];
    __shared__ int hist[FUSED_T / 32][256];          // per-warp digit counters / bases of the radix passes
    __shared__ float red[FUSED_T / 32][6];
    __shared__ int sm[34];
    __shared__ float bb[8];
    __shared__ int sbad, skv, sK;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5, NWF = FUSED_T / 32;
    const int b = blockIdx.x;
    const int base = A.uniform_N > 0 ? b * A.uniform_N : A.poff[b], N = A.uniform_N > 0 ? A.uniform_N : A.poff[b + 1] - base;
    if (A.uniform_N > 0 && tid == 0) {
        A.poff_out[b] = base;
        if (b == A.B - 1) A.poff_out[A.B] = base + N;
    }
    const float *P = A.pts + (size_t)base * 3;
    // ---- a1: bounding box + non-finite flag ----
    {
        float mn[3] = {FLT_MAX, FLT_MAX, FLT_MAX}, mx[3] = {-FLT_MAX, -FLT_MAX, -FLT_MAX};
        bool bad = false;
        // (four points per trip, all twelve loads first: the memory round trips of a trip overlap)
        for (int i0 = tid; i0 < N; i0 += 4 * FUSED_T) {
            float c[4][3];
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int a = 0; a < 3; ++a) c[u][a] = i0 + u * FUSED_T < N ? P[3 * (size_t)(i0 + u * FUSED_T) + a] : P[3 * (size_t)i0 + a];
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    const float v = c[u][a];
                    bad |= !(fabsf(v) <= FLT_MAX);
                    mn[a] = fminf(mn[a], v);
                    mx[a] = fmaxf(mx[a], v);
                }
        }
#pragma unroll
        for (int a = 0; a < 3; ++a)
            for (int o = 16; o > 0; o >>= 1) {
                mn[a] = fminf(mn[a], __shfl_xor_sync(0xffffffffu, mn[a], o));
                mx[a] = fmaxf(mx[a], __shfl_xor_sync(0xffffffffu, mx[a], o));
            }
        bad = __any_sync(0xffffffffu, bad);
        if (tid == 0) sbad = 0;
        __syncthreads();
        if (lane == 0) {
#pragma unroll
            for (int a = 0; a < 3; ++a) { red[w][a] = mn[a]; red[w][3 + a] = mx[a]; }
            if (bad) sbad = 1;
        }
        __syncthreads();
        if (tid < 3) {
            float lo = red[0][tid], hi = red[0][3 + tid];
            for (int i = 1; i < NWF; ++i) { lo = fminf(lo, red[i][tid]); hi = fmaxf(hi, red[i][3 + tid]); }
            bb[tid] = lo; bb[3 + tid] = hi;
            unsigned *g = A.bbox + b * BBOX_STRIDE;
            g[tid] = f2ord(lo); g[3 + tid] = f2ord(hi);
            if (tid == 0) {
                g[6] = sbad ? 1u : 0u;
                if (A.host_rb) A.host_rb[2 * A.B + b] = sbad;
            }
        }
        __syncthreads();
    }
    // shared-memory scratch, sized for the largest cloud of the batch: two key and two value buffers, the digit table
    unsigned *kin = reinterpret_cast<unsigned *>(fsm), *kout = kin + A.Nmax;
    int *vin = reinterpret_cast<int *>(kout + A.Nmax), *vout = vin + A.Nmax;
    int *const table = vout + A.Nmax;                              // digit-major [256][nchunk]
    // ---- a2: sort keys (Eq. 8: floor, then clamp; Hilbert voxel id + Morton sub-cell bits) ----
    {
        const float E = fmaxf(fmaxf(bb[3] - bb[0], bb[4] - bb[1]), bb[5] - bb[2]);
        float L = (1.0f + 1e-3f) * E / (float)A.n_vox;
        if (!(L > 0.0f)) L = 1.0f;
        const float invsub = (float)(1 << A.sb);
        for (int i0 = tid; i0 < N; i0 += 4 * FUSED_T) {
          float c[4][3];
#pragma unroll
          for (int u = 0; u < 4; ++u)
#pragma unroll
              for (int a = 0; a < 3; ++a) c[u][a] = i0 + u * FUSED_T < N ? P[3 * (size_t)(i0 + u * FUSED_T) + a] : 0.0f;
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const int i = i0 + u * FUSED_T;
            if (i >= N) break;
            unsigned v[3], s[3];
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const float t = (c[u][a] - bb[a]) / L;
                int c = (int)floorf(t);
                c = max(0, min(A.n_vox - 1, c));
                int sc = (int)floorf((t - (float)c) * invsub);
                sc = max(0, min((1 << A.sb) - 1, sc));
                v[a] = (unsigned)c;
                s[a] = (unsigned)sc;
            }
            const unsigned vid = hilbert3(v[0], v[1], v[2], A.hb);
            const unsigned sub = A.sb ? (spread3(s[0]) | (spread3(s[1]) << 1) | (spread3(s[2]) << 2)) : 0u;
            kin[i] = (vid << (3 * A.sb)) | sub;
            vin[i] = i;
          }
        }
        __syncthreads();
    }
    // ---- a3: stable LSD radix sort, 8 bits per pass; a warp owns chunks of FUSED_CHUNK keys ----
    {
        const int nchunk = (N + FUSED_CHUNK - 1) / FUSED_CHUNK;
        const int ts = nchunk | 1;        // odd row stride of the digit table: a warp's 32 digits hit 32 banks
        const unsigned lt = (1u << lane) - 1u;
        for (int shift = 0; shift < A.keybits; shift += 8) {
            if (ts != nchunk && tid < 256) table[tid * ts + nchunk] = 0;      // the pad column counts nothing (the scan below runs over it)
            for (int c0 = 0; c0 < nchunk; c0 += NWF) {
                const int c = c0 + w;
                for (int d = lane; d < 256; d += 32) hist[w][d] = 0;
                __syncwarp();
                if (c < nchunk) {
                    const int end = min(N, (c + 1) * FUSED_CHUNK);
                    unsigned kr[FUSED_CHUNK / 32];              // the whole chunk first: one memory round trip, not 16
#pragma unroll
                    for (int r = 0; r < FUSED_CHUNK / 32; ++r) { const int p = c * FUSED_CHUNK + 32 * r + lane; kr[r] = p < end ? kin[p] : 0u; }
#pragma unroll
                    for (int r = 0; r < FUSED_CHUNK / 32; ++r)
                        if (c * FUSED_CHUNK + 32 * r + lane < end) atomicAdd(&hist[w][(kr[r] >> shift) & 255u], 1);
                    __syncwarp();
                    for (int d = lane; d < 256; d += 32) table[d * ts + c] = hist[w][d];
                }
                __syncwarp();
            }
            __syncthreads();
            cta_scan_excl(table, table, 256 * ts, sm);
            for (int c0 = 0; c0 < nchunk; c0 += NWF) {
                const int c = c0 + w;
                if (c < nchunk) {
                    for (int d = lane; d < 256; d += 32) hist[w][d] = table[d * ts + c];
                    __syncwarp();
                    const int end = min(N, (c + 1) * FUSED_CHUNK);
                    // the chunk is loaded before the ranking loop, whose rounds are serially dependent through the
                    // shared counters: a global load inside each of them would put L2 latency on that chain
                    unsigned kr[FUSED_CHUNK / 32];
                    int vr[FUSED_CHUNK / 32];
#pragma unroll
                    for (int r = 0; r < FUSED_CHUNK / 32; ++r) {
                        const int p = c * FUSED_CHUNK + 32 * r + lane;
                        kr[r] = p < end ? kin[p] : 0u;
                        vr[r] = p < end ? vin[p] : 0;
                    }
#pragma unroll
                    for (int r = 0; r < FUSED_CHUNK / 32; ++r) {
                        if (c * FUSED_CHUNK + 32 * r >= end) break;      // warp-uniform
                        const bool valid = c * FUSED_CHUNK + 32 * r + lane < end;
                        const unsigned key = kr[r];
                        const int val = vr[r];
                        const unsigned d = valid ? ((key >> shift) & 255u) : 256u;
                        const unsigned peers = same_digit_lanes(d, valid);
                        const int rk = __popc(peers & lt);
                        int dst = 0;
                        if (valid) dst = hist[w][d] + rk;
                        __syncwarp();
                        if (valid && rk == 0) hist[w][d] += __popc(peers);
                        __syncwarp();
                        if (valid) { kout[dst] = key; vout[dst] = val; }
                    }
                }
                __syncwarp();
            }
            __syncthreads();
            unsigned *tk = kin; kin = kout; kout = tk;
            int *tv = vin; vin = vout; vout = tv;
        }
    }
    // ---- a5: grid voxels (heads -> rank -> offsets), tiles (ntiles -> base -> segments) ----
    // the sort's spare buffers are reused: heads -> F1, rank -> F2, then voff -> F1 (the head flags are recomputed from
    // the keys), tile counts and their scan -> F2 (in place; a voxel's tile count is recomputed from its length)
    int *const F1 = reinterpret_cast<int *>(kout), *const F2 = vout;
    const int subbits = 3 * A.sb;
    for (int p = tid; p < N; p += FUSED_T) F1[p] = (p == 0 || (kin[p] >> subbits) != (kin[p - 1] >> subbits)) ? 1 : 0;
    __syncthreads();
    {
        const int kvt = cta_scan_excl(F1, F2, N, sm);
        if (tid == 0) skv = kvt;
    }
    __syncthreads();
    const int kv = skv;
    int *const voff = F1;
    for (int p = tid; p < N; p += FUSED_T)
        if (p == 0 || (kin[p] >> subbits) != (kin[p - 1] >> subbits)) voff[F2[p]] = p;
    __syncthreads();
    auto tiles_of = [&](const int cnt) { return A.tile_points > 0 ? (cnt + A.tile_points - 1) / A.tile_points : 1; };
    for (int k = tid; k < N; k += FUSED_T) {
        int nt = 0;
        if (k < kv) nt = tiles_of((k + 1 < kv ? voff[k + 1] : N) - voff[k]);
        F2[k] = nt;
    }
    __syncthreads();
    {
        const int Kt = cta_scan_excl(F2, F2, N, sm);
        if (tid == 0) { sK = Kt; A.K_dev[b] = Kt; if (A.host_rb) A.host_rb[b] = Kt; }
    }
    __syncthreads();
    const int K = sK;
    const int *const tbase = F2;
    int2 *vseg = A.vseg + (size_t)b * A.K_cap;
    for (int k = tid; k < kv; k += FUSED_T) {
        const int off = voff[k];
        const int cnt = (k + 1 < kv ? voff[k + 1] : N) - off;
        const int nt = tiles_of(cnt);
        const int chunk = (cnt + nt - 1) / nt;
        int2 *dst = vseg + tbase[k];
        // (a packed copy {first point, count << 16} stays in shared memory for the sphere phase: the keys are not needed
        // any more, and N <= FUSED_MAX_N = 8 192 fits 16 bits)
        for (int t = 0; t < nt; ++t) {
            const int o = off + t * chunk, c = min(chunk, cnt - t * chunk);
            dst[t] = make_int2(o, c);
            kin[tbase[k] + t] = (unsigned)o | ((unsigned)c << 16);
        }
    }
    __syncthreads();                                       // voff / tbase (F1 / F2) are free from here on
    // ---- a4: gather AoS -> sorted SoA (+ permutation and its inverse).  Four points per trip with all loads first (the
    // memory round trips overlap); the sorted coordinates also stay in shared memory (x in place of the sorted values,
    // y and z in the two spare buffers) for the sphere phase ----
    float *px = A.px + base, *py = A.py + base, *pz = A.pz + base;
    int *porig = A.porig + base, *pinv = A.pinv + base;
    const unsigned *const pseg = kin;
    float *const sx = reinterpret_cast<float *>(vin), *const sy = reinterpret_cast<float *>(F1), *const sz = reinterpret_cast<float *>(F2);
    for (int p0 = tid; p0 < N; p0 += 4 * FUSED_T) {
        int idx[4];
        float c[4][3];
#pragma unroll
        for (int u = 0; u < 4; ++u) idx[u] = p0 + u * FUSED_T < N ? vin[p0 + u * FUSED_T] : 0;
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int a = 0; a < 3; ++a) c[u][a] = P[3 * (size_t)idx[u] + a];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int q = p0 + u * FUSED_T;
            if (q < N) {
                px[q] = c[u][0]; py[q] = c[u][1]; pz[q] = c[u][2];
                porig[q] = idx[u];
                pinv[idx[u]] = q;
                sx[q] = c[u][0]; sy[q] = c[u][1]; sz[q] = c[u][2];
            }
        }
    }
    __syncthreads();
    // ---- a6: tight bounding sphere per (tiled) voxel, 8 lanes per voxel (small clouds have small voxels: a whole
    // warp per voxel spends its time in shuffles); then the group spheres ----
    float4 *vgeom = A.vgeom + (size_t)b * A.K_cap;
    int local_max = 0;
    if ((long long)N <= 8ll * K) {
        // few points per voxel (uniform small clouds: 2-8): ONE thread per voxel, no shuffles -- eight lanes per voxel
        // would spend ~120 instructions per warp and pass on two or three points.  min / max are order-independent, so
        // the sphere is bit-identical either way
        for (int k = tid; k < K; k += FUSED_T) {
            const unsigned ps = pseg[k];
            const int off = (int)(ps & 0xffffu), cnt = (int)(ps >> 16);
            float mn[3] = {FLT_MAX, FLT_MAX, FLT_MAX}, mx[3] = {-FLT_MAX, -FLT_MAX, -FLT_MAX};
            for (int p = off; p < off + cnt; ++p) {
                mn[0] = fminf(mn[0], sx[p]); mx[0] = fmaxf(mx[0], sx[p]);
                mn[1] = fminf(mn[1], sy[p]); mx[1] = fmaxf(mx[1], sy[p]);
                mn[2] = fminf(mn[2], sz[p]); mx[2] = fmaxf(mx[2], sz[p]);
            }
            const float cx = __fadd_rn(__fmul_rn(0.5f, mn[0]), __fmul_rn(0.5f, mx[0]));
            const float cy = __fadd_rn(__fmul_rn(0.5f, mn[1]), __fmul_rn(0.5f, mx[1]));
            const float cz = __fadd_rn(__fmul_rn(0.5f, mn[2]), __fmul_rn(0.5f, mx[2]));
            float r2 = 0.0f;
            for (int p = off; p < off + cnt; ++p) r2 = fmaxf(r2, d2_rn(sx[p], sy[p], sz[p], cx, cy, cz));
            vgeom[k] = make_float4(cx, cy, cz, __fmul_rn(__fsqrt_rn(r2), 1.0f + 0x1p-20f));
            local_max = max(local_max, cnt);
        }
    } else {
        const int sub = lane & 7, grp = (w << 2) | (lane >> 3), NG = NWF * 4;
        for (int k0 = 0; k0 < K; k0 += NG) {
            const int k = k0 + grp;
            const unsigned ps = k < K ? pseg[k] : 0u;
            const int2 sg = make_int2((int)(ps & 0xffffu), (int)(ps >> 16));
            float mn[3] = {FLT_MAX, FLT_MAX, FLT_MAX}, mx[3] = {-FLT_MAX, -FLT_MAX, -FLT_MAX};
            for (int p = sg.x + sub; p < sg.x + sg.y; p += 8) {
                mn[0] = fminf(mn[0], sx[p]); mx[0] = fmaxf(mx[0], sx[p]);
                mn[1] = fminf(mn[1], sy[p]); mx[1] = fmaxf(mx[1], sy[p]);
                mn[2] = fminf(mn[2], sz[p]); mx[2] = fmaxf(mx[2], sz[p]);
            }
#pragma unroll
            for (int a = 0; a < 3; ++a)
                for (int o = 4; o > 0; o >>= 1) {
                    mn[a] = fminf(mn[a], __shfl_xor_sync(0xffffffffu, mn[a], o));
                    mx[a] = fmaxf(mx[a], __shfl_xor_sync(0xffffffffu, mx[a], o));
                }
            const float cx = __fadd_rn(__fmul_rn(0.5f, mn[0]), __fmul_rn(0.5f, mx[0]));
            const float cy = __fadd_rn(__fmul_rn(0.5f, mn[1]), __fmul_rn(0.5f, mx[1]));
            const float cz = __fadd_rn(__fmul_rn(0.5f, mn[2]), __fmul_rn(0.5f, mx[2]));
            float r2 = 0.0f;
            for (int p = sg.x + sub; p < sg.x + sg.y; p += 8) r2 = fmaxf(r2, d2_rn(sx[p], sy[p], sz[p], cx, cy, cz));
            for (int o = 4; o > 0; o >>= 1) r2 = fmaxf(r2, __shfl_xor_sync(0xffffffffu, r2, o));
            if (sub == 0 && k < K) {
                vgeom[k] = make_float4(cx, cy, cz, __fmul_rn(__fsqrt_rn(r2), 1.0f + 0x1p-20f));
                local_max = max(local_max, sg.y);
            }
        }
    }
    local_max = __reduce_max_sync(0xffffffffu, local_max);
    if (A.host_rb) {
        if (tid == 0) skv = 0;                              // (skv is free by now: reused as the CTA's largest segment)
        __syncthreads();
        if (lane == 0 && local_max > 0) atomicMax(&skv, local_max);
        __syncthreads();
        if (tid == 0) { A.host_rb[A.B + b] = skv; __threadfence_system(); }
    } else if (lane == 0 && local_max > 0) atomicMax(A.maxcnt, local_max);
    __syncthreads();
    float4 *ggeom = A.ggeom + (size_t)b * A.G_cap;
    const int G = (K + 31) / 32;
    for (int g = w; g < G; g += NWF) {
        const int k = g * 32 + lane;
        const bool in = k < K;
        const float4 v = in ? vgeom[k] : make_float4(0.f, 0.f, 0.f, 0.f);
        float mn[3] = {in ? v.x - v.w : FLT_MAX, in ? v.y - v.w : FLT_MAX, in ? v.z - v.w : FLT_MAX};
        float mx[3] = {in ? v.x + v.w : -FLT_MAX, in ? v.y + v.w : -FLT_MAX, in ? v.z + v.w : -FLT_MAX};
#pragma unroll
        for (int a = 0; a < 3; ++a)
            for (int o = 16; o > 0; o >>= 1) {
                mn[a] = fminf(mn[a], __shfl_xor_sync(0xffffffffu, mn[a], o));
                mx[a] = fmaxf(mx[a], __shfl_xor_sync(0xffffffffu, mx[a], o));
            }
        const float cx = __fadd_rn(__fmul_rn(0.5f, mn[0]), __fmul_rn(0.5f, mx[0]));
        const float cy = __fadd_rn(__fmul_rn(0.5f, mn[1]), __fmul_rn(0.5f, mx[1]));
        const float cz = __fadd_rn(__fmul_rn(0.5f, mn[2]), __fmul_rn(0.5f, mx[2]));
        float r = 0.0f;
        if (in) r = __fmul_rn(__fadd_rn(__fmul_rn(__fsqrt_rn(d2_rn(v.x, v.y, v.z, cx, cy, cz)), 1.0f + 0x1p-20f), v.w), 1.0f + 0x1p-20f);
        for (int o = 16; o > 0; o >>= 1) r = fmaxf(r, __shfl_xor_sync(0xffffffffu, r, o));
        if (lane == 0) ggeom[g] = make_float4(cx, cy, cz, r);
    }
}

// ---------------------------------------------------------------------------------------------
// a1-a6 in ONE launch for MID-SIZE clouds (FUSED_MAX_N < N <= CL_MAX_N = 155 648, e.g. config 2's 24 000 points): one
// thread-block CLUSTER of C CTAs per cloud.  CTA r owns the points (later: the sorted positions) [r Np, (r+1) Np);
// keys and values live in its shared memory as in k_build_fused, and the radix passes exchange across the cluster:
// every CTA publishes its 256 digit totals (read by the peers over DSMEM), derives the global output offset of each
// of its (digit, chunk) cells -- digit-major, then CTA rank, then chunk, which keeps the sort stable --, and scatters
// its keys straight into the owner's shared memory (st.shared::cluster).  The segment / tile phase scans every CTA's
// share in shared memory and chains the shares through per-CTA totals (DSMEM); the spheres are dealt over all warps
// of the cluster.  A dozen cluster barriers instead of 22 launches; same voxels, tiles and spheres as the chain
// (tests compare them).
// ---------------------------------------------------------------------------------------------
// ~6 000 points per CTA where that needs <= 16 CTAs (a cluster of more than 8 is "non-portable" but fits a B200 GPC);
// up to CL_PER_CTA_MAX per CTA beyond (what the 227 KB of shared memory hold next to the 35 KB of static arrays)
constexpr int CL_PER_CTA = 6144, CL_PER_CTA_MAX = 9728, CL_MAX_C = 16, CL_MAX_N = CL_MAX_C * CL_PER_CTA_MAX;
static inline int cluster_build_ctas(int N) { return std::min(CL_MAX_C, std::max(2, (N + CL_PER_CTA - 1) / CL_PER_CTA)); }
static inline size_t cluster_smem_bytes(int Np) { return (size_t)16 * Np + (size_t)1024 * (((Np + FUSED_CHUNK - 1) / FUSED_CHUNK) | 1); }

struct ClusterArgs {
    FusedArgs f;                    // (f.Nmax = positions per CTA of the largest cloud: sizes the shared-memory buffers)
    int *F1g;                       // [all points] first point of every grid voxel (global scratch)
};

// exclusive prefix sums of two int sequences of 256 elements held by threads 0..255 (one element each); whole CTA
__device__ __forceinline__ int2 scan256_pair(const int a, const int b, int *sm /* [34] */)
{
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    int ia = a, ib = b;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int ta = __shfl_up_sync(0xffffffffu, ia, o), tb = __shfl_up_sync(0xffffffffu, ib, o);
        if (lane >= o) { ia += ta; ib += tb; }
    }
    __syncthreads();
    if (w < 8 && lane == 31) { sm[w] = ia; sm[8 + w] = ib; }
    __syncthreads();
    int ca = 0, cb = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) { ca += i < w ? sm[i] : 0; cb += i < w ? sm[8 + i] : 0; }
    return make_int2(ca + ia - a, cb + ib - b);
}

__global__ void __launch_bounds__(FUSED_T, 1) k_build_cluster(const ClusterArgs CA)
{
    grid_dep_sync();
    const FusedArgs &A = CA.f;
    extern __shared__ __align__(16) unsigned char fsm[];
    __shared__ int hist[FUSED_T / 32][256];
    __shared__ float red[FUSED_T / 32][6];
    __shared__ float cred[8];        // this CTA's {lo x y z, hi x y z, non-finite flag, largest segment}: read by the peers
    __shared__ int tdig[256];        // this CTA's digit totals of the running radix pass: read by the peers
    __shared__ int fix[256];
    __shared__ int sm[34];
    __shared__ float bb[8];
    __shared__ int sbad, sK, smaxc;
    __shared__ int xch[2];           // this CTA's head / tile totals: read by the peers
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5, NWF = FUSED_T / 32;
    const int C = (int)cluster_nctarank(), r = (int)cluster_ctarank();
    const int b = blockIdx.x / C;
    const int base = A.uniform_N > 0 ? b * A.uniform_N : A.poff[b], N = A.uniform_N > 0 ? A.uniform_N : A.poff[b + 1] - base;
    if (A.uniform_N > 0 && tid == 0 && r == 0) {
        A.poff_out[b] = base;
        if (b == A.B - 1) A.poff_out[A.B] = base + N;
    }
    const float *P = A.pts + (size_t)base * 3;
    const int Np = (N + C - 1) / C;                          // points / sorted positions per CTA
    const int p0 = min(N, r * Np), n = min(N, p0 + Np) - p0; // this CTA's share
    // ---- a1: bounding box + non-finite flag: CTA partials, combined over the cluster ----
    {
        float mn[3] = {FLT_MAX, FLT_MAX, FLT_MAX}, mx[3] = {-FLT_MAX, -FLT_MAX, -FLT_MAX};
        bool bad = false;
        for (int j = tid; j < n; j += FUSED_T) {
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const float v = P[3 * (size_t)(p0 + j) + a];
                bad |= !(fabsf(v) <= FLT_MAX);
                mn[a] = fminf(mn[a], v);
                mx[a] = fmaxf(mx[a], v);
            }
        }
#pragma unroll
        for (int a = 0; a < 3; ++a)
            for (int o = 16; o > 0; o >>= 1) {
                mn[a] = fminf(mn[a], __shfl_xor_sync(0xffffffffu, mn[a], o));
                mx[a] = fmaxf(mx[a], __shfl_xor_sync(0xffffffffu, mx[a], o));
            }
        bad = __any_sync(0xffffffffu, bad);
        if (tid == 0) sbad = 0;
        __syncthreads();
        if (lane == 0) {
#pragma unroll
            for (int a = 0; a < 3; ++a) { red[w][a] = mn[a]; red[w][3 + a] = mx[a]; }
            if (bad) sbad = 1;
        }
        __syncthreads();
        if (tid < 3) {
            float lo = red[0][tid], hi = red[0][3 + tid];
            for (int i = 1; i < NWF; ++i) { lo = fminf(lo, red[i][tid]); hi = fmaxf(hi, red[i][3 + tid]); }
            cred[tid] = lo; cred[3 + tid] = hi;
            if (tid == 0) cred[6] = sbad ? 1.0f : 0.0f;
        }
        cluster_sync_all();
        if (tid < 3) {
            float lo = FLT_MAX, hi = -FLT_MAX;
            for (int q = 0; q < C; ++q) {
                lo = fminf(lo, __uint_as_float(ld_dsmem_u32(mapa(smem_u32(&cred[tid]), (unsigned)q))));
                hi = fmaxf(hi, __uint_as_float(ld_dsmem_u32(mapa(smem_u32(&cred[3 + tid]), (unsigned)q))));
            }
            bb[tid] = lo; bb[3 + tid] = hi;
            if (r == 0) {
                unsigned *g = A.bbox + b * BBOX_STRIDE;
                g[tid] = f2ord(lo); g[3 + tid] = f2ord(hi);
            }
            if (tid == 0 && r == 0) {
                int anybad = 0;
                for (int q = 0; q < C; ++q) anybad |= __uint_as_float(ld_dsmem_u32(mapa(smem_u32(&cred[6]), (unsigned)q))) != 0.0f ? 1 : 0;
                A.bbox[b * BBOX_STRIDE + 6] = anybad ? 1u : 0u;
                if (A.host_rb) A.host_rb[2 * A.B + b] = anybad;
            }
        }
        __syncthreads();
    }
    unsigned *kin = reinterpret_cast<unsigned *>(fsm), *kout = kin + A.Nmax;
    int *vin = reinterpret_cast<int *>(kout + A.Nmax), *vout = vin + A.Nmax;
    int *const table = vout + A.Nmax;                              // digit-major [256][nchunk]
    // ---- a2: sort keys of this CTA's points (the arithmetic of k_keys) ----
    {
        const float E = fmaxf(fmaxf(bb[3] - bb[0], bb[4] - bb[1]), bb[5] - bb[2]);
        float L = (1.0f + 1e-3f) * E / (float)A.n_vox;
        if (!(L > 0.0f)) L = 1.0f;
        const float invsub = (float)(1 << A.sb);
        for (int j = tid; j < n; j += FUSED_T) {
            const int i = p0 + j;
            unsigned v[3], s[3];
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const float t = (P[3 * (size_t)i + a] - bb[a]) / L;
                int c = (int)floorf(t);
                c = max(0, min(A.n_vox - 1, c));
                int sc = (int)floorf((t - (float)c) * invsub);
                sc = max(0, min((1 << A.sb) - 1, sc));
                v[a] = (unsigned)c;
                s[a] = (unsigned)sc;
            }
            const unsigned vid = hilbert3(v[0], v[1], v[2], A.hb);
            const unsigned sub = A.sb ? (spread3(s[0]) | (spread3(s[1]) << 1) | (spread3(s[2]) << 2)) : 0u;
            kin[j] = (vid << (3 * A.sb)) | sub;
            vin[j] = i;
        }
        __syncthreads();
    }
    // ---- a3: stable LSD radix sort across the cluster, 8 bits per pass ----
    {
        const int nchunk = (n + FUSED_CHUNK - 1) / FUSED_CHUNK;                 // this CTA's chunks (0 if it holds no point)
        const int ts = ((A.Nmax + FUSED_CHUNK - 1) / FUSED_CHUNK) | 1;          // odd row stride of the digit table
        const unsigned lt = (1u << lane) - 1u;
        for (int shift = 0; shift < A.keybits; shift += 8) {
            for (int i = tid; i < 256 * ts; i += FUSED_T) table[i] = 0;         // (chunks this CTA does not have count nothing)
            __syncthreads();
            for (int c0 = 0; c0 < nchunk; c0 += NWF) {
                const int c = c0 + w;
                for (int d = lane; d < 256; d += 32) hist[w][d] = 0;
                __syncwarp();
                if (c < nchunk) {
                    const int end = min(n, (c + 1) * FUSED_CHUNK);
                    unsigned kr[FUSED_CHUNK / 32];
#pragma unroll
                    for (int q = 0; q < FUSED_CHUNK / 32; ++q) { const int p = c * FUSED_CHUNK + 32 * q + lane; kr[q] = p < end ? kin[p] : 0u; }
#pragma unroll
                    for (int q = 0; q < FUSED_CHUNK / 32; ++q)
                        if (c * FUSED_CHUNK + 32 * q + lane < end) atomicAdd(&hist[w][(kr[q] >> shift) & 255u], 1);
                    __syncwarp();
                    for (int d = lane; d < 256; d += 32) table[d * ts + c] = hist[w][d];
                }
                __syncwarp();
            }
            __syncthreads();
            // this CTA's digit totals -> the peers; every CTA then knows where each of its digits starts in the output
            int mine = 0;
            if (tid < 256) {
                for (int c = 0; c < nchunk; ++c) mine += table[tid * ts + c];
                tdig[tid] = mine;
            }
            cluster_sync_all();
            int all = 0, before = 0;
            if (tid < 256)
                for (int q = 0; q < C; ++q) {
                    const int v = (int)ld_dsmem_u32(mapa(smem_u32(&tdig[tid]), (unsigned)q));
                    all += v;
                    before += q < r ? v : 0;
                }
            const int2 ex = scan256_pair(all, mine, sm);      // digits before d: in the whole cloud / in this CTA
            // global offset of (digit d, chunk c) = (all digits < d) + (digit d in the CTAs before this one) + (digit d in
            // this CTA's chunks before c); the local digit-major scan of the table below yields (this CTA's digits < d) +
            // (digit d in its chunks before c): fix[d] is the difference
            if (tid < 256) fix[tid] = ex.x + before - ex.y;
            __syncthreads();
            cta_scan_excl(table, table, 256 * ts, sm);
            for (int c0 = 0; c0 < nchunk; c0 += NWF) {
                const int c = c0 + w;
                if (c < nchunk) {
                    for (int d = lane; d < 256; d += 32) hist[w][d] = table[d * ts + c] + fix[d];
                    __syncwarp();
                    const int end = min(n, (c + 1) * FUSED_CHUNK);
                    unsigned kr[FUSED_CHUNK / 32];
                    int vr[FUSED_CHUNK / 32];
#pragma unroll
                    for (int q = 0; q < FUSED_CHUNK / 32; ++q) {
                        const int p = c * FUSED_CHUNK + 32 * q + lane;
                        kr[q] = p < end ? kin[p] : 0u;
                        vr[q] = p < end ? vin[p] : 0;
                    }
#pragma unroll
                    for (int q = 0; q < FUSED_CHUNK / 32; ++q) {
                        if (c * FUSED_CHUNK + 32 * q >= end) break;      // warp-uniform
                        const bool valid = c * FUSED_CHUNK + 32 * q + lane < end;
                        const unsigned key = kr[q];
                        const int val = vr[q];
                        const unsigned d = valid ? ((key >> shift) & 255u) : 256u;
                        const unsigned peers = same_digit_lanes(d, valid);
                        const int rk = __popc(peers & lt);
                        int dst = 0;
                        if (valid) dst = hist[w][d] + rk;
                        __syncwarp();
                        if (valid && rk == 0) hist[w][d] += __popc(peers);
                        __syncwarp();
                        if (valid) {                                     // straight into the owner's shared memory
                            const int q2 = dst / Np, li = dst - q2 * Np;
                            st_dsmem_u32(mapa(smem_u32(kout + li), (unsigned)q2), key);
                            st_dsmem_u32(mapa(smem_u32(vout + li), (unsigned)q2), (unsigned)val);
                        }
                    }
                }
                __syncwarp();
            }
            cluster_sync_all();                                          // every CTA's scatter has landed
            unsigned *tk = kin; kin = kout; kout = tk;
            int *tv = vin; vin = vout; vout = tv;
        }
    }
    // ---- a4: gather this CTA's sorted positions (AoS -> sorted SoA, permutation and its inverse) ----
    float *px = A.px + base, *py = A.py + base, *pz = A.pz + base;
    int *porig = A.porig + base, *pinv = A.pinv + base;
    for (int j0 = tid; j0 < n; j0 += 4 * FUSED_T) {
        int idx[4];
        float c[4][3];
#pragma unroll
        for (int u = 0; u < 4; ++u) idx[u] = j0 + u * FUSED_T < n ? vin[j0 + u * FUSED_T] : vin[j0];
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int a = 0; a < 3; ++a) c[u][a] = P[3 * (size_t)idx[u] + a];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int j = j0 + u * FUSED_T;
            if (j < n) {
                const int q = p0 + j;
                px[q] = c[u][0]; py[q] = c[u][1]; pz[q] = c[u][2];
                porig[q] = idx[u];
                pinv[idx[u]] = q;
            }
        }
    }
    __syncthreads();                                                     // (vin is free from here on)
    // ---- a5: grid voxels (heads -> rank -> offsets) and tiles (counts -> base -> segments), spread over the cluster: every
    // CTA scans its own share in shared memory; the shares are chained through per-CTA totals read over DSMEM ----
    int2 *vseg = A.vseg + (size_t)b * A.K_cap;
    {
        int *const F1 = reinterpret_cast<int *>(kout), *const F2 = vout;         // (free since the sort)
        int *const voffg = CA.F1g + base;                                        // first point of every grid voxel (global)
        const int subbits = 3 * A.sb;
        // heads of this CTA's positions; the key before its first position is the last key of the CTA before it
        unsigned prevk = 0u;
        if (r > 0 && n > 0) prevk = ld_dsmem_u32(mapa(smem_u32(kin + (Np - 1)), (unsigned)(r - 1)));
        for (int j = tid; j < n; j += FUSED_T) {
            const unsigned pk = j > 0 ? kin[j - 1] : prevk;
            F1[j] = (p0 + j == 0 || (kin[j] >> subbits) != (pk >> subbits)) ? 1 : 0;
        }
        __syncthreads();
        const int hc = cta_scan_excl(F1, F2, n, sm);                             // F2 = rank of a head among this CTA's heads
        if (tid == 0) xch[0] = hc;
        cluster_sync_all();
        int vbase = 0, kv = 0;
        for (int q = 0; q < C; ++q) {
            const int v = (int)ld_dsmem_u32(mapa(smem_u32(&xch[0]), (unsigned)q));
            vbase += q < r ? v : 0;
            kv += v;
        }
        for (int j = tid; j < n; j += FUSED_T)
            if (F1[j]) voffg[vbase + F2[j]] = p0 + j;
        cluster_sync_all();                                                      // voffg is complete
        // tiles: the grid voxels are dealt to the CTAs in contiguous shares
        const int Kp = (kv + C - 1) / C, k0 = min(kv, r * Kp), nk = min(kv, k0 + Kp) - k0;
        auto tiles_of = [&](const int cnt) { return A.tile_points > 0 ? (cnt + A.tile_points - 1) / A.tile_points : 1; };
        for (int kl = tid; kl < nk; kl += FUSED_T) {
            const int k = k0 + kl;
            F1[kl] = tiles_of((k + 1 < kv ? voffg[k + 1] : N) - voffg[k]);
        }
        __syncthreads();
        const int tc = cta_scan_excl(F1, F2, nk, sm);                            // F2 = first tile of a voxel among this CTA's tiles
        if (tid == 0) xch[1] = tc;
        cluster_sync_all();
        int tb = 0, Kt = 0;
        for (int q = 0; q < C; ++q) {
            const int v = (int)ld_dsmem_u32(mapa(smem_u32(&xch[1]), (unsigned)q));
            tb += q < r ? v : 0;
            Kt += v;
        }
        if (r == 0 && tid == 0) { A.K_dev[b] = Kt; if (A.host_rb) A.host_rb[b] = Kt; }
        for (int kl = tid; kl < nk; kl += FUSED_T) {
            const int k = k0 + kl;
            const int off = voffg[k];
            const int cnt = (k + 1 < kv ? voffg[k + 1] : N) - off;
            const int nt = F1[kl];
            const int chunk = (cnt + nt - 1) / nt;
            int2 *dst = vseg + tb + F2[kl];
            for (int t = 0; t < nt; ++t) dst[t] = make_int2(off + t * chunk, min(chunk, cnt - t * chunk));
        }
        sK = Kt;                                                                  // (every thread writes the same value)
    }
    cluster_sync_all();                                                          // vseg is complete
    const int K = sK;
    // ---- a6: tight bounding sphere per (tiled) voxel: eight lanes per voxel, four voxels per warp in flight (the points
    // come from global memory / L2: what counts is the number of round trips under way), voxels dealt over the cluster ----
    float4 *vgeom = A.vgeom + (size_t)b * A.K_cap;
    int local_max = 0;
    {
        const int sub = lane & 7, grp = (r * NWF + w) * 4 + (lane >> 3), NG = C * NWF * 4;
        for (int k0 = 0; k0 < K; k0 += NG) {
            const int k = k0 + grp;
            const int2 sg = k < K ? vseg[k] : make_int2(0, 0);
            float mn[3] = {FLT_MAX, FLT_MAX, FLT_MAX}, mx[3] = {-FLT_MAX, -FLT_MAX, -FLT_MAX};
            for (int p = sg.x + sub; p < sg.x + sg.y; p += 8) {
                mn[0] = fminf(mn[0], px[p]); mx[0] = fmaxf(mx[0], px[p]);
                mn[1] = fminf(mn[1], py[p]); mx[1] = fmaxf(mx[1], py[p]);
                mn[2] = fminf(mn[2], pz[p]); mx[2] = fmaxf(mx[2], pz[p]);
            }
#pragma unroll
            for (int a = 0; a < 3; ++a)
                for (int o = 4; o > 0; o >>= 1) {
                    mn[a] = fminf(mn[a], __shfl_xor_sync(0xffffffffu, mn[a], o));
                    mx[a] = fmaxf(mx[a], __shfl_xor_sync(0xffffffffu, mx[a], o));
                }
            const float cx = __fadd_rn(__fmul_rn(0.5f, mn[0]), __fmul_rn(0.5f, mx[0]));
            const float cy = __fadd_rn(__fmul_rn(0.5f, mn[1]), __fmul_rn(0.5f, mx[1]));
            const float cz = __fadd_rn(__fmul_rn(0.5f, mn[2]), __fmul_rn(0.5f, mx[2]));
            float r2 = 0.0f;
            for (int p = sg.x + sub; p < sg.x + sg.y; p += 8) r2 = fmaxf(r2, d2_rn(px[p], py[p], pz[p], cx, cy, cz));
            for (int o = 4; o > 0; o >>= 1) r2 = fmaxf(r2, __shfl_xor_sync(0xffffffffu, r2, o));
            if (sub == 0 && k < K) {
                vgeom[k] = make_float4(cx, cy, cz, __fmul_rn(__fsqrt_rn(r2), 1.0f + 0x1p-20f));
                local_max = max(local_max, sg.y);
            }
        }
    }
    local_max = __reduce_max_sync(0xffffffffu, local_max);
    if (tid == 0) smaxc = 0;
    __syncthreads();
    if (lane == 0 && local_max > 0) atomicMax(&smaxc, local_max);
    __syncthreads();
    if (tid == 0) cred[7] = __int_as_float(smaxc);
    cluster_sync_all();
    // ---- a6': group spheres (32 consecutive voxels), groups dealt over the cluster's warps ----
    float4 *ggeom = A.ggeom + (size_t)b * A.G_cap;
    const int G = (K + 31) / 32;
    for (int g = r * NWF + w; g < G; g += C * NWF) {
        const int k = g * 32 + lane;
        const bool in = k < K;
        const float4 v = in ? vgeom[k] : make_float4(0.f, 0.f, 0.f, 0.f);
        float mn[3] = {in ? v.x - v.w : FLT_MAX, in ? v.y - v.w : FLT_MAX, in ? v.z - v.w : FLT_MAX};
        float mx[3] = {in ? v.x + v.w : -FLT_MAX, in ? v.y + v.w : -FLT_MAX, in ? v.z + v.w : -FLT_MAX};
#pragma unroll
        for (int a = 0; a < 3; ++a)
            for (int o = 16; o > 0; o >>= 1) {
                mn[a] = fminf(mn[a], __shfl_xor_sync(0xffffffffu, mn[a], o));
                mx[a] = fmaxf(mx[a], __shfl_xor_sync(0xffffffffu, mx[a], o));
            }
        const float cx = __fadd_rn(__fmul_rn(0.5f, mn[0]), __fmul_rn(0.5f, mx[0]));
        const float cy = __fadd_rn(__fmul_rn(0.5f, mn[1]), __fmul_rn(0.5f, mx[1]));
        const float cz = __fadd_rn(__fmul_rn(0.5f, mn[2]), __fmul_rn(0.5f, mx[2]));
        float rr = 0.0f;
        if (in) rr = __fmul_rn(__fadd_rn(__fmul_rn(__fsqrt_rn(d2_rn(v.x, v.y, v.z, cx, cy, cz)), 1.0f + 0x1p-20f), v.w), 1.0f + 0x1p-20f);
        for (int o = 16; o > 0; o >>= 1) rr = fmaxf(rr, __shfl_xor_sync(0xffffffffu, rr, o));
        if (lane == 0) ggeom[g] = make_float4(cx, cy, cz, rr);
    }
    if (r == 0 && tid == 0) {
        int mc = 0;
        for (int q = 0; q < C; ++q) mc = max(mc, (int)ld_dsmem_u32(mapa(smem_u32(&cred[7]), (unsigned)q)));
        if (A.host_rb) { A.host_rb[A.B + b] = mc; __threadfence_system(); }
        else if (mc > 0) atomicMax(A.maxcnt, mc);
    }
    cluster_sync_all();              // no CTA may exit while a peer can still read its shared memory
}

// ---------------------------------------------------------------------------------------------
// host orchestration
// ---------------------------------------------------------------------------------------------
static int ilog2_ceil(unsigned long long v)
{
    int b = 0;
    while ((1ull << b) < v) ++b;
    return b;
}

static int auto_n_vox(int N)
{   // nearest power of two to (N/4)^(1/3): some tens of points per active voxel on surface-like clouds
    // (denser cells are cut into tiles of <= tile_points anyway).  Measured on C1-C5: the sampling time
    // is flat within a factor 4 of this value and rises when most voxels hold only 1-2 points.
    // A free parameter of the method; results do not depend on it.
    double c = std::cbrt((double)N / 4.0);
    int n = 1;
    while (n * 2 <= 1024 && std::fabs(std::log2((double)n * 2) - std::log2(c)) <= std::fabs(std::log2((double)n) - std::log2(c))) n *= 2;
    return n < 2 ? 2 : n;
}

// Stream-ordered allocations from a private pool that keeps freed memory (release threshold = max),
// so that a build + destroy cycle costs no cudaMalloc/cudaFree and no device synchronisation.
static cudaMemPool_t build_pool()
{
    static std::mutex mu;
    static cudaMemPool_t pools[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
    std::lock_guard<std::mutex> lock(mu);
    if (!pools[dev]) {
        cudaMemPoolProps props;
        memset(&props, 0, sizeof props);
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        if (cudaMemPoolCreate(&pools[dev], &props) != cudaSuccess) { cudaGetLastError(); pools[dev] = nullptr; return nullptr; }
        unsigned long long keep = ~0ull;
        cudaMemPoolSetAttribute(pools[dev], cudaMemPoolAttrReleaseThreshold, &keep);
    }
    return pools[dev];
}

static cudaError_t pool_alloc(void **p, size_t bytes, cudaStream_t st)
{
    cudaMemPool_t pool = build_pool();
    if (!pool) return cudaMalloc(p, bytes);
    return cudaMallocFromPoolAsync(p, bytes, pool, st);
}

cudaError_t dev_alloc_async(void **p, size_t bytes, cudaStream_t st) { return pool_alloc(p, bytes ? bytes : 4, st); }
void dev_free_async(void *p, cudaStream_t st)
{
    if (!p) return;
    if (build_pool()) cudaFreeAsync(p, st);
    else cudaFree(p);
}

void trim_pool()
{
    cudaMemPool_t pool = build_pool();
    if (pool) cudaMemPoolTrimTo(pool, 0);
}

struct Carver {    // hands out 256-byte aligned pieces of one allocation (first pass: sizes only)
    char *base = nullptr;
    size_t off = 0;
    template <class T> T *take(size_t count)
    {
        T *p = base ? reinterpret_cast<T *>(base + off) : nullptr;
        off += ((count ? count : 1) * sizeof(T) + 255) & ~(size_t)255;
        return p;
    }
};

void free_index(DeviceIndex &ix)
{
    if (ix.arena) {
        // stream-ordered: the memory is released after the last sampling kernel enqueued on that stream
        if (ix.arena_pooled) cudaFreeAsync(ix.arena, ix.last_stream);
        else cudaFree(ix.arena);
    }
    if (ix.gx) dev_free_async(ix.gx, ix.last_stream);
    free(ix.K_host);
    free(ix.poff_host);
    free(ix.rag_host);
    ix = DeviceIndex();
}

struct Scratch {
    unsigned *bbox, *kA, *kB;
    int *vA, *vB, *table, *bsum, *heads, *rank, *voff, *ntl, *tbase, *Kv;
};

// the single-launch build takes more than the default 48 KB of dynamic shared memory: opt in once per device
static bool fused_attr_set()
{
    static std::mutex mu;
    static bool done[64];
    int dev = 0;
    cudaGetDevice(&dev);
    std::lock_guard<std::mutex> lock(mu);
    if (dev >= 0 && dev < 64 && done[dev]) return true;
    if (cudaFuncSetAttribute(k_build_fused, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fused_smem_bytes(FUSED_MAX_N)) != cudaSuccess) return false;
    if (cudaFuncSetAttribute(k_build_cluster, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cluster_smem_bytes(CL_PER_CTA_MAX)) != cudaSuccess) return false;
    if (cudaFuncSetAttribute(k_build_cluster, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) return false;
    if (dev >= 0 && dev < 64) done[dev] = true;
    return true;
}

// Per-thread pinned host staging for the two small copies of a build (cloud offsets in, read-back block out): with a
// pageable buffer both copies are staged by the driver and cost several microseconds of host time each, which is a
// visible part of a small cloud's build.  Grown on demand, kept for the life of the thread (a build synchronises its
// stream before it returns, so the buffer is free again by then; portable + mapped, so that every device the thread
// builds on can write its read-back block into it); nullptr if pinned memory cannot be had.
static unsigned *pinned_stage(size_t words)
{
    struct Stage { unsigned *p = nullptr; size_t cap = 0; };
    static thread_local Stage t;
    if (words > t.cap) {
        if (t.p) cudaFreeHost(t.p);
        t.p = nullptr; t.cap = 0;
        const size_t want = std::max<size_t>(words * 2, 4096);
        if (cudaHostAlloc((void **)&t.p, want * sizeof(unsigned), cudaHostAllocMapped | cudaHostAllocPortable) != cudaSuccess) { cudaGetLastError(); t.p = nullptr; return nullptr; }
        t.cap = want;
    }
    return t.p;
}

int build_index(DeviceIndex &ix, const float *points, const fps_build_opts &o)
{
    // ix.poff_host[0..B] = first point of every cloud in the concatenated arrays (set by the caller);
    // N = the largest cloud: grids, the voxel bound and the radix chunks are sized for it
    const int B = ix.B, N = ix.N;
    const int *ph = ix.poff_host;
    cudaStream_t st = (cudaStream_t)o.stream;
    ix.last_stream = st;
    int n_vox = o.n_vox > 0 ? o.n_vox : auto_n_vox(N);
    if (n_vox > 1024) { set_error("n_vox=%d out of range [1,1024]", n_vox); return FPS_ERR_INVALID; }
    // tiles of <= 64 points by default; for very large clouds the tile grows so that the per-voxel state
    // of the sampling kernel (60 B per tile, shared memory of <= 15 worker CTAs) still fits
    int auto_tile = 64;
    while ((long long)auto_tile * 24000 < N) auto_tile *= 2;
    int tile_points = o.tile_points == 0 ? auto_tile : (o.tile_points < 0 ? 0 : o.tile_points);
    const int vbits = 3 * ilog2_ceil((unsigned long long)n_vox);
    int sb = tile_points > 0 ? (32 - vbits) / 3 : 0;
    if (sb > 4) sb = 4;
    // An index of small clouds built with default options is sampled by the small-cloud kernel (sample_batched.cu,
    // choose_batched_shape), which uses the sorted order only: 16 key bits -- two radix passes instead of three -- order
    // the points finely enough for its runs of 64 (measured: same sampling time, the build 5-8 us shorter)
    if (N <= 8192 && o.cluster_size == 0 && (o.local_warps == 0 || o.local_warps == 32) && !(o.flags & (FPS_FLAG_NO_BATCH | FPS_FLAG_PER_PICK)))
        while (sb > 0 && vbits + 3 * sb > 16) --sb;
    const int keybits = vbits + 3 * sb;
    ix.n_vox = n_vox;
    ix.tile_points = tile_points;
    ix.flags = o.flags;

    // upper bound of the (tiled) voxel count, known before anything runs: no host round-trip is
    // needed to size the voxel arrays
    const long long cells = (long long)n_vox * n_vox * n_vox;
    long long kb = std::min<long long>(N, cells) + (tile_points > 0 ? N / tile_points : 0);
    kb = std::min<long long>(kb, N);
    ix.K_cap = (int)((kb + 31) / 32 * 32);
    ix.G_cap = ix.K_cap / 32;

    const size_t BN = (size_t)ph[B];      // all points of the batch
    const int nchunk = (N + RS_CHUNK - 1) / RS_CHUNK;
    const size_t table_n = (size_t)256 * nchunk;       // per cloud
    const bool per_pick = o.flags & FPS_FLAG_PER_PICK;

    Scratch sc;
    unsigned *meta = nullptr;      // [0] = largest segment, then (persistent arena only)
    unsigned *rb = nullptr;        // the read-back block (persistent arena)
    auto carve = [&](Carver &c, bool persistent) {
        if (persistent) {
            ix.px = c.take<float>(BN); ix.py = c.take<float>(BN); ix.pz = c.take<float>(BN);
            ix.porig = c.take<int32_t>(BN); ix.pinv = c.take<int32_t>(BN); ix.Dp = c.take<float>(BN);
            ix.vgeom = c.take<float4>((size_t)B * ix.K_cap);
            ix.vseg = c.take<int2>((size_t)B * ix.K_cap);
            ix.ggeom = c.take<float4>((size_t)B * ix.G_cap);
            ix.vstate = per_pick ? c.take<uint4>((size_t)B * ix.K_cap) : nullptr;
            // read-back block: K per cloud, meta, the bounding boxes (with the non-finite flags) -- contiguous, so
            // that the one host round-trip of the build is ONE copy
            rb = c.take<unsigned>((size_t)B + 8 + (size_t)B * BBOX_STRIDE);
            ix.K_dev = reinterpret_cast<int32_t *>(rb);
            meta = rb ? rb + B : nullptr;
            sc.bbox = rb ? rb + B + 8 : nullptr;
            ix.poff_dev = c.take<int32_t>(B + 1);
            ix.rag_dev = c.take<int32_t>(3 * (size_t)(B + 1));
            ix.counters = c.take<unsigned long long>(NUM_COUNTERS);

        } else {
            sc.kA = c.take<unsigned>(BN); sc.kB = c.take<unsigned>(BN);
            sc.vA = c.take<int>(BN); sc.vB = c.take<int>(BN);
            sc.table = c.take<int>(table_n * B);
            sc.bsum = c.take<int>((size_t)scan_tmp_ints((int)std::max((size_t)N, table_n), B));
            sc.heads = c.take<int>(BN); sc.rank = c.take<int>(BN); sc.voff = c.take<int>(BN);
            sc.ntl = c.take<int>(BN); sc.tbase = c.take<int>(BN);
            sc.Kv = c.take<int>(B);
        }
    };
    const bool fused = N <= FUSED_MAX_N && !(o.flags & FPS_FLAG_CHAIN_BUILD);     // one launch, all intermediates in shared memory
    Carver sizeP, sizeS;
    carve(sizeP, true);
    carve(sizeS, false);
    void *arena = nullptr, *scratch = nullptr;
    ix.arena_pooled = build_pool() != nullptr;
    // (the single-launch build needs none of the chain's intermediate arrays)
    if (pool_alloc(&arena, sizeP.off, st) != cudaSuccess || (!fused && pool_alloc(&scratch, sizeS.off, st) != cudaSuccess)) {
        set_error("device allocation of %zu + %zu bytes failed: %s", sizeP.off, sizeS.off, cudaGetErrorString(cudaGetLastError()));
        if (arena) { if (ix.arena_pooled) cudaFreeAsync(arena, st); else cudaFree(arena); }
        return FPS_ERR_NOMEM;
    }
    ix.arena = arena;
    ix.device_bytes = (int64_t)sizeP.off;
    Carver cp, cs;
    cp.base = (char *)arena;
    cs.base = (char *)scratch;
    carve(cp, true);
    if (!fused) carve(cs, false);
    auto release_scratch = [&]() { if (scratch) { if (ix.arena_pooled) cudaFreeAsync(scratch, st); else cudaFree(scratch); } };

    LaunchLog log;
    const int sms = device_props().sm_count;
    const dim3 gN((N + 255) / 256, B);
    // a failing enqueue below must not leak the scratch block: every exit goes through release_scratch()
    const size_t rb_n = (size_t)B + 8 + (size_t)B * BBOX_STRIDE;
    unsigned *const stage = pinned_stage((size_t)(B + 1) + rb_n);      // [B + 1] offsets in, [rb_n] read-back out
    // single-launch build with pinned staging: the kernel writes the read-back values straight into the (mapped) host
    // block and, for equal-size clouds, computes the offsets itself -- no memset, no copy in, no copy out
    int *host_rb_dev = nullptr;
    // mid-size clouds: one launch too, one thread-block cluster per cloud (k_build_cluster)
    // (measured: C2 0.172 -> 0.112 ms, C4 0.240 -> 0.152 ms; a single cloud of 150 000 points on 16 CTAs takes 0.203 ms
    // against 0.164 ms for the chain, which spreads it over the whole GPU: beyond 8 192 points per CTA, or for one
    // cloud of more than 65 536 points, the chain stays)
    const bool clustered = !fused && N <= CL_MAX_N && (N + cluster_build_ctas(N) - 1) / cluster_build_ctas(N) <= 8192 && (N <= 65536 || B >= 2) &&
                           !(o.flags & FPS_FLAG_CHAIN_BUILD) && stage != nullptr;
    if ((fused || clustered) && stage && cudaHostGetDevicePointer((void **)&host_rb_dev, stage + (B + 1), 0) != cudaSuccess) { cudaGetLastError(); host_rb_dev = nullptr; }
    const bool zero_copy = host_rb_dev != nullptr, poff_in_kernel = zero_copy && !ix.ragged;
    unsigned *chain_rb_dev = nullptr;     // kernel chain: the last kernel copies the read-back block to the host
    const void *poff_src = ph;
    if (stage) { memcpy(stage, ph, sizeof(int32_t) * (B + 1)); poff_src = stage; }
    cudaError_t e0 = zero_copy ? cudaSuccess : cudaMemsetAsync(meta, 0, 8 * sizeof(unsigned), st);
    if (e0 == cudaSuccess && !poff_in_kernel) e0 = cudaMemcpyAsync(ix.poff_dev, poff_src, sizeof(int32_t) * (B + 1), cudaMemcpyHostToDevice, st);
    if (e0 != cudaSuccess) {
        set_error("index build: enqueueing the first copies failed: %s", cudaGetErrorString(e0));
        release_scratch();
        return FPS_ERR_CUDA;
    }
    const int *poff = ix.poff_dev;
    if (fused) {
        // small clouds: the whole build in ONE launch, one CTA per cloud (k_build_fused)
        FusedArgs fa;
        fa.pts = points; fa.poff = poff; fa.bbox = sc.bbox;
        fa.n_vox = n_vox; fa.hb = vbits / 3; fa.sb = sb; fa.keybits = keybits; fa.tile_points = tile_points;
        fa.K_cap = ix.K_cap; fa.G_cap = ix.G_cap; fa.Nmax = N;
        fa.px = ix.px; fa.py = ix.py; fa.pz = ix.pz; fa.porig = ix.porig; fa.pinv = ix.pinv;
        fa.vseg = ix.vseg; fa.vgeom = ix.vgeom; fa.ggeom = ix.ggeom; fa.K_dev = ix.K_dev;
        fa.maxcnt = reinterpret_cast<int *>(meta);
        fa.host_rb = host_rb_dev; fa.B = B;
        if (poff_in_kernel) { fa.uniform_N = N; fa.poff_out = ix.poff_dev; }
        if (!fused_attr_set()) {
            set_error("cudaFuncSetAttribute(k_build_fused) failed: %s", cudaGetErrorString(cudaGetLastError()));
            release_scratch();
            return FPS_ERR_CUDA;
        }
        launch_pdl_smem(log, fused_smem_bytes(N), k_build_fused, dim3(B), dim3(FUSED_T), st, fa);
    } else if (clustered && zero_copy) {
        const int C = cluster_build_ctas(N), Np = (N + C - 1) / C;
        ClusterArgs ca;
        FusedArgs &fa = ca.f;
        fa.pts = points; fa.poff = poff; fa.bbox = sc.bbox;
        fa.n_vox = n_vox; fa.hb = vbits / 3; fa.sb = sb; fa.keybits = keybits; fa.tile_points = tile_points;
        fa.K_cap = ix.K_cap; fa.G_cap = ix.G_cap; fa.Nmax = Np;
        fa.px = ix.px; fa.py = ix.py; fa.pz = ix.pz; fa.porig = ix.porig; fa.pinv = ix.pinv;
        fa.vseg = ix.vseg; fa.vgeom = ix.vgeom; fa.ggeom = ix.ggeom; fa.K_dev = ix.K_dev;
        fa.maxcnt = reinterpret_cast<int *>(meta);
        fa.host_rb = host_rb_dev; fa.B = B;
        if (poff_in_kernel) { fa.uniform_N = N; fa.poff_out = ix.poff_dev; }
        ca.F1g = sc.heads;
        if (!fused_attr_set()) {
            set_error("cudaFuncSetAttribute(k_build_cluster) failed: %s", cudaGetErrorString(cudaGetLastError()));
            release_scratch();
            return FPS_ERR_CUDA;
        }
        launch_pdl_cluster(log, cluster_smem_bytes(Np), C, k_build_cluster, dim3(B * C), dim3(FUSED_T), st, ca);
    } else {
    launch_pdl(log, k_bbox_init, dim3((B * BBOX_STRIDE + 255) / 256), dim3(256), st, sc.bbox, B);
    launch_pdl(log, k_bbox, dim3(dim3(std::max(1, std::min((N + 4095) / 4096, sms)), B)), dim3(256), st, points, poff, sc.bbox);
    launch_pdl(log, k_keys, dim3(gN), dim3(256), st, points, poff, sc.bbox, n_vox, vbits / 3, sb, sc.kA, sc.vA);

    // a3: LSD radix sort, 8 bits per pass
    unsigned *kin = sc.kA, *kout = sc.kB;
    int *vin = sc.vA, *vout = sc.vB;
    const dim3 gR((nchunk + RS_WARPS - 1) / RS_WARPS, B);
    for (int shift = 0; shift < keybits; shift += 8) {
        launch_pdl(log, k_radix_hist, dim3(gR), dim3(RS_WARPS * 32), st, kin, poff, nchunk, shift, sc.table);
        scan_exclusive(log, sc.table, sc.table, (int)table_n, (int)table_n, B, nullptr, sc.bsum, st);
        launch_pdl(log, k_radix_scatter, dim3(gR), dim3(RS_WARPS * 32), st, kin, vin, poff, nchunk, shift, sc.table, kout, vout);
        std::swap(kin, kout);
        std::swap(vin, vout);
    }

    // a5: grid voxels -> (tiled) segments; a4: gather; a6: spheres
    launch_pdl(log, k_heads, dim3(gN), dim3(256), st, kin, poff, 3 * sb, sc.heads);
    scan_exclusive(log, sc.heads, sc.rank, N, N, B, sc.Kv, sc.bsum, st, poff);
    launch_pdl(log, k_voxel_offsets, dim3(gN), dim3(256), st, sc.heads, sc.rank, poff, sc.voff);
    launch_pdl(log, k_ntiles, dim3(gN), dim3(256), st, sc.voff, sc.Kv, poff, tile_points, sc.ntl);
    scan_exclusive(log, sc.ntl, sc.tbase, N, N, B, ix.K_dev, sc.bsum, st, poff);
    launch_pdl(log, k_tiles, dim3(gN), dim3(256), st, sc.voff, sc.Kv, sc.ntl, sc.tbase, poff, ix.K_cap, ix.vseg);
    launch_pdl(log, k_gather, dim3(gN), dim3(256), st, points, vin, poff, ix.px, ix.py, ix.pz, ix.porig, ix.pinv);
    const int sphere_blocks = std::max(1, std::min((ix.K_cap + 7) / 8, sms * 8));
    launch_pdl(log, k_sphere, dim3(dim3(sphere_blocks, B)), dim3(256), st, ix.px, ix.py, ix.pz, ix.vseg, ix.K_dev, poff, ix.K_cap, ix.vgeom,
               reinterpret_cast<int *>(meta));
    const int group_blocks = std::max(1, std::min((ix.G_cap + 7) / 8, sms * 8));
    if (stage && cudaHostGetDevicePointer((void **)&chain_rb_dev, stage + (B + 1), 0) != cudaSuccess) { cudaGetLastError(); chain_rb_dev = nullptr; }
    launch_pdl(log, k_group_sphere, dim3(dim3(group_blocks, B)), dim3(256), st, ix.vgeom, ix.K_dev, ix.K_cap, ix.G_cap, ix.ggeom,
               (const unsigned *)rb, chain_rb_dev, (int)rb_n);
    }
    {
        const cudaError_t el = log.first_error != cudaSuccess ? log.first_error : cudaGetLastError();
        if (el != cudaSuccess) {
            set_error("a build kernel failed to launch: %s", cudaGetErrorString(el));
            cudaGetLastError();
            release_scratch();
            return FPS_ERR_CUDA;
        }
    }

    // the one host round-trip of the build: K per cloud, the non-finite flags, the largest segment
    ix.K_host = (int32_t *)malloc(sizeof(int32_t) * B);
    std::vector<unsigned> hrb_pageable(stage ? 0 : rb_n);
    unsigned *const hrb = stage ? stage + (B + 1) : hrb_pageable.data();
    if (!ix.K_host) { set_error("host malloc failed"); release_scratch(); return FPS_ERR_NOMEM; }
    cudaError_t e1 = (zero_copy || chain_rb_dev) ? cudaSuccess : cudaMemcpyAsync(hrb, rb, sizeof(unsigned) * rb_n, cudaMemcpyDeviceToHost, st);
    release_scratch();
    cudaError_t e4 = cudaStreamSynchronize(st);
    if (e1 != cudaSuccess || e4 != cudaSuccess) {
        set_error("index build failed on the device: %s", cudaGetErrorString(e4 != cudaSuccess ? e4 : e1));
        return FPS_ERR_CUDA;
    }
    if (zero_copy) {                      // [3][B]: K, largest segment, non-finite flag (written by k_build_fused)
        const int *h3 = reinterpret_cast<const int *>(hrb);
        memcpy(ix.K_host, h3, sizeof(int32_t) * B);
        ix.max_voxel_points = 0;
        for (int b = 0; b < B; ++b) ix.max_voxel_points = std::max(ix.max_voxel_points, h3[B + b]);
        for (int b = 0; b < B; ++b)
            if (h3[2 * B + b]) {
                set_error("cloud %d holds a NaN or infinite coordinate", b);
                return FPS_ERR_NONFINITE;
            }
    } else {
        memcpy(ix.K_host, hrb, sizeof(int32_t) * B);
        ix.max_voxel_points = (int)hrb[B];
        const unsigned *hb = hrb + B + 8;
        for (int b = 0; b < B; ++b)
            if (hb[(size_t)b * BBOX_STRIDE + 6]) {
                set_error("cloud %d holds a NaN or infinite coordinate", b);
                return FPS_ERR_NONFINITE;
            }
    }
    ix.K_max = 0;
    ix.K_total = 0;
    for (int b = 0; b < B; ++b) {
        ix.K_max = std::max(ix.K_max, ix.K_host[b]);
        ix.K_total += ix.K_host[b];
    }
    ix.build_launches = log.launches;
    return per_pick ? choose_launch_shape(ix, o) : choose_batched_shape(ix, o);
}

// ---------------------------------------------------------------------------------------------
// fps_sample_noalloc (radiusfps.h): the whole path a1-a13 for ONE cloud of <= FPS_NOALLOC_MAX_N points without a
// single device allocation.  The voxel index -- everything build_index() carves out of its arena: the sorted point
// arrays, Dist_p, the voxel and group records, the read-back block -- is scratch memory of such a call, and here it
// lives in a file-scope device array that every GPU loading the library holds until the process exits.
//
// In host code `g_noalloc_scratch` is only a stand-in for the symbol, not a device address: its address is resolved
// once per device, with that device current, by cudaGetSymbolAddress, and it is this pointer that the kernels get.
// Every call on a device shares the array and finds the previous call's contents in it; the one block that has to
// start at zero (meta: the running maximum of the segment sizes) is cleared on the stream before the build kernel;
// everything else is written before it is read (k_build_fused writes the whole index and the bounding box block,
// the sampling kernel initialises Dist_p).  Two calls that overlap on the GPU -- different streams without an
// ordering between them, or two host threads -- race on the array; on one stream they are ordered.
// ---------------------------------------------------------------------------------------------
static_assert(FPS_NOALLOC_MAX_N <= FUSED_MAX_N, "the no-allocation entry point uses the single-launch build");
static __device__ __align__(256) unsigned char g_noalloc_scratch[FPS_NOALLOC_SCRATCH_BYTES];

static int noalloc_scratch_ptr(unsigned char **out)
{
    static std::mutex mu;
    static unsigned char *ptr[64] = {};
    int dev = 0;
    RFPS_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) { set_error("device ordinal %d is not supported by fps_sample_noalloc", dev); return FPS_ERR_INVALID; }
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p) {
            set_error("cudaGetSymbolAddress(g_noalloc_scratch) failed on device %d: %s", dev, cudaGetErrorString(e));
            cudaGetLastError();
            return FPS_ERR_CUDA;
        }
        ptr[dev] = static_cast<unsigned char *>(p);
    }
    *out = ptr[dev];
    return FPS_OK;
}

int sample_noalloc(const float *points, int32_t N, int32_t M, int32_t start_idx, int32_t flags, int32_t *out_idx, float *out_mindist,
                   cudaStream_t st)
{
    if (N > FPS_NOALLOC_MAX_N) {
        set_error("fps_sample_noalloc: N=%d is above FPS_NOALLOC_MAX_N=%d (the static scratch array holds the index of one cloud of at most "
                  "that many points); use fps_index_build + fps_sample", N, (int)FPS_NOALLOC_MAX_N);
        return FPS_ERR_INVALID;
    }
    unsigned char *base = nullptr;
    const int rcp = noalloc_scratch_ptr(&base);
    if (rcp != FPS_OK) return rcp;

    // the same parameters as build_index() picks for this N
    int32_t poff_h[2] = {0, N}, K_h[1] = {0};
    DeviceIndex ix;
    ix.B = 1; ix.N = N;
    ix.poff_host = poff_h;            // (stack storage: this index is never handed to free_index)
    ix.K_host = K_h;
    ix.last_stream = st;
    fps_build_opts o;
    memset(&o, 0, sizeof o);
    o.flags = flags;
    o.stream = (void *)st;
    const int n_vox = auto_n_vox(N);
    const int tile_points = 64;
    const int vbits = 3 * ilog2_ceil((unsigned long long)n_vox);
    const int sb = std::min(4, (32 - vbits) / 3);
    const int keybits = vbits + 3 * sb;
    ix.n_vox = n_vox; ix.tile_points = tile_points; ix.flags = flags;
    const long long cells = (long long)n_vox * n_vox * n_vox;
    const long long kb = std::min<long long>(std::min<long long>(N, cells) + N / tile_points, N);
    ix.K_cap = (int)((kb + 31) / 32 * 32);
    ix.G_cap = ix.K_cap / 32;

    Carver c;
    c.base = reinterpret_cast<char *>(base);
    const size_t BN = (size_t)N;
    ix.px = c.take<float>(BN); ix.py = c.take<float>(BN); ix.pz = c.take<float>(BN);
    ix.porig = c.take<int32_t>(BN); ix.pinv = c.take<int32_t>(BN); ix.Dp = c.take<float>(BN);
    ix.vgeom = c.take<float4>((size_t)ix.K_cap);
    ix.vseg = c.take<int2>((size_t)ix.K_cap);
    ix.ggeom = c.take<float4>((size_t)ix.G_cap);
    constexpr size_t RB_N = 1 + 8 + BBOX_STRIDE;          // K, meta, the bounding box block (with the non-finite flag)
    unsigned *rb = c.take<unsigned>(RB_N);
    ix.K_dev = reinterpret_cast<int32_t *>(rb);
    unsigned *meta = rb + 1, *bbox = rb + 1 + 8;
    ix.poff_dev = c.take<int32_t>(2);
    ix.counters = c.take<unsigned long long>(NUM_COUNTERS);
    if (c.off > (size_t)FPS_NOALLOC_SCRATCH_BYTES) {
        set_error("fps_sample_noalloc: the index of N=%d points needs %zu bytes, the static scratch array holds %zu", N, c.off,
                  (size_t)FPS_NOALLOC_SCRATCH_BYTES);
        return FPS_ERR_INVALID;
    }
    ix.device_bytes = (int64_t)c.off;

    RFPS_CUDA(cudaMemsetAsync(meta, 0, 8 * sizeof(unsigned), st));     // the array keeps the last call's contents
    RFPS_CUDA(cudaMemcpyAsync(ix.poff_dev, poff_h, sizeof poff_h, cudaMemcpyHostToDevice, st));
    FusedArgs fa;
    fa.pts = points; fa.poff = ix.poff_dev; fa.bbox = bbox;
    fa.n_vox = n_vox; fa.hb = vbits / 3; fa.sb = sb; fa.keybits = keybits; fa.tile_points = tile_points;
    fa.K_cap = ix.K_cap; fa.G_cap = ix.G_cap; fa.Nmax = N;
    fa.px = ix.px; fa.py = ix.py; fa.pz = ix.pz; fa.porig = ix.porig; fa.pinv = ix.pinv;
    fa.vseg = ix.vseg; fa.vgeom = ix.vgeom; fa.ggeom = ix.ggeom; fa.K_dev = ix.K_dev;
    fa.maxcnt = reinterpret_cast<int *>(meta);
    if (!fused_attr_set()) { set_error("cudaFuncSetAttribute(k_build_fused) failed: %s", cudaGetErrorString(cudaGetLastError())); return FPS_ERR_CUDA; }
    LaunchLog log;
    launch_pdl_smem(log, fused_smem_bytes(N), k_build_fused, dim3(1), dim3(FUSED_T), st, fa);
    {
        const cudaError_t el = log.first_error != cudaSuccess ? log.first_error : cudaGetLastError();
        if (el != cudaSuccess) {
            set_error("the build kernel failed to launch: %s", cudaGetErrorString(el));
            cudaGetLastError();
            return FPS_ERR_CUDA;
        }
    }
    // the build's one host round-trip (K sizes the sampling kernel's shared memory; the non-finite flag)
    unsigned hrb[RB_N];
    RFPS_CUDA(cudaMemcpyAsync(hrb, rb, sizeof hrb, cudaMemcpyDeviceToHost, st));
    RFPS_CUDA(cudaStreamSynchronize(st));
    if (hrb[1 + 8 + 6]) { set_error("the cloud holds a NaN or infinite coordinate"); return FPS_ERR_NONFINITE; }
    K_h[0] = (int32_t)hrb[0];
    ix.max_voxel_points = (int)hrb[1];
    ix.K_max = K_h[0];
    ix.K_total = K_h[0];
    ix.build_launches = log.launches;
    int rcs = choose_batched_shape(ix, o);
    if (rcs == FPS_OK && ix.grid_ctas > 0) {               // grid mode would allocate exchange blocks: one cluster instead
        fps_build_opts oc = o;
        oc.cluster_size = std::max(1, std::min(8, N / 1024));
        rcs = choose_batched_shape(ix, oc);
    }
    if (rcs != FPS_OK) return rcs;
    if (ix.grid_ctas > 0) { set_error("fps_sample_noalloc: unexpected grid mode"); return FPS_ERR_INVALID; }
    return launch_sample_batched(ix, M, start_idx, nullptr, (int64_t)(M - 1), out_idx, out_mindist, st);
}

}  // namespace rfps
