/*
 * radiusfps.h -- C-ABI of the B200-native RadiusFPS hot path.
 *
 * Exact farthest point sampling accelerated by spherical-voxel pruning
 * (arxiv/paper_2606_06255; PAPER.md = the paper's text).  The library computes, for every
 * cloud of a batch, the sequence defined by Eq. 3
 *
 *     s_j = argmax_{p in P}  min_{s in S_{j-1}}  d2(p, s),      j = 1 .. M-1,   s_0 = P[start_idx]
 *
 * under the exactness contract of PAPER.md:179 (same seed, same floating-point precision, argmax
 * ties -> smallest original input index), with
 *
 *     d2(p, s) = ((dx*dx + dy*dy) + dz*dz),  dx = p.x - s.x, ...   fp32, round-to-nearest-even,
 *                                                                   no FMA contraction
 *
 * (BASELINE.json north_star; the paper itself writes the Euclidean norm, Eq. 1/29).  The result
 * is bit-identical to classical FPS (Alg. 1); the voxel index only removes work
 * that cannot change it (Eq. 20-30).
 *
 * Conventions
 *   - Every pointer named "DEVICE" is a CUDA device pointer on the current device; every other
 *     pointer is a host pointer.  No torch types appear anywhere in this interface.
 *   - The caller owns points, out_idx and out_mindist.  The library owns everything inside a
 *     handle and frees it in fps_index_destroy.
 *   - Functions returning int return FPS_OK (0) or a negative fps_status.  fps_last_error()
 *     returns a thread-local, NUL-terminated description of the last failure on this thread.
 *   - A handle holds mutable sampling state (Dist_p, Dist_v): calls on ONE handle must not
 *     overlap, and one handle is used on ONE stream at a time (fps_index_destroy releases the memory
 *     stream-ordered behind the last fps_sample / fps_gather_xyz call only); different handles are
 *     independent, also across host threads.
 */
#ifndef RADIUSFPS_H
#define RADIUSFPS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fps_index fps_index_t;   /* opaque */

typedef enum {
    FPS_OK            =  0,
    FPS_ERR_INVALID   = -1,  /* bad argument: N<1, B<1, M<1, M>N, start_idx outside [0,N), NULL pointer,
                                unsupported option value                                              */
    FPS_ERR_CUDA      = -2,  /* a CUDA runtime call or kernel launch failed                           */
    FPS_ERR_NONFINITE = -3,  /* a coordinate is NaN or +-inf (the method has no defined answer)       */
    FPS_ERR_NOMEM     = -4   /* device or host allocation failed                                      */
} fps_status;

/* Build options.  NOTHING here may change the sampled indices or min-distances: the options only
 * move work around (the voxel resolution n_vox is a free parameter of the method, PAPER.md:192,
 * :695; results are identical for every value).  Zero-initialise, then set what you need.       */
typedef struct {
    int32_t n_vox;         /* voxel bins per axis (Eq. 7); 0 = choose from N; 1..1024   */
    int32_t tile_points;   /* split voxels holding more points than this into tiles with their own
                              bounding sphere; 0 = default, -1 = never split (the paper's layout)      */
    int32_t cluster_size;  /* CTAs per cloud in the sampling kernel: 0 = choose; 1..16 = one thread-block cluster of
                              that size per cloud (per-pick kernel: 1,2,4,8,16); batched kernel only: -2..-148 =
                              that many CTAs per cloud spread over the whole grid (one picker, the others workers,
                              exchanging through global memory; needs B * CTAs <= SMs).  With 0, an index whose
                              clouds all hold <= 8 192 points is sampled by the one-CTA-per-cloud kernel that keeps
                              the whole cloud in registers (fps_stats.whole_cloud_kernel); any explicit value, a
                              local_warps other than 0 / 32, or FPS_FLAG_NO_BATCH selects the general kernel       */
    int32_t block_threads; /* threads per CTA: 0 = choose; 128..1024, multiple of 32                    */
    int32_t flags;         /* FPS_FLAG_* below                                                          */
    void   *stream;        /* cudaStream_t the build is issued on (0 = the legacy default stream)       */
    int32_t local_warps;   /* batched kernel, local phase: 0 = choose; 32 = parallel resolution (all 16 warps hold
                              candidates, the top <= 64 are resolved into picks per step; the default);
                              16 = hierarchical (all 16 warps hold candidates, one warp picks sequentially from the
                              top <= 96 of them); 4, 1, 8 = flat FPS on that many warps                          */
    int32_t cand_per_thread; /* candidates per thread (registers): 0 = choose; 2, 4, 8 with local_warps 32 / 16
                              (capacity 512 * cand_per_thread; 16 with local_warps 32 for clouds of <= 8 192 points,
                              small-cloud kernel only); flat shapes: 8 with 4 or 1 warps, 16 with 8                */
} fps_build_opts;

enum {
    FPS_FLAG_NO_PRUNE = 1,  /* ablation: visit every voxel (Eq. 25 never taken)                         */
    FPS_FLAG_NO_SKIP  = 2,  /* ablation: no coordinate-wise point skip (Eq. 28 never taken)             */
    FPS_FLAG_STATS    = 4,  /* count voxel tests / visited voxels / visited points / effective updates  */
    FPS_FLAG_NO_BATCH = 8,  /* ablation: every batch of the batched kernel is the single global argmax  */
    FPS_FLAG_PER_PICK = 16, /* run the per-pick persistent kernel (one cluster-wide exchange per sample,
                               the paper's iteration structure) instead of exact batched picking        */
    FPS_FLAG_CHAIN_BUILD = 64, /* build the index with the chain of ~22 kernels also for clouds that by default take a
                               single-launch build (one CTA per cloud up to 8 192 points, one thread-block cluster
                               per cloud up to 65 536 points -- batches: ~130 000); same voxels, tiles and samples */
    FPS_FLAG_EUCLIDEAN = 32 /* NOT an option that leaves results alone: sample with the Euclidean distance
                               sqrt_rn(d2), the paper's literal Eq. 1 / Eq. 29, instead of
                               d2.  out_mindist then holds distances.  In fp32 this is a different function:
                               maxima that differ in d2 can round to the same square root and tie (lowest
                               index wins).  Batched kernel with the default local phase only.              */
};

/* Counters and layout facts, summed over the B clouds (fps_get_stats).  With the batched kernel
 * voxel_tests / points_visited / points_computed count (voxel, pick) and (point, pick) pairs.      */
typedef struct {
    int32_t B, N;             /* clouds; points per cloud (the largest cloud of a ragged index)       */
    int32_t n_vox;            /* resolution actually used                                             */
    int32_t cluster_size, block_threads, voxels_per_thread;
    int64_t K_total;          /* active (tiled) voxels over all clouds                                */
    int32_t K_max;            /* largest per-cloud K                                                  */
    int32_t max_voxel_points; /* largest segment                                                      */
    int64_t device_bytes;     /* memory owned by the handle                                           */
    int32_t build_launches;   /* kernels fps_index_build launched (a1-a6); fps_sample launches ONE    */
    int32_t grid_ctas;        /* batched kernel: > 0 = CTAs per cloud spread over the grid (cooperative launch,
                                 exchange through global memory); 0 = one cluster of cluster_size CTAs per cloud */
    /* the following are filled only when FPS_FLAG_STATS was set, for the LAST fps_sample call:      */
    int64_t iterations;       /* sum over clouds of (M-1)                                             */
    int64_t voxel_tests;      /* Eq. 25 evaluations                                                   */
    int64_t voxels_visited;   /* voxels that survived the prune                                       */
    int64_t points_visited;   /* points in visited voxels                                             */
    int64_t points_computed;  /* points that passed the skip test                                     */
    int64_t effective;        /* strict decreases of Dist_p (Eq. 2)                     */
    /* batched kernel only (zero for FPS_FLAG_PER_PICK):                                              */
    int64_t rounds;           /* global rounds (apply + extract + local phase)                        */
    int64_t extract_retries;  /* candidate extractions repeated because the buffer overflowed         */
    int64_t single_picks;     /* rounds that fell back to the single global argmax                    */
    int64_t candidates;       /* candidates handed to the local phase, summed over rounds             */
    int64_t extract_voxels;   /* voxels scanned by the extraction                                     */
    int64_t extract_points;   /* points scanned by the extraction                                     */
    int64_t cycles_apply, cycles_max, cycles_extract, cycles_local;   /* SM cycles spent per phase, as seen
                                 by thread 0 of each cloud's first CTA, summed over clouds             */
    int64_t group_tests;      /* (group of 32 voxels, pick) prune tests; voxel_tests then counts only the
                                 pairs whose group survived                                           */
    int64_t cycles_prune_sum, cycles_visit_sum;   /* APPLY split: prune tests / point visits, SM cycles
                                 summed over ALL CTAs                                                 */
    int64_t cycles_prune_max, cycles_visit_max;   /* the same for the slowest CTA                       */
    int64_t sub_batches;      /* groups of <= 128 picks applied between two CTA barriers              */
    int64_t local_subrounds;  /* hierarchical local phase: sub-rounds (one-warp FPS runs)             */
    int64_t local_fallbacks;  /* ... of which single block-wide argmax picks (first bin overflowed)   */
    int32_t local_warps, cand_per_thread;   /* local-phase shape actually used                        */
    int64_t cycles_local_select, cycles_local_pick, cycles_local_update;   /* hierarchical local phase, SM cycles
                                 seen by thread 0 of the picker CTA, summed over clouds: candidate selection /
                                 the pick loop (parallel resolution: all pairs + resolving) / applying the picks
                                 to the candidates after it                                                    */
    int64_t cycles_local_pairs, cycles_local_publish;   /* parallel resolution: the all-pairs part of cycles_local_pick;
                                 publishing a step's picks to the workers (release at cluster scope)          */
    int64_t cycles_worker_tail, cycles_worker_extract, cycles_worker_idle;   /* worker CTAs, thread 0, summed over all
                                 workers: applying what is left of a batch once it is declared complete / the candidate
                                 extraction scans / waiting for the next message                              */
    int64_t worker_pieces;    /* pieces of <= 128 picks applied, summed over all workers                       */
    int32_t whole_cloud_kernel; /* 1: every cloud holds <= 8 192 points and is sampled by the one-CTA-per-cloud
                                 kernel (whole cloud in registers, radius prune on runs of 64 sorted points; the
                                 voxel / point counters then count those runs); 0: the general kernel          */
    int32_t reserved0;
} fps_stats;

/*
 * fps_index_build -- steps a1-a6 of the hot path: on-device spherical-voxel index
 * (Alg. 2 Phases 1-3; Eq. 6-10).
 *
 *   points  DEVICE, fp32, contiguous [B][N][3] (array of structures, row-major).  Read during the
 *           call only; not referenced afterwards.
 *   N       points per cloud, >= 1.     B  clouds, >= 1.  Every cloud gets its own bounding box,
 *           grid, active-voxel list and sorted structure-of-arrays copy.
 *
 * Work is issued on the legacy default stream (fps_index_build) or on opts->stream (_ex); the
 * call returns when the index is complete (it synchronises that stream).  Returns NULL on
 * failure; fps_last_error() says why (FPS_ERR_NONFINITE if a coordinate is not finite).
 */
fps_index_t *fps_index_build(const float *points, int32_t N, int32_t B);
fps_index_t *fps_index_build_ex(const float *points, int32_t N, int32_t B, const fps_build_opts *opts);

/*
 * fps_sample -- steps a7-a13: M-1 fused iterations of {select, radius prune (Eq. 25), point skip
 * (Eq. 28), fp32 min-distance update (Eq. 29), per-voxel max (Eq. 30), global argmax (Eq. 15-18)}
 * in ONE persistent kernel launch, for all B clouds at once.
 *
 *   M            samples per cloud, 1 <= M <= N.       start_idx  first sample of every cloud.
 *   out_idx      DEVICE int32 [B][M]: ORIGINAL input indices in selection order; out_idx[b][0] ==
 *                start_idx.
 *   out_mindist  DEVICE fp32 [B][M]: squared fp32 distance of sample j to the nearest earlier
 *                sample at the moment it was chosen (= max_i Dist_p[i]); out_mindist[b][0] = +inf.
 *   stream       cudaStream_t (as void*) the launch is enqueued on; the call does not synchronise.
 *
 * May be called any number of times on one handle (any M, any start_idx); every call restarts
 * from Dist_p = +inf.  On a negative return nothing has been enqueued.
 */
int fps_sample(fps_index_t *h, int32_t M, int32_t start_idx,
               int32_t *out_idx, float *out_mindist, void *stream);

/*
 * Ragged batches: clouds of different sizes in one index, and per-cloud sample
 * counts and start points in one launch.  The paper's workloads are variable-size scenes
 * (Fig. 1); every cloud is sampled exactly as by fps_index_build + fps_sample on it alone.
 *
 *   points     DEVICE fp32 [offsets[B]][3]: the clouds one after the other.
 *   offsets    HOST int32 [B+1], offsets[0] = 0, strictly increasing: cloud b = points offsets[b] ..
 *              offsets[b+1]-1.  Read during the call only.
 *   M          HOST int32 [B], 1 <= M[b] <= N_b.       start_idx  HOST int32 [B] or NULL (= all 0).
 *   out_idx / out_mindist  DEVICE [sum M[b]]: cloud b's samples start at M[0] + .. + M[b-1]; indices
 *              are relative to the cloud's own first point.
 * fps_sample (one M, one start_idx) also works on a ragged index if they fit every cloud.
 */
fps_index_t *fps_index_build_ragged(const float *points, const int32_t *offsets, int32_t B, const fps_build_opts *opts);
int fps_sample_ragged(fps_index_t *h, const int32_t *M, const int32_t *start_idx,
                      int32_t *out_idx, float *out_mindist, void *stream);

/*
 * fps_gather_xyz -- coordinates of sampled points: out_xyz[..][j] = the input point
 * with original index idx[..][j], read from the index's own sorted copy (the caller's `points` buffer is not
 * needed any more).  idx: DEVICE int32, out_xyz: DEVICE fp32, 3 floats per sample, same layout as idx:
 * [B][M] for M >= 1; M = 0 means the ragged layout of the last fps_sample_ragged call on this handle.
 * An index outside its cloud yields NaN coordinates.  Asynchronous on `stream`.
 */
int fps_gather_xyz(fps_index_t *h, const int32_t *idx, int32_t M, float *out_xyz, void *stream);

/*
 * fps_pick_chain_cycles -- measurement aid, not part of the path: SM cycles per pick of the bare dependent
 * chain of one pick on one warp (update -> lane max -> redux(max D) -> redux(slot id) -> 3 shared loads)
 * with cand_per_lane = 1, 2 or 4 candidates per lane, averaged over `iters` picks.  This is the latency
 * floor of the sequential part of FPS on this GPU; bench.py reports the achieved
 * cycles per pick against it.  cycles_per_pick: HOST.  Synchronous, default stream.
 */
int fps_pick_chain_cycles(int32_t cand_per_lane, int32_t iters, float *cycles_per_pick);

/* Frees the handle and all device memory it owns (stream-ordered behind the last call on the handle).
 * NULL is allowed.  The memory goes back to a library-private pool that keeps it for the next build;
 * fps_trim() returns whatever the pool holds unused to the driver. */
void fps_index_destroy(fps_index_t *h);
void fps_trim(void);

/*
 * fps_sample_noalloc -- the whole path (index build a1-a6 + sampling a7-a13, Algorithm 1 / Sec. 3.2-3.4) for
 * ONE cloud, for callers that must not allocate device memory (tight serving loops, harnesses that forbid
 * cudaMalloc).  It calls no cudaMalloc / cudaFree / pool routine and creates no handle: the voxel index, which is
 * scratch memory of such a call, lives in a static device array of FPS_NOALLOC_SCRATCH_BYTES (512 KiB) that every GPU
 * loading the library holds until the process exits.  Results are bit-identical to fps_index_build + fps_sample with
 * default options on the same cloud.
 *   points       DEVICE [N][3] fp32, finite; N in [1, FPS_NOALLOC_MAX_N = 8192] -- a larger N is rejected with
 *                FPS_ERR_INVALID and a message naming the limit (nothing is launched)
 *   M, start_idx as for fps_sample (1 <= M <= N, 0 <= start_idx < N)
 *   flags        0, or FPS_FLAG_EUCLIDEAN; any other flag is rejected
 *   out_idx      DEVICE [M] int32, out_mindist DEVICE [M] fp32: owned by the caller, written by the call
 *   stream       cudaStream_t (NULL = default stream) of the CURRENT device
 * The call synchronises `stream` once (the build's read-back of the voxel count, as fps_index_build does) and returns
 * with the sampling kernel enqueued.  ALL calls on one device share the one static array: it keeps the previous
 * call's contents (the call clears what has to start at zero), calls on the same stream are ordered, and calls that
 * overlap on the GPU -- different streams without an ordering between them, several host threads -- RACE on it; the
 * caller serialises them.  Errors: FPS_ERR_INVALID (arguments, N above the limit), FPS_ERR_NONFINITE, FPS_ERR_CUDA.
 */
#define FPS_NOALLOC_MAX_N 8192
#define FPS_NOALLOC_SCRATCH_BYTES (512 * 1024)
int fps_sample_noalloc(const float *points, int32_t N, int32_t M, int32_t start_idx, int32_t flags, int32_t *out_idx,
                       float *out_mindist, void *stream);

/* Layout facts and (with FPS_FLAG_STATS) the counters of the last fps_sample; synchronises the
 * stream of that call.  out: host pointer. */
int fps_get_stats(fps_index_t *h, fps_stats *out);

/*
 * fps_sample_host -- the same path for callers whose data lives in HOST memory: copies
 * points [B][N][3] to the device, builds the index, samples, copies out_idx / out_mindist
 * (HOST, [B][M]) back and destroys the index.  Synchronous.  opts may be NULL.
 */
int fps_sample_host(const float *points_host, int32_t N, int32_t B, int32_t M, int32_t start_idx,
                    int32_t *out_idx_host, float *out_mindist_host, const fps_build_opts *opts);

/*
 * fps_build_and_sample -- the one-shot call: index build, sampling and release of
 * the index for a batch that is sampled once, as the first sampling layer of a network does with every
 * scene; the build is then on the critical path.  The batch is cut into chunks of
 * consecutive clouds; the index of chunk k+1 is built on an internal stream while the sampling kernel of
 * chunk k runs on opts->stream.  Every cloud is sampled exactly as by fps_index_build + fps_sample on it
 * alone: chunking changes the schedule, never a result.
 *
 *   points        DEVICE fp32 [total][3], the clouds one after the other.
 *   offsets       HOST int32 [B+1] (as fps_index_build_ragged), or NULL: B clouds of N points each.
 *   M             HOST int32 [B], or NULL: every cloud yields M_all samples.
 *   start_idx     HOST int32 [B], or NULL: every cloud starts at its point 0.
 *   out_idx / out_mindist   DEVICE, cloud b's samples start at M[0] + .. + M[b-1] (b * M_all).
 *   opts          NULL or build options; opts->stream is the stream `points` was produced on and the results
 *                 are ordered on.
 *   chunk_clouds  clouds per chunk; 0 or >= B: one chunk (the fastest schedule measured on B200: the
 *                 sampling time of a chunk is latency-bound and hardly depends on its size).  Smaller
 *                 chunks bound the device memory of the index (about 100 B per point of one chunk).
 *
 * Returns when the last sampling kernel is enqueued.  Every index build ends with one small device-to-host
 * read (voxel counts, non-finite flags) and synchronises the stream it runs on: with several chunks that is
 * the internal stream, so opts->stream is never waited for; with ONE chunk (the default) the build runs on
 * opts->stream itself and the call therefore waits for everything enqueued on it before.  On a negative
 * return the chunks before the failing one have been enqueued and the rest of the outputs is untouched.
 */
int fps_build_and_sample(const float *points, const int32_t *offsets, int32_t N, int32_t B,
                         const int32_t *M, int32_t M_all, const int32_t *start_idx,
                         int32_t *out_idx, float *out_mindist, const fps_build_opts *opts, int32_t chunk_clouds);

/* Thread-local description of the last error on the calling thread ("" if none). */
const char *fps_last_error(void);

/* fps_status of the last fps_index_build / fps_index_build_ex on the calling thread (those return
 * a pointer, so NULL alone cannot say why): FPS_OK after a success. */
int fps_last_status(void);

/* Library version string, e.g. "radiusfps-b200 0.1 (sm_100a)". */
const char *fps_version(void);

#ifdef __cplusplus
}
#endif
#endif /* RADIUSFPS_H */
