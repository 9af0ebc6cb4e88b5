// api.cu -- the C-ABI of include/radiusfps.h: argument validation, error strings, handle lifetime.
// Every step of the path runs in the kernels of index_build.cu / sample_kernel.cu; there is no CPU
// fallback anywhere in this library.
#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "internal.h"

namespace rfps {

static thread_local char g_err[512] = "";
static thread_local int g_build_rc = 0;   // status of the last fps_index_build* on this thread
static thread_local int g_status = 0;     // status of the last failing call on this thread (fps_last_status)

void set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
}

const DeviceProps &device_props()
{
    static std::mutex mu;
    static DeviceProps props[64];
    static bool known[64] = {};
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= 64) dev = 0;
    std::lock_guard<std::mutex> lock(mu);
    if (!known[dev]) {
        cudaDeviceGetAttribute(&props[dev].sm_count, cudaDevAttrMultiProcessorCount, dev);
        cudaDeviceGetAttribute(&props[dev].max_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
        if (props[dev].sm_count <= 0) props[dev].sm_count = 1;
        known[dev] = true;
    }
    return props[dev];
}

}  // namespace rfps

using rfps::set_error;

extern "C" {

const char *fps_last_error(void) { return rfps::g_err; }
const char *fps_version(void) { return "radiusfps-b200 0.1 (sm_100a)"; }
int fps_last_status(void) { return rfps::g_status; }

// common body of the three build entry points: `offsets` (host, [B+1]) or uniform clouds of N points
static fps_index_t *build_common(const float *points, int32_t N, int32_t B, const int32_t *offsets, const fps_build_opts *opts)
{
    rfps::g_err[0] = 0;
    rfps::g_status = FPS_ERR_INVALID;
    if (!points) { set_error("points is NULL"); return nullptr; }
    if (B < 1) { set_error("B=%d must be >= 1", B); return nullptr; }
    if (B > 65535) { set_error("B=%d: at most 65535 clouds per index (split the batch, or use fps_build_and_sample with chunk_clouds)", B); return nullptr; }
    long long total = 0;
    int32_t nmax = 0;
    if (offsets) {
        if (offsets[0] != 0) { set_error("offsets[0]=%d must be 0", offsets[0]); return nullptr; }
        for (int b = 0; b < B; ++b) {
            const long long nb = (long long)offsets[b + 1] - offsets[b];
            if (nb < 1) { set_error("cloud %d holds %lld points; every cloud needs >= 1", b, nb); return nullptr; }
            if (nb > nmax) nmax = (int32_t)nb;
        }
        total = offsets[B];
    } else {
        if (N < 1) { set_error("N=%d and B=%d must be >= 1", N, B); return nullptr; }
        total = (long long)N * B;
        nmax = N;
    }
    if (total > (1ll << 30)) { set_error("the batch holds %lld points, more than 2^30", total); return nullptr; }
    fps_build_opts o;
    memset(&o, 0, sizeof o);
    if (opts) o = *opts;
    if (o.n_vox < 0 || o.n_vox > 1024) { set_error("n_vox=%d out of range [0,1024]", o.n_vox); return nullptr; }
    if ((o.flags & FPS_FLAG_EUCLIDEAN) && (o.flags & FPS_FLAG_PER_PICK)) {
        set_error("FPS_FLAG_EUCLIDEAN is not available with FPS_FLAG_PER_PICK");
        return nullptr;
    }
    fps_index_t *h = new (std::nothrow) fps_index_t();
    if (!h) { set_error("host allocation failed"); return nullptr; }
    h->ix.B = B;
    h->ix.N = nmax;
    h->ix.ragged = offsets != nullptr;
    h->ix.poff_host = (int32_t *)malloc(sizeof(int32_t) * ((size_t)B + 1));
    h->ix.rag_host = (int32_t *)malloc(sizeof(int32_t) * 3 * ((size_t)B + 1));
    if (!h->ix.poff_host || !h->ix.rag_host) {
        set_error("host allocation failed");
        free(h->ix.poff_host); free(h->ix.rag_host);
        delete h;
        return nullptr;
    }
    for (int b = 0; b <= B; ++b) h->ix.poff_host[b] = offsets ? offsets[b] : (int32_t)((long long)b * N);
    int rc = rfps::build_index(h->ix, points, o);
    rfps::g_build_rc = rc;
    rfps::g_status = rc;
    if (rc != FPS_OK) {
        cudaStreamSynchronize((cudaStream_t)o.stream);
        char keep[sizeof rfps::g_err];
        memcpy(keep, rfps::g_err, sizeof keep);
        rfps::free_index(h->ix);
        delete h;
        cudaGetLastError();
        memcpy(rfps::g_err, keep, sizeof keep);
        return nullptr;
    }
    return h;
}

fps_index_t *fps_index_build_ex(const float *points, int32_t N, int32_t B, const fps_build_opts *opts)
{
    return build_common(points, N, B, nullptr, opts);
}

fps_index_t *fps_index_build_ragged(const float *points, const int32_t *offsets, int32_t B, const fps_build_opts *opts)
{
    if (!offsets) { rfps::g_status = FPS_ERR_INVALID; set_error("offsets is NULL"); return nullptr; }
    return build_common(points, 0, B, offsets, opts);
}

fps_index_t *fps_index_build(const float *points, int32_t N, int32_t B)
{
    return fps_index_build_ex(points, N, B, nullptr);
}

int fps_sample(fps_index_t *h, int32_t M, int32_t start_idx, int32_t *out_idx, float *out_mindist, void *stream)
{
    rfps::g_err[0] = 0;
    if (!h) { set_error("handle is NULL"); return FPS_ERR_INVALID; }
    if (!out_idx || !out_mindist) { set_error("output pointer is NULL"); return FPS_ERR_INVALID; }
    if (M < 1 || M > h->ix.N) { set_error("M=%d must be in [1, N=%d]", M, h->ix.N); return FPS_ERR_INVALID; }
    if (start_idx < 0 || start_idx >= h->ix.N) {
        set_error("start_idx=%d must be in [0, N=%d)", start_idx, h->ix.N);
        return FPS_ERR_INVALID;
    }
    if (h->ix.ragged) {
        for (int b = 0; b < h->ix.B; ++b) {
            const int nb = h->ix.poff_host[b + 1] - h->ix.poff_host[b];
            if (M > nb || start_idx >= nb) {
                set_error("cloud %d holds %d points: M=%d / start_idx=%d do not fit (use fps_sample_ragged)", b, nb, M, start_idx);
                return FPS_ERR_INVALID;
            }
        }
    }
    const int64_t iters = (int64_t)h->ix.B * (M - 1);
    if (h->ix.flags & FPS_FLAG_PER_PICK)
        return rfps::launch_sample(h->ix, M, start_idx, nullptr, iters, out_idx, out_mindist, (cudaStream_t)stream);
    return rfps::launch_sample_batched(h->ix, M, start_idx, nullptr, iters, out_idx, out_mindist, (cudaStream_t)stream);
}

int fps_sample_ragged(fps_index_t *h, const int32_t *M, const int32_t *start_idx, int32_t *out_idx, float *out_mindist,
                      void *stream)
{
    rfps::g_err[0] = 0;
    if (!h) { set_error("handle is NULL"); return FPS_ERR_INVALID; }
    if (!M || !out_idx || !out_mindist) { set_error("NULL argument"); return FPS_ERR_INVALID; }
    rfps::DeviceIndex &ix = h->ix;
    const int B = ix.B;
    // validate every cloud before touching the handle's state (rag_host / rag_M_max describe the LAST GOOD call)
    for (int b = 0; b < B; ++b) {
        const int nb = ix.poff_host[b + 1] - ix.poff_host[b];
        const int sb = start_idx ? start_idx[b] : 0;
        if (M[b] < 1 || M[b] > nb) { set_error("M[%d]=%d must be in [1, N_b=%d]", b, M[b], nb); return FPS_ERR_INVALID; }
        if (sb < 0 || sb >= nb) { set_error("start_idx[%d]=%d must be in [0, N_b=%d)", b, sb, nb); return FPS_ERR_INVALID; }
    }
    int32_t *r = ix.rag_host;                 // [3][B+1]: M_b, start_b, output offsets
    long long off = 0;
    int64_t iters = 0;
    int32_t mmax = 0;
    for (int b = 0; b < B; ++b) {
        r[b] = M[b];
        r[(B + 1) + b] = start_idx ? start_idx[b] : 0;
        r[2 * (B + 1) + b] = (int32_t)off;
        off += M[b];
        iters += M[b] - 1;
        mmax = std::max(mmax, M[b]);
    }
    ix.rag_M_max = mmax;
    r[B] = 0; r[(B + 1) + B] = 0; r[2 * (B + 1) + B] = (int32_t)off;
    cudaStream_t st = (cudaStream_t)stream;
    // pageable source: the copy is staged before the call returns, so rag_host can be reused by the next call
    RFPS_CUDA(cudaMemcpyAsync(ix.rag_dev, r, sizeof(int32_t) * 3 * ((size_t)B + 1), cudaMemcpyHostToDevice, st));
    if (ix.flags & FPS_FLAG_PER_PICK) return rfps::launch_sample(ix, 0, 0, ix.rag_dev, iters, out_idx, out_mindist, st);
    return rfps::launch_sample_batched(ix, 0, 0, ix.rag_dev, iters, out_idx, out_mindist, st);
}

int fps_gather_xyz(fps_index_t *h, const int32_t *idx, int32_t M, float *out_xyz, void *stream)
{
    rfps::g_err[0] = 0;
    if (!h || !idx || !out_xyz) { set_error("NULL argument"); return FPS_ERR_INVALID; }
    if (M < 0) { set_error("M=%d must be >= 0", M); return FPS_ERR_INVALID; }
    if (M == 0) {
        if (h->ix.rag_M_max <= 0) { set_error("M=0 means 'the layout of the last fps_sample_ragged call', but there was none"); return FPS_ERR_INVALID; }
        return rfps::launch_gather_xyz(h->ix, idx, 0, h->ix.rag_M_max, h->ix.rag_dev, out_xyz, (cudaStream_t)stream);
    }
    return rfps::launch_gather_xyz(h->ix, idx, M, M, nullptr, out_xyz, (cudaStream_t)stream);
}

int fps_pick_chain_cycles(int32_t cand_per_lane, int32_t iters, float *cycles_per_pick)
{
    rfps::g_err[0] = 0;
    if (!cycles_per_pick || iters < 1) { set_error("bad argument"); return FPS_ERR_INVALID; }
    return rfps::measure_pick_chain(cand_per_lane, iters, cycles_per_pick);
}

void fps_trim(void) { rfps::trim_pool(); }

int fps_sample_noalloc(const float *points, int32_t N, int32_t M, int32_t start_idx, int32_t flags, int32_t *out_idx, float *out_mindist,
                       void *stream)
{
    rfps::g_err[0] = 0;
    int rc = FPS_ERR_INVALID;
    if (!points) set_error("points is NULL");
    else if (!out_idx || !out_mindist) set_error("output pointer is NULL");
    else if (N < 1) set_error("N=%d must be >= 1", N);
    else if (M < 1 || M > N) set_error("M=%d must be in [1, N=%d]", M, N);
    else if (start_idx < 0 || start_idx >= N) set_error("start_idx=%d must be in [0, N=%d)", start_idx, N);
    else if (flags & ~FPS_FLAG_EUCLIDEAN) set_error("fps_sample_noalloc takes flags 0 or FPS_FLAG_EUCLIDEAN, got %d", flags);
    else rc = rfps::sample_noalloc(points, N, M, start_idx, flags, out_idx, out_mindist, (cudaStream_t)stream);
    if (rc != FPS_OK) rfps::g_status = rc;
    return rc;
}

void fps_index_destroy(fps_index_t *h)
{
    if (!h) return;
    rfps::free_index(h->ix);
    delete h;
}

int fps_get_stats(fps_index_t *h, fps_stats *out)
{
    rfps::g_err[0] = 0;
    if (!h || !out) { set_error("NULL argument"); return FPS_ERR_INVALID; }
    const rfps::DeviceIndex &ix = h->ix;
    memset(out, 0, sizeof *out);
    out->B = ix.B; out->N = ix.N; out->n_vox = ix.n_vox;
    out->cluster_size = ix.cluster_size; out->block_threads = ix.block_threads; out->voxels_per_thread = ix.vpt;
    out->K_total = ix.K_total; out->K_max = ix.K_max; out->max_voxel_points = ix.max_voxel_points;
    out->device_bytes = ix.device_bytes;
    out->build_launches = ix.build_launches;
    out->grid_ctas = ix.grid_ctas;
    out->local_warps = ix.local_warps; out->cand_per_thread = ix.cand_per_thread;
    out->whole_cloud_kernel = ix.whole ? 1 : 0;
    if (ix.flags & FPS_FLAG_STATS) {
        unsigned long long c[rfps::NUM_COUNTERS];
        RFPS_CUDA(cudaStreamSynchronize(ix.last_stream));
        RFPS_CUDA(cudaMemcpy(c, ix.counters, sizeof c, cudaMemcpyDeviceToHost));
        out->iterations = ix.last_iterations;
        out->voxel_tests = (int64_t)c[0];
        out->voxels_visited = (int64_t)c[1];
        out->points_visited = (int64_t)c[2];
        out->points_computed = (int64_t)c[3];
        out->effective = (int64_t)c[4];
        if (!(ix.flags & FPS_FLAG_PER_PICK)) {
            out->rounds = (int64_t)c[5]; out->extract_retries = (int64_t)c[6]; out->single_picks = (int64_t)c[7];
            out->candidates = (int64_t)c[8]; out->extract_voxels = (int64_t)c[9]; out->extract_points = (int64_t)c[10];
            out->cycles_apply = (int64_t)c[11]; out->cycles_max = (int64_t)c[12];
            out->cycles_extract = (int64_t)c[13]; out->cycles_local = (int64_t)c[14];
            out->group_tests = (int64_t)c[15];
            out->cycles_prune_sum = (int64_t)c[16]; out->cycles_visit_sum = (int64_t)c[17];
            out->cycles_prune_max = (int64_t)c[18]; out->cycles_visit_max = (int64_t)c[19];
            out->sub_batches = (int64_t)c[20];
            out->local_subrounds = (int64_t)c[24]; out->local_fallbacks = (int64_t)c[25];
            out->cycles_local_select = (int64_t)c[21]; out->cycles_local_pick = (int64_t)c[22]; out->cycles_local_update = (int64_t)c[23];
            out->cycles_local_pairs = (int64_t)c[26]; out->cycles_local_publish = (int64_t)c[27];
            out->cycles_worker_tail = (int64_t)c[28]; out->cycles_worker_extract = (int64_t)c[29];
            out->cycles_worker_idle = (int64_t)c[30]; out->worker_pieces = (int64_t)c[31];
        }
    }
    return FPS_OK;
}

// The pipelined one-shot call builds on a stream of its own, ordered behind the caller's stream by an event.
// Both are created per call and destroyed when the call returns (cudaStreamDestroy / cudaEventDestroy release
// the objects once the work already enqueued has finished), so two host threads calling at the same time
// never share a stream or re-record each other's event.
struct PipelineStream {
    cudaStream_t bs = nullptr;
    cudaEvent_t ev = nullptr;
    ~PipelineStream()
    {
        if (ev) cudaEventDestroy(ev);
        if (bs) cudaStreamDestroy(bs);
    }
};

int fps_build_and_sample(const float *points, const int32_t *offsets, int32_t N, int32_t B, const int32_t *M, int32_t M_all,
                         const int32_t *start_idx, int32_t *out_idx, float *out_mindist, const fps_build_opts *opts,
                         int32_t chunk_clouds)
{
    rfps::g_err[0] = 0;
    if (!points || !out_idx || !out_mindist) { set_error("NULL argument"); return FPS_ERR_INVALID; }
    if (B < 1) { set_error("B=%d must be >= 1", B); return FPS_ERR_INVALID; }
    if (!offsets && N < 1) { set_error("N=%d must be >= 1 when offsets is NULL", N); return FPS_ERR_INVALID; }
    if (!M && M_all < 1) { set_error("M_all=%d must be >= 1 when M is NULL", M_all); return FPS_ERR_INVALID; }
    if (chunk_clouds < 0) { set_error("chunk_clouds=%d must be >= 0", chunk_clouds); return FPS_ERR_INVALID; }
    if (offsets && offsets[0] != 0) { set_error("offsets[0]=%d must be 0", offsets[0]); return FPS_ERR_INVALID; }
    fps_build_opts o;
    memset(&o, 0, sizeof o);
    if (opts) o = *opts;
    cudaStream_t us = (cudaStream_t)o.stream;
    // auto = one chunk: a chunk's sampling time is set by the latency of its longest cloud, not by how many
    // clouds it holds, and the chunks' sampling kernels run one after the other; measured on B200 the
    // build that chunking hides never outweighs that.  Chunks are for bounding the
    // memory of the index (about 100 B per point, held for one chunk at a time)
    int chunk = chunk_clouds == 0 ? B : chunk_clouds;
    if (chunk > B) chunk = B;
    const bool pipelined = chunk < B;
    cudaStream_t bs = us;
    PipelineStream ps;
    if (pipelined) {
        RFPS_CUDA(cudaStreamCreateWithFlags(&ps.bs, cudaStreamNonBlocking));
        RFPS_CUDA(cudaEventCreateWithFlags(&ps.ev, cudaEventDisableTiming));
        bs = ps.bs;
        // the builds read `points` on the internal stream: order it behind what the caller enqueued
        RFPS_CUDA(cudaEventRecord(ps.ev, us));
        RFPS_CUDA(cudaStreamWaitEvent(bs, ps.ev, 0));
    }
    o.stream = (void *)bs;
    std::vector<int32_t> loc;
    long long out_off = 0;
    for (int c0 = 0; c0 < B; c0 += chunk) {
        const int Bk = std::min(chunk, B - c0);
        const float *pk = points + 3 * (size_t)(offsets ? offsets[c0] : (long long)c0 * N);
        fps_index_t *h;
        if (offsets) {
            loc.resize((size_t)Bk + 1);
            for (int i = 0; i <= Bk; ++i) loc[i] = offsets[c0 + i] - offsets[c0];
            h = build_common(pk, 0, Bk, loc.data(), &o);
        } else {
            h = build_common(pk, N, Bk, nullptr, &o);
        }
        if (!h) return rfps::g_build_rc ? rfps::g_build_rc : FPS_ERR_INVALID;
        // the index is complete (the build synchronised its stream): sample it on the caller's stream,
        // behind the previous chunk, while the host goes on to build the next chunk
        int rc;
        long long mk = 0;
        if (!M && !start_idx) {
            rc = fps_sample(h, M_all, 0, out_idx + out_off, out_mindist + out_off, (void *)us);
            mk = (long long)M_all * Bk;
        } else {
            std::vector<int32_t> mm((size_t)Bk), ss((size_t)Bk);
            for (int i = 0; i < Bk; ++i) {
                mm[i] = M ? M[c0 + i] : M_all;
                ss[i] = start_idx ? start_idx[c0 + i] : 0;
                mk += mm[i] > 0 ? mm[i] : 0;
            }
            rc = fps_sample_ragged(h, mm.data(), ss.data(), out_idx + out_off, out_mindist + out_off, (void *)us);
        }
        fps_index_destroy(h);      // stream-ordered behind the sampling kernel just enqueued
        if (rc != FPS_OK) return rc;
        out_off += mk;
    }
    return FPS_OK;
}

int fps_sample_host(const float *points_host, int32_t N, int32_t B, int32_t M, int32_t start_idx,
                    int32_t *out_idx_host, float *out_mindist_host, const fps_build_opts *opts)
{
    rfps::g_err[0] = 0;
    if (!points_host || !out_idx_host || !out_mindist_host) { set_error("NULL argument"); return FPS_ERR_INVALID; }
    if (N < 1 || B < 1 || M < 1 || M > N || start_idx < 0 || start_idx >= N) {
        set_error("bad sizes N=%d B=%d M=%d start_idx=%d", N, B, M, start_idx);
        return FPS_ERR_INVALID;
    }
    fps_build_opts o;
    memset(&o, 0, sizeof o);
    if (opts) o = *opts;
    cudaStream_t st = (cudaStream_t)o.stream;
    float *d_pts = nullptr, *d_mind = nullptr;
    int32_t *d_idx = nullptr;
    const size_t pb = sizeof(float) * 3 * (size_t)N * B, ob = sizeof(int32_t) * (size_t)M * B;
    int rc = FPS_OK;
    fps_index_t *h = nullptr;
    auto fail = [&](int code) {
        rfps::dev_free_async(d_pts, st); rfps::dev_free_async(d_idx, st); rfps::dev_free_async(d_mind, st);
        if (h) fps_index_destroy(h);
        return code;
    };
    if (rfps::dev_alloc_async((void **)&d_pts, pb, st) != cudaSuccess || rfps::dev_alloc_async((void **)&d_idx, ob, st) != cudaSuccess ||
        rfps::dev_alloc_async((void **)&d_mind, ob, st) != cudaSuccess) {
        set_error("device allocation failed in fps_sample_host");
        cudaGetLastError();
        return fail(FPS_ERR_NOMEM);
    }
    if (cudaMemcpyAsync(d_pts, points_host, pb, cudaMemcpyHostToDevice, st) != cudaSuccess) {
        set_error("H2D copy failed: %s", cudaGetErrorString(cudaGetLastError()));
        return fail(FPS_ERR_CUDA);
    }
    h = fps_index_build_ex(d_pts, N, B, &o);
    if (!h) return fail(rfps::g_build_rc ? rfps::g_build_rc : FPS_ERR_INVALID);
    rc = fps_sample(h, M, start_idx, d_idx, d_mind, st);
    if (rc != FPS_OK) return fail(rc);
    if (cudaMemcpyAsync(out_idx_host, d_idx, ob, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaMemcpyAsync(out_mindist_host, d_mind, ob, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess) {
        set_error("D2H copy / kernel failed: %s", cudaGetErrorString(cudaGetLastError()));
        return fail(FPS_ERR_CUDA);
    }
    return fail(FPS_OK);
}

}  // extern "C"
