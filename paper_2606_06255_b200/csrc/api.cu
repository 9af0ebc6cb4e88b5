// api.cu -- the C-ABI of include/radiusfps.h: argument validation, error strings, handle lifetime.
// Every step of the path runs in the kernels of index_build.cu / sample_kernel.cu; there is no CPU
// fallback anywhere in this library.
#include <cstdlib>
#include <cstring>
#include <new>

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

}  // namespace rfps

using rfps::set_error;

extern "C" {

const char *fps_last_error(void) { return rfps::g_err; }
const char *fps_version(void) { return "radiusfps-b200 0.1 (sm_100a)"; }
int fps_last_status(void) { return rfps::g_status; }

fps_index_t *fps_index_build_ex(const float *points, int32_t N, int32_t B, const fps_build_opts *opts)
{
    rfps::g_err[0] = 0;
    rfps::g_status = FPS_ERR_INVALID;
    if (!points) { set_error("points is NULL"); return nullptr; }
    if (N < 1 || B < 1) { set_error("N=%d and B=%d must be >= 1", N, B); return nullptr; }
    if ((long long)N * B > (1ll << 30)) { set_error("B*N=%lld exceeds 2^30", (long long)N * B); return nullptr; }
    fps_build_opts o;
    memset(&o, 0, sizeof o);
    if (opts) o = *opts;
    if (o.n_vox < 0 || o.n_vox > 1024) { set_error("n_vox=%d out of range [0,1024]", o.n_vox); return nullptr; }
    fps_index_t *h = new (std::nothrow) fps_index_t();
    if (!h) { set_error("host allocation failed"); return nullptr; }
    h->ix.B = B;
    h->ix.N = N;
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
    if (h->ix.flags & FPS_FLAG_PER_PICK)
        return rfps::launch_sample(h->ix, M, start_idx, out_idx, out_mindist, (cudaStream_t)stream);
    return rfps::launch_sample_batched(h->ix, M, start_idx, out_idx, out_mindist, (cudaStream_t)stream);
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
    out->local_warps = ix.local_warps; out->cand_per_thread = ix.cand_per_thread;
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
            if (getenv("RFPS_DEBUG")) fprintf(stderr, "[rfps debug] local phase cycles (sum over clouds): select %llu pick-loop %llu apply %llu\n", c[21], c[22], c[23]);
        }
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
