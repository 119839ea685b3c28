// api.cu -- the C-ABI of include/imager.h: argument checks, plan life cycle, call sequencing.
#include <cstdarg>
#include <cstdio>
#include <cmath>
#include <new>
#include "common.cuh"

namespace imager {

static thread_local char g_err[512] = "";

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

int num_sms() {
    static int cached[64] = {};                      // per device ordinal; a B200 has 148
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
    if (!cached[dev]) {
        int n = 0;
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
        cached[dev] = n;
    }
    return cached[dev];
}

int cuda_fail(cudaError_t e, const char* what) {
    set_error("CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
    return e == cudaErrorMemoryAllocation ? IMAGER_ERR_NOMEM : IMAGER_ERR_CUDA;
}

static int check_params(const imager_params* p) {
    if (!p) { set_error("params is NULL"); return IMAGER_ERR_INVALID_ARG; }
    if (p->grid_size < 2 || (p->grid_size & 1) || p->grid_size > 32768) {
        set_error("grid_size must be even and in [2, 32768]"); return IMAGER_ERR_INVALID_ARG; }
    if (!((p->n_corr == 1 && p->n_pol == 1) || (p->n_corr == 4 && p->n_pol == 4))) {
        set_error("only n_corr = n_pol = 1 or 4 are built"); return IMAGER_ERR_UNSUPPORTED; }
    if (p->n_wplanes < 1 || p->n_wplanes > 4096) { set_error("n_wplanes out of range"); return IMAGER_ERR_INVALID_ARG; }
    if (p->n_wplanes > 1 && !(p->w_max > 0)) { set_error("w_max must be > 0 when n_wplanes > 1"); return IMAGER_ERR_INVALID_ARG; }
    if (p->support_min < 1 || p->support_max < p->support_min || p->support_max > 255 ||
        ((p->support_max - p->support_min) & 1)) {
        set_error("need 1 <= support_min <= support_max <= 255 with an even difference"); return IMAGER_ERR_INVALID_ARG; }
    if (p->support_max > p->grid_size) { set_error("support exceeds the grid"); return IMAGER_ERR_INVALID_ARG; }
    if (p->oversample < 1 || p->oversample > 128 || (p->oversample > 1 && (p->oversample & 1))) {
        set_error("oversample must be 1 or even, <= 128"); return IMAGER_ERR_INVALID_ARG; }
    if (p->n_aplanes < 1) { set_error("n_aplanes must be >= 1"); return IMAGER_ERR_INVALID_ARG; }
    if (p->kernel_mode < IMAGER_MODE_DELTA || p->kernel_mode > IMAGER_MODE_USER) {
        set_error("unknown kernel_mode"); return IMAGER_ERR_INVALID_ARG; }
    if (p->kernel_mode == IMAGER_MODE_DELTA &&
        !(p->support_min == 1 && p->support_max == 1 && p->oversample == 1 && p->n_wplanes == 1 && p->n_aplanes == 1 &&
          p->n_corr == 1)) {
        set_error("DELTA mode needs support 1, oversample 1, one plane, one correlation"); return IMAGER_ERR_INVALID_ARG; }
    if ((p->kernel_mode == IMAGER_MODE_AWPROJ_ADJOINT || p->kernel_mode == IMAGER_MODE_AWPROJ_PAPER) && p->n_corr != 4) {
        set_error("AWPROJ modes need n_corr = n_pol = 4"); return IMAGER_ERR_INVALID_ARG; }
    if ((p->kernel_mode == IMAGER_MODE_PSWF || p->kernel_mode == IMAGER_MODE_WPROJ ||
         p->kernel_mode == IMAGER_MODE_MOSAIC_PB) && p->n_corr != 1) {
        set_error("PSWF / WPROJ / MOSAIC_PB modes are single-polarisation"); return IMAGER_ERR_INVALID_ARG; }
    if (!(p->cell_size_rad > 0)) { set_error("cell_size_rad must be > 0"); return IMAGER_ERR_INVALID_ARG; }
    if (p->max_nvis < 0 || p->max_nvis > 2000000000LL) { set_error("max_nvis out of range"); return IMAGER_ERR_INVALID_ARG; }
    return 0;
}

static void free_plan(imager_plan* pl) {
    if (!pl) return;
    if (pl->index_done) cudaEventDestroy(pl->index_done);
    if (pl->d_tab_degrid && pl->d_tab_degrid != pl->d_tab_grid) cudaFree(pl->d_tab_degrid);
    cudaFree(pl->d_tab_grid);
    cudaFree(pl->d_set_offset);
    cudaFree(pl->d_set_support);
    cudaFree(pl->d_plane_support);
    cudaFree(pl->d_rec);
    cudaFree(pl->d_key[0]);
    cudaFree(pl->d_key[1]);
    cudaFree(pl->d_perm[0]);
    cudaFree(pl->d_perm[1]);
    cudaFree(pl->d_bucket_offset);
    cudaFree(pl->d_hist);
    cudaFree(pl->d_scan_tmp);
    cudaFree(pl->d_counters);
    cudaFree(pl->d_items);
    destroy_transform(pl);
    tiled_release(pl);
    delete pl;
}

}  // namespace imager

using namespace imager;

extern "C" const char* imager_last_error(void) { return g_err; }

extern "C" int imager_plan_create(const imager_params* params, void* cuda_stream, imager_plan** out_plan) {
    g_err[0] = 0;
    if (!out_plan) { set_error("out_plan is NULL"); return IMAGER_ERR_INVALID_ARG; }
    *out_plan = nullptr;
    int rc = check_params(params);
    if (rc) return rc;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        set_error("no CUDA device: libimager has no CPU fallback");
        return IMAGER_ERR_CUDA;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    imager_plan* pl = new (std::nothrow) imager_plan();
    if (!pl) return IMAGER_ERR_NOMEM;
    pl->p = *params;
    if (params->pointing_lm) pl->pointing_lm.assign(params->pointing_lm, params->pointing_lm + 2 * (size_t)params->n_aplanes);
    pl->p.pa_rad = nullptr;
    pl->p.pointing_lm = nullptr;
    pl->p.user_tables = pl->p.user_tables_degrid = nullptr;
    const imager_params& p = pl->p;
    const int P = p.n_wplanes, O = p.oversample;
    // R5: S_p = support_min + 2 rint(((support_max - support_min)/2) p/(P-1))
    pl->plane_support.resize(P);
    const int half = (p.support_max - p.support_min) / 2;
    for (int q = 0; q < P; ++q)
        pl->plane_support[q] = (P == 1) ? p.support_min
                                        : p.support_min + 2 * (int)std::nearbyint((double)(half * q) / (double)(P - 1));
    pl->n_sets = p.n_aplanes * (2 * P - 1);
    pl->set_support.resize(pl->n_sets);
    pl->set_offset.resize(pl->n_sets + 1);
    pl->set_offset[0] = 0;
    for (int k = 0; k < pl->n_sets; ++k) {
        const int sp = k % (2 * P - 1) - (P - 1);
        const int S = pl->plane_support[sp < 0 ? -sp : sp];
        pl->set_support[k] = S;
        pl->set_offset[k + 1] = pl->set_offset[k] + (int64_t)p.n_pol * p.n_corr * O * O * S * S;
    }
    pl->uv_scale = (double)O * (double)p.grid_size * p.cell_size_rad;       // R2: O*N exact, one rounding
    pl->w_scale = (P > 1) ? (double)(P - 1) / p.w_max : 0.0;
    pl->nt = (p.grid_size + kBucketTile - 1) / kBucketTile;
    const int64_t nb = (int64_t)pl->n_sets * pl->nt * pl->nt;
    if (nb * O * O >= (int64_t)kKeyDrop) {
        free_plan(pl);
        set_error("bucket key needs more than 32 bits");
        return IMAGER_ERR_UNSUPPORTED;
    }
    pl->n_buckets = (int)nb;
    pl->key_drop = (uint32_t)(nb * O * O);                // one more than the largest valid key
    pl->key_bits = 1;
    while (((int64_t)1 << pl->key_bits) <= nb * O * O) pl->key_bits++;      // bits of the drop key
    pl->sort_passes = (pl->key_bits + 7) / 8;
    const int64_t mv = p.max_nvis > 0 ? p.max_nvis : 1;
    const int64_t n_chunks = (mv + kSortChunk - 1) / kSortChunk;
    const int64_t hist_len = 256 * n_chunks;
    pl->scan_tmp_len = 0;
    for (int64_t n = std::max<int64_t>(hist_len, nb + 1); n > 1; n = (n + 1023) / 1024) pl->scan_tmp_len += (n + 1023) / 1024 + 1;
#define PLAN_CUDA(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { free_plan(pl); return cuda_fail(e__, #call); } } while (0)
    PLAN_CUDA(cudaMalloc(&pl->d_set_offset, (pl->n_sets + 1) * sizeof(int64_t)));
    PLAN_CUDA(cudaMalloc(&pl->d_set_support, pl->n_sets * sizeof(int32_t)));
    PLAN_CUDA(cudaMalloc(&pl->d_plane_support, P * sizeof(int32_t)));
    PLAN_CUDA(cudaMemcpyAsync(pl->d_set_offset, pl->set_offset.data(), (pl->n_sets + 1) * sizeof(int64_t), cudaMemcpyHostToDevice, st));
    PLAN_CUDA(cudaMemcpyAsync(pl->d_set_support, pl->set_support.data(), pl->n_sets * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    PLAN_CUDA(cudaMemcpyAsync(pl->d_plane_support, pl->plane_support.data(), P * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    PLAN_CUDA(cudaMalloc(&pl->d_rec, mv * sizeof(imager_record)));
    for (int i = 0; i < 2; ++i) {
        PLAN_CUDA(cudaMalloc(&pl->d_key[i], mv * sizeof(uint32_t)));
        PLAN_CUDA(cudaMalloc(&pl->d_perm[i], mv * sizeof(int32_t)));
    }
    PLAN_CUDA(cudaMalloc(&pl->d_bucket_offset, (nb + 1) * sizeof(int32_t)));
    PLAN_CUDA(cudaMalloc(&pl->d_hist, hist_len * sizeof(int32_t)));
    PLAN_CUDA(cudaMalloc(&pl->d_scan_tmp, (pl->scan_tmp_len + 16) * sizeof(int32_t)));
    PLAN_CUDA(cudaMalloc(&pl->d_counters, 64 * sizeof(int32_t)));
    PLAN_CUDA(cudaMemsetAsync(pl->d_counters, 0, 64 * sizeof(int32_t), st));
    pl->max_items = (int64_t)pl->n_sets * pl->nt * pl->nt;
    PLAN_CUDA(cudaMalloc(&pl->d_items, (pl->max_items + 1) * 4 * sizeof(int32_t)));
    PLAN_CUDA(cudaEventCreateWithFlags(&pl->index_done, cudaEventDisableTiming));
    PLAN_CUDA(cudaStreamSynchronize(st));
#undef PLAN_CUDA
    rc = build_tables(pl, params, st);
    if (rc) { free_plan(pl); return rc; }
    *out_plan = pl;
    return 0;
}

extern "C" int imager_plan_destroy(imager_plan* plan) {
    free_plan(plan);
    return 0;
}

static int ensure_index(imager_plan* pl, int64_t nvis, const float* uvw, const int32_t* a_index, uint32_t flags,
                        cudaStream_t st) {
    if (nvis < 0) { set_error("nvis < 0"); return IMAGER_ERR_INVALID_ARG; }
    if (nvis > pl->p.max_nvis) { set_error("nvis exceeds max_nvis"); return IMAGER_ERR_TOO_MANY_VIS; }
    if ((flags & IMAGER_REUSE_INDEX) && pl->index_valid && pl->indexed_nvis == nvis) return 0;
    if (nvis > 0 && !uvw) { set_error("uvw is NULL"); return IMAGER_ERR_INVALID_ARG; }
    const int rc = run_index_and_sort(pl, nvis, uvw, a_index, st);
    if (rc == 0 && pl->index_done) IMAGER_CUDA(cudaEventRecord(pl->index_done, st));
    return rc;
}

extern "C" int imager_index(imager_plan* plan, int64_t nvis, const float* uvw, const int32_t* a_index, void* cuda_stream) {
    g_err[0] = 0;
    if (!plan) { set_error("plan is NULL"); return IMAGER_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    plan->last_launches = 0;
    int rc = ensure_index(plan, nvis, uvw, a_index, 0, st);
    if (rc) return rc;
    return tiled_supported(plan) ? tiled_prepare(plan, nvis, st) : 0;
}

extern "C" int imager_grid(imager_plan* plan, int64_t nvis, const float* uvw, const float* vis, const float* weights,
                           const int32_t* a_index, float* grid, double* sum_weights, uint32_t flags, void* cuda_stream) {
    g_err[0] = 0;
    if (!plan || !grid || (nvis > 0 && (!vis || !weights))) { set_error("NULL argument"); return IMAGER_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    plan->last_launches = 0;
    int rc = ensure_index(plan, nvis, uvw, a_index, flags, st);
    if (rc) return rc;
    rc = launch_sum_weights(plan, nvis, (const float2*)vis, weights, sum_weights, st);
    if (rc) return rc;
    if (!(flags & IMAGER_PATH_REFERENCE) && tiled_supported(plan))
        return launch_grid_tiled(plan, nvis, (const float2*)vis, weights, (float2*)grid, st);
    return launch_grid_reference(plan, nvis, (const float2*)vis, weights, (float2*)grid, nullptr, st);
}

extern "C" int imager_degrid(imager_plan* plan, int64_t nvis, const float* uvw, const int32_t* a_index, const float* grid,
                             float* vis_out, uint32_t flags, void* cuda_stream) {
    g_err[0] = 0;
    if (!plan || !grid || (nvis > 0 && !vis_out)) { set_error("NULL argument"); return IMAGER_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    plan->last_launches = 0;
    int rc = ensure_index(plan, nvis, uvw, a_index, flags, st);
    if (rc) return rc;
    const int residual = (flags & IMAGER_DEGRID_RESIDUAL) ? 1 : 0;
    if (!(flags & IMAGER_PATH_REFERENCE) && tiled_supported(plan))
        return launch_degrid_tiled(plan, nvis, (const float2*)grid, (float2*)vis_out, residual, st);
    return launch_degrid_reference(plan, nvis, (const float2*)grid, (float2*)vis_out, nullptr, residual, st);
}

extern "C" int imager_grid_image_transform(imager_plan* plan, float* data, int32_t direction, double norm,
                                           void* cuda_stream) {
    g_err[0] = 0;
    if (!plan || !data) { set_error("NULL argument"); return IMAGER_ERR_INVALID_ARG; }
    return grid_image_transform(plan, (float2*)data, direction, norm, (cudaStream_t)cuda_stream);
}

extern "C" int imager_mosaic_correct(imager_plan* plan, float* image, void* cuda_stream) {
    g_err[0] = 0;
    if (!plan || !image) { set_error("NULL argument"); return IMAGER_ERR_INVALID_ARG; }
    if (plan->p.kernel_mode != IMAGER_MODE_MOSAIC_PB) {
        set_error("imager_mosaic_correct needs a MOSAIC_PB plan");
        return IMAGER_ERR_INVALID_ARG;
    }
    return mosaic_correct(plan, (float2*)image, (cudaStream_t)cuda_stream);
}

extern "C" int imager_debug_index(imager_plan* plan, int64_t nvis, const float* uvw, const int32_t* a_index,
                                  imager_record* records_out, int32_t* perm_out, uint32_t* keys_out,
                                  int32_t* bucket_offset_out, int64_t* n_kept_out, void* cuda_stream) {
    g_err[0] = 0;
    if (!plan) { set_error("plan is NULL"); return IMAGER_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    plan->last_launches = 0;
    int rc = ensure_index(plan, nvis, uvw, a_index, 0, st);
    if (rc) return rc;
    IMAGER_CUDA(cudaStreamSynchronize(st));
    const int b = plan->sorted_buf;
    if (records_out && nvis) IMAGER_CUDA(cudaMemcpy(records_out, plan->d_rec, nvis * sizeof(imager_record), cudaMemcpyDeviceToHost));
    if (perm_out && nvis) IMAGER_CUDA(cudaMemcpy(perm_out, plan->d_perm[b], nvis * sizeof(int32_t), cudaMemcpyDeviceToHost));
    if (keys_out && nvis) {
        IMAGER_CUDA(cudaMemcpy(keys_out, plan->d_key[b], nvis * sizeof(uint32_t), cudaMemcpyDeviceToHost));
        for (int64_t i = nvis - 1; i >= 0 && keys_out[i] == plan->key_drop; --i) keys_out[i] = kKeyDrop;   // sorted: drops last
    }
    if (bucket_offset_out)
        IMAGER_CUDA(cudaMemcpy(bucket_offset_out, plan->d_bucket_offset, ((size_t)plan->n_buckets + 1) * sizeof(int32_t), cudaMemcpyDeviceToHost));
    if (n_kept_out) {
        int32_t c[2];
        IMAGER_CUDA(cudaMemcpy(c, plan->d_counters, sizeof(c), cudaMemcpyDeviceToHost));
        *n_kept_out = c[0];
    }
    return 0;
}

extern "C" int imager_debug_kernels(imager_plan* plan, int32_t kset, int32_t which, float* host_out, int32_t* support_out) {
    g_err[0] = 0;
    if (!plan || kset < 0 || kset >= plan->n_sets) { set_error("bad plan / kset"); return IMAGER_ERR_INVALID_ARG; }
    if (support_out) *support_out = plan->set_support[kset];
    if (host_out) {
        const float2* src = (which ? plan->d_tab_degrid : plan->d_tab_grid) + plan->set_offset[kset];
        const int64_t n = plan->set_offset[kset + 1] - plan->set_offset[kset];
        IMAGER_CUDA(cudaMemcpy(host_out, src, n * sizeof(float2), cudaMemcpyDeviceToHost));
    }
    return 0;
}

extern "C" int imager_index_stats(imager_plan* plan, int64_t out[8], void* cuda_stream) {
    g_err[0] = 0;
    if (!plan || !out) { set_error("NULL argument"); return IMAGER_ERR_INVALID_ARG; }
    if (!plan->index_valid) { set_error("no index yet: call imager_index / imager_grid / imager_degrid first"); return IMAGER_ERR_INVALID_ARG; }
    return tiled_index_stats(plan, out, (cudaStream_t)cuda_stream);
}

extern "C" int imager_last_launch_count(imager_plan* plan) {
    return plan ? plan->last_launches : (int)IMAGER_ERR_INVALID_ARG;
}

extern "C" int imager_plan_path(imager_plan* plan, char* why_out, int32_t why_len) {
    g_err[0] = 0;
    if (!plan || why_len < 0 || (why_len > 0 && !why_out)) { set_error("NULL argument"); return IMAGER_ERR_INVALID_ARG; }
    const char* why = tiled_unsupported_reason(plan);
    if (why_len > 0) snprintf(why_out, (size_t)why_len, "%s", why ? why : "");
    return why ? 0 : 1;
}

extern "C" int imager_plan_info(imager_plan* plan, int64_t info_out[8]) {
    g_err[0] = 0;
    if (!plan || !info_out) { set_error("NULL argument"); return IMAGER_ERR_INVALID_ARG; }
    int32_t c[2] = {0, 0};
    // the counters are written by the last indexing, on whatever stream that ran (possibly a non-blocking one, which the
    // legacy-stream copy below would not wait for): wait for the event recorded behind it first
    if (plan->index_done) IMAGER_CUDA(cudaEventSynchronize(plan->index_done));
    IMAGER_CUDA(cudaMemcpy(c, plan->d_counters, sizeof(c), cudaMemcpyDeviceToHost));
    info_out[0] = plan->n_sets;
    info_out[1] = kBucketTile;
    info_out[2] = plan->n_buckets;
    info_out[3] = plan->key_bits;
    info_out[4] = c[1];
    info_out[5] = plan->last_launches;
    info_out[6] = plan->set_offset[plan->n_sets];
    info_out[7] = c[0];
    return 0;
}
