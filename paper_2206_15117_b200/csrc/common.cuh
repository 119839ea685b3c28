// common.cuh -- internal declarations shared by the translation units of libimager.so (sm_100a only).
// Nothing here is part of the C-ABI (include/imager.h is).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>
#include "../../include/imager.h"

namespace imager {

constexpr int kBucketTile = 32;          // bucketing tile (cells); DESIGN.md "Bucketing key"
constexpr uint32_t kKeyDrop = 0xFFFFFFFFu;   // exported key of a dropped visibility (the oracle's KEY_DROP)
constexpr int kSortChunk = 4096;         // items per CTA tile in the radix sort

int num_sms();                           // SMs of the current device (cudaDevAttrMultiProcessorCount, cached per device): launch sizes
void set_error(const char* fmt, ...);
int cuda_fail(cudaError_t e, const char* what);

#define IMAGER_CUDA(call)                                              \
    do {                                                               \
        cudaError_t e__ = (call);                                      \
        if (e__ != cudaSuccess) return ::imager::cuda_fail(e__, #call); \
    } while (0)

// R24: a sample (visibility k, correlation c) with zero weight, or with a weight or value that is not finite, is
// FLAGGED: it contributes (0, 0) to the grid and nothing to the sum of weights -- flagged data often carry NaN, and
// 0 * NaN would otherwise poison every cell of the footprint (and, in the tiled kernel, the padding around it).
__device__ __forceinline__ bool sample_flagged(float w, float2 v) {
    return w == 0.f || !isfinite(w) || !isfinite(v.x) || !isfinite(v.y);
}
__device__ __forceinline__ float2 weighted_sample(float w, float2 v) {
    return sample_flagged(w, v) ? make_float2(0.f, 0.f) : make_float2(w * v.x, w * v.y);
}

}  // namespace imager

struct imager_plan {
    imager_params p;                     // copy of the caller's params (host pointers cleared)
    int n_sets = 0, nt = 0, n_buckets = 0, key_bits = 0, sort_passes = 0;
    uint32_t key_drop = 0;               // internal sort key of a dropped visibility: n_buckets * O * O
    double uv_scale = 0, w_scale = 0;
    std::vector<int> plane_support;      // S_p, p = 0..P-1
    std::vector<int64_t> set_offset;     // per kernel set, in complex elements (n_sets + 1)
    std::vector<int> set_support;        // per kernel set

    float2* d_tab_grid = nullptr;        // canonical layout, sets back to back
    float2* d_tab_degrid = nullptr;      // == d_tab_grid unless the mode has separate degridding tables
    int64_t* d_set_offset = nullptr;     // [n_sets + 1]
    int32_t* d_set_support = nullptr;    // [n_sets]
    int32_t* d_plane_support = nullptr;  // [P]

    // index / bucketing state (valid for `indexed_nvis` visibilities once index_valid)
    imager_record* d_rec = nullptr;      // [max_nvis] input order
    uint32_t* d_key[2] = {nullptr, nullptr};
    int32_t* d_perm[2] = {nullptr, nullptr};
    int sorted_buf = 0;                  // which of d_key/d_perm holds the sorted result
    int32_t* d_bucket_offset = nullptr;  // [n_buckets + 1]
    int32_t* d_hist = nullptr;           // radix histograms [256 * n_tiles]
    int32_t* d_scan_tmp = nullptr;       // block sums of the scan, all levels
    int64_t scan_tmp_len = 0;
    int32_t* d_counters = nullptr;       // [0] n_kept, [1] n_dropped, [2..] work-queue heads
    int64_t indexed_nvis = -1;
    bool index_valid = false;
    int64_t index_epoch = 0;             // bumped by every re-indexing
    void* tiled = nullptr;               // gridder_tiled.cu state (TiledState*)

    // tiled path work list
    int32_t* d_items = nullptr;          // [max_items][4]
    int64_t max_items = 0;

    double* d_taper = nullptr;           // [N] psi(2(x-N/2)/N) for imager_grid_image_transform
    std::vector<double> pointing_lm;     // [n_aplanes][2] copy of the caller's pointing offsets (MOSAIC_PB)
    float* d_gamma = nullptr;            // [N][N] Eq. 1 weighting correction, built by the first imager_mosaic_correct
    void* fft_plan = nullptr;            // cufftHandle stored as intptr
    bool fft_ready = false;

    cudaEvent_t index_done = nullptr;    // recorded behind every (re)indexing, on the stream it ran on: imager_plan_info waits for it

    int last_launches = 0;
};

namespace imager {

// index_sort.cu
int run_index_and_sort(imager_plan* pl, int64_t nvis, const float* uvw, const int32_t* a_index, cudaStream_t st);
// in-place exclusive scan of n int32; tmp needs sum over levels of (ceil(n/1024)+1) ints
int exclusive_scan_i32(imager_plan* pl, int32_t* data, int64_t n, int32_t* tmp, cudaStream_t st);

// gridder_ref.cu
// set_mask (device, per kernel set, may be NULL): only visibilities of sets with a non-zero entry are processed
int launch_grid_reference(imager_plan* pl, int64_t nvis, const float2* vis, const float* weights, float2* grid,
                          const int32_t* set_mask, cudaStream_t st);
int launch_degrid_reference(imager_plan* pl, int64_t nvis, const float2* grid, float2* vis_out, const int32_t* set_mask,
                            int residual, cudaStream_t st);
int launch_sum_weights(imager_plan* pl, int64_t nvis, const float2* vis, const float* weights, double* sum_weights, cudaStream_t st);

// gridder_tiled.cu
bool tiled_supported(const imager_plan* pl);
const char* tiled_unsupported_reason(const imager_plan* pl);   // NULL = supported
int launch_grid_tiled(imager_plan* pl, int64_t nvis, const float2* vis, const float* weights, float2* grid,
                      cudaStream_t st);
int launch_degrid_tiled(imager_plan* pl, int64_t nvis, const float2* grid, float2* vis_out, int residual, cudaStream_t st);
void tiled_release(imager_plan* pl);
int tiled_prepare(imager_plan* pl, int64_t nvis, cudaStream_t st);
int tiled_index_stats(imager_plan* pl, int64_t out[8], cudaStream_t st);

// tables.cu
int build_tables(imager_plan* pl, const imager_params* user, cudaStream_t st);

// transform.cu
int grid_image_transform(imager_plan* pl, float2* data, int direction, double norm, cudaStream_t st);
int grid_image_transform_dev(imager_plan* pl, float2* data, int direction, const double* norm_dev, cudaStream_t st);
void destroy_transform(imager_plan* pl);
int mosaic_correct(imager_plan* pl, float2* image, cudaStream_t st);

}  // namespace imager
