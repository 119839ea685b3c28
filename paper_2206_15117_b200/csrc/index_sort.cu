// index_sort.cu -- hot-path steps A1 (index) and A2 (bucketing) of DESIGN.md.
//
// A1: one thread per visibility: uvw (float32, wavelengths) -> imager_record + 32-bit bucket key.
//     Integer results are defined by DESIGN.md R2-R5/R8 and must equal the oracle bit for bit:
//       q = rint(double(u) * uv_scale)            one IEEE multiply + round-half-even (cvt.rni.s64.f64)
//       i = floor((q + O/2)/O), o = q - i*O, g = i + N/2;  p = min(P-1, rint(|w| * w_scale)), sp = sign(w) p
//       kset = a*(2P-1) + sp + P-1;  drop if the S_p footprint leaves the grid
//       key  = ((kset*nt + gy/32)*nt + gx/32)*O*O + (oy+O/2)*O + (ox+O/2), dropped -> 0xFFFFFFFF
//       R17: non-finite u, v, w, |q| >= 2^30 or a_index outside [0, n_aplanes) -> dropped, record (0, 0, drop, 0)
//     Internally the drop key is n_buckets * O * O (one more than the largest valid key), so that the radix sort needs
//     only ceil(bits(n_buckets * O * O) / 8) passes; imager_debug_index exports it as 0xFFFFFFFF (the oracle's KEY_DROP).
// A2: stable LSD radix sort (8-bit digits) of (key, input index), then dense bucket offsets by binary search.
//     The sort is hand-written: per-tile (4096 items, one CTA) histograms -> exclusive scan -> stable scatter: ranks from
//     __match_any_sync within rows of 32 items, the tile sorted by digit in shared memory and written out in runs
//     (coalesced).  Stability makes the permutation unique, hence comparable bit-exactly.
#include "common.cuh"

namespace imager {

__device__ __forceinline__ int floor_div32(int a, int b) {      // b > 0
    const int q = a / b;
    return (a - q * b < 0) ? q - 1 : q;
}

// record and sort key of visibility k (the permutation starts as the identity: the first sort pass assumes it)
__device__ __forceinline__ uint32_t index_one(int64_t k, const float* __restrict__ uvw, const int32_t* __restrict__ a_index,
                                              double uv_scale, double w_scale, int N, int O, int P, int nt, int n_aplanes,
                                              uint32_t key_drop, const int32_t* __restrict__ plane_support,
                                              imager_record* __restrict__ rec, int32_t* __restrict__ counters) {
    float u = uvw[3 * k], v = uvw[3 * k + 1], w = uvw[3 * k + 2];
    int a = a_index ? a_index[k] : 0;
    const double su = __dmul_rn((double)u, uv_scale), sv = __dmul_rn((double)v, uv_scale);
    // R17: values that cannot be indexed are dropped before any cell or kernel-set index is formed from them
    const bool invalid = !(isfinite(u) && isfinite(v) && isfinite(w)) || !(fabs(su) < 1073741824.0) ||
                         !(fabs(sv) < 1073741824.0) || a < 0 || a >= n_aplanes;
    if (invalid) {
        imager_record r;
        r.gx = r.gy = 0;
        r.sub = 1u << 16;
        r.kset = 0;
        rec[k] = r;
        atomicAdd(&counters[1], 1);
        return key_drop;
    }
    // |su|, |sv| < 2^30 from here on: 32-bit integer arithmetic gives the same values as the 64-bit definition
    const int qx = __double2int_rn(su), qy = __double2int_rn(sv);
    const int half_o = O / 2;
    const int ix = floor_div32(qx + half_o, O), iy = floor_div32(qy + half_o, O);
    const int ox = qx - ix * O, oy = qy - iy * O;
    const int gx = ix + N / 2, gy = iy + N / 2;
    // p = min(P - 1, rint(|w| w_scale)): the comparison is made in double so that huge |w| clamps instead of wrapping
    const double sw = __dmul_rn(fabs((double)w), w_scale);
    const int p = sw >= (double)(P - 1) ? P - 1 : __double2int_rn(sw);
    const int sp = (w < 0.f) ? -p : p;
    const int kset = a * (2 * P - 1) + sp + P - 1;
    const int S = plane_support[p], h_lo = S / 2, h_hi = S - 1 - h_lo;
    const bool drop = (gx - h_lo < 0) || (gx + h_hi >= N) || (gy - h_lo < 0) || (gy + h_hi >= N);
    imager_record r;
    r.gx = gx;
    r.gy = gy;
    r.sub = (uint32_t)(ox + half_o) | ((uint32_t)(oy + half_o) << 8) | ((uint32_t)drop << 16);
    r.kset = kset;
    rec[k] = r;
    uint32_t kk = key_drop;
    if (!drop)                       // < 2^32 (checked at plan creation); gx, gy >= 0 here
        kk = (((uint32_t)kset * (uint32_t)nt + (uint32_t)gy / kBucketTile) * (uint32_t)nt + (uint32_t)gx / kBucketTile) * (uint32_t)(O * O) +
             (uint32_t)((oy + half_o) * O + (ox + half_o));
    else
        atomicAdd(&counters[1], 1);
    return kk;
}

// One CTA indexes one sort tile (kSortChunk visibilities) and leaves the tile's histogram of the first radix digit, so
// that the first sort pass needs no histogram pass of its own.  hist[d * n_tiles + tile], as radix_hist_kernel writes it.
__global__ void __launch_bounds__(256) index_kernel(int64_t nvis, const float* __restrict__ uvw, const int32_t* __restrict__ a_index,
                                                    double uv_scale, double w_scale, int N, int O, int P, int nt, int n_aplanes,
                                                    uint32_t key_drop, const int32_t* __restrict__ plane_support,
                                                    imager_record* __restrict__ rec, uint32_t* __restrict__ key,
                                                    int32_t* __restrict__ counters, int32_t* __restrict__ hist, int n_tiles) {
    __shared__ int32_t cnt[8][256];
    const int warp = threadIdx.x >> 5;
    for (int i = threadIdx.x & 31; i < 256; i += 32) cnt[warp][i] = 0;
    __syncwarp();
    const int64_t base = (int64_t)blockIdx.x * kSortChunk;
#pragma unroll 2
    for (int r = 0; r < kSortChunk / 256; ++r) {
        const int64_t k = base + r * 256 + threadIdx.x;
        if (k < nvis) {
            const uint32_t kk = index_one(k, uvw, a_index, uv_scale, w_scale, N, O, P, nt, n_aplanes, key_drop, plane_support, rec, counters);
            key[k] = kk;
            atomicAdd(&cnt[warp][kk & 255u], 1);
        }
    }
    __syncthreads();
    int t = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) t += cnt[w][threadIdx.x];
    hist[(int64_t)threadIdx.x * n_tiles + blockIdx.x] = t;
}


// ---- radix sort: one CTA owns a tile of kSortChunk consecutive items (8 warps x kSortRows rows of 32) ----
constexpr int kSortThreads = 256, kSortWarps = kSortThreads / 32, kSortRows = kSortChunk / kSortThreads;

__global__ void __launch_bounds__(kSortThreads) radix_hist_kernel(int64_t n, const uint32_t* __restrict__ key, int shift,
                                                                  int32_t* __restrict__ hist, int n_tiles) {
    __shared__ int32_t cnt[kSortWarps][256];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tile = blockIdx.x;
    for (int i = lane; i < 256; i += 32) cnt[warp][i] = 0;
    __syncwarp();
    const int64_t base = (int64_t)tile * kSortChunk + warp * (kSortRows * 32);
#pragma unroll 4
    for (int r = 0; r < kSortRows; ++r) {
        const int64_t idx = base + r * 32 + lane;
        if (idx < n) atomicAdd(&cnt[warp][(key[idx] >> shift) & 255u], 1);
    }
    __syncthreads();
    int t = 0;
#pragma unroll
    for (int w = 0; w < kSortWarps; ++w) t += cnt[w][threadIdx.x];
    hist[(int64_t)threadIdx.x * n_tiles + tile] = t;
}

// Stable scatter of one tile.  Ranks: per row of 32 consecutive items the lanes with the same digit find each other with
// __match_any_sync (rank = lower peers), per-warp digit counters order the rows, a prefix over the warps orders the
// warps: the tile is first sorted by digit in shared memory, then written out in runs of equal digit (coalesced), each
// run to the place the scanned histograms give it.  val_in == nullptr: the values are the input indices (first pass).
__global__ void __launch_bounds__(kSortThreads, 3) radix_scatter_kernel(int64_t n, const uint32_t* __restrict__ key_in,
                                                                     const int32_t* __restrict__ val_in,
                                                                     uint32_t* __restrict__ key_out, int32_t* __restrict__ val_out,
                                                                     int shift, const int32_t* __restrict__ hist_scanned, int n_tiles) {
    __shared__ int32_t wcount[kSortWarps][256];
    __shared__ int32_t dstart[256], gdelta[256], wsum[kSortWarps];
    __shared__ uint32_t s_key[kSortChunk];
    __shared__ int32_t s_val[kSortChunk];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tile = blockIdx.x;
    const unsigned lt_mask = (1u << lane) - 1u;
    for (int i = lane; i < 256; i += 32) wcount[warp][i] = 0;
    __syncwarp();
    const int64_t base = (int64_t)tile * kSortChunk + warp * (kSortRows * 32);
    uint32_t k[kSortRows];
    int32_t v[kSortRows];
    int32_t lrank[kSortRows];                   // rank of the item among those of its warp with the same digit
#pragma unroll
    for (int r = 0; r < kSortRows; ++r) {
        const int64_t idx = base + r * 32 + lane;
        k[r] = 0u;
        v[r] = 0;
        if (idx < n) {
            k[r] = key_in[idx];
            v[r] = val_in ? val_in[idx] : (int32_t)idx;
        }
    }
#pragma unroll
    for (int r = 0; r < kSortRows; ++r) {
        const int64_t idx = base + r * 32 + lane;
        const bool live = idx < n;
        const unsigned active = __ballot_sync(0xffffffffu, live);
        lrank[r] = 0;
        if (live) {
            const unsigned d = (k[r] >> shift) & 255u;
            const unsigned peers = __match_any_sync(active, d);
            const int rank = __popc(peers & lt_mask);
            lrank[r] = wcount[warp][d] + rank;
            __syncwarp(active);
            if (rank == 0) wcount[warp][d] += __popc(peers);
        }
        __syncwarp();
    }
    __syncthreads();
    {   // thread d: exclusive prefix of digit d over the warps, then of the digit totals over the digits
        const int d = threadIdx.x;
        int t = 0;
#pragma unroll
        for (int w = 0; w < kSortWarps; ++w) {
            const int c = wcount[w][d];
            wcount[w][d] = t;
            t += c;
        }
        int inc = t;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += y;
        }
        if (lane == 31) wsum[warp] = inc;
        __syncthreads();
        int woff = 0;
#pragma unroll
        for (int w = 0; w < kSortWarps; ++w)
            if (w < warp) woff += wsum[w];
        const int start = woff + inc - t;
        dstart[d] = start;
        gdelta[d] = hist_scanned[(int64_t)d * n_tiles + tile] - start;
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < kSortRows; ++r) {
        const int64_t idx = base + r * 32 + lane;
        if (idx < n) {
            const unsigned d = (k[r] >> shift) & 255u;
            const int pos = dstart[d] + wcount[warp][d] + lrank[r];
            s_key[pos] = k[r];
            s_val[pos] = v[r];
        }
    }
    __syncthreads();
    const int64_t left = n - (int64_t)tile * kSortChunk;
    const int count = left < kSortChunk ? (int)left : kSortChunk;
    for (int i = threadIdx.x; i < count; i += kSortThreads) {
        const uint32_t kk = s_key[i];
        const int dst = gdelta[(kk >> shift) & 255u] + i;
        key_out[dst] = kk;
        val_out[dst] = s_val[i];
    }
}

// ---- exclusive scan of int32 (1024 items per block), hierarchical ----
__global__ void scan_block_kernel(const int32_t* in, int32_t* out, int32_t* __restrict__ sums,   // in may alias out
                                  int64_t n) {
    __shared__ int32_t warp_tot[8];
    const int64_t base = (int64_t)blockIdx.x * 1024 + threadIdx.x * 4;
    int32_t v[4], t = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        v[j] = (base + j < n) ? in[base + j] : 0;
        t += v[j];
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int32_t inc = t;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        int32_t y = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += y;
    }
    if (lane == 31) warp_tot[warp] = inc;
    __syncthreads();
    int32_t woff = 0, total = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) {
        if (w < warp) woff += warp_tot[w];
        total += warp_tot[w];
    }
    int32_t run = woff + inc - t;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        if (base + j < n) out[base + j] = run;
        run += v[j];
    }
    if (threadIdx.x == 0 && sums) sums[blockIdx.x] = total;
}

__global__ void scan_add_kernel(int32_t* __restrict__ data, const int32_t* __restrict__ block_off, int64_t n) {
    const int64_t i = (int64_t)blockIdx.x * 1024 + threadIdx.x;
    const int32_t off = block_off[blockIdx.x];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int64_t idx = i + j * 256;
        if (idx < n) data[idx] += off;
    }
}

// data[i] += sum of the block totals before block i / 1024: every block sums its predecessors' totals itself (at most
// kDirectBlocks of them), which saves the scan of the totals and one launch per level
constexpr int kDirectBlocks = 4096;
__global__ void scan_add_direct_kernel(int32_t* __restrict__ data, const int32_t* __restrict__ block_sums, int64_t n) {
    __shared__ int32_t warp_tot[8];
    __shared__ int32_t s_off;
    int32_t t = 0;
    for (int j = threadIdx.x; j < (int)blockIdx.x; j += 256) t += block_sums[j];
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) t += __shfl_xor_sync(0xffffffffu, t, d);
    if ((threadIdx.x & 31) == 0) warp_tot[threadIdx.x >> 5] = t;
    __syncthreads();
    if (threadIdx.x == 0) {
        int32_t o = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) o += warp_tot[w];
        s_off = o;
    }
    __syncthreads();
    const int32_t off = s_off;
    const int64_t i = (int64_t)blockIdx.x * 1024 + threadIdx.x;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int64_t idx = i + j * 256;
        if (idx < n) data[idx] += off;
    }
}

static int exclusive_scan(imager_plan* pl, int32_t* data, int64_t n, int32_t* tmp, cudaStream_t st) {
    const int64_t nb = (n + 1023) / 1024;
    scan_block_kernel<<<(unsigned)nb, 256, 0, st>>>(data, data, nb > 1 ? tmp : nullptr, n);
    pl->last_launches++;
    if (nb > 1 && nb <= kDirectBlocks) {
        scan_add_direct_kernel<<<(unsigned)nb, 256, 0, st>>>(data, tmp, n);
        pl->last_launches++;
    } else if (nb > 1) {
        int rc = exclusive_scan(pl, tmp, nb, tmp + nb, st);
        if (rc) return rc;
        scan_add_kernel<<<(unsigned)nb, 256, 0, st>>>(data, tmp, n);
        pl->last_launches++;
    }
    return 0;
}

int exclusive_scan_i32(imager_plan* pl, int32_t* data, int64_t n, int32_t* tmp, cudaStream_t st) {
    return exclusive_scan(pl, data, n, tmp, st);
}

__global__ void bucket_offset_kernel(const uint32_t* __restrict__ skey, int64_t n, int n_buckets, int oo,
                                     int32_t* __restrict__ bucket_offset, int32_t* __restrict__ counters) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b > n_buckets) return;
    // lower_bound of b*O*O in the sorted keys (the drop key is larger than every bucket edge)
    const uint64_t edge = (uint64_t)b * (uint64_t)oo;
    int64_t lo = 0, hi = n;
    while (lo < hi) {
        const int64_t mid = (lo + hi) >> 1;
        if ((uint64_t)skey[mid] < edge) lo = mid + 1; else hi = mid;      // the drop key equals the last edge
    }
    bucket_offset[b] = (int32_t)lo;
    if (b == n_buckets) counters[0] = (int32_t)lo;      // n_kept
}

int run_index_and_sort(imager_plan* pl, int64_t nvis, const float* uvw, const int32_t* a_index, cudaStream_t st) {
    const imager_params& p = pl->p;
    IMAGER_CUDA(cudaMemsetAsync(pl->d_counters, 0, 64 * sizeof(int32_t), st));
    if (nvis > 0) {
        index_kernel<<<(unsigned)((nvis + kSortChunk - 1) / kSortChunk), 256, 0, st>>>(
            nvis, uvw, a_index, pl->uv_scale, pl->w_scale, p.grid_size, p.oversample, p.n_wplanes, pl->nt, p.n_aplanes,
            pl->key_drop, pl->d_plane_support, pl->d_rec, pl->d_key[0], pl->d_counters, pl->d_hist,
            (int)((nvis + kSortChunk - 1) / kSortChunk));
        pl->last_launches++;
    }
    int cur = 0;
    const int n_chunks = (int)((nvis + kSortChunk - 1) / kSortChunk);
    for (int pass = 0; pass < pl->sort_passes && nvis > 0; ++pass) {
        const int shift = 8 * pass;
        const unsigned blocks = (unsigned)n_chunks;
        if (pass > 0) {                           // the index kernel has left the histograms of the first digit
            radix_hist_kernel<<<blocks, kSortThreads, 0, st>>>(nvis, pl->d_key[cur], shift, pl->d_hist, n_chunks);
            pl->last_launches++;
        }
        int rc = exclusive_scan(pl, pl->d_hist, (int64_t)256 * n_chunks, pl->d_scan_tmp, st);
        if (rc) return rc;
        radix_scatter_kernel<<<blocks, kSortThreads, 0, st>>>(nvis, pl->d_key[cur], pass == 0 ? nullptr : pl->d_perm[cur],
                                                              pl->d_key[cur ^ 1], pl->d_perm[cur ^ 1], shift, pl->d_hist, n_chunks);
        pl->last_launches++;
        cur ^= 1;
    }
    pl->sorted_buf = cur;
    bucket_offset_kernel<<<(unsigned)((pl->n_buckets + 1 + 255) / 256), 256, 0, st>>>(
        pl->d_key[cur], nvis, pl->n_buckets, p.oversample * p.oversample, pl->d_bucket_offset, pl->d_counters);
    pl->last_launches++;
    IMAGER_CUDA(cudaGetLastError());
    pl->indexed_nvis = nvis;
    pl->index_valid = true;
    pl->index_epoch++;
    return 0;
}

}  // namespace imager
