// gridder_tiled.cu -- the output-stationary ("tiled") gridding / degridding kernels (hot-path steps A3, A6).
//
// Why this shape: every complex MAC needs one 8-byte tap that no other MAC can share
// (the tap index depends on visibility AND cell), so the shared-memory pipe (128 B/clk/SM, measured: 4.59e12
// LDS.64 lanes/s = 49 % of the FP32-FMA peak) is the binding unit, not HBM and not the FMA pipe.  The kernel
// therefore (1) keeps the grid cells in REGISTERS (a warp owns an 8 x 32 strip, 8 cells per lane, packed
// FFMA2 accumulators), (2) keeps one kernel set's oversampled table resident in SHARED memory, zero-padded and
// pitched so that LDS.64 is conflict-free, (3) streams bucket-sorted visibilities through warp ballots so
// that a warp only spends issue slots on visibilities whose footprint meets its strip, and (4) flushes a strip
// once per (kernel set, strip) with red.global.add.v2.f32.
//
//   work item  = (kernel set, slice group, strip row); CTAs pull items from a global queue (kset-major so the
//                resident table is reused); the 16 warps of a CTA pull 8x32 strips of that row from a shared counter
//   table unit = "slice group": all O*O sub-cell slices of the set if they fit in shared memory, else one oy row
//                (O slices), else one slice; sets that do not fit at all take the reference kernels
#include "common.cuh"

namespace imager {

constexpr int kStripW = 8, kStripH = 32, kSlots = 8, kPad = 3;
constexpr int kTiledThreads = 512;
constexpr int kMaxSmem = 227 * 1024;

struct SetPlan {           // per kernel set, host-built at first use
    int32_t pitch;         // taps per padded row, = 8 mod 16 (conflict-free LDS.64 for an 8x4 lane block)
    int32_t group_slices;  // sub-cell slices resident at once (O*O, O or 1); 0 = not tiled (reference path)
    int32_t n_groups;
    int32_t item_base;     // first work item of this set
};

__device__ __forceinline__ void ffma2(float2& d, const float2 a, const float2 b) {
    unsigned long long dd = *reinterpret_cast<unsigned long long*>(&d);
    asm("fma.rn.f32x2 %0, %1, %2, %0;"
        : "+l"(dd)
        : "l"(*reinterpret_cast<const unsigned long long*>(&a)), "l"(*reinterpret_cast<const unsigned long long*>(&b)));
    d = *reinterpret_cast<float2*>(&dd);
}

// sorted-order geometry: word0 = gx | gy << 16, word1 = oy_idx * O + ox_idx  (kept visibilities only)
__global__ void sorted_geo_kernel(const int32_t* __restrict__ counters, const int32_t* __restrict__ perm,
                                  const imager_record* __restrict__ rec, int O, uint2* __restrict__ sgeo) {
    const int n_kept = counters[0];
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_kept; i += gridDim.x * blockDim.x) {
        const imager_record r = rec[perm[i]];
        sgeo[i] = make_uint2((uint32_t)r.gx | ((uint32_t)r.gy << 16), ((r.sub >> 8) & 255u) * O + (r.sub & 255u));
    }
}

// sorted-order weighted visibilities  w_kc * V_kc
template <int NC>
__global__ void gather_values_kernel(const int32_t* __restrict__ counters, const int32_t* __restrict__ perm,
                                     const float2* __restrict__ vis, const float* __restrict__ weights,
                                     float2* __restrict__ sval) {
    const int n_kept = counters[0];
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_kept; i += gridDim.x * blockDim.x) {
        const int64_t k = perm[i];
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const float2 v = vis[k * NC + c];
            const float w = weights[k * NC + c];
            sval[(int64_t)i * NC + c] = make_float2(w * v.x, w * v.y);
        }
    }
}

struct TiledArgs {
    const int32_t* bucket_offset;
    const uint2* sgeo;
    const float2* sval;
    const float2* tab;
    const int64_t* set_offset;
    const int32_t* set_support;
    const SetPlan* set_plan;
    int32_t* queue;          // global work-item counter
    int n_sets, n_items, N, O, nt, strip_rows, strips_per_row;
};

// copy one slice group of kernel set `kset` into shared memory: [slice][row -3 .. S+2][pitch], zero padded
__device__ void load_table_group(const TiledArgs& a, int kset, int group, const SetPlan sp, int S, float2* smem) {
    const float2* T = a.tab + a.set_offset[kset];
    const int rows = S + 2 * kPad;
    const int per_slice = rows * sp.pitch;
    const int total = sp.group_slices * per_slice;
    for (int i = threadIdx.x; i < total; i += blockDim.x) {
        const int sl = i / per_slice, rem = i - sl * per_slice;
        const int row = rem / sp.pitch - kPad, col = rem - (rem / sp.pitch) * sp.pitch;
        float2 v = make_float2(0.f, 0.f);
        if (row >= 0 && row < S && col < S) v = __ldg(&T[((int64_t)(group * sp.group_slices + sl) * S + row) * S + col]);
        smem[i] = v;
    }
}

__global__ void __launch_bounds__(kTiledThreads, 1) grid_tiled_kernel(const TiledArgs a, float2* __restrict__ grid) {
    extern __shared__ float2 smem[];
    __shared__ int s_item, s_strip;
    const int lane = threadIdx.x & 31, lx = lane & 7, ly = lane >> 3;
    int cur_kset = -1, cur_group = -1;
    for (;;) {
        __syncthreads();                                   // everyone is done with the previous item (and s_item)
        if (threadIdx.x == 0) {
            s_item = atomicAdd(a.queue, 1);
            s_strip = 0;
        }
        __syncthreads();
        const int item = s_item;
        if (item >= a.n_items) break;
        // decode: items are laid out set-major: item_base[kset] + group * strip_rows + sy
        int kset = 0;
        {   // n_sets is small (<= a few hundred): linear search from the current set
            kset = cur_kset < 0 ? 0 : cur_kset;
            while (kset + 1 < a.n_sets && item >= a.set_plan[kset + 1].item_base) ++kset;
        }
        const SetPlan sp = a.set_plan[kset];
        if (sp.group_slices == 0) continue;                // set handled by the reference kernel (has no items anyway)
        const int local = item - sp.item_base;
        const int group = local / a.strip_rows, sy = local - group * a.strip_rows;
        const int S = a.set_support[kset], h_lo = S / 2, h_hi = S - 1 - h_lo;
        const int Yw = sy * kStripH;
        // bucket rows whose visibilities can reach this strip row
        const int by_lo = max(0, Yw - h_hi) / kBucketTile;
        const int by_hi = min(a.nt - 1, (Yw + kStripH - 1 + h_lo) / kBucketTile);
        const int row_count = a.bucket_offset[(kset * a.nt + by_hi + 1) * a.nt] - a.bucket_offset[(kset * a.nt + by_lo) * a.nt];
        if (row_count == 0) continue;                      // uniform across the CTA
        if (kset != cur_kset || group != cur_group) {
            load_table_group(a, kset, group, sp, S, smem);
            cur_kset = kset;
            cur_group = group;
            __syncthreads();
        }
        const int slice_stride = (S + 2 * kPad) * sp.pitch;       // in float2
        const int slot_step = 4 * sp.pitch;                       // rows advance by 4 per slot
        const int sub_lo = group * sp.group_slices;
        for (;;) {
            int sx = 0;
            if (lane == 0) sx = atomicAdd(&s_strip, 1);
            sx = __shfl_sync(0xffffffffu, sx, 0);
            if (sx >= a.strips_per_row) break;
            const int Xw = sx * kStripW;
            const int bx_lo = max(0, Xw - h_hi) / kBucketTile;
            const int bx_hi = min(a.nt - 1, (Xw + kStripW - 1 + h_lo) / kBucketTile);
            float2 A[kSlots], B[kSlots];
#pragma unroll
            for (int j = 0; j < kSlots; ++j) A[j] = B[j] = make_float2(0.f, 0.f);
            bool any = false;
            for (int by = by_lo; by <= by_hi; ++by) {
                const int b0 = (kset * a.nt + by) * a.nt;
                const int beg = a.bucket_offset[b0 + bx_lo], end = a.bucket_offset[b0 + bx_hi + 1];   // contiguous in bx
                for (int i0 = beg; i0 < end; i0 += 32) {
                    const int idx = i0 + lane;
                    uint2 g = make_uint2(0u, 0u);
                    float2 v = make_float2(0.f, 0.f);
                    bool hit = false;
                    if (idx < end) {
                        g = a.sgeo[idx];
                        const int gx = (int)(g.x & 0xffffu), gy = (int)(g.x >> 16);
                        const int dx0 = Xw - (gx - h_lo), dy0 = Yw - (gy - h_lo);
                        const int sub = (int)g.y - sub_lo;
                        hit = (dx0 + kStripW > 0) && (dx0 < S) && (dy0 + kStripH > 0) && (dy0 < S) &&
                              ((unsigned)sub < (unsigned)sp.group_slices);
                        if (hit) v = a.sval[idx];
                    }
                    unsigned m = __ballot_sync(0xffffffffu, hit);
                    any |= (m != 0u);
                    while (m) {
                        const int src = __ffs(m) - 1;
                        m &= m - 1;
                        const uint32_t gxy = __shfl_sync(0xffffffffu, g.x, src);
                        const int sub = (int)__shfl_sync(0xffffffffu, g.y, src) - sub_lo;
                        const float vr = __shfl_sync(0xffffffffu, v.x, src), vi = __shfl_sync(0xffffffffu, v.y, src);
                        const int gx = (int)(gxy & 0xffffu), gy = (int)(gxy >> 16);
                        const int dy0 = Yw - (gy - h_lo);                 // tap row of the strip's first row
                        const int col = Xw + lx - (gx - h_lo);
                        // slots whose 4-row group meets the footprint rows [0, S)
                        const int jl = (dy0 + 3 < 0) ? (-dy0) / 4 : 0;      // first j with dy0 + 4j + 3 >= 0
                        const int jh = min(kSlots, (S - 1 - dy0) / 4 + 1);  // one past the last j with dy0 + 4j <= S-1
                        if ((unsigned)col < (unsigned)S) {
                            const float2* tp = smem + sub * slice_stride + (dy0 + ly + kPad) * sp.pitch + col;
                            const float2 vrr = make_float2(vr, vr), vii = make_float2(vi, vi);
#pragma unroll
                            for (int j = 0; j < kSlots; ++j) {
                                if (j >= jl && j < jh) {
                                    const float2 t = tp[j * slot_step];
                                    ffma2(A[j], t, vrr);
                                    ffma2(B[j], t, vii);
                                }
                            }
                        }
                    }
                }
            }
            if (any) {
#pragma unroll
                for (int j = 0; j < kSlots; ++j) {
                    const float re = A[j].x - B[j].y, im = A[j].y + B[j].x;
                    if (re != 0.f || im != 0.f)
                        atomicAdd(&grid[(int64_t)(Yw + ly + 4 * j) * a.N + Xw + lx], make_float2(re, im));
                }
            }
        }
    }
}

// ---- host side -------------------------------------------------------------------------------------------

struct TiledState {
    std::vector<SetPlan> plan;
    SetPlan* d_plan = nullptr;
    int32_t* d_ref_mask = nullptr;        // per set: 1 = no tiled plan (reference kernels handle it)
    int64_t geo_epoch = -1;
    uint2* d_sgeo = nullptr;
    float2* d_sval = nullptr;
    int n_items = 0, smem_bytes = 0;
    bool any_tiled = false, any_ref = false;
};

bool tiled_supported(const imager_plan* pl) {
    const imager_params& p = pl->p;
    return p.n_corr == 1 && p.n_pol == 1 && p.grid_size % kStripH == 0 && p.grid_size <= 32768 &&
           pl->p.kernel_mode != IMAGER_MODE_DELTA;
}

static TiledState* state_of(imager_plan* pl) {
    if (pl->tiled) return static_cast<TiledState*>(pl->tiled);
    TiledState* st = new TiledState();
    const imager_params& p = pl->p;
    const int O = p.oversample, strip_rows = p.grid_size / kStripH;
    st->plan.resize(pl->n_sets);
    int items = 0;
    for (int k = 0; k < pl->n_sets; ++k) {
        const int S = pl->set_support[k];
        SetPlan sp;
        sp.pitch = ((S + 7) / 16) * 16 + 8;                 // smallest value >= S that is 8 mod 16
        if (sp.pitch < S) sp.pitch += 16;
        const int64_t slice_bytes = (int64_t)(S + 2 * kPad) * sp.pitch * 8;
        sp.group_slices = 0;
        for (int gsl : {O * O, O, 1})
            if (gsl * slice_bytes <= kMaxSmem - 1024) { sp.group_slices = gsl; break; }
        sp.n_groups = sp.group_slices ? (O * O) / sp.group_slices : 0;
        sp.item_base = items;
        items += sp.n_groups * strip_rows;
        if (sp.group_slices) {
            st->any_tiled = true;
            st->smem_bytes = std::max<int>(st->smem_bytes, (int)(sp.group_slices * slice_bytes));
        } else {
            st->any_ref = true;
        }
        st->plan[k] = sp;
    }
    st->n_items = items;
    pl->tiled = st;
    return st;
}

void tiled_release(imager_plan* pl) {
    if (!pl->tiled) return;
    TiledState* st = static_cast<TiledState*>(pl->tiled);
    cudaFree(st->d_plan);
    cudaFree(st->d_ref_mask);
    cudaFree(st->d_sgeo);
    cudaFree(st->d_sval);
    delete st;
    pl->tiled = nullptr;
}

static int prepare(imager_plan* pl, TiledState* st, int64_t nvis, cudaStream_t stream) {
    const int64_t mv = std::max<int64_t>(pl->p.max_nvis, 1);
    if (!st->d_plan) {
        IMAGER_CUDA(cudaMalloc(&st->d_plan, pl->n_sets * sizeof(SetPlan)));
        IMAGER_CUDA(cudaMemcpyAsync(st->d_plan, st->plan.data(), pl->n_sets * sizeof(SetPlan), cudaMemcpyHostToDevice, stream));
        std::vector<int32_t> mask(pl->n_sets);
        for (int k = 0; k < pl->n_sets; ++k) mask[k] = st->plan[k].group_slices == 0;
        IMAGER_CUDA(cudaMalloc(&st->d_ref_mask, pl->n_sets * sizeof(int32_t)));
        IMAGER_CUDA(cudaMemcpyAsync(st->d_ref_mask, mask.data(), pl->n_sets * sizeof(int32_t), cudaMemcpyHostToDevice, stream));
        IMAGER_CUDA(cudaStreamSynchronize(stream));     // one-off: the host vectors above go out of scope
        IMAGER_CUDA(cudaMalloc(&st->d_sgeo, mv * sizeof(uint2)));
        IMAGER_CUDA(cudaMalloc(&st->d_sval, mv * pl->p.n_corr * sizeof(float2)));
        IMAGER_CUDA(cudaFuncSetAttribute(grid_tiled_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem - 1024));
    }
    if (st->geo_epoch != pl->index_epoch) {
        sorted_geo_kernel<<<4 * kNumSMs, 256, 0, stream>>>(pl->d_counters, pl->d_perm[pl->sorted_buf], pl->d_rec,
                                                           pl->p.oversample, st->d_sgeo);
        pl->last_launches++;
        st->geo_epoch = pl->index_epoch;
    }
    return 0;
}

int launch_grid_tiled(imager_plan* pl, int64_t nvis, const float2* vis, const float* weights, float2* grid,
                      cudaStream_t stream) {
    if (nvis == 0) return 0;
    TiledState* st = state_of(pl);
    int rc = prepare(pl, st, nvis, stream);
    if (rc) return rc;
    if (st->any_ref) {
        rc = launch_grid_reference(pl, nvis, vis, weights, grid, st->d_ref_mask, stream);   // sets without a tiled plan
        if (rc) return rc;
    }
    if (!st->any_tiled) return 0;
    gather_values_kernel<1><<<4 * kNumSMs, 256, 0, stream>>>(pl->d_counters, pl->d_perm[pl->sorted_buf], vis, weights, st->d_sval);
    IMAGER_CUDA(cudaMemsetAsync(pl->d_counters + 8, 0, sizeof(int32_t), stream));
    TiledArgs a;
    a.bucket_offset = pl->d_bucket_offset;
    a.sgeo = st->d_sgeo;
    a.sval = st->d_sval;
    a.tab = pl->d_tab_grid;
    a.set_offset = pl->d_set_offset;
    a.set_support = pl->d_set_support;
    a.set_plan = st->d_plan;
    a.queue = pl->d_counters + 8;
    a.n_sets = pl->n_sets;
    a.n_items = st->n_items;
    a.N = pl->p.grid_size;
    a.O = pl->p.oversample;
    a.nt = pl->nt;
    a.strip_rows = pl->p.grid_size / kStripH;
    a.strips_per_row = pl->p.grid_size / kStripW;
    grid_tiled_kernel<<<kNumSMs, kTiledThreads, st->smem_bytes, stream>>>(a, grid);
    pl->last_launches += 2;
    IMAGER_CUDA(cudaGetLastError());
    return 0;
}

int launch_degrid_tiled(imager_plan* pl, int64_t nvis, const float2* grid, float2* vis_out, cudaStream_t stream) {
    return launch_degrid_reference(pl, nvis, grid, vis_out, nullptr, stream);
}

}  // namespace imager
