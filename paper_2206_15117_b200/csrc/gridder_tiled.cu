// gridder_tiled.cu -- the output-stationary ("tiled") gridding kernel (hot-path step A3) and its work planner.
//
// Why this shape: every complex MAC needs one 8-byte tap that no other MAC can share
// (the tap index depends on visibility AND cell), so the shared-memory pipe (128 B/clk/SM; measured 4.59e12
// LDS.64 lanes/s = 49 % of the FP32-FMA peak) is the binding unit, not HBM and not the FMA pipe.  The kernel
//   (1) keeps grid cells in REGISTERS: a warp owns a 16 x 32 strip, its 8 x 4 lane block is replicated 2 x 8
//       times (16 cells per lane, packed FFMA2 accumulators), so idle lanes only occur where a footprint edge
//       cuts an 8 x 4 block;
//   (2) keeps one "unit" (a kernel set, or a group of its sub-cell slices) resident in SHARED memory, rows
//       zero-padded by 3 and pitched to 8 mod 16 taps so that LDS.64 of an 8 x 4 lane block is conflict-free;
//   (3) streams bucket-sorted visibilities: 32 candidates per batch are tested against the strip by one lane
//       each, the hits are compacted into per-warp descriptors in shared memory and replayed; a descriptor
//       carries the precomputed tap address and the first/last active row group, so a hit costs one broadcast
//       LDS.128 plus a Duff-style entry into the unrolled row-group chain (1 LDS.64 + 2 FFMA2 per group);
//   (4) flushes a strip once per work entry with red.global.add.v2.f32.
// Work planning (device side, at index time, cached while uvw is unchanged): entry = (unit, strip, part) with at
// most kChunk candidate visibilities; blocks of kBlockEntries entries of one unit are pulled by persistent CTAs
// from a global queue, the 16 warps of a CTA pull entries of the block from a shared counter.
#include "common.cuh"

namespace imager {

constexpr int kLaneW = 8, kLaneH = 4;                 // lane block
constexpr int kNX = 2, kNY = 8;                       // replications: strip = 16 x 32 cells
constexpr int kStripW = kLaneW * kNX, kStripH = kLaneH * kNY, kPad = kLaneH - 1;
constexpr int kTiledThreads = 512, kWarps = kTiledThreads / 32;
constexpr int kChunk = 512;                           // candidate visibilities per work entry
constexpr int kBlockEntries = 64;                     // entries per CTA-level block
constexpr int kStageBytes = kWarps * 32 * 16;         // per-warp hit descriptors
constexpr int kMaxSmem = 227 * 1024;
constexpr int64_t kMaxPlanCells = 48 << 20;           // (unit, strip) pairs the planner may enumerate

struct SetPlan {           // per kernel set (host-built)
    int32_t pitch;         // taps per padded row, = 8 mod 16
    int32_t group_slices;  // sub-cell slices resident at once (O*O, O or 1); 0 = not tiled (reference path)
    int32_t n_groups;
    int32_t unit_base;     // first unit of this set; unit = unit_base + group
};

struct Entry { int32_t unit, strip, part, pad; };
struct Block { int32_t kset, group, first, count; };

__device__ __forceinline__ void ffma2(float2& d, const float2 a, const float2 b) {
    unsigned long long dd = *reinterpret_cast<unsigned long long*>(&d);
    asm("fma.rn.f32x2 %0, %1, %2, %0;"
        : "+l"(dd)
        : "l"(*reinterpret_cast<const unsigned long long*>(&a)), "l"(*reinterpret_cast<const unsigned long long*>(&b)));
    d = *reinterpret_cast<float2*>(&dd);
}

__device__ __forceinline__ float2 lds64(uint32_t addr) {
    float2 v;
    asm("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
    return v;
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

struct Geometry {
    int N, O, nt, strips_per_row, n_strips, n_sets, n_units;
};

// candidate visibilities of (kset, strip): the bucket rows / columns whose footprints can reach the strip
__device__ __forceinline__ void strip_buckets(const Geometry& g, int strip, int S, int& Xw, int& Yw, int& bx_lo, int& bx_hi,
                                              int& by_lo, int& by_hi) {
    const int sy = strip / g.strips_per_row, sx = strip - sy * g.strips_per_row;
    const int h_lo = S / 2, h_hi = S - 1 - h_lo;
    Xw = sx * kStripW;
    Yw = sy * kStripH;
    bx_lo = max(0, Xw - h_hi) / kBucketTile;
    bx_hi = min(g.nt - 1, (Xw + kStripW - 1 + h_lo) / kBucketTile);
    by_lo = max(0, Yw - h_hi) / kBucketTile;
    by_hi = min(g.nt - 1, (Yw + kStripH - 1 + h_lo) / kBucketTile);
}

// ---- planner ---------------------------------------------------------------------------------------------
// parts[unit * n_strips + strip] = ceil(candidates / kChunk)
__global__ void plan_count_kernel(const Geometry g, const SetPlan* __restrict__ set_plan, const int32_t* __restrict__ unit_set,
                                  const int32_t* __restrict__ set_support, const int32_t* __restrict__ bucket_offset,
                                  int32_t* __restrict__ parts) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i > (int64_t)g.n_units * g.n_strips) return;
    if (i == (int64_t)g.n_units * g.n_strips) { parts[i] = 0; return; }
    const int unit = (int)(i / g.n_strips), strip = (int)(i - (int64_t)unit * g.n_strips);
    const int kset = unit_set[unit];
    int Xw, Yw, bx_lo, bx_hi, by_lo, by_hi;
    strip_buckets(g, strip, set_support[kset], Xw, Yw, bx_lo, bx_hi, by_lo, by_hi);
    int c = 0;
    for (int by = by_lo; by <= by_hi; ++by) {
        const int b0 = (kset * g.nt + by) * g.nt;
        c += bucket_offset[b0 + bx_hi + 1] - bucket_offset[b0 + bx_lo];
    }
    parts[i] = (c + kChunk - 1) / kChunk;
}

__global__ void plan_fill_kernel(const Geometry g, const int32_t* __restrict__ entry_start, Entry* __restrict__ entries) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (int64_t)g.n_units * g.n_strips) return;
    const int unit = (int)(i / g.n_strips), strip = (int)(i - (int64_t)unit * g.n_strips);
    const int e0 = entry_start[i], e1 = entry_start[i + 1];
    for (int e = e0; e < e1; ++e) entries[e] = Entry{unit, strip, e - e0, 0};
}

// one thread block: blocks of at most kBlockEntries entries, never spanning two units
__global__ void plan_blocks_kernel(const Geometry g, const SetPlan* __restrict__ set_plan, const int32_t* __restrict__ unit_set,
                                   const int32_t* __restrict__ entry_start, Block* __restrict__ blocks,
                                   int32_t* __restrict__ n_blocks) {
    __shared__ int s_total;
    if (threadIdx.x == 0) s_total = 0;
    __syncthreads();
    for (int u0 = 0; u0 < g.n_units; u0 += blockDim.x) {
        const int u = u0 + threadIdx.x;
        int first = 0, cnt = 0;
        if (u < g.n_units) {
            first = entry_start[(int64_t)u * g.n_strips];
            cnt = entry_start[(int64_t)(u + 1) * g.n_strips] - first;
        }
        const int nb = (cnt + kBlockEntries - 1) / kBlockEntries;
        const int base = nb ? atomicAdd(&s_total, nb) : 0;            // block order is irrelevant
        if (nb) {
            const int kset = unit_set[u];
            for (int b = 0; b < nb; ++b)
                blocks[base + b] = Block{kset, u - set_plan[kset].unit_base, first + b * kBlockEntries,
                                         min(kBlockEntries, cnt - b * kBlockEntries)};
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) *n_blocks = s_total;
}

// ---- the gridding kernel ---------------------------------------------------------------------------------
struct TiledArgs {
    Geometry g;
    const int32_t* bucket_offset;
    const uint2* sgeo;
    const float2* sval;
    const float2* tab;
    const int64_t* set_offset;
    const int32_t* set_support;
    const SetPlan* set_plan;
    const Entry* entries;
    const Block* blocks;
    const int32_t* n_blocks;
    int32_t* queue;
};

// copy one slice group of kernel set `kset` into shared memory: [slice][row -3 .. S+2][pitch], zero padded
__device__ void load_table_group(const TiledArgs& a, int kset, int group, const SetPlan sp, int S, float2* tab_s) {
    const float2* T = a.tab + a.set_offset[kset];
    const int rows = S + 2 * kPad;
    const int per_slice = rows * sp.pitch;
    const int total = sp.group_slices * per_slice;
    for (int i = threadIdx.x; i < total; i += blockDim.x) {
        const int sl = i / per_slice, rem = i - sl * per_slice;
        const int r = rem / sp.pitch, row = r - kPad, col = rem - r * sp.pitch;
        float2 v = make_float2(0.f, 0.f);
        if (row >= 0 && row < S && col < S) v = __ldg(&T[((int64_t)(group * sp.group_slices + sl) * S + row) * S + col]);
        tab_s[i] = v;
    }
}

// one row group: tap loads for the two 8-column halves of the strip, 2 FFMA2 each (A += t*vr, B += t*vi)
#define IMAGER_SLOT_BOTH(j)                                \
    {                                                      \
        const float2 t0 = lds64(addr0 + (j) * step0);      \
        const float2 t1 = lds64(addr1 + (j) * step1);      \
        ffma2(A0[j], t0, vrr);                             \
        ffma2(B0[j], t0, vii);                             \
        ffma2(A1[j], t1, vrr);                             \
        ffma2(B1[j], t1, vii);                             \
    }
#define IMAGER_SLOT_LEFT(j)                                \
    {                                                      \
        const float2 t0 = lds64(addr0 + (j) * step0);      \
        ffma2(A0[j], t0, vrr);                             \
        ffma2(B0[j], t0, vii);                             \
    }
#define IMAGER_SLOT_RIGHT(j)                               \
    {                                                      \
        const float2 t1 = lds64(addr1 + (j) * step1);      \
        ffma2(A1[j], t1, vrr);                             \
        ffma2(B1[j], t1, vii);                             \
    }
// enter the unrolled row-group chain at jl, leave after jh - 1 (jl, jh are warp-uniform: they come from a REDUX)
#define IMAGER_CHAIN(SLOT)                         \
    switch (jl) {                                  \
        case 0: SLOT(0) if (jh == 1) break;        \
        case 1: SLOT(1) if (jh == 2) break;        \
        case 2: SLOT(2) if (jh == 3) break;        \
        case 3: SLOT(3) if (jh == 4) break;        \
        case 4: SLOT(4) if (jh == 5) break;        \
        case 5: SLOT(5) if (jh == 6) break;        \
        case 6: SLOT(6) if (jh == 7) break;        \
        case 7: SLOT(7)                            \
    }

__global__ void __launch_bounds__(kTiledThreads, 1) grid_tiled_kernel(const TiledArgs a, float2* __restrict__ grid) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint4* stage = reinterpret_cast<uint4*>(smem_raw) + (threadIdx.x >> 5) * 32;       // this warp's descriptors
    float2* tab_s = reinterpret_cast<float2*>(smem_raw + kStageBytes);
    const uint32_t tab_addr = (uint32_t)__cvta_generic_to_shared(tab_s);
    __shared__ int s_block, s_next;
    const int lane = threadIdx.x & 31, lx = lane & (kLaneW - 1), ly = lane >> 3;
    const Geometry g = a.g;
    const int n_blocks = *a.n_blocks;
    int cur_kset = -1, cur_group = -1;
    for (;;) {
        __syncthreads();                                   // everyone is done with the previous block
        if (threadIdx.x == 0) {
            s_block = atomicAdd(a.queue, 1);
            s_next = 0;
        }
        __syncthreads();
        if (s_block >= n_blocks) break;
        const Block blk = a.blocks[s_block];
        const SetPlan sp = a.set_plan[blk.kset];
        const int S = a.set_support[blk.kset], h_lo = S / 2;
        if (blk.kset != cur_kset || blk.group != cur_group) {
            load_table_group(a, blk.kset, blk.group, sp, S, tab_s);
            cur_kset = blk.kset;
            cur_group = blk.group;
            __syncthreads();
        }
        const int slice_bytes = (S + 2 * kPad) * sp.pitch * 8;
        const int step_bytes = kLaneH * sp.pitch * 8;              // one row group down
        const int sub_lo = blk.group * sp.group_slices;
        const uint32_t lane_off = (uint32_t)((ly * sp.pitch + lx) * 8);
        for (;;) {
            int ei = 0;
            if (lane == 0) ei = atomicAdd(&s_next, 1);
            ei = __shfl_sync(0xffffffffu, ei, 0);
            if (ei >= blk.count) break;
            const Entry ent = a.entries[blk.first + ei];
            int Xw, Yw, bx_lo, bx_hi, by_lo, by_hi;
            strip_buckets(g, ent.strip, S, Xw, Yw, bx_lo, bx_hi, by_lo, by_hi);
            float2 A0[kNY], B0[kNY], A1[kNY], B1[kNY];
#pragma unroll
            for (int j = 0; j < kNY; ++j) A0[j] = B0[j] = A1[j] = B1[j] = make_float2(0.f, 0.f);
            bool any = false;
            int skip = ent.part * kChunk, take = kChunk;
            for (int by = by_lo; by <= by_hi && take > 0; ++by) {
                const int b0 = (blk.kset * g.nt + by) * g.nt;
                const int r0 = a.bucket_offset[b0 + bx_lo], r1 = a.bucket_offset[b0 + bx_hi + 1];
                if (skip >= r1 - r0) { skip -= r1 - r0; continue; }
                const int beg = r0 + skip, end = min(r1, beg + take);
                skip = 0;
                take -= end - beg;
                for (int i0 = beg; i0 < end; i0 += 32) {
                    const int idx = i0 + lane;
                    bool hit = false;
                    uint32_t packed = 0u;
                    if (idx < end) {
                        const uint2 geo = a.sgeo[idx];
                        const int gx = (int)(geo.x & 0xffffu), gy = (int)(geo.x >> 16);
                        const int dx0 = Xw - (gx - h_lo), dy0 = Yw - (gy - h_lo);   // tap coordinates of the strip origin
                        const int sub = (int)geo.y - sub_lo;
                        hit = (dx0 + kStripW > 0) && (dx0 < S) && (dy0 + kStripH > 0) && (dy0 < S) &&
                              ((unsigned)sub < (unsigned)sp.group_slices);
                        if (hit) {
                            const float2 v = a.sval[idx];
                            const int jl = (dy0 + kPad < 0) ? (-dy0) / kLaneH : 0;        // first group reaching row 0
                            const int jh = min(kNY, (S - 1 - dy0) / kLaneH + 1);          // one past the last group
                            const uint32_t left = (dx0 + kLaneW > 0) ? 1u : 0u;           // x-half 0 meets the footprint
                            const uint32_t right = (dx0 + kLaneW < S) ? 1u : 0u;          // x-half 1 meets the footprint
                            uint4 desc;                                                   // address may wrap; valid taps do not
                            desc.x = tab_addr + (uint32_t)(sub * slice_bytes + ((dy0 + kPad) * sp.pitch + dx0) * 8);
                            desc.y = __float_as_uint(v.x);
                            desc.z = __float_as_uint(v.y);
                            desc.w = 0u;
                            stage[lane] = desc;
                            packed = (uint32_t)jl | ((uint32_t)(jh - 1) << 3) | (left << 6) | (right << 7) |
                                     ((uint32_t)(dx0 & 0xff) << 8);
                        }
                    }
                    unsigned m = __ballot_sync(0xffffffffu, hit);
                    if (m == 0u) continue;
                    any = true;
                    __syncwarp();
                    while (m) {                                    // m, src, ctrl are warp-uniform by construction
                        const int src = __ffs(m) - 1;
                        m &= m - 1;
                        const uint32_t ctrl = __reduce_or_sync(0xffffffffu, lane == src ? packed : 0u);
                        const uint4 d = stage[src];                // broadcast LDS.128
                        const int jl = (int)(ctrl & 7u), jh = (int)((ctrl >> 3) & 7u) + 1;
                        const int c0 = (int)(int8_t)((ctrl >> 8) & 0xffu) + lx;           // this lane's tap column, x-half 0
                        const float vr = __uint_as_float(d.y), vi = __uint_as_float(d.z);
                        const float2 vrr = make_float2(vr, vr), vii = make_float2(vi, vi);
                        // lanes outside the footprint columns read a zero tap (first pad element) with step 0
                        const bool v0 = (unsigned)c0 < (unsigned)S, v1 = (unsigned)(c0 + kLaneW) < (unsigned)S;
                        const uint32_t addr0 = v0 ? d.x + lane_off : tab_addr, step0 = v0 ? (uint32_t)step_bytes : 0u;
                        const uint32_t addr1 = v1 ? d.x + lane_off + kLaneW * 8 : tab_addr, step1 = v1 ? (uint32_t)step_bytes : 0u;
                        const uint32_t halves = ctrl & 0xc0u;
                        if (halves == 0xc0u) {
                            IMAGER_CHAIN(IMAGER_SLOT_BOTH)
                        } else if (halves == 0x40u) {
                            IMAGER_CHAIN(IMAGER_SLOT_LEFT)
                        } else {
                            IMAGER_CHAIN(IMAGER_SLOT_RIGHT)
                        }
                    }
                    __syncwarp();
                }
            }
            if (any) {
#pragma unroll
                for (int j = 0; j < kNY; ++j) {
                    const int64_t cell = (int64_t)(Yw + ly + kLaneH * j) * g.N + Xw + lx;
                    float re = A0[j].x - B0[j].y, im = A0[j].y + B0[j].x;
                    if (re != 0.f || im != 0.f) atomicAdd(&grid[cell], make_float2(re, im));
                    re = A1[j].x - B1[j].y;
                    im = A1[j].y + B1[j].x;
                    if (re != 0.f || im != 0.f) atomicAdd(&grid[cell + kLaneW], make_float2(re, im));
                }
            }
        }
    }
}

// ---- host side -------------------------------------------------------------------------------------------

struct TiledState {
    std::vector<SetPlan> plan;
    std::vector<int32_t> unit_set;
    SetPlan* d_plan = nullptr;
    int32_t* d_unit_set = nullptr;
    int32_t* d_ref_mask = nullptr;        // per set: 1 = no tiled plan (reference kernels handle it)
    int32_t* d_parts = nullptr;           // [n_units * n_strips + 1] -> scanned into entry starts
    int32_t* d_scan_tmp = nullptr;
    Entry* d_entries = nullptr;
    Block* d_blocks = nullptr;
    int64_t max_entries = 0, max_blocks = 0;
    uint2* d_sgeo = nullptr;
    float2* d_sval = nullptr;
    int64_t geo_epoch = -1;
    Geometry g;
    int smem_bytes = 0;
    bool any_tiled = false, any_ref = false, usable = true;
};

bool tiled_supported(const imager_plan* pl) {
    const imager_params& p = pl->p;
    if (!(p.n_corr == 1 && p.n_pol == 1 && p.grid_size % kStripH == 0 && p.grid_size <= 32768 &&
          p.kernel_mode != IMAGER_MODE_DELTA))
        return false;
    const int64_t n_strips = (int64_t)(p.grid_size / kStripW) * (p.grid_size / kStripH);
    return (int64_t)pl->n_sets * p.oversample * p.oversample * n_strips <= kMaxPlanCells;   // conservative (all groups)
}

static TiledState* state_of(imager_plan* pl) {
    if (pl->tiled) return static_cast<TiledState*>(pl->tiled);
    TiledState* st = new TiledState();
    const imager_params& p = pl->p;
    const int O = p.oversample;
    st->plan.resize(pl->n_sets);
    int units = 0;
    for (int k = 0; k < pl->n_sets; ++k) {
        const int S = pl->set_support[k];
        SetPlan sp;
        sp.pitch = ((S + 7) / 16) * 16 + 8;                 // smallest value >= S that is 8 mod 16
        const int64_t slice_bytes = (int64_t)(S + 2 * kPad) * sp.pitch * 8;
        sp.group_slices = 0;
        for (int gsl : {O * O, O, 1})
            if (gsl * slice_bytes <= kMaxSmem - 1024 - kStageBytes) { sp.group_slices = gsl; break; }
        sp.n_groups = sp.group_slices ? (O * O) / sp.group_slices : 0;
        sp.unit_base = units;
        units += sp.n_groups;
        for (int q = 0; q < sp.n_groups; ++q) st->unit_set.push_back(k);
        if (sp.group_slices) {
            st->any_tiled = true;
            st->smem_bytes = std::max<int>(st->smem_bytes, (int)(sp.group_slices * slice_bytes) + kStageBytes);
        } else {
            st->any_ref = true;
        }
        st->plan[k] = sp;
    }
    Geometry& g = st->g;
    g.N = p.grid_size;
    g.O = O;
    g.nt = pl->nt;
    g.strips_per_row = p.grid_size / kStripW;
    g.n_strips = g.strips_per_row * (p.grid_size / kStripH);
    g.n_sets = pl->n_sets;
    g.n_units = units;
    pl->tiled = st;
    return st;
}

void tiled_release(imager_plan* pl) {
    if (!pl->tiled) return;
    TiledState* st = static_cast<TiledState*>(pl->tiled);
    cudaFree(st->d_plan);
    cudaFree(st->d_unit_set);
    cudaFree(st->d_ref_mask);
    cudaFree(st->d_parts);
    cudaFree(st->d_scan_tmp);
    cudaFree(st->d_entries);
    cudaFree(st->d_blocks);
    cudaFree(st->d_sgeo);
    cudaFree(st->d_sval);
    delete st;
    pl->tiled = nullptr;
}

static int prepare(imager_plan* pl, TiledState* st, cudaStream_t stream) {
    const int64_t mv = std::max<int64_t>(pl->p.max_nvis, 1);
    const Geometry& g = st->g;
    const int64_t n_cells = (int64_t)g.n_units * g.n_strips;
    if (!st->d_plan) {
        std::vector<int32_t> mask(pl->n_sets);
        for (int k = 0; k < pl->n_sets; ++k) mask[k] = st->plan[k].group_slices == 0;
        IMAGER_CUDA(cudaMalloc(&st->d_plan, pl->n_sets * sizeof(SetPlan)));
        IMAGER_CUDA(cudaMalloc(&st->d_ref_mask, pl->n_sets * sizeof(int32_t)));
        IMAGER_CUDA(cudaMalloc(&st->d_unit_set, std::max<size_t>(1, st->unit_set.size()) * sizeof(int32_t)));
        IMAGER_CUDA(cudaMemcpyAsync(st->d_plan, st->plan.data(), pl->n_sets * sizeof(SetPlan), cudaMemcpyHostToDevice, stream));
        IMAGER_CUDA(cudaMemcpyAsync(st->d_ref_mask, mask.data(), pl->n_sets * sizeof(int32_t), cudaMemcpyHostToDevice, stream));
        IMAGER_CUDA(cudaMemcpyAsync(st->d_unit_set, st->unit_set.data(), st->unit_set.size() * sizeof(int32_t),
                                    cudaMemcpyHostToDevice, stream));
        IMAGER_CUDA(cudaStreamSynchronize(stream));     // one-off: `mask` goes out of scope
        // every visibility is a candidate of at most ceil((32+S+W)/W) * ceil((32+S+H)/H) strips; bound with S = 255
        st->max_entries = n_cells + 2 + (mv * 20 * 11) / kChunk;
        st->max_blocks = g.n_units + st->max_entries / kBlockEntries + 2;
        int64_t tmp_len = 16;
        for (int64_t n = n_cells + 1; n > 1; n = (n + 1023) / 1024) tmp_len += (n + 1023) / 1024 + 1;
        IMAGER_CUDA(cudaMalloc(&st->d_parts, (n_cells + 1) * sizeof(int32_t)));
        IMAGER_CUDA(cudaMalloc(&st->d_scan_tmp, tmp_len * sizeof(int32_t)));
        IMAGER_CUDA(cudaMalloc(&st->d_entries, st->max_entries * sizeof(Entry)));
        IMAGER_CUDA(cudaMalloc(&st->d_blocks, st->max_blocks * sizeof(Block)));
        IMAGER_CUDA(cudaMalloc(&st->d_sgeo, mv * sizeof(uint2)));
        IMAGER_CUDA(cudaMalloc(&st->d_sval, mv * pl->p.n_corr * sizeof(float2)));
        IMAGER_CUDA(cudaFuncSetAttribute(grid_tiled_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem - 1024));
    }
    if (st->geo_epoch != pl->index_epoch) {
        sorted_geo_kernel<<<4 * kNumSMs, 256, 0, stream>>>(pl->d_counters, pl->d_perm[pl->sorted_buf], pl->d_rec,
                                                           pl->p.oversample, st->d_sgeo);
        const unsigned nb = (unsigned)((n_cells + 1 + 255) / 256);
        plan_count_kernel<<<nb, 256, 0, stream>>>(g, st->d_plan, st->d_unit_set, pl->d_set_support, pl->d_bucket_offset,
                                                  st->d_parts);
        pl->last_launches += 2;
        int rc = exclusive_scan_i32(pl, st->d_parts, n_cells + 1, st->d_scan_tmp, stream);
        if (rc) return rc;
        plan_fill_kernel<<<nb, 256, 0, stream>>>(g, st->d_parts, st->d_entries);
        plan_blocks_kernel<<<1, 1024, 0, stream>>>(g, st->d_plan, st->d_unit_set, st->d_parts, st->d_blocks, pl->d_counters + 9);
        pl->last_launches += 2;
        st->geo_epoch = pl->index_epoch;
    }
    return 0;
}

int launch_grid_tiled(imager_plan* pl, int64_t nvis, const float2* vis, const float* weights, float2* grid,
                      cudaStream_t stream) {
    if (nvis == 0) return 0;
    TiledState* st = state_of(pl);
    int rc = prepare(pl, st, stream);
    if (rc) return rc;
    if (st->any_ref) {
        rc = launch_grid_reference(pl, nvis, vis, weights, grid, st->d_ref_mask, stream);   // sets without a tiled plan
        if (rc) return rc;
    }
    if (!st->any_tiled) return 0;
    gather_values_kernel<1><<<4 * kNumSMs, 256, 0, stream>>>(pl->d_counters, pl->d_perm[pl->sorted_buf], vis, weights, st->d_sval);
    IMAGER_CUDA(cudaMemsetAsync(pl->d_counters + 8, 0, sizeof(int32_t), stream));
    TiledArgs a;
    a.g = st->g;
    a.bucket_offset = pl->d_bucket_offset;
    a.sgeo = st->d_sgeo;
    a.sval = st->d_sval;
    a.tab = pl->d_tab_grid;
    a.set_offset = pl->d_set_offset;
    a.set_support = pl->d_set_support;
    a.set_plan = st->d_plan;
    a.entries = st->d_entries;
    a.blocks = st->d_blocks;
    a.n_blocks = pl->d_counters + 9;
    a.queue = pl->d_counters + 8;
    grid_tiled_kernel<<<kNumSMs, kTiledThreads, st->smem_bytes, stream>>>(a, grid);
    pl->last_launches += 2;
    IMAGER_CUDA(cudaGetLastError());
    return 0;
}

int launch_degrid_tiled(imager_plan* pl, int64_t nvis, const float2* grid, float2* vis_out, cudaStream_t stream) {
    return launch_degrid_reference(pl, nvis, grid, vis_out, nullptr, stream);
}

}  // namespace imager
