// gridder_tiled.cu -- the output-stationary ("tiled") gridding and degridding kernels (hot-path steps A3 / A6) and
// their work planner (part of A2).  DESIGN.md section 6.2.
//
// Why this shape: every complex MAC needs one 8-byte tap that no other MAC can share (the tap index depends on
// visibility AND cell), and on sm_100a ANY shared-memory load of up to 8 bytes per lane occupies the LSU pipe for
// 2.1 clocks per warp instruction whatever its lane mask or address pattern (profiles/r1_lds_mask_probe.md), so the
// binding unit is shared-memory load INSTRUCTIONS, not HBM and not the FMA pipe (1 LDS.64 + 2 FFMA2 per 32 complex
// MACs = 50 % of the FP32 peak at best).  The kernels therefore
//   (1) keep grid cells in REGISTERS: a warp owns a 16 x 32 strip, its 8 x 4 lane block replicated 2 x 8 times
//       ("slots": 16 cells per lane), one packed accumulator per cell (complex MAC = two FFMA2 with operand modifiers);
//   (2) keep one unit (kernel set x group of sub-cell slices x Mueller element) resident in SHARED memory, rows
//       zero-padded by 3, columns by 7, pitched to 8 mod 16 taps: an 8 x 4 lane block reads conflict-free, and
//       lanes beyond a footprint edge read zeros without any per-lane test;
//   (3) replay precomputed HITS: a hit is one (visibility, strip) pair with the tap address of the strip origin
//       and the range of slots its footprint meets.  The hit lists are built on the device when (uvw, a_index)
//       are indexed and are cached while those do not change (IMAGER_REUSE_INDEX: every major cycle after the
//       first).  Hits are replayed in runs of equal slot range: one REDUX + ballot per run, then per hit one broadcast
//       LDS.128 (value and tap address, loaded a hit ahead) and straight-line code specialised for the range
//       (1 LDS.64 + 2 FFMA2 per slot, nothing else);
//   (4) gridding flushes a strip once per work item with red.global.add.v2.f32; degridding loads the strip once
//       per item, writes each hit's 32 partial sums with one STS.64, sums 16 hits at a time by a transposed read and
//       one shuffle stage, and adds the result to the visibility with one red.global.add.v2.f32.
// Work planning (visibility-centric; a warp counts the lanes that meet each strip of its window with one ballot and
// issues one atomic per strip): hits per (geometry unit, strip) are counted, scanned, emitted and counting-sorted by
// slot-range variant; item = up to kItemHits hits of one (unit, strip); block =
// consecutive items of one unit with about kBlockHits hits, times one Mueller element (s, c); persistent CTAs pull
// blocks from a two-ended global queue (small blocks last), their warps pull items of the block from a shared counter.
#include "common.cuh"

namespace imager {

// ---- checked build (-DIMAGER_CHECKED=1 -> libimager_checked.so): every index formed below is tested against its
// bounds and violations are counted per check (imager_debug_violations) instead of being dereferenced blindly ----
#ifndef IMAGER_CHECKED
#define IMAGER_CHECKED 0
#endif
__device__ unsigned long long g_violations[16];
#if IMAGER_CHECKED
#define IMAGER_CHECK(k, cond) ((cond) ? true : (atomicAdd(&g_violations[k], 1ull), false))
#else
#define IMAGER_CHECK(k, cond) (true)
#endif
enum { kChkHitPlace = 0, kChkVisIndex = 1, kChkTapAddr = 2, kChkStrip = 3, kChkItem = 4, kChkBlock = 5, kChkHash = 6, kChkWindow = 7 };

constexpr int kLaneW = 8, kLaneH = 4;                 // lane block
constexpr int kNX = 2, kNY = 8;                       // replications: strip = 16 x 32 cells
constexpr int kStripW = kLaneW * kNX, kStripH = kLaneH * kNY;
constexpr int kPadY = kLaneH - 1, kPadX = kLaneW - 1;
#ifndef IMAGER_DEGRID_THREADS
#define IMAGER_DEGRID_THREADS 512
#endif
constexpr int kTiledThreads = IMAGER_DEGRID_THREADS, kWarps = kTiledThreads / 32;   // degridding kernel
#ifndef IMAGER_GRID_THREADS
#define IMAGER_GRID_THREADS 768
#endif
constexpr int kGridThreads = IMAGER_GRID_THREADS;     // gridding kernel: threads per CTA (one CTA per SM)
#ifndef IMAGER_CHUNK3
#define IMAGER_CHUNK3 4
#endif
#ifndef IMAGER_ITEM_HITS
#define IMAGER_ITEM_HITS 384
#endif
#ifndef IMAGER_BLOCK_HITS
#define IMAGER_BLOCK_HITS 73728
#endif
constexpr int kItemHits = IMAGER_ITEM_HITS;                        // hits per work item (one flush / strip load each)
constexpr int kBlockHits = IMAGER_BLOCK_HITS;                     // hits per CTA-level block
constexpr int kStageBytes = kWarps * 32 * 8;          // per-warp hit descriptors (degridding): 32 x {tap address, sorted index}
constexpr int kStageSlots = 40;                       // gridding: 32 descriptors + the one read past a batch's end
constexpr int kGridStageBytes = (kGridThreads / 32) * kStageSlots * 16;
constexpr int kMaxSmem = 227 * 1024;
#ifndef IMAGER_RED_SLOTS
#define IMAGER_RED_SLOTS 16
#endif
constexpr int kRedSlots = IMAGER_RED_SLOTS;            // degridding: hits per transposed reduction (8, 16 or 32)
constexpr int kRedBytes = kWarps * kRedSlots * 32 * 8;
constexpr int kTableBudget = kMaxSmem - (kStageBytes + kRedBytes > kGridStageBytes ? kStageBytes + kRedBytes : kGridStageBytes) - 1024;   // 1 KB: static
static_assert(kTableBudget >= (127 + 2 * kPadY) * 152 * 8, "a support-127 slice (BASELINE.json configs[4]: 133 rows x 152 taps) must fit the table budget");
constexpr int64_t kMaxPlanCells = (int64_t)1 << 30;   // (geometry unit, strip) pairs: 12 bytes of planner state each
constexpr uint32_t kTapBias = 1u << 20;

struct SetPlan {           // per kernel set (host-built)
    int32_t pitch;         // taps per padded row, = 8 mod 16, >= S + 2 kPadX
    int32_t rows;          // S + 2 kPadY
    int32_t group_slices;  // sub-cell slices resident at once (a power of two <= O*O)
    int32_t n_groups;
    int32_t gu_base;       // first geometry unit of this set; gu = gu_base + group
    int32_t pad[3];
};

struct Item { int32_t strip, hit_begin, hit_count, pad; };
struct Block { int32_t gu, sc, item_begin, item_count; };

struct Geometry {
    int N, O, nt, strips_per_row, n_strips, n_sets, n_gu, n_pol, n_corr;
};

__device__ __forceinline__ float2 lds64(uint32_t addr) {
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
    return v;
}

// sorted-order geometry: word0 = gx | gy << 16, word1 = (oy_idx * O + ox_idx) | kernel set << kSubBits  (kept visibilities)
constexpr int kSubBits = 14;                          // O <= 128: sub-cell slice index < 2^14
constexpr uint32_t kSubMask = (1u << kSubBits) - 1u;
__global__ void sorted_geo_kernel(const int32_t* __restrict__ counters, const int32_t* __restrict__ perm,
                                  const imager_record* __restrict__ rec, int O, uint2* __restrict__ sgeo) {
    const int n_kept = counters[0];
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_kept; i += gridDim.x * blockDim.x) {
        const imager_record r = rec[perm[i]];
        sgeo[i] = make_uint2((uint32_t)r.gx | ((uint32_t)r.gy << 16),
                             (((r.sub >> 8) & 255u) * O + (r.sub & 255u)) | ((uint32_t)r.kset << kSubBits));
    }
}

// ---- exact pre-summation of duplicates (S16 / R16: "pre-summing duplicate (cell, sub-cell, plane, A-plane)
// visibilities is exact algebra") -----------------------------------------------------------------------------
// Visibilities with the same (kernel set, cell, sub-cell) use the same taps on the same cells: gridding grids the SUM of
// their weighted values once, degridding predicts one value and copies it.  rep[i] = the smallest sorted index with
// i's geometry among the kDedupeChunk consecutive sorted visibilities of i's chunk (equal geometries are neighbours in
// the sorted order up to the tile's other visibilities; a duplicate in another chunk is simply not merged).
#ifndef IMAGER_DEDUPE
#define IMAGER_DEDUPE 1
#endif
constexpr int kDedupeChunk = 4096, kDedupeSlots = 8192;          // shared hash table: load factor <= 0.5
constexpr int kDedupeSmem = kDedupeSlots * 12;
constexpr uint32_t kMergedFlag = 0x8000u;                       // bit 15 of sgeo.x (gx < 2^15): merged into another one
constexpr int kDedupeThreads = 1024, kDedupePer = kDedupeChunk / kDedupeThreads;   // 2 CTAs per SM: 64 warps hide the gather
// Fused with the sorted-geometry pass: one CTA builds sgeo for kDedupeChunk consecutive sorted visibilities, finds their
// representatives through a shared hash table (min sorted index per geometry) and flags the merged ones.
__global__ void __launch_bounds__(kDedupeThreads, 2) sorted_geo_dedupe_kernel(const int32_t* __restrict__ counters,
                                                                           const int32_t* __restrict__ perm,
                                                                           const imager_record* __restrict__ rec, int O,
                                                                           uint2* __restrict__ sgeo, int32_t* __restrict__ rep) {
    extern __shared__ __align__(16) unsigned char dedupe_smem[];
    unsigned long long* s_key = reinterpret_cast<unsigned long long*>(dedupe_smem);
    int32_t* s_idx = reinterpret_cast<int32_t*>(dedupe_smem + kDedupeSlots * sizeof(unsigned long long));
    const int n_kept = counters[0];
    const int c0 = blockIdx.x * kDedupeChunk;
    if (c0 >= n_kept) return;
    const int c1 = min(n_kept, c0 + kDedupeChunk);
    uint2 geo[kDedupePer];
#pragma unroll
    for (int j = 0; j < kDedupePer; ++j) {
        const int i = c0 + j * kDedupeThreads + threadIdx.x;
        if (i < c1) {
            const imager_record r = rec[perm[i]];
            geo[j] = make_uint2((uint32_t)r.gx | ((uint32_t)r.gy << 16),
                                (((r.sub >> 8) & 255u) * O + (r.sub & 255u)) | ((uint32_t)r.kset << kSubBits));
        }
    }
    for (int q = threadIdx.x; q < kDedupeSlots; q += blockDim.x) {
        s_key[q] = ~0ull;                                               // no geometry has all bits set (kset < 2^18)
        s_idx[q] = 0x7fffffff;
    }
    __syncthreads();
    for (int pass = 0; pass < 2; ++pass) {                              // 0: insert (min index per geometry), 1: look up
#pragma unroll
        for (int j = 0; j < kDedupePer; ++j) {
            const int i = c0 + j * kDedupeThreads + threadIdx.x;
            if (i >= c1) continue;
            const unsigned long long key = ((unsigned long long)geo[j].y << 32) | geo[j].x;
            uint32_t h = (uint32_t)((key * 0x9E3779B97F4A7C15ull) >> 51) & (kDedupeSlots - 1);
            for (int probes = 0;; ++probes) {
                const unsigned long long old = pass == 0 ? atomicCAS(&s_key[h], ~0ull, key) : s_key[h];
                if (old == key || (pass == 0 && old == ~0ull)) break;
                if (!IMAGER_CHECK(kChkHash, probes < kDedupeSlots)) break;      // load factor <= 0.5: cannot happen
                h = (h + 1) & (kDedupeSlots - 1);
            }
            if (pass == 0) {
                atomicMin(&s_idx[h], i);
            } else {
                const int r = s_idx[h];
                IMAGER_CHECK(kChkHash, r >= c0 && r <= i);
                rep[i] = r;
                sgeo[i] = make_uint2(geo[j].x | (r != i ? kMergedFlag : 0u), geo[j].y);
            }
        }
        __syncthreads();
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
            sval[(int64_t)i * NC + c] = weighted_sample(w, v);                  // R24
        }
    }
}

// gather_values + accumulate_duplicates in one pass: a CTA owns one dedupe chunk (a merged visibility and its
// representative are always in the same chunk), gathers the weighted values into shared memory, adds the merged ones
// to their representatives there, and writes the chunk out once.
template <int NC>
__global__ void __launch_bounds__(1024) gather_merge_values_kernel(const int32_t* __restrict__ counters, const int32_t* __restrict__ perm,
                                                                   const int32_t* __restrict__ rep, const float2* __restrict__ vis,
                                                                   const float* __restrict__ weights, float2* __restrict__ sval) {
    extern __shared__ __align__(16) unsigned char gm_smem[];
    float2* s_val = reinterpret_cast<float2*>(gm_smem);                   // [kDedupeChunk][NC]
    const int n_kept = counters[0];
    const int c0 = blockIdx.x * kDedupeChunk;
    if (c0 >= n_kept) return;
    const int c1 = min(n_kept, c0 + kDedupeChunk);
    for (int i = c0 + threadIdx.x; i < c1; i += blockDim.x) {
        const int64_t k = perm[i];
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const float2 v = vis[k * NC + c];
            const float w = weights[k * NC + c];
            s_val[(i - c0) * NC + c] = weighted_sample(w, v);                // R24
        }
    }
    __syncthreads();
    for (int i = c0 + threadIdx.x; i < c1; i += blockDim.x) {
        const int r = rep[i];
        if (r == i) continue;
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const float2 v = s_val[(i - c0) * NC + c];                    // a merged one is never a representative: not modified
            atomicAdd(&s_val[(r - c0) * NC + c].x, v.x);
            atomicAdd(&s_val[(r - c0) * NC + c].y, v.y);
        }
    }
    __syncthreads();
    for (int q = threadIdx.x; q < (c1 - c0) * NC; q += blockDim.x) sval[(int64_t)c0 * NC + q] = s_val[q];
}

// degridding epilogue: sorted-order sums -> vis_out in input order (dropped visibilities predict 0); with `residual`
// the prediction is subtracted from what vis_out holds (V - V_model, the major-cycle update)
template <int NC>
__global__ void scatter_values_kernel(int64_t nvis, const int32_t* __restrict__ counters, const int32_t* __restrict__ perm,
                                      const int32_t* __restrict__ rep, const float2* __restrict__ sval, int residual,
                                      float2* __restrict__ vis_out) {
    const int n_kept = counters[0];
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvis; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t k = perm[i];
        const int64_t src = (rep && i < n_kept) ? rep[i] : i;              // merged duplicates share one prediction
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const float2 m = i < n_kept ? sval[src * NC + c] : make_float2(0.f, 0.f);
            float2* o = vis_out + k * NC + c;
            *o = residual ? make_float2(o->x - m.x, o->y - m.y) : m;
        }
    }
}

// ---- planner ---------------------------------------------------------------------------------------------
// A hit of (gu, strip): a kept visibility of the unit's kernel set whose sub-cell slice is in the unit's group and
// whose footprint meets the strip.  Record: .x = sorted index of the visibility,
// .y = (tap offset of the strip origin within the group's shared-memory image + kTapBias) | ctrl << 24,
// ctrl = jl | (jh - 1) << 3 | halves << 6: slots jl .. jh-1 of x-half 0 (bit 6) and / or 1 (bit 7).
struct PlanArgs {
    Geometry g;
    const SetPlan* set_plan;
    const int32_t* gu_set;
    const int32_t* set_support;
    const uint2* sgeo;
    int64_t cap_hits;          // capacity of the hit-record arrays (checked build)
};

// ctrl byte of a candidate against a strip, or 0 if it is no hit (a hit always has bit 6 or 7 set)
__device__ __forceinline__ uint32_t hit_ctrl(int dx0, int dy0, int S, int sub, int group_slices) {
    const bool hit = (dx0 + kStripW > 0) && (dx0 < S) && (dy0 + kStripH > 0) && (dy0 < S) &&
                     ((unsigned)sub < (unsigned)group_slices);
    if (!hit) return 0u;
    const int jl = (dy0 + kPadY < 0) ? (-dy0) / kLaneH : 0;        // first slot reaching row 0
    const int jh = min(kNY, (S - 1 - dy0) / kLaneH + 1);           // one past the last slot
    const uint32_t left = (dx0 + kLaneW > 0) ? 1u : 0u;            // x-half 0 meets the footprint
    const uint32_t right = (dx0 + kLaneW < S) ? 1u : 0u;           // x-half 1 meets the footprint
    return (uint32_t)jl | ((uint32_t)(jh - 1) << 3) | (left << 6) | (right << 7);
}

// dense variant number of a ctrl byte (108 values)
#define IMAGER_VARIANT(H, JL, JH1) (((H) - 1) * 36 + (JL) * 8 - ((JL) * ((JL) - 1)) / 2 + (JH1) - (JL))
constexpr int kVariants = 108;

__device__ __forceinline__ uint32_t ctrl_variant(uint32_t ctrl) {
    const int jl = (int)(ctrl & 7u), jh1 = (int)((ctrl >> 3) & 7u), h = (int)(ctrl >> 6);
    return (uint32_t)IMAGER_VARIANT(h, jl, jh1);
}


// Hit counts per (gu, strip), visibility-centric and warp-aggregated.  The lanes of a warp hold 32 consecutive sorted
// visibilities: mostly one kernel set and one or two neighbouring 32 x 32 tiles, so their footprints meet the same few
// strips.  Per group of lanes with the same geometry unit the warp walks the bounding box of the group's strips (the
// "window", at most kWindowMax strips) and counts the lanes that meet each strip with one ballot: no __match_any_sync
// (the MIO queue was the limit of the match-based version: short_scoreboard 19.6, mio_throttle 15.8 stalls per issue),
// one atomic per (warp, strip).  Lane t keeps the count of window strip t (and t + 32).
constexpr int kWindowMax = 64;
// the strips a kept visibility meets: sx0 .. sx0 + nsx - 1, sy0 .. sy0 + nsy - 1 of geometry unit gu
struct VisHits {
    int gu, nsx, nsy, n, x0, y0, sx0, sy0, S, subl, kset;
};
__device__ __forceinline__ VisHits vis_hits(const PlanArgs& a, const uint2 geo) {
    VisHits v;
    const int gx = (int)(geo.x & 0x7fffu), gy = (int)(geo.x >> 16);           // bit 15: merged flag
    const int sub = (int)(geo.y & kSubMask);
    v.kset = (int)(geo.y >> kSubBits);
    const SetPlan sp = a.set_plan[v.kset];
    v.S = a.set_support[v.kset];
    const int h_lo = v.S / 2, group = sub / sp.group_slices;
    v.subl = sub - group * sp.group_slices;
    v.x0 = gx - h_lo;                                                  // footprint origin, inside the grid for kept ones
    v.y0 = gy - h_lo;
    v.sx0 = v.x0 / kStripW;
    v.sy0 = v.y0 / kStripH;
    v.nsx = (v.x0 + v.S - 1) / kStripW - v.sx0 + 1;
    v.nsy = (v.y0 + v.S - 1) / kStripH - v.sy0 + 1;
    v.n = v.nsx * v.nsy;
    v.gu = sp.gu_base + group;
    return v;
}

// One group of a warp's lanes (same geometry unit) and the window of strips they meet
struct HitWindow {
    unsigned group;            // lanes of the group
    int gu, x_lo, y_lo, w, h;  // window = strips x_lo .. x_lo + w - 1, y_lo .. y_lo + h - 1
};
__device__ __forceinline__ HitWindow next_window(const VisHits& v, bool valid, unsigned pending) {
    HitWindow win;
    const int leader = __ffs(pending) - 1;
    win.gu = __shfl_sync(0xffffffffu, v.gu, leader);
    const bool mine = valid && v.gu == win.gu;
    win.group = __ballot_sync(0xffffffffu, mine);
    win.x_lo = __reduce_min_sync(0xffffffffu, mine ? v.sx0 : 0x7fffffff);
    win.y_lo = __reduce_min_sync(0xffffffffu, mine ? v.sy0 : 0x7fffffff);
    win.w = __reduce_max_sync(0xffffffffu, mine ? v.sx0 + v.nsx : 0) - win.x_lo;
    win.h = __reduce_max_sync(0xffffffffu, mine ? v.sy0 + v.nsy : 0) - win.y_lo;
    IMAGER_CHECK(kChkWindow, win.x_lo >= 0 && win.y_lo >= 0 && win.w >= 1 && win.h >= 1);
    return win;
}

__global__ void count_hits_kernel(const PlanArgs a, const int32_t* __restrict__ counters, int32_t* __restrict__ hits,
                                  unsigned long long* __restrict__ total) {
    const Geometry& g = a.g;
    const int n_kept = counters[0];
    const int lane = threadIdx.x & 31;
    int mine_total = 0;                        // hits of this thread's visibilities (the 64-bit total guards the int32 scan)
    for (int i0 = (blockIdx.x * blockDim.x + threadIdx.x) - lane; i0 < n_kept; i0 += gridDim.x * blockDim.x) {
        const int i = i0 + lane;
        VisHits v;
        v.n = 0;
        v.gu = -1;
        if (i < n_kept) {
            const uint2 geo = a.sgeo[i];
            if (!(geo.x & 0x8000u)) v = vis_hits(a, geo);                      // merged duplicates have no hits of their own
        }
        mine_total += v.n;
        const bool valid = v.n > 0;
        unsigned pending = __ballot_sync(0xffffffffu, valid);
        while (pending) {
            const HitWindow win = next_window(v, valid, pending);
            const bool mine = (win.group >> lane) & 1u;
            const int64_t cell0 = (int64_t)win.gu * g.n_strips;
            IMAGER_CHECK(kChkWindow, win.gu >= 0 && win.gu < g.n_gu && win.x_lo + win.w <= g.strips_per_row &&
                                         (win.y_lo + win.h) * g.strips_per_row <= g.n_strips);
            if (win.w * win.h <= kWindowMax) {
                int cnt0 = 0, cnt1 = 0, t = 0;
                for (int Y = win.y_lo; Y < win.y_lo + win.h; ++Y)
                    for (int X = win.x_lo; X < win.x_lo + win.w; ++X, ++t) {
                        const bool in = mine && (unsigned)(X - v.sx0) < (unsigned)v.nsx && (unsigned)(Y - v.sy0) < (unsigned)v.nsy;
                        const int c = __popc(__ballot_sync(0xffffffffu, in));
                        if (lane == (t & 31)) {
                            if (t < 32) cnt0 = c; else cnt1 = c;
                        }
                    }
                if (cnt0) {
                    const int ty = lane / win.w;
                    atomicAdd(hits + cell0 + (int64_t)(win.y_lo + ty) * g.strips_per_row + win.x_lo + (lane - ty * win.w), cnt0);
                }
                if (cnt1) {
                    const int t1 = lane + 32, ty = t1 / win.w;
                    atomicAdd(hits + cell0 + (int64_t)(win.y_lo + ty) * g.strips_per_row + win.x_lo + (t1 - ty * win.w), cnt1);
                }
            } else if (mine) {                 // a group that straddles the end of a tile row: every lane on its own
                for (int ty = 0; ty < v.nsy; ++ty)
                    for (int tx = 0; tx < v.nsx; ++tx)
                        atomicAdd(hits + cell0 + (int64_t)(v.sy0 + ty) * g.strips_per_row + v.sx0 + tx, 1);
            }
            pending &= ~win.group;
        }
    }
    mine_total = __reduce_add_sync(0xffffffffu, mine_total);   // < 2^31: a thread sees at most 2^31 / gridDim visibilities x 162 strips
    if (lane == 0 && mine_total) atomicAdd(total, (unsigned long long)mine_total);
}

// totals -> mapped host memory: [0] hits (64-bit), [1] items (low word; high word 0)
__global__ void publish_totals_kernel(const unsigned long long* __restrict__ total, const int32_t* __restrict__ n_items,
                                      int64_t* __restrict__ host_totals) {
    host_totals[0] = (int64_t)*total;
    host_totals[1] = (int64_t)(uint32_t)*n_items;
    __threadfence_system();
}

// items[cell] = ceil(hits[cell] / kItemHits); entry n_cells (the terminator of the exclusive scans) is 0 in both
__global__ void items_from_hits_kernel(int64_t n_cells, const int32_t* __restrict__ hits, int32_t* __restrict__ items) {
    for (int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; c <= n_cells; c += (int64_t)gridDim.x * blockDim.x)
        items[c] = c < n_cells ? (hits[c] + kItemHits - 1) / kItemHits : 0;
}

// Unsorted hit records, visibility-centric: the same walk as count_hits_kernel.  Per window strip one lane reserves
// the places of the warp's hits with ONE atomic on the cell's cursor; a lane's hit takes place hit_start[cell] + that
// base + its rank among the lanes that meet the strip.
__device__ __forceinline__ void emit_one(const VisHits& v, int i, int X, int Y, int pitch, int slice_taps, int group_slices,
                                         int64_t pos, uint2* __restrict__ hit_tmp, const int32_t* __restrict__ range) {
    const int dx0 = X * kStripW - v.x0, dy0 = Y * kStripH - v.y0;          // taps of the strip origin
    const uint32_t ctrl = hit_ctrl(dx0, dy0, v.S, v.subl, group_slices);
    const int tapoff = v.subl * slice_taps + (dy0 + kPadY) * pitch + dx0 + kPadX;
    if (!IMAGER_CHECK(kChkHitPlace, ctrl != 0u && pos >= range[0] && pos < range[1])) return;   // range = hit_start + cell
    hit_tmp[pos] = make_uint2((uint32_t)i, (uint32_t)(tapoff + (int)kTapBias) | (ctrl << 24));
}

__global__ void emit_hits_kernel(const PlanArgs a, const int32_t* __restrict__ counters, const int32_t* __restrict__ hit_start,
                                 int32_t* __restrict__ cursor, uint2* __restrict__ hit_tmp) {
    const Geometry& g = a.g;
    const int n_kept = counters[0];
    const int lane = threadIdx.x & 31;
    const unsigned lt_mask = (1u << lane) - 1u;
    for (int i0 = (blockIdx.x * blockDim.x + threadIdx.x) - lane; i0 < n_kept; i0 += gridDim.x * blockDim.x) {
        const int i = i0 + lane;
        VisHits v;
        v.n = 0;
        v.gu = -1;
        int pitch = 0, slice_taps = 0, group_slices = 1;
        uint2 geo = make_uint2(0x8000u, 0u);
        if (i < n_kept) geo = a.sgeo[i];
        if (!(geo.x & 0x8000u)) {
            v = vis_hits(a, geo);
            const SetPlan sp = a.set_plan[v.kset];
            pitch = sp.pitch;
            slice_taps = sp.rows * sp.pitch;
            group_slices = sp.group_slices;
        }
        const bool valid = v.n > 0;
        unsigned pending = __ballot_sync(0xffffffffu, valid);
        while (pending) {
            const HitWindow win = next_window(v, valid, pending);
            const bool mine = (win.group >> lane) & 1u;
            const int64_t cell0 = (int64_t)win.gu * g.n_strips;
            IMAGER_CHECK(kChkWindow, win.gu >= 0 && win.gu < g.n_gu && win.x_lo + win.w <= g.strips_per_row &&
                                         (win.y_lo + win.h) * g.strips_per_row <= g.n_strips);
            if (win.w * win.h <= kWindowMax) {
                int cnt0 = 0, cnt1 = 0, t = 0;
                unsigned bal0 = 0u, bal1 = 0u;                               // lane t: the lanes that meet window strip t / t + 32
                for (int Y = win.y_lo; Y < win.y_lo + win.h; ++Y)
                    for (int X = win.x_lo; X < win.x_lo + win.w; ++X, ++t) {
                        const bool in = mine && (unsigned)(X - v.sx0) < (unsigned)v.nsx && (unsigned)(Y - v.sy0) < (unsigned)v.nsy;
                        const unsigned b = __ballot_sync(0xffffffffu, in);
                        if (lane == (t & 31)) {
                            if (t < 32) {
                                cnt0 = __popc(b);
                                bal0 = b;
                            } else {
                                cnt1 = __popc(b);
                                bal1 = b;
                            }
                        }
                    }
                int pos0 = 0, pos1 = 0;                                       // first place of window strip `lane` / `lane + 32`
                if (cnt0) {
                    const int ty = lane / win.w;
                    const int64_t cell = cell0 + (int64_t)(win.y_lo + ty) * g.strips_per_row + win.x_lo + (lane - ty * win.w);
                    pos0 = hit_start[cell] + atomicAdd(cursor + cell, cnt0);
                }
                if (cnt1) {
                    const int t1 = lane + 32, ty = t1 / win.w;
                    const int64_t cell = cell0 + (int64_t)(win.y_lo + ty) * g.strips_per_row + win.x_lo + (t1 - ty * win.w);
                    pos1 = hit_start[cell] + atomicAdd(cursor + cell, cnt1);
                }
                // every lane walks its own strips: place = the strip's base + this lane's rank among the lanes that meet it
                const bool big = win.w * win.h > 32;                           // warp-uniform
                const int n_own = mine ? v.n : 0;
                const int n_max = __reduce_max_sync(0xffffffffu, n_own);
                int tx = 0, ty = 0;
                for (int q = 0; q < n_max; ++q) {
                    const bool on = q < n_own;
                    const int X = v.sx0 + tx, Y = v.sy0 + ty;
                    const int wi = on ? (Y - win.y_lo) * win.w + (X - win.x_lo) : 0;
                    int base = __shfl_sync(0xffffffffu, pos0, wi & 31);
                    unsigned b = __shfl_sync(0xffffffffu, bal0, wi & 31);
                    if (big) {
                        const int base1 = __shfl_sync(0xffffffffu, pos1, wi & 31);
                        const unsigned b1 = __shfl_sync(0xffffffffu, bal1, wi & 31);
                        if (wi >= 32) {
                            base = base1;
                            b = b1;
                        }
                    }
                    if (on) emit_one(v, i, X, Y, pitch, slice_taps, group_slices, (int64_t)base + __popc(b & lt_mask), hit_tmp,
                                     hit_start + cell0 + (int64_t)Y * g.strips_per_row + X);
                    if (++tx == v.nsx) {
                        tx = 0;
                        ++ty;
                    }
                }
            } else if (mine) {
                for (int ty = 0; ty < v.nsy; ++ty)
                    for (int tx = 0; tx < v.nsx; ++tx) {
                        const int64_t cell = cell0 + (int64_t)(v.sy0 + ty) * g.strips_per_row + v.sx0 + tx;
                        emit_one(v, i, v.sx0 + tx, v.sy0 + ty, pitch, slice_taps, group_slices,
                                 (int64_t)hit_start[cell] + atomicAdd(cursor + cell, 1), hit_tmp, hit_start + cell);
                    }
            }
            pending &= ~win.group;
        }
    }
}

// item records: one thread per (gu, strip); item = up to kItemHits consecutive hits of the cell
__global__ void make_items_kernel(const Geometry g, const int32_t* __restrict__ hits, const int32_t* __restrict__ items,
                                  Item* __restrict__ item_rec) {
    const int64_t n_cells = (int64_t)g.n_gu * g.n_strips;
    for (int64_t cell = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; cell < n_cells; cell += (int64_t)gridDim.x * blockDim.x) {
        const int out = hits[cell], n_hits = hits[cell + 1] - out;
        if (n_hits == 0) continue;
        const int gu = (int)(cell / g.n_strips), strip = (int)(cell - (int64_t)gu * g.n_strips);
        const int i0 = items[cell], n_items = items[cell + 1] - i0;
        for (int p = 0; p < n_items; ++p)
            item_rec[i0 + p] = Item{strip, out + p * kItemHits, min(kItemHits, n_hits - p * kItemHits), gu};
    }
}

// One warp per sort unit: counting sort of the unit's hit records by variant (hit_tmp -> hit_rec), so that the kernels
// replay runs of hits with the same slot range.  A unit = the consecutive items of one (gu, strip) whose first hit
// falls into the same kSortSpan-aligned window of the hit array: at most kSortSpan hits, whatever the cell's size.
#ifndef IMAGER_SORT_ITEMS
#define IMAGER_SORT_ITEMS 2
#endif
constexpr int kSortSpan = IMAGER_SORT_ITEMS * kItemHits;
__global__ void __launch_bounds__(256, 4) sort_items_kernel(int n_items, const Item* __restrict__ item_rec,
                                                         const uint2* __restrict__ hit_tmp, uint2* __restrict__ hit_rec) {
    __shared__ int32_t s_bin[8][128];
    const int item = (int)(((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5);
    const int lane = threadIdx.x & 31, warp = (threadIdx.x >> 5) & 7;
    if (item >= n_items) return;
    const Item it = item_rec[item];
    const int window = it.hit_begin / kSortSpan;
    if (item > 0) {                                            // not the first item of its unit: nothing to do
        const Item pv = item_rec[item - 1];
        if (pv.strip == it.strip && pv.pad == it.pad && pv.hit_begin / kSortSpan == window) return;
    }
    const int out = it.hit_begin;
    int n_hits = it.hit_count;
    for (int k = 1; k < kSortSpan / kItemHits && item + k < n_items; ++k) {
        const Item nx = item_rec[item + k];
        if (nx.strip != it.strip || nx.pad != it.pad || nx.hit_begin / kSortSpan != window) break;
        n_hits += nx.hit_count;
    }
    constexpr int kPer = kSortSpan / 32;
    uint2 r[kPer];
    for (int q = lane; q < 128; q += 32) s_bin[warp][q] = 0;
    __syncwarp();
#pragma unroll
    for (int k = 0; k < kPer; ++k) {
        const int q = k * 32 + lane;
        r[k] = make_uint2(0u, 0u);
        if (q < n_hits) r[k] = hit_tmp[out + q];
    }
#pragma unroll
    for (int k = 0; k < kPer; ++k)
        if (k * 32 + lane < n_hits) atomicAdd(&s_bin[warp][ctrl_variant(r[k].y >> 24)], 1);
    __syncwarp();
    {                                                          // exclusive prefix of the 108 bins, 4 per lane
        int c[4], t = 0;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            c[q] = s_bin[warp][4 * lane + q];
            t += c[q];
        }
        int inc = t;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, inc, d);
            if (lane >= d) inc += y;
        }
        int run = inc - t;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            s_bin[warp][4 * lane + q] = run;
            run += c[q];
        }
    }
    __syncwarp();
    // scatter: a hit takes the next free place of its variant's range (order within a variant is irrelevant)
#pragma unroll
    for (int k = 0; k < kPer; ++k)
        if (k * 32 + lane < n_hits) hit_rec[out + atomicAdd(&s_bin[warp][ctrl_variant(r[k].y >> 24)], 1)] = r[k];
}

// one thread block per geometry unit: blocks of whole items, replicated for every Mueller element sc = s * n_corr + c.
// All but the last 1/kTailFrac of a unit's blocks go to the FRONT of `blocks` (about kBlockHits hits each), the rest into
// blocks of kBlockHits / kTailDiv hits at its BACK; the work queue serves the front part first, so that the kernel
// ends on small blocks (a short tail) without paying their overhead throughout.
#ifndef IMAGER_TAIL_DIV
#define IMAGER_TAIL_DIV 4
#endif
#ifndef IMAGER_TAIL_FRAC
#define IMAGER_TAIL_FRAC 16
#endif
constexpr int kTailDiv = IMAGER_TAIL_DIV, kTailFrac = IMAGER_TAIL_FRAC;
__device__ __forceinline__ int first_item_at(const Item* __restrict__ item_rec, int lo, int hi, int64_t limit) {
    while (lo < hi) {                                     // first item whose hit_begin >= limit
        const int mid = (lo + hi) >> 1;
        if (item_rec[mid].hit_begin < limit) lo = mid + 1; else hi = mid;
    }
    return lo;
}

__global__ void plan_blocks_kernel(const Geometry g, const int32_t* __restrict__ hit_start, const int32_t* __restrict__ item_start,
                                   const Item* __restrict__ item_rec, Block* __restrict__ blocks, int32_t* __restrict__ n_front,
                                   int32_t* __restrict__ n_back, int cap_blocks) {
    __shared__ int s_front, s_back;
    const int gu = blockIdx.x;
    const int n_sc = g.n_pol * g.n_corr;
    const int64_t c0 = (int64_t)gu * g.n_strips, c1 = c0 + g.n_strips;
    const int h0 = hit_start[c0], h1 = hit_start[c1], i0 = item_start[c0], i1 = item_start[c1];
    if (h1 == h0) return;
    const int nb_all = (h1 - h0 + kBlockHits - 1) / kBlockHits;
    const int nb_front = nb_all - (nb_all + kTailFrac - 1) / kTailFrac;   // whole big blocks in the front part
    const int64_t hs = (int64_t)h0 + (int64_t)nb_front * kBlockHits;  // the tail part starts here
    constexpr int kSmall = kBlockHits / kTailDiv;
    const int nb_back = (int)((h1 - hs + kSmall - 1) / kSmall);
    if (threadIdx.x == 0) {
        s_front = atomicAdd(n_front, nb_front * n_sc);
        s_back = atomicAdd(n_back, nb_back * n_sc);
    }
    __syncthreads();
    const int is = first_item_at(item_rec, i0, i1, hs);               // first item of the tail part
    for (int b = threadIdx.x; b < nb_front + nb_back; b += blockDim.x) {
        const bool front = b < nb_front;
        const int k = front ? b : b - nb_front, nbk = front ? nb_front : nb_back;
        const int64_t lo_hit = front ? (int64_t)h0 + (int64_t)k * kBlockHits : hs + (int64_t)k * kSmall;
        const int64_t hi_hit = front ? lo_hit + kBlockHits : lo_hit + kSmall;
        const int first = (k == 0) ? (front ? i0 : is) : first_item_at(item_rec, i0, i1, lo_hit);
        const int last = (k == nbk - 1) ? (front ? is : i1) : first_item_at(item_rec, i0, i1, hi_hit);
        const int cnt = max(last - first, 0);                         // items are whole: a small block may come out empty
        for (int sc = 0; sc < n_sc; ++sc) {
            const int slot = front ? s_front + sc * nb_front + k : cap_blocks - 1 - (s_back + sc * nb_back + k);
            blocks[slot] = Block{gu, sc, first, cnt};
        }
    }
}

// ---- the kernels -----------------------------------------------------------------------------------------
struct TiledArgs {
    Geometry g;
    const uint2* hit_rec;
    const Item* items;
    const Block* blocks;
    const int32_t* n_front;     // blocks at the front of `blocks` (served first)
    const int32_t* n_back;      // blocks at its back: entry cap_blocks - 1 - k
    int32_t cap_blocks;
    int32_t* queue;
    const float2* tab;
    const int64_t* set_offset;
    const int32_t* set_support;
    const SetPlan* set_plan;
    const int32_t* gu_set;
    int64_t n_hits;             // totals of the plan (checked build)
    int32_t n_items;
};

// checked build: a staged hit must stay inside the resident table group, name a kept visibility and a strip of the grid
__device__ __forceinline__ bool check_hit(const TiledArgs& a, const SetPlan& sp, const Item& it, bool live, uint2 rec) {
#if IMAGER_CHECKED
    bool ok = IMAGER_CHECK(kChkStrip, it.strip >= 0 && it.strip < a.g.n_strips && it.hit_begin >= 0 &&
                                          (int64_t)it.hit_begin + it.hit_count <= a.n_hits);
    if (live) {
        const uint32_t ctrl = rec.y >> 24;
        const int tapoff = (int)(rec.y & 0xffffffu) - (int)kTapBias;
        const int jl = (int)(ctrl & 7u), jh1 = (int)((ctrl >> 3) & 7u);
        const int lo = tapoff + jl * kLaneH * sp.pitch + ((ctrl & 0x40u) ? 0 : kLaneW);
        const int hi = tapoff + (jh1 * kLaneH + kLaneH - 1) * sp.pitch + ((ctrl & 0x80u) ? kStripW - 1 : kLaneW - 1);
        ok = IMAGER_CHECK(kChkTapAddr, (ctrl >> 6) != 0u && jl <= jh1 && lo >= 0 && hi < sp.group_slices * sp.rows * sp.pitch) && ok;
        ok = IMAGER_CHECK(kChkVisIndex, (int)rec.x >= 0 && (int)rec.x < a.queue[-8]) && ok;     // queue = counters + 8; counters[0] = n_kept
    }
    return ok;
#else
    return true;
#endif
}

// copy one slice group of element sc of kernel set `kset` into shared memory: [slice][row -3 .. S+2][col -7 ..], zero padded
__device__ void load_table_group(const TiledArgs& a, int kset, int group, int sc, const SetPlan sp, int S, float2* tab_s) {
    const int OO = a.g.O * a.g.O;
    const float2* T = a.tab + a.set_offset[kset] + ((int64_t)sc * OO + (int64_t)group * sp.group_slices) * S * S;
    const int per_slice = sp.rows * sp.pitch;
    const int total = sp.group_slices * per_slice;
    for (int i = threadIdx.x; i < total; i += blockDim.x) {
        const int sl = i / per_slice, rem = i - sl * per_slice;
        const int r = rem / sp.pitch, row = r - kPadY, col = rem - r * sp.pitch - kPadX;
        float2 v = make_float2(0.f, 0.f);
        if (row >= 0 && row < S && col >= 0 && col < S) v = __ldg(&T[((int64_t)sl * S + row) * S + col]);
        tab_s[i] = v;
    }
}

// ---- gridding bodies: a run of `cnt` staged hits with the same slot range, straight-line code per hit -----------
// slot j, x-half h: tap at addr + j * step + 64 h; A += t * vr, B += t * vi  (re = A.x - B.y, im = A.y + B.x at the flush)
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
    uint4 d;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(d.x), "=r"(d.y), "=r"(d.z), "=r"(d.w) : "r"(addr));
    return d;
}

__device__ __forceinline__ uint32_t lds32(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}

typedef unsigned long long u64;

__device__ __forceinline__ u64 pack2(float x, float y) {
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(x), "f"(y));
    return r;
}

__device__ __forceinline__ float2 unpack2(u64 v) {
    float2 r;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v));
    return r;
}

__device__ __forceinline__ void ffma2p(u64& d, u64 a, u64 b) { asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(d) : "l"(a), "l"(b)); }

// One complex MAC  acc += t * v  as two FFMA2 on ONE packed accumulator: acc += (t.re, t.im) * (v.re, v.re), then
// acc += (t.im, t.re) * (-v.im, v.im).  ptxas folds the swapped pair and the sign pattern into operand modifiers
// (FFMA2 R, -R.F32x2.LO_HI.NP, R.F32, R): no extra instruction, two registers per owned cell.
__device__ __forceinline__ void cmac_re(u64& acc, float2 t, float vr) { ffma2p(acc, pack2(t.x, t.y), pack2(vr, vr)); }
__device__ __forceinline__ void cmac_im(u64& acc, float2 t, float vi) { ffma2p(acc, pack2(t.y, t.x), pack2(-vi, vi)); }

// A run: `cnt` consecutive staged hits with the same slot range.  A hit's descriptor {value.x, value.y, tap address, -}
// is ONE broadcast LDS.128 (one wavefront), loaded a hit ahead; `d` carries the prefetched descriptor across runs.
template <int H, int JL, int JH>
__device__ __forceinline__ void grid_run(u64 (&C0)[kNY], u64 (&C1)[kNY], uint4& d, uint32_t desc_addr, int cnt,
                                         const uint32_t lane_off, const uint32_t (&step)[kNY]) {
#pragma unroll 1
    do {                                                     // cnt >= 1
        const uint32_t addr = d.z + lane_off;
        const float vx = __uint_as_float(d.x), vy = __uint_as_float(d.y);
        desc_addr += 16;
        d = lds128(desc_addr);                               // the next hit of the batch (one past it at its end: unused)
        // at most 8 tap loads in flight: chunks of 4 slots (both halves) or 8 slots (one half)
        constexpr int kChunk = (H == 3) ? IMAGER_CHUNK3 : 8;
#pragma unroll
        for (int j0 = JL; j0 < JH; j0 += kChunk) {
            float2 t0[kChunk], t1[kChunk];
#pragma unroll
            for (int j = j0; j < j0 + kChunk && j < JH; ++j) {
                if (H & 1) t0[j - j0] = lds64(addr + step[j]);
                if (H & 2) t1[j - j0] = lds64(addr + step[j] + kLaneW * 8);
            }
#pragma unroll
            for (int j = j0; j < j0 + kChunk && j < JH; ++j) {
                if (H & 1) cmac_re(C0[j], t0[j - j0], vx);
                if (H & 2) cmac_re(C1[j], t1[j - j0], vx);
            }
#pragma unroll
            for (int j = j0; j < j0 + kChunk && j < JH; ++j) {
                if (H & 1) cmac_im(C0[j], t0[j - j0], vy);
                if (H & 2) cmac_im(C1[j], t1[j - j0], vy);
            }
        }
    } while (--cnt > 0);
}

#define IMAGER_CASE(FN, H, JL, JH1) \
    case IMAGER_VARIANT(H, JL, JH1): FN<H, JL, (JH1) + 1> IMAGER_BODY_ARGS; break;
#define IMAGER_CASES_H(FN, H)                                                                                           \
    IMAGER_CASE(FN, H, 0, 0) IMAGER_CASE(FN, H, 0, 1) IMAGER_CASE(FN, H, 0, 2) IMAGER_CASE(FN, H, 0, 3)                  \
    IMAGER_CASE(FN, H, 0, 4) IMAGER_CASE(FN, H, 0, 5) IMAGER_CASE(FN, H, 0, 6) IMAGER_CASE(FN, H, 0, 7)                  \
    IMAGER_CASE(FN, H, 1, 1) IMAGER_CASE(FN, H, 1, 2) IMAGER_CASE(FN, H, 1, 3) IMAGER_CASE(FN, H, 1, 4)                  \
    IMAGER_CASE(FN, H, 1, 5) IMAGER_CASE(FN, H, 1, 6) IMAGER_CASE(FN, H, 1, 7)                                           \
    IMAGER_CASE(FN, H, 2, 2) IMAGER_CASE(FN, H, 2, 3) IMAGER_CASE(FN, H, 2, 4) IMAGER_CASE(FN, H, 2, 5)                  \
    IMAGER_CASE(FN, H, 2, 6) IMAGER_CASE(FN, H, 2, 7)                                                                    \
    IMAGER_CASE(FN, H, 3, 3) IMAGER_CASE(FN, H, 3, 4) IMAGER_CASE(FN, H, 3, 5) IMAGER_CASE(FN, H, 3, 6)                  \
    IMAGER_CASE(FN, H, 3, 7)                                                                                             \
    IMAGER_CASE(FN, H, 4, 4) IMAGER_CASE(FN, H, 4, 5) IMAGER_CASE(FN, H, 4, 6) IMAGER_CASE(FN, H, 4, 7)                  \
    IMAGER_CASE(FN, H, 5, 5) IMAGER_CASE(FN, H, 5, 6) IMAGER_CASE(FN, H, 5, 7)                                           \
    IMAGER_CASE(FN, H, 6, 6) IMAGER_CASE(FN, H, 6, 7)                                                                    \
    IMAGER_CASE(FN, H, 7, 7)
#define IMAGER_DISPATCH(FN, variant)   \
    switch (variant) {                 \
        IMAGER_CASES_H(FN, 1)          \
        IMAGER_CASES_H(FN, 2)          \
        IMAGER_CASES_H(FN, 3)          \
        default: break;                \
    }

// slot mask of a ctrl byte: bits 0-7 x-half 0, bits 8-15 x-half 1
__device__ __forceinline__ uint32_t ctrl_slot_mask(uint32_t ctrl) {
    const uint32_t jl = ctrl & 7u, jh = ((ctrl >> 3) & 7u) + 1u;
    const uint32_t rows = (1u << jh) - (1u << jl);
    return ((ctrl & 0x40u) ? rows : 0u) | ((ctrl & 0x80u) ? rows << 8 : 0u);
}

template <int NC>
__global__ void __launch_bounds__(kGridThreads, 1)
grid_tiled_kernel(const TiledArgs a, const float2* __restrict__ sval, float2* __restrict__ grid) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint4* stage = reinterpret_cast<uint4*>(smem_raw) + (threadIdx.x >> 5) * kStageSlots;  // this warp's descriptors
    float2* tab_s = reinterpret_cast<float2*>(smem_raw + kGridStageBytes);
    const uint32_t tab_addr = (uint32_t)__cvta_generic_to_shared(tab_s);
    const uint32_t stage_addr = (uint32_t)__cvta_generic_to_shared(stage);
    __shared__ int s_block, s_next;
    const int lane = threadIdx.x & 31, lx = lane & (kLaneW - 1), ly = lane >> 3;
    const Geometry g = a.g;
    const int n_front = *a.n_front, n_blocks = n_front + *a.n_back;
    int cur_gu = -1, cur_sc = -1;
    for (;;) {
        __syncthreads();                                   // everyone is done with the previous block
        if (threadIdx.x == 0) {
            s_block = atomicAdd(a.queue, 1);
            s_next = 0;
        }
        __syncthreads();
        if (s_block >= n_blocks) break;
        const Block blk = a.blocks[s_block < n_front ? s_block : a.cap_blocks - 1 - (s_block - n_front)];
        if (blk.item_count == 0) continue;
        if (!IMAGER_CHECK(kChkBlock, n_blocks <= a.cap_blocks && blk.gu >= 0 && blk.gu < g.n_gu && blk.sc >= 0 && blk.sc < g.n_pol * g.n_corr &&
                                         blk.item_begin >= 0 && blk.item_begin + blk.item_count <= a.n_items)) continue;
        const int kset = a.gu_set[blk.gu];
        const SetPlan sp = a.set_plan[kset];
        const int S = a.set_support[kset];
        if (blk.gu != cur_gu || blk.sc != cur_sc) {
            load_table_group(a, kset, blk.gu - sp.gu_base, blk.sc, sp, S, tab_s);
            cur_gu = blk.gu;
            cur_sc = blk.sc;
            __syncthreads();
        }
        const int s_pol = blk.sc / g.n_corr, c_corr = blk.sc - s_pol * g.n_corr;
        float2* gplane = grid + (int64_t)s_pol * g.N * g.N;
        // byte offsets of the 8 slots; each REDUX yields a uniform register, so that a tap load is LDS [R + UR] with
        // no per-slot address arithmetic
        uint32_t step[kNY];
#pragma unroll
        for (int j = 0; j < kNY; ++j) step[j] = __reduce_or_sync(0xffffffffu, (uint32_t)(j * kLaneH * sp.pitch * 8));
        const uint32_t lane_off = (uint32_t)((ly * sp.pitch + lx) * 8);
        for (;;) {
            int ii = 0;
            if (lane == 0) ii = atomicAdd(&s_next, 1);
            ii = __shfl_sync(0xffffffffu, ii, 0);
            if (ii >= blk.item_count) break;
            const Item it = a.items[blk.item_begin + ii];
            u64 C0[kNY], C1[kNY];
#pragma unroll
            for (int j = 0; j < kNY; ++j) C0[j] = C1[j] = 0ull;
            uint32_t touched = 0u;
            // software pipeline over batches of 32 hits (one per lane): the records of batch b + 2 and the values of
            // batch b + 1 are in flight while batch b is replayed
            uint2 rec = make_uint2(0u, 0u), rec1 = make_uint2(0u, 0u);
            float2 val = make_float2(0.f, 0.f);
            if (lane < it.hit_count) rec = a.hit_rec[it.hit_begin + lane];
            if (lane + 32 < it.hit_count) rec1 = a.hit_rec[it.hit_begin + 32 + lane];
            if (lane < it.hit_count) val = sval[(int64_t)rec.x * NC + c_corr];
            for (int b0 = 0; b0 < it.hit_count; b0 += 32) {
                const int n = min(32, it.hit_count - b0);
                if (!check_hit(a, sp, it, lane < n, rec)) rec = make_uint2(0u, kTapBias | (0x40u << 24));   // checked build: a harmless hit
                const uint32_t my_ctrl = lane < n ? rec.y >> 24 : 0x40u;
                const uint32_t my_variant = ctrl_variant(my_ctrl);
                stage[lane] = make_uint4(__float_as_uint(val.x), __float_as_uint(val.y),
                                         tab_addr + (uint32_t)(((int)(rec.y & 0xffffffu) - (int)kTapBias) * 8), rec.x);
                if (lane < n) touched |= ctrl_slot_mask(my_ctrl);
                rec = rec1;
                if (b0 + 32 + lane < it.hit_count) val = sval[(int64_t)rec.x * NC + c_corr];
                if (b0 + 64 + lane < it.hit_count) rec1 = a.hit_rec[it.hit_begin + b0 + 64 + lane];
                __syncwarp();
                uint4 d = lds128(stage_addr);
                for (int h = 0; h < n;) {                                   // runs of equal variant (the planner sorted them)
                    const uint32_t variant = __reduce_or_sync(0xffffffffu, lane == h ? my_variant : 0u);   // warp-uniform
                    const int cnt = __popc(__ballot_sync(0xffffffffu, lane >= h && lane < n && my_variant == variant));
                    const uint32_t desc_addr = stage_addr + h * 16;
#define IMAGER_BODY_ARGS (C0, C1, d, desc_addr, cnt, lane_off, step)
                    IMAGER_DISPATCH(grid_run, variant)
#undef IMAGER_BODY_ARGS
                    h += cnt;
                }
                __syncwarp();
            }
            touched = __reduce_or_sync(0xffffffffu, touched);
            const int sy = it.strip / g.strips_per_row, sx = it.strip - sy * g.strips_per_row;
            float2* gp = gplane + (int64_t)(sy * kStripH + ly) * g.N + sx * kStripW + lx;
#pragma unroll
            for (int j = 0; j < kNY; ++j) {
                if (touched & (1u << j)) {
                    const float2 c = unpack2(C0[j]);
                    if (c.x != 0.f || c.y != 0.f) atomicAdd(gp + (int64_t)(kLaneH * j) * g.N, c);
                }
                if (touched & (0x100u << j)) {
                    const float2 c = unpack2(C1[j]);
                    if (c.x != 0.f || c.y != 0.f) atomicAdd(gp + (int64_t)(kLaneH * j) * g.N + kLaneW, c);
                }
            }
        }
    }
}


// ---- degridding ------------------------------------------------------------------------------------------
// Same hits, same ownership: the warp holds its strip of the grid in registers; a hit's lanes accumulate
// sum conj(t) g over their cells:  P += t * g.x, Q += t * g.y,  conj(t) g = (P.x + Q.y) + i (Q.x - P.y).
// The 32 partial sums of a hit go to a per-warp shared buffer red[slot][lane]; every kRedSlots = 16 hits the buffer is
// summed by a transposed read (lane = slot + 16 * half sums 16 columns, one shuffle stage joins the halves) and the result is
// added to the visibility's sorted-order sum with one red.global.add.v2.f32 per hit.  (Measured alternative, DESIGN.md
// section 6.4: the same sum by one mma.sync.m16n8k8 per hit with a TF32 head / tail split takes the reduction off the
// shared-memory pipe -- 77 % -> 54 % busy -- but the longer bodies miss the instruction cache more: 4.9 ms against 4.1.)

__device__ __forceinline__ void sts64(uint32_t addr, float2 v) {
    asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(addr), "f"(v.x), "f"(v.y) : "memory");
}

// conj(t) * g on one packed accumulator: acc += (t.re, t.im) * (g.re, -g.re), then acc += (t.im, t.re) * (g.im, g.im)
__device__ __forceinline__ void dmac_re(u64& acc, float2 t, float gr) { ffma2p(acc, pack2(t.x, t.y), pack2(gr, -gr)); }
__device__ __forceinline__ void dmac_im(u64& acc, float2 t, float gi) { ffma2p(acc, pack2(t.y, t.x), pack2(gi, gi)); }
__device__ __forceinline__ u64 add2p(u64 a, u64 b) {
    u64 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}

template <int H, int JL, int JH>
__device__ __forceinline__ void degrid_run(const float2 (&G0)[kNY], const float2 (&G1)[kNY], uint32_t desc_addr, int cnt,
                                           uint32_t red_addr, const uint32_t lane_off, const uint32_t (&step)[kNY]) {
    uint32_t a_cur = lds32(desc_addr);
#pragma unroll 1
    do {                                                     // cnt >= 1
        desc_addr += 8;
        const uint32_t a_next = lds32(desc_addr);            // one past the run at its end: unused
        const uint32_t addr = a_cur + lane_off;
        u64 P[2][2] = {{0ull, 0ull}, {0ull, 0ull}};          // [x-half][slot parity]: four independent FFMA2 chains
        constexpr int kChunk = (H == 3) ? 4 : 8;
#pragma unroll
        for (int j0 = JL; j0 < JH; j0 += kChunk) {
            float2 t0[kChunk], t1[kChunk];
#pragma unroll
            for (int j = j0; j < j0 + kChunk && j < JH; ++j) {
                if (H & 1) t0[j - j0] = lds64(addr + step[j]);
                if (H & 2) t1[j - j0] = lds64(addr + step[j] + kLaneW * 8);
            }
#pragma unroll
            for (int j = j0; j < j0 + kChunk && j < JH; ++j) {
                if (H & 1) dmac_re(P[0][j & 1], t0[j - j0], G0[j].x);
                if (H & 2) dmac_re(P[1][j & 1], t1[j - j0], G1[j].x);
            }
#pragma unroll
            for (int j = j0; j < j0 + kChunk && j < JH; ++j) {
                if (H & 1) dmac_im(P[0][j & 1], t0[j - j0], G0[j].y);
                if (H & 2) dmac_im(P[1][j & 1], t1[j - j0], G1[j].y);
            }
        }
        u64 sum;
        if (H == 3) sum = add2p(add2p(P[0][0], P[0][1]), add2p(P[1][0], P[1][1]));
        else if (H == 1) sum = add2p(P[0][0], P[0][1]);
        else sum = add2p(P[1][0], P[1][1]);
        sts64(red_addr, unpack2(sum));
        red_addr += 32 * 8;
        a_cur = a_next;
    } while (--cnt > 0);
}

template <int NC>
__global__ void __launch_bounds__(kTiledThreads, 1)
degrid_tiled_kernel(const TiledArgs a, const float2* __restrict__ grid, float2* __restrict__ ssum) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5;
    uint2* stage = reinterpret_cast<uint2*>(smem_raw) + warp * 32;                       // {tap address, sorted index}
    float2* red = reinterpret_cast<float2*>(smem_raw + kStageBytes) + warp * kRedSlots * 32;
    float2* tab_s = reinterpret_cast<float2*>(smem_raw + kStageBytes + kRedBytes);
    const uint32_t tab_addr = (uint32_t)__cvta_generic_to_shared(tab_s);
    const uint32_t stage_addr = (uint32_t)__cvta_generic_to_shared(stage);
    const uint32_t red_base = (uint32_t)__cvta_generic_to_shared(red);
    __shared__ int s_block, s_next;
    const int lane = threadIdx.x & 31, lx = lane & (kLaneW - 1), ly = lane >> 3;
    const Geometry g = a.g;
    const int n_front = *a.n_front, n_blocks = n_front + *a.n_back;
    int cur_gu = -1, cur_sc = -1;
    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) {
            s_block = atomicAdd(a.queue, 1);
            s_next = 0;
        }
        __syncthreads();
        if (s_block >= n_blocks) break;
        const Block blk = a.blocks[s_block < n_front ? s_block : a.cap_blocks - 1 - (s_block - n_front)];
        if (blk.item_count == 0) continue;
        if (!IMAGER_CHECK(kChkBlock, n_blocks <= a.cap_blocks && blk.gu >= 0 && blk.gu < g.n_gu && blk.sc >= 0 && blk.sc < g.n_pol * g.n_corr &&
                                         blk.item_begin >= 0 && blk.item_begin + blk.item_count <= a.n_items)) continue;
        const int kset = a.gu_set[blk.gu];
        const SetPlan sp = a.set_plan[kset];
        const int S = a.set_support[kset];
        if (blk.gu != cur_gu || blk.sc != cur_sc) {
            load_table_group(a, kset, blk.gu - sp.gu_base, blk.sc, sp, S, tab_s);
            cur_gu = blk.gu;
            cur_sc = blk.sc;
            __syncthreads();
        }
        const int s_pol = blk.sc / g.n_corr, c_corr = blk.sc - s_pol * g.n_corr;
        const float2* gplane = grid + (int64_t)s_pol * g.N * g.N;
        uint32_t step[kNY];
#pragma unroll
        for (int j = 0; j < kNY; ++j) step[j] = __reduce_or_sync(0xffffffffu, (uint32_t)(j * kLaneH * sp.pitch * 8));
        const uint32_t lane_off = (uint32_t)((ly * sp.pitch + lx) * 8);
        for (;;) {
            int ii = 0;
            if (lane == 0) ii = atomicAdd(&s_next, 1);
            ii = __shfl_sync(0xffffffffu, ii, 0);
            if (ii >= blk.item_count) break;
            const Item it = a.items[blk.item_begin + ii];
            const int sy = it.strip / g.strips_per_row, sx = it.strip - sy * g.strips_per_row;
            const float2* gp = gplane + (int64_t)(sy * kStripH + ly) * g.N + sx * kStripW + lx;
            float2 G0[kNY], G1[kNY];
#pragma unroll
            for (int j = 0; j < kNY; ++j) {
                G0[j] = __ldg(gp + (int64_t)(kLaneH * j) * g.N);
                G1[j] = __ldg(gp + (int64_t)(kLaneH * j) * g.N + kLaneW);
            }
            uint2 rec = make_uint2(0u, 0u), rec1 = make_uint2(0u, 0u);
            if (lane < it.hit_count) rec = a.hit_rec[it.hit_begin + lane];
            if (lane + 32 < it.hit_count) rec1 = a.hit_rec[it.hit_begin + 32 + lane];
            for (int b0 = 0; b0 < it.hit_count; b0 += 32) {
                const int n = min(32, it.hit_count - b0);
                if (!check_hit(a, sp, it, lane < n, rec)) rec = make_uint2(0u, kTapBias | (0x40u << 24));   // checked build: a harmless hit
                const uint32_t my_ctrl = lane < n ? rec.y >> 24 : 0x40u;
                const uint32_t my_variant = ctrl_variant(my_ctrl);
                stage[lane] = make_uint2(tab_addr + (uint32_t)(((int)(rec.y & 0xffffffu) - (int)kTapBias) * 8), rec.x);
                rec = rec1;
                if (b0 + 64 + lane < it.hit_count) rec1 = a.hit_rec[it.hit_begin + b0 + 64 + lane];
                __syncwarp();
                for (int h = 0; h < n;) {
                    const uint32_t variant = __reduce_or_sync(0xffffffffu, lane == h ? my_variant : 0u);   // warp-uniform
                    int cnt = __popc(__ballot_sync(0xffffffffu, lane >= h && lane < n && my_variant == variant));
                    cnt = min(cnt, kRedSlots - (h & (kRedSlots - 1)));          // runs do not cross a reduction batch
                    const uint32_t desc_addr = stage_addr + h * 8;
                    const uint32_t red_addr = red_base + (uint32_t)(((h & (kRedSlots - 1)) * 32 + lane) * 8);
#define IMAGER_BODY_ARGS (G0, G1, desc_addr, cnt, red_addr, lane_off, step)
                    IMAGER_DISPATCH(degrid_run, variant)
#undef IMAGER_BODY_ARGS
                    h += cnt;
                    if ((h & (kRedSlots - 1)) == 0 || h == n) {
                        // transposed reduction of hits [h0, h)
                        const int h0 = (h - 1) & ~(kRedSlots - 1);
                        __syncwarp();
                        // lane = slot + kRedSlots * part sums the kRedCols columns of its part
                        constexpr int kRedParts = 32 / kRedSlots, kRedCols = 32 / kRedParts;
                        const int slot = lane & (kRedSlots - 1), q = lane / kRedSlots;
                        float2 acc = make_float2(0.f, 0.f);
                        if (h0 + slot < h) {
#pragma unroll
                            for (int k = 0; k < kRedCols; ++k) {
                                const float2 v = lds64(red_base + (uint32_t)((slot * 32 + kRedCols * q + ((k + slot) & (kRedCols - 1))) * 8));
                                acc.x += v.x;
                                acc.y += v.y;
                            }
                        }
#pragma unroll
                        for (int d = kRedSlots; d < 32; d <<= 1) {
                            acc.x += __shfl_xor_sync(0xffffffffu, acc.x, d);
                            acc.y += __shfl_xor_sync(0xffffffffu, acc.y, d);
                        }
                        if (lane < kRedSlots && h0 + lane < h) {
                            const uint32_t idx = stage[h0 + lane].y;
                            atomicAdd(&ssum[(int64_t)idx * NC + c_corr], acc);
                        }
                        __syncwarp();
                    }
                }
                __syncwarp();
            }
        }
    }
}



// ---- host side -------------------------------------------------------------------------------------------

struct TiledState {
    std::vector<SetPlan> plan;
    std::vector<int32_t> gu_set;
    SetPlan* d_plan = nullptr;
    int32_t* d_gu_set = nullptr;
    int32_t* d_hits = nullptr;            // [n_cells + 1] -> scanned into hit starts
    int32_t* d_items = nullptr;           // [n_cells + 1] -> scanned into item starts
    int32_t* d_scan_tmp = nullptr;
    uint2* d_hit_rec = nullptr;
    uint2* d_hit_tmp = nullptr;           // unsorted hit records (planner scratch)
    int32_t* d_cursor = nullptr;          // [n_cells + 1] fill cursors of emit_hits_kernel
    Item* d_item_rec = nullptr;
    Block* d_blocks = nullptr;
    int64_t cap_hits = 0, cap_items = 0, cap_blocks = 0, cap_tmp = 0;
    int64_t* h_totals = nullptr;          // pinned, mapped [2]: hits (64-bit count), items -- written by publish_totals_kernel
    int64_t* d_h_totals = nullptr;        // the device's address of h_totals
    unsigned long long* d_total = nullptr;  // 64-bit hit count of count_hits_kernel
    bool initialised = false;             // set once every allocation of the first prepare() has succeeded
    uint2* d_sgeo = nullptr;
    int32_t* d_rep = nullptr;             // [max_nvis] representative of every sorted visibility (IMAGER_DEDUPE)
    float2* d_sval = nullptr;
    int64_t plan_epoch = -1;
    int32_t blocks_cap = 0;               // the two-ended block queue lives in d_blocks[0 .. blocks_cap)
    Geometry g;
    int smem_bytes = 0;                   // the largest resident table group (the kernels add their staging)
};

// taps per padded table row: >= S + 2 kPadX and such that the lane block of a half-warp wavefront reads conflict-free
// (8 x 2 lanes: 8 mod 16)
static int table_pitch(int S) {
    return ((S + 2 * kPadX + 7) / 16) * 16 + 8;
}

// NULL if the tiled kernels can run this plan, else the reason they cannot (imager_plan_path reports it)
const char* tiled_unsupported_reason(const imager_plan* pl) {
    const imager_params& p = pl->p;
    if (p.grid_size % kStripH != 0) return "grid_size is not a multiple of the 32-cell strip height";
    if (p.grid_size > 32768) return "grid_size exceeds 32768";
    if (pl->n_sets >= (1 << (32 - kSubBits))) return "too many kernel sets for the hit record's set field";
    // every slice (with its padding) must fit in shared memory, and the planner enumerates (gu, strip) pairs
    const int64_t n_strips = (int64_t)(p.grid_size / kStripW) * (p.grid_size / kStripH);
    int64_t n_gu = 0;
    for (int k = 0; k < pl->n_sets; ++k) {
        const int S = pl->set_support[k];
        const int pitch = table_pitch(S);
        const int64_t slice_bytes = (int64_t)(S + 2 * kPadY) * pitch * 8;
        if (slice_bytes > kTableBudget) return "one sub-cell slice of the largest kernel exceeds the shared-memory table budget";
        int gs = p.oversample * p.oversample;
        while (gs > 1 && gs * slice_bytes > kTableBudget) gs >>= 1;
        if ((p.oversample * p.oversample) % gs) return "oversample^2 is not a multiple of the sub-cell group size";
        n_gu += (p.oversample * p.oversample) / gs;
    }
    if (n_gu * n_strips > kMaxPlanCells) return "(kernel slice group, strip) pairs exceed the planner's table";
    return nullptr;
}

bool tiled_supported(const imager_plan* pl) { return tiled_unsupported_reason(pl) == nullptr; }

static TiledState* state_of(imager_plan* pl) {
    if (pl->tiled) return static_cast<TiledState*>(pl->tiled);
    TiledState* st = new TiledState();
    const imager_params& p = pl->p;
    const int OO = p.oversample * p.oversample;
    st->plan.resize(pl->n_sets);
    int n_gu = 0;
    for (int k = 0; k < pl->n_sets; ++k) {
        const int S = pl->set_support[k];
        SetPlan sp = {};
        sp.pitch = table_pitch(S);
        sp.rows = S + 2 * kPadY;
        const int64_t slice_bytes = (int64_t)sp.rows * sp.pitch * 8;
        int gs = OO;
        while (gs > 1 && gs * slice_bytes > kTableBudget) gs >>= 1;
        sp.group_slices = gs;
        sp.n_groups = OO / gs;
        sp.gu_base = n_gu;
        n_gu += sp.n_groups;
        for (int q = 0; q < sp.n_groups; ++q) st->gu_set.push_back(k);
        st->smem_bytes = std::max<int>(st->smem_bytes, (int)(gs * slice_bytes));
        st->plan[k] = sp;
    }
    Geometry& g = st->g;
    g.N = p.grid_size;
    g.O = p.oversample;
    g.nt = pl->nt;
    g.strips_per_row = p.grid_size / kStripW;
    g.n_strips = g.strips_per_row * (p.grid_size / kStripH);
    g.n_sets = pl->n_sets;
    g.n_gu = n_gu;
    g.n_pol = p.n_pol;
    g.n_corr = p.n_corr;
    pl->tiled = st;
    return st;
}

void tiled_release(imager_plan* pl) {
    if (!pl->tiled) return;
    TiledState* st = static_cast<TiledState*>(pl->tiled);
    cudaFree(st->d_plan);
    cudaFree(st->d_gu_set);
    cudaFree(st->d_hits);
    cudaFree(st->d_items);
    cudaFree(st->d_scan_tmp);
    cudaFree(st->d_hit_rec);
    cudaFree(st->d_hit_tmp);
    cudaFree(st->d_cursor);
    cudaFree(st->d_item_rec);
    cudaFree(st->d_blocks);
    cudaFree(st->d_sgeo);
    cudaFree(st->d_rep);
    cudaFree(st->d_sval);
    cudaFree(st->d_total);
    if (st->h_totals) cudaFreeHost(st->h_totals);
    delete st;
    pl->tiled = nullptr;
}

template <typename T>
static int grow(T** ptr, int64_t* cap, int64_t need) {
    if (need <= *cap) return 0;
    if (*ptr) IMAGER_CUDA(cudaFree(*ptr));
    *ptr = nullptr;
    *cap = 0;
    const int64_t n = need + need / 8 + 1024;
    IMAGER_CUDA(cudaMalloc(ptr, n * sizeof(T)));
    *cap = n;
    return 0;
}

// One-time allocations of the tiled path.  The hit lists are pre-sized from max_nvis and the mean number of strips a
// footprint meets (over the kernel sets), so that in the steady state -- and normally in the first call too -- no hot
// call allocates; prepare() still grows them if a data set needs more.
static int init_buffers(imager_plan* pl, TiledState* st, cudaStream_t stream) {
    const int64_t mv = std::max<int64_t>(pl->p.max_nvis, 1);
    const Geometry& g = st->g;
    const int64_t n_cells = (int64_t)g.n_gu * g.n_strips;
    IMAGER_CUDA(cudaMalloc(&st->d_plan, pl->n_sets * sizeof(SetPlan)));
    IMAGER_CUDA(cudaMalloc(&st->d_gu_set, st->gu_set.size() * sizeof(int32_t)));
    IMAGER_CUDA(cudaMemcpyAsync(st->d_plan, st->plan.data(), pl->n_sets * sizeof(SetPlan), cudaMemcpyHostToDevice, stream));
    IMAGER_CUDA(cudaMemcpyAsync(st->d_gu_set, st->gu_set.data(), st->gu_set.size() * sizeof(int32_t),
                                cudaMemcpyHostToDevice, stream));
    int64_t tmp_len = 16;
    for (int64_t n = n_cells + 1; n > 1; n = (n + 1023) / 1024) tmp_len += (n + 1023) / 1024 + 1;
    IMAGER_CUDA(cudaMalloc(&st->d_hits, (n_cells + 1) * sizeof(int32_t)));
    IMAGER_CUDA(cudaMalloc(&st->d_items, (n_cells + 1) * sizeof(int32_t)));
    IMAGER_CUDA(cudaMalloc(&st->d_cursor, (n_cells + 1) * sizeof(int32_t)));
    IMAGER_CUDA(cudaMalloc(&st->d_scan_tmp, tmp_len * sizeof(int32_t)));
    IMAGER_CUDA(cudaMalloc(&st->d_sgeo, mv * sizeof(uint2)));
#if IMAGER_DEDUPE
    IMAGER_CUDA(cudaMalloc(&st->d_rep, mv * sizeof(int32_t)));
    IMAGER_CUDA(cudaFuncSetAttribute(sorted_geo_dedupe_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kDedupeSmem));
    IMAGER_CUDA(cudaFuncSetAttribute(gather_merge_values_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     kDedupeChunk * 4 * (int)sizeof(float2)));
#endif
    IMAGER_CUDA(cudaMalloc(&st->d_sval, mv * pl->p.n_corr * sizeof(float2)));
    IMAGER_CUDA(cudaMalloc(&st->d_total, sizeof(unsigned long long)));
    IMAGER_CUDA(cudaHostAlloc(&st->h_totals, 2 * sizeof(int64_t), cudaHostAllocMapped));
    IMAGER_CUDA(cudaHostGetDevicePointer(&st->d_h_totals, st->h_totals, 0));
    st->h_totals[0] = st->h_totals[1] = 0;
    IMAGER_CUDA(cudaFuncSetAttribute(grid_tiled_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem - 1024));
    IMAGER_CUDA(cudaFuncSetAttribute(grid_tiled_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem - 1024));
    IMAGER_CUDA(cudaFuncSetAttribute(degrid_tiled_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem - 1024));
    IMAGER_CUDA(cudaFuncSetAttribute(degrid_tiled_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem - 1024));
    // expected strips per footprint: a footprint of S cells starting anywhere meets (S - 1) / W + 1 strips on average
    double per_vis = 0.0;
    for (int k = 0; k < pl->n_sets; ++k) {
        const double S = pl->set_support[k];
        per_vis += ((S - 1.0) / kStripW + 1.0) * ((S - 1.0) / kStripH + 1.0);
    }
    per_vis /= std::max(pl->n_sets, 1);
    const int64_t est_hits = std::min<int64_t>((int64_t)(per_vis * 1.25 * (double)mv) + 4096, (int64_t)0x7ffffff0);
    int rc = grow(&st->d_hit_rec, &st->cap_hits, est_hits);
    if (!rc) rc = grow(&st->d_hit_tmp, &st->cap_tmp, est_hits);
    if (!rc) rc = grow(&st->d_item_rec, &st->cap_items, est_hits / kItemHits + n_cells / 8 + 1024);
    return rc;
}

// (Re)build the hit lists, items and blocks for the current index.  Synchronises the stream once (the sizes of the
// lists are read back: they bound the launches that follow and guard the 32-bit offsets); cached until the next
// re-indexing.  Limit per call: fewer than 2^31 hits (visibility x strip pairs) -- larger data sets are fed in chunks
// (gridding accumulates into the caller's grid).
static int prepare(imager_plan* pl, TiledState* st, cudaStream_t stream) {
    const Geometry& g = st->g;
    const int64_t n_cells = (int64_t)g.n_gu * g.n_strips;
    if (!st->initialised) {
        const int rc = init_buffers(pl, st, stream);
        if (rc) {                                     // start clean at the next call instead of running on half a state
            tiled_release(pl);
            return rc;
        }
        st->initialised = true;
    }
    if (st->plan_epoch == pl->index_epoch) return 0;
#if IMAGER_DEDUPE
    sorted_geo_dedupe_kernel<<<(unsigned)((pl->indexed_nvis + kDedupeChunk - 1) / kDedupeChunk), kDedupeThreads, kDedupeSmem, stream>>>(
        pl->d_counters, pl->d_perm[pl->sorted_buf], pl->d_rec, pl->p.oversample, st->d_sgeo, st->d_rep);
#else
    sorted_geo_kernel<<<4 * num_sms(), 256, 0, stream>>>(pl->d_counters, pl->d_perm[pl->sorted_buf], pl->d_rec,
                                                       pl->p.oversample, st->d_sgeo);
#endif
    PlanArgs pa;
    pa.g = g;
    pa.set_plan = st->d_plan;
    pa.gu_set = st->d_gu_set;
    pa.set_support = pl->d_set_support;
    pa.sgeo = st->d_sgeo;
    pa.cap_hits = 0;
    IMAGER_CUDA(cudaMemsetAsync(st->d_hits, 0, (n_cells + 1) * sizeof(int32_t), stream));
    IMAGER_CUDA(cudaMemsetAsync(st->d_total, 0, sizeof(unsigned long long), stream));
    count_hits_kernel<<<8 * num_sms(), 256, 0, stream>>>(pa, pl->d_counters, st->d_hits, st->d_total);
    items_from_hits_kernel<<<2 * num_sms(), 256, 0, stream>>>(n_cells, st->d_hits, st->d_items);
    pl->last_launches += 3;
    int rc = exclusive_scan_i32(pl, st->d_hits, n_cells + 1, st->d_scan_tmp, stream);
    if (rc) return rc;
    rc = exclusive_scan_i32(pl, st->d_items, n_cells + 1, st->d_scan_tmp, stream);
    if (rc) return rc;
    // The two totals reach the host through a store into mapped pinned memory, not through a D2H copy: a copy would queue
    // behind whatever the caller has on the device-to-host copy engine (a 97 MB copy of predictions held this 8-byte
    // read-back up for 0.9 ms per step in bench.py's end-to-end loop).
    publish_totals_kernel<<<1, 1, 0, stream>>>(st->d_total, st->d_items + n_cells, st->d_h_totals);
    pl->last_launches += 1;
    int32_t* h_items32 = reinterpret_cast<int32_t*>(&st->h_totals[1]);
    IMAGER_CUDA(cudaStreamSynchronize(stream));
    const int64_t n_hits = st->h_totals[0], n_items = h_items32[0];
    if (n_hits > (int64_t)0x7ffffff0) {              // the 32-bit scan above has wrapped: nothing after this point may use it
        set_error("%lld hits (visibility x strip pairs) in one call exceed the limit of 2^31: feed the visibilities in chunks",
                  (long long)n_hits);
        return IMAGER_ERR_TOO_MANY_VIS;
    }
    const int n_sc = g.n_pol * g.n_corr;
    const int64_t max_blocks = (n_hits / kBlockHits + n_hits / (kTailFrac * (kBlockHits / kTailDiv)) + (int64_t)g.n_gu * (2 * kTailDiv + 4) + 4) * n_sc;
    if (max_blocks > 0x7fffffff) {
        set_error("too many work blocks");
        return IMAGER_ERR_UNSUPPORTED;
    }
    st->blocks_cap = (int32_t)max_blocks;
    rc = grow(&st->d_hit_rec, &st->cap_hits, n_hits + 1);
    if (rc) return rc;
    rc = grow(&st->d_item_rec, &st->cap_items, n_items + 1);
    if (rc) return rc;
    rc = grow(&st->d_blocks, &st->cap_blocks, max_blocks + 1);
    if (rc) return rc;
    rc = grow(&st->d_hit_tmp, &st->cap_tmp, n_hits + 1);
    if (rc) return rc;
    IMAGER_CUDA(cudaMemsetAsync(st->d_cursor, 0, (n_cells + 1) * sizeof(int32_t), stream));
    emit_hits_kernel<<<8 * num_sms(), 256, 0, stream>>>(pa, pl->d_counters, st->d_hits, st->d_cursor, st->d_hit_tmp);
    make_items_kernel<<<8 * num_sms(), 256, 0, stream>>>(g, st->d_hits, st->d_items, st->d_item_rec);
    if (n_items > 0)
        sort_items_kernel<<<(unsigned)((n_items + 7) / 8), 256, 0, stream>>>((int)n_items, st->d_item_rec, st->d_hit_tmp,
                                                                             st->d_hit_rec);
    pl->last_launches += 2;
    IMAGER_CUDA(cudaMemsetAsync(pl->d_counters + 9, 0, sizeof(int32_t), stream));
    IMAGER_CUDA(cudaMemsetAsync(pl->d_counters + 12, 0, sizeof(int32_t), stream));
    plan_blocks_kernel<<<g.n_gu, 128, 0, stream>>>(g, st->d_hits, st->d_items, st->d_item_rec, st->d_blocks, pl->d_counters + 9,
                                                   pl->d_counters + 12, st->blocks_cap);
    pl->last_launches += 2;
    IMAGER_CUDA(cudaGetLastError());
    st->plan_epoch = pl->index_epoch;
    return 0;
}

static void fill_args(imager_plan* pl, TiledState* st, TiledArgs& a, const float2* tab) {
    a.g = st->g;
    a.hit_rec = st->d_hit_rec;
    a.items = st->d_item_rec;
    a.blocks = st->d_blocks;
    a.n_front = pl->d_counters + 9;
    a.n_back = pl->d_counters + 12;
    a.cap_blocks = st->blocks_cap;
    a.queue = pl->d_counters + 8;
    a.tab = tab;
    a.set_offset = pl->d_set_offset;
    a.set_support = pl->d_set_support;
    a.set_plan = st->d_plan;
    a.gu_set = st->d_gu_set;
    a.n_hits = st->h_totals ? st->h_totals[0] : 0;
    a.n_items = st->h_totals ? *reinterpret_cast<int32_t*>(&st->h_totals[1]) : 0;
}

// imager_index_stats: sums over the sorted kept visibilities.  out: [0] sum S^2 of all kept, [1] sum S^2 of those that
// are not merged duplicates, [2] merged duplicates.  sgeo == nullptr (no tiled plan yet): nothing is merged.
__global__ void index_stats_kernel(const int32_t* __restrict__ counters, const int32_t* __restrict__ perm,
                                   const imager_record* __restrict__ rec, const int32_t* __restrict__ set_support,
                                   const uint2* __restrict__ sgeo, unsigned long long* __restrict__ out) {
    const int n_kept = counters[0];
    unsigned long long all = 0, own = 0, merged = 0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_kept; i += gridDim.x * blockDim.x) {
        const unsigned long long S = (unsigned long long)set_support[rec[perm[i]].kset];
        const bool m = sgeo && (sgeo[i].x & kMergedFlag);
        all += S * S;
        own += m ? 0ull : S * S;
        merged += m ? 1ull : 0ull;
    }
    for (int d = 16; d > 0; d >>= 1) {
        all += __shfl_xor_sync(0xffffffffu, all, d);
        own += __shfl_xor_sync(0xffffffffu, own, d);
        merged += __shfl_xor_sync(0xffffffffu, merged, d);
    }
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(out + 0, all);
        atomicAdd(out + 1, own);
        atomicAdd(out + 2, merged);
    }
}

int tiled_index_stats(imager_plan* pl, int64_t out[8], cudaStream_t stream) {
    TiledState* st = pl->tiled ? static_cast<TiledState*>(pl->tiled) : nullptr;
    const bool planned = st && st->initialised && st->plan_epoch == pl->index_epoch;
    unsigned long long* d_out = nullptr;
    IMAGER_CUDA(cudaMalloc(&d_out, 3 * sizeof(unsigned long long)));
    cudaError_t e = cudaMemsetAsync(d_out, 0, 3 * sizeof(unsigned long long), stream);
    unsigned long long h[3] = {0, 0, 0};
    int32_t c[2] = {0, 0};
    if (e == cudaSuccess) {
        index_stats_kernel<<<4 * num_sms(), 256, 0, stream>>>(pl->d_counters, pl->d_perm[pl->sorted_buf], pl->d_rec,
                                                            pl->d_set_support, planned ? st->d_sgeo : nullptr, d_out);
        e = cudaMemcpyAsync(h, d_out, sizeof(h), cudaMemcpyDeviceToHost, stream);
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(c, pl->d_counters, sizeof(c), cudaMemcpyDeviceToHost, stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
    cudaFree(d_out);
    if (e != cudaSuccess) return cuda_fail(e, "imager_index_stats");
    const int64_t n_sc = (int64_t)pl->p.n_corr * pl->p.n_pol;
    out[0] = c[0];
    out[1] = c[1];
    out[2] = (int64_t)h[2];
    out[3] = n_sc * (int64_t)h[0];
    out[4] = n_sc * (int64_t)h[1];
    out[5] = planned ? st->h_totals[0] : 0;
    out[6] = planned ? (int64_t) * reinterpret_cast<int32_t*>(&st->h_totals[1]) : 0;
    out[7] = 0;
    return 0;
}

// hit lists for the current index (imager_index: planning ahead of the first gridding / degridding call)
int tiled_prepare(imager_plan* pl, int64_t nvis, cudaStream_t stream) {
    if (nvis == 0) return 0;
    return prepare(pl, state_of(pl), stream);
}

int launch_grid_tiled(imager_plan* pl, int64_t nvis, const float2* vis, const float* weights, float2* grid,
                      cudaStream_t stream) {
    if (nvis == 0) return 0;
    TiledState* st = state_of(pl);
    int rc = prepare(pl, st, stream);
    if (rc) return rc;
    const unsigned gb = 4 * num_sms();
    if (st->d_rep) {                          // duplicates pre-summed: gather and merge in one pass over the dedupe chunks
        const unsigned chunks = (unsigned)((pl->indexed_nvis + kDedupeChunk - 1) / kDedupeChunk);
        if (pl->p.n_corr == 1)
            gather_merge_values_kernel<1><<<chunks, 1024, kDedupeChunk * 1 * sizeof(float2), stream>>>(
                pl->d_counters, pl->d_perm[pl->sorted_buf], st->d_rep, vis, weights, st->d_sval);
        else
            gather_merge_values_kernel<4><<<chunks, 1024, kDedupeChunk * 4 * sizeof(float2), stream>>>(
                pl->d_counters, pl->d_perm[pl->sorted_buf], st->d_rep, vis, weights, st->d_sval);
    } else if (pl->p.n_corr == 1) {
        gather_values_kernel<1><<<gb, 256, 0, stream>>>(pl->d_counters, pl->d_perm[pl->sorted_buf], vis, weights, st->d_sval);
    } else {
        gather_values_kernel<4><<<gb, 256, 0, stream>>>(pl->d_counters, pl->d_perm[pl->sorted_buf], vis, weights, st->d_sval);
    }
    IMAGER_CUDA(cudaMemsetAsync(pl->d_counters + 8, 0, sizeof(int32_t), stream));
    TiledArgs a;
    fill_args(pl, st, a, pl->d_tab_grid);
    if (pl->p.n_corr == 1)
        grid_tiled_kernel<1><<<num_sms(), kGridThreads, st->smem_bytes + kGridStageBytes, stream>>>(a, st->d_sval, grid);
    else
        grid_tiled_kernel<4><<<num_sms(), kGridThreads, st->smem_bytes + kGridStageBytes, stream>>>(a, st->d_sval, grid);
    pl->last_launches += 2;
    IMAGER_CUDA(cudaGetLastError());
    return 0;
}

int launch_degrid_tiled(imager_plan* pl, int64_t nvis, const float2* grid, float2* vis_out, int residual, cudaStream_t stream) {
    if (nvis == 0) return 0;
    TiledState* st = state_of(pl);
    int rc = prepare(pl, st, stream);
    if (rc) return rc;
    const int nc = pl->p.n_corr;
    IMAGER_CUDA(cudaMemsetAsync(st->d_sval, 0, (size_t)nvis * nc * sizeof(float2), stream));
    IMAGER_CUDA(cudaMemsetAsync(pl->d_counters + 8, 0, sizeof(int32_t), stream));
    TiledArgs a;
    fill_args(pl, st, a, pl->d_tab_degrid);
    const int smem = st->smem_bytes + kStageBytes + kRedBytes;
    const unsigned gb = 4 * num_sms();
    if (nc == 1) {
        degrid_tiled_kernel<1><<<num_sms(), kTiledThreads, smem, stream>>>(a, grid, st->d_sval);
        scatter_values_kernel<1><<<gb, 256, 0, stream>>>(nvis, pl->d_counters, pl->d_perm[pl->sorted_buf], st->d_rep, st->d_sval, residual, vis_out);
    } else {
        degrid_tiled_kernel<4><<<num_sms(), kTiledThreads, smem, stream>>>(a, grid, st->d_sval);
        scatter_values_kernel<4><<<gb, 256, 0, stream>>>(nvis, pl->d_counters, pl->d_perm[pl->sorted_buf], st->d_rep, st->d_sval, residual, vis_out);
    }
    pl->last_launches += 2;
    IMAGER_CUDA(cudaGetLastError());
    return 0;
}

}  // namespace imager

extern "C" int imager_debug_violations(int64_t out[16]) {
    if (!out) return IMAGER_ERR_INVALID_ARG;
    unsigned long long h[16] = {0};
    cudaError_t e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaMemcpyFromSymbol(h, imager::g_violations, sizeof(h));
    if (e != cudaSuccess) return imager::cuda_fail(e, "imager_debug_violations");
    for (int k = 0; k < 16; ++k) out[k] = (int64_t)h[k];
    return IMAGER_CHECKED ? 1 : 0;
}
