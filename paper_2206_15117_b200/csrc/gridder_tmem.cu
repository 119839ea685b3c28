// gridder_tmem.cu -- gridding / degridding with the kernel taps in TENSOR MEMORY (hot-path steps A3 / A6) and the
// planner that feeds them.  DESIGN.md section 6.3.
//
// Why (profiles/r1_port_probe.md): one complex MAC needs one private 8-byte tap per lane.  Shared memory (and L1,
// and the texture path: one port) delivers 16 taps/clk/SM = half of what the FP32 pipe consumes; tcgen05.ld delivers
// 32 taps/clk/SM from TMEM, concurrently with shared memory.  TMEM's restriction is that lane i of a warp reads only
// TMEM lane 32 (warp % 4) + i at a warp-uniform column.  So the lane <-> tap relation is made FIXED:
//   lane (lx, ly) handles the taps (ty, tx) of any footprint with  ty = ly + 4 J,  tx = lx + 8 I,
// i.e. the 8 x 4 lane block is aligned to the FOOTPRINT (origin fx = gx - S/2, fy = gy - S/2), not to the grid, and
// the lane's TMEM row holds R[slice][I][J] = T[slice][ly + 4 J][lx + 8 I] (zero beyond S): column 2 ((sl EI + I) EJ + J).
// The cells a lane owns then depend on the visibility's alignment class a = (fx mod 8, fy mod 4): 32 classes, each
// with its own strip lattice, shifted by (ax, ay) against the grid.  A warp accumulates a 16 x 32 strip of ONE class
// in registers over a RUN of hits (same class, same strip), adds it into a private shared-memory tile of its 32 x 32
// region (39 x 35 cells with the shifts; plain load-add-store: the tile is private to the warp) when the run ends,
// and adds the tile to the grid with red.global.add.v2.f32 once per work item.  No lane is spent on a footprint edge
// (only on rounding S up to multiples of 8 and 4), the FP32 pipe and the TMEM port are the co-binding units, and the
// shared-memory port carries only the run flushes and one descriptor load per hit.
//
// Work planning: geometry unit gu = (kernel set, group of sub-cell slices that fit one lane's 240 TMEM taps);
// cell = (gu, 32 x 32 region); hits of a cell are sorted by run key (class, strip); item = up to kItemHits
// consecutive hits of a cell; block = consecutive items of a gu with about kBlockHits hits, times one Mueller element.
// Persistent CTAs pull blocks from a global queue (loading the gu's tables into TMEM when it changes), their 16
// warps pull items from a shared counter.
#include "common.cuh"

namespace imager {

namespace tm {

constexpr int kLaneW = 8, kLaneH = 4;
constexpr int kStripW = 16, kStripH = 32, kNY = 8;
constexpr int kRegion = 32;                            // = kBucketTile
constexpr int kThreads = 512, kWarps = kThreads / 32;
constexpr int kTmemTaps = 240;                         // taps per lane (480 of the 512 columns; 16 taps of read slack)
constexpr int kItemHits = 512;
constexpr int kBlockHits = 65536;
constexpr int kTileRows = kRegion + kLaneH - 1;        // 35
constexpr int kTileCols = kRegion + kLaneW - 1;        // 39
constexpr int kTilePitch = 40;                         // cells; = 8 mod 16: an 8 x 4 lane block is conflict-free
constexpr int kTileBytes = kTileRows * kTilePitch * 8; // 11200
constexpr int kStageBytes = kWarps * 32 * 8;
constexpr int kSmemBytes = kStageBytes + kWarps * kTileBytes;   // 187,392
constexpr int64_t kMaxPlanCells = 48 << 20;

static_assert(kRegion == kBucketTile, "regions are the bucketing tiles");

struct SetPlan {           // per kernel set (host-built)
    int32_t EI, EJ;        // footprint blocks: ceil(S / 8), ceil(S / 4)
    int32_t group_slices;  // sub-cell slices resident at once
    int32_t n_groups;
    int32_t gu_base;
    int32_t pad[3];
};

struct Item { int32_t region, hit_begin, hit_count, gu; };
struct Block { int32_t gu, sc, item_begin, item_count; };

struct Geometry {
    int N, O, nt, n_regions, n_sets, n_gu, n_pol, n_corr;
};

// hit record: .x = sorted index of the visibility,
// .y = tap index of the first tap (8 bits) | jl << 8 | (jh - 1) << 11 | halves << 14 | run key << 16 (class * 2 + strip)
__device__ __forceinline__ uint32_t pack_ctrl(int tap, int jl, int jh, int halves, int run) {
    return (uint32_t)tap | ((uint32_t)jl << 8) | ((uint32_t)(jh - 1) << 11) | ((uint32_t)halves << 14) | ((uint32_t)run << 16);
}

struct PlanArgs {
    Geometry g;
    const SetPlan* set_plan;
    const int32_t* gu_set;
    const int32_t* set_support;
    const int32_t* bucket_offset;
    const uint2* sgeo;
};

// ctrl word of candidate (gx, gy, sub) against strip `st` of region (rx, ry) for its own class, or 0xffffffff if no hit
__device__ __forceinline__ uint32_t hit_ctrl(int gx, int gy, int subl, int S, const SetPlan& sp, int rx, int ry, int st) {
    const int h_lo = S >> 1;
    const int fx = gx - h_lo, fy = gy - h_lo;                 // >= 0 for kept visibilities
    const int ax = fx & 7, ay = fy & 3;
    const int H = sp.EJ * 4;
    const int Y0 = ry * kRegion + ay, X0 = rx * kRegion + ax + st * kStripW;
    const int jl = max(0, (fy - Y0) >> 2);                    // exact: fy - Y0 is a multiple of 4
    const int jh = min(kNY, (fy + H - Y0) >> 2);
    const int I0 = (X0 - fx) >> 3;                            // exact: multiple of 8; may be negative
    const int h0 = (I0 >= 0 && I0 < sp.EI) ? 1 : 0, h1 = (I0 + 1 >= 0 && I0 + 1 < sp.EI) ? 2 : 0;
    if (jl >= jh || (h0 | h1) == 0 || (unsigned)subl >= (unsigned)sp.group_slices) return 0xffffffffu;
    const int J0 = (Y0 + 4 * jl - fy) >> 2;
    const int tap = (subl * sp.EI + (h0 ? I0 : I0 + 1)) * sp.EJ + J0;
    return pack_ctrl(tap, jl, jh, h0 | h1, (ax + 8 * ay) * 2 + st);
}

// candidate buckets of (kset, region): those whose visibilities' padded footprints can reach the region's strips
__device__ __forceinline__ void region_buckets(const Geometry& g, int rx, int ry, int S, const SetPlan& sp, int& bx_lo,
                                               int& bx_hi, int& by_lo, int& by_hi) {
    const int h_lo = S >> 1, W = sp.EI * 8, H = sp.EJ * 4;
    // hit needs fx + W > 32 rx and fx < 32 rx + 39  (fx = gx - h_lo), same in y with H and 35
    bx_lo = max(0, rx * kRegion + h_lo - W + 1) / kRegion;
    bx_hi = min(g.nt - 1, (rx * kRegion + kTileCols - 1 + h_lo) / kRegion);
    by_lo = max(0, ry * kRegion + h_lo - H + 1) / kRegion;
    by_hi = min(g.nt - 1, (ry * kRegion + kTileRows - 1 + h_lo) / kRegion);
}

// sort bin of a hit within its cell: run key major (64), slot range (jl, jh - 1) minor (36): hits of a run that share
// a slot range are replayed by one pass through the same straight-line code
constexpr int kPlanWarps = 4, kPlanBins = 64 * 36, kBinsPerLane = kPlanBins / 32;
__device__ __forceinline__ uint32_t hit_bin(uint32_t ctrl) {
    const uint32_t jl = (ctrl >> 8) & 7u, jh1 = (ctrl >> 11) & 7u;
    return (ctrl >> 16) * 36u + (jl * 8u - (jl * (jl - 1u)) / 2u + jh1 - jl);
}

// MODE 0: count hits / items of every cell; MODE 1: write the hit records sorted by bin (stable) and the items.
// One warp per cell (gu, region).
template <int MODE>
__global__ void __launch_bounds__(kPlanWarps * 32) plan_hits_kernel(const PlanArgs a, int32_t* __restrict__ hits,
                                                                    int32_t* __restrict__ items, uint2* __restrict__ hit_rec,
                                                                    Item* __restrict__ item_rec) {
    __shared__ int32_t s_bin[MODE ? kPlanWarps : 1][MODE ? kPlanBins : 1];
    const Geometry& g = a.g;
    const int64_t cell = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t n_cells = (int64_t)g.n_gu * g.n_regions;
    const int lane = threadIdx.x & 31, warp = (threadIdx.x >> 5) % kPlanWarps;
    if (cell > n_cells) return;
    if (cell == n_cells) {
        if (MODE == 0 && lane == 0) hits[cell] = items[cell] = 0;
        return;
    }
    const int gu = (int)(cell / g.n_regions), region = (int)(cell - (int64_t)gu * g.n_regions);
    const int ry = region / g.nt, rx = region - ry * g.nt;
    const int kset = a.gu_set[gu];
    const SetPlan sp = a.set_plan[kset];
    const int S = a.set_support[kset];
    const int sub_lo = (gu - sp.gu_base) * sp.group_slices;
    int bx_lo, bx_hi, by_lo, by_hi;
    region_buckets(g, rx, ry, S, sp, bx_lo, bx_hi, by_lo, by_hi);
    int out = 0;
    if (MODE == 1) {
        out = hits[cell];
        const int n_hits = hits[cell + 1] - out;
        if (n_hits == 0) return;
        const int i0 = items[cell], n_items = items[cell + 1] - i0;
        for (int p = lane; p < n_items; p += 32)
            item_rec[i0 + p] = Item{region, out + p * kItemHits, min(kItemHits, n_hits - p * kItemHits), gu};
        for (int v = lane; v < kPlanBins; v += 32) s_bin[warp][v] = 0;
        __syncwarp();
    }
    const unsigned lt_mask = (1u << lane) - 1u;
    int count = 0;
    for (int pass = 0; pass <= MODE; ++pass) {
        if (MODE == 1 && pass == 1) {                        // exclusive prefix of the bins, kBinsPerLane per lane
            __syncwarp();
            int t = 0;
            for (int q = 0; q < kBinsPerLane; ++q) t += s_bin[warp][kBinsPerLane * lane + q];
            int inc = t;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, inc, d);
                if (lane >= d) inc += y;
            }
            int run = inc - t;
            for (int q = 0; q < kBinsPerLane; ++q) {
                const int c = s_bin[warp][kBinsPerLane * lane + q];
                s_bin[warp][kBinsPerLane * lane + q] = run;
                run += c;
            }
            __syncwarp();
        }
        for (int by = by_lo; by <= by_hi; ++by) {
            const int b0 = (kset * g.nt + by) * g.nt;
            const int r0 = a.bucket_offset[b0 + bx_lo], r1 = a.bucket_offset[b0 + bx_hi + 1];
            for (int i0 = r0; i0 < r1; i0 += 32) {
                const int idx = i0 + lane;
                uint32_t ctrl[2] = {0xffffffffu, 0xffffffffu};
                if (idx < r1) {
                    const uint2 geo = a.sgeo[idx];
                    const int gx = (int)(geo.x & 0xffffu), gy = (int)(geo.x >> 16), subl = (int)geo.y - sub_lo;
                    ctrl[0] = hit_ctrl(gx, gy, subl, S, sp, rx, ry, 0);
                    ctrl[1] = hit_ctrl(gx, gy, subl, S, sp, rx, ry, 1);
                }
#pragma unroll
                for (int st = 0; st < 2; ++st) {
                    const bool hit = ctrl[st] != 0xffffffffu;
                    const unsigned m = __ballot_sync(0xffffffffu, hit);
                    if (MODE == 0) {
                        count += __popc(m);
                    } else if (m) {
                        const uint32_t bin = hit ? hit_bin(ctrl[st]) : (uint32_t)(kPlanBins + lane);   // misses match nobody
                        if (pass == 0) {
                            if (hit) atomicAdd(&s_bin[warp][bin], 1);
                        } else {
                            const unsigned peers = __match_any_sync(0xffffffffu, bin);
                            const int leader = __ffs(peers) - 1, rank = __popc(peers & lt_mask);
                            int base = 0;
                            if (lane == leader && hit) {
                                base = s_bin[warp][bin];
                                s_bin[warp][bin] = base + __popc(peers);
                            }
                            base = __shfl_sync(0xffffffffu, base, leader);
                            if (hit) hit_rec[out + base + rank] = make_uint2((uint32_t)idx, ctrl[st]);
                            __syncwarp();
                        }
                    }
                }
            }
        }
    }
    if (MODE == 0 && lane == 0) {
        hits[cell] = count;
        items[cell] = (count + kItemHits - 1) / kItemHits;
    }
}

// one thread block per geometry unit: blocks of about kBlockHits hits (whole items), one copy per Mueller element
__global__ void plan_blocks_kernel(const Geometry g, const int32_t* __restrict__ hit_start, const int32_t* __restrict__ item_start,
                                   const Item* __restrict__ item_rec, Block* __restrict__ blocks, int32_t* __restrict__ n_blocks,
                                   int max_blocks) {
    __shared__ int s_base;
    const int gu = blockIdx.x;
    const int n_sc = g.n_pol * g.n_corr;
    const int64_t c0 = (int64_t)gu * g.n_regions, c1 = c0 + g.n_regions;
    const int h0 = hit_start[c0], h1 = hit_start[c1], i0 = item_start[c0], i1 = item_start[c1];
    if (h1 == h0) return;
    const int nb = (h1 - h0 + kBlockHits - 1) / kBlockHits;
    if (threadIdx.x == 0) s_base = atomicAdd(n_blocks, nb * n_sc);
    __syncthreads();
    const int base = s_base;
    if (base + nb * n_sc > max_blocks) return;                    // cannot happen: max_blocks is an upper bound
    for (int b = threadIdx.x; b < nb; b += blockDim.x) {
        // items [first, last): hit_begin in [h0 + b K, h0 + (b + 1) K)
        int bounds[2];
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int64_t limit = (int64_t)h0 + (int64_t)(b + e) * kBlockHits;
            int lo = i0, hi = i1;
            while (lo < hi) {
                const int mid = (lo + hi) >> 1;
                if (item_rec[mid].hit_begin < limit) lo = mid + 1; else hi = mid;
            }
            bounds[e] = lo;
        }
        if (b == nb - 1) bounds[1] = i1;
        for (int sc = 0; sc < n_sc; ++sc) blocks[base + sc * nb + b] = Block{gu, sc, bounds[0], bounds[1] - bounds[0]};
    }
}


// ---- device helpers --------------------------------------------------------------------------------------
struct TmArgs {
    Geometry g;
    const uint2* hit_rec;
    const Item* items;
    const Block* blocks;
    const int32_t* n_blocks;
    int32_t* queue;
    const float2* tab;
    const int64_t* set_offset;
    const int32_t* set_support;
    const SetPlan* set_plan;
    const int32_t* gu_set;
};

typedef unsigned long long u64;

// d += (tap.re, tap.im) * (v, v) with the tap given as the two 32-bit registers tcgen05.ld wrote
__device__ __forceinline__ void ffma2_tap(u64& d, uint32_t t_re, uint32_t t_im, u64 v) {
    asm("{\n\t.reg .b64 t;\n\tmov.b64 t, {%1, %2};\n\tfma.rn.f32x2 %0, t, %3, %0;\n\t}" : "+l"(d) : "r"(t_re), "r"(t_im), "l"(v));
}

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

__device__ __forceinline__ float2 lds64(uint32_t addr) {
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
    return v;
}

__device__ __forceinline__ uint4 lds128(uint32_t addr) {
    uint4 d;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(d.x), "=r"(d.y), "=r"(d.z), "=r"(d.w) : "r"(addr));
    return d;
}

__device__ __forceinline__ void sts64(uint32_t addr, float2 v) {
    asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(addr), "f"(v.x), "f"(v.y) : "memory");
}

// tcgen05.ld.32x32b: every lane reads consecutive 32-bit columns of ITS OWN TMEM lane, starting at a warp-uniform column
__device__ __forceinline__ void ldtm2(uint32_t* t, uint32_t taddr) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(t[0]), "=r"(t[1]) : "r"(taddr));
}
__device__ __forceinline__ void ldtm4(uint32_t* t, uint32_t taddr) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(t[0]), "=r"(t[1]), "=r"(t[2]), "=r"(t[3]) : "r"(taddr));
}
__device__ __forceinline__ void ldtm8(uint32_t* t, uint32_t taddr) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(t[0]), "=r"(t[1]), "=r"(t[2]), "=r"(t[3]), "=r"(t[4]), "=r"(t[5]), "=r"(t[6]), "=r"(t[7]) : "r"(taddr));
}
__device__ __forceinline__ void ldtm16(uint32_t* t, uint32_t taddr) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                 : "=r"(t[0]), "=r"(t[1]), "=r"(t[2]), "=r"(t[3]), "=r"(t[4]), "=r"(t[5]), "=r"(t[6]), "=r"(t[7]), "=r"(t[8]),
                   "=r"(t[9]), "=r"(t[10]), "=r"(t[11]), "=r"(t[12]), "=r"(t[13]), "=r"(t[14]), "=r"(t[15])
                 : "r"(taddr));
}

// NT taps (2 NT columns) into t[0 .. 2 NT): exact sizes, so that no TMEM bandwidth is spent on taps nobody uses
template <int NT>
__device__ __forceinline__ void load_taps(uint32_t (&t)[16], uint32_t taddr) {
    if (NT == 8) {
        ldtm16(t, taddr);
    } else {
        int o = 0;
        if (NT & 4) { ldtm8(t + o, taddr + o); o += 8; }
        if (NT & 2) { ldtm4(t + o, taddr + o); o += 4; }
        if (NT & 1) { ldtm2(t + o, taddr + o); }
    }
}

// wait for the loads, and make every later use of t depend on the wait
__device__ __forceinline__ void wait_taps(uint32_t (&t)[16]) {
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+r"(t[0]), "+r"(t[1]), "+r"(t[2]), "+r"(t[3]), "+r"(t[4]), "+r"(t[5]), "+r"(t[6]), "+r"(t[7]), "+r"(t[8]),
                   "+r"(t[9]), "+r"(t[10]), "+r"(t[11]), "+r"(t[12]), "+r"(t[13]), "+r"(t[14]), "+r"(t[15])
                 :: "memory");
}
__device__ __forceinline__ void touch_taps(uint32_t (&t)[16]) {
    asm volatile("" : "+r"(t[0]), "+r"(t[1]), "+r"(t[2]), "+r"(t[3]), "+r"(t[4]), "+r"(t[5]), "+r"(t[6]), "+r"(t[7]), "+r"(t[8]),
                      "+r"(t[9]), "+r"(t[10]), "+r"(t[11]), "+r"(t[12]), "+r"(t[13]), "+r"(t[14]), "+r"(t[15])
                 :: "memory");
}

// one geometry unit's tables for Mueller element sc -> TMEM.  All 16 warps: warp w fills quarter (w >> 2) of the
// entries of quadrant (w & 3) (the four quadrants hold the same data: a warp can only read its own quadrant).
__device__ void load_tables_tmem(const TmArgs& a, int kset, int group, int sc, const SetPlan sp, int S, uint32_t tmem_base) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, lx = lane & 7, ly = lane >> 3;
    const int OO = a.g.O * a.g.O, E = sp.EI * sp.EJ, n = sp.group_slices * E;
    const float2* T = a.tab + a.set_offset[kset] + ((int64_t)sc * OO + (int64_t)group * sp.group_slices) * S * S;
    const int chunk = (n + 3) >> 2, e0 = (warp >> 2) * chunk, e1 = min(n, e0 + chunk);
    const uint32_t row = tmem_base + ((uint32_t)((warp & 3) * 32) << 16);
    for (int e = e0; e < e1; ++e) {
        const int sl = e / E, rem = e - sl * E, I = rem / sp.EJ, J = rem - I * sp.EJ;
        const int ty = ly + 4 * J, tx = lx + 8 * I;
        float2 v = make_float2(0.f, 0.f);
        if (ty < S && tx < S) v = __ldg(&T[((int64_t)sl * S + ty) * S + tx]);
        asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(row + 2 * e), "r"(__float_as_uint(v.x)),
                     "r"(__float_as_uint(v.y)) : "memory");
    }
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}

// variant number of a slot range (jl, jh - 1): 1 .. 36 (0 is "no hit")
#define TM_V36(JL, JH1) (1 + (JL) * 8 - ((JL) * ((JL) - 1)) / 2 + (JH1) - (JL))

// control word of a hit, built once per batch by the lane that holds the hit and broadcast with REDUX (so that it is
// warp-uniform for the compiler): variant [5:0] | halves [7:6] | run key [14:8] | tap index [23:16]
__device__ __forceinline__ uint32_t control_word(uint32_t ctrl) {
    const int jl = (int)((ctrl >> 8) & 7u), jh1 = (int)((ctrl >> 11) & 7u);
    return (uint32_t)TM_V36(jl, jh1) | (((ctrl >> 14) & 3u) << 6) | ((ctrl >> 16) << 8) | ((ctrl & 255u) << 16);
}
constexpr uint32_t kKeyMask = 0x7f3fu;                 // variant + run key
constexpr uint32_t kEndWord = 37u | (64u << 8);        // terminator: a run key no hit has, a variant with no body

#define TM_CASE(FN, JL, JH1) \
    case TM_V36(JL, JH1): FN<JL, (JH1) + 1> TM_BODY_ARGS; break;
#define TM_DISPATCH(FN, variant)                                                                     \
    switch (variant) {                                                                               \
        TM_CASE(FN, 0, 0) TM_CASE(FN, 0, 1) TM_CASE(FN, 0, 2) TM_CASE(FN, 0, 3)                      \
        TM_CASE(FN, 0, 4) TM_CASE(FN, 0, 5) TM_CASE(FN, 0, 6) TM_CASE(FN, 0, 7)                      \
        TM_CASE(FN, 1, 1) TM_CASE(FN, 1, 2) TM_CASE(FN, 1, 3) TM_CASE(FN, 1, 4)                      \
        TM_CASE(FN, 1, 5) TM_CASE(FN, 1, 6) TM_CASE(FN, 1, 7)                                        \
        TM_CASE(FN, 2, 2) TM_CASE(FN, 2, 3) TM_CASE(FN, 2, 4) TM_CASE(FN, 2, 5)                      \
        TM_CASE(FN, 2, 6) TM_CASE(FN, 2, 7)                                                          \
        TM_CASE(FN, 3, 3) TM_CASE(FN, 3, 4) TM_CASE(FN, 3, 5) TM_CASE(FN, 3, 6) TM_CASE(FN, 3, 7)    \
        TM_CASE(FN, 4, 4) TM_CASE(FN, 4, 5) TM_CASE(FN, 4, 6) TM_CASE(FN, 4, 7)                      \
        TM_CASE(FN, 5, 5) TM_CASE(FN, 5, 6) TM_CASE(FN, 5, 7)                                        \
        TM_CASE(FN, 6, 6) TM_CASE(FN, 6, 7)                                                          \
        TM_CASE(FN, 7, 7)                                                                            \
        default: w = 0u; break;                                                                      \
    }

// ---- gridding --------------------------------------------------------------------------------------------
// Loop state of a warp replaying one batch of staged hits.
struct Replay {
    uint32_t w;          // control word of the current hit (warp-uniform; 0 past the end of the batch)
    uint32_t my_w;       // control word of the hit this lane staged
    uint32_t saddr;      // shared address of the current hit's value
    uint32_t touched;    // slots of the register strip written in the current run (bits 0-7 half 0, 8-15 half 1)
    int h;               // index of the current hit in the batch
};

// A sub-run: consecutive hits with the same run key and the same slot range JL .. JH-1.  Per hit: the taps of the
// x-halves it meets from TMEM (exact sizes), then A += t * (vr, vr), B += t * (vi, vi)
// (re = A.x - B.y, im = A.y + B.x when the run is flushed).
template <int JL, int JH>
__device__ __forceinline__ void grid_subrun(u64 (&A0)[kNY], u64 (&B0)[kNY], u64 (&A1)[kNY], u64 (&B1)[kNY], Replay& r,
                                            const uint32_t tmem_row, const uint32_t ej2, const int lane) {
    constexpr int NT = JH - JL;
    constexpr uint32_t kRows = (1u << JH) - (1u << JL);
    const uint32_t key = r.w & kKeyMask;
    uint32_t w = r.w, saddr = r.saddr, touched = r.touched;
    int h = r.h;
#pragma unroll 1
    do {
        const float2 v = lds64(saddr);
        const uint32_t taddr = tmem_row + ((w >> 15) & 0x1feu);
        const bool half0 = (w & 0x40u) != 0u, half1 = (w & 0x80u) != 0u;
        // both halves are always fetched (a half the hit does not meet yields taps nobody uses): no control flow
        // around the loads
        uint32_t t0[16], t1[16];
        load_taps<NT>(t0, taddr);
        load_taps<NT>(t1, half0 ? taddr + ej2 : taddr);
        saddr += 8;
        ++h;
        w = __reduce_or_sync(0xffffffffu, lane == h ? r.my_w : 0u);              // the next hit
        wait_taps(t0);
        touch_taps(t1);
        const u64 vrr = pack2(v.x, v.x), vii = pack2(v.y, v.y);
        if (half0) {
#pragma unroll
            for (int q = 0; q < NT; ++q) {
                ffma2_tap(A0[JL + q], t0[2 * q], t0[2 * q + 1], vrr);
                ffma2_tap(B0[JL + q], t0[2 * q], t0[2 * q + 1], vii);
            }
            touched |= kRows;
        }
        if (half1) {
#pragma unroll
            for (int q = 0; q < NT; ++q) {
                ffma2_tap(A1[JL + q], t1[2 * q], t1[2 * q + 1], vrr);
                ffma2_tap(B1[JL + q], t1[2 * q], t1[2 * q + 1], vii);
            }
            touched |= kRows << 8;
        }
    } while ((w & kKeyMask) == key);
    r.w = w;
    r.saddr = saddr;
    r.touched = touched;
    r.h = h;
}

// add the touched slots of the register strip into the warp's private tile and clear them
__device__ __forceinline__ void flush_run(u64 (&A0)[kNY], u64 (&B0)[kNY], u64 (&A1)[kNY], u64 (&B1)[kNY], uint32_t touched,
                                          uint32_t base) {
#pragma unroll
    for (int j = 0; j < kNY; ++j) {
        if (touched & (1u << j)) {
            const float2 a = unpack2(A0[j]), b = unpack2(B0[j]);
            const uint32_t addr = base + (uint32_t)(j * kLaneH * kTilePitch * 8);
            float2 p = lds64(addr);
            p.x += a.x - b.y;
            p.y += a.y + b.x;
            sts64(addr, p);
            A0[j] = B0[j] = 0ull;
        }
        if (touched & (0x100u << j)) {
            const float2 a = unpack2(A1[j]), b = unpack2(B1[j]);
            const uint32_t addr = base + (uint32_t)(j * kLaneH * kTilePitch * 8 + kLaneW * 8);
            float2 p = lds64(addr);
            p.x += a.x - b.y;
            p.y += a.y + b.x;
            sts64(addr, p);
            A1[j] = B1[j] = 0ull;
        }
    }
}

// byte offset, within a tile, of the strip-origin cell of this lane for run key `run` (class * 2 + strip)
__device__ __forceinline__ uint32_t run_tile_offset(uint32_t run, int lx, int ly) {
    const uint32_t st = run & 1u, ax = (run >> 1) & 7u, ay = run >> 4;
    return ((ay + ly) * kTilePitch + ax + st * kStripW + lx) * 8u;
}

__device__ __forceinline__ uint32_t tmem_alloc_all(uint32_t* slot) {
    if ((threadIdx.x >> 5) == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"((uint32_t)__cvta_generic_to_shared(slot)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    return *slot;
}

__device__ __forceinline__ void tmem_free_all(uint32_t base) {
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if ((threadIdx.x >> 5) == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(base) : "memory");
}

template <int NC>
__global__ void __launch_bounds__(kThreads, 1)
grid_tmem_kernel(const TmArgs a, const float2* __restrict__ sval, float2* __restrict__ grid) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ int s_block, s_next;
    __shared__ uint32_t s_tmem;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, lx = lane & (kLaneW - 1), ly = lane >> 3;
    float2* stage = reinterpret_cast<float2*>(smem_raw + warp * 32 * 8);
    float2* tile = reinterpret_cast<float2*>(smem_raw + kStageBytes + warp * kTileBytes);
    const uint32_t stage_addr = (uint32_t)__cvta_generic_to_shared(stage);
    const uint32_t tile_addr = (uint32_t)__cvta_generic_to_shared(tile);
    const uint32_t tmem_base = tmem_alloc_all(&s_tmem);
    const uint32_t tmem_row = __reduce_or_sync(0xffffffffu, tmem_base + ((uint32_t)((warp & 3) * 32) << 16));
    for (int i = lane; i < kTileRows * kTilePitch; i += 32) tile[i] = make_float2(0.f, 0.f);
    __syncwarp();
    const Geometry g = a.g;
    const int n_blocks = *a.n_blocks;
    int cur_gu = -1, cur_sc = -1;
    for (;;) {
        __syncthreads();                                   // everyone is done with the previous block (and its tables)
        if (threadIdx.x == 0) {
            s_block = atomicAdd(a.queue, 1);
            s_next = 0;
        }
        __syncthreads();
        if (s_block >= n_blocks) break;
        const Block blk = a.blocks[s_block];
        const int kset = a.gu_set[blk.gu];
        const SetPlan sp = a.set_plan[kset];
        if (blk.gu != cur_gu || blk.sc != cur_sc) {
            load_tables_tmem(a, kset, blk.gu - sp.gu_base, blk.sc, sp, a.set_support[kset], tmem_base);
            cur_gu = blk.gu;
            cur_sc = blk.sc;
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncthreads();
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        }
        const int s_pol = blk.sc / g.n_corr, c_corr = blk.sc - s_pol * g.n_corr;
        float2* gplane = grid + (int64_t)s_pol * g.N * g.N;
        const uint32_t ej2 = __reduce_or_sync(0xffffffffu, (uint32_t)(2 * sp.EJ));
        for (;;) {
            int ii = 0;
            if (lane == 0) ii = atomicAdd(&s_next, 1);
            ii = __shfl_sync(0xffffffffu, ii, 0);
            if (ii >= blk.item_count) break;
            const Item it = a.items[blk.item_begin + ii];
            u64 A0[kNY], B0[kNY], A1[kNY], B1[kNY];
#pragma unroll
            for (int j = 0; j < kNY; ++j) A0[j] = B0[j] = A1[j] = B1[j] = 0ull;
            uint32_t cur_run = 64u;
            Replay r;
            r.touched = 0u;
            uint2 rec = make_uint2(0u, 0u), rec1 = make_uint2(0u, 0u);
            float2 val = make_float2(0.f, 0.f);
            if (lane < it.hit_count) rec = a.hit_rec[it.hit_begin + lane];
            if (lane + 32 < it.hit_count) rec1 = a.hit_rec[it.hit_begin + 32 + lane];
            if (lane < it.hit_count) val = sval[(int64_t)rec.x * NC + c_corr];
            // batches of 32 hits, then one batch holding only the terminator (it flushes the last run)
            for (int b0 = 0; b0 < it.hit_count + 32; b0 += 32) {
                const int n = min(32, it.hit_count - b0);
                r.my_w = lane < n ? control_word(rec.y) : ((n <= 0 && lane == 0) ? kEndWord : 0u);
                stage[lane] = val;
                rec = rec1;
                if (b0 + 32 + lane < it.hit_count) val = sval[(int64_t)rec.x * NC + c_corr];
                if (b0 + 64 + lane < it.hit_count) rec1 = a.hit_rec[it.hit_begin + b0 + 64 + lane];
                __syncwarp();
                r.h = 0;
                r.saddr = stage_addr;
                r.w = __reduce_or_sync(0xffffffffu, lane == 0 ? r.my_w : 0u);
#pragma unroll 1
                while (r.w != 0u) {
                    const uint32_t run = (r.w >> 8) & 0x7fu;
                    if (run != cur_run) {
                        if (r.touched) {
                            flush_run(A0, B0, A1, B1, r.touched, tile_addr + run_tile_offset(cur_run, lx, ly));
                            __syncwarp();
                        }
                        cur_run = run;
                        r.touched = 0u;
                    }
                    uint32_t& w = r.w;
#define TM_BODY_ARGS (A0, B0, A1, B1, r, tmem_row, ej2, lane)
                    TM_DISPATCH(grid_subrun, r.w & 0x3fu)
#undef TM_BODY_ARGS
                }
                __syncwarp();
            }
            // the tile -> the grid (cells inside the grid, non-zero values only); the tile is left zeroed
            const int ry = it.region / g.nt, rx = it.region - ry * g.nt;
            int row = 0, col = lane;
            for (int i = lane; i < kTileRows * kTilePitch; i += 32) {
                const float2 p = tile[i];
                if (p.x != 0.f || p.y != 0.f) {
                    tile[i] = make_float2(0.f, 0.f);
                    const int gy = ry * kRegion + row, gx = rx * kRegion + col;
                    if (gx < g.N && gy < g.N) atomicAdd(gplane + (int64_t)gy * g.N + gx, p);
                }
                col += 32;
                if (col >= kTilePitch) {
                    col -= kTilePitch;
                    ++row;
                }
            }
            __syncwarp();
        }
    }
    tmem_free_all(tmem_base);
}

// ---- small streaming kernels (sorted-order copies of the per-visibility data) ------------------------------
__global__ void sorted_geo_kernel(const int32_t* __restrict__ counters, const int32_t* __restrict__ perm,
                                  const imager_record* __restrict__ rec, int O, uint2* __restrict__ sgeo) {
    const int n_kept = counters[0];
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_kept; i += gridDim.x * blockDim.x) {
        const imager_record r = rec[perm[i]];
        sgeo[i] = make_uint2((uint32_t)r.gx | ((uint32_t)r.gy << 16), ((r.sub >> 8) & 255u) * O + (r.sub & 255u));
    }
}

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

template <int NC>
__global__ void scatter_values_kernel(int64_t nvis, const int32_t* __restrict__ counters, const int32_t* __restrict__ perm,
                                      const float2* __restrict__ sval, float2* __restrict__ vis_out) {
    const int n_kept = counters[0];
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvis; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t k = perm[i];
#pragma unroll
        for (int c = 0; c < NC; ++c) vis_out[k * NC + c] = i < n_kept ? sval[i * NC + c] : make_float2(0.f, 0.f);
    }
}

// ---- host side -------------------------------------------------------------------------------------------
struct TmState {
    std::vector<SetPlan> plan;
    std::vector<int32_t> gu_set;
    SetPlan* d_plan = nullptr;
    int32_t* d_gu_set = nullptr;
    int32_t* d_hits = nullptr;            // [n_cells + 1] -> scanned into hit starts
    int32_t* d_items = nullptr;           // [n_cells + 1] -> scanned into item starts
    int32_t* d_scan_tmp = nullptr;
    uint2* d_hit_rec = nullptr;
    Item* d_item_rec = nullptr;
    Block* d_blocks = nullptr;
    int64_t cap_hits = 0, cap_items = 0, cap_blocks = 0;
    int32_t* h_totals = nullptr;          // pinned [2]
    uint2* d_sgeo = nullptr;
    float2* d_sval = nullptr;
    int64_t plan_epoch = -1;
    Geometry g;
};

static int slices_per_group(int S, int OO, int& EI, int& EJ) {
    EI = (S + kLaneW - 1) / kLaneW;
    EJ = (S + kLaneH - 1) / kLaneH;
    const int E = EI * EJ;
    if (E > kTmemTaps) return 0;
    int gs = 1;
    while (gs * 2 <= OO && OO % (gs * 2) == 0 && gs * 2 * E <= kTmemTaps) gs *= 2;
    return gs;
}

}  // namespace tm

bool tmem_supported(const imager_plan* pl) {
    const imager_params& p = pl->p;
    if (p.grid_size % tm::kRegion != 0 || p.grid_size > 32768) return false;
    const int OO = p.oversample * p.oversample;
    const int64_t n_regions = (int64_t)(p.grid_size / tm::kRegion) * (p.grid_size / tm::kRegion);
    int64_t n_gu = 0;
    for (int k = 0; k < pl->n_sets; ++k) {
        int EI, EJ;
        const int gs = tm::slices_per_group(pl->set_support[k], OO, EI, EJ);
        if (gs == 0) return false;
        n_gu += OO / gs;
    }
    return n_gu * n_regions <= tm::kMaxPlanCells;
}

namespace tm {

static TmState* state_of(imager_plan* pl) {
    if (pl->tmem) return static_cast<TmState*>(pl->tmem);
    TmState* st = new TmState();
    const imager_params& p = pl->p;
    const int OO = p.oversample * p.oversample;
    st->plan.resize(pl->n_sets);
    int n_gu = 0;
    for (int k = 0; k < pl->n_sets; ++k) {
        SetPlan sp = {};
        sp.group_slices = slices_per_group(pl->set_support[k], OO, sp.EI, sp.EJ);
        sp.n_groups = OO / sp.group_slices;
        sp.gu_base = n_gu;
        n_gu += sp.n_groups;
        for (int q = 0; q < sp.n_groups; ++q) st->gu_set.push_back(k);
        st->plan[k] = sp;
    }
    Geometry& g = st->g;
    g.N = p.grid_size;
    g.O = p.oversample;
    g.nt = pl->nt;
    g.n_regions = pl->nt * pl->nt;
    g.n_sets = pl->n_sets;
    g.n_gu = n_gu;
    g.n_pol = p.n_pol;
    g.n_corr = p.n_corr;
    pl->tmem = st;
    return st;
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

// (Re)build hit lists, items and blocks for the current index.  Synchronises the stream once (the list sizes are
// read back to size their storage); cached until the next re-indexing.
static int prepare(imager_plan* pl, TmState* st, cudaStream_t stream) {
    const int64_t mv = std::max<int64_t>(pl->p.max_nvis, 1);
    const Geometry& g = st->g;
    const int64_t n_cells = (int64_t)g.n_gu * g.n_regions;
    if (!st->d_plan) {
        IMAGER_CUDA(cudaMalloc(&st->d_plan, pl->n_sets * sizeof(SetPlan)));
        IMAGER_CUDA(cudaMalloc(&st->d_gu_set, st->gu_set.size() * sizeof(int32_t)));
        IMAGER_CUDA(cudaMemcpyAsync(st->d_plan, st->plan.data(), pl->n_sets * sizeof(SetPlan), cudaMemcpyHostToDevice, stream));
        IMAGER_CUDA(cudaMemcpyAsync(st->d_gu_set, st->gu_set.data(), st->gu_set.size() * sizeof(int32_t),
                                    cudaMemcpyHostToDevice, stream));
        int64_t tmp_len = 16;
        for (int64_t n = n_cells + 1; n > 1; n = (n + 1023) / 1024) tmp_len += (n + 1023) / 1024 + 1;
        IMAGER_CUDA(cudaMalloc(&st->d_hits, (n_cells + 1) * sizeof(int32_t)));
        IMAGER_CUDA(cudaMalloc(&st->d_items, (n_cells + 1) * sizeof(int32_t)));
        IMAGER_CUDA(cudaMalloc(&st->d_scan_tmp, tmp_len * sizeof(int32_t)));
        IMAGER_CUDA(cudaMalloc(&st->d_sgeo, mv * sizeof(uint2)));
        IMAGER_CUDA(cudaMalloc(&st->d_sval, mv * pl->p.n_corr * sizeof(float2)));
        IMAGER_CUDA(cudaMallocHost(&st->h_totals, 2 * sizeof(int32_t)));
    }
    if (st->plan_epoch == pl->index_epoch) return 0;
    sorted_geo_kernel<<<4 * kNumSMs, 256, 0, stream>>>(pl->d_counters, pl->d_perm[pl->sorted_buf], pl->d_rec,
                                                       pl->p.oversample, st->d_sgeo);
    PlanArgs pa;
    pa.g = g;
    pa.set_plan = st->d_plan;
    pa.gu_set = st->d_gu_set;
    pa.set_support = pl->d_set_support;
    pa.bucket_offset = pl->d_bucket_offset;
    pa.sgeo = st->d_sgeo;
    const unsigned nb = (unsigned)((n_cells + 1 + kPlanWarps - 1) / kPlanWarps);
    plan_hits_kernel<0><<<nb, kPlanWarps * 32, 0, stream>>>(pa, st->d_hits, st->d_items, nullptr, nullptr);
    pl->last_launches += 2;
    int rc = exclusive_scan_i32(pl, st->d_hits, n_cells + 1, st->d_scan_tmp, stream);
    if (rc) return rc;
    rc = exclusive_scan_i32(pl, st->d_items, n_cells + 1, st->d_scan_tmp, stream);
    if (rc) return rc;
    IMAGER_CUDA(cudaMemcpyAsync(&st->h_totals[0], st->d_hits + n_cells, sizeof(int32_t), cudaMemcpyDeviceToHost, stream));
    IMAGER_CUDA(cudaMemcpyAsync(&st->h_totals[1], st->d_items + n_cells, sizeof(int32_t), cudaMemcpyDeviceToHost, stream));
    IMAGER_CUDA(cudaStreamSynchronize(stream));
    const int64_t n_hits = st->h_totals[0], n_items = st->h_totals[1];
    if (n_hits < 0 || n_items < 0) {
        set_error("hit lists exceed 2^31 entries");
        return IMAGER_ERR_UNSUPPORTED;
    }
    const int n_sc = g.n_pol * g.n_corr;
    const int64_t max_blocks = ((int64_t)g.n_gu + n_hits / kBlockHits + 1) * n_sc;
    rc = grow(&st->d_hit_rec, &st->cap_hits, n_hits + 1);
    if (rc) return rc;
    rc = grow(&st->d_item_rec, &st->cap_items, n_items + 1);
    if (rc) return rc;
    rc = grow(&st->d_blocks, &st->cap_blocks, max_blocks + 1);
    if (rc) return rc;
    plan_hits_kernel<1><<<nb, kPlanWarps * 32, 0, stream>>>(pa, st->d_hits, st->d_items, st->d_hit_rec, st->d_item_rec);
    IMAGER_CUDA(cudaMemsetAsync(pl->d_counters + 11, 0, sizeof(int32_t), stream));
    plan_blocks_kernel<<<g.n_gu, 128, 0, stream>>>(g, st->d_hits, st->d_items, st->d_item_rec, st->d_blocks, pl->d_counters + 11,
                                                   (int)std::min<int64_t>(st->cap_blocks, 0x7fffffff));
    pl->last_launches += 2;
    IMAGER_CUDA(cudaGetLastError());
    st->plan_epoch = pl->index_epoch;
    return 0;
}

static void fill_args(imager_plan* pl, TmState* st, TmArgs& a, const float2* tab) {
    a.g = st->g;
    a.hit_rec = st->d_hit_rec;
    a.items = st->d_item_rec;
    a.blocks = st->d_blocks;
    a.n_blocks = pl->d_counters + 11;
    a.queue = pl->d_counters + 10;
    a.tab = tab;
    a.set_offset = pl->d_set_offset;
    a.set_support = pl->d_set_support;
    a.set_plan = st->d_plan;
    a.gu_set = st->d_gu_set;
}

}  // namespace tm

void tmem_release(imager_plan* pl) {
    if (!pl->tmem) return;
    tm::TmState* st = static_cast<tm::TmState*>(pl->tmem);
    cudaFree(st->d_plan);
    cudaFree(st->d_gu_set);
    cudaFree(st->d_hits);
    cudaFree(st->d_items);
    cudaFree(st->d_scan_tmp);
    cudaFree(st->d_hit_rec);
    cudaFree(st->d_item_rec);
    cudaFree(st->d_blocks);
    cudaFree(st->d_sgeo);
    cudaFree(st->d_sval);
    if (st->h_totals) cudaFreeHost(st->h_totals);
    delete st;
    pl->tmem = nullptr;
}

int launch_grid_tmem(imager_plan* pl, int64_t nvis, const float2* vis, const float* weights, float2* grid, cudaStream_t stream) {
    using namespace tm;
    if (nvis == 0) return 0;
    TmState* st = state_of(pl);
    int rc = prepare(pl, st, stream);
    if (rc) return rc;
    static bool attr_set = false;
    if (!attr_set) {
        IMAGER_CUDA(cudaFuncSetAttribute(grid_tmem_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes));
        IMAGER_CUDA(cudaFuncSetAttribute(grid_tmem_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes));
        attr_set = true;
    }
    const unsigned gb = 4 * kNumSMs;
    if (pl->p.n_corr == 1)
        gather_values_kernel<1><<<gb, 256, 0, stream>>>(pl->d_counters, pl->d_perm[pl->sorted_buf], vis, weights, st->d_sval);
    else
        gather_values_kernel<4><<<gb, 256, 0, stream>>>(pl->d_counters, pl->d_perm[pl->sorted_buf], vis, weights, st->d_sval);
    IMAGER_CUDA(cudaMemsetAsync(pl->d_counters + 10, 0, sizeof(int32_t), stream));
    TmArgs a;
    fill_args(pl, st, a, pl->d_tab_grid);
    if (pl->p.n_corr == 1)
        grid_tmem_kernel<1><<<kNumSMs, kThreads, kSmemBytes, stream>>>(a, st->d_sval, grid);
    else
        grid_tmem_kernel<4><<<kNumSMs, kThreads, kSmemBytes, stream>>>(a, st->d_sval, grid);
    pl->last_launches += 2;
    IMAGER_CUDA(cudaGetLastError());
    return 0;
}

int launch_degrid_tmem(imager_plan* pl, int64_t nvis, const float2* grid, float2* vis_out, cudaStream_t stream) {
    return launch_degrid_tiled(pl, nvis, grid, vis_out, 0, stream);
}

}  // namespace imager
