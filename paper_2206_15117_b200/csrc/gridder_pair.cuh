// gridder_pair.cuh -- gridding / degridding kernels that replay TWO hits per warp instruction (IMAGER_PAIR = 1).
// Included by gridder_tiled.cu, inside namespace imager, after the shared helpers (TiledArgs, lds64, cmac_*, ...).
//
// Why (profiles/r1_lds_mask_probe.md, r1b_ncu_grid_degrid.md): the kernels are bound by shared-memory load
// INSTRUCTIONS (2.1 clk each whatever the lane mask or the number of distinct addresses), and with an 8 x 4 lane block
// only 70 % of a tap load's lanes fall inside a footprint.  Here each half-warp is a 4 x 4 lane block with its own hit
// (the hardware serves an LDS.64 half-warp by half-warp, so the two hits cannot conflict), which cuts the waste at the
// footprint edges to (S+3)^2 / S^2, serves two hit descriptors with one broadcast-per-half-warp LDS.128, and halves
// the reduction traffic of degridding.  Counted on config 2: 310 M instead of 364 M shared-memory instructions per
// gridding launch, 380 M instead of 463 M per degridding launch, for 1.42 x the hits (16 x 16 strips).
//
// Both half-warps own the SAME 16 x 16 strip (4 x 4 slots per lane): gridding keeps two partial accumulators per cell
// (one per half-warp) and both are added to the grid when the item ends; degridding keeps two copies of the strip.
// Hits of a run (same slot range) are taken two at a time; the second half-warp idles on the odd one.
//
// STATUS: parity-green (tests/test_gpu_parity.py and the full-size sampled tests pass with -DIMAGER_PAIR=1) but NOT the
// default: on config 2 the shared-memory instructions drop as counted (341 M instead of 383 M per gridding launch), yet
// the kernel is slower (3.23-3.40 ms against 3.08 ms; degridding 4.47-4.70 against 4.40; config 3 87 against 70 ms):
// about 50 of the 100 slot-range bodies are live at once on 16 x 16 strips, the warps wait for instruction fetch
// (no_instruction 4.3 stalls per issue against 0.8), and 1.42 x the hits cost 1.42 x the gathers, flushes and planner.
// Kept behind the macro as the starting point for a variant-poor version.
#pragma once

// ---- dispatch over the 100 slot-range variants -------------------------------------------------------------
#define PAIR_CASE(FN, IL, IH1, JL, JH1) \
    case IMAGER_VARIANT(IL, IH1, JL, JH1): FN<IL, (IH1) + 1, JL, (JH1) + 1> IMAGER_BODY_ARGS; break;
#define PAIR_CASES_J(FN, IL, IH1)                                                                               \
    PAIR_CASE(FN, IL, IH1, 0, 0) PAIR_CASE(FN, IL, IH1, 0, 1) PAIR_CASE(FN, IL, IH1, 0, 2) PAIR_CASE(FN, IL, IH1, 0, 3) \
    PAIR_CASE(FN, IL, IH1, 1, 1) PAIR_CASE(FN, IL, IH1, 1, 2) PAIR_CASE(FN, IL, IH1, 1, 3)                       \
    PAIR_CASE(FN, IL, IH1, 2, 2) PAIR_CASE(FN, IL, IH1, 2, 3) PAIR_CASE(FN, IL, IH1, 3, 3)
#define PAIR_DISPATCH(FN, variant)                                                              \
    switch (variant) {                                                                          \
        PAIR_CASES_J(FN, 0, 0) PAIR_CASES_J(FN, 0, 1) PAIR_CASES_J(FN, 0, 2) PAIR_CASES_J(FN, 0, 3) \
        PAIR_CASES_J(FN, 1, 1) PAIR_CASES_J(FN, 1, 2) PAIR_CASES_J(FN, 1, 3)                    \
        PAIR_CASES_J(FN, 2, 2) PAIR_CASES_J(FN, 2, 3) PAIR_CASES_J(FN, 3, 3)                    \
        default: break;                                                                         \
    }

// slot mask of a ctrl byte: bit 4 i + j for x-slot i, y-slot j
__device__ __forceinline__ uint32_t pair_slot_mask(uint32_t ctrl) {
    const uint32_t il = ctrl & 3u, ih = ((ctrl >> 2) & 3u) + 1u, jl = (ctrl >> 4) & 3u, jh = (ctrl >> 6) + 1u;
    const uint32_t rows = (1u << jh) - (1u << jl);
    const uint32_t cols = ((1u << (4u * ih)) - (1u << (4u * il))) / 15u;       // 0x1111 pattern over the x-slots
    return rows * cols;
}

constexpr uint32_t kNoVariant = 127u;       // lanes beyond the batch: matches no body

// ---- gridding ----------------------------------------------------------------------------------------------
// A run: `cnt` consecutive staged hits (stage slots h .. h + cnt - 1) with the same slot range.  Half-warp q takes hits
// h + q, h + q + 2, ...; on an odd count the second half-warp repeats the last hit with a zero value.
template <int IL, int IH, int JL, int JH>
__device__ __forceinline__ void grid_run_pair(u64 (&C)[kNX][kNY], const uint32_t stage_addr, const int h, const int cnt, const int q,
                                              const uint32_t lane_off, const uint32_t (&step)[kNY]) {
    const int h_last = h + cnt - 1;
    int hq = h + q;
    uint4 d = lds128(stage_addr + 16u * (uint32_t)min(hq, h_last));
    int iters = (cnt + 1) >> 1;
#pragma unroll 1
    do {
        const bool valid = hq <= h_last;
        const uint32_t addr = d.z + lane_off;
        const float vx = valid ? __uint_as_float(d.x) : 0.f, vy = valid ? __uint_as_float(d.y) : 0.f;
        hq += 2;
        d = lds128(stage_addr + 16u * (uint32_t)min(hq, h_last));            // the next pair (a repeat at the run's end)
        constexpr int NI = IH - IL;
        constexpr int kRows = (NI >= 3) ? 2 : 4;                              // at most 8 tap loads in flight
#pragma unroll
        for (int j0 = JL; j0 < JH; j0 += kRows) {
            float2 t[kRows][NI];
#pragma unroll
            for (int j = j0; j < j0 + kRows && j < JH; ++j)
#pragma unroll
                for (int i = IL; i < IH; ++i) t[j - j0][i - IL] = lds64(addr + step[j] + (uint32_t)(i * kLaneW * 8));
#pragma unroll
            for (int j = j0; j < j0 + kRows && j < JH; ++j)
#pragma unroll
                for (int i = IL; i < IH; ++i) cmac_re(C[i][j], t[j - j0][i - IL], vx);
#pragma unroll
            for (int j = j0; j < j0 + kRows && j < JH; ++j)
#pragma unroll
                for (int i = IL; i < IH; ++i) cmac_im(C[i][j], t[j - j0][i - IL], vy);
        }
    } while (--iters > 0);
}

template <int NC>
__global__ void __launch_bounds__(kGridThreads, 1)
grid_pair_kernel(const TiledArgs a, const float2* __restrict__ sval, float2* __restrict__ grid) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint4* stage = reinterpret_cast<uint4*>(smem_raw) + (threadIdx.x >> 5) * kStageSlots;  // this warp's descriptors
    float2* tab_s = reinterpret_cast<float2*>(smem_raw + kGridStageBytes);
    const uint32_t tab_addr = (uint32_t)__cvta_generic_to_shared(tab_s);
    const uint32_t stage_addr = (uint32_t)__cvta_generic_to_shared(stage);
    __shared__ int s_block, s_next;
    const int lane = threadIdx.x & 31, q = lane >> 4, lx = lane & (kLaneW - 1), ly = (lane >> 2) & (kLaneH - 1);
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
        uint32_t step[kNY];                                // byte offsets of the y-slots, in uniform registers
#pragma unroll
        for (int j = 0; j < kNY; ++j) step[j] = __reduce_or_sync(0xffffffffu, (uint32_t)(j * kLaneH * sp.pitch * 8));
        const uint32_t lane_off = (uint32_t)((ly * sp.pitch + lx) * 8);
        for (;;) {
            int ii = 0;
            if (lane == 0) ii = atomicAdd(&s_next, 1);
            ii = __shfl_sync(0xffffffffu, ii, 0);
            if (ii >= blk.item_count) break;
            const Item it = a.items[blk.item_begin + ii];
            u64 C[kNX][kNY];
#pragma unroll
            for (int i = 0; i < kNX; ++i)
#pragma unroll
                for (int j = 0; j < kNY; ++j) C[i][j] = 0ull;
            uint32_t touched = 0u;
            uint2 rec = make_uint2(0u, 0u), rec1 = make_uint2(0u, 0u);
            float2 val = make_float2(0.f, 0.f);
            if (lane < it.hit_count) rec = a.hit_rec[it.hit_begin + lane];
            if (lane + 32 < it.hit_count) rec1 = a.hit_rec[it.hit_begin + 32 + lane];
            if (lane < it.hit_count) val = sval[(int64_t)rec.x * NC + c_corr];
            for (int b0 = 0; b0 < it.hit_count; b0 += 32) {
                const int n = min(32, it.hit_count - b0);
                const uint32_t my_ctrl = rec.y >> 24;
                const uint32_t my_variant = lane < n ? ctrl_variant(my_ctrl) : kNoVariant;
                stage[lane] = make_uint4(__float_as_uint(val.x), __float_as_uint(val.y),
                                         tab_addr + (uint32_t)(((int)(rec.y & 0xffffffu) - (int)kTapBias) * 8), rec.x);
                if (lane < n) touched |= pair_slot_mask(my_ctrl);
                rec = rec1;
                if (b0 + 32 + lane < it.hit_count) val = sval[(int64_t)rec.x * NC + c_corr];
                if (b0 + 64 + lane < it.hit_count) rec1 = a.hit_rec[it.hit_begin + b0 + 64 + lane];
                __syncwarp();
                for (int h = 0; h < n;) {                                   // runs of equal variant (the planner sorted them)
                    const uint32_t variant = __reduce_or_sync(0xffffffffu, lane == h ? my_variant : 0u);   // warp-uniform
                    const int cnt = __popc(__ballot_sync(0xffffffffu, lane >= h && lane < n && my_variant == variant));
#define IMAGER_BODY_ARGS (C, stage_addr, h, cnt, q, lane_off, step)
                    PAIR_DISPATCH(grid_run_pair, variant)
#undef IMAGER_BODY_ARGS
                    h += cnt;
                }
                __syncwarp();
            }
            touched = __reduce_or_sync(0xffffffffu, touched);
            // both half-warps add their partial strips to the grid
            const int sy = it.strip / g.strips_per_row, sx = it.strip - sy * g.strips_per_row;
            float2* gp = gplane + (int64_t)(sy * kStripH + ly) * g.N + sx * kStripW + lx;
#pragma unroll
            for (int i = 0; i < kNX; ++i)
#pragma unroll
                for (int j = 0; j < kNY; ++j)
                    if (touched & (1u << (4 * i + j))) {
                        const float2 c = unpack2(C[i][j]);
                        if (c.x != 0.f || c.y != 0.f) atomicAdd(gp + (int64_t)(kLaneH * j) * g.N + kLaneW * i, c);
                    }
        }
    }
}

// ---- degridding --------------------------------------------------------------------------------------------
// Each half-warp holds the strip in registers and accumulates sum conj(t) g over its lanes' cells for its own hit.
// Per pair of hits one STS.64 writes the 2 x 16 partial sums to red[pair slot][lane]; every 8 pairs (16 hits) lane
// L = 2 u + part sums 8 of the 16 partials of hit u by a transposed read, one shuffle joins the two parts, and the
// sum is added to the visibility with one red.global.add.v2.f32.
constexpr int kPairSlots = kRedSlots;                       // pair slots per reduction: 8 x 32 x 8 bytes per warp

template <int IL, int IH, int JL, int JH>
__device__ __forceinline__ void degrid_run_pair(const float2 (&G)[kNX][kNY], const uint32_t stage_addr, const int h, const int cnt,
                                                const int iters_in, const int q, uint32_t red_addr, const uint32_t lane_off,
                                                const uint32_t (&step)[kNY]) {
    const int h_last = h + cnt - 1;
    int hq = h + q;
    uint32_t a_cur = lds32(stage_addr + 8u * (uint32_t)min(hq, h_last));
    int iters = iters_in;
#pragma unroll 1
    do {
        const uint32_t addr = a_cur + lane_off;
        hq += 2;
        a_cur = lds32(stage_addr + 8u * (uint32_t)min(hq, h_last));            // the next pair (a repeat at the run's end)
        u64 P[4] = {0ull, 0ull, 0ull, 0ull};                                    // four independent FFMA2 chains
        constexpr int NI = IH - IL;
        constexpr int kRows = (NI >= 3) ? 2 : 4;
#pragma unroll
        for (int j0 = JL; j0 < JH; j0 += kRows) {
            float2 t[kRows][NI];
#pragma unroll
            for (int j = j0; j < j0 + kRows && j < JH; ++j)
#pragma unroll
                for (int i = IL; i < IH; ++i) t[j - j0][i - IL] = lds64(addr + step[j] + (uint32_t)(i * kLaneW * 8));
#pragma unroll
            for (int j = j0; j < j0 + kRows && j < JH; ++j)
#pragma unroll
                for (int i = IL; i < IH; ++i) dmac_re(P[(i + 2 * j) & 3], t[j - j0][i - IL], G[i][j].x);
#pragma unroll
            for (int j = j0; j < j0 + kRows && j < JH; ++j)
#pragma unroll
                for (int i = IL; i < IH; ++i) dmac_im(P[(i + 2 * j) & 3], t[j - j0][i - IL], G[i][j].y);
        }
        sts64(red_addr, unpack2(add2p(add2p(P[0], P[1]), add2p(P[2], P[3]))));
        red_addr += 32 * 8;
    } while (--iters > 0);
}

template <int NC>
__global__ void __launch_bounds__(kTiledThreads, 1)
degrid_pair_kernel(const TiledArgs a, const float2* __restrict__ grid, float2* __restrict__ ssum) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5;
    uint2* stage = reinterpret_cast<uint2*>(smem_raw) + warp * kStageSlots;               // {tap address, sorted index}
    float2* red = reinterpret_cast<float2*>(smem_raw + kStageBytes) + warp * kPairSlots * 32;
    float2* tab_s = reinterpret_cast<float2*>(smem_raw + kStageBytes + kRedBytes);
    const uint32_t tab_addr = (uint32_t)__cvta_generic_to_shared(tab_s);
    const uint32_t stage_addr = (uint32_t)__cvta_generic_to_shared(stage);
    const uint32_t red_base = (uint32_t)__cvta_generic_to_shared(red);
    __shared__ int s_block, s_next;
    const int lane = threadIdx.x & 31, q = lane >> 4, lx = lane & (kLaneW - 1), ly = (lane >> 2) & (kLaneH - 1);
    const int red_slot = lane >> 2, red_q = (lane >> 1) & 1, red_part = lane & 1;       // reduction role: hit 2 red_slot + red_q
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
            float2 G[kNX][kNY];
#pragma unroll
            for (int i = 0; i < kNX; ++i)
#pragma unroll
                for (int j = 0; j < kNY; ++j) G[i][j] = __ldg(gp + (int64_t)(kLaneH * j) * g.N + kLaneW * i);
            uint2 rec = make_uint2(0u, 0u), rec1 = make_uint2(0u, 0u);
            if (lane < it.hit_count) rec = a.hit_rec[it.hit_begin + lane];
            if (lane + 32 < it.hit_count) rec1 = a.hit_rec[it.hit_begin + 32 + lane];
            for (int b0 = 0; b0 < it.hit_count; b0 += 32) {
                const int n = min(32, it.hit_count - b0);
                const uint32_t my_variant = lane < n ? ctrl_variant(rec.y >> 24) : kNoVariant;
                stage[lane] = make_uint2(tab_addr + (uint32_t)(((int)(rec.y & 0xffffffu) - (int)kTapBias) * 8), rec.x);
                rec = rec1;
                if (b0 + 64 + lane < it.hit_count) rec1 = a.hit_rec[it.hit_begin + b0 + 64 + lane];
                __syncwarp();
                int ps = 0;                                     // pair slots filled since the last reduction
                int my_red_hit = -1;                            // stage slot of the hit this lane reduces, or -1
                for (int h = 0; h < n;) {
                    const uint32_t variant = __reduce_or_sync(0xffffffffu, lane == h ? my_variant : 0u);   // warp-uniform
                    int cnt = __popc(__ballot_sync(0xffffffffu, lane >= h && lane < n && my_variant == variant));
                    const int iters = min((cnt + 1) >> 1, kPairSlots - ps);      // runs do not cross a reduction batch
                    cnt = min(cnt, 2 * iters);
                    const uint32_t red_addr = red_base + (uint32_t)((ps * 32 + lane) * 8);
#define IMAGER_BODY_ARGS (G, stage_addr, h, cnt, iters, q, red_addr, lane_off, step)
                    PAIR_DISPATCH(degrid_run_pair, variant)
#undef IMAGER_BODY_ARGS
                    if (red_slot >= ps && red_slot < ps + iters) {
                        const int hit = h + 2 * (red_slot - ps) + red_q;
                        my_red_hit = hit < h + cnt ? hit : -1;
                    }
                    ps += iters;
                    h += cnt;
                    if (ps == kPairSlots || h == n) {
                        __syncwarp();
                        float2 acc = make_float2(0.f, 0.f);
                        if (my_red_hit >= 0) {
#pragma unroll
                            for (int k = 0; k < 8; ++k) {
                                const float2 v = lds64(red_base + (uint32_t)((red_slot * 32 + 16 * red_q + 8 * red_part +
                                                                              ((k + (lane >> 1)) & 7)) * 8));
                                acc.x += v.x;
                                acc.y += v.y;
                            }
                        }
                        acc.x += __shfl_xor_sync(0xffffffffu, acc.x, 1);
                        acc.y += __shfl_xor_sync(0xffffffffu, acc.y, 1);
                        if (red_part == 0 && my_red_hit >= 0) {
                            const uint32_t idx = stage[my_red_hit].y;
                            atomicAdd(&ssum[(int64_t)idx * NC + c_corr], acc);
                        }
                        ps = 0;
                        my_red_hit = -1;
                        __syncwarp();
                    }
                }
                __syncwarp();
            }
        }
    }
}
