// gridder_ref.cu -- the simple hot-path kernels: one warp per visibility, any n_corr / n_pol / support.
//   gridding   (A3): each lane walks taps t = lane, lane+32, ... of the S x S footprint and adds
//                    sum_c T[s][c][oy][ox][dy][dx] * (w_kc V_kc) to the grid with one red.global.add.v2.f32 per cell
//   degridding (A6): each lane accumulates conj(T) * G over its taps, then a warp-shuffle reduction
// They serve every shape the tiled kernels (gridder_tiled.cu) do not cover, and are selectable with
// IMAGER_PATH_REFERENCE for A/B checks.  Visibilities are walked in bucket-sorted order so that a warp's
// neighbours touch nearby cells and the same kernel slices (L2 locality).
#include "common.cuh"

namespace imager {

template <int NC, int NP>
__global__ void __launch_bounds__(256)
grid_ref_kernel(const int32_t* __restrict__ counters, const int32_t* __restrict__ perm,
                const imager_record* __restrict__ rec, const float2* __restrict__ vis,
                const float* __restrict__ weights, const float2* __restrict__ tab,
                const int64_t* __restrict__ set_offset, const int32_t* __restrict__ set_support,
                const int32_t* __restrict__ set_mask, int N, int O, float2* __restrict__ grid) {
    const int n_kept = counters[0];
    const int lane = threadIdx.x & 31;
    const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t n_warps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t i = warp0; i < n_kept; i += n_warps) {
        const int k = perm[i];
        const imager_record r = rec[k];
        if (set_mask && !set_mask[r.kset]) continue;
        const int S = set_support[r.kset], h_lo = S / 2, SS = S * S;
        const int sub = (int)((r.sub >> 8) & 255u) * O + (int)(r.sub & 255u);
        float2 val[NC];
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const float2 v = vis[(int64_t)k * NC + c];
            const float w = weights[(int64_t)k * NC + c];
            val[c] = weighted_sample(w, v);                                  // R24
        }
        const float2* T = tab + set_offset[r.kset] + (int64_t)sub * SS;
        const int64_t elem_stride = (int64_t)O * O * SS;
        for (int t = lane; t < SS; t += 32) {
            const int dy = t / S, dx = t - dy * S;
            const int64_t cell = (int64_t)(r.gy - h_lo + dy) * N + (r.gx - h_lo + dx);
#pragma unroll
            for (int s = 0; s < NP; ++s) {
                float ar = 0.f, ai = 0.f;
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    const float2 tp = __ldg(&T[(int64_t)(s * NC + c) * elem_stride + t]);
                    ar = fmaf(tp.x, val[c].x, ar);
                    ar = fmaf(-tp.y, val[c].y, ar);
                    ai = fmaf(tp.x, val[c].y, ai);
                    ai = fmaf(tp.y, val[c].x, ai);
                }
                atomicAdd(&grid[(int64_t)s * N * N + cell], make_float2(ar, ai));
            }
        }
    }
}

template <int NC, int NP>
__global__ void __launch_bounds__(256)
degrid_ref_kernel(int64_t nvis, const imager_record* __restrict__ rec, const int32_t* __restrict__ perm,
                  const float2* __restrict__ grid, const float2* __restrict__ tab,
                  const int64_t* __restrict__ set_offset, const int32_t* __restrict__ set_support,
                  const int32_t* __restrict__ set_mask, int N, int O, int residual, float2* __restrict__ vis_out) {
    const int lane = threadIdx.x & 31;
    const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t n_warps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t i = warp0; i < nvis; i += n_warps) {
        const int k = perm[i];                          // sorted order: dropped visibilities come last
        const imager_record r = rec[k];
        if (set_mask && !set_mask[r.kset] && !((r.sub >> 16) & 1u)) continue;     // dropped ones are always written (0)
        float2 acc[NC];
#pragma unroll
        for (int c = 0; c < NC; ++c) acc[c] = make_float2(0.f, 0.f);
        if (!((r.sub >> 16) & 1u)) {
            const int S = set_support[r.kset], h_lo = S / 2, SS = S * S;
            const int sub = (int)((r.sub >> 8) & 255u) * O + (int)(r.sub & 255u);
            const float2* T = tab + set_offset[r.kset] + (int64_t)sub * SS;
            const int64_t elem_stride = (int64_t)O * O * SS;
            for (int t = lane; t < SS; t += 32) {
                const int dy = t / S, dx = t - dy * S;
                const int64_t cell = (int64_t)(r.gy - h_lo + dy) * N + (r.gx - h_lo + dx);
#pragma unroll
                for (int s = 0; s < NP; ++s) {
                    const float2 g = __ldg(&grid[(int64_t)s * N * N + cell]);
#pragma unroll
                    for (int c = 0; c < NC; ++c) {
                        const float2 tp = __ldg(&T[(int64_t)(s * NC + c) * elem_stride + t]);
                        // conj(tp) * g
                        acc[c].x = fmaf(tp.x, g.x, acc[c].x);
                        acc[c].x = fmaf(tp.y, g.y, acc[c].x);
                        acc[c].y = fmaf(tp.x, g.y, acc[c].y);
                        acc[c].y = fmaf(-tp.y, g.x, acc[c].y);
                    }
                }
            }
        }
#pragma unroll
        for (int c = 0; c < NC; ++c) {
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) {
                acc[c].x += __shfl_xor_sync(0xffffffffu, acc[c].x, d);
                acc[c].y += __shfl_xor_sync(0xffffffffu, acc[c].y, d);
            }
        }
        if (lane == 0) {
#pragma unroll
            for (int c = 0; c < NC; ++c) {
                float2* o = vis_out + (int64_t)k * NC + c;
                *o = residual ? make_float2(o->x - acc[c].x, o->y - acc[c].y) : acc[c];
            }
        }
    }
}

template <int NC>
__global__ void sum_weights_kernel(int64_t nvis, const imager_record* __restrict__ rec, const float2* __restrict__ vis,
                                   const float* __restrict__ weights, double* __restrict__ sum_weights) {
    double acc[NC];
#pragma unroll
    for (int c = 0; c < NC; ++c) acc[c] = 0.0;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < nvis; k += (int64_t)gridDim.x * blockDim.x) {
        if ((rec[k].sub >> 16) & 1u) continue;
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const float w = weights[k * NC + c];
            if (!sample_flagged(w, vis[k * NC + c])) acc[c] += (double)w;           // R24: a flagged sample carries no weight
        }
    }
#pragma unroll
    for (int c = 0; c < NC; ++c) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) acc[c] += __shfl_xor_sync(0xffffffffu, acc[c], d);
        if ((threadIdx.x & 31) == 0 && acc[c] != 0.0) atomicAdd(&sum_weights[c], acc[c]);
    }
}

int launch_sum_weights(imager_plan* pl, int64_t nvis, const float2* vis, const float* weights, double* sum_weights, cudaStream_t st) {
    if (!sum_weights || nvis == 0) return 0;
    const unsigned blocks = (unsigned)std::min<int64_t>((nvis + 255) / 256, 4 * num_sms());
    if (pl->p.n_corr == 1) sum_weights_kernel<1><<<blocks, 256, 0, st>>>(nvis, pl->d_rec, vis, weights, sum_weights);
    else sum_weights_kernel<4><<<blocks, 256, 0, st>>>(nvis, pl->d_rec, vis, weights, sum_weights);
    pl->last_launches++;
    IMAGER_CUDA(cudaGetLastError());
    return 0;
}

int launch_grid_reference(imager_plan* pl, int64_t nvis, const float2* vis, const float* weights, float2* grid,
                          const int32_t* set_mask, cudaStream_t st) {
    if (nvis == 0) return 0;
    const unsigned blocks = (unsigned)std::min<int64_t>((nvis + 7) / 8, 16 * num_sms());
    const int N = pl->p.grid_size, O = pl->p.oversample;
    if (pl->p.n_corr == 1)
        grid_ref_kernel<1, 1><<<blocks, 256, 0, st>>>(pl->d_counters, pl->d_perm[pl->sorted_buf], pl->d_rec, vis, weights,
                                                      pl->d_tab_grid, pl->d_set_offset, pl->d_set_support, set_mask, N, O, grid);
    else
        grid_ref_kernel<4, 4><<<blocks, 256, 0, st>>>(pl->d_counters, pl->d_perm[pl->sorted_buf], pl->d_rec, vis, weights,
                                                      pl->d_tab_grid, pl->d_set_offset, pl->d_set_support, set_mask, N, O, grid);
    pl->last_launches++;
    IMAGER_CUDA(cudaGetLastError());
    return 0;
}

int launch_degrid_reference(imager_plan* pl, int64_t nvis, const float2* grid, float2* vis_out, const int32_t* set_mask,
                            int residual, cudaStream_t st) {
    if (nvis == 0) return 0;
    const unsigned blocks = (unsigned)std::min<int64_t>((nvis + 7) / 8, 16 * num_sms());
    const int N = pl->p.grid_size, O = pl->p.oversample;
    if (pl->p.n_corr == 1)
        degrid_ref_kernel<1, 1><<<blocks, 256, 0, st>>>(nvis, pl->d_rec, pl->d_perm[pl->sorted_buf], grid, pl->d_tab_degrid,
                                                        pl->d_set_offset, pl->d_set_support, set_mask, N, O, residual, vis_out);
    else
        degrid_ref_kernel<4, 4><<<blocks, 256, 0, st>>>(nvis, pl->d_rec, pl->d_perm[pl->sorted_buf], grid, pl->d_tab_degrid,
                                                        pl->d_set_offset, pl->d_set_support, set_mask, N, O, residual, vis_out);
    pl->last_launches++;
    IMAGER_CUDA(cudaGetLastError());
    return 0;
}

}  // namespace imager
