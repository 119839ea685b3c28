// mosaic.cu -- image-domain mosaic: image-plane reprojection and the per-component loops.
//
// PAPER.md:46 "For image-domain mosaics, an image of each mosaic component is generated with the phase position at its
// centre, and image-plane reprojection is used to construct the mosaic at a common phase position.  Prior to the
// degridding stage of cleaning the model image is reprojected to the phase position of each mosaic component, and multiple
// FFT and degridding steps are performed."  Readings (R21-R23): frames related by the translation of the
// pointing offsets (small field); bilinear interpolation, zero outside the source, a component image used only inside its
// inner half; mosaic = sum_i w_i B_i reproject_i[I_i] with w_i = sum of weights of component i / total and B the Airy power
// beam centred on the component -- the linear mosaic the UV-domain path forms with its beam kernels, so that
// the same Eq. 1 correction applies afterwards.
//
// Every component goes through the hot path with its own small grid: imager_grid (index + bucket + grid) -> cuFFT + taper
// -> reproject-accumulate; and backwards reproject -> cuFFT -> imager_degrid.  "Multiple FFT and degridding steps" are
// exactly this loop; it runs on one stream with one plan (the component grid) and never synchronises beyond the one wait
// of each indexing step.
#include "common.cuh"

namespace imager {

// dst(l, m) (+)= scale * B * bilinear(src at (l - shift_l, m - shift_m)); coordinates and weights in double, data float32.
// beam: 0 none, 1 centred on the source frame, 2 centred on the target frame.  inner_half: source pixels outside
// [n/4, 3n/4) count as zero.  scale_dev (may be NULL): multiply by 1 / *scale_dev (0 counts as 1).
__global__ void reproject_kernel(const float2* __restrict__ src, int n_src, double cell_src, float2* __restrict__ dst, int n_dst,
                                 double cell_dst, double shift_l, double shift_m, int beam, double dish, double freq, int inner_half,
                                 int accumulate, const double* __restrict__ scale_dev) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y;
    if (x >= n_dst) return;
    const double l = (x - n_dst / 2) * cell_dst, m = (y - n_dst / 2) * cell_dst;
    const double ls = l - shift_l, ms = m - shift_m;
    const double fx = ls / cell_src + n_src / 2, fy = ms / cell_src + n_src / 2;
    const double x0f = floor(fx), y0f = floor(fy);
    const double tx = fx - x0f, ty = fy - y0f;
    const int lo = inner_half ? n_src / 4 : 0, hi = inner_half ? 3 * (n_src / 4) : n_src;
    double ar = 0.0, ai = 0.0;
    if (x0f >= -1.0 && x0f <= (double)n_src && y0f >= -1.0 && y0f <= (double)n_src) {
        const int x0 = (int)x0f, y0 = (int)y0f;
#pragma unroll
        for (int dy = 0; dy < 2; ++dy)
#pragma unroll
            for (int dx = 0; dx < 2; ++dx) {
                const int yy = y0 + dy, xx = x0 + dx;
                if (yy < lo || yy >= hi || xx < lo || xx >= hi) continue;
                const double w = (dy ? ty : 1.0 - ty) * (dx ? tx : 1.0 - tx);
                const float2 v = src[(int64_t)yy * n_src + xx];
                ar += w * (double)v.x;
                ai += w * (double)v.y;
            }
    }
    double f = 1.0;
    if (beam) {
        const double rho = beam == 1 ? hypot(ls, ms) : hypot(l, m);
        const double xx = M_PI * dish * rho * freq / 299792458.0;
        const double e = xx == 0.0 ? 1.0 : 2.0 * j1(xx) / xx;
        f = e * e;
    }
    if (scale_dev && *scale_dev != 0.0) f /= *scale_dev;
    float2* o = dst + (int64_t)y * n_dst + x;
    const float2 add = make_float2((float)(ar * f), (float)(ai * f));
    *o = accumulate ? make_float2(o->x + add.x, o->y + add.y) : add;
}

int launch_reproject(const float2* src, int n_src, double cell_src, float2* dst, int n_dst, double cell_dst, double shift_l,
                     double shift_m, int beam, double dish, double freq, int inner_half, int accumulate, const double* scale_dev,
                     cudaStream_t st) {
    reproject_kernel<<<dim3((n_dst + 127) / 128, n_dst), 128, 0, st>>>(src, n_src, cell_src, dst, n_dst, cell_dst, shift_l, shift_m,
                                                                      beam, dish, freq, inner_half, accumulate, scale_dev);
    IMAGER_CUDA(cudaGetLastError());
    return 0;
}

__global__ void scale_by_inverse_kernel(int64_t n, float2* __restrict__ v, const double* __restrict__ denom) {
    const double d = *denom == 0.0 ? 1.0 : *denom;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        v[i] = make_float2((float)(v[i].x / d), (float)(v[i].y / d));
}

}  // namespace imager

using namespace imager;

extern "C" int imager_reproject(const float* src, int32_t n_src, double cell_src, float* dst, int32_t n_dst, double cell_dst,
                                double shift_l, double shift_m, int32_t beam, double dish_diameter_m, double freq_hz,
                                int32_t inner_half, int32_t accumulate, void* cuda_stream) {
    if (!src || !dst || n_src < 2 || n_dst < 2 || !(cell_src > 0) || !(cell_dst > 0) || beam < 0 || beam > 2) {
        set_error("imager_reproject: NULL argument or bad size");
        return IMAGER_ERR_INVALID_ARG;
    }
    return launch_reproject((const float2*)src, n_src, cell_src, (float2*)dst, n_dst, cell_dst, shift_l, shift_m, beam,
                            dish_diameter_m, freq_hz, inner_half, accumulate, nullptr, (cudaStream_t)cuda_stream);
}

static int check_mosaic_args(imager_plan* plan, int32_t n_point, const int64_t* nvis, const void* const* uvw, const double* lm,
                             const void* image, int32_t n_mosaic, double cell_mosaic) {
    if (!plan || n_point < 1 || !nvis || !uvw || !lm || !image || n_mosaic < 2 || !(cell_mosaic > 0)) {
        set_error("image-domain mosaic: NULL argument or bad size");
        return IMAGER_ERR_INVALID_ARG;
    }
    if (plan->p.n_pol != 1 || plan->p.n_corr != 1 || plan->p.n_aplanes != 1) {
        set_error("image-domain mosaic needs a single-polarisation component plan with one A-plane");
        return IMAGER_ERR_UNSUPPORTED;
    }
    const int mode = plan->p.kernel_mode;
    if (mode == IMAGER_MODE_MOSAIC_PB || mode == IMAGER_MODE_AWPROJ_ADJOINT || mode == IMAGER_MODE_AWPROJ_PAPER) {
        // the beam is applied here, in the image plane (reproject): a plan whose gridding kernel already holds it would apply it twice
        set_error("image-domain mosaic needs a plan WITHOUT a beam in its kernels (PSWF, WPROJ, or USER tables of that kind); "
                  "kernel_mode %d carries the primary beam", mode);
        return IMAGER_ERR_UNSUPPORTED;
    }
    return 0;
}

extern "C" int imager_mosaic_grid(imager_plan* plan, int32_t n_point, const int64_t* nvis, const float* const* uvw,
                                  const float* const* vis, const float* const* weights, const double* pointing_lm,
                                  float* mosaic_image, int32_t n_mosaic, double cell_mosaic, double* sum_weights,
                                  void* cuda_stream) {
    int rc = check_mosaic_args(plan, n_point, nvis, (const void* const*)uvw, pointing_lm, mosaic_image, n_mosaic, cell_mosaic);
    if (rc) return rc;
    if (!vis || !weights) { set_error("imager_mosaic_grid: NULL argument"); return IMAGER_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int n = plan->p.grid_size;
    const int64_t npix = (int64_t)n * n, nmos = (int64_t)n_mosaic * n_mosaic;
    float2* work = nullptr;
    double* total = nullptr;
    int launches = 0;
    auto done = [&](int code) {                          // every exit frees what was allocated so far
        if (work) cudaFreeAsync(work, st);
        if (total) cudaFreeAsync(total, st);
        plan->last_launches = launches;
        return code;
    };
#define MOSAIC_CUDA(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return done(cuda_fail(e__, #call)); } while (0)
    MOSAIC_CUDA(cudaMallocAsync(&work, npix * sizeof(float2), st));
    MOSAIC_CUDA(cudaMallocAsync(&total, sizeof(double), st));
    MOSAIC_CUDA(cudaMemsetAsync(total, 0, sizeof(double), st));
    MOSAIC_CUDA(cudaMemsetAsync(mosaic_image, 0, nmos * sizeof(float2), st));
    for (int i = 0; i < n_point; ++i) {
        // component i at its own phase centre: grid (A1 + A2 + A3), transform with the taper but WITHOUT the division by its
        // sum of weights (w_i I_i = FFT(G_i) / psi psi / total: the component's own sum cancels, R23)
        MOSAIC_CUDA(cudaMemsetAsync(work, 0, npix * sizeof(float2), st));
        rc = imager_grid(plan, nvis[i], uvw[i], vis[i], weights[i], nullptr, (float*)work, total, 0, cuda_stream);
        launches += plan->last_launches;
        if (rc) return done(rc);
        rc = grid_image_transform(plan, work, +1, 1.0, st);
        if (rc) return done(rc);
        rc = launch_reproject(work, n, plan->p.cell_size_rad, (float2*)mosaic_image, n_mosaic, cell_mosaic, pointing_lm[2 * i],
                              pointing_lm[2 * i + 1], 1, plan->p.dish_diameter_m, plan->p.freq_hz, 1, 1, nullptr, st);
        if (rc) return done(rc);
        launches += 4;
    }
    scale_by_inverse_kernel<<<4 * num_sms(), 256, 0, st>>>(nmos, (float2*)mosaic_image, total);
    if (sum_weights) MOSAIC_CUDA(cudaMemcpyAsync(sum_weights, total, sizeof(double), cudaMemcpyDeviceToDevice, st));
    MOSAIC_CUDA(cudaGetLastError());
    return done(0);
}

extern "C" int imager_mosaic_degrid(imager_plan* plan, int32_t n_point, const int64_t* nvis, const float* const* uvw,
                                    const double* pointing_lm, const float* model_image, int32_t n_mosaic, double cell_mosaic,
                                    float* const* vis_out, uint32_t flags, void* cuda_stream) {
    int rc = check_mosaic_args(plan, n_point, nvis, (const void* const*)uvw, pointing_lm, model_image, n_mosaic, cell_mosaic);
    if (rc) return rc;
    if (!vis_out) { set_error("imager_mosaic_degrid: NULL argument"); return IMAGER_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int n = plan->p.grid_size;
    float2* work = nullptr;
    IMAGER_CUDA(cudaMallocAsync(&work, (int64_t)n * n * sizeof(float2), st));
    int launches = 0;
    auto done = [&](int code) {
        cudaFreeAsync(work, st);
        plan->last_launches = launches;
        return code;
    };
    for (int i = 0; i < n_point; ++i) {
        // the model as component i sees it: B(l', m') model(l' + l_i, m' + m_i) on its own frame, then A5 and A6
        rc = launch_reproject((const float2*)model_image, n_mosaic, cell_mosaic, work, n, plan->p.cell_size_rad, -pointing_lm[2 * i],
                              -pointing_lm[2 * i + 1], 2, plan->p.dish_diameter_m, plan->p.freq_hz, 0, 0, nullptr, st);
        if (rc) return done(rc);
        rc = grid_image_transform(plan, work, -1, 1.0, st);
        if (rc) return done(rc);
        rc = imager_degrid(plan, nvis[i], uvw[i], nullptr, (const float*)work, vis_out[i], flags & IMAGER_DEGRID_RESIDUAL, cuda_stream);
        launches += plan->last_launches + 4;
        if (rc) return done(rc);
    }
    MOSAIC_CUDA(cudaGetLastError());
#undef MOSAIC_CUDA
    return done(0);
}
