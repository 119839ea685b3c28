// transform.cu -- surrounding stages A4 / A5 (built, outside the timed hot path): grid <-> image with cuFFT and
// the taper correction.  Signs follow the visibility equation, Eq. 2: V = sum I exp[+2 pi i (ul+vm+..)],
// so grid -> image is the FORWARD DFT and image -> grid the unnormalised inverse, both centred on (N/2, N/2)
// (R1).  For even N the centring is two (-1)^(x+y) sign flips, fused here with the division by
// psi(l) psi(m) (the image-domain anti-aliasing function the kernel tables were built from).
#include <cufft.h>
#include "common.cuh"
#include "pswf.h"

namespace imager {

// norm_dev (device, may be NULL) overrides `norm`: the sum of weights of a gridding call that is still in flight
__global__ void flip_scale_kernel(float2* __restrict__ data, int N, const double* __restrict__ taper, int divide,
                                  double norm, const double* __restrict__ norm_dev) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y;
    if (x >= N) return;
    if (norm_dev) norm = (*norm_dev == 0.0) ? 1.0 : *norm_dev;
    double f = ((x + y) & 1) ? -1.0 : 1.0;
    if (divide) f /= (taper[x] * taper[y] * norm);
    float2 v = data[(int64_t)y * N + x];
    v.x = (float)(v.x * f);
    v.y = (float)(v.y * f);
    data[(int64_t)y * N + x] = v;
}

static int transform_impl(imager_plan* pl, float2* data, int direction, double norm, const double* norm_dev, cudaStream_t st);

int grid_image_transform(imager_plan* pl, float2* data, int direction, double norm, cudaStream_t st) {
    return transform_impl(pl, data, direction, norm, nullptr, st);
}

int grid_image_transform_dev(imager_plan* pl, float2* data, int direction, const double* norm_dev, cudaStream_t st) {
    return transform_impl(pl, data, direction, 1.0, norm_dev, st);
}

static int transform_impl(imager_plan* pl, float2* data, int direction, double norm, const double* norm_dev, cudaStream_t st) {
    const int N = pl->p.grid_size;
    if (direction != 1 && direction != -1) {
        set_error("direction must be +1 or -1");
        return IMAGER_ERR_INVALID_ARG;
    }
    if (!pl->fft_ready) {
        Pswf psi(pl->p.pswf_support > 0 ? pl->p.pswf_support : 7);
        std::vector<double> t(N);
        for (int x = 0; x < N; ++x) t[x] = psi(2.0 * (x - N / 2) / N);
        if (!pl->d_taper) IMAGER_CUDA(cudaMalloc(&pl->d_taper, N * sizeof(double)));
        IMAGER_CUDA(cudaMemcpy(pl->d_taper, t.data(), N * sizeof(double), cudaMemcpyHostToDevice));
        cufftHandle h;
        if (cufftPlan2d(&h, N, N, CUFFT_C2C) != CUFFT_SUCCESS) {
            cudaFree(pl->d_taper);                            // a retry starts clean
            pl->d_taper = nullptr;
            set_error("cufftPlan2d(%d) failed", N);
            return IMAGER_ERR_CUDA;
        }
        pl->fft_plan = (void*)(intptr_t)h;
        pl->fft_ready = true;
    }
    cufftHandle h = (cufftHandle)(intptr_t)pl->fft_plan;
    if (cufftSetStream(h, st) != CUFFT_SUCCESS) {
        set_error("cufftSetStream failed");
        return IMAGER_ERR_CUDA;
    }
    if (norm == 0.0) norm = 1.0;
    const dim3 grid((N + 255) / 256, N);
    for (int s = 0; s < pl->p.n_pol; ++s) {
        float2* plane = data + (int64_t)s * N * N;
        flip_scale_kernel<<<grid, 256, 0, st>>>(plane, N, pl->d_taper, direction == -1, 1.0, nullptr);
        if (cufftExecC2C(h, (cufftComplex*)plane, (cufftComplex*)plane, direction == 1 ? CUFFT_FORWARD : CUFFT_INVERSE) !=
            CUFFT_SUCCESS) {
            set_error("cufftExecC2C failed");
            return IMAGER_ERR_CUDA;
        }
        flip_scale_kernel<<<grid, 256, 0, st>>>(plane, N, pl->d_taper, direction == 1, norm, direction == 1 ? norm_dev : nullptr);
    }
    IMAGER_CUDA(cudaGetLastError());
    return 0;
}

// ---- Eq. 1: UV-domain mosaic weighting correction ---------------------------------------------
// ssq(l,m) = sum_i B_i(l,m)^2 with B_i = E^2(l - l_i, m - m_i), E = 2 J1(x) / x, x = pi D rho nu / c;
// gamma = [sqrt(ssq) / max sqrt(ssq)] * [1 / ssq] = 1 / (max_root * sqrt(ssq)).
__global__ void mosaic_ssq_kernel(int N, double cell, double dish, double freq, int n_point, const double* __restrict__ lm,
                                  double* __restrict__ ssq, unsigned long long* __restrict__ max_bits) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y;
    if (x >= N) return;
    const double l = (x - N / 2) * cell, m = (y - N / 2) * cell;
    double s = 0.0;
    for (int i = 0; i < n_point; ++i) {
        const double xx = M_PI * dish * hypot(l - lm[2 * i], m - lm[2 * i + 1]) * freq / 299792458.0;
        const double e = xx == 0.0 ? 1.0 : 2.0 * j1(xx) / xx;
        const double b = e * e;
        s += b * b;
    }
    ssq[(int64_t)y * N + x] = s;
    atomicMax(max_bits, (unsigned long long)__double_as_longlong(sqrt(s)));      // non-negative doubles order as integers
}

__global__ void mosaic_gamma_kernel(int64_t n, const double* __restrict__ ssq, const unsigned long long* __restrict__ max_bits,
                                    float* __restrict__ gamma) {
    const double mx = __longlong_as_double((long long)*max_bits);
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        gamma[i] = (float)(1.0 / (mx * sqrt(ssq[i])));
}

__global__ void mosaic_apply_kernel(int64_t n, int n_pol, const float* __restrict__ gamma, float2* __restrict__ image) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float gmm = gamma[i];
        for (int s = 0; s < n_pol; ++s) {
            float2 v = image[s * n + i];
            v.x *= gmm;
            v.y *= gmm;
            image[s * n + i] = v;
        }
    }
}

int mosaic_correct(imager_plan* pl, float2* image, cudaStream_t st) {
    const int N = pl->p.grid_size, na = pl->p.n_aplanes;
    const int64_t n = (int64_t)N * N;
    if (!pl->d_gamma) {
        std::vector<double> lm(2 * (size_t)na, 0.0);
        if (!pl->pointing_lm.empty()) lm = pl->pointing_lm;
        double *d_lm = nullptr, *d_ssq = nullptr;
        unsigned long long* d_max = nullptr;
        float* d_gamma = nullptr;
        cudaError_t e = cudaMalloc(&d_lm, lm.size() * sizeof(double));
        if (e == cudaSuccess) e = cudaMalloc(&d_ssq, n * sizeof(double));
        if (e == cudaSuccess) e = cudaMalloc(&d_max, sizeof(unsigned long long));
        if (e == cudaSuccess) e = cudaMalloc(&d_gamma, n * sizeof(float));
        if (e == cudaSuccess) e = cudaMemcpyAsync(d_lm, lm.data(), lm.size() * sizeof(double), cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) e = cudaMemsetAsync(d_max, 0, sizeof(unsigned long long), st);
        if (e == cudaSuccess) {
            mosaic_ssq_kernel<<<dim3((N + 127) / 128, N), 128, 0, st>>>(N, pl->p.cell_size_rad, pl->p.dish_diameter_m, pl->p.freq_hz,
                                                                       na, d_lm, d_ssq, d_max);
            mosaic_gamma_kernel<<<4 * num_sms(), 256, 0, st>>>(n, d_ssq, d_max, d_gamma);
            e = cudaStreamSynchronize(st);                      // lm (host vector) and the scratch are released below
        }
        cudaFree(d_lm);
        cudaFree(d_ssq);
        cudaFree(d_max);
        if (e != cudaSuccess) {
            cudaFree(d_gamma);
            return cuda_fail(e, "mosaic_correct: building gamma");
        }
        pl->d_gamma = d_gamma;
    }
    mosaic_apply_kernel<<<4 * num_sms(), 256, 0, st>>>(n, pl->p.n_pol, pl->d_gamma, image);
    IMAGER_CUDA(cudaGetLastError());
    return 0;
}

void destroy_transform(imager_plan* pl) {
    if (pl->d_gamma) cudaFree(pl->d_gamma);
    pl->d_gamma = nullptr;
    if (pl->fft_ready) cufftDestroy((cufftHandle)(intptr_t)pl->fft_plan);
    if (pl->d_taper) cudaFree(pl->d_taper);
    pl->fft_ready = false;
    pl->d_taper = nullptr;
}

}  // namespace imager
