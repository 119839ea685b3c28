// transform.cu -- surrounding stages A4 / A5 (built, outside the timed hot path): grid <-> image with cuFFT and
// the taper correction.  Signs follow the visibility equation, Eq. 2: V = sum I exp[+2 pi i (ul+vm+..)],
// so grid -> image is the FORWARD DFT and image -> grid the unnormalised inverse, both centred on (N/2, N/2)
// (R1).  For even N the centring is two (-1)^(x+y) sign flips, fused here with the division by
// psi(l) psi(m) (the image-domain anti-aliasing function the kernel tables were built from).
#include <cufft.h>
#include "common.cuh"
#include "pswf.h"

namespace imager {

__global__ void flip_scale_kernel(float2* __restrict__ data, int N, const double* __restrict__ taper, int divide,
                                  double norm) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y;
    if (x >= N) return;
    double f = ((x + y) & 1) ? -1.0 : 1.0;
    if (divide) f /= (taper[x] * taper[y] * norm);
    float2 v = data[(int64_t)y * N + x];
    v.x = (float)(v.x * f);
    v.y = (float)(v.y * f);
    data[(int64_t)y * N + x] = v;
}

int grid_image_transform(imager_plan* pl, float2* data, int direction, double norm, cudaStream_t st) {
    const int N = pl->p.grid_size;
    if (direction != 1 && direction != -1) {
        set_error("direction must be +1 or -1");
        return IMAGER_ERR_INVALID_ARG;
    }
    if (!pl->fft_ready) {
        Pswf psi(pl->p.pswf_support > 0 ? pl->p.pswf_support : 7);
        std::vector<double> t(N);
        for (int x = 0; x < N; ++x) t[x] = psi(2.0 * (x - N / 2) / N);
        IMAGER_CUDA(cudaMalloc(&pl->d_taper, N * sizeof(double)));
        IMAGER_CUDA(cudaMemcpy(pl->d_taper, t.data(), N * sizeof(double), cudaMemcpyHostToDevice));
        cufftHandle h;
        if (cufftPlan2d(&h, N, N, CUFFT_C2C) != CUFFT_SUCCESS) {
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
        flip_scale_kernel<<<grid, 256, 0, st>>>(plane, N, pl->d_taper, direction == -1, 1.0);
        if (cufftExecC2C(h, (cufftComplex*)plane, (cufftComplex*)plane, direction == 1 ? CUFFT_FORWARD : CUFFT_INVERSE) !=
            CUFFT_SUCCESS) {
            set_error("cufftExecC2C failed");
            return IMAGER_ERR_CUDA;
        }
        flip_scale_kernel<<<grid, 256, 0, st>>>(plane, N, pl->d_taper, direction == 1, norm);
    }
    IMAGER_CUDA(cudaGetLastError());
    return 0;
}

void destroy_transform(imager_plan* pl) {
    if (pl->fft_ready) cufftDestroy((cufftHandle)(intptr_t)pl->fft_plan);
    if (pl->d_taper) cudaFree(pl->d_taper);
    pl->fft_ready = false;
    pl->d_taper = nullptr;
}

}  // namespace imager
