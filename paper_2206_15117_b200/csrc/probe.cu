// probe.cu -- micro-benchmarks of the two SM units the gridding / degridding kernels are bound by, kept in
// the library so that the numbers the design and bench.py's `lsu_floor_ms` rest on can be re-measured from the tree
// (tests/test_zy_gpu_microbench.py):
//   * the shared-memory (LSU) data pipe: clocks per warp-wide LDS.64 instruction per SM, with all 32 lanes active and with
//     only 16 (the claim: one LSU instruction of <= 8 bytes per lane costs about 2.1 clk per SM whatever its lane mask);
//   * the FP32 pipe: clocks per warp-wide FFMA2 (fma.rn.f32x2) instruction per SM.
// One CTA of 1024 threads per SM (32 warps, 8 per scheduler); every warp issues kUnroll independent instructions per loop
// trip; a CTA times itself with clock64 between two barriers.  Not part of the hot path.
#include "common.cuh"

namespace imager {

constexpr int kProbeThreads = 1024;
constexpr int kProbeUnroll = 8;

// mode 0: all lanes load; mode 1: lanes 0..15 only
__global__ void __launch_bounds__(kProbeThreads) lds64_probe_kernel(int iters, int mode, long long* __restrict__ clocks,
                                                                   float2* __restrict__ sink) {
    __shared__ float2 buf[4096];                                       // 32 KB
    for (int i = threadIdx.x; i < 4096; i += blockDim.x) buf[i] = make_float2((float)i, 1.f);
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const bool active = mode == 0 || lane < 16;
    float2 acc[kProbeUnroll];
#pragma unroll
    for (int u = 0; u < kProbeUnroll; ++u) acc[u] = make_float2(0.f, 0.f);
    const uint32_t buf0 = (uint32_t)__cvta_generic_to_shared(buf);
    const uint32_t off = (uint32_t)((warp * 32 + lane) * 8);             // a conflict-free 256-byte row per warp
    __syncthreads();
    const long long t0 = clock64();
    if (active) {
        for (int it = 0; it < iters; ++it) {
            // the address moves with the trip (8 rows of 2 KB apart) so that the compiler cannot merge the loads of
            // successive trips; largest offset 8184 + 7 * 256 + 7 * 2048 < 32 KB
            const uint32_t a = buf0 + off + (uint32_t)((it & 7) << 11);
#pragma unroll
            for (int u = 0; u < kProbeUnroll; ++u) {
                float x, y;
                asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(x), "=f"(y) : "r"(a + (uint32_t)(u * 256)) : "memory");
                acc[u].x += x;
                acc[u].y += y;
            }
        }
    }
    __syncthreads();
    const long long t1 = clock64();
    if (threadIdx.x == 0) clocks[blockIdx.x] = t1 - t0;
    float2 s = make_float2(0.f, 0.f);
#pragma unroll
    for (int u = 0; u < kProbeUnroll; ++u) { s.x += acc[u].x; s.y += acc[u].y; }
    if (s.x == -1.f) sink[threadIdx.x] = s;                            // keeps the loads alive, never taken
}

__global__ void __launch_bounds__(kProbeThreads) ffma2_probe_kernel(int iters, long long* __restrict__ clocks,
                                                                   float2* __restrict__ sink) {
    unsigned long long acc[kProbeUnroll];
    const float seed = 1.0f + (float)threadIdx.x * 1e-6f;
    unsigned long long m, c;
    asm volatile("mov.b64 %0, {%1, %2};" : "=l"(m) : "f"(0.999999f), "f"(1.000001f));
    asm volatile("mov.b64 %0, {%1, %2};" : "=l"(c) : "f"(1e-7f), "f"(-1e-7f));
#pragma unroll
    for (int u = 0; u < kProbeUnroll; ++u) asm volatile("mov.b64 %0, {%1, %2};" : "=l"(acc[u]) : "f"(seed + u), "f"(seed - u));
    __syncthreads();
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < kProbeUnroll; ++u) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(acc[u]) : "l"(m), "l"(c));
    }
    __syncthreads();
    const long long t1 = clock64();
    if (threadIdx.x == 0) clocks[blockIdx.x] = t1 - t0;
    float sx = 0.f;
#pragma unroll
    for (int u = 0; u < kProbeUnroll; ++u) {
        float x, y;
        asm volatile("mov.b64 {%0, %1}, %2;" : "=f"(x), "=f"(y) : "l"(acc[u]));
        sx += x + y;
    }
    if (sx == -1.f) sink[threadIdx.x] = make_float2(sx, 0.f);
}

}  // namespace imager

using namespace imager;

extern "C" int imager_debug_probe(double out[4], void* cuda_stream) {
    if (!out) { set_error("imager_debug_probe: out is NULL"); return IMAGER_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, n_sm = 0;
    IMAGER_CUDA(cudaGetDevice(&dev));
    IMAGER_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    long long* d_clk = nullptr;
    float2* d_sink = nullptr;
    IMAGER_CUDA(cudaMalloc(&d_clk, 3 * n_sm * sizeof(long long)));
    if (cudaMalloc(&d_sink, kProbeThreads * sizeof(float2)) != cudaSuccess) {
        cudaFree(d_clk);
        return cuda_fail(cudaErrorMemoryAllocation, "cudaMalloc(sink)");
    }
    const int iters = 4096;
    for (int rep = 0; rep < 2; ++rep) {                                // first round warms the instruction cache and clocks
        lds64_probe_kernel<<<n_sm, kProbeThreads, 0, st>>>(iters, 0, d_clk, d_sink);
        lds64_probe_kernel<<<n_sm, kProbeThreads, 0, st>>>(iters, 1, d_clk + n_sm, d_sink);
        ffma2_probe_kernel<<<n_sm, kProbeThreads, 0, st>>>(iters, d_clk + 2 * n_sm, d_sink);
    }
    std::vector<long long> h(3 * n_sm);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = cudaMemcpy(h.data(), d_clk, h.size() * sizeof(long long), cudaMemcpyDeviceToHost);
    cudaFree(d_clk);
    cudaFree(d_sink);
    if (e != cudaSuccess) return cuda_fail(e, "imager_debug_probe");
    const double warp_inst = (double)(kProbeThreads / 32) * iters * kProbeUnroll;       // per SM
    for (int k = 0; k < 3; ++k) {
        double sum = 0;
        for (int b = 0; b < n_sm; ++b) sum += (double)h[k * n_sm + b];
        out[k] = sum / n_sm / warp_inst;                               // clocks per warp instruction per SM (mean over SMs)
    }
    out[3] = (double)n_sm;
    return 0;
}
