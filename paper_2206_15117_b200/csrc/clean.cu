// clean.cu -- the minor cycle and the Cotton-Schwab major-cycle loop around the hot path.
//
// PAPER.md:27 "The output images are cleaned using an implementation of the Cotton-Schwab algorithm [6], which accepts many
// of the usual parameters such as the number of clean cycles, the loop gain, the cycle factor, and a threshold stopping
// criterion"; PAPER.md:110 counts Hogbom cleaning among the "more iterative processes" that "are less able to take full
// advantage of parallelisation" (hence the device-side control below: the host never waits on it).  The paper gives
// neither in symbols; readings R18-R20 state them:
//   R18  Hogbom: p = first pixel (row-major) of the window with the largest |R|; a = gain * R[p]; model[p] += a;
//        R[q] -= a * B[q - p + c] wherever that PSF sample exists (c = N/2); up to n_iter times.
//   R19  the cycle stops when |R[p]| < max(threshold, cycle_factor * sidelobe * |R[p_0]|), sidelobe = max |B| outside the
//        3 x 3 pixels around the PSF centre, p_0 the first peak of the cycle.
//   R20  major cycle: residual visibilities V - V_model (model image -> grid -> degrid) -> grid -> residual image -> minor
//        cycle; the PSF is the dirty image of unit visibilities; the window is the inner half of the field.
// The peak search decides an integer, so it is taken in one fixed precision: every arithmetic step is ONE IEEE float32
// operation (__fmul_rn, __fsub_rn, __fadd_rn: never contracted into an FMA), in the order R18 / R19 write them, and ties go to
// the lowest row-major index -- which makes peak positions and component values comparable bit for bit with the oracle.
//
// Device-side control: an iteration is two launches, `hogbom_update_kernel` (subtract the previous component from the
// whole image and find every block's largest |R| inside the window, fused in one pass over the image) and
// `hogbom_pick_kernel` (one block: the global peak, the stop test, the new component).  The host never reads anything
// back: once the stop test fails the remaining launches see `done` and return at once.
#include "common.cuh"
#include <mutex>

namespace imager {

struct HogbomCtrl {
    float a;          // component to subtract in the next update (0 if none)
    int32_t p;        // its pixel (row-major), -1 if none
    float stop;       // R19, fixed by the first iteration
    int32_t done;     // the stop test has failed (or nothing is left to do)
    int32_t n_comp;   // components found so far
    int32_t iter;     // iterations started
    float sidelobe;   // max |B| outside the 3 x 3 centre
    int32_t pad;
};

constexpr int kCleanThreads = 256;

// larger |v| wins; ties go to the lower index (the first maximum in row-major order)
__device__ __forceinline__ void arg_better(float& bv, int& bi, float v, int i) {
    if (v > bv || (v == bv && i < bi)) {
        bv = v;
        bi = i;
    }
}

__global__ void psf_sidelobe_kernel(const float* __restrict__ psf, int n, HogbomCtrl* __restrict__ ctrl) {
    __shared__ float s[kCleanThreads];
    const int c = n / 2;
    float m = 0.f;
    for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < (int64_t)n * n; q += (int64_t)gridDim.x * blockDim.x) {
        const int y = (int)(q / n), x = (int)(q - (int64_t)y * n);
        if (abs(y - c) <= 1 && abs(x - c) <= 1) continue;
        m = fmaxf(m, fabsf(psf[q]));
    }
    s[threadIdx.x] = m;
    __syncthreads();
    for (int d = blockDim.x / 2; d > 0; d >>= 1) {
        if (threadIdx.x < d) s[threadIdx.x] = fmaxf(s[threadIdx.x], s[threadIdx.x + d]);
        __syncthreads();
    }
    if (threadIdx.x == 0) atomicMax(reinterpret_cast<int*>(&ctrl->sidelobe), __float_as_int(s[0]));   // non-negative floats
}

__global__ void __launch_bounds__(kCleanThreads)
hogbom_update_kernel(float* __restrict__ res, const float* __restrict__ psf, int n, int y0, int x0, int y1, int x1,
                     const HogbomCtrl* __restrict__ ctrl, float* __restrict__ part_val, int32_t* __restrict__ part_idx) {
    __shared__ float s_v[kCleanThreads];
    __shared__ int s_i[kCleanThreads];
    if (ctrl->done) return;
    const float a = ctrl->a;
    const int p = ctrl->p, c = n / 2;
    const int py = p >= 0 ? p / n : 0, px = p >= 0 ? p - py * n : 0;
    float bv = -1.f;
    int bi = 0x7fffffff;
    for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < (int64_t)n * n; q += (int64_t)gridDim.x * blockDim.x) {
        const int y = (int)(q / n), x = (int)(q - (int64_t)y * n);
        float r = res[q];
        if (p >= 0) {
            const int by = y - py + c, bx = x - px + c;
            if (by >= 0 && by < n && bx >= 0 && bx < n) {
                r = __fsub_rn(r, __fmul_rn(a, psf[(int64_t)by * n + bx]));
                res[q] = r;
            }
        }
        if (y >= y0 && y < y1 && x >= x0 && x < x1) arg_better(bv, bi, fabsf(r), (int)q);
    }
    s_v[threadIdx.x] = bv;
    s_i[threadIdx.x] = bi;
    __syncthreads();
    for (int d = blockDim.x / 2; d > 0; d >>= 1) {
        if (threadIdx.x < d) arg_better(s_v[threadIdx.x], s_i[threadIdx.x], s_v[threadIdx.x + d], s_i[threadIdx.x + d]);
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        part_val[blockIdx.x] = s_v[0];
        part_idx[blockIdx.x] = s_i[0];
    }
}

// `last` = 1: the call after the final iteration only retires the pending component (nothing more is picked)
__global__ void __launch_bounds__(kCleanThreads)
hogbom_pick_kernel(const float* __restrict__ res, float* __restrict__ model, int n, int n_parts, const float* __restrict__ part_val,
                   const int32_t* __restrict__ part_idx, float gain, float threshold, float cycle_factor, int last,
                   HogbomCtrl* __restrict__ ctrl, float* __restrict__ comps) {
    __shared__ float s_v[kCleanThreads];
    __shared__ int s_i[kCleanThreads];
    if (ctrl->done) return;
    float bv = -1.f;
    int bi = 0x7fffffff;
    for (int k = threadIdx.x; k < n_parts; k += blockDim.x) arg_better(bv, bi, part_val[k], part_idx[k]);
    s_v[threadIdx.x] = bv;
    s_i[threadIdx.x] = bi;
    __syncthreads();
    for (int d = blockDim.x / 2; d > 0; d >>= 1) {
        if (threadIdx.x < d) arg_better(s_v[threadIdx.x], s_i[threadIdx.x], s_v[threadIdx.x + d], s_i[threadIdx.x + d]);
        __syncthreads();
    }
    if (threadIdx.x != 0) return;
    ctrl->a = 0.f;
    ctrl->p = -1;
    if (last || s_i[0] == 0x7fffffff) {                 // nothing left to pick (or an empty window)
        ctrl->done = 1;
        return;
    }
    const int p = s_i[0];
    const float peak = res[p];
    if (ctrl->iter == 0) ctrl->stop = fmaxf(threshold, __fmul_rn(__fmul_rn(cycle_factor, ctrl->sidelobe), fabsf(peak)));
    ctrl->iter += 1;
    if (!(fabsf(peak) >= ctrl->stop)) {
        ctrl->done = 1;
        return;
    }
    const float a = __fmul_rn(gain, peak);
    model[p] = __fadd_rn(model[p], a);
    if (comps) {
        const int k = ctrl->n_comp;
        comps[3 * k] = (float)(p / n);
        comps[3 * k + 1] = (float)(p - (p / n) * n);
        comps[3 * k + 2] = a;
    }
    ctrl->n_comp += 1;
    ctrl->a = a;
    ctrl->p = p;
}

__global__ void store_count_kernel(const HogbomCtrl* __restrict__ ctrl, int32_t* __restrict__ n_out) { *n_out = ctrl->n_comp; }

// The minor cycle on device buffers; scratch is stream-ordered (cudaMallocAsync), nothing is read back.
int run_hogbom(float* residual, const float* psf, float* model, int n, const int32_t window[4], float gain, float threshold,
               float cycle_factor, int n_iter, float* components_out, int32_t* n_components_out, cudaStream_t st, int* launches) {
    const int y0 = std::max(0, window[0]), x0 = std::max(0, window[1]), y1 = std::min(n, window[2]), x1 = std::min(n, window[3]);
    const int blocks = (int)std::min<int64_t>(((int64_t)n * n + kCleanThreads - 1) / kCleanThreads, 4 * num_sms());
    HogbomCtrl* ctrl = nullptr;
    float* part_val = nullptr;
    int32_t* part_idx = nullptr;
    auto fail = [&](cudaError_t e, const char* what) {      // an exit on error frees what was allocated so far
        if (ctrl) cudaFreeAsync(ctrl, st);
        if (part_val) cudaFreeAsync(part_val, st);
        if (part_idx) cudaFreeAsync(part_idx, st);
        return cuda_fail(e, what);
    };
#define HOGBOM_CUDA(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return fail(e__, #call); } while (0)
    HOGBOM_CUDA(cudaMallocAsync(&ctrl, sizeof(HogbomCtrl), st));
    HOGBOM_CUDA(cudaMallocAsync(&part_val, blocks * sizeof(float), st));
    HOGBOM_CUDA(cudaMallocAsync(&part_idx, blocks * sizeof(int32_t), st));
    HogbomCtrl init = {};
    init.p = -1;
    if (y1 <= y0 || x1 <= x0 || n_iter <= 0) init.done = 1;
    HOGBOM_CUDA(cudaMemcpyAsync(ctrl, &init, sizeof(init), cudaMemcpyHostToDevice, st));   // pageable source: copied before return
    psf_sidelobe_kernel<<<blocks, kCleanThreads, 0, st>>>(psf, n, ctrl);
    int count = 1;
    for (int it = 0; it <= n_iter; ++it) {
        hogbom_update_kernel<<<blocks, kCleanThreads, 0, st>>>(residual, psf, n, y0, x0, y1, x1, ctrl, part_val, part_idx);
        hogbom_pick_kernel<<<1, kCleanThreads, 0, st>>>(residual, model, n, blocks, part_val, part_idx, gain, threshold,
                                                        cycle_factor, it == n_iter, ctrl, components_out);
        count += 2;
    }
    if (n_components_out) {
        store_count_kernel<<<1, 1, 0, st>>>(ctrl, n_components_out);
        ++count;
    }
    HOGBOM_CUDA(cudaGetLastError());
#undef HOGBOM_CUDA
    IMAGER_CUDA(cudaFreeAsync(ctrl, st));
    IMAGER_CUDA(cudaFreeAsync(part_val, st));
    IMAGER_CUDA(cudaFreeAsync(part_idx, st));
    if (launches) *launches += count;
    return 0;
}

// ---- major cycle -----------------------------------------------------------------------------------------------
__global__ void fill_ones_kernel(int64_t n, float2* __restrict__ v) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        v[i] = make_float2(1.f, 0.f);
}
__global__ void real_part_kernel(int64_t n, const float2* __restrict__ in, float* __restrict__ out) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) out[i] = in[i].x;
}
// total += cycle (one float32 addition per pixel, as the oracle's), and the complex model image for A5
__global__ void add_model_kernel(int64_t n, float* __restrict__ total, const float* __restrict__ cycle, float2* __restrict__ image) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float t = __fadd_rn(total[i], cycle[i]);
        total[i] = t;
        image[i] = make_float2(t, 0.f);
    }
}

}  // namespace imager

using namespace imager;

extern "C" int imager_hogbom(float* residual, const float* psf, float* model, int32_t n, const int32_t window[4], float gain,
                             float threshold, float cycle_factor, int32_t n_iter, float* components_out,
                             int32_t* n_components_out, void* cuda_stream) {
    if (!residual || !psf || !model || !window || n < 2 || n > 32768) {
        set_error("imager_hogbom: NULL argument or bad size");
        return IMAGER_ERR_INVALID_ARG;
    }
    return run_hogbom(residual, psf, model, n, window, gain, threshold, cycle_factor, n_iter, components_out, n_components_out,
                      (cudaStream_t)cuda_stream, nullptr);
}

extern "C" int imager_clean(imager_plan* plan, int64_t nvis, const float* uvw, const float* vis, const float* weights,
                            const int32_t* a_index, const imager_clean_params* cp, float* model_image, float* residual_image,
                            float* residual_vis, float* psf_out, int32_t* n_components_out, void* cuda_stream) {
    if (!plan || !cp || !model_image || !residual_image || !residual_vis || (nvis > 0 && (!uvw || !vis || !weights))) {
        set_error("imager_clean: NULL argument");
        return IMAGER_ERR_INVALID_ARG;
    }
    if (plan->p.n_pol != 1 || plan->p.n_corr != 1) {
        set_error("imager_clean is built for single-polarisation plans");
        return IMAGER_ERR_UNSUPPORTED;
    }
    if (cp->n_major < 1 || cp->n_iter < 0 || !(cp->gain > 0.f)) {
        set_error("imager_clean: need n_major >= 1, n_iter >= 0, gain > 0");
        return IMAGER_ERR_INVALID_ARG;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int n = plan->p.grid_size;
    const int64_t npix = (int64_t)n * n;
    const unsigned gb = 4 * num_sms();
    float2* work = nullptr;                      // [N][N] complex: grid <-> image
    float *psf = nullptr, *cycle = nullptr;
    double* sumwt = nullptr;
    IMAGER_CUDA(cudaMallocAsync(&work, npix * sizeof(float2), st));
    IMAGER_CUDA(cudaMallocAsync(&psf, npix * sizeof(float), st));
    IMAGER_CUDA(cudaMallocAsync(&cycle, npix * sizeof(float), st));
    IMAGER_CUDA(cudaMallocAsync(&sumwt, sizeof(double), st));
    int rc = 0, launches = 0;
    auto done = [&](int code) {
        cudaFreeAsync(work, st);
        cudaFreeAsync(psf, st);
        cudaFreeAsync(cycle, st);
        cudaFreeAsync(sumwt, st);
        plan->last_launches = launches;
        return code;
    };
#define CLEAN_CUDA(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return done(cuda_fail(e__, #call)); } while (0)
#define CLEAN_RC(call) do { rc = (call); launches += plan->last_launches; if (rc) return done(rc); } while (0)
    // A1 + A2 once; every later call reuses the index (the steady state of the loop)
    CLEAN_RC(imager_index(plan, nvis, uvw, a_index, cuda_stream));
    // PSF: the dirty image of unit visibilities
    CLEAN_CUDA(cudaMemsetAsync(work, 0, npix * sizeof(float2), st));
    CLEAN_CUDA(cudaMemsetAsync(sumwt, 0, sizeof(double), st));
    fill_ones_kernel<<<gb, 256, 0, st>>>(nvis, (float2*)residual_vis);
    CLEAN_RC(imager_grid(plan, nvis, uvw, residual_vis, weights, a_index, (float*)work, sumwt, IMAGER_REUSE_INDEX, cuda_stream));
    CLEAN_RC(grid_image_transform_dev(plan, work, +1, sumwt, st));
    real_part_kernel<<<gb, 256, 0, st>>>(npix, work, psf);
    if (psf_out) CLEAN_CUDA(cudaMemcpyAsync(psf_out, psf, npix * sizeof(float), cudaMemcpyDeviceToDevice, st));
    CLEAN_CUDA(cudaMemsetAsync(model_image, 0, npix * sizeof(float), st));
    CLEAN_CUDA(cudaMemcpyAsync(residual_vis, vis, nvis * sizeof(float2), cudaMemcpyDeviceToDevice, st));
    launches += 2;
    const int q = n / 4;
    const int32_t window[4] = {q, q, 3 * q, 3 * q};
    for (int m = 0; m < cp->n_major; ++m) {
        CLEAN_CUDA(cudaMemsetAsync(work, 0, npix * sizeof(float2), st));
        CLEAN_RC(imager_grid(plan, nvis, uvw, residual_vis, weights, a_index, (float*)work, nullptr, IMAGER_REUSE_INDEX, cuda_stream));
        CLEAN_RC(grid_image_transform_dev(plan, work, +1, sumwt, st));
        real_part_kernel<<<gb, 256, 0, st>>>(npix, work, residual_image);
        CLEAN_CUDA(cudaMemsetAsync(cycle, 0, npix * sizeof(float), st));
        rc = run_hogbom(residual_image, psf, cycle, n, window, cp->gain, cp->threshold, cp->cycle_factor, cp->n_iter, nullptr,
                        n_components_out ? n_components_out + m : nullptr, st, &launches);
        if (rc) return done(rc);
        add_model_kernel<<<gb, 256, 0, st>>>(npix, model_image, cycle, work);
        CLEAN_RC(grid_image_transform_dev(plan, work, -1, nullptr, st));
        CLEAN_CUDA(cudaMemcpyAsync(residual_vis, vis, nvis * sizeof(float2), cudaMemcpyDeviceToDevice, st));
        CLEAN_RC(imager_degrid(plan, nvis, uvw, a_index, (const float*)work, residual_vis, IMAGER_REUSE_INDEX | IMAGER_DEGRID_RESIDUAL,
                               cuda_stream));
        launches += 2;
    }
    CLEAN_CUDA(cudaGetLastError());
#undef CLEAN_CUDA
#undef CLEAN_RC
    return done(0);
}

// ---- the minor cycle for callers that may not allocate (imager_hogbom_static) ------------------------------------------
//
// imager_hogbom takes its three scratch buffers (control block, per-block peak values, per-block peak indices) from the
// stream-ordered pool on every call.  That is no good to a caller whose device memory was shared out once at start-up and
// who must not touch the allocator afterwards: an imaging loop that sits beside a correlator or beamformer on the same GPU
// with every byte of HBM already promised, a process running under a framework whose caching allocator owns the whole
// device, or a real-time loop that cannot afford the allocator's locks, its possible pool growth or the device-wide wait a
// cudaMalloc / cudaFree may bring.  For them the same kernels run here on scratch that is part of the library image: a
// file-scope device array, resident on every GPU that loads libimager.so from the moment the module is loaded until the
// process exits, whether or not this entry point is ever called.
//
// Size: 256 bytes of control block + one (value, index) pair per thread block, one block per 1024 pixels, sized for
// images up to IMAGER_HOGBOM_STATIC_MAX_N = 4096 pixels a side: 256 + 16384 * 8 = 131,328 bytes per GPU.
//
// `g_hogbom_scratch` below is a DEVICE symbol.  Device code may name it; in host code the identifier is only the host
// shadow of the symbol and is NOT a device address (handing `g_hogbom_scratch` itself to a kernel would fault, or on a
// system where the GPU can reach host memory quietly work on the wrong bytes).  Host code gets the real address once per
// device from cudaGetSymbolAddress, with that device current, and passes that pointer to the kernels.
namespace imager {

constexpr int kStaticMaxN = IMAGER_HOGBOM_STATIC_MAX_N;
constexpr int kStaticPixelsPerBlock = 1024;                                            // 256 threads x 4 pixels
constexpr int kStaticMaxParts = (kStaticMaxN / 32) * (kStaticMaxN / 32);               // 16384 blocks at the largest image
constexpr size_t kStaticCtrlBytes = 256;
constexpr size_t kStaticScratchBytes = kStaticCtrlBytes + (size_t)kStaticMaxParts * (sizeof(float) + sizeof(int32_t));
constexpr int kStaticMaxDevices = 64;
static_assert(sizeof(HogbomCtrl) <= kStaticCtrlBytes, "control block outgrew its slot");
static_assert((int64_t)kStaticMaxParts * kStaticPixelsPerBlock == (int64_t)kStaticMaxN * kStaticMaxN, "block count of the largest image");

static __device__ __align__(256) unsigned char g_hogbom_scratch[kStaticScratchBytes];

static std::mutex g_static_mutex;
static unsigned char* g_static_addr[kStaticMaxDevices] = {};       // device address of g_hogbom_scratch, per device ordinal

// The array keeps whatever the previous call left in it: the control block is rewritten in full here (the sidelobe level
// is built with atomicMax and the counters are incremented, so both must start from zero); the per-block pairs need no
// clearing, every block of an update launch overwrites its own pair before the pick kernel reads it.
__global__ void hogbom_static_reset_kernel(HogbomCtrl* __restrict__ ctrl, int done) {
    HogbomCtrl c;
    c.a = 0.f;
    c.p = -1;
    c.stop = 0.f;
    c.done = done;
    c.n_comp = 0;
    c.iter = 0;
    c.sidelobe = 0.f;
    c.pad = 0;
    *ctrl = c;
}

// Set-up, once per device: resolve the device address of the scratch array for the CURRENT device and remember it.
static int static_scratch_address(unsigned char** out) {
    int dev = -1;
    IMAGER_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) {
        set_error("imager_hogbom_static: device ordinal %d is outside the %d this build keeps addresses for", dev, kStaticMaxDevices);
        return IMAGER_ERR_UNSUPPORTED;
    }
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_addr[dev]) {
        void* p = nullptr;
        IMAGER_CUDA(cudaGetSymbolAddress(&p, g_hogbom_scratch));
        if (!p) {
            set_error("imager_hogbom_static: cudaGetSymbolAddress returned a null address");
            return IMAGER_ERR_CUDA;
        }
        g_static_addr[dev] = static_cast<unsigned char*>(p);
    }
    *out = g_static_addr[dev];
    return 0;
}

}  // namespace imager

extern "C" int imager_hogbom_static(float* residual, const float* psf, float* model, int32_t n, const int32_t window[4],
                                    float gain, float threshold, float cycle_factor, int32_t n_iter, float* components_out,
                                    int32_t* n_components_out, void* cuda_stream) {
    if (!residual || !psf || !model || !window || n < 2) {
        set_error("imager_hogbom_static: NULL argument or bad size");
        return IMAGER_ERR_INVALID_ARG;
    }
    if (n > kStaticMaxN) {
        set_error("imager_hogbom_static: image side n = %d exceeds IMAGER_HOGBOM_STATIC_MAX_N = %d (the built-in scratch holds one "
                  "peak per 1024 pixels of a %d x %d image); use imager_hogbom, which allocates, for larger images",
                  n, kStaticMaxN, kStaticMaxN, kStaticMaxN);
        return IMAGER_ERR_UNSUPPORTED;
    }
    unsigned char* base = nullptr;
    if (int rc = static_scratch_address(&base)) return rc;
    HogbomCtrl* ctrl = reinterpret_cast<HogbomCtrl*>(base);
    float* part_val = reinterpret_cast<float*>(base + kStaticCtrlBytes);
    int32_t* part_idx = reinterpret_cast<int32_t*>(base + kStaticCtrlBytes + (size_t)kStaticMaxParts * sizeof(float));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int y0 = std::max(0, window[0]), x0 = std::max(0, window[1]), y1 = std::min(n, window[2]), x1 = std::min(n, window[3]);
    const int blocks = (int)(((int64_t)n * n + kStaticPixelsPerBlock - 1) / kStaticPixelsPerBlock);    // <= kStaticMaxParts
    hogbom_static_reset_kernel<<<1, 1, 0, st>>>(ctrl, (y1 <= y0 || x1 <= x0 || n_iter <= 0) ? 1 : 0);
    psf_sidelobe_kernel<<<blocks, kCleanThreads, 0, st>>>(psf, n, ctrl);
    for (int it = 0; it <= n_iter; ++it) {
        hogbom_update_kernel<<<blocks, kCleanThreads, 0, st>>>(residual, psf, n, y0, x0, y1, x1, ctrl, part_val, part_idx);
        hogbom_pick_kernel<<<1, kCleanThreads, 0, st>>>(residual, model, n, blocks, part_val, part_idx, gain, threshold,
                                                        cycle_factor, it == n_iter, ctrl, components_out);
    }
    if (n_components_out) store_count_kernel<<<1, 1, 0, st>>>(ctrl, n_components_out);
    IMAGER_CUDA(cudaGetLastError());
    return 0;
}
