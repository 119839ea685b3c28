/* imager.h -- C-ABI of libimager.so: the gridding / degridding hot path of the GPU imager of
 * arxiv/paper_2206_15117 ("A GPU-based Imager with Polarised Primary-beam Correction"), built for one
 * NVIDIA B200 (sm_100a).  Citations "P:NN" are lines of the paper text; "R<n>" are the readings
 * listed in DESIGN.md where the paper is silent.
 *
 * What is computed:
 *   gridding    G[s][gy+dy][gx+dx] += sum_c T[kset][s][c][oy][ox][dy][dx] * (w_kc * V_kc)
 *   degridding  V_kc = sum_s sum_{dy,dx} conj(T_d[kset][s][c][oy][ox][dy][dx]) * G[s][gy+dy][gx+dx]
 * with T = anti-aliasing function x w-correction term x Mueller-matrix cell (or its inverse), Fourier
 * transformed to the UV domain, oversampled O times per cell and looked up at the nearest sub-cell.
 * (gx,gy), (ox,oy), the signed w-plane and the kernel set `kset` of a visibility follow R2-R5.
 *
 * General rules
 *   - Every pointer argument says "dev" (CUDA device memory, caller-owned, e.g. a torch tensor) or "host".
 *   - The library never allocates or frees caller memory.  All device work is enqueued on the given
 *     cuda_stream (a cudaStream_t passed as void*; NULL = the legacy default stream).
 *   - Synchronisation contract.  imager_grid / imager_degrid with IMAGER_REUSE_INDEX (the steady state of a major-cycle
 *     loop) only enqueue work: no host wait, no allocation.  A call that (re)indexes -- imager_index, or the first
 *     imager_grid / imager_degrid after new (uvw, a_index) -- waits ONCE for cuda_stream (cudaStreamSynchronize: the
 *     sizes of the hit lists are read back to bound the launches that follow and to guard their 32-bit offsets) and may
 *     grow plan-owned scratch if the data need more than the estimate made at the first call.  Never a device-wide
 *     synchronisation.  Plan creation and the debug / statistics exports synchronise.
 *   - A plan is bound to ONE stream at a time: its work queues and cached hit lists are plan state, so calls on the
 *     same plan must be issued on the same stream (or be ordered by the caller); use one plan per concurrent stream.
 *   - Limits per call: nvis <= max_nvis, and fewer than 2^31 hits (visibility x 16 x 32-cell strip pairs; about 4 per
 *     visibility at support 15, 15 at support 63) -- IMAGER_ERR_TOO_MANY_VIS otherwise.  Larger data sets are fed in
 *     chunks: gridding accumulates into the caller's grid, degridding is per visibility.
 *   - Every call returns 0 on success or a negative imager_status.  No exceptions, no abort, no printing.
 *     imager_last_error() gives a thread-local message for the last failure on this thread.
 *     Asynchronous CUDA faults surface on the next call or at the caller's synchronisation.
 *   - There is no CPU fallback: without a CUDA device every call fails with IMAGER_ERR_CUDA.
 */
#ifndef IMAGER_H_
#define IMAGER_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum imager_status {
    IMAGER_OK = 0,
    IMAGER_ERR_INVALID_ARG = -1,
    IMAGER_ERR_UNSUPPORTED = -2,
    IMAGER_ERR_NOMEM = -3,
    IMAGER_ERR_CUDA = -4,
    IMAGER_ERR_TOO_MANY_VIS = -5
} imager_status;

/* kernel_mode: which image-domain function the kernel tables are the transform of (R6, R9-R11) */
enum {
    IMAGER_MODE_DELTA = 0,          /* S = 1, O = 1, T = 1 (test mode: a visibility lands on one cell)            */
    IMAGER_MODE_PSWF = 1,           /* psi(l) psi(m): prolate-spheroidal anti-aliasing function only        */
    IMAGER_MODE_WPROJ = 2,          /* psi psi exp(-2 pi i w_p (n-1)): w-projection                          */
    IMAGER_MODE_AWPROJ_ADJOINT = 3, /* 4x4: (M S^-1)^H cells x psi psi x w-term; degridding is the exact adjoint   */
    IMAGER_MODE_AWPROJ_PAPER = 4,   /* 4x4: gridding from (M^S')^-1 S with Eq. 6, degridding as mode 3  */
    IMAGER_MODE_MOSAIC_PB = 5,      /* psi psi E^2(l - l_a, m - m_a): primary beam as gridding kernel       */
    IMAGER_MODE_USER = 6            /* tables supplied by the caller                                               */
};

/* flags of imager_grid / imager_degrid */
enum {
    IMAGER_REUSE_INDEX = 1u,        /* uvw / a_index / nvis unchanged since the previous grid or degrid call on this
                                       plan: skip indexing and bucketing (the steady state of a major-cycle loop) */
    IMAGER_PATH_REFERENCE = 2u,     /* use the simple one-warp-per-visibility kernels instead of the tiled ones
                                       (same results up to summation order; for tests and A/B timing)             */
    IMAGER_DEGRID_RESIDUAL = 16u    /* imager_degrid: vis_out holds the observed visibilities on entry and the
                                       residuals V - V_model on return (the major-cycle update), fused into
                                       the kernel's epilogue; dropped visibilities are left as they are           */
};

typedef struct imager_plan imager_plan;   /* opaque, owned by the library */

/* Plain data, copied at imager_plan_create; the caller may free it (and what it points to) afterwards. */
typedef struct imager_params {
    int32_t grid_size;        /* N (even): grids are [n_pol][N][N] complex64, row-major, u = v = 0 at cell (N/2, N/2)  */
    int32_t n_corr;           /* 1 or 4 correlations per visibility, order XX*, XY*, YX*, YY*                   */
    int32_t n_pol;            /* 1 or 4 output grids, order I, Q, U, V (Eq. 4-5)                             */
    int32_t n_wplanes;        /* P >= 1 planes in |w| from 0 to w_max ("configurable number of w-planes"; R4)    */
    int32_t support_min;      /* taps per side on plane 0                                                              */
    int32_t support_max;      /* taps per side on plane P-1; S_p per R5; (support_max - support_min) must be even     */
    int32_t oversample;       /* O sub-cells per cell (even, or 1)                                                     */
    int32_t n_aplanes;        /* A-planes: parallactic-angle bins or mosaic pointings (P:90 averaging; R12); >= 1     */
    int32_t kernel_mode;      /* IMAGER_MODE_*                                                                         */
    int32_t pswf_support;     /* S_ps of the anti-aliasing function psi = S00(pi S_ps / 2, eta); 0 means 7            */
    double cell_size_rad;     /* image cell in radians; the uv cell is 1 / (N * cell) wavelengths                      */
    double w_max;             /* wavelengths; ignored if P == 1                                                        */
    double dish_diameter_m;   /* Airy beam E = 2 J1(x)/x, x = pi D rho / lambda (AWPROJ_*, MOSAIC_PB)                  */
    double freq_hz;           /* frequency the beam is evaluated at                                                    */
    double leakage[4];        /* d1.re, d1.im, d2.re, d2.im of D = [[1, d1], [d2, 1]] (AWPROJ_*)                       */
    double beam_eps;          /* epsilon of Eq. 6, AWPROJ_PAPER only; 0 means 0.2                              */
    const double* pa_rad;     /* host [n_aplanes] parallactic angle per A-plane (AWPROJ_*), or NULL = zeros           */
    const double* pointing_lm;/* host [n_aplanes][2] pointing offsets (l, m) in radians (MOSAIC_PB), or NULL = zeros  */
    const float* user_tables;        /* host, USER mode: gridding tables, complex64 interleaved, the sets
                                        kset = a*(2P-1) + (sp+P-1) back to back, each [n_pol][n_corr][O][O][S][S]     */
    const float* user_tables_degrid; /* host, USER mode: degridding tables in the same layout, or NULL = same tables  */
    int64_t max_nvis;         /* scratch is sized for this many visibilities per call                                  */
} imager_params;

/* 16-byte index record of one visibility (R2-R5, R8); exported by imager_debug_index, compared bit-exactly
 * with the oracle. */
typedef struct imager_record {
    int32_t gx, gy;           /* grid cell of the visibility (may lie outside the grid if dropped)                     */
    uint32_t sub;             /* (ox + O/2) | (oy + O/2) << 8 | drop << 16                                             */
    int32_t kset;             /* kernel set a*(2P-1) + (sp + P-1)                                                      */
} imager_record;

/* Create a plan: validates params, builds the kernel tables on the device (or uploads USER tables) and
 * allocates scratch for max_nvis visibilities.  Synchronises cuda_stream before returning.
 * Errors: INVALID_ARG (bad sizes, NULL), UNSUPPORTED (mode / shape combination not built), NOMEM, CUDA. */
int imager_plan_create(const imager_params* params, void* cuda_stream, imager_plan** out_plan);

/* Steps A1 + A2 on their own: index and bucket (uvw, a_index) and plan the work lists of the gridding / degridding
 * kernels, so that later imager_grid / imager_degrid calls with IMAGER_REUSE_INDEX start at once (e.g. while the
 * visibilities are still being copied to the device).  uvw dev float32 [nvis][3], a_index dev int32 [nvis] or NULL.
 * Synchronises the stream once (the list sizes are read back).  Errors: INVALID_ARG, TOO_MANY_VIS (nvis > max_nvis or
 * 2^31 hits or more), NOMEM, CUDA. */
int imager_index(imager_plan* plan, int64_t nvis, const float* uvw, const int32_t* a_index, void* cuda_stream);

/* Gridding.  Accumulates into `grid` (the caller zeroes it); visibilities whose footprint leaves the
 * grid are skipped and counted (R8), and so are invalid ones (R17: u, v or w not finite or beyond 2^30 fine cells,
 * a_index outside [0, n_aplanes)): nothing is ever indexed from them.  uvw dev float32 [nvis][3] in wavelengths ("baseline vectors ... in
 * units of wavelength"); vis dev complex64 [nvis][n_corr]; weights dev float32 [nvis][n_corr]; a_index dev
 * int32 [nvis] in [0, n_aplanes) or NULL (= 0); grid dev complex64 [n_pol][N][N]; sum_weights dev double
 * [n_corr] or NULL, accumulated with the weights of the kept visibilities.
 * Errors: INVALID_ARG, TOO_MANY_VIS (nvis > max_nvis), CUDA. */
int imager_grid(imager_plan* plan, int64_t nvis, const float* uvw, const float* vis, const float* weights,
                const int32_t* a_index, float* grid, double* sum_weights, uint32_t flags, void* cuda_stream);

/* Degridding: predicts vis_out dev complex64 [nvis][n_corr] (overwritten, input order) from grid dev
 * complex64 [n_pol][N][N]; dropped visibilities predict 0.  Weights play no part.  With IMAGER_DEGRID_RESIDUAL the
 * prediction is subtracted from what vis_out holds instead (vis_out := vis_out - V_model). */
int imager_degrid(imager_plan* plan, int64_t nvis, const float* uvw, const int32_t* a_index, const float* grid,
                  float* vis_out, uint32_t flags, void* cuda_stream);

/* Destroy a plan and free everything it owns.  NULL is a no-op. */
int imager_plan_destroy(imager_plan* plan);

/* ---- surrounding stages, built but outside the timed hot path (BASELINE.json north_star item 3) ---- */

/* (The survey's proposed `imager_taper_correct` lives inside this call: the division by psi psi is fused with the
 * centring sign flips around the cuFFT transform.)
 * direction = +1: grid -> image: centred forward DFT (cuFFT) of each [N][N] plane in place, then divide by
 * psi(l) psi(m) and by norm (pass the sum of weights; 0 means 1).  direction = -1: image -> grid: divide by
 * psi psi, then the centred unnormalised inverse DFT (R1: signs follow Eq. 2).  data dev complex64. */
int imager_grid_image_transform(imager_plan* plan, float* data, int32_t direction, double norm, void* cuda_stream);

/* UV-domain mosaic weighting correction, Eq. 1: multiplies every [N][N] plane of `image` (dev complex64
 * [n_pol][N][N], pixel (N/2, N/2) at l = m = 0, the output of imager_grid_image_transform(+1)) in place by
 * gamma(l,m) = [sqrt(sum_i B_i^2) / max sqrt(sum_i B_i^2)] * [1 / sum_i B_i^2], B_i(l,m) = E^2(l - l_i, m - m_i) the
 * power beam of pointing i (the gridding kernel of MOSAIC_PB mode; E the Airy pattern of dish_diameter_m at freq_hz).
 * gamma is built on the device at the first call and cached in the plan.  Errors: INVALID_ARG (NULL, plan not in
 * MOSAIC_PB mode), NOMEM, CUDA. */
int imager_mosaic_correct(imager_plan* plan, float* image, void* cuda_stream);

/* ---- the loop around the hot path: minor cycle and Cotton-Schwab major cycles ---- */

/* Hogbom minor cycle (R18, R19) on device images, all float32 [n][n] row-major: `residual` is updated in
 * place, `psf` has its peak (1) at pixel (n/2, n/2), the components found are ADDED to `model`.  window = {y0, x0, y1, x1}
 * (half-open) limits the peak search.  Repeats up to n_iter times: p = first pixel (row-major) of the window with the
 * largest |residual|; stop if |residual[p]| < max(threshold, cycle_factor * sidelobe * |first peak|), sidelobe = the largest
 * |psf| outside the 3 x 3 pixels at its centre; a = gain * residual[p]; model[p] += a; residual[q] -= a * psf[q - p + c]
 * wherever that psf sample exists.  Each step is one IEEE float32 operation (no fused multiply-add), so that peak positions
 * and component values are reproducible bit for bit.  components_out dev float32 [n_iter][3] = (y, x, a) in the order
 * found, or NULL; n_components_out dev int32 [1] or NULL.  Enqueues 2 n_iter + 3 kernels on cuda_stream (one more with
 * n_components_out) whatever happens: the stop test is taken on the device, and once it has fired the launches still queued
 * return at once (a few microseconds each: choose n_iter as a bound, not as a wish); nothing is read back and nothing synchronises.  Errors: INVALID_ARG, NOMEM, CUDA. */
int imager_hogbom(float* residual, const float* psf, float* model, int32_t n, const int32_t window[4], float gain,
                  float threshold, float cycle_factor, int32_t n_iter, float* components_out, int32_t* n_components_out,
                  void* cuda_stream);

/* The same minor cycle for callers that must not allocate device memory.  imager_hogbom above takes three small scratch
 * buffers from the stream-ordered pool (cudaMallocAsync / cudaFreeAsync) on every call.  Some users of this library cannot
 * do that: a pipeline that shares one GPU with a correlator or beamformer and had all of its HBM handed out at start-up, a
 * process in which a framework's caching allocator already owns the device, a real-time loop that cannot take the
 * allocator's locks, pool growth or the device-wide wait that cudaMalloc / cudaFree can cause.  This entry point calls no
 * cudaMalloc, cudaMallocAsync, cudaFree or any library routine that allocates; its scratch is an array built into
 * libimager.so (file-scope `static __device__` in csrc/clean.cu): 131,328 bytes (256 of control block + 16384 per-block peak
 * records of 8 bytes), held by EVERY GPU that loads the library from the moment it is loaded until the process exits,
 * used or not.  The caller still passes every input and output.
 *   - Arguments, arithmetic, results and stream behaviour are those of imager_hogbom: residual / model / components are
 *     bit-identical between the two calls.  Enqueues 2 n_iter + 5 kernels, never synchronises.
 *   - Limit: n <= IMAGER_HOGBOM_STATIC_MAX_N (the scratch holds one peak record per 1024 pixels of a 4096 x 4096 image).
 *     A larger n is refused with IMAGER_ERR_UNSUPPORTED and a message naming the limit; nothing is enqueued.
 *   - Set-up: the FIRST call on each device (with that device current) looks up the array's device address
 *     (cudaGetSymbolAddress, return code checked; the first use may also make the CUDA runtime load the library's module
 *     on that device) and keeps it for later calls on that device.  Make that first call ahead of time: before any stream
 *     capture is begun, and outside whatever section of the caller's loop may not make such runtime calls.
 *   - One array per GPU, shared by every call in the process.  It keeps the previous call's contents; the entry point
 *     rewrites what has to start from zero (the control block) at the head of its own work queue, so back-to-back calls on
 *     ONE stream are fine.  Two calls whose kernels can overlap on the same GPU (different streams without an ordering
 *     event, different host threads) RACE on the array and give wrong results: order them, or use imager_hogbom for all
 *     but one of them.
 * Errors: INVALID_ARG (NULL, n < 2), UNSUPPORTED (n beyond the limit; device ordinal >= 64), CUDA. */
#define IMAGER_HOGBOM_STATIC_MAX_N 4096
int imager_hogbom_static(float* residual, const float* psf, float* model, int32_t n, const int32_t window[4], float gain,
                         float threshold, float cycle_factor, int32_t n_iter, float* components_out,
                         int32_t* n_components_out, void* cuda_stream);

typedef struct imager_clean_params {
    int32_t n_major;          /* major (Cotton-Schwab) cycles, >= 1 ("number of clean cycles")                      */
    int32_t n_iter;           /* minor-cycle iterations per major cycle                                                    */
    float gain;               /* loop gain                                                                          */
    float threshold;          /* stop level in image units                                                          */
    float cycle_factor;       /* R19: a minor cycle ends at cycle_factor * PSF sidelobe * its first peak            */
} imager_clean_params;

/* Cotton-Schwab loop (R20) for single-polarisation plans: indexes (uvw, a_index) once, forms the PSF as the
 * dirty image of unit visibilities, then n_major times: grids the residual visibilities (imager_grid, index reused),
 * transforms (cuFFT + taper), runs the minor cycle inside the inner half of the field, transforms the accumulated model
 * back and subtracts its prediction from the observed visibilities (imager_degrid with IMAGER_DEGRID_RESIDUAL).
 * vis, weights dev [nvis]; model_image dev float32 [N][N] (overwritten: the clean components); residual_image dev float32
 * [N][N] (the last cycle's image after its minor cycle); residual_vis dev complex64 [nvis] (V - V_model after the last
 * cycle); psf_out dev float32 [N][N] or NULL; n_components_out dev int32 [n_major] or NULL.  Synchronises once (the
 * indexing step); everything else is enqueued.  Errors: INVALID_ARG, UNSUPPORTED (n_pol != 1), TOO_MANY_VIS, NOMEM, CUDA. */
int imager_clean(imager_plan* plan, int64_t nvis, const float* uvw, const float* vis, const float* weights,
                 const int32_t* a_index, const imager_clean_params* params, float* model_image, float* residual_image,
                 float* residual_vis, float* psf_out, int32_t* n_components_out, void* cuda_stream);

/* ---- image-domain mosaic (R21-R23) ---- */

/* Image-plane reprojection (R22): dst(l, m) (+)= B * bilinear(src at (l - shift_l, m - shift_m)), zero outside the source.
 * src dev complex64 [n_src][n_src] with cell cell_src, dst dev complex64 [n_dst][n_dst] with cell cell_dst (radians), pixel
 * (n/2, n/2) the origin of either frame, l along the last axis.  beam: 0 none, 1 = Airy power beam E^2 (dish_diameter_m,
 * freq_hz) centred on the SOURCE frame (forward: component -> mosaic), 2 = centred on the TARGET frame (backward: model ->
 * component).  inner_half != 0: only source pixels n/4 <= x, y < 3n/4 count.  accumulate != 0 adds to dst.  Enqueues one
 * kernel.  Errors: INVALID_ARG, CUDA. */
int imager_reproject(const float* src, int32_t n_src, double cell_src, float* dst, int32_t n_dst, double cell_dst,
                     double shift_l, double shift_m, int32_t beam, double dish_diameter_m, double freq_hz, int32_t inner_half,
                     int32_t accumulate, void* cuda_stream);

/* Image-domain mosaic, forward (R23): every component i = 0 .. n_point-1 (visibilities referred to ITS OWN phase
 * centre) is gridded on the plan's grid (imager_grid: index + bucket + grid), transformed (cuFFT + taper), weighted by the
 * Airy power beam of the plan (dish_diameter_m, freq_hz) and reprojected to the mosaic frame at offset pointing_lm[i];
 * mosaic_image = sum_i w_i B_i reproject_i[I_i], w_i = component i's sum of weights / the total.  `plan`: single
 * polarisation, one A-plane, kernel mode PSWF, WPROJ, DELTA or USER tables of that kind (a MOSAIC_PB or AWPROJ_* plan is refused
 * with UNSUPPORTED: its kernels already hold the beam, which this call applies in the image plane).  nvis host [n_point]; uvw, vis, weights host arrays of n_point DEVICE
 * pointers ([nvis_i][3] float32, [nvis_i] complex64, [nvis_i] float32); pointing_lm host [n_point][2] radians;
 * mosaic_image dev complex64 [n_mosaic][n_mosaic] (OVERWRITTEN), cell_mosaic radians; sum_weights dev double [1] or NULL
 * (the total).  Synchronises once per component (its indexing step).  Errors: INVALID_ARG, UNSUPPORTED, TOO_MANY_VIS
 * (a component larger than max_nvis), NOMEM, CUDA. */
int imager_mosaic_grid(imager_plan* plan, int32_t n_point, const int64_t* nvis, const float* const* uvw,
                       const float* const* vis, const float* const* weights, const double* pointing_lm, float* mosaic_image,
                       int32_t n_mosaic, double cell_mosaic, double* sum_weights, void* cuda_stream);

/* Image-domain mosaic, backward ("the model image is reprojected to the phase position of each mosaic component, and
 * multiple FFT and degridding steps are performed"): per component, model_image is reprojected to the component frame,
 * multiplied by the beam, transformed to the grid (taper + cuFFT) and degridded at the component's uvw into vis_out[i]
 * (dev complex64 [nvis_i]; flags: 0 or IMAGER_DEGRID_RESIDUAL).  Arguments as imager_mosaic_grid. */
int imager_mosaic_degrid(imager_plan* plan, int32_t n_point, const int64_t* nvis, const float* const* uvw,
                         const double* pointing_lm, const float* model_image, int32_t n_mosaic, double cell_mosaic,
                         float* const* vis_out, uint32_t flags, void* cuda_stream);

/* ---- test / debug exports (synchronise; not part of the hot path) ---- */

/* Runs indexing + bucketing for (uvw, a_index) and copies out: records host [nvis], perm host int32 [nvis]
 * (sorted position -> input index, stable), sorted keys host uint32 [nvis], bucket_offset host int32
 * [n_buckets + 1] (see imager_plan_info), n_kept.  Any output pointer may be NULL. */
int imager_debug_index(imager_plan* plan, int64_t nvis, const float* uvw, const int32_t* a_index,
                       imager_record* records_out, int32_t* perm_out, uint32_t* keys_out,
                       int32_t* bucket_offset_out, int64_t* n_kept_out, void* cuda_stream);

/* Copies kernel set `kset` (gridding tables if which == 0, degridding if 1) to host_out in the canonical
 * layout [n_pol][n_corr][O][O][S][S] complex64 and writes its support S.  host_out may be NULL (size query). */
int imager_debug_kernels(imager_plan* plan, int32_t kset, int32_t which, float* host_out, int32_t* support_out);

/* info: [0] n_sets, [1] bucket tile size, [2] n_buckets, [3] key bits, [4] dropped visibilities of the last
 * indexing, [5] GPU kernel launches issued by the last imager_grid / imager_degrid call, [6] complex elements of one
 * table set collection, [7] kept visibilities of the last indexing.  [4] and [7] are read back after waiting for the
 * last indexing of this plan (an event recorded behind it on the stream it ran on, non-blocking streams included); no
 * device-wide synchronisation. */
int imager_plan_info(imager_plan* plan, int64_t info_out[8]);

/* Which kernels imager_grid / imager_degrid will run for this plan (without IMAGER_PATH_REFERENCE): returns 1 for the tiled
 * kernels (the fast path every number in bench.py is about), 0 for the one-warp-per-visibility reference kernels -- the
 * library falls back to them, with the same results and several times the run time, for shapes the tiled kernels are not
 * built for -- and then writes the reason into why_out (host char [why_len], NUL-terminated, "" when tiled; may be NULL
 * with why_len 0).  Fixed at plan creation; no device work, no synchronisation.  < 0 on error (INVALID_ARG). */
int imager_plan_path(imager_plan* plan, char* why_out, int32_t why_len);

/* Statistics of the current index (built by the last imager_index / imager_grid / imager_degrid / imager_debug_index
 * call); synchronises cuda_stream.  out[0] kept visibilities, [1] dropped ones, [2] duplicates merged into another
 * visibility of the same (kernel set, cell, sub-cell) (pre-summed: exact algebra, R16), [3] nominal complex
 * multiply-accumulates of one gridding (= one degridding) pass, n_corr n_pol sum over kept visibilities of S^2,
 * [4] the complex multiply-accumulates the tiled kernels execute (merged duplicates excluded), [5] hits (visibility x
 * 16 x 32 strip pairs) and [6] work items of the tiled plan (0 before it is built), [7] 0.
 * Errors: INVALID_ARG (NULL, no index yet), CUDA. */
int imager_index_stats(imager_plan* plan, int64_t out[8], void* cuda_stream);

/* Number of GPU kernels the last imager_grid / imager_degrid / imager_debug_index call on this plan launched
 * (host-side counter, no synchronisation); negative status on a NULL plan. */
int imager_last_launch_count(imager_plan* plan);

/* Self-checks of a CHECKED build (libimager_checked.so, compiled with -DIMAGER_CHECKED=1: every index the planner and the
 * tiled kernels form -- hit-record places, visibility indices, shared-memory tap addresses, strips, work items -- is
 * tested against its bounds on the device and violations are counted instead of being dereferenced blindly; the pool's
 * compute-sanitizer is closed).  out[k], k = 0..15: violations of check k since the library was
 * loaded (k: 0 hit place, 1 visibility index of a hit, 2 tap address, 3 strip, 4 item range, 5 block range, 6 hash
 * table, 7 window strip).  Returns 1 for a checked build, 0 for the normal build (out is zeroed), < 0 on error.
 * Synchronises the device. */
int imager_debug_violations(int64_t out[16]);

/* Micro-benchmarks of the two SM units that bound the gridding / degridding kernels, so that the numbers
 * the design and bench.py's `lsu_floor_ms` rest on can be re-measured: out[0] clocks per warp-wide LDS.64 instruction per
 * SM with all 32 lanes active, out[1] the same with 16 lanes active, out[2] clocks per warp-wide FFMA2 (fma.rn.f32x2)
 * instruction per SM, out[3] the SM count.  Allocates and frees 4 KB of device memory, launches six small kernels (one
 * 1024-thread CTA per SM, a few hundred microseconds), synchronises cuda_stream.  Errors: INVALID_ARG, NOMEM, CUDA. */
int imager_debug_probe(double out[4], void* cuda_stream);

/* Thread-local message of the last failing call on this thread ("" if none); valid until the next call. */
const char* imager_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* IMAGER_H_ */
