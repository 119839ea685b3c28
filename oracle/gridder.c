/* CPU ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE (see oracle/__init__.py).
 *
 * Steps O4 (gridding) and O5 (degridding) of DESIGN.md, i.e. textbook convolutional gridding with an
 * oversampled lookup table, which is what PAPER.md:86-88 and :110 name without writing out:
 *
 *   O4  for k in input order, not dropped:  val_c = w_kc * V_kc
 *         G[s][gy+dy][gx+dx] += sum_c T[kset_k][s][c][oy][ox][dy][dx] * val_c      (complex128 accumulation)
 *         A[s][gy+dy][gx+dx] += sum_c |T| * |val_c|                                  (parity normaliser)
 *         sumwt[c] += w_kc                                                         (kept visibilities only)
 *   O5  V_kc = sum_s sum_{dy,dx} conj(T[kset_k][s][c][oy][ox][dy][dx]) * G[s][gy+dy][gx+dx],
 *         B_kc = sum |T| * |G|;  dropped visibilities predict 0.
 *
 * Plain C, no intrinsics, no blocking.  OpenMP only splits the OUTPUT (row bands of the grid for O4, visibilities
 * for O5), so every output element is still accumulated in input order by exactly one thread: deterministic.
 * Tables are complex64 (as a GPU holds them), promoted to double before any arithmetic.
 */
#include <stdint.h>
#include <stdlib.h>
#include <math.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* table element (s, c, oy_idx, ox_idx, dy_idx, dx_idx) of a set with support S, oversampling O */
static inline int64_t tap_index(int n_corr, int O, int S, int s, int c, int oy, int ox, int dy, int dx) {
    return (((((int64_t)s * n_corr + c) * O + oy) * O + ox) * S + dy) * S + dx;
}

/* Reading R24 (extends R9 "omega = 0 contributes 0"): sample j = (visibility, correlation) is FLAGGED when its
 * weight is zero or its weight or value is not finite; a flagged sample contributes (0, 0) and no weight. */
static int sample_flagged(const float* weights, const float* vis, int64_t j) {
    return weights[j] == 0.0f || !isfinite(weights[j]) || !isfinite(vis[2 * j]) || !isfinite(vis[2 * j + 1]);
}

/* O4.  grid, norm: [n_pol][N][N] (grid as interleaved re,im doubles), accumulated into.
 * If sample_rowptr != NULL only the listed cells are computed: sample_rowptr[N+1] is a CSR over rows of
 * sample_x (sorted), and outputs are written to sample_out[n_pol][n_samples] (re,im) / sample_norm instead. */
int oracle_grid(int64_t nvis, int N, int n_corr, int n_pol, int O,
                const int64_t* gx, const int64_t* gy, const int64_t* ox, const int64_t* oy,
                const int64_t* kset, const int64_t* support, const uint8_t* drop,
                const float* vis, const float* weights,
                const float* tables, const int64_t* table_offset,
                double* grid, double* norm, double* sumwt,
                const int64_t* sample_rowptr, const int64_t* sample_x, int64_t n_samples,
                double* sample_out, double* sample_norm, int n_threads) {
    if (n_threads < 1) n_threads = 1;
    const int half_o = O / 2;
#pragma omp parallel num_threads(n_threads)
    {
#ifdef _OPENMP
        const int tid = omp_get_thread_num(), nt = omp_get_num_threads();
#else
        const int tid = 0, nt = 1;
#endif
        const int64_t row0 = (int64_t)N * tid / nt, row1 = (int64_t)N * (tid + 1) / nt;
        for (int64_t k = 0; k < nvis; ++k) {
            if (drop[k]) continue;
            const int S = (int)support[k], h_lo = S / 2;
            const int64_t y_lo = gy[k] - h_lo, y_hi = y_lo + S;      /* rows [y_lo, y_hi) */
            if (y_hi <= row0 || y_lo >= row1) continue;
            const float* T = tables + 2 * table_offset[kset[k]];
            const int oyi = (int)oy[k] + half_o, oxi = (int)ox[k] + half_o;
            double vr[4], vi[4], va[4];
            for (int c = 0; c < n_corr; ++c) {
                const double w = (double)weights[k * n_corr + c];
                vr[c] = w * (double)vis[2 * (k * n_corr + c)];
                vi[c] = w * (double)vis[2 * (k * n_corr + c) + 1];
                if (sample_flagged(weights, vis, k * n_corr + c)) vr[c] = vi[c] = 0.0;   /* R24 */
                va[c] = hypot(vr[c], vi[c]);
            }
            for (int dy = 0; dy < S; ++dy) {
                const int64_t y = y_lo + dy;
                if (y < row0 || y >= row1) continue;
                if (sample_rowptr) {
                    for (int64_t j = sample_rowptr[y]; j < sample_rowptr[y + 1]; ++j) {
                        const int64_t dx = sample_x[j] - (gx[k] - h_lo);
                        if (dx < 0 || dx >= S) continue;
                        for (int s = 0; s < n_pol; ++s) {
                            double ar = 0, ai = 0, an = 0;
                            for (int c = 0; c < n_corr; ++c) {
                                const int64_t t = tap_index(n_corr, O, S, s, c, oyi, oxi, dy, (int)dx);
                                const double tr = T[2 * t], ti = T[2 * t + 1];
                                ar += tr * vr[c] - ti * vi[c];
                                ai += tr * vi[c] + ti * vr[c];
                                an += hypot(tr, ti) * va[c];
                            }
                            sample_out[2 * (s * n_samples + j)] += ar;
                            sample_out[2 * (s * n_samples + j) + 1] += ai;
                            sample_norm[s * n_samples + j] += an;
                        }
                    }
                    continue;
                }
                for (int dx = 0; dx < S; ++dx) {
                    const int64_t x = gx[k] - h_lo + dx;
                    for (int s = 0; s < n_pol; ++s) {
                        double ar = 0, ai = 0, an = 0;
                        for (int c = 0; c < n_corr; ++c) {
                            const int64_t t = tap_index(n_corr, O, S, s, c, oyi, oxi, dy, dx);
                            const double tr = T[2 * t], ti = T[2 * t + 1];
                            ar += tr * vr[c] - ti * vi[c];
                            ai += tr * vi[c] + ti * vr[c];
                            an += hypot(tr, ti) * va[c];
                        }
                        const int64_t cell = ((int64_t)s * N + y) * N + x;
                        grid[2 * cell] += ar;
                        grid[2 * cell + 1] += ai;
                        norm[cell] += an;
                    }
                }
            }
        }
    }
    for (int64_t k = 0; k < nvis; ++k)                              /* dropped visibilities carry no weight (R8) */
        if (!drop[k])
            for (int c = 0; c < n_corr; ++c)
                if (!sample_flagged(weights, vis, k * n_corr + c)) sumwt[c] += (double)weights[k * n_corr + c];   /* R24 */
    return 0;
}

/* O5.  grid: complex64 [n_pol][N][N] (what the GPU is given), promoted to double.
 * vis_out [nvis][n_corr] (re,im doubles), norm_out [nvis][n_corr]. */
int oracle_degrid(int64_t nvis, int N, int n_corr, int n_pol, int O,
                  const int64_t* gx, const int64_t* gy, const int64_t* ox, const int64_t* oy,
                  const int64_t* kset, const int64_t* support, const uint8_t* drop,
                  const float* grid, const float* tables, const int64_t* table_offset,
                  double* vis_out, double* norm_out, int n_threads) {
    if (n_threads < 1) n_threads = 1;
    const int half_o = O / 2;
#pragma omp parallel for schedule(static) num_threads(n_threads)
    for (int64_t k = 0; k < nvis; ++k) {
        for (int c = 0; c < n_corr; ++c) {
            vis_out[2 * (k * n_corr + c)] = vis_out[2 * (k * n_corr + c) + 1] = 0.0;
            norm_out[k * n_corr + c] = 0.0;
        }
        if (drop[k]) continue;
        const int S = (int)support[k], h_lo = S / 2;
        const float* T = tables + 2 * table_offset[kset[k]];
        const int oyi = (int)oy[k] + half_o, oxi = (int)ox[k] + half_o;
        for (int c = 0; c < n_corr; ++c) {
            double ar = 0, ai = 0, an = 0;
            for (int s = 0; s < n_pol; ++s)
                for (int dy = 0; dy < S; ++dy)
                    for (int dx = 0; dx < S; ++dx) {
                        const int64_t t = tap_index(n_corr, O, S, s, c, oyi, oxi, dy, dx);
                        const double tr = T[2 * t], ti = -(double)T[2 * t + 1];        /* conj(T) */
                        const int64_t cell = ((int64_t)s * N + (gy[k] - h_lo + dy)) * N + (gx[k] - h_lo + dx);
                        const double gr = grid[2 * cell], gi = grid[2 * cell + 1];
                        ar += tr * gr - ti * gi;
                        ai += tr * gi + ti * gr;
                        an += hypot(tr, ti) * hypot(gr, gi);
                    }
            vis_out[2 * (k * n_corr + c)] = ar;
            vis_out[2 * (k * n_corr + c) + 1] = ai;
            norm_out[k * n_corr + c] = an;
        }
    }
    return 0;
}
