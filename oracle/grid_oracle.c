/* O4 — convolutional gridding oracle, G1-G7 (TEST INFRASTRUCTURE ONLY).
 *
 * Plain fp64 C loops written from the definition in SURVEY.md §8(c) O4 /
 * DESIGN.md; shares no code with the CUDA path.  What is gridded: PAPER.md:30
 * (each visibility is convolved with the w-dependent kernel and projected on
 * a 2-D plane), PAPER.md:80, 84 (one contribution per support cell, S x S per
 * visibility, accumulated into the uv-grid), PAPER.md:56 (row x channel data).
 *
 * G1  f = freq[c]/c0; u = uvw[r][0] f; v = uvw[r][1] f; w = uvw[r][2] f
 * G2  p = clamp(floor((w + w_max)/dw), 0, Nw-1),  dw = 2 w_max / Nw
 * G3  x = u/du + N/2; X = floor(x Q + 0.5); Y = X - (S-2) Q/2;
 *     j0 = floor_div(Y, Q); o = Y - j0 Q          (same for v)
 * G4  window outside the grid -> skipped and counted, no wrap-around
 * G5  grid[j0v+iv][j0u+iu] += (weight vis) K[p][ov][ou][iv][iu]
 * G6  G1-G3 in IEEE fp64 in exactly this order, no FMA contraction
 *     (compile with -ffp-contract=off)
 * G7  natural weights, one polarisation, every visibility gridded once.
 *
 * The OpenMP mode models the paper's CPU method: static
 * split of the rows over threads, a private grid per thread, then a sum.
 * Complex arithmetic is written out in real form.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC grid_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define C0 299792458.0

typedef struct {
    int64_t n_gridded, n_skipped_oob, n_skipped_zero_weight, n_clamped_w, n_updates;
} oracle_stats;

/* floor division for a possibly negative numerator, positive denominator */
static int64_t floor_div(int64_t a, int64_t b) {
    int64_t q = a / b;
    if ((a % b != 0) && (a < 0)) q -= 1;
    return q;
}

/* G3 for one axis.  x_lambda is the coordinate in wavelengths. */
void oracle_index_map(double x_lambda, int N, double cell, int S, int Q,
                      int64_t *j0, int *o) {
    double fov = (double)N * cell;
    double du = 1.0 / fov;
    double x = x_lambda / du + (double)(N / 2);
    int64_t X = (int64_t)floor(x * (double)Q + 0.5);
    int64_t Y = X - (int64_t)((S - 2) * Q / 2);
    *j0 = floor_div(Y, Q);
    *o = (int)(Y - (*j0) * Q);
}

/* G2.  *clamped is set when |w| > w_max. */
int oracle_plane(double w, double w_max, int Nw, int *clamped) {
    *clamped = fabs(w) > w_max;
    double dw = 2.0 * w_max / (double)Nw;
    if (!(dw > 0.0)) return 0;               /* w_max = 0: single w value, plane 0 */
    double fp = floor((w + w_max) / dw);
    if (fp < 0.0) return 0;
    if (fp > (double)(Nw - 1)) return Nw - 1;
    return (int)fp;
}

static void grid_rows(const double *uvw, const float *vis, const float *weight,
                      const double *freq, int64_t row0, int64_t row1, int nchan,
                      const double *K, const int *support, const int64_t *plane_offset,
                      int Nw, int Q, int N, double cell, double w_max,
                      double *grid, oracle_stats *st) {
    for (int64_t r = row0; r < row1; ++r) {
        for (int c = 0; c < nchan; ++c) {
            double wt = (double)weight[r * nchan + c];
            if (wt == 0.0) { st->n_skipped_zero_weight++; continue; }
            double f = freq[c] / C0;                                    /* G1 */
            double u = uvw[3 * r + 0] * f;
            double v = uvw[3 * r + 1] * f;
            double w = uvw[3 * r + 2] * f;
            int clamped;
            int p = oracle_plane(w, w_max, Nw, &clamped);               /* G2 */
            int S = support[p];
            int64_t j0u, j0v; int ou, ov;
            oracle_index_map(u, N, cell, S, Q, &j0u, &ou);              /* G3 */
            oracle_index_map(v, N, cell, S, Q, &j0v, &ov);
            if (j0u < 0 || j0v < 0 || j0u + S > N || j0v + S > N) {     /* G4 */
                st->n_skipped_oob++; continue;
            }
            if (clamped) st->n_clamped_w++;
            double vr = wt * (double)vis[2 * (r * nchan + c) + 0];
            double vi = wt * (double)vis[2 * (r * nchan + c) + 1];
            const double *Ks = K + 2 * (plane_offset[p] + ((int64_t)ov * Q + ou) * S * S);
            for (int iv = 0; iv < S; ++iv) {                            /* G5 */
                double *g = grid + 2 * ((j0v + iv) * (int64_t)N + j0u);
                const double *k = Ks + 2 * (int64_t)iv * S;
                for (int iu = 0; iu < S; ++iu) {
                    double kr = k[2 * iu], ki = k[2 * iu + 1];
                    g[2 * iu]     += vr * kr - vi * ki;
                    g[2 * iu + 1] += vr * ki + vi * kr;
                }
            }
            st->n_gridded++;
            st->n_updates += (int64_t)S * S;
        }
    }
}

/* grid is ACCUMULATED INTO (caller zeroes).  stats_out: 5 int64.  nthreads<=1: serial. */
int oracle_grid(const double *uvw, const float *vis, const float *weight, const double *freq,
                int64_t nrow, int nchan, const double *K, const int *support,
                const int64_t *plane_offset, int Nw, int Q, int N, double cell, double w_max,
                double *grid, int64_t *stats_out, int nthreads) {
    oracle_stats tot; memset(&tot, 0, sizeof tot);
    if (nthreads <= 1) {
        grid_rows(uvw, vis, weight, freq, 0, nrow, nchan, K, support, plane_offset,
                  Nw, Q, N, cell, w_max, grid, &tot);
    } else {
#ifdef _OPENMP
        int64_t gsz = 2 * (int64_t)N * N;
        double **priv = (double **)calloc((size_t)nthreads, sizeof(double *));
        oracle_stats *sts = (oracle_stats *)calloc((size_t)nthreads, sizeof(oracle_stats));
        if (!priv || !sts) return -1;
        int fail = 0;
#pragma omp parallel num_threads(nthreads)
        {
            int t = omp_get_thread_num();
            int nt = omp_get_num_threads();
            priv[t] = (double *)calloc((size_t)gsz, sizeof(double));
            if (!priv[t]) {
#pragma omp atomic write
                fail = 1;
            } else {
                int64_t r0 = nrow * t / nt, r1 = nrow * (t + 1) / nt;   /* static row split */
                grid_rows(uvw, vis, weight, freq, r0, r1, nchan, K, support, plane_offset,
                          Nw, Q, N, cell, w_max, priv[t], &sts[t]);
            }
#pragma omp barrier
            if (!fail) {
#pragma omp for schedule(static)
                for (int64_t i = 0; i < gsz; ++i) {                     /* sum of sub-grids */
                    double s = 0.0;
                    for (int k = 0; k < nt; ++k) s += priv[k][i];
                    grid[i] += s;
                }
            }
        }
        for (int t = 0; t < nthreads; ++t) {
            tot.n_gridded += sts[t].n_gridded;
            tot.n_skipped_oob += sts[t].n_skipped_oob;
            tot.n_skipped_zero_weight += sts[t].n_skipped_zero_weight;
            tot.n_clamped_w += sts[t].n_clamped_w;
            tot.n_updates += sts[t].n_updates;
            free(priv[t]);
        }
        free(priv); free(sts);
        if (fail) return -1;
#else
        return -2;
#endif
    }
    stats_out[0] = tot.n_gridded; stats_out[1] = tot.n_skipped_oob;
    stats_out[2] = tot.n_skipped_zero_weight; stats_out[3] = tot.n_clamped_w;
    stats_out[4] = tot.n_updates;
    return 0;
}

/* Degridding, the adjoint of oracle_grid with unit weights (PAPER.md:36 names it as
 * the companion operation of gridding):
 *   vis[r][c] = sum_{iv,iu} grid[j0v+iv][j0u+iu] * conj(K[p][ov][ou][iv][iu])
 * with plane, window and sub-cell offsets exactly as in G1-G4; a visibility whose window is not fully inside the
 * grid is predicted as 0 (counted).  vis_out: complex128 pairs [nrow][nchan].  counts_out: {n_predicted, n_outside}. */
int oracle_degrid(const double *uvw, const double *freq, int64_t nrow, int nchan, const double *K,
                  const int *support, const int64_t *plane_offset, int Nw, int Q, int N, double cell,
                  double w_max, const double *grid, double *vis_out, int64_t *counts_out) {
    int64_t n_pred = 0, n_out = 0;
    for (int64_t r = 0; r < nrow; ++r) {
        for (int c = 0; c < nchan; ++c) {
            double f = freq[c] / C0;
            double u = uvw[3 * r + 0] * f, v = uvw[3 * r + 1] * f, w = uvw[3 * r + 2] * f;
            int clamped;
            int p = oracle_plane(w, w_max, Nw, &clamped);
            int S = support[p];
            int64_t j0u, j0v; int ou, ov;
            oracle_index_map(u, N, cell, S, Q, &j0u, &ou);
            oracle_index_map(v, N, cell, S, Q, &j0v, &ov);
            double sr = 0.0, si = 0.0;
            if (j0u < 0 || j0v < 0 || j0u + S > N || j0v + S > N) {
                n_out++;
            } else {
                const double *Ks = K + 2 * (plane_offset[p] + ((int64_t)ov * Q + ou) * S * S);
                for (int iv = 0; iv < S; ++iv) {
                    const double *g = grid + 2 * ((j0v + iv) * (int64_t)N + j0u);
                    const double *k = Ks + 2 * (int64_t)iv * S;
                    for (int iu = 0; iu < S; ++iu) {
                        double gr = g[2 * iu], gi = g[2 * iu + 1], kr = k[2 * iu], ki = k[2 * iu + 1];
                        sr += gr * kr + gi * ki;          /* g * conj(k) */
                        si += gi * kr - gr * ki;
                    }
                }
                n_pred++;
            }
            vis_out[2 * (r * nchan + c)] = sr;
            vis_out[2 * (r * nchan + c) + 1] = si;
        }
    }
    counts_out[0] = n_pred; counts_out[1] = n_out;
    return 0;
}

/* P11: flux conservation, evaluated WITHOUT a grid, in O(nvis):
 *   sum_cells grid            = sum_k wt_k V_k sigma [p_k][ov_k][ou_k],         sigma  = sum_{iv,iu} K
 *   sum_cells grid * ju       = sum_k wt_k V_k (j0u_k sigma + sigma_u),         sigma_u = sum_{iv,iu} iu K
 *   sum_cells grid * jv       = sum_k wt_k V_k (j0v_k sigma + sigma_v),         sigma_v = sum_{iv,iu} iv K
 * (the two first moments also pin WHERE the flux went: a window placed one cell off changes them).
 * The caller supplies the slice sums: sig[3 * s + {0,1,2}] complex (re, im pairs) for slice s = soff[p] + ov Q + ou,
 * soff[p] = p Q^2.  Plane, window and sub-cell offsets, validity and counters exactly as in grid_rows (G1-G4).
 * out: 8 doubles = {sum re, im; u-moment re, im; v-moment re, im; L1 = sum |wt V| |sigma|, 0}; stats_out: 5 int64. */
int oracle_flux(const double *uvw, const float *vis, const float *weight, const double *freq,
                int64_t nrow, int nchan, const double *sig, const int *support,
                int Nw, int Q, int N, double cell, double w_max,
                double *out, int64_t *stats_out, int nthreads) {
    double a0r = 0, a0i = 0, aur = 0, aui = 0, avr = 0, avi = 0, l1 = 0;
    int64_t ng = 0, noob = 0, nzero = 0, nclamp = 0, nupd = 0;
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for schedule(static) num_threads(nthreads) \
    reduction(+ : a0r, a0i, aur, aui, avr, avi, l1, ng, noob, nzero, nclamp, nupd)
    for (int64_t r = 0; r < nrow; ++r) {
        for (int c = 0; c < nchan; ++c) {
            double wt = (double)weight[r * nchan + c];
            if (wt == 0.0) { nzero++; continue; }
            double f = freq[c] / C0;
            double u = uvw[3 * r + 0] * f, v = uvw[3 * r + 1] * f, w = uvw[3 * r + 2] * f;
            int clamped;
            int p = oracle_plane(w, w_max, Nw, &clamped);
            int S = support[p];
            int64_t j0u, j0v; int ou, ov;
            oracle_index_map(u, N, cell, S, Q, &j0u, &ou);
            oracle_index_map(v, N, cell, S, Q, &j0v, &ov);
            if (j0u < 0 || j0v < 0 || j0u + S > N || j0v + S > N) { noob++; continue; }
            if (clamped) nclamp++;
            double vr = wt * (double)vis[2 * (r * nchan + c) + 0];
            double vi = wt * (double)vis[2 * (r * nchan + c) + 1];
            const double *sg = sig + 6 * (((int64_t)p * Q + ov) * Q + ou);
            double s0r = sg[0], s0i = sg[1];
            double sur = (double)j0u * s0r + sg[2], sui = (double)j0u * s0i + sg[3];
            double svr = (double)j0v * s0r + sg[4], svi = (double)j0v * s0i + sg[5];
            a0r += vr * s0r - vi * s0i; a0i += vr * s0i + vi * s0r;
            aur += vr * sur - vi * sui; aui += vr * sui + vi * sur;
            avr += vr * svr - vi * svi; avi += vr * svi + vi * svr;
            l1 += sqrt(vr * vr + vi * vi) * sqrt(s0r * s0r + s0i * s0i);
            ng++; nupd += (int64_t)S * S;
        }
    }
    out[0] = a0r; out[1] = a0i; out[2] = aur; out[3] = aui; out[4] = avr; out[5] = avi; out[6] = l1; out[7] = 0.0;
    stats_out[0] = ng; stats_out[1] = noob; stats_out[2] = nzero; stats_out[3] = nclamp; stats_out[4] = nupd;
    return 0;
}

/* The gridded value of single cells, one by one (G5 read as a gather; for checking full-size GPU runs on sampled
 * outputs): cell (cv[k], cu[k]) = sum over every visibility whose window covers it,
 *     j0v <= cv < j0v + S  and  j0u <= cu < j0u + S,
 * of wt V K[p][ov][ou][cv - j0v][cu - j0u].  Plane, window, sub-cell offsets and validity exactly as in grid_rows
 * (G1-G4): every visibility is tested against every requested cell, nothing cleverer.
 * out: 2 doubles per cell (re, im); l1_out: sum of |wt V| |K| per cell (the scale of its rounding error).
 * Threads split the rows; each sums into its own copy, the copies are added in thread order. */
int oracle_cells(const double *uvw, const float *vis, const float *weight, const double *freq,
                 int64_t nrow, int nchan, const double *K, const int *support, const int64_t *plane_offset,
                 int Nw, int Q, int N, double cell, double w_max,
                 const int *cu, const int *cv, int ncell, double *out, double *l1_out, int nthreads) {
    if (nthreads < 1) nthreads = 1;
    double *acc = (double *)calloc((size_t)nthreads * 3 * (size_t)(ncell > 0 ? ncell : 1), sizeof(double));
    if (!acc) return -1;
#pragma omp parallel num_threads(nthreads)
    {
#ifdef _OPENMP
        int t = omp_get_thread_num(), nt = omp_get_num_threads();
#else
        int t = 0, nt = 1;
#endif
        double *a = acc + (size_t)t * 3 * ncell;
        int64_t r0 = nrow * t / nt, r1 = nrow * (t + 1) / nt;
        for (int64_t r = r0; r < r1; ++r) {
            for (int c = 0; c < nchan; ++c) {
                double wt = (double)weight[r * nchan + c];
                if (wt == 0.0) continue;
                double f = freq[c] / C0;
                double u = uvw[3 * r + 0] * f, v = uvw[3 * r + 1] * f, w = uvw[3 * r + 2] * f;
                int clamped;
                int p = oracle_plane(w, w_max, Nw, &clamped);
                int S = support[p];
                int64_t j0u, j0v; int ou, ov;
                oracle_index_map(u, N, cell, S, Q, &j0u, &ou);
                oracle_index_map(v, N, cell, S, Q, &j0v, &ov);
                if (j0u < 0 || j0v < 0 || j0u + S > N || j0v + S > N) continue;
                double vr = wt * (double)vis[2 * (r * nchan + c) + 0];
                double vi = wt * (double)vis[2 * (r * nchan + c) + 1];
                const double *Ks = K + 2 * (plane_offset[p] + ((int64_t)ov * Q + ou) * S * S);
                for (int k = 0; k < ncell; ++k) {
                    int64_t iv = (int64_t)cv[k] - j0v, iu = (int64_t)cu[k] - j0u;
                    if (iv < 0 || iv >= S || iu < 0 || iu >= S) continue;
                    double kr = Ks[2 * (iv * S + iu)], ki = Ks[2 * (iv * S + iu) + 1];
                    a[3 * k]     += vr * kr - vi * ki;
                    a[3 * k + 1] += vr * ki + vi * kr;
                    a[3 * k + 2] += sqrt(vr * vr + vi * vi) * sqrt(kr * kr + ki * ki);
                }
            }
        }
    }
    for (int k = 0; k < ncell; ++k) {
        double sr = 0, si = 0, sl = 0;
        for (int t = 0; t < nthreads; ++t) {
            sr += acc[((size_t)t * ncell + k) * 3]; si += acc[((size_t)t * ncell + k) * 3 + 1]; sl += acc[((size_t)t * ncell + k) * 3 + 2];
        }
        out[2 * k] = sr; out[2 * k + 1] = si; l1_out[k] = sl;
    }
    free(acc);
    return 0;
}

int oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
