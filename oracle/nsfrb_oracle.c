/*
 * nsfrb_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, float64 CPU statement of what the NSFRB image-plane single-pulse
 * search computes (arxiv 2510.18136, "cerberus" search stage).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load this file.  It shares no code, header, table or constant with the CUDA path
 * (the csrc/ directory of the product package).
 *
 * What the paper fixes (PAPER.md = /root/reference/PAPER.md):
 *   - L73-L75 (sec. 2.2): images are de-dispersed over trial DMs with pre-computed
 *     per-channel shift indices, boxcar filtered over trial widths, "normalized by
 *     the running standard deviation to compute the S/N", and "final candidates are
 *     found by taking the maximum S/N (and its TOA) over time"; a S/N threshold
 *     identifies candidates.
 *   - L83 (sec. 2.2, text before Eq. 2): the dispersive delay across the band is
 *     (4.15 ms) DM (nu_min^-2 - nu_max^-2), nu in GHz  => constant 4.15e-3 s,
 *     reference = highest frequency.
 *   - L98 (footnote 12): the shifts are an integer lookup table; x5 DM at x5
 *     coarser sampling re-uses the same table.
 *   - L130 (sec. 3.2): the noise estimate is instantaneous and includes the pulse.
 *   - L146 (sec. 3.3): one candidate per searched time series.
 * Everything the paper leaves open follows the readings R1-R23 listed in DESIGN.md
 * (taken from SURVEY.md sec. 8(c)).  The steps below are labelled O1..O7 / S1..S6 as
 * there.
 *
 * Definition, per pixel p (cube I[c][t][p], float32, promoted to double on read):
 *   O1  f_ref = max_c f[c]
 *       x[k][c] = ((4.15e-3 * dm[k]) * (1/(f[c]*f[c]) - 1/(f_ref*f_ref))) / tsamp
 *       d[k][c] = (int) floor(x[k][c] + 0.5);  dmax_k = max_c d[k][c];  T_k = nt - dmax_k
 *   O2  D_k[t]  = sum_c I[c][t + d[k][c]][p],  0 <= t < T_k      (c = 0..nchan-1 in order)
 *   O3  mu_k = mean_t D_k[t];  var_k = mean_t (D_k[t]-mu_k)^2 (population, two pass)
 *   O4  P_k[0] = 0;  P_k[t+1] = P_k[t] + (D_k[t] - mu_k)
 *   O5  S(k,j,t) = (P_k[t+w_j] - P_k[t]) / (sigma_k sqrt(w_j)),  0 <= t <= T_k - w_j
 *       (S = 0 where sigma_k == 0)
 *   O6  snr[p] = max S, argmax[p] = lexicographically smallest (k,j,t) attaining it
 *       (-inf and (-1,-1,-1) if no cell is defined)
 *   O7  candidate iff snr[p] > threshold (strict)
 * Streaming restriction (S5): only windows whose last raw sample index
 *   t + w_j - 1 + dmax_k  >= raw_end_min   are evaluated (offline: raw_end_min = 0);
 *   mu/sigma still span every valid sample (S4).  Reported t gets t_offset added (S6).
 *
 * Parity pins (tests/test_oracle_pins.py): delay hand value and printed tables,
 * table-reuse identity, DM=0 == channel sum, w=1 == normalised series, numpy.convolve,
 * noise-free pulse closed form sqrt(T_k - w), injected-pulse closed form, offset/scale/
 * channel-permutation/duplicate-DM/time-shift invariances, brute force on tiny cubes,
 * streaming == offline on the ring contents.  Absolute S/N values on noisy cubes beyond
 * those pins: "parity unpinned" (the oracle is then the authority).
 */
#include <math.h>
#include <pthread.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_DISP_CONST_S 4.15e-3 /* PAPER.md:L83, reading R1 */

/* ---- O1: delay table ------------------------------------------------------------ */
int nsfrb_oracle_delays(int nchan, const double *freqs_GHz, double tsamp_s, int ndm,
                        const double *dm_list, int32_t *delays /* [ndm][nchan] */)
{
    if (nchan < 1 || ndm < 1 || !freqs_GHz || !dm_list || !delays || !(tsamp_s > 0.0))
        return -1;
    double f_ref = freqs_GHz[0];
    for (int c = 1; c < nchan; ++c)
        if (freqs_GHz[c] > f_ref) f_ref = freqs_GHz[c];
    for (int k = 0; k < ndm; ++k) {
        for (int c = 0; c < nchan; ++c) {
            double f = freqs_GHz[c];
            double x = ((ORACLE_DISP_CONST_S * dm_list[k]) *
                        (1.0 / (f * f) - 1.0 / (f_ref * f_ref))) / tsamp_s;
            delays[(size_t)k * nchan + c] = (int32_t)floor(x + 0.5);
        }
    }
    return 0;
}

/* ---- one pixel, steps O2..O6 ------------------------------------------------------ */
typedef struct {
    const float *cube;       /* [nchan][nt][npix] */
    int64_t npix;            /* pixel stride of the cube */
    int nchan, nt;
    const int32_t *delays;   /* [ndm][nchan] */
    int ndm;
    const int32_t *widths;   /* [nw] */
    int nw;
    int64_t raw_end_min;     /* S5 */
    int64_t t_offset;        /* S6 */
    int brute;               /* 1: O(w) direct boxcar sums, no prefix array */
    const double *sigma_norm; /* NULL, or [n_sel][ndm]: the standard deviation S is normalised by (reading R30:
                                 the "running standard deviation") instead of this call's own sigma_k */
} oracle_problem;

/* scratch: D[nt], P[nt+1] */
static void oracle_one_pixel(const oracle_problem *q, int64_t p, const double *sigma_norm /* [ndm] or NULL */,
                             double *D, double *P,
                             double *snr_out, int64_t *arg_out /* [3] */,
                             double *mu_out /* [ndm] or NULL */,
                             double *sigma_out /* [ndm] or NULL */,
                             double *best_out /* [ndm][nw] or NULL */,
                             int64_t *best_t_out /* [ndm][nw] or NULL */)
{
    const int nchan = q->nchan, nt = q->nt;
    double best = -INFINITY;
    int64_t bk = -1, bj = -1, bt = -1;

    for (int k = 0; k < q->ndm; ++k) {
        const int32_t *dk = q->delays + (size_t)k * nchan;
        int dmax = 0;
        for (int c = 0; c < nchan; ++c)
            if (dk[c] > dmax) dmax = dk[c];
        const int T = nt - dmax; /* T_k */
        if (mu_out) mu_out[k] = NAN;
        if (sigma_out) sigma_out[k] = NAN;
        if (best_out)
            for (int j = 0; j < q->nw; ++j) {
                best_out[(size_t)k * q->nw + j] = -INFINITY;
                best_t_out[(size_t)k * q->nw + j] = -1;
            }
        if (T < 1) continue;

        /* O2 */
        for (int t = 0; t < T; ++t) {
            double s = 0.0;
            for (int c = 0; c < nchan; ++c)
                s += (double)q->cube[((size_t)c * nt + (size_t)(t + dk[c])) * (size_t)q->npix + (size_t)p];
            D[t] = s;
        }
        /* O3 */
        double mu = 0.0;
        for (int t = 0; t < T; ++t) mu += D[t];
        mu /= (double)T;
        double var = 0.0;
        for (int t = 0; t < T; ++t) var += (D[t] - mu) * (D[t] - mu);
        var /= (double)T;
        const double sigma = sqrt(var);
        if (mu_out) mu_out[k] = mu;
        if (sigma_out) sigma_out[k] = sigma;
        /* O4 */
        if (!q->brute) {
            P[0] = 0.0;
            for (int t = 0; t < T; ++t) P[t + 1] = P[t] + (D[t] - mu);
        }
        /* O5, O6 */
        for (int j = 0; j < q->nw; ++j) {
            const int w = q->widths[j];
            if (w > T) continue;
            const double snorm = sigma_norm ? sigma_norm[k] : sigma; /* O5: sigma_k, or the caller's running one */
            const double norm = snorm * sqrt((double)w);
            double kj_best = -INFINITY;
            int64_t kj_t = -1;
            for (int t = 0; t <= T - w; ++t) {
                if ((int64_t)t + w - 1 + dmax < q->raw_end_min) continue; /* S5 */
                double B;
                if (q->brute) {
                    B = 0.0;
                    for (int u = t; u < t + w; ++u) B += D[u] - mu;
                } else {
                    B = P[t + w] - P[t];
                }
                const double S = (snorm == 0.0) ? 0.0 : B / norm;
                if (S > kj_best) { kj_best = S; kj_t = t; }
            }
            if (best_out) {
                best_out[(size_t)k * q->nw + j] = kj_best;
                best_t_out[(size_t)k * q->nw + j] = kj_t < 0 ? -1 : kj_t + q->t_offset;
            }
            /* strict '>' while scanning (k, j, t) in increasing order keeps the
               lexicographically smallest arg-max (O6, reading R17) */
            if (kj_t >= 0 && kj_best > best) {
                best = kj_best; bk = k; bj = j; bt = kj_t + q->t_offset;
            }
        }
    }
    *snr_out = best;
    arg_out[0] = bk; arg_out[1] = bj; arg_out[2] = bt;
}

typedef struct {
    const oracle_problem *q;
    const int64_t *pixels; /* list of pixel indices or NULL = 0..n-1 */
    int64_t begin, end, stride;
    double *snr; int64_t *argmax;
    double *mu, *sigma, *best; int64_t *best_t;
    int rc;
} oracle_job;

static void *oracle_worker(void *arg)
{
    oracle_job *jb = (oracle_job *)arg;
    const oracle_problem *q = jb->q;
    double *D = (double *)malloc(sizeof(double) * (size_t)(q->nt + 1));
    double *P = (double *)malloc(sizeof(double) * (size_t)(q->nt + 2));
    if (!D || !P) { free(D); free(P); jb->rc = -2; return NULL; }
    const size_t kw = (size_t)q->ndm * (size_t)q->nw;
    for (int64_t i = jb->begin; i < jb->end; i += jb->stride) {
        const int64_t p = jb->pixels ? jb->pixels[i] : i;
        oracle_one_pixel(q, p, q->sigma_norm ? q->sigma_norm + (size_t)i * q->ndm : NULL, D, P,
                         &jb->snr[i], &jb->argmax[3 * i],
                         jb->mu ? jb->mu + (size_t)i * q->ndm : NULL,
                         jb->sigma ? jb->sigma + (size_t)i * q->ndm : NULL,
                         jb->best ? jb->best + (size_t)i * kw : NULL,
                         jb->best_t ? jb->best_t + (size_t)i * kw : NULL);
    }
    free(D); free(P);
    jb->rc = 0;
    return NULL;
}

/*
 * Search n_sel pixels of the cube.  pixels == NULL means pixels 0..n_sel-1.
 * Outputs (all indexed by position in the selection):
 *   snr[n_sel] (double), argmax[n_sel][3] (int64: dm_idx, width_idx, t),
 *   optional mu[n_sel][ndm], sigma[n_sel][ndm], best[n_sel][ndm][nw], best_t[...].
 * nthreads >= 1: pixels are dealt round-robin to that many pthreads (each pixel is
 * still computed by one thread, start to finish).
 */
int nsfrb_oracle_search_norm(const float *cube, int64_t npix, int nchan, int nt,
                             const int32_t *delays, int ndm, const int32_t *widths, int nw,
                             int64_t raw_end_min, int64_t t_offset, int brute,
                             const int64_t *pixels, int64_t n_sel, int nthreads,
                             double *snr, int64_t *argmax,
                             double *mu, double *sigma, double *best, int64_t *best_t,
                             const double *sigma_norm);

int nsfrb_oracle_search(const float *cube, int64_t npix, int nchan, int nt,
                        const int32_t *delays, int ndm, const int32_t *widths, int nw,
                        int64_t raw_end_min, int64_t t_offset, int brute,
                        const int64_t *pixels, int64_t n_sel, int nthreads,
                        double *snr, int64_t *argmax,
                        double *mu, double *sigma, double *best, int64_t *best_t)
{
    return nsfrb_oracle_search_norm(cube, npix, nchan, nt, delays, ndm, widths, nw, raw_end_min, t_offset, brute,
                                    pixels, n_sel, nthreads, snr, argmax, mu, sigma, best, best_t, NULL);
}

/* As nsfrb_oracle_search, but S(k,j,t) is normalised by sigma_norm[i][k] (i = position in the selection) when
 * sigma_norm != NULL -- NEXT 1 / reading R30: the running standard deviation carried across pushes.  mu_k and the
 * boxcar sums are this call's; the sigma output still reports this call's own sigma_k. */
int nsfrb_oracle_search_norm(const float *cube, int64_t npix, int nchan, int nt,
                             const int32_t *delays, int ndm, const int32_t *widths, int nw,
                             int64_t raw_end_min, int64_t t_offset, int brute,
                             const int64_t *pixels, int64_t n_sel, int nthreads,
                             double *snr, int64_t *argmax,
                             double *mu, double *sigma, double *best, int64_t *best_t,
                             const double *sigma_norm)
{
    if (!cube || !delays || !widths || !snr || !argmax) return -1;
    if (npix < 1 || nchan < 1 || nt < 1 || ndm < 1 || nw < 1 || n_sel < 0) return -1;
    for (int j = 0; j < nw; ++j) if (widths[j] < 1) return -1;
    for (int i = 0; i < ndm * nchan; ++i) if (delays[i] < 0) return -1;
    if (pixels)
        for (int64_t i = 0; i < n_sel; ++i)
            if (pixels[i] < 0 || pixels[i] >= npix) return -1;
    if (!pixels && n_sel > npix) return -1;
    if (nthreads < 1) nthreads = 1;
    if (nthreads > 256) nthreads = 256;
    if ((int64_t)nthreads > n_sel) nthreads = n_sel > 0 ? (int)n_sel : 1;

    oracle_problem q;
    q.cube = cube; q.npix = npix; q.nchan = nchan; q.nt = nt;
    q.delays = delays; q.ndm = ndm; q.widths = widths; q.nw = nw;
    q.raw_end_min = raw_end_min; q.t_offset = t_offset; q.brute = brute;
    q.sigma_norm = sigma_norm;

    oracle_job jobs[256];
    pthread_t th[256];
    for (int i = 0; i < nthreads; ++i) {
        jobs[i].q = &q; jobs[i].pixels = pixels;
        jobs[i].begin = i; jobs[i].end = n_sel; jobs[i].stride = nthreads;
        jobs[i].snr = snr; jobs[i].argmax = argmax;
        jobs[i].mu = mu; jobs[i].sigma = sigma; jobs[i].best = best; jobs[i].best_t = best_t;
        jobs[i].rc = 0;
    }
    if (nthreads == 1) {
        oracle_worker(&jobs[0]);
        return jobs[0].rc;
    }
    for (int i = 0; i < nthreads; ++i)
        if (pthread_create(&th[i], NULL, oracle_worker, &jobs[i]) != 0) {
            for (int r = 0; r < i; ++r) pthread_join(th[r], NULL);
            return -3;
        }
    int rc = 0;
    for (int i = 0; i < nthreads; ++i) {
        pthread_join(th[i], NULL);
        if (jobs[i].rc != 0) rc = jobs[i].rc;
    }
    return rc;
}

/*
 * S(k,j,t) of one cell of one pixel (O2..O5), for adjudicating near-ties.  t is the
 * window start in the same frame the search reports (t_offset is subtracted first).
 * Returns NaN when the cell is not defined (w > T_k, t out of range, or excluded by S5).
 */
double nsfrb_oracle_snr_at(const float *cube, int64_t npix, int nchan, int nt,
                           const int32_t *delays, int ndm, const int32_t *widths, int nw,
                           int64_t raw_end_min, int64_t t_offset,
                           int64_t p, int k, int j, int64_t t_abs)
{
    if (!cube || !delays || !widths) return NAN;
    if (p < 0 || p >= npix || k < 0 || k >= ndm || j < 0 || j >= nw) return NAN;
    const int32_t *dk = delays + (size_t)k * nchan;
    int dmax = 0;
    for (int c = 0; c < nchan; ++c) if (dk[c] > dmax) dmax = dk[c];
    const int T = nt - dmax;
    const int w = widths[j];
    const int64_t t = t_abs - t_offset;
    if (T < 1 || w > T || t < 0 || t > T - w) return NAN;
    if (t + w - 1 + dmax < raw_end_min) return NAN;
    double mu = 0.0;
    for (int u = 0; u < T; ++u) {
        double s = 0.0;
        for (int c = 0; c < nchan; ++c)
            s += (double)cube[((size_t)c * nt + (size_t)(u + dk[c])) * (size_t)npix + (size_t)p];
        mu += s;
    }
    mu /= (double)T;
    double var = 0.0, B = 0.0;
    for (int u = 0; u < T; ++u) {
        double s = 0.0;
        for (int c = 0; c < nchan; ++c)
            s += (double)cube[((size_t)c * nt + (size_t)(u + dk[c])) * (size_t)npix + (size_t)p];
        var += (s - mu) * (s - mu);
        if (u >= t && u < t + w) B += s - mu;
    }
    var /= (double)T;
    const double sigma = sqrt(var);
    if (sigma == 0.0) return 0.0;
    return B / (sigma * sqrt((double)w));
}

/* Exact number of cells (p,k,j,t) one offline call evaluates per pixel:
 * sum_k sum_j max(0, T_k - w_j + 1). */
int64_t nsfrb_oracle_cells_per_pixel(int nchan, int nt, const int32_t *delays, int ndm,
                                     const int32_t *widths, int nw)
{
    int64_t n = 0;
    for (int k = 0; k < ndm; ++k) {
        int dmax = 0;
        for (int c = 0; c < nchan; ++c)
            if (delays[(size_t)k * nchan + c] > dmax) dmax = delays[(size_t)k * nchan + c];
        const int T = nt - dmax;
        for (int j = 0; j < nw; ++j)
            if (T - widths[j] + 1 > 0) n += T - widths[j] + 1;
    }
    return n;
}

/* NEXT 2: time binning of the image stack, PAPER.md:L77/L81 ("bins images to 0.67 s (x5) and 10.05 s
 * (x75)" before re-searching with the same widths and, by footnote 12 L98, the same shift table at 5x the DM).
 * Reading R24: out[c][u][p] = sum_{i<factor} in[c][u*factor + i][p] for u < floor(nt/factor); the
 * trailing nt mod factor samples are dropped; a sum, not a mean (the S/N of O5 is scale-free).  float64 accumulate,
 * result rounded once to float32 (the search takes a float32 cube). */
int nsfrb_oracle_bin(const float *in, int nchan, int nt, int64_t npix, int factor, float *out)
{
    if (!in || !out || nchan < 1 || nt < 1 || npix < 1 || factor < 1) return -1;
    const int nb = nt / factor;
    for (int c = 0; c < nchan; ++c)
        for (int u = 0; u < nb; ++u)
            for (int64_t p = 0; p < npix; ++p) {
                double s = 0.0;
                for (int i = 0; i < factor; ++i) s += (double)in[((size_t)c * nt + (size_t)u * factor + i) * npix + p];
                out[((size_t)c * nb + u) * npix + p] = (float)s;
            }
    return 0;
}
