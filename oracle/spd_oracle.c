/*
 * spd_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, float64 CPU statement of what the single-pulse-detection hot path of
 * arXiv 1611.09704 (Adamek & Armour) computes, written from /root/reference/PAPER.md
 * before any CUDA kernel existed.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load this library.  It shares no code, header,
 * table or helper with paper_1611_09704_b200/csrc/ and neither side imports the other.
 *
 * Every function follows the paper's order and notation; there is no blocking, fusion or
 * reordering beyond "OpenMP over DM rows" (rows are independent: "on each of
 * DM trial").  Readings of garbled / silent passages are those of SURVEY.md §8(c) and are
 * listed in DESIGN.md ("Readings of the paper").
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): P1 two-pass numpy mean/std, P2 closed
 * forms, P3 eq.2 merge-order invariance, P4 rectangular-pulse closed form (Figure 1),
 * P5 constant input (tie-break + row-end rule), P6 brute-force O(n*Nmax^2) inner sums,
 * P7 pure-noise normalisation, P8 sigma table end points, P9 candidate set = brute filter,
 * P10 (tests/test_oracle_decimated.py) for O5, decimation in time + boxcar: level 0 = O3, decimated
 * series = block sums, every level = explicit sums over the original samples, on-grid pulse = A sqrt(W),
 * off-grid sensitivity >= sqrt(0.9); P11 (tests/test_oracle_pins.py) for O3r, per-row statistics: every row equals
 * O3 on that row alone with that row's numpy two-pass mean / std.
 * No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ---------------------------------------------------------------------------------------
 * O1  mean and standard deviation  (section 2.1, eq. 1 and eq. 2)
 * ------------------------------------------------------------------------------------- */

typedef struct { uint64_t m; double T, S; } chan_t;   /* m samples, T = sum, S = sum of squared deviations */

/* eq. 1: streaming update with the j-th sample x_j.
 * Reading A1: the printed (j x_j - T_{1,j}) lacks its square; restored (Chan, Golub & LeVeque, ref. [2]).
 *   T_{1,j} = T_{1,j-1} + x_j
 *   S_{1,j} = S_{1,j-1} + (j x_j - T_{1,j})^2 / (j (j-1))                                   */
static void chan_push(chan_t *a, double x)
{
    if (a->m == 0) { a->m = 1; a->T = x; a->S = 0.0; return; }
    double j = (double)(a->m + 1);
    a->T += x;
    double d = j * x - a->T;
    a->S += d * d / (j * (j - 1.0));
    a->m += 1;
}

/* eq. 2: merge set 1..m (a) with set m+1..m+n (b), exactly as printed:
 *   S_{1,m+n} = S_{1,m} + S_{m+1,m+n} + m/(n(m+n)) * ( (n/m) T_{1,m} - T_{m+1,m+n} )^2
 *   T_{1,m+n} = T_{1,m} + T_{m+1,m+n}
 * A side with zero samples is skipped.                                                     */
static void chan_merge(chan_t *a, const chan_t *b)
{
    if (b->m == 0) return;
    if (a->m == 0) { *a = *b; return; }
    double m = (double)a->m, n = (double)b->m;
    double d = (n / m) * a->T - b->T;
    a->S = a->S + b->S + m / (n * (m + n)) * d * d;
    a->T = a->T + b->T;
    a->m += b->m;
}

/* A stream of values is cut into blocks of `block` samples ("equal sized blocks",
 * PAPER.md:44); each block runs eq. 1; blocks are folded left to right with eq. 2.       */
typedef struct { chan_t total, cur; uint64_t block; } chan_stream_t;

static void stream_init(chan_stream_t *s, uint64_t block) { memset(s, 0, sizeof *s); s->block = block ? block : 1000; }
static void stream_push(chan_stream_t *s, double x)
{
    chan_push(&s->cur, x);
    if (s->cur.m == s->block) { chan_merge(&s->total, &s->cur); memset(&s->cur, 0, sizeof s->cur); }
}
static void stream_finish(chan_stream_t *s) { chan_merge(&s->total, &s->cur); memset(&s->cur, 0, sizeof s->cur); }

/* out[0..4] = { n, T, S, mu = T/n, sigma = sqrt(S/n) }   (population form, reading A2).
 * One estimate for the whole array passed in (reading A3).                                  */
void spd_oracle_stats(const float *x, int64_t n_dm, int64_t n_t, int64_t row_stride, int64_t block, double *out)
{
    chan_stream_t s; stream_init(&s, (uint64_t)block);
    for (int64_t d = 0; d < n_dm; ++d)
        for (int64_t t = 0; t < n_t; ++t)
            stream_push(&s, (double)x[d * row_stride + t]);
    stream_finish(&s);
    double n = (double)s.total.m;
    out[0] = n; out[1] = s.total.T; out[2] = s.total.S;
    out[3] = s.total.T / n; out[4] = sqrt(s.total.S / n);
}

/* eq. 2 exposed on its own so that tests can fold partial results in any order (pin P3).
 * a and b are {m, T, S} triples (m as double); a is updated in place.                       */
void spd_oracle_merge(double *a, const double *b)
{
    chan_t A = { (uint64_t)a[0], a[1], a[2] }, B = { (uint64_t)b[0], b[1], b[2] };
    chan_merge(&A, &B);
    a[0] = (double)A.m; a[1] = A.T; a[2] = A.S;
}

/* eq. 1 alone over a contiguous float64 vector -> {m, T, S} (pins P1-P3).                    */
void spd_oracle_chan_run(const double *x, int64_t n, double *out)
{
    chan_t a; memset(&a, 0, sizeof a);
    for (int64_t i = 0; i < n; ++i) chan_push(&a, x[i]);
    out[0] = (double)a.m; out[1] = a.T; out[2] = a.S;
}

/* O1b  "true value of standard deviation after applying Nmax-sampled boxcar".
 * Reading A11: population std of the SUMS B_Nmax(t) over every full window t in [0, n_t-Nmax]
 * of every row.  b is the direct sum of Nmax samples, taken from a float64 prefix sum of the row.
 * out = { n', T', S', mean', sigma_Nmax }.                                                  */
void spd_oracle_sigma_nmax(const float *x, int64_t n_dm, int64_t n_t, int64_t row_stride, int nmax,
                           int64_t block, double *out)
{
    chan_stream_t s; stream_init(&s, (uint64_t)block);
    double *P = (double *)malloc((size_t)(n_t + 1) * sizeof(double));
    for (int64_t d = 0; d < n_dm; ++d) {
        const float *row = x + d * row_stride;
        P[0] = 0.0;
        for (int64_t t = 0; t < n_t; ++t) P[t + 1] = P[t] + (double)row[t];
        for (int64_t t = 0; t + nmax <= n_t; ++t) stream_push(&s, P[t + nmax] - P[t]);
    }
    free(P);
    stream_finish(&s);
    double n = (double)s.total.m;
    out[0] = n; out[1] = s.total.T; out[2] = s.total.S;
    out[3] = n > 0 ? s.total.T / n : NAN; out[4] = n > 0 ? sqrt(s.total.S / n) : NAN;
}

/* ---------------------------------------------------------------------------------------
 * O2  sigma after an N-sample boxcar  (section 2.2)
 *   mode 0: eq. 4   sigma_N = sqrt(N) sigma
 *   mode 1: eq. 5   sigma_N = sqrt(N) sigma + (N-1) sigma_Nmax / (Nmax-1)     (literal, reading A10)
 *   mode 2: anchored variant (not in the paper; exact at N=1 and N=Nmax):
 *           sigma_N = sqrt(N) sigma + (N-1) (sigma_Nmax - sqrt(Nmax) sigma) / (Nmax-1)
 * Nmax = 1 drops the linear term (0/0).  sig[w-1] = sigma_w for w = 1..nmax.                */
void spd_oracle_sigma_table(double sigma, double sigma_nmax, int nmax, int mode, double *sig)
{
    for (int w = 1; w <= nmax; ++w) {
        double s = sqrt((double)w) * sigma;
        if (mode == 1 && nmax > 1) s += (double)(w - 1) * sigma_nmax / (double)(nmax - 1);
        if (mode == 2 && nmax > 1) s += (double)(w - 1) * (sigma_nmax - sqrt((double)nmax) * sigma) / (double)(nmax - 1);
        sig[w - 1] = s;
    }
}

/* ---------------------------------------------------------------------------------------
 * O3  boxcar filters, SNR, max over width  (section 2.3, Algorithm 1)
 *
 * Readings A5-A7, A9: the boxcar is start-anchored and forward, B_N(t) = sum_{k<N} x[t+k];
 * SNR_N(t) = (B_N(t) - N mu) / sigma_N; widths ascend from 1 and a strict ">" keeps the
 * smallest width on ties; only widths that fit in the row are evaluated (N <= n_t - t).
 * Outputs per sample: snr = max_N SNR_N, width = smallest N attaining it,
 * margin = best - second best (+inf when a single width was evaluated).  Any of the three
 * output pointers may be NULL.                                                              */
void spd_oracle_sweep(const float *x, int64_t n_dm, int64_t n_t, int64_t row_stride,
                      double mu, const double *sig, int nmax,
                      double *snr, int32_t *width, double *margin)
{
    #pragma omp parallel for schedule(dynamic, 1)
    for (int64_t d = 0; d < n_dm; ++d) {
        const float *row = x + d * row_stride;
        for (int64_t t = 0; t < n_t; ++t) {
            double B = 0.0, best = -INFINITY, second = -INFINITY;
            int32_t W = 1;
            int64_t wmax = n_t - t < (int64_t)nmax ? n_t - t : (int64_t)nmax;
            for (int64_t w = 1; w <= wmax; ++w) {
                B += (double)row[t + w - 1];
                double s = (B - (double)w * mu) / sig[w - 1];
                if (s > best) { second = best; best = s; W = (int32_t)w; }
                else if (s > second) second = s;
            }
            int64_t o = d * n_t + t;
            if (snr)    snr[o] = best;
            if (width)  width[o] = W;
            if (margin) margin[o] = best - second;   /* +inf when second = -inf */
        }
    }
}

/* SNR of ONE width at every sample (debug plane for pin P7); samples whose window does not
 * fit get NaN.                                                                               */
void spd_oracle_snr_fixed_width(const float *x, int64_t n_dm, int64_t n_t, int64_t row_stride,
                                double mu, double sigma_w, int w, double *snr)
{
    for (int64_t d = 0; d < n_dm; ++d) {
        const float *row = x + d * row_stride;
        for (int64_t t = 0; t < n_t; ++t) {
            if (t + w > n_t) { snr[d * n_t + t] = NAN; continue; }
            double B = 0.0;
            for (int k = 0; k < w; ++k) B += (double)row[t + k];
            snr[d * n_t + t] = (B - (double)w * mu) / sigma_w;
        }
    }
}

/* SNR of listed (dm, t, width) triples by direct summation: used by the comparator to judge
 * a width that differs from the oracle's inside a near-tie.  Width that does not fit -> NaN. */
void spd_oracle_snr_at(const float *x, int64_t n_t, int64_t row_stride, double mu, const double *sig, int nmax,
                       const int64_t *dm, const int64_t *t, const int32_t *w, int64_t count, double *out)
{
    for (int64_t i = 0; i < count; ++i) {
        if (w[i] < 1 || w[i] > nmax || t[i] + w[i] > n_t) { out[i] = NAN; continue; }
        const float *row = x + dm[i] * row_stride;
        double B = 0.0;
        for (int k = 0; k < w[i]; ++k) B += (double)row[t[i] + k];
        out[i] = (B - (double)w[i] * mu) / sig[w[i] - 1];
    }
}

/* ---------------------------------------------------------------------------------------
 * O4  candidate selection  (section 2.4)
 * Readings A12-A15: keep every sample of the max-over-width plane with SNR >= f_T; the plane
 * is not modified; the result is a list of (DM row, start time, SNR, width), one entry per
 * sample, no clustering.  The list is returned in (dm, t) order (any order is correct).
 * Returns the number of hits; writes at most `capacity` of them.                             */
int64_t spd_oracle_candidates(const double *snr, const int32_t *width, int64_t n_dm, int64_t n_t, double f_T,
                              int64_t capacity, int64_t *c_dm, int64_t *c_t, double *c_snr, int32_t *c_width)
{
    int64_t count = 0;
    for (int64_t d = 0; d < n_dm; ++d)
        for (int64_t t = 0; t < n_t; ++t) {
            double s = snr[d * n_t + t];
            if (s >= f_T) {
                if (count < capacity) { c_dm[count] = d; c_t[count] = t; c_snr[count] = s; c_width[count] = width[d * n_t + t]; }
                ++count;
            }
        }
    return count;
}

/* ---------------------------------------------------------------------------------------
 * O5  decimation in time + boxcar for wide filters  (section 3: "we will use a
 * combination of boxcar filtering with the decimation in time of the input data")
 *
 * The paper names the route but gives no algorithm; this is reading A20 of DESIGN.md, written out
 * step by step.  It is an APPROXIMATION of the exhaustive search O3: the width grid gets coarser
 * with width (PAPER.md:21, :69 warn about the sensitivity this costs).
 *
 *   level 0:  x_0 = x.  Boxcars of every width w' = 1..W0 at every sample: exactly O3 with Nmax = W0.
 *   level l:  x_l[i] = x_{l-1}[2i] + x_{l-1}[2i+1],  i < n_l = floor(n_{l-1} / 2)      (decimation by 2)
 *             boxcars of widths w' = W0/2+1 .. W0 (in decimated samples) at every decimated sample i;
 *             one of them covers N = w' 2^l samples of x starting at t = i 2^l, so
 *                 SNR = (B - N mu) / sigma_N      with sigma_N from O2 for the EFFECTIVE width N
 *             (mu, sigma are those of x: nothing is re-measured per level).  Widths
 *             w' <= W0/2 are left to the finer levels, which cover them at twice the resolution.
 *   Only widths that fit are evaluated (reading A9): w' <= n_l - i.  A position where none of the
 *   level's widths fits gets snr = -inf, width = 0.
 *
 * This function does ONE level on an already decimated row block xl (float64, [n_dm][n_l]):
 *   lvl = l, sig[N-1] = sigma_N for N = 1..W0 2^l, wmin = smallest width evaluated (1 at level 0, W0/2+1 above).
 * Outputs per decimated sample: snr, width = EFFECTIVE width N (0 if none), margin = best - second.  */
void spd_oracle_sweep_level(const double *xl, int64_t n_dm, int64_t n_l, double mu, const double *sig,
                            int w0, int wmin, int lvl, double *snr, int32_t *width, double *margin)
{
    const int64_t D = (int64_t)1 << lvl;
    #pragma omp parallel for schedule(dynamic, 1)
    for (int64_t d = 0; d < n_dm; ++d) {
        const double *row = xl + d * n_l;
        for (int64_t i = 0; i < n_l; ++i) {
            double B = 0.0, best = -INFINITY, second = -INFINITY;
            int32_t W = 0;
            int64_t wmax = n_l - i < (int64_t)w0 ? n_l - i : (int64_t)w0;
            for (int64_t w = 1; w <= wmax; ++w) {
                B += row[i + w - 1];
                if (w < wmin) continue;
                int64_t N = w * D;
                double s = (B - (double)N * mu) / sig[N - 1];
                if (s > best) { second = best; best = s; W = (int32_t)N; }
                else if (s > second) second = s;
            }
            int64_t o = d * n_l + i;
            snr[o] = best; width[o] = W; margin[o] = best - second;
        }
    }
}

/* x_l[i] = x_{l-1}[2i] + x_{l-1}[2i+1] for one level (float64 in, float64 out, [n_dm][n_prev] -> [n_dm][n_prev/2]) */
void spd_oracle_decimate2(const double *xp, int64_t n_dm, int64_t n_prev, double *xl)
{
    const int64_t n_l = n_prev / 2;
    for (int64_t d = 0; d < n_dm; ++d)
        for (int64_t i = 0; i < n_l; ++i)
            xl[d * n_l + i] = xp[d * n_prev + 2 * i] + xp[d * n_prev + 2 * i + 1];
}

/* ---------------------------------------------------------------------------------------
 * O3r  the sweep with ONE (mu, sigma_N table) PER DM ROW  ("for the dataset": reading A3
 * takes one estimate per call; per-row statistics, A3's alternative, is what heterogeneous data wants,
 * SURVEY.md 8(f) f3).  Same loop as O3, with mu[d] and sig[d * nmax + (w-1)] in place of mu and sig[w-1].
 * The per-row statistics themselves are O1 / O1b called on one row at a time (no new arithmetic).     */
void spd_oracle_sweep_rows(const float *x, int64_t n_dm, int64_t n_t, int64_t row_stride,
                           const double *mu, const double *sig, int nmax,
                           double *snr, int32_t *width, double *margin)
{
    #pragma omp parallel for schedule(dynamic, 1)
    for (int64_t d = 0; d < n_dm; ++d) {
        const float *row = x + d * row_stride;
        const double *sg = sig + d * (int64_t)nmax;
        for (int64_t t = 0; t < n_t; ++t) {
            double B = 0.0, best = -INFINITY, second = -INFINITY;
            int32_t W = 1;
            int64_t wmax = n_t - t < (int64_t)nmax ? n_t - t : (int64_t)nmax;
            for (int64_t w = 1; w <= wmax; ++w) {
                B += (double)row[t + w - 1];
                double s = (B - (double)w * mu[d]) / sg[w - 1];
                if (s > best) { second = best; best = s; W = (int32_t)w; }
                else if (s > second) second = s;
            }
            int64_t o = d * n_t + t;
            if (snr)    snr[o] = best;
            if (width)  width[o] = W;
            if (margin) margin[o] = best - second;
        }
    }
}
