/*
 * gce_oracle.c -- CPU oracle for the Conditional Entropy (P, Pdot) period search.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code with the CUDA path (paper_2006_06866_b200/csrc) and neither
 * includes the other.  Host pointers only; plain C; fp64 throughout.
 *
 * Written from /root/reference/PAPER.md (Katz et al., arXiv 2006.06866):
 *   - magnitude normalisation            PAPER.md:96   (reading Q2 of DESIGN.md: min/max -> [0,1]; the paper's own
 *                                                       per-filter median / std step as an option, reading Q19)
 *   - phase fold with Pdot, Eq. 3
 *   - 2-D phase x magnitude histogram     PAPER.md:106  (non-overlapping bins; the 50 %-overlapping variant: reading Q3)
 *   - conditional entropy, Eq. 4
 *   - minimum CE = best (P, Pdot)
 *   - significance, Eq. 5
 *
 * The method is a brute-force grid evaluation ("the actual CE algorithm is
 * effectively the same"), so the oracle is the plain definition written out.  Because the
 * phase-bin index is a discontinuous function of an fp64 value near 1e6 cycles, "plain"
 * includes a FROZEN operation order (reading Q4):
 *
 *     invP = 1/P                       (IEEE RN division)
 *     c    = ((-0.5*Pdot)*invP)*invP   (left to right)
 *     a = dt*invP ; b = dt2*c ; x = a + b        (three RN operations, never fused)
 *     y = x * n_phase ; I = floor(y) ; j = I mod n_phase (floored modulus)
 *
 * Build:  gcc -O2 -std=c11 -ffp-contract=off -fno-fast-math -fopenmp -shared -fPIC
 * (-ffp-contract=off is REQUIRED: a fused multiply-add changes bin indices.)
 *
 * Pins (tests/test_oracle_pins.py, all -m "not gpu"): dyadic hand folds, hand count tables
 * with closed-form CE (0, ln 2, 1/2 ln 2, 0.6059391565991873), scipy.stats.entropy identity
 * H(m,phi) - H(phi), exact rational refold, Eq. 6 closed form, numpy.histogram marginals,
 * invariants 0 <= CE <= H(m), noiseless recovery; N2 overlap: hand tables, exact-rational interval
 * membership, CE_plain <= CE_overlap <= CE_plain + ln 2; S0 normalisation: hand closed forms, numpy.median /
 * numpy.std per filter, one-filter bin invariance, a two-filter merged light curve.  Parity with a CE value printed in the
 * paper: UNPINNED (the paper prints none).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define GCE_ORACLE_OK 0
#define GCE_ORACLE_EINVAL -1

/* ---------------------------------------------------------------------------------------
 * S0 (optional, NEXT item N4)  the paper's normalisation: "subtract from each
 * observation the median magnitude value, and then we divide by the standard deviation of the
 * magnitude values ... this allows us to combine observations from different filters into one
 * input light curve".  Per filter f of one light curve, over the points k with filt[k] == f in
 * light-curve order (reading Q19):
 *     med  = median (middle value, or the mean of the two middle values: (a + b) * 0.5)
 *     mean = (((v_0 + v_1) + v_2) + ...) / n_f              sequential sum, RN
 *     sd   = sqrt( (((d_0^2 + d_1^2) + ...) / n_f) ),  d_k = v_k - mean   population (ddof 0)
 *     u_k  = (v_k - med) / sd ;  sd == 0 (one point, or all equal) -> u_k = 0
 * The merged u then goes through S1 (min/max bins over the merged range) unchanged.
 * filt == NULL: one filter.  Filter ids 0 .. 7.
 * ------------------------------------------------------------------------------------- */
static int cmp_double(const void *a, const void *b)
{
    const double x = *(const double *)a, y = *(const double *)b;
    return (x > y) - (x < y);
}

int gce_oracle_normalise_filters(const double *m, const int32_t *filt, int64_t n, double *u)
{
    if (n < 0) return GCE_ORACLE_EINVAL;
    double *v = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
    if (!v) return GCE_ORACLE_EINVAL;
    for (int32_t f = 0; f < 8; ++f) {
        int64_t nf = 0;
        for (int64_t k = 0; k < n; ++k) {
            const int32_t fk = filt ? filt[k] : 0;
            if (fk < 0 || fk > 7) { free(v); return GCE_ORACLE_EINVAL; }
            if (fk == f) v[nf++] = m[k];
        }
        if (nf == 0) continue;
        double sum = 0.0;
        for (int64_t i = 0; i < nf; ++i) sum = sum + v[i];
        const double mean = sum / (double)nf;
        double ss = 0.0;
        for (int64_t i = 0; i < nf; ++i) {
            const double d = v[i] - mean;
            ss = ss + d * d;
        }
        const double sd = sqrt(ss / (double)nf);
        qsort(v, (size_t)nf, sizeof(double), cmp_double);
        const double med = (nf % 2) ? v[(nf - 1) / 2] : (v[nf / 2 - 1] + v[nf / 2]) * 0.5;
        for (int64_t k = 0; k < n; ++k) {
            if ((filt ? filt[k] : 0) != f) continue;
            u[k] = (sd == 0.0) ? 0.0 : (m[k] - med) / sd;
        }
    }
    free(v);
    return GCE_ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------
 * S1  preprocess one light curve (north_star (2)): t0 = min t, dt = t - t0,
 * dt2 = dt*dt, min/max normalise m to [0,1], magnitude bin i = min(floor(u*n_mag), n_mag-1).
 * All magnitudes equal (range 0) -> every point in bin 0 (reading Q12).
 * ------------------------------------------------------------------------------------- */
int gce_oracle_preprocess(const double *t, const double *m, int64_t n, int32_t n_mag,
                          double *dt, double *dt2, int32_t *mbin)
{
    if (n < 0 || n_mag < 1) return GCE_ORACLE_EINVAL;
    if (n == 0) return GCE_ORACLE_OK;
    double t0 = t[0], m_lo = m[0], m_hi = m[0];
    for (int64_t k = 1; k < n; ++k) {
        if (t[k] < t0) t0 = t[k];
        if (m[k] < m_lo) m_lo = m[k];
        if (m[k] > m_hi) m_hi = m[k];
    }
    const double r = m_hi - m_lo;
    for (int64_t k = 0; k < n; ++k) {
        dt[k] = t[k] - t0;
        dt2[k] = dt[k] * dt[k];
        if (r == 0.0) {
            mbin[k] = 0;
        } else {
            const double u = (m[k] - m_lo) / r;
            int32_t i = (int32_t)floor(u * (double)n_mag);
            if (i > n_mag - 1) i = n_mag - 1; /* u == 1 belongs to the last (closed) bin, Q6 */
            mbin[k] = i;
        }
    }
    return GCE_ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------
 * S2  fold (Eq. 3): P*phi = (t - 1/2 (Pdot/P) t^2) mod P, then / P.
 * In cycles: x = t/P - 1/2 Pdot t^2 / P^2 ; phase = x mod 1 ; bin j = floor(n_phase*phase).
 * Frozen order as in the header.  Writes the phase bin of every point.
 * ------------------------------------------------------------------------------------- */
static inline int32_t fold_bin(double dtk, double dt2k, double invP, double c, int32_t n_phase)
{
    const double a = dtk * invP;
    const double b = dt2k * c;
    const double x = a + b;
    const double y = x * (double)n_phase;
    const int64_t I = (int64_t)floor(y);
    int64_t j = I % (int64_t)n_phase;
    if (j < 0) j += n_phase; /* floored modulus: phase always in [0,1), Q5 */
    return (int32_t)j;
}

static inline void trial_constants(double P, double Pdot, double *invP, double *c)
{
    *invP = 1.0 / P;
    *c = ((-0.5 * Pdot) * (*invP)) * (*invP);
}

int gce_oracle_fold_bins(const double *dt, const double *dt2, int64_t n, double P, double Pdot,
                         int32_t n_phase, int32_t *phase_bin, double *x_out /* may be NULL */)
{
    if (n < 0 || n_phase < 1) return GCE_ORACLE_EINVAL;
    double invP, c;
    trial_constants(P, Pdot, &invP, &c);
    for (int64_t k = 0; k < n; ++k) {
        phase_bin[k] = fold_bin(dt[k], dt2[k], invP, c, n_phase);
        if (x_out) x_out[k] = dt[k] * invP + dt2[k] * c; /* same three RN ops (no contraction) */
    }
    return GCE_ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------
 * S3  2-D histogram: cnt[j][i] = number of points in phase bin j and
 * magnitude bin i.  Layout [n_phase][n_mag], row-major.
 * ------------------------------------------------------------------------------------- */
static void histogram_one_trial(const double *dt, const double *dt2, const int32_t *mbin, int64_t n,
                                double P, double Pdot, int32_t n_phase, int32_t n_mag, int64_t *cnt)
{
    double invP, c;
    trial_constants(P, Pdot, &invP, &c);
    memset(cnt, 0, sizeof(int64_t) * (size_t)n_phase * (size_t)n_mag);
    for (int64_t k = 0; k < n; ++k) {
        const int32_t j = fold_bin(dt[k], dt2[k], invP, c, n_phase);
        cnt[(int64_t)j * n_mag + mbin[k]] += 1;
    }
}

/* ---------------------------------------------------------------------------------------
 * S4  conditional entropy (Eq. 4):
 *   H_c = sum_{i,j} p(m_i,phi_j) ln( p(phi_j) / p(m_i,phi_j) ),
 *   p(m_i,phi_j) = n_ij/N, p(phi_j) = sum_i n_ij / N (Q8); empty cells contribute 0 (Q7).
 * N == 0 -> NaN (Q12).
 * ------------------------------------------------------------------------------------- */
double gce_oracle_ce_from_counts(const int64_t *cnt, int32_t n_phase, int32_t n_mag, int64_t N)
{
    if (N <= 0) return NAN;
    double ce = 0.0;
    for (int32_t j = 0; j < n_phase; ++j) {
        int64_t n_j = 0;
        for (int32_t i = 0; i < n_mag; ++i) n_j += cnt[(int64_t)j * n_mag + i];
        for (int32_t i = 0; i < n_mag; ++i) {
            const int64_t n_ij = cnt[(int64_t)j * n_mag + i];
            if (n_ij > 0) ce += ((double)n_ij / (double)N) * log((double)n_j / (double)n_ij);
        }
    }
    return ce;
}

/* Counts of selected trials of ONE light curve (already preprocessed). q = ip*n_pdot + ipd. */
int gce_oracle_histogram(const double *dt, const double *dt2, const int32_t *mbin, int64_t n,
                         const double *periods, int64_t n_p, const double *pdots, int64_t n_pdot,
                         int32_t n_phase, int32_t n_mag, const int64_t *trial_q, int64_t n_trials,
                         int64_t *out_counts /* [n_trials][n_phase][n_mag] */)
{
    if (n < 0 || n_phase < 1 || n_mag < 1 || n_p < 0 || n_pdot < 1) return GCE_ORACLE_EINVAL;
    for (int64_t s = 0; s < n_trials; ++s) {
        const int64_t q = trial_q[s];
        if (q < 0 || q >= n_p * n_pdot) return GCE_ORACLE_EINVAL;
        histogram_one_trial(dt, dt2, mbin, n, periods[q / n_pdot], pdots[q % n_pdot], n_phase, n_mag,
                            out_counts + s * (int64_t)n_phase * n_mag);
    }
    return GCE_ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------
 * The search: every light curve x every (P, Pdot).  out_ce layout [n_lc][n_p][n_pdot],
 * Pdot fastest (Q10).  OpenMP over periods; each thread has its own count table.
 * ------------------------------------------------------------------------------------- */
/* ---------------------------------------------------------------------------------------
 * NEXT item N2 -- 50 % overlapping phase bins ("each histogram bin has a 50% overlap
 * with each adjacent bin", Fig. 3 caption :162 "50 phase bins that overlap by 50% with surrounding
 * bins").  Reading Q3: phase axis only, cyclic.  The n_phase bins have
 * width 2/n_phase and start 1/n_phase apart: bin k covers the phases [(k-1)/n_phase, (k+1)/n_phase)
 * (mod 1), i.e. the two cells k-1 and k of the plain n_phase-cell grid of S2/S3.  Every point
 * therefore lies in exactly two bins, the table holds 2N entries, and probabilities are
 * normalised by 2N:  c[k][i] = n[k][i] + n[k-1 mod n_phase][i].  Eq. 4 is then applied to c.
 * ------------------------------------------------------------------------------------- */
int gce_oracle_overlap_counts(const int64_t *cnt, int32_t n_phase, int32_t n_mag, int64_t *out)
{
    if (n_phase < 1 || n_mag < 1) return GCE_ORACLE_EINVAL;
    for (int32_t k = 0; k < n_phase; ++k) {
        const int32_t km = (k + n_phase - 1) % n_phase;
        for (int32_t i = 0; i < n_mag; ++i)
            out[(int64_t)k * n_mag + i] = cnt[(int64_t)k * n_mag + i] + cnt[(int64_t)km * n_mag + i];
    }
    return GCE_ORACLE_OK;
}

static double ce_one_trial(const int64_t *cnt, int64_t *tmp, int32_t n_phase, int32_t n_mag, int64_t n, int overlap)
{
    if (!overlap) return gce_oracle_ce_from_counts(cnt, n_phase, n_mag, n);
    gce_oracle_overlap_counts(cnt, n_phase, n_mag, tmp);
    return gce_oracle_ce_from_counts(tmp, n_phase, n_mag, 2 * n);
}

static int ce_search_impl(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                          const double *periods, int64_t n_p, const double *pdots, int64_t n_pdot,
                          int32_t n_phase, int32_t n_mag, double *out_ce, int32_t n_threads, int overlap)
{
    if (n_lc < 0 || n_p < 0 || n_pdot < 1 || n_phase < 1 || n_mag < 1) return GCE_ORACLE_EINVAL;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
    for (int32_t l = 0; l < n_lc; ++l) {
        const int64_t off = lc_offsets[l], n = lc_offsets[l + 1] - off;
        if (n < 0) return GCE_ORACLE_EINVAL;
        double *dt = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
        double *dt2 = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
        int32_t *mbin = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
        gce_oracle_preprocess(times + off, mags + off, n, n_mag, dt, dt2, mbin);
        double *ce_l = out_ce + (int64_t)l * n_p * n_pdot;
#pragma omp parallel
        {
            int64_t *cnt = (int64_t *)malloc(sizeof(int64_t) * 2 * (size_t)n_phase * (size_t)n_mag);
            int64_t *tmp = cnt + (size_t)n_phase * (size_t)n_mag;
#pragma omp for schedule(static)
            for (int64_t ip = 0; ip < n_p; ++ip) {
                for (int64_t ipd = 0; ipd < n_pdot; ++ipd) {
                    histogram_one_trial(dt, dt2, mbin, n, periods[ip], pdots[ipd], n_phase, n_mag, cnt);
                    ce_l[ip * n_pdot + ipd] = ce_one_trial(cnt, tmp, n_phase, n_mag, n, overlap);
                }
            }
            free(cnt);
        }
        free(dt); free(dt2); free(mbin);
    }
    return GCE_ORACLE_OK;
}

int gce_oracle_ce_search(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                         const double *periods, int64_t n_p, const double *pdots, int64_t n_pdot,
                         int32_t n_phase, int32_t n_mag, double *out_ce, int32_t n_threads)
{
    return ce_search_impl(times, mags, lc_offsets, n_lc, periods, n_p, pdots, n_pdot, n_phase, n_mag, out_ce,
                          n_threads, 0);
}

int gce_oracle_ce_search_overlap(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                                 const double *periods, int64_t n_p, const double *pdots, int64_t n_pdot,
                                 int32_t n_phase, int32_t n_mag, double *out_ce, int32_t n_threads)
{
    return ce_search_impl(times, mags, lc_offsets, n_lc, periods, n_p, pdots, n_pdot, n_phase, n_mag, out_ce,
                          n_threads, 1);
}

/* CE at a list of flat trial indices (the same list for every light curve): sampled parity at
 * full-size grids.  out_ce layout [n_lc][n_trials]. */
static int ce_at_impl(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                      const double *periods, int64_t n_p, const double *pdots, int64_t n_pdot,
                      int32_t n_phase, int32_t n_mag, const int64_t *trial_q, int64_t n_trials,
                      double *out_ce, int32_t n_threads, int overlap)
{
    if (n_lc < 0 || n_p < 0 || n_pdot < 1 || n_phase < 1 || n_mag < 1) return GCE_ORACLE_EINVAL;
    for (int64_t s = 0; s < n_trials; ++s)
        if (trial_q[s] < 0 || trial_q[s] >= n_p * n_pdot) return GCE_ORACLE_EINVAL;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
    for (int32_t l = 0; l < n_lc; ++l) {
        const int64_t off = lc_offsets[l], n = lc_offsets[l + 1] - off;
        if (n < 0) return GCE_ORACLE_EINVAL;
        double *dt = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
        double *dt2 = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
        int32_t *mbin = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
        gce_oracle_preprocess(times + off, mags + off, n, n_mag, dt, dt2, mbin);
#pragma omp parallel
        {
            int64_t *cnt = (int64_t *)malloc(sizeof(int64_t) * 2 * (size_t)n_phase * (size_t)n_mag);
            int64_t *tmp = cnt + (size_t)n_phase * (size_t)n_mag;
#pragma omp for schedule(static)
            for (int64_t s = 0; s < n_trials; ++s) {
                const int64_t q = trial_q[s];
                histogram_one_trial(dt, dt2, mbin, n, periods[q / n_pdot], pdots[q % n_pdot], n_phase, n_mag, cnt);
                out_ce[(int64_t)l * n_trials + s] = ce_one_trial(cnt, tmp, n_phase, n_mag, n, overlap);
            }
            free(cnt);
        }
        free(dt); free(dt2); free(mbin);
    }
    return GCE_ORACLE_OK;
}

int gce_oracle_ce_at(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                     const double *periods, int64_t n_p, const double *pdots, int64_t n_pdot,
                     int32_t n_phase, int32_t n_mag, const int64_t *trial_q, int64_t n_trials,
                     double *out_ce, int32_t n_threads)
{
    return ce_at_impl(times, mags, lc_offsets, n_lc, periods, n_p, pdots, n_pdot, n_phase, n_mag, trial_q, n_trials,
                      out_ce, n_threads, 0);
}

int gce_oracle_ce_at_overlap(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                             const double *periods, int64_t n_p, const double *pdots, int64_t n_pdot,
                             int32_t n_phase, int32_t n_mag, const int64_t *trial_q, int64_t n_trials,
                             double *out_ce, int32_t n_threads)
{
    return ce_at_impl(times, mags, lc_offsets, n_lc, periods, n_p, pdots, n_pdot, n_phase, n_mag, trial_q, n_trials,
                      out_ce, n_threads, 1);
}

/* ---------------------------------------------------------------------------------------
 * S5  best / top-k ("the lowest Conditional Entropy value indicates the most
 * likely period", :112): trials ordered by (CE ascending, flat index q ascending) (Q9); the
 * first k are returned.  One scan with a sorted list of the k best so far; a later trial only
 * displaces an entry when its CE is strictly smaller, so equal CE keeps the smaller q first.
 * NaN CE (empty light curve) never enters; unused slots get idx = -1, val = NaN.
 * ------------------------------------------------------------------------------------- */
int gce_oracle_topk(const double *ce, int64_t n_trials, int32_t k, int64_t *out_idx, double *out_val)
{
    if (k < 0 || n_trials < 0) return GCE_ORACLE_EINVAL;
    int32_t filled = 0;
    for (int32_t r = 0; r < k; ++r) { out_idx[r] = -1; out_val[r] = NAN; }
    for (int64_t q = 0; q < n_trials; ++q) {
        const double v = ce[q];
        if (v != v) continue;
        if (filled == k && !(v < out_val[k - 1])) continue;
        int32_t pos = filled < k ? filled : k - 1;
        while (pos > 0 && v < out_val[pos - 1]) {
            out_val[pos] = out_val[pos - 1];
            out_idx[pos] = out_idx[pos - 1];
            --pos;
        }
        out_val[pos] = v;
        out_idx[pos] = q;
        if (filled < k) ++filled;
    }
    return GCE_ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------
 * Significance (Eq. 5): rho = (mu - H_c,min) / sigma with mu, sigma the mean
 * and (population, Q13) standard deviation of all CE values of one light curve.
 * Two-pass mean / variance.  out = {mu, sigma, rho}.
 * ------------------------------------------------------------------------------------- */
int gce_oracle_significance(const double *ce, int64_t n_trials, double *out3)
{
    if (n_trials <= 0) { out3[0] = out3[1] = out3[2] = NAN; return GCE_ORACLE_OK; }
    double sum = 0.0, mn = ce[0];
    for (int64_t q = 0; q < n_trials; ++q) { sum += ce[q]; if (ce[q] < mn) mn = ce[q]; }
    const double mu = sum / (double)n_trials;
    double ss = 0.0;
    for (int64_t q = 0; q < n_trials; ++q) { const double d = ce[q] - mu; ss += d * d; }
    const double sigma = sqrt(ss / (double)n_trials);
    out3[0] = mu; out3[1] = sigma; out3[2] = (mu - mn) / sigma;
    return GCE_ORACLE_OK;
}

int gce_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
