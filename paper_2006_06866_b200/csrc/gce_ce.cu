// gce_ce.cu -- B200 (sm_100a) kernels and C ABI of the Conditional Entropy (P, Pdot) search.
//
// Path (citations are PAPER.md lines of arXiv 2006.06866):
//   k_preprocess  S1  t0 / min-max / magnitude bin per point, points grouped by magnitude bin      (:96)
//                     (+ the fixed-point table L(k) = k ln k used by S4, built by the same launch)
//   k_search      S2  fp64 fold, Eq. 3, frozen operation order               (:100)
//                 S3  per-trial private histogram in shared memory                                 (:106)
//                 S4  N*CE = sum_j L(n_j) - sum_ij L(n_ij), exact integer accumulation, Eq. 4      (:108)
//                 S5  CE cube store + per-warp running top-k                                       (:49, :112)
//   k_merge_topk  S5  per-light-curve merge of the per-CTA candidates
//
// Design (B200-first): one THREAD owns R consecutive trials (the paper's one-thread-
// per-grid-point idea, :152, kept because it makes every shared-memory access conflict-free).  The R trials of a
// thread share one period whenever n_pdot % R == 0, so a = dt * invP is computed once per point.  The whole light
// curve is staged in shared memory by TMA bulk copies (cp.async.bulk + mbarrier) once per CTA and read by every
// thread as a broadcast LDS.128; light curves longer than the buffer are streamed through two half buffers.
// Points are pre-grouped by magnitude bin so a trial only needs a 1-D phase histogram at a time (the paper's
// memory insight, :152); counters are 16-bit pairs in a [bin][thread] column layout (bank = lane), updated with
// one RED.shared per point-fold; the phase marginal lives in registers (compile-time n_phi) and the entropy is
// accumulated in 2^-42 fixed point so CE does not depend on summation order.  The phase bin is
// floor(y) - n_phi * floor(x) from two round-down magic adds (exact for |y| < 2^51, no integer division: on sm_100
// IMAD.HI is quarter rate and slows the FP64 pipe, measured in DESIGN.md section 7); where the shared memory allows
// 2 n_phi + 1 counter rows, the trials of a thread share one floor(x) (gce_search.cuh, "MODE 1 / 2").  No tensor
// cores: this is a histogram/entropy path, not a contraction.
//
// This translation unit must be compiled with -fmad=false; the fold additionally uses explicit _rn/_rd
// intrinsics, which are never contracted.
#include <vector>

#include "gce_common.cuh"
#include "gce_preprocess.cuh"
#include "gce_debug.cuh"
#include "gce_select.cuh"
#include "gce_probe.cuh"

namespace {

// ------------------------------------------------------------------------------------------------ host side
thread_local int g_last_cuda_error = 0;

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

constexpr int kMaxThreadsSmemMarg = 640;  // launch bound of the shared-memory-marginal kernels (<= 102 registers)
constexpr int kMinPoints = 640;           // smallest point buffer
constexpr int kMinCtasPerSm = 8, kMaxCtasPerSm = 16;   // CTAs per SM over the whole launch
constexpr double kPointFoldsPerCta = 2.0e7;            // work per CTA the plan aims for
// SMs of the B200 the launch plan is tuned for.  Deliberately a constant, not a device query: the plan (and with it the
// workspace layout and the split of the partial sums) is decided from the sizes alone, so that gce_ce_workspace_bytes
// needs no device and every GPU gives the same CTA split.  On a part with another SM count the results stay the same
// and only the fill of the last round of CTAs degrades.
constexpr int64_t kNumSms = 148;

size_t search_smem_fixed() {  // mbarriers, seg row, Eq. 5 accumulators, the warps' top-k lists + thresholds, light-curve scalars
    return sizeof(uint64_t) * 2 + sizeof(int) * (GCE_CE_MAX_BINS + 4) + sizeof(uint64_t) * kMaxWarps * kStatWords +
           sizeof(int64_t) * kMaxWarps * 64 + sizeof(int64_t) * kMaxWarps * 2 + sizeof(double) * 2;
}
// counter rows of one thread: histogram (n_phi + 1 rows, the last one catches RN(x * n_phi) == n_phi * (floor(x) + 1)),
// plus n_phi marginal rows when the marginal is not in registers; RW words each
size_t search_smem_per_thread(int n_phi, int R, bool regm, bool ext = false, bool wide = false) {
    const int hist_rows = ext ? 2 * n_phi + 1 : n_phi + 1;
    return (size_t)(wide ? R : (R + 1) / 2) * (size_t)(regm ? hist_rows : hist_rows + n_phi) * sizeof(uint32_t);
}

// Points per light curve this call accepts, and whether it needs the 32-bit counters: the 16-bit range unless the
// caller has announced longer light curves (gce_ce_params.max_lc_points).
int64_t narrow_limit(const gce_ce_params *prm) { return prm->overlap ? GCE_CE_MAX_POINTS_OVERLAP : GCE_CE_MAX_POINTS; }
bool is_wide(const gce_ce_params *prm) { return (int64_t)prm->max_lc_points > narrow_limit(prm); }
int64_t points_limit(const gce_ce_params *prm) { return is_wide(prm) ? (int64_t)prm->max_lc_points : narrow_limit(prm); }

// Fixed-point shift of the k ln k table: the largest shift, between 42 and 52 for tables within the 16-bit counter range
// and at most 42 beyond it, that keeps L(k_max) 2^shift below 2^60 (narrow) / 2^61 (wide) -- and with it every sum of
// table entries of one trial, which is at most L(k_max).  Short tables (a call whose light curves are short: k_max is
// bounded by the call's total_points) leave spare bits in the 64-bit sums, and spending them shrinks the quantisation
// term of CE (reading Q21): k_max = 200 -> 2^-49, 1000 -> 2^-47, 5000 -> 2^-44, >= 11 000 -> 2^-42 as before.
// Eq. 5 needs more than S < 2^61: a warp adds up to 128 squares of d = S - K in 128 bits, so |d| <= max(S, K) must stay
// below 2^60.5.  S and K are at most mult N ln(n_m) 2^shift and at most L(k_max) 2^shift: narrow calls stay below
// min(2^60, 65535 * 4.16 * 2^42 = 2^60.1), and beyond the 16-bit range ln(k_max) > 11.09 > ln 64, so
// N ln(n_m) 2^shift < L(k_max) 2^shift * 4.16 / 11.09 < 2^59.6.
int table_shift(int64_t ltab_n) {
    const double kmax = (double)(ltab_n - 1);
    if (kmax < 2.0) return 52;  // the table is all zeros
    const int bits = (int)ceil(log2(kmax * log(kmax)));
    if (kmax <= (double)GCE_CE_MAX_POINTS) {
        const int s = 60 - bits;
        return s < kLfixShift ? kLfixShift : (s > 52 ? 52 : s);
    }
    return 61 - bits < kLfixShift ? 61 - bits : kLfixShift;
}

// Trials per thread and whether they share a period: from the grid shape alone (also used by gce_ce_debug_bins).
void plan_trials(int64_t n_pdot, int n_phi, int *R, bool *share_p) {
    if (n_pdot % 4 == 0) { *R = 4; *share_p = true; }
    else if (n_pdot % 2 == 0) { *R = 2; *share_p = true; }
    else { *R = 4; *share_p = false; }
    // 50 phase bins (the paper's production binning): the register marginal of R = 4 trials would take
    // 100 registers, so a thread owns R = 2 trials and 512 threads still fit (measured 2x the generic variant)
    if (n_phi == 50) { *R = 2; *share_p = (n_pdot % 2 == 0); }
}

Plan make_plan(int32_t n_lc, int64_t total_points, int64_t n_trials, int64_t n_pdot, int n_phi, bool wide) {
    Plan p;
    p.wide = wide;
    plan_trials(n_pdot, wide ? 0 : n_phi, &p.R, &p.share_p);
    const int64_t avail = (int64_t)kSmemLimit - (int64_t)search_smem_fixed();
    const bool templ = !wide && (n_phi == 15 || n_phi == 20 || n_phi == 30 || n_phi == 50);  // wide counters: generic family
    // point buffer wanted: the average light curve plus a quarter (the per-LC lengths live on the device; a longer
    // light curve is streamed through the buffer in two halves instead of staying resident)
    const int64_t avg = n_lc > 0 ? (total_points + n_lc - 1) / n_lc : 0;
    int64_t want_pts = (avg + avg / 4 + 15) / 8 * 8;
    if (want_pts < kMinPoints) want_pts = kMinPoints;
    if (want_pts > 8192) want_pts = 8192;
    auto threads_beside = [&](int64_t pts, bool regm) {
        int64_t nt = (avail - (pts + 2) * (int64_t)sizeof(double2)) / (int64_t)search_smem_per_thread(n_phi, p.R, regm, false, wide);
        return nt < 0 ? 0 : nt / 32 * 32;
    };
    int64_t nt_s = threads_beside(want_pts, false);
    if (nt_s > kMaxThreadsSmemMarg) nt_s = kMaxThreadsSmemMarg;
    const bool regm_fits = templ && threads_beside(kMinPoints, true) >= nt_regm(n_phi);
    // measured on C3: register marginals beat 608 threads with shared-memory marginals (83.7 vs
    // 86.8 ms), so the register variant is taken whenever it fits; its thread count is per family (nt_regm)
    if (regm_fits) {
        p.regm = true;
        p.nt = nt_regm(n_phi);
    } else {
        p.regm = false;
        if (nt_s < 32) nt_s = threads_beside(kMinPoints, false);
        if (nt_s > kMaxThreadsSmemMarg) nt_s = kMaxThreadsSmemMarg;
        p.nt = (int)nt_s;  // >= 32: 64 x 64 bins with R = 4 leave room for 192 threads
    }
    p.nphi_t = (templ && p.regm) ? n_phi : 0;  // compile-time n_phi kernels exist with register marginals only
    // extended rows (one FP64 instruction fewer per two point-folds, C3: 83 -> 77 ms): instantiated for n_phi = 15 and
    // 20 with R = 4 trials sharing a period; taken when the whole average light curve still fits beside the counters
    p.ext = p.regm && p.share_p && p.R == 4 && (n_phi == 15 || n_phi == 20) && n_pdot > 1 &&
            (avail - (int64_t)search_smem_per_thread(n_phi, p.R, true, true) * p.nt) / (int64_t)sizeof(double2) - 2 >= want_pts;
    const int64_t planes = (int64_t)search_smem_per_thread(n_phi, p.R, p.regm, p.ext, wide) * p.nt;
    int64_t cap = (avail - planes) / (int64_t)sizeof(double2) - 2;  // - 2: read-ahead slack of the hot loop
    cap = cap / 8 * 8;
    if (cap > 8192) cap = 8192;  // 128 KB of points; longer light curves are streamed
    p.cap_points = (int)cap;
    p.smem = (size_t)(cap + 2) * sizeof(double2) + search_smem_fixed() + (size_t)planes;
    const int64_t tile = (int64_t)p.nt * p.R;
    p.tiles_per_lc = n_trials > 0 ? (n_trials + tile - 1) / tile : 0;
    // CTAs over the whole launch: enough for dynamic balance at the tail, few enough that a CTA's set-up (zeroing its
    // counters, staging the light curve, merging its top-k) stays small against its work -- about 2e7 point-folds per
    // CTA, between 8 and 16 CTAs per SM (measured: C4 9.14 -> 9.03 ms from 16 to 8 per SM; C5 indifferent between 8 and
    // 64 except 48: +1.3 %); at least one tile per job
    const int64_t lcs = n_lc > 0 ? n_lc : 1;
    int64_t ctas = (int64_t)((double)total_points * (double)n_trials / kPointFoldsPerCta);
    if (ctas < kNumSms * kMinCtasPerSm) ctas = kNumSms * kMinCtasPerSm;
    if (ctas > kNumSms * kMaxCtasPerSm) ctas = kNumSms * kMaxCtasPerSm;
    int64_t want = (ctas + lcs - 1) / lcs;
    if (want > p.tiles_per_lc) want = p.tiles_per_lc;
    if (want < 1) want = 1;
    if (want > 4096) want = 4096;
    // One CTA per SM at a time and CTAs of about equal length: the launch takes ceil(CTAs / kNumSms) rounds, so a CTA count
    // just above a multiple of kNumSms wastes most of its last round (P1: 100 light curves x 24 jobs = 16.2 rounds).  Up to
    // twice the jobs are taken when that fills the last round better.
    auto fill = [&](int64_t j) {
        const double rounds = (double)(lcs * j) / (double)kNumSms;
        return rounds / ceil(rounds);
    };
    int64_t best = want;
    for (int64_t j = want + 1; j <= 2 * want && j <= p.tiles_per_lc && j <= 4096; ++j)
        if (fill(j) > fill(best) + 1e-9) best = j;
    want = best;
    p.jobs_per_lc = (int)want;
    return p;
}

struct Layout {
    size_t pts, seg, info, ltab, part_S, part_q, part_stats, mnorm, total;
    int ltab_n;
};

Layout make_layout(int64_t total_points, int32_t n_lc, int64_t n_trials, int64_t n_pdot, const gce_ce_params *prm) {
    Layout L;
    size_t o = 0;
    L.pts = o; o = align_up(o + sizeof(double2) * (size_t)(total_points > 0 ? total_points : 1), 256);
    L.seg = o; o = align_up(o + sizeof(int32_t) * (size_t)(n_lc > 0 ? n_lc : 1) * (prm->n_mag_bins + 1), 256);
    L.info = o; o = align_up(o + sizeof(LcInfo) * (size_t)(n_lc > 0 ? n_lc : 1), 256);
    // largest count looked up: the longest light curve's N, or 2N with overlapping bins
    int64_t longest = total_points < points_limit(prm) ? total_points : points_limit(prm);
    int64_t tn = (prm->overlap ? 2 : 1) * longest;
    if (!is_wide(prm) && tn > GCE_CE_MAX_POINTS) tn = GCE_CE_MAX_POINTS;
    L.ltab_n = (int)tn + 1;
    L.ltab = o; o = align_up(o + sizeof(int64_t) * (size_t)L.ltab_n, 256);
    const Plan p = make_plan(n_lc, total_points, n_trials, n_pdot, prm->n_phase_bins, is_wide(prm));
    const size_t parts = (size_t)(n_lc > 0 ? n_lc : 1) * (size_t)p.jobs_per_lc * (size_t)(prm->top_k > 0 ? prm->top_k : 1);
    L.part_S = o; o = align_up(o + sizeof(int64_t) * parts, 256);
    L.part_q = o; o = align_up(o + sizeof(int64_t) * parts, 256);
    L.part_stats = o;
    if (prm->want_stats) o = align_up(o + sizeof(uint64_t) * kStatWords * (size_t)(n_lc > 0 ? n_lc : 1) * (size_t)p.jobs_per_lc, 256);
    L.mnorm = o;
    if (prm->normalise) o = align_up(o + sizeof(double) * (size_t)(total_points > 0 ? total_points : 1), 256);
    L.total = o;
    return L;
}

int check_params(const gce_ce_params *prm) {
    if (!prm) return GCE_CE_ERR_POINTER;
    if (prm->n_phase_bins < 1 || prm->n_phase_bins > GCE_CE_MAX_BINS) return GCE_CE_ERR_RANGE;
    if (prm->n_mag_bins < 1 || prm->n_mag_bins > GCE_CE_MAX_BINS) return GCE_CE_ERR_RANGE;
    if (prm->top_k < 0 || prm->top_k > GCE_CE_MAX_TOPK) return GCE_CE_ERR_RANGE;
    if (prm->ce_fp64 != 0 && prm->ce_fp64 != 1) return GCE_CE_ERR_RANGE;
    if (prm->want_stats != 0 && prm->want_stats != 1) return GCE_CE_ERR_RANGE;
    if (prm->overlap != 0 && prm->overlap != 1) return GCE_CE_ERR_RANGE;
    if (prm->max_lc_points < 0 || prm->max_lc_points > GCE_CE_MAX_POINTS_WIDE) return GCE_CE_ERR_RANGE;
    if (prm->normalise != 0 && prm->normalise != 1) return GCE_CE_ERR_RANGE;
    return GCE_CE_OK;
}

int check_sizes(int32_t n_lc, int64_t total_points, int64_t n_p, int64_t n_pdot) {
    if (n_lc < 0 || total_points < 0 || n_p < 0 || n_pdot < 1) return GCE_CE_ERR_RANGE;
    if (n_lc > (1 << 24)) return GCE_CE_ERR_RANGE;
    if (n_p > 0 && n_pdot > (int64_t)0x7fffffffffffLL / n_p) return GCE_CE_ERR_RANGE;
    return GCE_CE_OK;
}

// Light-curve lengths from a HOST copy of lc_offsets: non-negative and within the counter range.
int check_lengths_host(const int64_t *lc_offsets, int32_t n_lc, const gce_ce_params *prm) {
    if (n_lc > 0 && lc_offsets[0] != 0) return GCE_CE_ERR_RANGE;
    const int64_t lim = points_limit(prm);
    for (int32_t l = 0; l < n_lc; ++l) {
        const int64_t n = lc_offsets[l + 1] - lc_offsets[l];
        if (n < 0 || n > lim) return GCE_CE_ERR_RANGE;
    }
    return GCE_CE_OK;
}

// Host entries: raise max_lc_points to the longest light curve when that is beyond the 16-bit range.
void host_set_max_lc_points(const int64_t *lc_offsets, int32_t n_lc, gce_ce_params *prm) {
    int64_t longest = 0;
    for (int32_t l = 0; l < n_lc; ++l) {
        const int64_t n = lc_offsets[l + 1] - lc_offsets[l];
        if (n > longest) longest = n;
    }
    if (longest > narrow_limit(prm) && longest <= GCE_CE_MAX_POINTS_WIDE && longest > (int64_t)prm->max_lc_points)
        prm->max_lc_points = (int32_t)longest;
}

int cuda_fail(cudaError_t e) {
    g_last_cuda_error = (int)e;
    return GCE_CE_ERR_CUDA;
}

int dispatch_search(const SearchParams &sp, const Plan &plan, bool dump, int32_t n_lc, cudaStream_t st) {
    cudaError_t e = cudaErrorInvalidValue;
    switch (plan.nphi_t) {
        case 0: e = dump ? launch_search_n0_d1(sp, plan, n_lc, st) : launch_search_n0_d0(sp, plan, n_lc, st); break;
        case 15: e = dump ? launch_search_n15_d1(sp, plan, n_lc, st) : launch_search_n15_d0(sp, plan, n_lc, st); break;
        case 20: e = dump ? launch_search_n20_d1(sp, plan, n_lc, st) : launch_search_n20_d0(sp, plan, n_lc, st); break;
        case 30: e = dump ? launch_search_n30_d1(sp, plan, n_lc, st) : launch_search_n30_d0(sp, plan, n_lc, st); break;
        case 50: e = dump ? launch_search_n50_d1(sp, plan, n_lc, st) : launch_search_n50_d0(sp, plan, n_lc, st); break;
        default: break;
    }
    return e == cudaSuccess ? GCE_CE_OK : cuda_fail(e);
}

}  // namespace

// ================================================================================================ C ABI
extern "C" {

const char *gce_ce_version(void) { return "gce-b200 0.3 (sm_100a)"; }

const char *gce_ce_strerror(int code) {
    switch (code) {
        case GCE_CE_OK: return "ok";
        case GCE_CE_ERR_POINTER: return "null or inconsistent pointer arguments";
        case GCE_CE_ERR_RANGE: return "size, bin count, light-curve length or option out of range";
        case GCE_CE_ERR_WORKSPACE: return "workspace too small or misaligned";
        case GCE_CE_ERR_CUDA: return "CUDA runtime error (see gce_ce_last_cuda_error)";
        case GCE_CE_ERR_STATIC_LIMIT: return "call needs more scratch than GCE_CE_STATIC_SCRATCH_BYTES (use gce_ce_search with a workspace)";
        default: return "unknown error code";
    }
}

int gce_ce_last_cuda_error(void) { return g_last_cuda_error; }

int gce_ce_launch_count(int32_t n_lc, int64_t n_p, const gce_ce_params *prm, int partial) {
    if (!prm || n_lc <= 0) return 0;
    // [normalise], preprocess (+ table), search (when the grid is not empty), [merge_topk], [merge_stats: Eq. 5 and every partial blob]
    return (prm->normalise ? 1 : 0) + 1 + (n_p > 0 ? 1 : 0) + (prm->top_k > 0 ? 1 : 0) + ((prm->want_stats || partial) ? 1 : 0);
}

int gce_ce_workspace_bytes(int64_t total_points, int32_t n_lc, int64_t n_p, int64_t n_pdot, const gce_ce_params *prm,
                           size_t *bytes) {
    if (!bytes) return GCE_CE_ERR_POINTER;
    int rc = check_params(prm);
    if (rc) return rc;
    rc = check_sizes(n_lc, total_points, n_p, n_pdot);
    if (rc) return rc;
    *bytes = make_layout(total_points, n_lc, n_p * n_pdot, n_pdot, prm).total;
    return GCE_CE_OK;
}

// Every fallible host-side step (argument, plan and workspace checks) comes before the first launch; after that only a
// failing launch or event record can return an error, and then the outputs are undefined.
static int run_search(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                      int64_t total_points, const double *periods, int64_t n_p, const double *pdots, int64_t n_pdot,
                      const gce_ce_params *prm, void *out_ce, int64_t *out_best_idx, float *out_best_ce, double *out_stats,
                      const int64_t *trial_q, int64_t n_dump, uint32_t *out_counts, double *out_ce_at, int64_t ip_begin,
                      int64_t *out_partial, void *workspace, size_t workspace_bytes, void *stream) {
    // periods / n_p describe THIS call's period range; ip_begin is its offset in the caller's grid (0 for a whole grid)
    const bool dump = out_counts != nullptr;
    int rc = check_params(prm);
    if (rc) return rc;
    rc = check_sizes(n_lc, total_points, n_p, n_pdot);
    if (rc) return rc;
    if (!lc_offsets || !workspace) return GCE_CE_ERR_POINTER;
    if (total_points > 0 && (!times || !mags)) return GCE_CE_ERR_POINTER;
    if (n_p > 0 && !periods) return GCE_CE_ERR_POINTER;
    if (!pdots) return GCE_CE_ERR_POINTER;
    if (dump) {
        if (n_dump < 0 || n_dump > 0x7fffffff) return GCE_CE_ERR_RANGE;
        if (n_dump > 0 && !trial_q) return GCE_CE_ERR_POINTER;
    } else {
        if (out_partial) {
            if (out_best_idx || out_best_ce || out_stats) return GCE_CE_ERR_POINTER;
        } else {
            if (!out_ce && !out_best_idx && !out_stats) return GCE_CE_ERR_POINTER;
            if ((prm->want_stats != 0) != (out_stats != nullptr)) return GCE_CE_ERR_POINTER;
            if ((prm->top_k > 0) != (out_best_idx != nullptr)) return GCE_CE_ERR_POINTER;
            if (out_best_ce && !out_best_idx) return GCE_CE_ERR_POINTER;
        }
    }
    // more points than every light curve could hold within the counter range: some light curve must be too long
    const int64_t max_points = points_limit(prm);
    if (total_points > (int64_t)n_lc * max_points) return GCE_CE_ERR_RANGE;
    const int64_t n_trials = n_p * n_pdot;
    const int mult = prm->overlap ? 2 : 1;
    const Layout L = make_layout(total_points, n_lc, n_trials, n_pdot, prm);
    if (workspace_bytes < L.total || (reinterpret_cast<uintptr_t>(workspace) & 255u)) return GCE_CE_ERR_WORKSPACE;
    if (n_lc == 0) return GCE_CE_OK;

    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    if (dump && n_dump > 0) {  // the dump kernels only write the cells that hold points; first launch-side effect of the call
        cudaError_t em = cudaMemsetAsync(out_counts, 0, sizeof(uint32_t) * (size_t)n_lc * (size_t)n_dump * prm->n_phase_bins * prm->n_mag_bins, st);
        if (em != cudaSuccess) return cuda_fail(em);
    }
    unsigned char *ws = reinterpret_cast<unsigned char *>(workspace);
    double2 *pts = reinterpret_cast<double2 *>(ws + L.pts);
    int32_t *seg = reinterpret_cast<int32_t *>(ws + L.seg);
    LcInfo *info = reinterpret_cast<LcInfo *>(ws + L.info);
    int64_t *ltab = reinterpret_cast<int64_t *>(ws + L.ltab);

    const Plan plan = make_plan(n_lc, total_points, n_trials, n_pdot, prm->n_phase_bins, is_wide(prm));
    SearchParams sp;
    memset(&sp, 0, sizeof(sp));
    sp.pts = pts; sp.seg = seg; sp.info = info; sp.lc_offsets = lc_offsets; sp.ltab = ltab;
    sp.periods = periods; sp.pdots = pdots; sp.trial_q = trial_q; sp.n_dump = n_dump;
    sp.n_p = n_p; sp.n_pdot = n_pdot; sp.n_trials = n_trials;
    sp.q_off = ip_begin * n_pdot;
    sp.jobs_per_lc = plan.jobs_per_lc;
    sp.tiles_per_lc = plan.tiles_per_lc;
    sp.cap_points = plan.cap_points;
    sp.n_phi = prm->n_phase_bins; sp.n_m = prm->n_mag_bins;
    sp.ltab_n = L.ltab_n;
    sp.top_k = dump ? 0 : prm->top_k;
    sp.ce_fp64 = prm->ce_fp64;
    sp.overlap = prm->overlap;
    sp.out_ce = out_ce;
    sp.part_S = reinterpret_cast<int64_t *>(ws + L.part_S);
    sp.part_q = reinterpret_cast<int64_t *>(ws + L.part_q);
    sp.part_stats = (!dump && prm->want_stats) ? reinterpret_cast<uint64_t *>(ws + L.part_stats) : nullptr;
    sp.out_counts = out_counts; sp.out_ce_at = out_ce_at;

    const double *mags_used = mags;
    if (prm->normalise && total_points > 0) {  // S0 (N4): per-filter median / std into the workspace
        double *mnorm = reinterpret_cast<double *>(ws + L.mnorm);
        k_normalise<<<n_lc, 256, 0, st>>>(mags, prm->filter_ids, lc_offsets, mnorm);
        cudaError_t en = cudaGetLastError();
        if (en != cudaSuccess) return cuda_fail(en);
        mags_used = mnorm;
    }
    k_preprocess<<<n_lc + (L.ltab_n + 255) / 256, 256, 0, st>>>(times, mags_used, lc_offsets, n_lc, prm->n_mag_bins, pts, seg, info,
                                                              ltab, L.ltab_n, table_shift(L.ltab_n), mult, (int)max_points);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);
    if (prm->ev_search_begin) {
        e = cudaEventRecord(reinterpret_cast<cudaEvent_t>(prm->ev_search_begin), st);
        if (e != cudaSuccess) return cuda_fail(e);
    }
    if (n_trials > 0 && !(dump && n_dump == 0)) {
        rc = dispatch_search(sp, plan, dump, n_lc, st);
        if (rc) return rc;
    }
    if (prm->ev_search_end) {
        e = cudaEventRecord(reinterpret_cast<cudaEvent_t>(prm->ev_search_end), st);
        if (e != cudaSuccess) return cuda_fail(e);
    }
    const int K = prm->top_k;
    const int n_jobs = n_trials > 0 ? plan.jobs_per_lc : 0;
    const int W = partial_words(K);
    if (!dump && K > 0) {
        k_merge_topk<<<n_lc, 32, 0, st>>>(sp.part_S, sp.part_q, (int64_t)plan.jobs_per_lc * K, K, n_jobs, K, info, nullptr, 0,
                                          mult, out_best_idx, out_best_ce, out_partial, W);
        e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(e);
    }
    if (!dump && (prm->want_stats || out_partial)) {
        k_merge_stats<<<n_lc, 32, 0, st>>>(sp.part_stats, (int64_t)plan.jobs_per_lc * kStatWords, kStatWords,
                                           prm->want_stats ? n_jobs : 0, info, nullptr, 0, mult, out_stats,
                                           out_partial ? out_partial + 2 * K : nullptr, W);
        e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(e);
    }
    return GCE_CE_OK;
}

int gce_ce_search(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                  int64_t total_points, const double *periods, int64_t n_p, const double *pdots, int64_t n_pdot,
                  const gce_ce_params *prm, void *out_ce, int64_t *out_best_idx, float *out_best_ce, double *out_stats,
                  void *workspace, size_t workspace_bytes, void *stream) {
    return run_search(times, mags, lc_offsets, n_lc, total_points, periods, n_p, pdots, n_pdot, prm, out_ce,
                      out_best_idx, out_best_ce, out_stats, nullptr, 0, nullptr, nullptr, 0, nullptr, workspace, workspace_bytes, stream);
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------ gce_ce_search_static
// Scratch of the entry point for callers that may not allocate (guests of another program's GPU process: no allocator
// handed to them, cudaMalloc banned because it stalls the device and may fail late; see include/gce_ce.h).  The array is
// part of this translation unit's device image: every GPU that loads the library holds these 8 MiB until the process
// exits.  In HOST code the name below is only the handle the runtime registered for the symbol -- it is not a device
// address and must never be passed to a kernel (the kernel would fault, or where the GPU can reach host memory, quietly
// work on the wrong bytes).  Host code gets the device address once per device from cudaGetSymbolAddress, with that
// device current, and passes THAT pointer on.
static __device__ __align__(256) unsigned char g_static_scratch[GCE_CE_STATIC_SCRATCH_BYTES];

namespace {
std::mutex g_static_mutex;
void *g_static_addr[64] = {};  // device address of g_static_scratch on each device, 0 = not looked up yet

// Device address of the scratch array on the current device; the first call per device does the look-up.
cudaError_t static_scratch_addr(void **addr) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_addr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return e;
        if (!p || (reinterpret_cast<uintptr_t>(p) & 255u)) return cudaErrorInvalidSymbol;
        g_static_addr[dev] = p;
    }
    *addr = g_static_addr[dev];
    return cudaSuccess;
}
}  // namespace

extern "C" {

// No cudaMalloc / cudaFree / pool call anywhere below: size checks on the host, one address look-up, then run_search,
// which only launches kernels and records the caller's events.  The scratch is shared by every call on the device and
// is not cleared: each call writes what it later reads (the existing path runs on uninitialised workspaces too).
int gce_ce_search_static(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                         int64_t total_points, const double *periods, int64_t n_p, const double *pdots, int64_t n_pdot,
                         const gce_ce_params *prm, void *out_ce, int64_t *out_best_idx, float *out_best_ce,
                         double *out_stats, void *stream) {
    int rc = check_params(prm);
    if (rc) return rc;
    rc = check_sizes(n_lc, total_points, n_p, n_pdot);
    if (rc) return rc;
    if (total_points > (int64_t)n_lc * points_limit(prm)) return GCE_CE_ERR_RANGE;  // some light curve is too long (as in run_search)
    if (make_layout(total_points, n_lc, n_p * n_pdot, n_pdot, prm).total > (size_t)GCE_CE_STATIC_SCRATCH_BYTES)
        return GCE_CE_ERR_STATIC_LIMIT;
    void *scratch = nullptr;
    const cudaError_t e = static_scratch_addr(&scratch);
    if (e != cudaSuccess) return cuda_fail(e);
    return run_search(times, mags, lc_offsets, n_lc, total_points, periods, n_p, pdots, n_pdot, prm, out_ce, out_best_idx,
                      out_best_ce, out_stats, nullptr, 0, nullptr, nullptr, 0, nullptr, scratch,
                      (size_t)GCE_CE_STATIC_SCRATCH_BYTES, stream);
}

size_t gce_ce_partial_words(int32_t top_k) { return (size_t)partial_words(top_k < 0 ? 0 : top_k); }

int gce_ce_search_partial(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                          int64_t total_points, const double *periods, int64_t n_p, const double *pdots, int64_t n_pdot,
                          const gce_ce_params *prm, int64_t ip_begin, int64_t ip_end, void *out_ce, int64_t *out_partial,
                          void *workspace, size_t workspace_bytes, void *stream) {
    if (!out_partial) return GCE_CE_ERR_POINTER;
    if (ip_begin < 0 || ip_end < ip_begin || ip_end > n_p) return GCE_CE_ERR_RANGE;
    return run_search(times, mags, lc_offsets, n_lc, total_points, periods ? periods + ip_begin : periods, ip_end - ip_begin,
                      pdots, n_pdot, prm, out_ce, nullptr, nullptr, nullptr, nullptr, 0, nullptr, nullptr, ip_begin,
                      out_partial, workspace, workspace_bytes, stream);
}

int gce_ce_merge_partials(const int64_t *partials, int32_t n_parts, int32_t n_lc, const gce_ce_params *prm,
                          int64_t *out_best_idx, float *out_best_ce, double *out_stats, void *stream) {
    int rc = check_params(prm);
    if (rc) return rc;
    if (n_parts < 1 || n_lc < 0) return GCE_CE_ERR_RANGE;
    if (!partials) return GCE_CE_ERR_POINTER;
    if ((prm->want_stats != 0) != (out_stats != nullptr)) return GCE_CE_ERR_POINTER;
    if ((prm->top_k > 0) != (out_best_idx != nullptr)) return GCE_CE_ERR_POINTER;
    if (out_best_ce && !out_best_idx) return GCE_CE_ERR_POINTER;
    if (n_lc == 0) return GCE_CE_OK;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    const int K = prm->top_k, W = partial_words(K), mult = prm->overlap ? 2 : 1;
    const int64_t *npts = partials + 2 * K + kStatWords;  // N and the pivot, identical in every part
    if (K > 0) {
        k_merge_topk<<<n_lc, 32, 0, st>>>(partials, partials + K, W, (int64_t)n_lc * W, n_parts, K, nullptr, npts, W, mult,
                                          out_best_idx, out_best_ce, nullptr, 0);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(e);
    }
    if (prm->want_stats) {
        k_merge_stats<<<n_lc, 32, 0, st>>>(reinterpret_cast<const uint64_t *>(partials + 2 * K), W, (int64_t)n_lc * W, n_parts,
                                           nullptr, npts, W, mult, out_stats, nullptr, 0);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(e);
    }
    return GCE_CE_OK;
}

int gce_ce_merge_partials_to_partial(const int64_t *partials, int32_t n_parts, int32_t n_lc, const gce_ce_params *prm,
                                     int64_t *out_partial, void *stream) {
    int rc = check_params(prm);
    if (rc) return rc;
    if (n_parts < 1 || n_lc < 0) return GCE_CE_ERR_RANGE;
    if (!partials || !out_partial) return GCE_CE_ERR_POINTER;
    if (n_lc == 0) return GCE_CE_OK;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    const int K = prm->top_k, W = partial_words(K), mult = prm->overlap ? 2 : 1;
    const int64_t *npts = partials + 2 * K + kStatWords;
    if (K > 0) {
        k_merge_topk<<<n_lc, 32, 0, st>>>(partials, partials + K, W, (int64_t)n_lc * W, n_parts, K, nullptr, npts, W, mult,
                                          nullptr, nullptr, out_partial, W);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(e);
    }
    k_merge_stats<<<n_lc, 32, 0, st>>>(reinterpret_cast<const uint64_t *>(partials + 2 * K), W, (int64_t)n_lc * W, n_parts,
                                       nullptr, npts, W, mult, nullptr, out_partial + 2 * K, W);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);
    return GCE_CE_OK;
}

int gce_ce_debug_histogram(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                           int64_t total_points, const double *periods, int64_t n_p, const double *pdots,
                           int64_t n_pdot, const gce_ce_params *prm, const int64_t *trial_q, int64_t n_trials,
                           uint32_t *out_counts, double *out_ce_at, void *workspace, size_t workspace_bytes,
                           void *stream) {
    if (!out_counts) return GCE_CE_ERR_POINTER;
    return run_search(times, mags, lc_offsets, n_lc, total_points, periods, n_p, pdots, n_pdot, prm, nullptr, nullptr,
                      nullptr, nullptr, trial_q, n_trials, out_counts, out_ce_at, 0, nullptr, workspace, workspace_bytes, stream);
}

int gce_ce_debug_bins(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                      const double *periods, int64_t n_p, const double *pdots, int64_t n_pdot, const gce_ce_params *prm,
                      int32_t lc, int64_t q, int32_t fold_mode, int32_t *out_phase_bin, int32_t *out_mag_bin,
                      int32_t *out_fold_mode, void *stream) {
    int rc = check_params(prm);
    if (rc) return rc;
    if (!times || !mags || !lc_offsets || !periods || !pdots || !out_phase_bin || !out_mag_bin) return GCE_CE_ERR_POINTER;
    if (n_pdot < 1 || n_p < 1 || lc < 0 || lc >= n_lc || q < 0 || q >= n_p * n_pdot) return GCE_CE_ERR_RANGE;
    if (fold_mode < GCE_CE_FOLD_AUTO || fold_mode > GCE_CE_FOLD_PDOT_ZERO) return GCE_CE_ERR_RANGE;
    int R;
    bool share_p;
    plan_trials(n_pdot, is_wide(prm) ? 0 : prm->n_phase_bins, &R, &share_p);  // as make_plan: wide calls run the generic family
    SearchParams sp;
    memset(&sp, 0, sizeof(sp));
    sp.periods = periods; sp.pdots = pdots;
    sp.n_p = n_p; sp.n_pdot = n_pdot; sp.n_trials = n_p * n_pdot;
    sp.n_phi = prm->n_phase_bins; sp.n_m = prm->n_mag_bins;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    if (R == 4 && share_p) k_debug_bins<4, true><<<1, 256, 0, st>>>(times, mags, lc_offsets, sp, lc, q, fold_mode, out_phase_bin, out_mag_bin, out_fold_mode);
    else if (R == 2 && share_p) k_debug_bins<2, true><<<1, 256, 0, st>>>(times, mags, lc_offsets, sp, lc, q, fold_mode, out_phase_bin, out_mag_bin, out_fold_mode);
    else if (R == 4) k_debug_bins<4, false><<<1, 256, 0, st>>>(times, mags, lc_offsets, sp, lc, q, fold_mode, out_phase_bin, out_mag_bin, out_fold_mode);
    else k_debug_bins<2, false><<<1, 256, 0, st>>>(times, mags, lc_offsets, sp, lc, q, fold_mode, out_phase_bin, out_mag_bin, out_fold_mode);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);
    return GCE_CE_OK;
}

int gce_ce_probe_rate(int32_t kind, double *rate_host) {
    if (!rate_host) return GCE_CE_ERR_POINTER;
    if (kind != GCE_CE_PROBE_FP64 && kind != GCE_CE_PROBE_SHARED) return GCE_CE_ERR_RANGE;
    int dev = 0, n_sm = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return cuda_fail(e);
    void *sink = nullptr;
    long long *out = nullptr;
    int rc = GCE_CE_OK;
    std::vector<long long> h((size_t)2 * n_sm);
    do {
        if ((e = cudaMalloc(&sink, (size_t)n_sm * 1024 * sizeof(double))) != cudaSuccess) { rc = cuda_fail(e); break; }
        if ((e = cudaMalloc(&out, sizeof(long long) * 2 * (size_t)n_sm)) != cudaSuccess) { rc = cuda_fail(e); break; }
        for (int pass = 0; pass < 2; ++pass) {  // the first pass warms up (clocks, instruction cache)
            const int iters = pass == 0 ? 200 : 20000;
            if (kind == GCE_CE_PROBE_FP64) k_probe_fp64<<<n_sm, 1024>>>(static_cast<double *>(sink), out, iters, 1.0000001);
            else k_probe_shared<<<n_sm, 1024>>>(static_cast<unsigned *>(sink), out, iters);
            if ((e = cudaGetLastError()) != cudaSuccess) break;
        }
        if (e != cudaSuccess) { rc = cuda_fail(e); break; }
        if ((e = cudaMemcpy(h.data(), out, sizeof(long long) * 2 * (size_t)n_sm, cudaMemcpyDeviceToHost)) != cudaSuccess) { rc = cuda_fail(e); break; }
        double sum = 0.0;
        for (int i = 0; i < n_sm; ++i) sum += (double)h[2 * i] / (double)(h[2 * i + 1] > 0 ? h[2 * i + 1] : 1);
        *rate_host = sum / n_sm;  // mean over the SMs of operations per clock of that SM
    } while (0);
    if (sink) cudaFree(sink);
    if (out) cudaFree(out);
    return rc;
}

int gce_ce_validate_host(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                         const double *periods, int64_t n_p, const double *pdots, int64_t n_pdot,
                         const gce_ce_params *prm_in) {
    int rc = check_params(prm_in);
    if (rc) return rc;
    if (!lc_offsets) return GCE_CE_ERR_POINTER;
    if (n_lc < 0 || n_p < 0 || n_pdot < 1) return GCE_CE_ERR_RANGE;
    if (lc_offsets[0] != 0) return GCE_CE_ERR_RANGE;
    gce_ce_params prm_local = *prm_in;  // what gce_ce_search_host would accept: lengths up to GCE_CE_MAX_POINTS_WIDE
    host_set_max_lc_points(lc_offsets, n_lc, &prm_local);
    const gce_ce_params *prm = &prm_local;
    rc = check_lengths_host(lc_offsets, n_lc, prm);
    if (rc) return rc;
    const int64_t total = lc_offsets[n_lc];
    if (total > 0 && (!times || !mags)) return GCE_CE_ERR_POINTER;
    for (int64_t k = 0; k < total; ++k)
        if (!(times[k] - times[k] == 0.0) || !(mags[k] - mags[k] == 0.0)) return GCE_CE_ERR_RANGE;  // NaN / inf
    if (prm->normalise && prm->filter_ids)  // a HOST pointer here
        for (int64_t k = 0; k < total; ++k)
            if (prm->filter_ids[k] < 0 || prm->filter_ids[k] >= GCE_CE_MAX_FILTERS) return GCE_CE_ERR_RANGE;
    if (n_p > 0 && !periods) return GCE_CE_ERR_POINTER;
    if (!pdots) return GCE_CE_ERR_POINTER;
    for (int64_t i = 0; i < n_p; ++i)
        if (!(periods[i] > 0.0) || !(periods[i] - periods[i] == 0.0)) return GCE_CE_ERR_RANGE;
    for (int64_t i = 0; i < n_pdot; ++i)
        if (!(pdots[i] - pdots[i] == 0.0)) return GCE_CE_ERR_RANGE;
    return GCE_CE_OK;
}

// Device memory of the host-buffer entry points comes from a library-private stream-ordered pool per device whose
// release threshold keeps up to 1 GiB cached between calls (the default pool hands everything back to the driver at
// every synchronisation, which costs 20 - 200 ms per call for a few hundred MB).  gce_ce_host_release() trims it.
static cudaMemPool_t g_host_pool[64] = {};
static std::mutex g_host_pool_mutex;

static cudaError_t host_pool(cudaMemPool_t *pool) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_host_pool_mutex);
    if (!g_host_pool[dev]) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t mp = nullptr;
        e = cudaMemPoolCreate(&mp, &props);
        if (e != cudaSuccess) return e;
        uint64_t keep = 1ull << 30;
        e = cudaMemPoolSetAttribute(mp, cudaMemPoolAttrReleaseThreshold, &keep);
        if (e != cudaSuccess) { cudaMemPoolDestroy(mp); return e; }
        g_host_pool[dev] = mp;
    }
    *pool = g_host_pool[dev];
    return cudaSuccess;
}

int gce_ce_host_release(void) {
    std::lock_guard<std::mutex> lock(g_host_pool_mutex);
    for (int d = 0; d < 64; ++d)
        if (g_host_pool[d]) {
            cudaError_t e = cudaMemPoolTrimTo(g_host_pool[d], 0);
            if (e != cudaSuccess) return cuda_fail(e);
        }
    return GCE_CE_OK;
}

// Streams, events and pool allocations of one host-entry call; everything is released by the destructor, whatever path
// the call leaves on.  CU(x): run a CUDA call, on failure record it and leave the do { } while (0) block.
namespace {
struct HostCall {
    cudaMemPool_t pool = nullptr;
    cudaStream_t st = nullptr, st2 = nullptr;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    void *mem[16] = {};
    int n_mem = 0;
    cudaError_t alloc(void **p, size_t bytes) {
        cudaError_t e = cudaMallocFromPoolAsync(p, bytes ? bytes : 16, pool, st);
        if (e == cudaSuccess) mem[n_mem++] = *p;
        return e;
    }
    ~HostCall() {
        if (st2) cudaStreamSynchronize(st2);
        for (int i = 0; i < n_mem; ++i) cudaFreeAsync(mem[i], st);
        if (st) cudaStreamSynchronize(st);
        for (cudaEvent_t e : ev)
            if (e) cudaEventDestroy(e);
        if (st2) cudaStreamDestroy(st2);
        if (st) cudaStreamDestroy(st);
    }
};
}  // namespace
#define CU(x)                                   \
    {                                           \
        const cudaError_t cu_e_ = (x);          \
        if (cu_e_ != cudaSuccess) {             \
            rc = cuda_fail(cu_e_);              \
            break;                              \
        }                                       \
    }

// Host-buffer entry with the cube requested and a grid worth splitting: the period axis is cut into chunks searched
// back to back on one stream (gce_ce_search_partial, exact merge at the end) while a second stream copies each finished
// cube slice to the caller's buffer, so the device-to-host transfer of the cube overlaps the search of the next chunk.
static int search_host_pipelined(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                                 int64_t total, const double *periods, int64_t n_p, const double *pdots, int64_t n_pdot,
                                 const gce_ce_params *prm_in, void *out_ce, int64_t *out_best_idx, float *out_best_ce,
                                 double *out_stats, int n_chunks) {
    gce_ce_params prm_dev = *prm_in;  // filter_ids: the caller's HOST pointer is replaced by a device copy below
    const gce_ce_params *prm = &prm_dev;
    const int32_t *filt_host = prm_in->normalise ? prm_in->filter_ids : nullptr;
    const size_t esz = prm->ce_fp64 ? 8 : 4;
    const int64_t chunk = (n_p + n_chunks - 1) / n_chunks;
    const size_t k = (size_t)prm->top_k, W = gce_ce_partial_words(prm->top_k);
    size_t ws_bytes = 0;
    int rc = gce_ce_workspace_bytes(total, n_lc, chunk, n_pdot, prm, &ws_bytes);
    if (rc) return rc;
    HostCall hc;
    void *d_t = nullptr, *d_m = nullptr, *d_off = nullptr, *d_p = nullptr, *d_pd = nullptr, *d_ws = nullptr;
    void *d_sl[2] = {nullptr, nullptr}, *d_part = nullptr, *d_idx = nullptr, *d_bce = nullptr, *d_st = nullptr;
    const size_t slice_bytes = (size_t)n_lc * (size_t)chunk * (size_t)n_pdot * esz;
    do {
        CU(host_pool(&hc.pool));
        CU(cudaStreamCreateWithFlags(&hc.st, cudaStreamNonBlocking));
        CU(cudaStreamCreateWithFlags(&hc.st2, cudaStreamNonBlocking));
        bool ev_ok = true;
        for (int i = 0; i < 4 && ev_ok; ++i) {
            const cudaError_t e = cudaEventCreateWithFlags(&hc.ev[i], cudaEventDisableTiming);
            if (e != cudaSuccess) { rc = cuda_fail(e); ev_ok = false; }
        }
        if (!ev_ok) break;
        cudaEvent_t *ev_done = hc.ev, *ev_free = hc.ev + 2;
        cudaStream_t st = hc.st, st2 = hc.st2;
        CU(hc.alloc(&d_t, 8 * (size_t)total)); CU(hc.alloc(&d_m, 8 * (size_t)total));
        CU(hc.alloc(&d_off, 8 * (size_t)(n_lc + 1))); CU(hc.alloc(&d_p, 8 * (size_t)n_p));
        CU(hc.alloc(&d_pd, 8 * (size_t)n_pdot)); CU(hc.alloc(&d_ws, ws_bytes));
        CU(hc.alloc(&d_sl[0], slice_bytes)); CU(hc.alloc(&d_sl[1], slice_bytes));
        CU(hc.alloc(&d_part, 8 * W * (size_t)n_lc * (size_t)n_chunks)); CU(hc.alloc(&d_idx, 8 * (size_t)n_lc * k));
        CU(hc.alloc(&d_bce, 4 * (size_t)n_lc * k)); CU(hc.alloc(&d_st, 32 * (size_t)n_lc));
        if (filt_host) {
            void *d_filt = nullptr;
            CU(hc.alloc(&d_filt, 4 * (size_t)total));
            CU(cudaMemcpyAsync(d_filt, filt_host, 4 * (size_t)total, cudaMemcpyHostToDevice, st));
            prm_dev.filter_ids = static_cast<const int32_t *>(d_filt);
        }
        CU(cudaMemcpyAsync(d_t, times, 8 * (size_t)total, cudaMemcpyHostToDevice, st));
        CU(cudaMemcpyAsync(d_m, mags, 8 * (size_t)total, cudaMemcpyHostToDevice, st));
        CU(cudaMemcpyAsync(d_off, lc_offsets, 8 * (size_t)(n_lc + 1), cudaMemcpyHostToDevice, st));
        CU(cudaMemcpyAsync(d_p, periods, 8 * (size_t)n_p, cudaMemcpyHostToDevice, st));
        CU(cudaMemcpyAsync(d_pd, pdots, 8 * (size_t)n_pdot, cudaMemcpyHostToDevice, st));
        int n_done = 0;
        for (int c = 0; c < n_chunks && rc == GCE_CE_OK; ++c) {
            const int64_t a = (int64_t)c * chunk, b = a + chunk < n_p ? a + chunk : n_p;
            if (a >= b) break;
            const int buf = c & 1;
            cudaError_t e = cudaSuccess;
            if (c >= 2) e = cudaStreamWaitEvent(st, ev_free[buf], 0);  // the copy that last read this slice buffer is done
            if (e != cudaSuccess) { rc = cuda_fail(e); break; }
            rc = gce_ce_search_partial((const double *)d_t, (const double *)d_m, (const int64_t *)d_off, n_lc, total,
                                       (const double *)d_p, n_p, (const double *)d_pd, n_pdot, prm, a, b, d_sl[buf],
                                       (int64_t *)d_part + (size_t)c * (size_t)n_lc * W, d_ws, ws_bytes, st);
            if (rc) break;
            ++n_done;
            const size_t width = (size_t)(b - a) * (size_t)n_pdot * esz;  // one light curve's rows of this slice
            if ((e = cudaEventRecord(ev_done[buf], st)) != cudaSuccess || (e = cudaStreamWaitEvent(st2, ev_done[buf], 0)) != cudaSuccess ||
                (e = cudaMemcpy2DAsync(static_cast<unsigned char *>(out_ce) + (size_t)a * (size_t)n_pdot * esz,
                                       (size_t)n_p * (size_t)n_pdot * esz, d_sl[buf], width, width, (size_t)n_lc,
                                       cudaMemcpyDeviceToHost, st2)) != cudaSuccess ||
                (e = cudaEventRecord(ev_free[buf], st2)) != cudaSuccess) { rc = cuda_fail(e); break; }
        }
        if (rc) break;
        if (k || prm->want_stats) {
            rc = gce_ce_merge_partials((const int64_t *)d_part, n_done, n_lc, prm, out_best_idx ? (int64_t *)d_idx : nullptr,
                                       out_best_ce ? (float *)d_bce : nullptr, out_stats ? (double *)d_st : nullptr, st);
            if (rc) break;
        }
        if (out_best_idx && k) CU(cudaMemcpyAsync(out_best_idx, d_idx, 8 * (size_t)n_lc * k, cudaMemcpyDeviceToHost, st));
        if (out_best_ce && k) CU(cudaMemcpyAsync(out_best_ce, d_bce, 4 * (size_t)n_lc * k, cudaMemcpyDeviceToHost, st));
        if (out_stats) CU(cudaMemcpyAsync(out_stats, d_st, 32 * (size_t)n_lc, cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st2));
        CU(cudaStreamSynchronize(st));
    } while (0);
    return rc;
}

int gce_ce_search_host(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                       const double *periods, int64_t n_p, const double *pdots, int64_t n_pdot,
                       const gce_ce_params *prm_in, void *out_ce, int64_t *out_best_idx, float *out_best_ce,
                       double *out_stats) {
    int rc = check_params(prm_in);
    if (rc) return rc;
    if (!lc_offsets || n_lc < 0) return GCE_CE_ERR_POINTER;
    gce_ce_params prm_local = *prm_in;
    host_set_max_lc_points(lc_offsets, n_lc, &prm_local);  // the host entry sees the lengths: longer light curves -> 32-bit counters
    const gce_ce_params *prm = &prm_local;
    const int64_t total = lc_offsets[n_lc];
    rc = check_sizes(n_lc, total, n_p, n_pdot);
    if (rc) return rc;
    rc = check_lengths_host(lc_offsets, n_lc, prm);  // the host entry sees the offsets: a checked error, not NaN
    if (rc) return rc;
    if (total > 0 && (!times || !mags)) return GCE_CE_ERR_POINTER;
    if ((n_p > 0 && !periods) || !pdots) return GCE_CE_ERR_POINTER;
    if (!out_ce && !out_best_idx && !out_stats) return GCE_CE_ERR_POINTER;
    if ((prm->want_stats != 0) != (out_stats != nullptr)) return GCE_CE_ERR_POINTER;
    if ((prm->top_k > 0) != (out_best_idx != nullptr)) return GCE_CE_ERR_POINTER;
    if (out_best_ce && !out_best_idx) return GCE_CE_ERR_POINTER;
    if (prm->normalise && prm->filter_ids)  // a HOST array here: ids outside 0 .. GCE_CE_MAX_FILTERS - 1 are refused, not masked
        for (int64_t i = 0; i < total; ++i)
            if (prm->filter_ids[i] < 0 || prm->filter_ids[i] >= GCE_CE_MAX_FILTERS) return GCE_CE_ERR_RANGE;
    // a cube of at least 64 MB over at least 64 periods: overlap its transfer with the search, 8 chunks
    if (out_ce && n_lc > 0 && total > 0 && n_p >= 64 &&
        (size_t)n_lc * (size_t)n_p * (size_t)n_pdot * (prm->ce_fp64 ? 8 : 4) >= ((size_t)64 << 20))
        return search_host_pipelined(times, mags, lc_offsets, n_lc, total, periods, n_p, pdots, n_pdot, prm, out_ce,
                                     out_best_idx, out_best_ce, out_stats, 8);
    size_t ws_bytes = 0;
    rc = gce_ce_workspace_bytes(total, n_lc, n_p, n_pdot, prm, &ws_bytes);
    if (rc) return rc;
    const size_t n_trials = (size_t)n_p * (size_t)n_pdot;
    const size_t ce_bytes = out_ce ? (size_t)n_lc * n_trials * (prm->ce_fp64 ? 8 : 4) : 0;
    const size_t k = (size_t)prm->top_k;

    HostCall hc;
    void *d_t = nullptr, *d_m = nullptr, *d_off = nullptr, *d_p = nullptr, *d_pd = nullptr, *d_ws = nullptr;
    void *d_ce = nullptr, *d_idx = nullptr, *d_bce = nullptr, *d_st = nullptr;
    do {
        CU(host_pool(&hc.pool));
        CU(cudaStreamCreateWithFlags(&hc.st, cudaStreamNonBlocking));
        cudaStream_t st = hc.st;
        CU(hc.alloc(&d_t, 8 * (size_t)total)); CU(hc.alloc(&d_m, 8 * (size_t)total));
        CU(hc.alloc(&d_off, 8 * (size_t)(n_lc + 1))); CU(hc.alloc(&d_p, 8 * (size_t)n_p));
        CU(hc.alloc(&d_pd, 8 * (size_t)n_pdot)); CU(hc.alloc(&d_ws, ws_bytes));
        CU(hc.alloc(&d_ce, ce_bytes)); CU(hc.alloc(&d_idx, 8 * (size_t)n_lc * k));
        CU(hc.alloc(&d_bce, 4 * (size_t)n_lc * k)); CU(hc.alloc(&d_st, 32 * (size_t)n_lc));
        if (prm_in->normalise && prm_in->filter_ids && total) {  // the caller's HOST filter ids -> device copy
            void *d_filt = nullptr;
            CU(hc.alloc(&d_filt, 4 * (size_t)total));
            CU(cudaMemcpyAsync(d_filt, prm_in->filter_ids, 4 * (size_t)total, cudaMemcpyHostToDevice, st));
            prm_local.filter_ids = static_cast<const int32_t *>(d_filt);
        }
        if (total) {
            CU(cudaMemcpyAsync(d_t, times, 8 * (size_t)total, cudaMemcpyHostToDevice, st));
            CU(cudaMemcpyAsync(d_m, mags, 8 * (size_t)total, cudaMemcpyHostToDevice, st));
        }
        CU(cudaMemcpyAsync(d_off, lc_offsets, 8 * (size_t)(n_lc + 1), cudaMemcpyHostToDevice, st));
        if (n_p) CU(cudaMemcpyAsync(d_p, periods, 8 * (size_t)n_p, cudaMemcpyHostToDevice, st));
        CU(cudaMemcpyAsync(d_pd, pdots, 8 * (size_t)n_pdot, cudaMemcpyHostToDevice, st));
        rc = gce_ce_search((const double *)d_t, (const double *)d_m, (const int64_t *)d_off, n_lc, total,
                           (const double *)d_p, n_p, (const double *)d_pd, n_pdot, prm, out_ce ? d_ce : nullptr,
                           out_best_idx ? (int64_t *)d_idx : nullptr, out_best_ce ? (float *)d_bce : nullptr,
                           out_stats ? (double *)d_st : nullptr, d_ws, ws_bytes, st);
        if (rc) break;
        if (out_ce && ce_bytes) CU(cudaMemcpyAsync(out_ce, d_ce, ce_bytes, cudaMemcpyDeviceToHost, st));
        if (out_best_idx && k && n_lc) CU(cudaMemcpyAsync(out_best_idx, d_idx, 8 * (size_t)n_lc * k, cudaMemcpyDeviceToHost, st));
        if (out_best_ce && k && n_lc) CU(cudaMemcpyAsync(out_best_ce, d_bce, 4 * (size_t)n_lc * k, cudaMemcpyDeviceToHost, st));
        if (out_stats && n_lc) CU(cudaMemcpyAsync(out_stats, d_st, 32 * (size_t)n_lc, cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
    } while (0);
    return rc;
}
#undef CU

}  // extern "C"
