/*
 * gce_ce.h -- C ABI of the B200-native Conditional Entropy (P, Pdot) period search.
 *
 * What the library computes (Katz et al., arXiv 2006.06866; citations are lines of PAPER.md):
 *   for every light curve and every trial (P, Pdot) of a caller-supplied grid
 *     S1  normalise: t0 = min t, magnitudes min/max-scaled to [0,1], magnitude bin per point   (:96)
 *     S2  fold each time to a phase that includes the Pdot term, Eq. 3                          (:100-102)
 *     S3  bin the points into an n_phase x n_mag histogram                                      (:106)
 *     S4  CE = sum_ij p(m_i,phi_j) ln( p(phi_j) / p(m_i,phi_j) ), Eq. 4                         (:108-110)
 *     S5  store CE and/or select the k smallest per light curve (minimum = best period)         (:49, :112)
 *   optionally the significance statistics of Eq. 5 (:112-116).
 * The arithmetic (operation order of the fp64 fold, bin edge ownership, tie rule) is frozen in
 * DESIGN.md section 3; histogram counts and bin indices are bit-exact against that definition.
 *
 * Conventions
 *   - Plain C types only.  Pointers are DEVICE pointers unless the parameter name ends in _host or the
 *     function name ends in _host.  All arrays are caller-owned; the library never frees or retains them.
 *   - gce_ce_search and the debug calls only enqueue work on `stream` (a cudaStream_t passed as void*,
 *     NULL = default stream) and return without synchronising; results are valid once the stream has
 *     reached that point.  gce_ce_search_host synchronises before returning.
 *   - Return value: 0 (GCE_CE_OK) = enqueued.  Negative = error: argument, size, plan and workspace checks all
 *     run before the first launch, so for every code except GCE_CE_ERR_CUDA nothing was enqueued; after
 *     GCE_CE_ERR_CUDA (a launch or event record failed) the outputs are undefined.
 *   - No global mutable state on the device-pointer calls; re-entrant across streams as long as each call has its
 *     own workspace.  The *_host entry points allocate from a library-private, thread-safe memory pool per device
 *     that keeps up to 1 GiB cached between calls; gce_ce_host_release() returns it to the driver.
 *   - `times` need not be sorted.  `periods` are in the unit of `times`; `pdots` are dimensionless (s/s), any
 *     sign (:228).  Trials are addressed by the flat index q = ip * n_pdot + ipd.
 *   - Values that need device data to validate (non-monotone lc_offsets, P <= 0, non-finite inputs) are
 *     undefined behaviour on the device-pointer calls; gce_ce_validate_host checks host copies.  Light curves of
 *     any length up to GCE_CE_MAX_POINTS_WIDE are searched; beyond GCE_CE_MAX_POINTS (GCE_CE_MAX_POINTS_OVERLAP with
 *     overlap = 1) the device-pointer caller must say so in gce_ce_params.max_lc_points (the lengths live on the
 *     device; the *_host calls see the offsets and set it themselves).  A light curve longer than the call's limit
 *     is never folded with wrapped counters: the device-pointer calls return GCE_CE_ERR_RANGE when total_points
 *     alone proves it and otherwise treat that light curve as empty (CE = NaN, best index -1); the *_host calls
 *     return GCE_CE_ERR_RANGE beyond GCE_CE_MAX_POINTS_WIDE.
 *   - A light curve with N = 0 yields CE = NaN for every trial and best index -1; N = 1 yields CE = 0.
 *   - There is no CPU fallback anywhere in this library.
 */
#ifndef GCE_CE_H_
#define GCE_CE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GCE_CE_OK 0
#define GCE_CE_ERR_POINTER (-1)   /* NULL / inconsistent pointer combination                       */
#define GCE_CE_ERR_RANGE (-2)     /* a size or bin count is out of range                           */
#define GCE_CE_ERR_WORKSPACE (-3) /* workspace too small or misaligned                             */
#define GCE_CE_ERR_CUDA (-4)      /* a CUDA runtime call failed; see gce_ce_last_cuda_error()       */
#define GCE_CE_ERR_STATIC_LIMIT (-5) /* gce_ce_search_static only: the call needs more scratch than
                                      * GCE_CE_STATIC_SCRATCH_BYTES; use gce_ce_search with a workspace */

#define GCE_CE_MAX_BINS 64         /* n_phase_bins and n_mag_bins are each in 1..64                 */
#define GCE_CE_MAX_TOPK 32         /* top_k is in 0..32                                             */
#define GCE_CE_MAX_FILTERS 8       /* filter ids are in 0..7 (normalise = 1)                        */
#define GCE_CE_MAX_POINTS 65535    /* points per light curve with the default 16-bit counters       */
#define GCE_CE_MAX_POINTS_OVERLAP 32767 /* ... with overlap = 1 (the table holds 2N entries)            */
#define GCE_CE_MAX_POINTS_WIDE (1 << 26) /* ... of a call that announces longer light curves (max_lc_points) */

typedef struct gce_ce_params {
    int32_t n_phase_bins; /* n_phi, 1..64                                                         */
    int32_t n_mag_bins;   /* n_m,   1..64                                                         */
    int32_t top_k;        /* 0 = no selection output; 1..32 = keep the k smallest CE per LC        */
    int32_t ce_fp64;      /* 0: out_ce is float[...]; 1: out_ce is double[...]                     */
    int32_t want_stats;   /* 1: out_stats receives the Eq. 5 statistics (requires out_stats)      */
    int32_t overlap;      /* 0: plain bins (hot path).  1: 50 % overlapping phase bins (:106, :162):
                           * n_phase_bins bins of width 2/n_phase_bins, bin k = plain cells k-1 and k (cyclic),
                           * every point counted twice, p = c / 2N.  gce_ce_debug_bins ignores it.          */
    int32_t max_lc_points; /* 0: every light curve has at most GCE_CE_MAX_POINTS (_OVERLAP) points.  Larger (up to
                           * GCE_CE_MAX_POINTS_WIDE): an upper bound on the longest light curve of this call -- the
                           * search then runs with 32-bit counters and a k ln k table of that length (the paper's
                           * "base" variant for light curves of any length, :154).  gce_ce_search_host sets it itself. */
    int32_t normalise;    /* 0: magnitudes are min/max-scaled per light curve (north_star, reading Q2).
                           * 1: the paper's normalisation first (:96): per light curve and per filter, subtract the
                           * median and divide by the standard deviation of that filter's magnitudes, so that the
                           * filters can be merged into one light curve; the merged values are then min/max-binned as
                           * before.  With one filter the bins equal those of normalise = 0 in exact arithmetic.     */
    /* Optional cudaEvent_t handles (NULL = none), recorded on `stream` immediately before / after the
     * fold+bin+entropy kernel, so a harness can time the dominant kernel alone without a profiler.    */
    void *ev_search_begin;
    void *ev_search_end;
    /* normalise = 1 only: int32[total_points], the filter (0 .. GCE_CE_MAX_FILTERS - 1) of every point; NULL = all points
     * belong to one filter.  A DEVICE pointer for the device-pointer calls, a HOST pointer for the *_host calls.  An id
     * outside 0 .. GCE_CE_MAX_FILTERS - 1 is refused (GCE_CE_ERR_RANGE) by gce_ce_search_host and gce_ce_validate_host,
     * which see the array; on the device-pointer calls it is undefined behaviour like the other device-side values
     * (the kernel uses the low three bits).  Cost of normalise = 1: sequential sums are part of the frozen arithmetic,
     * so one thread per filter walks each light curve -- negligible at 1e3 points, seconds near GCE_CE_MAX_POINTS_WIDE. */
    const int32_t *filter_ids;
} gce_ce_params;

/* Bytes of device workspace gce_ce_search needs for these sizes (256-byte aligned base required).
 * total_points = lc_offsets[n_lc] (the caller knows it on the host). */
int gce_ce_workspace_bytes(int64_t total_points, int32_t n_lc, int64_t n_p, int64_t n_pdot,
                           const gce_ce_params *prm_host, size_t *bytes_host);

/*
 * The search (S1..S5).  Layouts:
 *   times, mags      double[total_points], light curves back to back (CSR)
 *   lc_offsets       int64[n_lc + 1], lc_offsets[0] = 0, non-decreasing
 *   periods          double[n_p], pdots double[n_pdot]
 *   out_ce           NULL, or [n_lc][n_p][n_pdot] (Pdot fastest) float or double per prm->ce_fp64
 *   out_best_idx     NULL (iff top_k == 0), or int64[n_lc][top_k]: flat q of the k smallest CE, ascending by
 *                    (CE, q); -1 where fewer than k trials exist or N = 0
 *   out_best_ce      NULL, or float[n_lc][top_k] matching out_best_idx (NaN where idx = -1)
 *   out_stats        NULL (iff want_stats == 0), or double[n_lc][4] = {mean CE, population std, min CE,
 *                    rho = (mean-min)/std} over all trials of the light curve (Eq. 5); exact
 *                    integer partial sums inside, so the values do not depend on the CTA split; std = 0 exactly
 *                    and rho = NaN when every trial has the same CE; all NaN for N = 0
 * At least one of out_ce / out_best_idx / out_stats must be non-NULL.
 */
int gce_ce_search(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                  int64_t total_points, const double *periods, int64_t n_p, const double *pdots,
                  int64_t n_pdot, const gce_ce_params *prm_host, void *out_ce, int64_t *out_best_idx,
                  float *out_best_ce, double *out_stats, void *workspace, size_t workspace_bytes,
                  void *stream);

/*
 * The same search for callers that cannot allocate device memory at all.
 *
 * Who this is for: code that runs as a guest inside somebody else's GPU process -- a survey alert broker, an
 * acquisition daemon, a plug-in of a pipeline that reserved the whole card for its own pool at start-up.  Such a host
 * hands the guest input and output buffers and a stream, but no allocator; cudaMalloc is off limits there because it
 * stalls every stream of the device while it runs, and because it can fail long after start-up once the host has claimed
 * the memory.  gce_ce_search still needs a workspace from somebody; this entry point needs none.
 *
 * How: the scratch memory (grouped points, magnitude-bin segments, the k ln k table, the per-CTA top-k and Eq. 5
 * partials) lives in an array of GCE_CE_STATIC_SCRATCH_BYTES that is compiled into the library's device image.  Every
 * GPU on which the library gets loaded carries that array from load until the process exits, whether or not this entry
 * point is ever called.  The call itself runs no cudaMalloc, no cudaFree and no other routine that allocates: it looks
 * up the array's device address (first call on each device, see below), checks the sizes and enqueues the same kernels,
 * in the same launch configuration, as gce_ce_search -- the results are the same bits.
 *
 * Arguments, layouts, return codes and stream semantics are those of gce_ce_search, minus workspace / workspace_bytes.
 * One more return code: GCE_CE_ERR_STATIC_LIMIT when gce_ce_workspace_bytes(total_points, n_lc, n_p, n_pdot, prm) for this
 * call exceeds GCE_CE_STATIC_SCRATCH_BYTES (nothing is enqueued; the caller can make the same comparison up front).  For
 * scale: 16 bytes per point, 8 bytes per k ln k entry (at most 65 536 entries without max_lc_points), and 16 * top_k + 64
 * bytes per CTA of the search launch.  All five BASELINE.json configs fit (C3: 64 000 points, 1.5 MiB; C4: 200 000 points
 * in 1000 light curves, 3.8 MiB; C5: 2.3 MiB), as does the paper's production grid; a batch of about 450 000 points is
 * where the limit is reached.
 *
 * Set-up: the first call on each device, made with that device current, asks the runtime for the array's address
 * (cudaGetSymbolAddress; this may load the library's device code on that device) and remembers it.  Make that first
 * call before the stream is put into capture mode.  Later calls on the device only read the remembered address.
 *
 * Sharing: there is ONE array per device and process.  Every call on that device uses it, whatever the stream or host
 * thread, and it keeps the previous call's contents.  Nothing in it has to start at zero -- each call writes every word
 * before it reads it -- so no clearing is done or needed.  But two calls whose kernels can be on the GPU at the same time
 * (different streams without an ordering between them, or two host threads on one device) overwrite each other's
 * scratch and both return garbage: order them yourself (same stream, or events).  Calls on different devices, and
 * gce_ce_search calls with their own workspaces, do not interfere.
 */
#define GCE_CE_STATIC_SCRATCH_BYTES (8u << 20)
int gce_ce_search_static(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                         int64_t total_points, const double *periods, int64_t n_p, const double *pdots,
                         int64_t n_pdot, const gce_ce_params *prm_host, void *out_ce, int64_t *out_best_idx,
                         float *out_best_ce, double *out_stats, void *stream);

/* Same call with HOST buffers for every array: allocates device memory, copies inputs in, runs the
 * search, copies the requested outputs back and synchronises.  Convenience / end-to-end timing entry. */
int gce_ce_search_host(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                       const double *periods, int64_t n_p, const double *pdots, int64_t n_pdot,
                       const gce_ce_params *prm_host, void *out_ce, int64_t *out_best_idx,
                       float *out_best_ce, double *out_stats);

/*
 * Period sub-ranges and exact merging (NEXT item N4; "batching over light curves / Pdots" with the
 * per-batch minima merged afterwards; SURVEY.md section 8e period-axis split across GPUs).
 *
 * gce_ce_search_partial searches the periods [ip_begin, ip_end) of the grid for every light curve and writes, instead
 * of the final selection, one PARTIAL blob per light curve:
 *   out_partial   int64[n_lc][gce_ce_partial_words(top_k)] =
 *                 { S[top_k] ascending, q[top_k], 8 words of Eq. 5 sums, N, pivot }
 *                 with S = N * CE * 2^shift as an exact integer (shift = the call's table shift, 42 .. 52 by the length of
 *                 the k ln k table and less beyond 65 536 entries; it travels in the blob's N word, so blobs of one
 *                 problem merge whatever their period ranges; INT64_MAX where fewer than top_k trials exist) and q the
 *                 flat index in the WHOLE grid (ip * n_pdot + ipd); the Eq. 5 words are filled when want_stats = 1.
 *   out_ce        NULL, or the cube slice [n_lc][ip_end - ip_begin][n_pdot]
 *   periods       the whole grid double[n_p]; workspace as for gce_ce_workspace_bytes(total_points, n_lc,
 *                 ip_end - ip_begin, n_pdot, prm)
 * gce_ce_merge_partials merges n_parts such blob arrays, int64[n_parts][n_lc][words] (disjoint period ranges of the same
 * light curves and the same prm; device memory, e.g. gathered from other batches or GPUs), into out_best_idx /
 * out_best_ce / out_stats exactly as gce_ce_search would have written them for the union of the ranges: all keys and
 * sums are integers, so the result is bit-identical however the grid was split.
 */
size_t gce_ce_partial_words(int32_t top_k);

int gce_ce_search_partial(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                          int64_t total_points, const double *periods, int64_t n_p, const double *pdots,
                          int64_t n_pdot, const gce_ce_params *prm_host, int64_t ip_begin, int64_t ip_end,
                          void *out_ce, int64_t *out_partial, void *workspace, size_t workspace_bytes, void *stream);

int gce_ce_merge_partials(const int64_t *partials, int32_t n_parts, int32_t n_lc, const gce_ce_params *prm_host,
                          int64_t *out_best_idx, float *out_best_ce, double *out_stats, void *stream);

/* Same merge, but the result is again one partial blob array int64[n_lc][words] (hierarchical merging: the chunks of
 * one GPU first, then one blob array per GPU over the interconnect). */
int gce_ce_merge_partials_to_partial(const int64_t *partials, int32_t n_parts, int32_t n_lc,
                                     const gce_ce_params *prm_host, int64_t *out_partial, void *stream);

/* Returns the cached device memory of the *_host entry points to the driver (see Conventions). */
int gce_ce_host_release(void);

/* Test-only: the search kernel gce_ce_search would launch for this grid -- same plan, same instantiation compiled in
 * dump mode, same tiles, warps and fold modes -- restricted to the tiles that hold a listed trial.  trial_q is a device
 * list int64[n_trials] of distinct flat trial indices q = ip * n_pdot + ipd of the (n_p x n_pdot) grid, the same for
 * every light curve.  Writes the count table Eq. 4 is evaluated on,
 *   out_counts uint32[n_lc][n_trials][n_phase_bins][n_mag_bins]      (phase-major, n_ij; with prm->overlap = 1 the
 *                                                                     overlapped table c[k][i] = n[k][i] + n[k-1][i])
 * and, if out_ce_at != NULL, double[n_lc][n_trials] CE of those trials.  Workspace as for gce_ce_workspace_bytes(
 * total_points, n_lc, n_p, n_pdot, prm).  top_k and want_stats are ignored. */
int gce_ce_debug_histogram(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                           int64_t total_points, const double *periods, int64_t n_p, const double *pdots,
                           int64_t n_pdot, const gce_ce_params *prm_host, const int64_t *trial_q,
                           int64_t n_trials, uint32_t *out_counts, double *out_ce_at, void *workspace,
                           size_t workspace_bytes, void *stream);

/* Test-only: phase bin and magnitude bin of every point of light curve `lc` for trial q, in the caller's
 * point order: out_phase_bin int32[N], out_mag_bin int32[N].  The bins come from the search kernel's own fold
 * functions, called with the thread context the search builds for trial q (its R - 1 slot neighbours, slots sorted by
 * c where floors can be shared).  fold_mode selects which of the kernel's fold variants runs: GCE_CE_FOLD_AUTO = the one
 * the owning thread qualifies for, or one of them forced; out_fold_mode (device int32[1], may be NULL) receives the
 * variant used, or -1 -- and every bin is -1 -- when the forced variant's precondition does not hold for this trial.
 * prm->normalise is ignored (the magnitude bins are those of min/max scaling of `mags` as given). */
#define GCE_CE_FOLD_AUTO 0
#define GCE_CE_FOLD_PLAIN 1     /* j = floor(y) - n_phi floor(x), one floor(x) per trial; needs |y| < 2^51        */
#define GCE_CE_FOLD_PAIR 2      /* the two trials of a counter word share floor(x); needs them within one cycle  */
#define GCE_CE_FOLD_QUAD 3      /* all trials of the thread share floor(x); needs them within one cycle          */
#define GCE_CE_FOLD_GENERIC 4   /* 64-bit integer floor and modulus, any |y| < 2^62                              */
#define GCE_CE_FOLD_PDOT_ZERO 5 /* every c of the thread is +-0: x = a                                           */
int gce_ce_debug_bins(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                      const double *periods, int64_t n_p, const double *pdots, int64_t n_pdot,
                      const gce_ce_params *prm_host, int32_t lc, int64_t q, int32_t fold_mode,
                      int32_t *out_phase_bin, int32_t *out_mag_bin, int32_t *out_fold_mode, void *stream);

/* Synchronous argument checker on HOST copies of the arrays (the hot call never synchronises).
 * Returns GCE_CE_OK or the first error found. */
int gce_ce_validate_host(const double *times_host, const double *mags_host, const int64_t *lc_offsets_host,
                         int32_t n_lc, const double *periods_host, int64_t n_p, const double *pdots_host,
                         int64_t n_pdot, const gce_ce_params *prm_host);

/* Number of kernels one gce_ce_search (partial = 0) or gce_ce_search_partial (partial = 1) call over n_p periods
 * enqueues for these arguments (for launch accounting). */
int gce_ce_launch_count(int32_t n_lc, int64_t n_p, const gce_ce_params *prm_host, int partial);

/* Diagnostic, not part of the search ABI and excluded from its stability promise (bench.py uses it to confirm the
 * roofline denominators; it allocates with cudaMalloc and synchronises).  Measures on the current device the per-SM issue rate a roofline denominator assumes, with a
 * probe kernel of 1024 threads per SM timed by the SM's own clock counter (so the figure is per clock, whatever the
 * clock).  GCE_CE_PROBE_FP64: FP64 lane-operations per SM per clock from independent DADD / DMUL chains (nominal 64 on
 * B200).  GCE_CE_PROBE_SHARED: shared-memory wavefronts per SM per clock from conflict-free RED.shared (nominal 1). */
#define GCE_CE_PROBE_FP64 0
#define GCE_CE_PROBE_SHARED 1
int gce_ce_probe_rate(int32_t kind, double *rate_host);

const char *gce_ce_strerror(int code);
int gce_ce_last_cuda_error(void); /* cudaError_t of the most recent GCE_CE_ERR_CUDA on this thread */
const char *gce_ce_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GCE_CE_H_ */
