// gce_ce.cu -- B200 (sm_100a) kernels and C ABI of the Conditional Entropy (P, Pdot) search.
//
// Path (citations are PAPER.md lines of arXiv 2006.06866):
//   k_preprocess  S1  t0 / min-max / magnitude bin per point, points grouped by magnitude bin      (:96)
//   k_ltab            fixed-point table L(k) = k ln k used by S4
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
// IMAD.HI is quarter rate and slows the FP64 pipe, measured in DESIGN.md section 7).  No tensor cores: this is a
// histogram/entropy path, not a contraction.
//
// This translation unit must be compiled with -fmad=false; the fold additionally uses explicit _rn/_rd
// intrinsics, which are never contracted.
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>
#include <string.h>

#include "gce_ce.h"

#ifndef GCE_HIST_ATOMIC
#define GCE_HIST_ATOMIC 1 /* 1: ATOMS.ADD without return; 0: LDS + IADD + STS (thread-private, race-free) */
#endif

namespace {

constexpr int kLtabSmem = 1024;   // entries of the L table mirrored in shared memory
constexpr int kLfixShift = 42;    // L table fixed point: 2^-42
constexpr double kMagic = 6755399441055744.0;  // 1.5 * 2^52: RD-add puts floor(y) in the low mantissa word
constexpr double kYSafe = 2251799813685248.0;  // 2^51: |y| below this -> the magic-add floor is exact
constexpr int64_t kInfS = INT64_MAX;
constexpr int kSmemLimit = 227 * 1024 - 8 * kLtabSmem;  // dynamic shared memory per CTA: 227 KB minus the static L table
constexpr int kStatWords = 8;     // partial Eq. 5 sums: n, sum d (i128), sum d^2 (u192), min S, pad; d = S - K
constexpr int kMaxWarps = 20;     // warps per CTA of the largest variant (640 threads)
constexpr int kCloseGroup = 5;    // phase bins whose read-and-clear atomics are in flight together in S4

struct FalseT { static constexpr bool value = false; };
struct TrueT { static constexpr bool value = true; };

struct LcInfo {
    int32_t n;
    int32_t pad;
    double dt_max;
    int64_t K;  // N * H(m) in 2^-42 fixed point = L(N) - sum_i L(points in magnitude bin i): CE <= H(m), pivot of the Eq. 5 sums
};

struct SearchParams {
    const double2 *pts;        // [total_points] (dt, dt2), grouped by magnitude bin inside each light curve
    const int32_t *seg;        // [n_lc][n_m + 1] segment offsets relative to the light curve start
    const LcInfo *info;        // [n_lc]
    const int64_t *lc_offsets; // [n_lc + 1]
    const int64_t *ltab;       // [ltab_n] fixed-point k ln k
    const double *periods;
    const double *pdots;
    const int64_t *trial_q;    // DUMP only
    int64_t n_p, n_pdot, n_trials;
    int64_t q_off;             // flat index of this call's first trial in the caller's grid (period sub-range)
    int64_t tiles_per_lc;
    int32_t jobs_per_lc;
    int32_t n_phi, n_m;
    int32_t cap_points;        // capacity of the shared-memory point buffer (multiple of 8)
    int32_t ltab_n;
    int32_t top_k;
    int32_t ce_fp64;
    int32_t overlap;           // N2: 50 %-overlapping phase bins
    void *out_ce;              // cube or NULL
    int64_t *part_S, *part_q;  // [n_lc][jobs_per_lc][top_k]
    uint64_t *part_stats;      // [n_lc][jobs_per_lc][kStatWords] partial Eq. 5 sums, or NULL
    uint32_t *out_counts;      // DUMP only
    double *out_ce_at;         // DUMP only
};

// ------------------------------------------------------------------------------------------------ helpers
__device__ __forceinline__ uint32_t smem_u32(const void *p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// TMA bulk copy global -> shared, completion counted in bytes on an mbarrier (SASS: UBLKCP).
__device__ __forceinline__ void tma_load_bulk(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// (S, q) lexicographic order: exact integer N*CE first, then flat trial index (tie rule Q9).
__device__ __forceinline__ bool key_less(int64_t s1, int64_t q1, int64_t s2, int64_t q2) {
    return (s1 < s2) || (s1 == s2 && q1 < q2);
}

// Warp-distributed sorted list: lane l holds the l-th best (S, q); lanes >= k hold +inf.
struct WarpTopK {
    int64_t S, q;       // this lane's element
    int64_t thrS, thrq; // the k-th (worst kept) element, replicated
    int k;
    __device__ __forceinline__ void reset(int k_) {
        k = k_;
        S = kInfS; q = kInfS; thrS = kInfS; thrq = kInfS;
    }
    // Every lane offers one candidate (cS = kInfS for "none"); warp-uniform call.
    __device__ __forceinline__ void offer(int64_t cS, int64_t cq) {
        const int lane = threadIdx.x & 31;
        unsigned mask = __ballot_sync(0xffffffffu, key_less(cS, cq, thrS, thrq));
        while (mask) {
            const int src = __ffs(mask) - 1;
            mask &= mask - 1;
            const int64_t xS = __shfl_sync(0xffffffffu, cS, src);
            const int64_t xq = __shfl_sync(0xffffffffu, cq, src);
            if (!key_less(xS, xq, thrS, thrq)) continue;  // threshold moved since the ballot
            const int pos = __popc(__ballot_sync(0xffffffffu, key_less(S, q, xS, xq)));
            const int64_t upS = __shfl_up_sync(0xffffffffu, S, 1);
            const int64_t upq = __shfl_up_sync(0xffffffffu, q, 1);
            if (lane == pos) { S = xS; q = xq; }
            else if (lane > pos) { S = upS; q = upq; }
            if (lane >= k) { S = kInfS; q = kInfS; }
            thrS = __shfl_sync(0xffffffffu, S, k - 1);
            thrq = __shfl_sync(0xffffffffu, q, k - 1);
        }
    }
};

// ---- Eq. 5 statistics (NEXT item N1): exact integer partial sums of d = S - K over trials, S = N*CE*2^42.
// Word layout (kStatWords u64): [0] n, [1..2] sum d (two's-complement i128), [3..5] sum d^2 (u192), [6] min S, [7] max S.
typedef unsigned __int128 u128_t;
__device__ __forceinline__ u128_t shfl_xor_u128(u128_t v, int o) {
    uint64_t lo = (uint64_t)v, hi = (uint64_t)(v >> 64);
    lo = __shfl_xor_sync(0xffffffffu, lo, o);
    hi = __shfl_xor_sync(0xffffffffu, hi, o);
    return ((u128_t)hi << 64) | lo;
}
__device__ __forceinline__ void stat_init(uint64_t *st) {
    st[0] = st[1] = st[2] = st[3] = st[4] = st[5] = 0;
    st[6] = (uint64_t)kInfS;
    st[7] = (uint64_t)INT64_MIN;
}
// st += (n, a, b, mn, mx); a is an i128 passed as its two's-complement bits, b < 2^128
__device__ __forceinline__ void stat_add(uint64_t *st, uint64_t n, u128_t a, u128_t b, uint64_t b_hi, int64_t mn, int64_t mx) {
    st[0] += n;
    const u128_t A = (((u128_t)st[2] << 64) | st[1]) + a;
    st[1] = (uint64_t)A; st[2] = (uint64_t)(A >> 64);
    const u128_t B = (((u128_t)st[4] << 64) | st[3]) + b;
    st[3] = (uint64_t)B; st[4] = (uint64_t)(B >> 64);
    st[5] += b_hi + (B < b ? 1u : 0u);
    if (mn < (int64_t)st[6]) st[6] = (uint64_t)mn;
    if (mx > (int64_t)st[7]) st[7] = (uint64_t)mx;
}
__device__ __forceinline__ void stat_merge(uint64_t *st, const uint64_t *o) {
    stat_add(st, o[0], ((u128_t)o[2] << 64) | o[1], ((u128_t)o[4] << 64) | o[3], o[5], (int64_t)o[6], (int64_t)o[7]);
}

// S1 magnitude bin: min(floor(((m - m_lo) / r) * n_m), n_m - 1); r == 0 -> 0.
__device__ __forceinline__ int mag_bin(double m, double m_lo, double r, int n_m) {
    if (r == 0.0) return 0;
    const double u = __ddiv_rn(__dsub_rn(m, m_lo), r);
    const int i = __double2int_rd(__dmul_rn(u, (double)n_m));
    return i < n_m - 1 ? i : n_m - 1;
}

// S2, slow generic form (any |y| < 2^62): exactly the listing of DESIGN.md section 3.
__device__ __forceinline__ int fold_bin_generic(double dt, double dt2, double invP, double c, int n_phi) {
    const double a = __dmul_rn(dt, invP);
    const double b = __dmul_rn(dt2, c);
    const double x = __dadd_rn(a, b);
    const double y = __dmul_rn(x, (double)n_phi);
    const long long I = __double2ll_rd(y);
    long long j = I % (long long)n_phi;
    if (j < 0) j += n_phi;
    return (int)j;
}

__device__ __forceinline__ void trial_constants(double P, double Pdot, double &invP, double &c) {
    invP = __ddiv_rn(1.0, P);
    c = __dmul_rn(__dmul_rn(__dmul_rn(-0.5, Pdot), invP), invP);
}

struct MinMax3 {
    double tmin, tmax, mmin, mmax;
};

__device__ __forceinline__ MinMax3 block_minmax(MinMax3 v, MinMax3 *sh) {
    for (int o = 16; o > 0; o >>= 1) {
        const double a = __shfl_xor_sync(0xffffffffu, v.tmin, o);
        const double b = __shfl_xor_sync(0xffffffffu, v.tmax, o);
        const double c = __shfl_xor_sync(0xffffffffu, v.mmin, o);
        const double d = __shfl_xor_sync(0xffffffffu, v.mmax, o);
        v.tmin = a < v.tmin ? a : v.tmin;
        v.tmax = b > v.tmax ? b : v.tmax;
        v.mmin = c < v.mmin ? c : v.mmin;
        v.mmax = d > v.mmax ? d : v.mmax;
    }
    const int w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    if ((threadIdx.x & 31) == 0) sh[w] = v;
    __syncthreads();
    MinMax3 r = sh[0];
    for (int i = 1; i < nw; ++i) {
        r.tmin = sh[i].tmin < r.tmin ? sh[i].tmin : r.tmin;
        r.tmax = sh[i].tmax > r.tmax ? sh[i].tmax : r.tmax;
        r.mmin = sh[i].mmin < r.mmin ? sh[i].mmin : r.mmin;
        r.mmax = sh[i].mmax > r.mmax ? sh[i].mmax : r.mmax;
    }
    __syncthreads();
    return r;
}

// ------------------------------------------------------------------------------------------------ S1
// One CTA per light curve.  Output points are permuted so equal magnitude bins are contiguous (counts do not
// depend on point order); seg[lc][i] is the first point of magnitude bin i, seg[lc][n_m] = N.
__global__ void __launch_bounds__(256) k_preprocess(const double *__restrict__ times, const double *__restrict__ mags,
                                                    const int64_t *__restrict__ lc_offsets, int n_m,
                                                    double2 *__restrict__ pts, int32_t *__restrict__ seg,
                                                    LcInfo *__restrict__ info, const int64_t *__restrict__ ltab, const int mult) {
    __shared__ MinMax3 sh_red[8];
    __shared__ int sh_cnt[GCE_CE_MAX_BINS + 1];
    __shared__ int sh_cur[GCE_CE_MAX_BINS];
    const int lc = blockIdx.x;
    const int64_t off = lc_offsets[lc];
    const int n = (int)(lc_offsets[lc + 1] - off);
    const double *t = times + off, *m = mags + off;

    MinMax3 v{CUDART_INF, -CUDART_INF, CUDART_INF, -CUDART_INF};
    for (int k = threadIdx.x; k < n; k += blockDim.x) {
        const double tk = t[k], mk = m[k];
        v.tmin = tk < v.tmin ? tk : v.tmin;
        v.tmax = tk > v.tmax ? tk : v.tmax;
        v.mmin = mk < v.mmin ? mk : v.mmin;
        v.mmax = mk > v.mmax ? mk : v.mmax;
    }
    v = block_minmax(v, sh_red);
    const double t0 = v.tmin, m_lo = v.mmin, r = __dsub_rn(v.mmax, v.mmin);

    for (int i = threadIdx.x; i <= n_m; i += blockDim.x) sh_cnt[i] = 0;
    __syncthreads();
    for (int k = threadIdx.x; k < n; k += blockDim.x) atomicAdd(&sh_cnt[mag_bin(m[k], m_lo, r, n_m)], 1);
    __syncthreads();
    if (threadIdx.x == 0) {
        int acc = 0;
        int64_t K = ltab[mult * n];  // mult = 2 with overlapping phase bins: the table holds 2N entries
        for (int i = 0; i < n_m; ++i) {
            const int c = sh_cnt[i];
            seg[(int64_t)lc * (n_m + 1) + i] = acc;
            sh_cur[i] = acc;
            acc += c;
            K -= ltab[mult * c];
        }
        info[lc].K = K;
        seg[(int64_t)lc * (n_m + 1) + n_m] = acc;
        info[lc].n = n;
        info[lc].pad = 0;
        info[lc].dt_max = n > 0 ? __dsub_rn(v.tmax, t0) : 0.0;
    }
    __syncthreads();
    for (int k = threadIdx.x; k < n; k += blockDim.x) {
        const int i = mag_bin(m[k], m_lo, r, n_m);
        const int pos = atomicAdd(&sh_cur[i], 1);
        const double dt = __dsub_rn(t[k], t0);
        pts[off + pos] = make_double2(dt, __dmul_rn(dt, dt));
    }
}

// L(k) = k ln k in 2^-42 fixed point (k < 2^16 -> L < 2^20, so sums of up to N entries fit in int64).
__global__ void k_ltab(int64_t *__restrict__ ltab, int n) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) ltab[k] = k < 2 ? 0 : __double2ll_rn(ldexp((double)k * log((double)k), kLfixShift));
}

// ------------------------------------------------------------------------------------------------ S2..S5
__device__ __forceinline__ void red_add_u32(uint32_t addr, uint32_t inc) {
    asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(addr), "r"(inc) : "memory");
}

// read-and-clear of one counter word in one LSU instruction (ATOMS.EXCH)
__device__ __forceinline__ uint32_t exch0_u32(uint32_t addr) {
    uint32_t w;
    asm volatile("atom.shared.exch.b32 %0, [%1], %2;" : "=r"(w) : "r"(addr), "r"(0u) : "memory");
    return w;
}

// L(k) = k ln k in 2^-42 fixed point for the two 16-bit counter fields of a word.  The fields count in units of
// 2^us: us = 3 whenever every count of the light curve fits 13 bits (N, or 2N with overlapping bins, <= 8191), so that a
// field IS the byte offset of its table entry.  BIG = false: the caller guarantees us == 3 and counts < kLtabSmem (a
// bound on the number of points that can be in the cell): mask / shift, one LDS.64 each.  BIG = true: any us, first
// kLtabSmem entries from shared memory, the rest from global.
template <bool BIG>
__device__ __forceinline__ void ltab_pair(const int64_t *__restrict__ sL, const int64_t *__restrict__ gL, const uint32_t w,
                                          const uint32_t us, int64_t &v0, int64_t &v1) {
    if (!BIG) {
        const unsigned char *b = reinterpret_cast<const unsigned char *>(sL);
        v0 = *reinterpret_cast<const int64_t *>(b + (w & 0xfff8u));
        v1 = *reinterpret_cast<const int64_t *>(b + (w >> 16));
    } else {
        const uint32_t c0 = (w & 0xffffu) >> us, c1 = w >> (16u + us);
        v0 = sL[c0 & (kLtabSmem - 1)];
        v1 = sL[c1 & (kLtabSmem - 1)];
        if (c0 >= (uint32_t)kLtabSmem) v0 = gL[c0];
        if (c1 >= (uint32_t)kLtabSmem) v1 = gL[c1];
    }
}

// S2 + S3 for one point and the R trials of this thread (DESIGN.md section 3; PAPER.md:100 Eq. 3, :106).
//   a = dt*invP ; b = dt2*c ; x = a + b ; y = x*n_phi          (RN each, never fused)
//   j = floor(y) - n_phi*floor(x)                               two exact round-down magic adds, |y| < 2^51
// j equals floor(y) mod n_phi except when RN(x*n_phi) lands exactly on the next multiple of n_phi, where it is
// n_phi: that count goes to an extra histogram row that is folded into row 0 when the segment is closed.
// PZ: every trial of the thread has c = +-0, so x = a bit for bit (a >= +0) and two operations are skipped.
template <int R, bool SHARE_P, bool PZ>
__device__ __forceinline__ void fold_bin_add(const double2 p, const double (&invP)[R], const double (&cc)[R],
                                             const double nphi_d, const uint32_t negn, const uint32_t rs,
                                             const uint32_t (&hb)[(R + 1) / 2], const uint32_t inc0, const uint32_t inc1) {
    double a;
    if (SHARE_P) a = __dmul_rn(p.x, invP[0]);
#pragma unroll
    for (int r = 0; r < R; ++r) {
        if (!SHARE_P) a = __dmul_rn(p.x, invP[r]);
        const double x = PZ ? a : __dadd_rn(a, __dmul_rn(p.y, cc[r]));
        const double y = __dmul_rn(x, nphi_d);
        const uint32_t Iy = (uint32_t)__double2loint(__dadd_rd(y, kMagic));
        const uint32_t Ix = (uint32_t)__double2loint(__dadd_rd(x, kMagic));
        const uint32_t j = Iy + Ix * negn;
        red_add_u32(j * rs + hb[r >> 1], (r & 1) ? inc1 : inc0);
    }
}

// Hot loop over the points [kk, ke) of one shared-memory buffer (all of one magnitude bin).  The next two points are
// loaded before the current two are folded (the RED asm statements are compiler barriers, so the loads would otherwise
// sit behind the previous iteration's atomics and the first DMUL would wait for them); the last trip reads up to two
// entries past ke, which are inside the buffer's slack and never used.
template <int R, bool SHARE_P, bool PZ>
__device__ __forceinline__ void fold_range(const double2 *__restrict__ sp, int kk, const int ke, const double (&invP)[R],
                                           const double (&cc)[R], const double nphi_d, const uint32_t negn,
                                           const uint32_t rs, const uint32_t (&hb)[(R + 1) / 2], const uint32_t inc0,
                                           const uint32_t inc1) {
    if (ke - kk >= 4) {
        double2 a0 = sp[kk], a1 = sp[kk + 1];
        do {
            const double2 b0 = sp[kk + 2], b1 = sp[kk + 3];
            fold_bin_add<R, SHARE_P, PZ>(a0, invP, cc, nphi_d, negn, rs, hb, inc0, inc1);
            fold_bin_add<R, SHARE_P, PZ>(a1, invP, cc, nphi_d, negn, rs, hb, inc0, inc1);
            a0 = sp[kk + 4];
            a1 = sp[kk + 5];
            fold_bin_add<R, SHARE_P, PZ>(b0, invP, cc, nphi_d, negn, rs, hb, inc0, inc1);
            fold_bin_add<R, SHARE_P, PZ>(b1, invP, cc, nphi_d, negn, rs, hb, inc0, inc1);
            kk += 4;
        } while (ke - kk >= 4);
    }
    for (; kk < ke; ++kk) fold_bin_add<R, SHARE_P, PZ>(sp[kk], invP, cc, nphi_d, negn, rs, hb, inc0, inc1);
}

// Rare path (|y| >= 2^51 for some point): the listing of DESIGN.md section 3 with 64-bit integers.
template <int R, bool SHARE_P>
__device__ __forceinline__ void fold_range_generic(const double2 *__restrict__ sp, int kk, const int ke,
                                                   const double (&invP)[R], const double (&cc)[R], const int n_phi,
                                                   const uint32_t rs, const uint32_t (&hb)[(R + 1) / 2],
                                                   const uint32_t inc0, const uint32_t inc1) {
    for (; kk < ke; ++kk) {
        const double2 p = sp[kk];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int j = fold_bin_generic(p.x, p.y, invP[SHARE_P ? 0 : r], cc[r], n_phi);
            red_add_u32((uint32_t)j * rs + hb[r >> 1], (r & 1) ? inc1 : inc0);
        }
    }
}

// S4, first half: close magnitude bin `seg_i`.  fetch_word reads and clears this thread's counter word of phase bin j
// (two 16-bit counts, trials 2*w2 and 2*w2+1); close_word adds it to the phase marginal and accumulates sum L(n_ij).
__device__ __forceinline__ uint32_t fetch_word(const int j, const int n_phi, const uint32_t rs, const uint32_t hbw) {
    uint32_t w = exch0_u32(hbw + (uint32_t)j * rs);
    if (j == 0) w += exch0_u32(hbw + (uint32_t)n_phi * rs);  // phase bin 0 takes over the overflow row
    return w;
}

template <int R, bool DUMP, bool BIG>
__device__ __forceinline__ void close_word(const uint32_t w, const int j, const int w2, const int n_phi, const uint32_t us,
                                           int64_t (&S2)[R], const int64_t *__restrict__ sL, const SearchParams &prm,
                                           const int lc, const int64_t s0, const bool (&valid)[R], const int seg_i) {
    int64_t v0, v1;
    ltab_pair<BIG>(sL, prm.ltab, w, us, v0, v1);
    S2[2 * w2] += v0;
    if (2 * w2 + 1 < R) S2[(2 * w2 + 1) < R ? 2 * w2 + 1 : 0] += v1;
    if (DUMP) {
        const uint32_t c0 = (w & 0xffffu) >> us, c1 = w >> (16u + us);
        if (valid[2 * w2])
            prm.out_counts[(((int64_t)lc * prm.n_trials + s0 + 2 * w2) * n_phi + j) * prm.n_m + seg_i] = c0;
        if (2 * w2 + 1 < R && valid[(2 * w2 + 1) < R ? 2 * w2 + 1 : 0])
            prm.out_counts[(((int64_t)lc * prm.n_trials + s0 + 2 * w2 + 1) * n_phi + j) * prm.n_m + seg_i] = c1;
    }
}

// All phase bins of magnitude bin seg_i.  The phase marginal is a register array (REGM, compile-time n_phi) or a second
// set of counter rows in shared memory updated with one RED per word (no registers, so more threads fit per SM).
// With a compile-time n_phi the read-and-clear atomics of kCloseGroup phase bins are issued back to back before
// their results are used, so their latency overlaps.
// OVL (NEXT item N2): 50 %-overlapping phase bins -- bin k holds the plain cells k-1 and k (cyclic), so
// the looked-up count is w[k] + w[k-1] (packed 16-bit pairs; needs 2N <= 65535); the folds and the plain marginal are
// unchanged, the overlap costs one add per word.
template <int NPHI, bool REGM, int R, bool DUMP, bool BIG, bool OVL>
__device__ __forceinline__ void close_mag_bin(const int n_phi, const uint32_t rs, const uint32_t marg_off, const uint32_t us,
                                              const uint32_t (&hb)[(R + 1) / 2],
                                              uint32_t (&mg)[REGM ? NPHI : 1][(R + 1) / 2], int64_t (&S2)[R],
                                              const int64_t *__restrict__ sL, const SearchParams &prm, const int lc,
                                              const int64_t s0, const bool (&valid)[R], const int seg_i) {
    constexpr int RW = (R + 1) / 2;
    uint32_t prev[RW], first[RW];
    if (NPHI > 0) {
        constexpr int NP = NPHI > 0 ? NPHI : 1;
        constexpr int G = NP % kCloseGroup == 0 ? kCloseGroup : 1;
#pragma unroll
        for (int j0 = 0; j0 < NP; j0 += G) {
            uint32_t w[G][RW];
#pragma unroll
            for (int jj = 0; jj < G; ++jj)
#pragma unroll
                for (int w2 = 0; w2 < RW; ++w2) w[jj][w2] = fetch_word(j0 + jj, n_phi, rs, hb[w2]);
#pragma unroll
            for (int jj = 0; jj < G; ++jj)
#pragma unroll
                for (int w2 = 0; w2 < RW; ++w2) {
                    const uint32_t ww = w[jj][w2];
                    if (REGM) mg[REGM ? j0 + jj : 0][w2] += ww;
                    else red_add_u32(hb[w2] + marg_off + (uint32_t)(j0 + jj - w2) * rs, ww);
                    if (!OVL) close_word<R, DUMP, BIG>(ww, j0 + jj, w2, n_phi, us, S2, sL, prm, lc, s0, valid, seg_i);
                    else {
                        if (j0 + jj == 0) first[w2] = ww;
                        else close_word<R, DUMP, BIG>(ww + prev[w2], j0 + jj, w2, n_phi, us, S2, sL, prm, lc, s0, valid, seg_i);
                        prev[w2] = ww;
                    }
                }
        }
    } else {
        for (int j = 0; j < n_phi; ++j) {
#pragma unroll
            for (int w2 = 0; w2 < RW; ++w2) {
                const uint32_t ww = fetch_word(j, n_phi, rs, hb[w2]);
                red_add_u32(hb[w2] + marg_off + (uint32_t)(j - w2) * rs, ww);
                if (!OVL) close_word<R, DUMP, BIG>(ww, j, w2, n_phi, us, S2, sL, prm, lc, s0, valid, seg_i);
                else {
                    if (j == 0) first[w2] = ww;
                    else close_word<R, DUMP, BIG>(ww + prev[w2], j, w2, n_phi, us, S2, sL, prm, lc, s0, valid, seg_i);
                    prev[w2] = ww;
                }
            }
        }
    }
    if (OVL) {  // bin 0 = cells n_phi-1 and 0
#pragma unroll
        for (int w2 = 0; w2 < RW; ++w2)
            close_word<R, DUMP, BIG>(first[w2] + prev[w2], 0, w2, n_phi, us, S2, sL, prm, lc, s0, valid, seg_i);
    }
}

// NPHI > 0: compile-time n_phi (unrolled S4); NPHI == 0: any n_phi <= 64.  REGM: phase marginal in registers, exactly
// 512 threads per CTA; otherwise the marginal is a second set of counter rows in shared memory, threads per CTA =
// prm.nt (any multiple of 32 up to 640), which leaves registers for a fifth warp per sub-partition when the shared
// memory allows it.  R = trials per thread.  SHARE_P: the R trials of a thread share one period (n_pdot % R == 0).
// DUMP: test mode, trials come from a list and the count tables are written out.
template <int NPHI, bool REGM, int R, bool SHARE_P, bool DUMP>
__global__ void __launch_bounds__(REGM ? 512 : 640, 1) k_search(const SearchParams prm) {
    static_assert(!REGM || NPHI > 0, "register marginals need a compile-time n_phi");
    constexpr int RW = (R + 1) / 2;  // 32-bit words per (bin, thread): two 16-bit counters each
    constexpr int NPHI_REG = REGM ? NPHI : 1;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int NT = REGM ? 512 : (int)blockDim.x, NW = NT >> 5;
    const int tid = threadIdx.x, lane = tid & 31;
    const int n_phi = NPHI > 0 ? NPHI : prm.n_phi, n_m = prm.n_m;
    const uint32_t rs = (uint32_t)NT * 4u;  // bytes between the counter rows of consecutive phase bins

    // shared-memory carve-up (dynamic part; the L table is static so that lookups are LDS.64 [offset + const]), points last
    __shared__ __align__(16) int64_t sL[kLtabSmem];  // static: its shared address is a link-time constant
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw);                     // [2]
    int *sseg = reinterpret_cast<int *>(full + 2);                               // [n_m + 1] (<= 65)
    uint64_t *sstat = reinterpret_cast<uint64_t *>(sseg + GCE_CE_MAX_BINS + 4);  // [kMaxWarps][kStatWords]
    uint32_t *hist = reinterpret_cast<uint32_t *>(sstat + kMaxWarps * kStatWords); // [RW][n_phi + 1][NT], 16-byte aligned
    const uint32_t plane = (uint32_t)(n_phi + 1) * rs;                           // bytes per counter-word plane
    // shared-memory marginal (!REGM): RW planes of n_phi rows after the histogram; word (w2, j) of this thread is at
    // hb[w2] + marg_off + (j - w2) * rs
    const uint32_t marg_off = (uint32_t)RW * plane;
    const uint32_t hist_words = (uint32_t)(REGM ? RW * (n_phi + 1) : RW * (2 * n_phi + 1)) * (uint32_t)NT;
    double2 *spts = reinterpret_cast<double2 *>(hist + hist_words);              // [cap_points + 2]

    const int lc = blockIdx.x / prm.jobs_per_lc;
    const int job = blockIdx.x % prm.jobs_per_lc;
    const int64_t tile_lo = prm.tiles_per_lc * job / prm.jobs_per_lc;
    const int64_t tile_hi = prm.tiles_per_lc * (job + 1) / prm.jobs_per_lc;
    const int n_tiles = (int)(tile_hi - tile_lo);
    const int N = prm.info[lc].n;
    const double dt_max = prm.info[lc].dt_max;
    const int64_t K = prm.info[lc].K;
    const double2 *gpts = prm.pts + prm.lc_offsets[lc];
    const bool single = N <= prm.cap_points;            // the whole light curve stays resident for every tile
    const int CH = single ? N : prm.cap_points / 2;     // else: streamed through two half buffers, per tile
    const int n_chunks = N > 0 ? (N + CH - 1) / CH : 0;
    const int total_seq = single ? n_chunks : n_tiles * n_chunks;
    const int64_t TILE = (int64_t)NT * R;

    auto issue_chunk = [&](int g) {  // thread 0 only: TMA bulk copy of sequence element g into its buffer
        const int c = g % n_chunks, buf = single ? 0 : (g & 1);
        const int cnt = min(CH, N - c * CH);
        mbar_expect_tx(&full[buf], (uint32_t)cnt * 16u);
        for (int o = 0; o < cnt; o += 2048)
            tma_load_bulk(spts + (size_t)buf * CH + o, gpts + (size_t)c * CH + o, (uint32_t)min(2048, cnt - o) * 16u, &full[buf]);
    };

    // ---- prologue: zero histograms, stage table / segments, start the point loads
    for (uint32_t i = tid; i < hist_words; i += NT) hist[i] = 0u;
    for (int i = tid; i < kLtabSmem; i += NT) sL[i] = i < prm.ltab_n ? prm.ltab[i] : 0;
    for (int i = tid; i <= n_m; i += NT) sseg[i] = prm.seg[(int64_t)lc * (n_m + 1) + i];
    if (tid < NW) stat_init(sstat + tid * kStatWords);
    if (tid == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        if (n_tiles > 0)
            for (int g = 0; g < 2 && g < total_seq; ++g) issue_chunk(g);
    }
    __syncthreads();

    WarpTopK top;
    top.reset(prm.top_k > 0 ? prm.top_k : 1);

    const double nphi_d = (double)n_phi;
    const uint32_t negn = 0u - (uint32_t)n_phi;
    uint32_t hb[RW];
#pragma unroll
    for (int w2 = 0; w2 < RW; ++w2) hb[w2] = smem_u32(hist) + (uint32_t)tid * 4u + (uint32_t)w2 * plane;
    const bool ovl = !DUMP && prm.overlap != 0;  // N2: 2N table entries per trial
    const double ce_scale = N > 0 ? ldexp(1.0, -kLfixShift) / (double)(ovl ? 2 * N : N) : 0.0;
    const uint32_t us = ((ovl ? 2 : 1) * N <= 8191) ? 3u : 0u;  // counter unit 2^us: a field is its table entry's byte offset
    const uint32_t inc0 = 1u << us, inc1 = 0x10000u << us;
    uint32_t mg[NPHI_REG][RW];  // phase marginal n_j of the R trials (NPHI > 0), packed like the histogram
#pragma unroll
    for (int j = 0; j < NPHI_REG; ++j)
#pragma unroll
        for (int w2 = 0; w2 < RW; ++w2) mg[j][w2] = 0u;

    // Warps that share an SM sub-partition (warp id mod 4) start at different magnitude bins, a quarter of the points
    // apart, so that one warp's S4 (no FP64) overlaps the others' folds (FP64-bound).  Counts and the integer entropy
    // sums do not depend on the order of the bins.  Streamed light curves are processed in storage order.
    int rot = 0;
    if (single && n_m > 1) {
        const int groups = (NW + 3) >> 2;
        const int target = (int)((int64_t)N * (tid >> 7) / groups);
        while (rot + 1 < n_m && sseg[rot + 1] <= target) ++rot;
    }
    int g = 0;  // position in this CTA's chunk sequence (streamed mode)
    for (int tl = 0; tl < n_tiles; ++tl) {
        const int64_t s0 = (tile_lo + tl) * TILE + (int64_t)tid * R;  // first trial slot of this thread
        // ---- per-trial constants
        double invP[R], cc[R];  // SHARE_P: only invP[0] is used
        int64_t qv[R];
        bool valid[R];
        bool fast = true, pz = true;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int64_t s = s0 + r;
            valid[r] = s < prm.n_trials;
            int64_t q = 0;
            if (valid[r]) q = DUMP ? prm.trial_q[s] : s;
            qv[r] = q + prm.q_off;  // reported index: flat q of the caller's whole grid
            double ip = 0.0, c = 0.0;
            if (valid[r] && (!SHARE_P || r == 0)) ip = __ddiv_rn(1.0, prm.periods[q / prm.n_pdot]);
            if (SHARE_P && r > 0) ip = invP[0];
            if (valid[r]) c = __dmul_rn(__dmul_rn(__dmul_rn(-0.5, prm.pdots[q % prm.n_pdot]), ip), ip);
            invP[r] = ip;
            cc[r] = c;
            // conservative bound on |y|: below 2^51 the magic-add floors are exact
            fast = fast && (nphi_d * (dt_max * fabs(ip) + dt_max * dt_max * fabs(c)) * 1.000001 < kYSafe);
            pz = pz && (c == 0.0);
        }
        fast = __all_sync(0xffffffffu, fast);
        pz = __all_sync(0xffffffffu, pz);

        int64_t S2[R];
#pragma unroll
        for (int r = 0; r < R; ++r) S2[r] = 0;

        int seg_s = 0;  // magnitude bins finished so far, counted in this warp's (rotated) order
        for (int c = 0; c < n_chunks; ++c) {
            const int buf = single ? 0 : (g & 1);
            if (!single || tl == 0) mbar_wait(&full[buf], single ? 0u : (uint32_t)((g >> 1) & 1));
            const double2 *sp = spts + (size_t)buf * CH;
            const int k_base = c * CH;
            const int k_end = min(N, k_base + CH);
            while (seg_s < n_m) {
                int seg_i = seg_s + rot;
                if (seg_i >= n_m) seg_i -= n_m;
                const int b0 = sseg[seg_i], b1 = sseg[seg_i + 1];
                const int lo = max(b0, k_base) - k_base, hi = min(b1, k_end) - k_base;
                // ---------------- hot loop: fold + bin the points of magnitude bin seg_i that are in this buffer
                if (lo < hi) {
                    if (fast) {
                        if (pz) fold_range<R, SHARE_P, true>(sp, lo, hi, invP, cc, nphi_d, negn, rs, hb, inc0, inc1);
                        else fold_range<R, SHARE_P, false>(sp, lo, hi, invP, cc, nphi_d, negn, rs, hb, inc0, inc1);
                    } else {
                        fold_range_generic<R, SHARE_P>(sp, lo, hi, invP, cc, n_phi, rs, hb, inc0, inc1);
                    }
                }
                if (b1 > k_end) break;  // the bin continues in the next buffer
                // ---------------- S4: the bin is complete; a cell holds at most b1 - b0 points
                if (b1 > b0) {
                    // a cell of this bin holds at most b1 - b0 points (twice that with overlapping bins)
                    if (!ovl) {
                        if (us == 3u && b1 - b0 < kLtabSmem)
                            close_mag_bin<NPHI, REGM, R, DUMP, false, false>(n_phi, rs, marg_off, us, hb, mg, S2, sL, prm, lc, s0, valid, seg_i);
                        else
                            close_mag_bin<NPHI, REGM, R, DUMP, true, false>(n_phi, rs, marg_off, us, hb, mg, S2, sL, prm, lc, s0, valid, seg_i);
                    } else if (!DUMP) {
                        if (us == 3u && 2 * (b1 - b0) < kLtabSmem)
                            close_mag_bin<NPHI, REGM, R, false, false, true>(n_phi, rs, marg_off, us, hb, mg, S2, sL, prm, lc, s0, valid, seg_i);
                        else
                            close_mag_bin<NPHI, REGM, R, false, true, true>(n_phi, rs, marg_off, us, hb, mg, S2, sL, prm, lc, s0, valid, seg_i);
                    }
                }
                ++seg_s;
            }
            if (!single) {  // streamed mode: everyone is done with this half buffer -> refill it with element g + 2
                __syncthreads();
                if (tid == 0 && g + 2 < total_seq) issue_chunk(g + 2);
                ++g;
            }
        }

        // ---------------- finish the trials: S1 = sum_j L(n_j), CE, outputs
        int64_t S1[R];
#pragma unroll
        for (int r = 0; r < R; ++r) S1[r] = 0;
        if (N > 0) {
            auto add_marg = [&](const uint32_t w, const int w2, auto big) {
                int64_t v0, v1;
                ltab_pair<decltype(big)::value>(sL, prm.ltab, w, us, v0, v1);
                S1[2 * w2] += v0;
                if (2 * w2 + 1 < R) S1[(2 * w2 + 1) < R ? 2 * w2 + 1 : 0] += v1;
            };
            auto marg_pass = [&](auto big, auto ovlt) {
                constexpr bool OVL = decltype(ovlt)::value;
                uint32_t prev[RW], first[RW];
                if (REGM) {
#pragma unroll
                    for (int j = 0; j < NPHI_REG; ++j)
#pragma unroll
                        for (int w2 = 0; w2 < RW; ++w2) {
                            const uint32_t ww = mg[j][w2];
                            mg[j][w2] = 0u;
                            if (!OVL) add_marg(ww, w2, big);
                            else { if (j == 0) first[w2] = ww; else add_marg(ww + prev[w2], w2, big); prev[w2] = ww; }
                        }
                } else {
                    for (int j = 0; j < n_phi; ++j)
#pragma unroll
                        for (int w2 = 0; w2 < RW; ++w2) {
                            const uint32_t ww = exch0_u32(hb[w2] + marg_off + (uint32_t)(j - w2) * rs);
                            if (!OVL) add_marg(ww, w2, big);
                            else { if (j == 0) first[w2] = ww; else add_marg(ww + prev[w2], w2, big); prev[w2] = ww; }
                        }
                }
                if (OVL) {
#pragma unroll
                    for (int w2 = 0; w2 < RW; ++w2) add_marg(first[w2] + prev[w2], w2, big);
                }
            };
            if (!ovl) { if (us == 3u && N < kLtabSmem) marg_pass(FalseT{}, FalseT{}); else marg_pass(TrueT{}, FalseT{}); }
            else { if (us == 3u && 2 * N < kLtabSmem) marg_pass(FalseT{}, TrueT{}); else marg_pass(TrueT{}, TrueT{}); }
        }
        double ce[R];
        int64_t S[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            S[r] = S1[r] - S2[r];  // = N * CE * 2^42, exact
            ce[r] = N > 0 ? (double)S[r] * ce_scale : CUDART_NAN;
        }
        if (DUMP) {
#pragma unroll
            for (int r = 0; r < R; ++r)
                if (valid[r] && prm.out_ce_at) prm.out_ce_at[(int64_t)lc * prm.n_trials + s0 + r] = ce[r];
        } else {
            if (prm.out_ce) {
                const int64_t o = (int64_t)lc * prm.n_trials + s0;  // q == slot outside DUMP
                float *o32 = reinterpret_cast<float *>(prm.out_ce) + o;
                if (R == 4 && !prm.ce_fp64 && valid[R - 1] && (reinterpret_cast<uintptr_t>(o32) & 15u) == 0) {
                    *reinterpret_cast<float4 *>(o32) = make_float4((float)ce[0], (float)ce[1 % R], (float)ce[2 % R], (float)ce[3 % R]);
                } else {
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        if (!valid[r]) continue;
                        if (prm.ce_fp64) reinterpret_cast<double *>(prm.out_ce)[o + r] = ce[r];
                        else o32[r] = (float)ce[r];
                    }
                }
            }
            if (prm.top_k > 0) {
#pragma unroll
                for (int r = 0; r < R; ++r) top.offer((valid[r] && N > 0) ? S[r] : kInfS, (valid[r] && N > 0) ? qv[r] : kInfS);
            }
            if (prm.part_stats != nullptr && N > 0) {  // Eq. 5 partial sums of this tile, warp-reduced, exact integers
                __int128 a = 0;
                u128_t b = 0;
                int64_t mn = kInfS, mx = INT64_MIN;
                uint32_t cnt = 0;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    if (!valid[r]) continue;
                    const int64_t d = S[r] - K;   // |d| < 2^60
                    a += d;
                    b += (u128_t)((__int128)d * d);
                    mn = S[r] < mn ? S[r] : mn;
                    mx = S[r] > mx ? S[r] : mx;
                    ++cnt;
                }
                u128_t au = (u128_t)a;
                for (int o = 16; o > 0; o >>= 1) {
                    au += shfl_xor_u128(au, o);
                    b += shfl_xor_u128(b, o);            // <= 32 * R * 2^120 < 2^128
                    const int64_t m2 = __shfl_xor_sync(0xffffffffu, mn, o), m3 = __shfl_xor_sync(0xffffffffu, mx, o);
                    mn = m2 < mn ? m2 : mn;
                    mx = m3 > mx ? m3 : mx;
                    cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
                }
                if (lane == 0) stat_add(sstat + (tid >> 5) * kStatWords, cnt, au, b, 0, mn, mx);
            }
        }
    }

    // ---------------- per-CTA Eq. 5 partial sums -> part_stats[lc][job]
    if (!DUMP && prm.part_stats != nullptr) {
        __syncthreads();
        if (tid == 0) {
            uint64_t tot[kStatWords];
            stat_init(tot);
            for (int w = 0; w < NW; ++w) stat_merge(tot, sstat + w * kStatWords);
            uint64_t *o = prm.part_stats + ((int64_t)lc * prm.jobs_per_lc + job) * kStatWords;
            for (int i = 0; i < kStatWords; ++i) o[i] = tot[i];
        }
    }

    // ---------------- per-CTA merge of the warps' top-k lists -> partial[lc][job][k]
    if (!DUMP && prm.top_k > 0) {
        const int K = prm.top_k;
        __syncthreads();  // every issued TMA load has been consumed: the point buffer is idle, reuse it as scratch
        int64_t *scr = reinterpret_cast<int64_t *>(spts);  // 16 * NW * K <= 10 KB <= cap_points * 16 (cap >= kMinPoints)
        if (lane < K) {
            scr[2 * ((tid >> 5) * K + lane)] = top.S;
            scr[2 * ((tid >> 5) * K + lane) + 1] = top.q;
        }
        __syncthreads();
        if (tid < 32) {
            top.reset(K);
            for (int e = 0; e < NW * K; e += 32) {
                const int i = e + lane;
                const int64_t cS = i < NW * K ? scr[2 * i] : kInfS;
                const int64_t cq = i < NW * K ? scr[2 * i + 1] : kInfS;
                top.offer(cS, cq);
            }
            if (lane < K) {
                const int64_t o = ((int64_t)lc * prm.jobs_per_lc + job) * K + lane;
                prm.part_S[o] = top.S;
                prm.part_q[o] = top.q;
            }
        }
    }
}

// ---- S5 / Eq. 5 merges.  One warp per light curve.  The candidates / partial sums of light curve lc live at
// base[lc * lc_stride + p * part_stride + ...], p < n_parts: inside one call the parts are the CTAs (jobs) of k_search,
// in gce_ce_merge_partials they are the caller's partial blobs (period ranges, batches, GPUs).  Keys are
// the exact integers (S = N*CE*2^42, flat q), so the merged result does not depend on the split.
// Partial blob of one light curve (int64 words): [0,K) S ascending, [K,2K) q, [2K,2K+8) Eq. 5 sums, [2K+8] N, [2K+9] pivot.
__host__ __device__ inline int partial_words(int K) { return 2 * K + kStatWords + 2; }

__global__ void __launch_bounds__(32) k_merge_topk(const int64_t *__restrict__ S, const int64_t *__restrict__ q,
                                                   int64_t lc_stride, int64_t part_stride, int n_parts, int K,
                                                   const LcInfo *__restrict__ info, const int64_t *__restrict__ npts,
                                                   int64_t npts_stride, int mult, int64_t *__restrict__ out_idx,
                                                   float *__restrict__ out_ce, int64_t *__restrict__ out_raw,
                                                   int64_t raw_stride) {
    const int lc = blockIdx.x, lane = threadIdx.x;
    WarpTopK top;
    top.reset(K);
    const int total = n_parts * K;
    for (int e = 0; e < total; e += 32) {
        const int i = e + lane;
        const int64_t at = (int64_t)lc * lc_stride + (int64_t)(i / K) * part_stride + (i % K);
        top.offer(i < total ? S[at] : kInfS, i < total ? q[at] : kInfS);
    }
    if (lane >= K) return;
    if (out_raw) {  // partial blob: exact keys, kInfS where fewer than K trials exist
        out_raw[(int64_t)lc * raw_stride + lane] = top.S;
        out_raw[(int64_t)lc * raw_stride + K + lane] = top.q;
        return;
    }
    const bool have = top.S != kInfS;
    const int64_t n = info ? (int64_t)info[lc].n : npts[(int64_t)lc * npts_stride];
    out_idx[(int64_t)lc * K + lane] = have ? top.q : -1;
    if (out_ce) out_ce[(int64_t)lc * K + lane] = have ? (float)((double)top.S * (ldexp(1.0, -kLfixShift) / (double)(mult * n))) : CUDART_NAN_F;
}

// Eq. 5: sums the partials (exact integers) and converts once to fp64:
// out_stats[lc] = {mean CE, population std, min CE, rho = (mean - min) / std}; or writes the raw sums to a partial blob.
__device__ __forceinline__ double u128_to_double(u128_t v) {
    return (double)(uint64_t)(v >> 64) * 18446744073709551616.0 + (double)(uint64_t)v;
}
__global__ void __launch_bounds__(32) k_merge_stats(const uint64_t *__restrict__ part, int64_t lc_stride, int64_t part_stride,
                                                    int n_parts, const LcInfo *__restrict__ info,
                                                    const int64_t *__restrict__ npts, int64_t npts_stride, int mult,
                                                    double *__restrict__ out_stats, int64_t *__restrict__ out_raw,
                                                    int64_t raw_stride) {
    __shared__ uint64_t sh[32][kStatWords];
    const int lc = blockIdx.x, lane = threadIdx.x;
    uint64_t acc[kStatWords];
    stat_init(acc);
    for (int j = lane; j < n_parts; j += 32) stat_merge(acc, part + (int64_t)lc * lc_stride + (int64_t)j * part_stride);
    for (int i = 0; i < kStatWords; ++i) sh[lane][i] = acc[i];
    __syncwarp();
    if (lane != 0) return;
    for (int l = 1; l < 32; ++l) stat_merge(acc, sh[l]);
    const int64_t n_pts = info ? (int64_t)info[lc].n : npts[(int64_t)lc * npts_stride];
    const int64_t pivot = info ? info[lc].K : npts[(int64_t)lc * npts_stride + 1];
    if (out_raw) {
        int64_t *o = out_raw + (int64_t)lc * raw_stride;
        for (int i = 0; i < kStatWords; ++i) o[i] = (int64_t)acc[i];
        o[kStatWords] = n_pts;
        o[kStatWords + 1] = pivot;
        return;
    }
    double *o = out_stats + (int64_t)lc * 4;
    if (acc[0] == 0 || n_pts <= 0) { o[0] = o[1] = o[2] = o[3] = CUDART_NAN; return; }
    const double n = (double)acc[0];
    const u128_t A = ((u128_t)acc[2] << 64) | acc[1];
    const bool neg = (acc[2] >> 63) != 0;
    const double sum_d = neg ? -u128_to_double((u128_t)0 - A) : u128_to_double(A);
    const double sum_d2 = (double)acc[5] * 3.4028236692093846e38 + u128_to_double(((u128_t)acc[4] << 64) | acc[3]);
    const double scale = ldexp(1.0, -kLfixShift) / (double)(mult * n_pts);
    const double mean_d = sum_d / n;
    double var = sum_d2 / n - mean_d * mean_d;
    if (var < 0.0 || acc[6] == acc[7]) var = 0.0;  // min == max: every trial has the same CE, the spread is exactly 0
    const double mean = ((double)pivot + mean_d) * scale;
    const double sd = sqrt(var) * scale;
    const double mn = (double)(int64_t)acc[6] * scale;
    o[0] = mean; o[1] = sd; o[2] = mn; o[3] = (mean - mn) / sd;
}

// Test-only: bins of one light curve for one trial, caller's point order (same device functions as the path).
__global__ void k_debug_bins(const double *__restrict__ times, const double *__restrict__ mags,
                             const int64_t *__restrict__ lc_offsets, const double *__restrict__ periods,
                             const double *__restrict__ pdots, int64_t n_pdot, int n_phi, int n_m, int lc, int64_t q,
                             uint32_t mod_mul, uint32_t mod_bias, double y_safe, int32_t *__restrict__ out_phase,
                             int32_t *__restrict__ out_mag) {
    __shared__ MinMax3 sh_red[8];
    const int64_t off = lc_offsets[lc];
    const int n = (int)(lc_offsets[lc + 1] - off);
    const double *t = times + off, *m = mags + off;
    MinMax3 v{CUDART_INF, -CUDART_INF, CUDART_INF, -CUDART_INF};
    for (int k = threadIdx.x; k < n; k += blockDim.x) {
        const double tk = t[k], mk = m[k];
        v.tmin = tk < v.tmin ? tk : v.tmin;
        v.tmax = tk > v.tmax ? tk : v.tmax;
        v.mmin = mk < v.mmin ? mk : v.mmin;
        v.mmax = mk > v.mmax ? mk : v.mmax;
    }
    v = block_minmax(v, sh_red);
    const double r = __dsub_rn(v.mmax, v.mmin);
    double invP, c;
    trial_constants(periods[q / n_pdot], pdots[q % n_pdot], invP, c);
    const double dt_max = n > 0 ? __dsub_rn(v.tmax, v.tmin) : 0.0;
    const bool fast = (double)n_phi * (dt_max * fabs(invP) + dt_max * dt_max * fabs(c)) * 1.000001 < y_safe;
    const double magic_b = kMagic + (double)mod_bias;
    for (int k = threadIdx.x; k < n; k += blockDim.x) {
        const double dt = __dsub_rn(t[k], v.tmin), dt2 = __dmul_rn(dt, dt);
        int j;
        if (fast) {
            const double y = __dmul_rn(__dadd_rn(__dmul_rn(dt, invP), __dmul_rn(dt2, c)), (double)n_phi);
            const uint32_t Iu = (uint32_t)__double2loint(__dadd_rd(y, magic_b));
            j = (int)(Iu - __umulhi(Iu, mod_mul) * (uint32_t)n_phi);
        } else {
            j = fold_bin_generic(dt, dt2, invP, c, n_phi);
        }
        out_phase[k] = j;
        out_mag[k] = mag_bin(m[k], v.mmin, r, n_m);
    }
}

// ------------------------------------------------------------------------------------------------ host side
thread_local int g_last_cuda_error = 0;

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// Which kernel variant runs, with how many threads, over how many CTAs: decided from sizes only (deterministic, no
// device query), so gce_ce_workspace_bytes and gce_ce_search agree.
struct Plan {
    int R;             // trials per thread
    bool share_p;      // the R trials of a thread share one period
    int nphi_t;        // compile-time n_phi of the kernel (15, 20, 30) or 0 = generic
    bool regm;         // phase marginal in registers (512 threads) instead of shared memory
    int nt;            // threads per CTA (multiple of 32)
    int cap_points;    // shared-memory point buffer capacity
    size_t smem;       // dynamic shared memory per CTA
    int64_t tiles_per_lc;
    int jobs_per_lc;
};

constexpr int kMaxThreadsSmemMarg = 640;  // launch bound of the shared-memory-marginal kernels (<= 102 registers)
constexpr int kMinPoints = 640;           // smallest point buffer; also the top-k merge scratch (16 B x 20 warps x 32)

size_t search_smem_fixed() {
    return sizeof(uint64_t) * 2 + sizeof(int) * (GCE_CE_MAX_BINS + 4) +
           sizeof(uint64_t) * kMaxWarps * kStatWords;
}
// counter rows of one thread: histogram (n_phi + 1 rows, the last one catches RN(x * n_phi) == n_phi * (floor(x) + 1)),
// plus n_phi marginal rows when the marginal is not in registers; RW words each
size_t search_smem_per_thread(int n_phi, int R, bool regm) {
    return (size_t)((R + 1) / 2) * (size_t)(regm ? n_phi + 1 : 2 * n_phi + 1) * sizeof(uint32_t);
}

Plan make_plan(int32_t n_lc, int64_t total_points, int64_t n_trials, int64_t n_pdot, int n_phi, bool dump) {
    Plan p;
    if (dump) { p.R = 2; p.share_p = false; }
    else if (n_pdot % 4 == 0) { p.R = 4; p.share_p = true; }
    else if (n_pdot % 2 == 0) { p.R = 2; p.share_p = true; }
    else { p.R = 4; p.share_p = false; }
    const int64_t avail = (int64_t)kSmemLimit - (int64_t)search_smem_fixed();
    const bool templ = !dump && (n_phi == 15 || n_phi == 20 || n_phi == 30 || n_phi == 50);
    // 50 phase bins (the paper's production binning): the register marginal of R = 4 trials would take
    // 100 registers, so a thread owns R = 2 trials and 512 threads still fit (measured 2x the generic variant)
    if (!dump && n_phi == 50) { p.R = 2; p.share_p = (n_pdot % 2 == 0); }
    // point buffer wanted: the average light curve plus a quarter (the per-LC lengths live on the device; a longer
    // light curve is streamed through the buffer in two halves instead of staying resident)
    const int64_t avg = n_lc > 0 ? (total_points + n_lc - 1) / n_lc : 0;
    int64_t want_pts = (avg + avg / 4 + 15) / 8 * 8;
    if (want_pts < kMinPoints) want_pts = kMinPoints;
    if (want_pts > 8192) want_pts = 8192;
    auto threads_beside = [&](int64_t pts, bool regm) {
        int64_t nt = (avail - (pts + 2) * (int64_t)sizeof(double2)) / (int64_t)search_smem_per_thread(n_phi, p.R, regm);
        return nt < 0 ? 0 : nt / 32 * 32;
    };
    int64_t nt_s = threads_beside(want_pts, false);
    if (nt_s > kMaxThreadsSmemMarg) nt_s = kMaxThreadsSmemMarg;
    const bool regm_fits = templ && threads_beside(kMinPoints, true) >= 512;
    // measured on C3: 512 threads with register marginals beat 608 threads with shared-memory
    // marginals (83.7 vs 86.8 ms), so the register variant is taken whenever it fits
    if (regm_fits) {
        p.regm = true;
        p.nt = 512;
    } else {
        p.regm = false;
        if (nt_s < 32) nt_s = threads_beside(kMinPoints, false);
        if (nt_s > kMaxThreadsSmemMarg) nt_s = kMaxThreadsSmemMarg;
        p.nt = (int)nt_s;  // >= 32: 64 x 64 bins with R = 4 leave room for 192 threads
    }
    p.nphi_t = templ ? n_phi : 0;
    const int64_t planes = (int64_t)search_smem_per_thread(n_phi, p.R, p.regm) * p.nt;
    int64_t cap = (avail - planes) / (int64_t)sizeof(double2) - 2;  // - 2: read-ahead slack of the hot loop
    cap = cap / 8 * 8;
    if (cap > 8192) cap = 8192;  // 128 KB of points; longer light curves are streamed
    p.cap_points = (int)cap;
    p.smem = (size_t)(cap + 2) * sizeof(double2) + search_smem_fixed() + (size_t)planes;
    const int64_t tile = (int64_t)p.nt * p.R;
    p.tiles_per_lc = n_trials > 0 ? (n_trials + tile - 1) / tile : 0;
    // ~16 CTAs per SM overall for dynamic balance, at least one tile per job
    int64_t want = (148LL * 16 + (n_lc > 0 ? n_lc : 1) - 1) / (n_lc > 0 ? n_lc : 1);
    if (want > p.tiles_per_lc) want = p.tiles_per_lc;
    if (want < 1) want = 1;
    if (want > 4096) want = 4096;
    p.jobs_per_lc = (int)want;
    return p;
}

struct Layout {
    size_t pts, seg, info, ltab, part_S, part_q, part_stats, total;
    int ltab_n;
};

Layout make_layout(int64_t total_points, int32_t n_lc, int64_t n_trials, int64_t n_pdot, const gce_ce_params *prm, bool dump) {
    Layout L;
    size_t o = 0;
    L.pts = o; o = align_up(o + sizeof(double2) * (size_t)(total_points > 0 ? total_points : 1), 256);
    L.seg = o; o = align_up(o + sizeof(int32_t) * (size_t)(n_lc > 0 ? n_lc : 1) * (prm->n_mag_bins + 1), 256);
    L.info = o; o = align_up(o + sizeof(LcInfo) * (size_t)(n_lc > 0 ? n_lc : 1), 256);
    int64_t tn = (prm->overlap ? 2 : 1) * total_points;  // largest count looked up: N, or 2N with overlapping bins
    if (tn > GCE_CE_MAX_POINTS) tn = GCE_CE_MAX_POINTS;
    L.ltab_n = (int)tn + 1;
    L.ltab = o; o = align_up(o + sizeof(int64_t) * (size_t)L.ltab_n, 256);
    const Plan p = make_plan(n_lc, total_points, n_trials, n_pdot, prm->n_phase_bins, dump);
    const size_t parts = (size_t)(n_lc > 0 ? n_lc : 1) * (size_t)p.jobs_per_lc * (size_t)(prm->top_k > 0 ? prm->top_k : 1);
    L.part_S = o; o = align_up(o + sizeof(int64_t) * parts, 256);
    L.part_q = o; o = align_up(o + sizeof(int64_t) * parts, 256);
    L.part_stats = o;
    if (prm->want_stats) o = align_up(o + sizeof(uint64_t) * kStatWords * (size_t)(n_lc > 0 ? n_lc : 1) * (size_t)p.jobs_per_lc, 256);
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
    if (prm->reserved[0] != 0 || prm->reserved[1] != 0) return GCE_CE_ERR_RANGE;
    return GCE_CE_OK;
}

int check_sizes(int32_t n_lc, int64_t total_points, int64_t n_p, int64_t n_pdot) {
    if (n_lc < 0 || total_points < 0 || n_p < 0 || n_pdot < 1) return GCE_CE_ERR_RANGE;
    if (n_lc > (1 << 24)) return GCE_CE_ERR_RANGE;
    if (n_p > 0 && n_pdot > (int64_t)0x7fffffffffffLL / n_p) return GCE_CE_ERR_RANGE;
    return GCE_CE_OK;
}

// Exact 32-bit floor-mod constants: q = umulhi(I, M) equals I / d for I < nmax.
void mod_constants(int d, uint32_t *mul, uint32_t *bias, double *y_safe) {
    if (d == 1) { *mul = 0; *bias = 0; *y_safe = -1.0; return; }  // always the generic path (j = 0)
    const uint64_t M = (1ULL << 32) / (uint64_t)d + 1;
    const uint64_t e = M * (uint64_t)d - (1ULL << 32);
    const uint64_t nmax = 0xffffffffULL / e;
    const uint64_t half = nmax / 2;
    const uint64_t B = half / (uint64_t)d * (uint64_t)d;
    *mul = (uint32_t)M;
    *bias = (uint32_t)B;
    *y_safe = (double)(B - (uint64_t)d - 2);
}

int cuda_fail(cudaError_t e) {
    g_last_cuda_error = (int)e;
    return GCE_CE_ERR_CUDA;
}

template <int NPHI, bool REGM, int R, bool SHARE_P, bool DUMP>
int launch_search(const SearchParams &sp, const Plan &plan, int32_t n_lc, cudaStream_t st) {
    auto kern = k_search<NPHI, REGM, R, SHARE_P, DUMP>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)plan.smem);
    if (e != cudaSuccess) return cuda_fail(e);
    const unsigned grid = (unsigned)((int64_t)n_lc * plan.jobs_per_lc);
    kern<<<grid, plan.nt, plan.smem, st>>>(sp);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);
    return GCE_CE_OK;
}

template <int NPHI, bool REGM>
int launch_search_variant(const SearchParams &sp, const Plan &plan, int32_t n_lc, cudaStream_t st) {
    if (plan.share_p && plan.R == 4) return launch_search<NPHI, REGM, 4, true, false>(sp, plan, n_lc, st);
    if (plan.share_p && plan.R == 2) return launch_search<NPHI, REGM, 2, true, false>(sp, plan, n_lc, st);
    return launch_search<NPHI, REGM, 4, false, false>(sp, plan, n_lc, st);
}

int dispatch_search(const SearchParams &sp, const Plan &plan, bool dump, int32_t n_lc, cudaStream_t st) {
    if (dump) return launch_search<0, false, 2, false, true>(sp, plan, n_lc, st);
    switch (plan.nphi_t) {
        case 15: return plan.regm ? launch_search_variant<15, true>(sp, plan, n_lc, st) : launch_search_variant<15, false>(sp, plan, n_lc, st);
        case 20: return plan.regm ? launch_search_variant<20, true>(sp, plan, n_lc, st) : launch_search_variant<20, false>(sp, plan, n_lc, st);
        case 30: return plan.regm ? launch_search_variant<30, true>(sp, plan, n_lc, st) : launch_search_variant<30, false>(sp, plan, n_lc, st);
        case 50:
            if (plan.regm && plan.R == 2)
                return plan.share_p ? launch_search<50, true, 2, true, false>(sp, plan, n_lc, st)
                                    : launch_search<50, true, 2, false, false>(sp, plan, n_lc, st);
            return launch_search_variant<0, false>(sp, plan, n_lc, st);
        default: return launch_search_variant<0, false>(sp, plan, n_lc, st);
    }
}

}  // namespace

// ================================================================================================ C ABI
extern "C" {

const char *gce_ce_version(void) { return "gce-b200 0.1 (sm_100a)"; }

const char *gce_ce_strerror(int code) {
    switch (code) {
        case GCE_CE_OK: return "ok";
        case GCE_CE_ERR_POINTER: return "null or inconsistent pointer arguments";
        case GCE_CE_ERR_RANGE: return "size, bin count or option out of range";
        case GCE_CE_ERR_WORKSPACE: return "workspace too small or misaligned";
        case GCE_CE_ERR_CUDA: return "CUDA runtime error (see gce_ce_last_cuda_error)";
        default: return "unknown error code";
    }
}

int gce_ce_last_cuda_error(void) { return g_last_cuda_error; }

int gce_ce_launch_count(int32_t n_lc, const gce_ce_params *prm) {
    if (!prm || n_lc <= 0) return 0;
    return 3 + (prm->top_k > 0 ? 1 : 0) + (prm->want_stats ? 1 : 0);  // ltab, preprocess, search, [merge_topk], [merge_stats]
}

int gce_ce_workspace_bytes(int64_t total_points, int32_t n_lc, int64_t n_p, int64_t n_pdot, const gce_ce_params *prm,
                           size_t *bytes) {
    if (!bytes) return GCE_CE_ERR_POINTER;
    int rc = check_params(prm);
    if (rc) return rc;
    rc = check_sizes(n_lc, total_points, n_p, n_pdot);
    if (rc) return rc;
    *bytes = make_layout(total_points, n_lc, n_p * n_pdot, n_pdot, prm, false).total;
    return GCE_CE_OK;
}

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
        if (!trial_q || n_dump < 0) return GCE_CE_ERR_POINTER;
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
    const int64_t n_trials = dump ? n_dump : n_p * n_pdot;
    gce_ce_params lay_prm = *prm;
    if (dump) { lay_prm.top_k = 0; lay_prm.want_stats = 0; lay_prm.overlap = 0; }  // the debug dump is always the plain table
    const int mult = lay_prm.overlap ? 2 : 1;
    const Layout L = make_layout(total_points, n_lc, n_trials, dump ? 1 : n_pdot, &lay_prm, dump);
    if (workspace_bytes < L.total || (reinterpret_cast<uintptr_t>(workspace) & 255u)) return GCE_CE_ERR_WORKSPACE;
    if (n_lc == 0) return GCE_CE_OK;

    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    unsigned char *ws = reinterpret_cast<unsigned char *>(workspace);
    double2 *pts = reinterpret_cast<double2 *>(ws + L.pts);
    int32_t *seg = reinterpret_cast<int32_t *>(ws + L.seg);
    LcInfo *info = reinterpret_cast<LcInfo *>(ws + L.info);
    int64_t *ltab = reinterpret_cast<int64_t *>(ws + L.ltab);

    k_ltab<<<(L.ltab_n + 255) / 256, 256, 0, st>>>(ltab, L.ltab_n);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);
    k_preprocess<<<n_lc, 256, 0, st>>>(times, mags, lc_offsets, prm->n_mag_bins, pts, seg, info, ltab, mult);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);

    const Plan plan = make_plan(n_lc, total_points, n_trials, dump ? 1 : n_pdot, prm->n_phase_bins, dump);
    SearchParams sp;
    memset(&sp, 0, sizeof(sp));
    sp.pts = pts; sp.seg = seg; sp.info = info; sp.lc_offsets = lc_offsets; sp.ltab = ltab;
    sp.periods = periods; sp.pdots = pdots; sp.trial_q = trial_q;
    sp.n_p = n_p; sp.n_pdot = n_pdot; sp.n_trials = n_trials;
    sp.q_off = dump ? 0 : ip_begin * n_pdot;
    sp.jobs_per_lc = plan.jobs_per_lc;
    sp.tiles_per_lc = plan.tiles_per_lc;
    sp.cap_points = plan.cap_points;
    sp.n_phi = prm->n_phase_bins; sp.n_m = prm->n_mag_bins;
    sp.ltab_n = L.ltab_n;
    sp.top_k = dump ? 0 : prm->top_k;
    sp.ce_fp64 = prm->ce_fp64;
    sp.overlap = lay_prm.overlap;
    sp.out_ce = out_ce;
    sp.part_S = reinterpret_cast<int64_t *>(ws + L.part_S);
    sp.part_q = reinterpret_cast<int64_t *>(ws + L.part_q);
    sp.part_stats = (!dump && prm->want_stats) ? reinterpret_cast<uint64_t *>(ws + L.part_stats) : nullptr;
    sp.out_counts = out_counts; sp.out_ce_at = out_ce_at;

    if (prm->ev_search_begin) {
        e = cudaEventRecord(reinterpret_cast<cudaEvent_t>(prm->ev_search_begin), st);
        if (e != cudaSuccess) return cuda_fail(e);
    }
    if (n_trials > 0) {
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
    int rc = check_params(prm);
    if (rc) return rc;
    if (n_lc > 0 && n_trials > 0) {
        cudaError_t e = cudaMemsetAsync(out_counts, 0,
                                        sizeof(uint32_t) * (size_t)n_lc * (size_t)n_trials * prm->n_phase_bins * prm->n_mag_bins,
                                        reinterpret_cast<cudaStream_t>(stream));
        if (e != cudaSuccess) return cuda_fail(e);
    }
    return run_search(times, mags, lc_offsets, n_lc, total_points, periods, n_p, pdots, n_pdot, prm, nullptr, nullptr,
                      nullptr, nullptr, trial_q, n_trials, out_counts, out_ce_at, 0, nullptr, workspace, workspace_bytes, stream);
}

int gce_ce_debug_bins(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                      const double *periods, int64_t n_p, const double *pdots, int64_t n_pdot, const gce_ce_params *prm,
                      int32_t lc, int64_t q, int32_t *out_phase_bin, int32_t *out_mag_bin, void *stream) {
    int rc = check_params(prm);
    if (rc) return rc;
    if (!times || !mags || !lc_offsets || !periods || !pdots || !out_phase_bin || !out_mag_bin) return GCE_CE_ERR_POINTER;
    if (n_pdot < 1 || n_p < 1 || lc < 0 || lc >= n_lc || q < 0 || q >= n_p * n_pdot) return GCE_CE_ERR_RANGE;
    uint32_t mul, bias;
    double y_safe;
    mod_constants(prm->n_phase_bins, &mul, &bias, &y_safe);
    k_debug_bins<<<1, 256, 0, reinterpret_cast<cudaStream_t>(stream)>>>(times, mags, lc_offsets, periods, pdots, n_pdot,
                                                                       prm->n_phase_bins, prm->n_mag_bins, lc, q, mul,
                                                                       bias, y_safe, out_phase_bin, out_mag_bin);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);
    return GCE_CE_OK;
}

int gce_ce_validate_host(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                         const double *periods, int64_t n_p, const double *pdots, int64_t n_pdot,
                         const gce_ce_params *prm) {
    int rc = check_params(prm);
    if (rc) return rc;
    if (!lc_offsets) return GCE_CE_ERR_POINTER;
    if (n_lc < 0 || n_p < 0 || n_pdot < 1) return GCE_CE_ERR_RANGE;
    if (lc_offsets[0] != 0) return GCE_CE_ERR_RANGE;
    for (int32_t l = 0; l < n_lc; ++l) {
        const int64_t n = lc_offsets[l + 1] - lc_offsets[l];
        if (n < 0 || n > GCE_CE_MAX_POINTS) return GCE_CE_ERR_RANGE;
    }
    const int64_t total = lc_offsets[n_lc];
    if (total > 0 && (!times || !mags)) return GCE_CE_ERR_POINTER;
    for (int64_t k = 0; k < total; ++k)
        if (!(times[k] - times[k] == 0.0) || !(mags[k] - mags[k] == 0.0)) return GCE_CE_ERR_RANGE;  // NaN / inf
    if (n_p > 0 && !periods) return GCE_CE_ERR_POINTER;
    if (!pdots) return GCE_CE_ERR_POINTER;
    for (int64_t i = 0; i < n_p; ++i)
        if (!(periods[i] > 0.0) || !(periods[i] - periods[i] == 0.0)) return GCE_CE_ERR_RANGE;
    for (int64_t i = 0; i < n_pdot; ++i)
        if (!(pdots[i] - pdots[i] == 0.0)) return GCE_CE_ERR_RANGE;
    return GCE_CE_OK;
}

// Host-buffer entry with the cube requested and a grid worth splitting: the period axis is cut into chunks searched
// back to back on one stream (gce_ce_search_partial, exact merge at the end) while a second stream copies each finished
// cube slice to the caller's buffer, so the device-to-host transfer of the cube overlaps the search of the next chunk.
static int search_host_pipelined(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                                 int64_t total, const double *periods, int64_t n_p, const double *pdots, int64_t n_pdot,
                                 const gce_ce_params *prm, void *out_ce, int64_t *out_best_idx, float *out_best_ce,
                                 double *out_stats, int n_chunks) {
    const size_t esz = prm->ce_fp64 ? 8 : 4;
    const int64_t chunk = (n_p + n_chunks - 1) / n_chunks;
    const size_t k = (size_t)prm->top_k, W = gce_ce_partial_words(prm->top_k);
    size_t ws_bytes = 0;
    int rc = gce_ce_workspace_bytes(total, n_lc, chunk, n_pdot, prm, &ws_bytes);
    if (rc) return rc;
    cudaStream_t st = nullptr, st2 = nullptr;
    cudaEvent_t ev_done[2] = {nullptr, nullptr}, ev_free[2] = {nullptr, nullptr};
    cudaError_t e = cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking);
    if (e != cudaSuccess) return cuda_fail(e);
    e = cudaStreamCreateWithFlags(&st2, cudaStreamNonBlocking);
    if (e != cudaSuccess) { cudaStreamDestroy(st); return cuda_fail(e); }
    for (int b = 0; b < 2; ++b) {
        cudaEventCreateWithFlags(&ev_done[b], cudaEventDisableTiming);
        cudaEventCreateWithFlags(&ev_free[b], cudaEventDisableTiming);
    }
    void *d_t = nullptr, *d_m = nullptr, *d_off = nullptr, *d_p = nullptr, *d_pd = nullptr, *d_ws = nullptr;
    void *d_sl[2] = {nullptr, nullptr}, *d_part = nullptr, *d_idx = nullptr, *d_bce = nullptr, *d_st = nullptr;
    auto dalloc = [&](void **p, size_t bytes) { return cudaMallocAsync(p, bytes ? bytes : 16, st); };
    const size_t slice_bytes = (size_t)n_lc * (size_t)chunk * (size_t)n_pdot * esz;
    rc = GCE_CE_OK;
    do {
        if ((e = dalloc(&d_t, 8 * (size_t)total)) || (e = dalloc(&d_m, 8 * (size_t)total)) ||
            (e = dalloc(&d_off, 8 * (size_t)(n_lc + 1))) || (e = dalloc(&d_p, 8 * (size_t)n_p)) ||
            (e = dalloc(&d_pd, 8 * (size_t)n_pdot)) || (e = dalloc(&d_ws, ws_bytes)) ||
            (e = dalloc(&d_sl[0], slice_bytes)) || (e = dalloc(&d_sl[1], slice_bytes)) ||
            (e = dalloc(&d_part, 8 * W * (size_t)n_lc * (size_t)n_chunks)) || (e = dalloc(&d_idx, 8 * (size_t)n_lc * k)) ||
            (e = dalloc(&d_bce, 4 * (size_t)n_lc * k)) || (e = dalloc(&d_st, 32 * (size_t)n_lc))) { rc = cuda_fail(e); break; }
        cudaMemcpyAsync(d_t, times, 8 * (size_t)total, cudaMemcpyHostToDevice, st);
        cudaMemcpyAsync(d_m, mags, 8 * (size_t)total, cudaMemcpyHostToDevice, st);
        cudaMemcpyAsync(d_off, lc_offsets, 8 * (size_t)(n_lc + 1), cudaMemcpyHostToDevice, st);
        cudaMemcpyAsync(d_p, periods, 8 * (size_t)n_p, cudaMemcpyHostToDevice, st);
        cudaMemcpyAsync(d_pd, pdots, 8 * (size_t)n_pdot, cudaMemcpyHostToDevice, st);
        int n_done = 0;
        for (int c = 0; c < n_chunks && rc == GCE_CE_OK; ++c) {
            const int64_t a = (int64_t)c * chunk, b = a + chunk < n_p ? a + chunk : n_p;
            if (a >= b) break;
            const int buf = c & 1;
            if (c >= 2) cudaStreamWaitEvent(st, ev_free[buf], 0);  // the copy that last read this slice buffer is done
            rc = gce_ce_search_partial((const double *)d_t, (const double *)d_m, (const int64_t *)d_off, n_lc, total,
                                       (const double *)d_p, n_p, (const double *)d_pd, n_pdot, prm, a, b, d_sl[buf],
                                       (int64_t *)d_part + (size_t)c * (size_t)n_lc * W, d_ws, ws_bytes, st);
            if (rc) break;
            ++n_done;
            cudaEventRecord(ev_done[buf], st);
            cudaStreamWaitEvent(st2, ev_done[buf], 0);
            const size_t width = (size_t)(b - a) * (size_t)n_pdot * esz;  // one light curve's rows of this slice
            e = cudaMemcpy2DAsync(static_cast<unsigned char *>(out_ce) + (size_t)a * (size_t)n_pdot * esz,
                                  (size_t)n_p * (size_t)n_pdot * esz, d_sl[buf], width, width, (size_t)n_lc,
                                  cudaMemcpyDeviceToHost, st2);
            if (e != cudaSuccess) { rc = cuda_fail(e); break; }
            cudaEventRecord(ev_free[buf], st2);
        }
        if (rc) break;
        if (k || prm->want_stats) {
            rc = gce_ce_merge_partials((const int64_t *)d_part, n_done, n_lc, prm, out_best_idx ? (int64_t *)d_idx : nullptr,
                                       out_best_ce ? (float *)d_bce : nullptr, out_stats ? (double *)d_st : nullptr, st);
            if (rc) break;
        }
        if (out_best_idx && k) cudaMemcpyAsync(out_best_idx, d_idx, 8 * (size_t)n_lc * k, cudaMemcpyDeviceToHost, st);
        if (out_best_ce && k) cudaMemcpyAsync(out_best_ce, d_bce, 4 * (size_t)n_lc * k, cudaMemcpyDeviceToHost, st);
        if (out_stats) cudaMemcpyAsync(out_stats, d_st, 32 * (size_t)n_lc, cudaMemcpyDeviceToHost, st);
    } while (0);
    e = cudaStreamSynchronize(st2);
    if (e != cudaSuccess && rc == GCE_CE_OK) rc = cuda_fail(e);
    void *frees[] = {d_t, d_m, d_off, d_p, d_pd, d_ws, d_sl[0], d_sl[1], d_part, d_idx, d_bce, d_st};
    for (void *p : frees)
        if (p) cudaFreeAsync(p, st);
    e = cudaStreamSynchronize(st);
    if (e != cudaSuccess && rc == GCE_CE_OK) rc = cuda_fail(e);
    for (int b = 0; b < 2; ++b) { cudaEventDestroy(ev_done[b]); cudaEventDestroy(ev_free[b]); }
    cudaStreamDestroy(st2);
    cudaStreamDestroy(st);
    return rc;
}

int gce_ce_search_host(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                       const double *periods, int64_t n_p, const double *pdots, int64_t n_pdot,
                       const gce_ce_params *prm, void *out_ce, int64_t *out_best_idx, float *out_best_ce,
                       double *out_stats) {
    int rc = check_params(prm);
    if (rc) return rc;
    if (!lc_offsets || n_lc < 0) return GCE_CE_ERR_POINTER;
    const int64_t total = lc_offsets[n_lc];
    rc = check_sizes(n_lc, total, n_p, n_pdot);
    if (rc) return rc;
    if ((prm->want_stats != 0) != (out_stats != nullptr)) return GCE_CE_ERR_POINTER;
    if ((prm->top_k > 0) != (out_best_idx != nullptr)) return GCE_CE_ERR_POINTER;
    if (out_best_ce && !out_best_idx) return GCE_CE_ERR_POINTER;
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

    cudaStream_t st;
    cudaError_t e = cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking);
    if (e != cudaSuccess) return cuda_fail(e);
    void *d_t = nullptr, *d_m = nullptr, *d_off = nullptr, *d_p = nullptr, *d_pd = nullptr, *d_ws = nullptr;
    void *d_ce = nullptr, *d_idx = nullptr, *d_bce = nullptr, *d_st = nullptr;
    auto dalloc = [&](void **p, size_t bytes) { return cudaMallocAsync(p, bytes ? bytes : 16, st); };
    rc = GCE_CE_OK;
    do {
        if ((e = dalloc(&d_t, 8 * (size_t)total)) || (e = dalloc(&d_m, 8 * (size_t)total)) ||
            (e = dalloc(&d_off, 8 * (size_t)(n_lc + 1))) || (e = dalloc(&d_p, 8 * (size_t)n_p)) ||
            (e = dalloc(&d_pd, 8 * (size_t)n_pdot)) || (e = dalloc(&d_ws, ws_bytes)) ||
            (e = dalloc(&d_ce, ce_bytes)) || (e = dalloc(&d_idx, 8 * (size_t)n_lc * k)) ||
            (e = dalloc(&d_bce, 4 * (size_t)n_lc * k)) || (e = dalloc(&d_st, 32 * (size_t)n_lc))) { rc = cuda_fail(e); break; }
        if (total) {
            cudaMemcpyAsync(d_t, times, 8 * (size_t)total, cudaMemcpyHostToDevice, st);
            cudaMemcpyAsync(d_m, mags, 8 * (size_t)total, cudaMemcpyHostToDevice, st);
        }
        cudaMemcpyAsync(d_off, lc_offsets, 8 * (size_t)(n_lc + 1), cudaMemcpyHostToDevice, st);
        if (n_p) cudaMemcpyAsync(d_p, periods, 8 * (size_t)n_p, cudaMemcpyHostToDevice, st);
        cudaMemcpyAsync(d_pd, pdots, 8 * (size_t)n_pdot, cudaMemcpyHostToDevice, st);
        rc = gce_ce_search((const double *)d_t, (const double *)d_m, (const int64_t *)d_off, n_lc, total,
                           (const double *)d_p, n_p, (const double *)d_pd, n_pdot, prm, out_ce ? d_ce : nullptr,
                           out_best_idx ? (int64_t *)d_idx : nullptr, out_best_ce ? (float *)d_bce : nullptr,
                           out_stats ? (double *)d_st : nullptr, d_ws, ws_bytes, st);
        if (rc) break;
        if (out_ce && ce_bytes) cudaMemcpyAsync(out_ce, d_ce, ce_bytes, cudaMemcpyDeviceToHost, st);
        if (out_best_idx && k) cudaMemcpyAsync(out_best_idx, d_idx, 8 * (size_t)n_lc * k, cudaMemcpyDeviceToHost, st);
        if (out_best_ce && k) cudaMemcpyAsync(out_best_ce, d_bce, 4 * (size_t)n_lc * k, cudaMemcpyDeviceToHost, st);
        if (out_stats && n_lc) cudaMemcpyAsync(out_stats, d_st, 32 * (size_t)n_lc, cudaMemcpyDeviceToHost, st);
    } while (0);
    void *frees[] = {d_t, d_m, d_off, d_p, d_pd, d_ws, d_ce, d_idx, d_bce, d_st};
    for (void *p : frees)
        if (p) cudaFreeAsync(p, st);
    e = cudaStreamSynchronize(st);
    if (e != cudaSuccess && rc == GCE_CE_OK) rc = cuda_fail(e);
    cudaStreamDestroy(st);
    return rc;
}

}  // extern "C"
