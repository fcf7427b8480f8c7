// gce_search.cuh -- S2..S5: the fold + bin + entropy kernel (k_search)
// Part of the single translation unit gce_ce.cu (compiled with -fmad=false); see the header comment there.
#pragma once
#include "gce_common.cuh"

namespace {

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

// WIDE counters (one 32-bit counter per trial, light curves beyond the 16-bit range): plain count, any size.
__device__ __forceinline__ int64_t ltab_one(const int64_t *__restrict__ sL, const int64_t *__restrict__ gL, const uint32_t c) {
    return c < (uint32_t)kLtabSmem ? sL[c] : gL[c];
}

// Counter words per thread: two 16-bit counters per word (WSH = 1) or one 32-bit counter per word (WSH = 0, WIDE).
__host__ __device__ constexpr int n_words(int R, int WSH) { return WSH ? (R + 1) / 2 : R; }

// S2 + S3 for one point and the R trials of this thread (DESIGN.md section 3; PAPER.md:100 Eq. 3, :106).
//   a = dt*invP ; b = dt2*c ; x = a + b ; y = x*n_phi          (RN each, never fused)
//   j = floor(y) - n_phi*floor(x)                               two exact round-down magic adds, |y| < 2^51
// j equals floor(y) mod n_phi except when RN(x*n_phi) lands exactly on the next multiple of n_phi, where it is
// n_phi: that count goes to an extra histogram row that is folded into row 0 when the segment is closed.
// PZ: every trial of the thread has c = +-0, so x = a bit for bit (a >= +0) and two operations are skipped.
// MODE 1 / 2 (only with extended counter rows, EXT in k_search): trials share a floor(x).  The caller has sorted the
// thread's trials by c, largest first, so that for every point x_0 >= x_1 >= ... (dt2 >= 0, RN is monotone), and has
// checked per tile that the trials sharing a floor stay less than one cycle apart over the whole light curve:
//   MODE 1: the two trials of a counter word share floor(x) of the odd slot   ((c_even - c_odd) * dt_max^2 < 1)
//   MODE 2: all R trials share floor(x) of the last slot                       ((c_0 - c_{R-1}) * dt_max^2 < 1)
// Then every j = floor(y) - n_phi * floor(x_base) lies in [0, 2 n_phi]; rows n_phi .. 2 n_phi are folded back (mod
// n_phi) when the magnitude bin is closed.  Fewer FP64 instructions and one row-offset multiply-add per counter word
// instead of per trial, the same bits.
// SINK receives (address of the counter word, slot r): the search kernel adds the slot's increment there with one RED
// (RedSink); the per-point bin dump of gce_ce_debug_bins records the row instead (rs = 1, hb = 0: the address IS the row).
struct RedSink {
    uint32_t inc0, inc1;  // increments of the even / odd trial of a counter word (16-bit fields)
    __device__ __forceinline__ void operator()(const uint32_t addr, const int r) const { red_add_u32(addr, (r & 1) ? inc1 : inc0); }
};

template <int R, bool SHARE_P, bool PZ, int MODE, int WSH = 1, typename SINK>
__device__ __forceinline__ void fold_bin_add(const double2 p, const double (&invP)[R], const double (&cc)[R],
                                             const double nphi_d, const uint32_t negn, const uint32_t rs,
                                             const uint32_t (&hb)[n_words(R, WSH)], const SINK &sink) {
    double a;
    if (SHARE_P) a = __dmul_rn(p.x, invP[0]);
    if constexpr (MODE != 0) {
        static_assert(MODE == 0 || (SHARE_P && !PZ && R % 2 == 0 && WSH == 1), "shared floors need one period, Pdot != 0 and packed counters");
        double x[R];
#pragma unroll
        for (int r = 0; r < R; ++r) x[r] = __dadd_rn(a, __dmul_rn(p.y, cc[r]));
        uint32_t Ix = 0;
        if (MODE == 2) Ix = (uint32_t)__double2loint(__dadd_rd(x[R - 1], kMagic));
#pragma unroll
        for (int r = 0; r < R; r += 2) {
            if (MODE == 1) Ix = (uint32_t)__double2loint(__dadd_rd(x[(r + 1) % R], kMagic));
            const uint32_t base = Ix * (negn * rs) + hb[r >> 1];  // one multiply-add for the word's common row offset
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const double y = __dmul_rn(x[(r + h) % R], nphi_d);
                const uint32_t Iy = (uint32_t)__double2loint(__dadd_rd(y, kMagic));
                sink(Iy * rs + base, r + h);
            }
        }
    } else {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (!SHARE_P) a = __dmul_rn(p.x, invP[r]);
            const double x = PZ ? a : __dadd_rn(a, __dmul_rn(p.y, cc[r]));
            const double y = __dmul_rn(x, nphi_d);
            const uint32_t Iy = (uint32_t)__double2loint(__dadd_rd(y, kMagic));
            const uint32_t Ix = (uint32_t)__double2loint(__dadd_rd(x, kMagic));
            // floor(x)'s row offset is ready before floor(y): one multiply-add between floor(y) and the RED
            const uint32_t t = Ix * (negn * rs) + hb[r >> WSH];
            sink(Iy * rs + t, r);
        }
    }
}

template <int R, bool SHARE_P, bool PZ, int MODE, int WSH = 1, typename SINK>
__device__ __forceinline__ void fold_range(const double2 *__restrict__ sp, int kk, const int ke, const double (&invP)[R],
                                           const double (&cc)[R], const double nphi_d, const uint32_t negn,
                                           const uint32_t rs, const uint32_t (&hb)[n_words(R, WSH)], const SINK &sink) {
    // Four points per trip, the next two read ahead (the buffer has two spare points).  The two source forms compile to
    // different ptxas schedules; each fold mode takes the one that measured faster (C5 / C4: -2 %, C3: +1 % otherwise).
    if constexpr (MODE == 0) {
        if (ke - kk >= 4) {
            double2 a[2], b[2];
#pragma unroll
            for (int g = 0; g < 2; ++g) a[g] = sp[kk + g];
            do {
#pragma unroll
                for (int g = 0; g < 2; ++g) b[g] = sp[kk + 2 + g];
#pragma unroll
                for (int g = 0; g < 2; ++g) fold_bin_add<R, SHARE_P, PZ, MODE, WSH>(a[g], invP, cc, nphi_d, negn, rs, hb, sink);
#pragma unroll
                for (int g = 0; g < 2; ++g) a[g] = sp[kk + 4 + g];
#pragma unroll
                for (int g = 0; g < 2; ++g) fold_bin_add<R, SHARE_P, PZ, MODE, WSH>(b[g], invP, cc, nphi_d, negn, rs, hb, sink);
                kk += 4;
            } while (ke - kk >= 4);
        }
    } else {
        if (ke - kk >= 4) {
            double2 a0 = sp[kk], a1 = sp[kk + 1];
            do {
                const double2 b0 = sp[kk + 2], b1 = sp[kk + 3];
                fold_bin_add<R, SHARE_P, PZ, MODE, WSH>(a0, invP, cc, nphi_d, negn, rs, hb, sink);
                fold_bin_add<R, SHARE_P, PZ, MODE, WSH>(a1, invP, cc, nphi_d, negn, rs, hb, sink);
                a0 = sp[kk + 4];
                a1 = sp[kk + 5];
                fold_bin_add<R, SHARE_P, PZ, MODE, WSH>(b0, invP, cc, nphi_d, negn, rs, hb, sink);
                fold_bin_add<R, SHARE_P, PZ, MODE, WSH>(b1, invP, cc, nphi_d, negn, rs, hb, sink);
                kk += 4;
            } while (ke - kk >= 4);
        }
    }
    for (; kk < ke; ++kk) fold_bin_add<R, SHARE_P, PZ, MODE, WSH>(sp[kk], invP, cc, nphi_d, negn, rs, hb, sink);
}


// Rare path (|y| >= 2^51 for some point): the listing of DESIGN.md section 3 with 64-bit integers.
template <int R, bool SHARE_P, int WSH = 1, typename SINK>
__device__ __forceinline__ void fold_bin_add_generic(const double2 p, const double (&invP)[R], const double (&cc)[R],
                                                     const int n_phi, const uint32_t rs, const uint32_t (&hb)[n_words(R, WSH)],
                                                     const SINK &sink) {
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int j = fold_bin_generic(p.x, p.y, invP[SHARE_P ? 0 : r], cc[r], n_phi);
        sink((uint32_t)j * rs + hb[r >> WSH], r);
    }
}
template <int R, bool SHARE_P, int WSH = 1, typename SINK>
__device__ __forceinline__ void fold_range_generic(const double2 *__restrict__ sp, int kk, const int ke,
                                                   const double (&invP)[R], const double (&cc)[R], const int n_phi,
                                                   const uint32_t rs, const uint32_t (&hb)[n_words(R, WSH)], const SINK &sink) {
    for (; kk < ke; ++kk) fold_bin_add_generic<R, SHARE_P, WSH>(sp[kk], invP, cc, n_phi, rs, hb, sink);
}

// S4, first half: close magnitude bin `seg_i`.  fetch_word reads and clears this thread's counter word of phase bin j
// (two 16-bit counts, trials 2*w2 and 2*w2+1); close_word adds it to the phase marginal and accumulates sum L(n_ij).
template <bool EXT>
__device__ __forceinline__ uint32_t fetch_word(const int j, const int n_phi, const uint32_t rs, const uint32_t hbw) {
    uint32_t w = exch0_u32(hbw + (uint32_t)j * rs);
    if (EXT) w += exch0_u32(hbw + (uint32_t)(j + n_phi) * rs);  // extended rows n_phi .. 2 n_phi - 1 fold back mod n_phi
    if (j == 0) w += exch0_u32(hbw + (uint32_t)(EXT ? 2 * n_phi : n_phi) * rs);  // phase bin 0 takes over the last row
    return w;
}

// DUMP (gce_ce_debug_histogram): dpos[r] is the position of slot r's trial in the caller's list (-1: not listed); the
// count this word contributes to Eq. 4 is written to out_counts[lc][dpos][j][seg_i].
template <int R, bool DUMP, bool BIG, bool WIDE>
__device__ __forceinline__ void close_word(const uint32_t w, const int j, const int w2, const int n_phi, const uint32_t us,
                                           int64_t (&S2)[R], const int64_t *__restrict__ sL, const SearchParams &prm,
                                           const int lc, const int (&dpos)[R], const int seg_i) {
    if constexpr (WIDE) {  // word w2 is the 32-bit count of trial slot w2
        S2[w2 < R ? w2 : 0] += ltab_one(sL, prm.ltab, w);
        if (DUMP) {
            const int d0 = dpos[w2 < R ? w2 : 0];
            if (d0 >= 0) prm.out_counts[(((int64_t)lc * prm.n_dump + d0) * n_phi + j) * prm.n_m + seg_i] = w;
        }
    } else {
        int64_t v0, v1;
        ltab_pair<BIG>(sL, prm.ltab, w, us, v0, v1);
        S2[(2 * w2) < R ? 2 * w2 : 0] += v0;
        if (2 * w2 + 1 < R) S2[(2 * w2 + 1) < R ? 2 * w2 + 1 : 0] += v1;
        if (DUMP) {
            const uint32_t c0 = (w & 0xffffu) >> us, c1 = w >> (16u + us);
            const int d0 = dpos[(2 * w2) < R ? 2 * w2 : 0], d1 = dpos[(2 * w2 + 1) < R ? 2 * w2 + 1 : 0];
            if (d0 >= 0) prm.out_counts[(((int64_t)lc * prm.n_dump + d0) * n_phi + j) * prm.n_m + seg_i] = c0;
            if (2 * w2 + 1 < R && d1 >= 0) prm.out_counts[(((int64_t)lc * prm.n_dump + d1) * n_phi + j) * prm.n_m + seg_i] = c1;
        }
    }
}

// All phase bins of magnitude bin seg_i.  The phase marginal is a register array (REGM, compile-time n_phi) or a second
// set of counter rows in shared memory updated with one RED per word (no registers, so more threads fit per SM).
// With a compile-time n_phi the read-and-clear atomics of kCloseGroup phase bins are issued back to back before
// their results are used, so their latency overlaps.
// OVL (NEXT item N2): 50 %-overlapping phase bins -- bin k holds the plain cells k-1 and k (cyclic), so
// the looked-up count is w[k] + w[k-1] (packed 16-bit pairs; needs 2N <= 65535); the folds and the plain marginal are
// unchanged, the overlap costs one add per word.
template <int NPHI, bool REGM, int R, bool DUMP, bool BIG, bool OVL, bool EXT, bool WIDE>
__device__ __forceinline__ void close_mag_bin(const int n_phi, const uint32_t rs, const uint32_t marg_off, const uint32_t us,
                                              const uint32_t (&hb)[n_words(R, WIDE ? 0 : 1)],
                                              uint32_t (&mg)[REGM ? NPHI : 1][n_words(R, WIDE ? 0 : 1)], int64_t (&S2)[R],
                                              const int64_t *__restrict__ sL, const SearchParams &prm, const int lc,
                                              const int (&dpos)[R], const int seg_i) {
    constexpr int RW = n_words(R, WIDE ? 0 : 1);
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
                for (int w2 = 0; w2 < RW; ++w2) w[jj][w2] = fetch_word<EXT>(j0 + jj, n_phi, rs, hb[w2]);
#pragma unroll
            for (int jj = 0; jj < G; ++jj)
#pragma unroll
                for (int w2 = 0; w2 < RW; ++w2) {
                    const uint32_t ww = w[jj][w2];
                    if (REGM) mg[REGM ? j0 + jj : 0][w2] += ww;
                    else red_add_u32(hb[w2] + marg_off + (uint32_t)(j0 + jj - w2) * rs, ww);
                    if (!OVL) close_word<R, DUMP, BIG, WIDE>(ww, j0 + jj, w2, n_phi, us, S2, sL, prm, lc, dpos, seg_i);
                    else {
                        if (j0 + jj == 0) first[w2] = ww;
                        else close_word<R, DUMP, BIG, WIDE>(ww + prev[w2], j0 + jj, w2, n_phi, us, S2, sL, prm, lc, dpos, seg_i);
                        prev[w2] = ww;
                    }
                }
        }
    } else {
        for (int j = 0; j < n_phi; ++j) {
#pragma unroll
            for (int w2 = 0; w2 < RW; ++w2) {
                const uint32_t ww = fetch_word<EXT>(j, n_phi, rs, hb[w2]);
                red_add_u32(hb[w2] + marg_off + (uint32_t)(j - w2) * rs, ww);
                if (!OVL) close_word<R, DUMP, BIG, WIDE>(ww, j, w2, n_phi, us, S2, sL, prm, lc, dpos, seg_i);
                else {
                    if (j == 0) first[w2] = ww;
                    else close_word<R, DUMP, BIG, WIDE>(ww + prev[w2], j, w2, n_phi, us, S2, sL, prm, lc, dpos, seg_i);
                    prev[w2] = ww;
                }
            }
        }
    }
    if (OVL) {  // bin 0 = cells n_phi-1 and 0
#pragma unroll
        for (int w2 = 0; w2 < RW; ++w2)
            close_word<R, DUMP, BIG, WIDE>(first[w2] + prev[w2], 0, w2, n_phi, us, S2, sL, prm, lc, dpos, seg_i);
    }
}

// Per-trial constants of the R consecutive trial slots s0 .. s0 + R - 1 of one thread:
// invP = 1/P, c = ((-0.5 * Pdot) * invP) * invP.  fast: every |y| of the light curve stays below 2^51, so the magic-add
// floors are exact; pz: every c is +-0 (then x = a bit for bit).  Shared by k_search and k_debug_bins.
template <int R, bool SHARE_P>
__device__ __forceinline__ void trial_slot_constants(const SearchParams &prm, const int64_t s0, const double nphi_d,
                                                     const double dt_max, double (&invP)[R], double (&cc)[R],
                                                     int64_t (&qv)[R], bool (&valid)[R], bool &fast, bool &pz) {
    fast = true;
    pz = true;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int64_t s = s0 + r;
        valid[r] = s < prm.n_trials;
        const int64_t q = valid[r] ? s : 0;
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
}

// EXT: sort the thread's trial slots by c, largest first (so x_0 >= x_1 >= ... for every point: dt2 >= 0 and RN is
// monotone), keeping qv / valid / org with their trial, and report how far apart the phases get over the light curve:
// pair_ok: the two trials of every counter word stay within one cycle, quad_ok: all R trials do.
template <int R>
__device__ __forceinline__ void sort_slots_by_c(double (&cc)[R], int64_t (&qv)[R], bool (&valid)[R], int (&org)[R],
                                                const double dt_max, bool &pair_ok, bool &quad_ok) {
    auto cswap = [&](const int i, const int j) {  // compare-exchange: afterwards cc[i] >= cc[j]
        if (cc[i] < cc[j]) {
            const double tc = cc[i]; cc[i] = cc[j]; cc[j] = tc;
            const int64_t tq = qv[i]; qv[i] = qv[j]; qv[j] = tq;
            const bool tv = valid[i]; valid[i] = valid[j]; valid[j] = tv;
            const int to = org[i]; org[i] = org[j]; org[j] = to;
        }
    };
    if (R == 4) { cswap(0, 1 % R); cswap(2 % R, 3 % R); cswap(0, 2 % R); cswap(1 % R, 3 % R); cswap(1 % R, 2 % R); }
    else cswap(0, 1 % R);
    const double d2 = dt_max * dt_max;
#pragma unroll
    for (int w2 = 0; w2 < (R + 1) / 2; ++w2) pair_ok = pair_ok && ((cc[2 * w2] - cc[(2 * w2 + 1) % R]) * d2 < 0.999);
    quad_ok = quad_ok && ((cc[0] - cc[R - 1]) * d2 < 0.999);
}

// NPHI > 0: compile-time n_phi (unrolled S4); NPHI == 0: any n_phi <= 64.  REGM: phase marginal in registers (needs a
// compile-time n_phi); otherwise the marginal is a second set of counter rows in shared memory.  NTC: compile-time
// threads per CTA, or 0 = blockDim.x (any multiple of 32 up to 640).  R = trials per thread.  SHARE_P: the R trials of a
// thread share one period (n_pdot % R == 0).  EXT: 2 n_phi + 1 counter rows, shared floors (fold_bin_add MODE 1 / 2).
// DUMP (gce_ce_debug_histogram): the same kernel, plan and tiles as the search, but only tiles that hold a listed trial
// are processed and, instead of the search outputs, the count tables (and CE) of the listed trials are written.
// WIDE (NEXT item N3, "light curves of any length"): one 32-bit counter per trial instead of two 16-bit
// fields per word, for calls whose light curves may exceed the 16-bit range (gce_ce_params.max_lc_points); counts are
// looked up directly (no byte-offset trick), the k ln k table is as long as the longest light curve.
template <int NPHI, bool REGM, int R, bool SHARE_P, bool DUMP, bool EXT, int NTC, bool WIDE = false>
__global__ void __launch_bounds__(NTC > 0 ? NTC : 640, 1) k_search(const SearchParams prm) {
    static_assert(!REGM || NPHI > 0, "register marginals need a compile-time n_phi");
    static_assert(!EXT || (SHARE_P && R % 2 == 0 && !WIDE), "extended rows serve trial pairs that share a period");
    static_assert(!WIDE || !REGM, "wide counters: generic family only");
    constexpr int WSH = WIDE ? 0 : 1;
    constexpr int RW = n_words(R, WSH);  // 32-bit words per (bin, thread): two 16-bit counters each, or one 32-bit counter
    constexpr int NPHI_REG = REGM ? NPHI : 1;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int NT = NTC > 0 ? NTC : (int)blockDim.x, NW = NT >> 5;
    const int tid = threadIdx.x, lane = tid & 31;
    const int n_phi = NPHI > 0 ? NPHI : prm.n_phi, n_m = prm.n_m;
    const uint32_t rs = (uint32_t)NT * 4u;  // bytes between the counter rows of consecutive phase bins

    // shared-memory carve-up (dynamic part; the L table is static so that lookups are LDS.64 [offset + const]), points last
    __shared__ __align__(16) int64_t sL[kLtabSmem];  // static: its shared address is a link-time constant
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw);                     // [2]
    int *sseg = reinterpret_cast<int *>(full + 2);                               // [n_m + 1] (<= 65)
    uint64_t *sstat = reinterpret_cast<uint64_t *>(sseg + GCE_CE_MAX_BINS + 4);  // [kMaxWarps][kStatWords]
    // Cold per-tile state lives in shared memory, not in registers, so that the hot loop has the register file to
    // itself (it is register-starved: with the phase marginals in registers ptxas otherwise issues the dependent FP64
    // instructions of a chain back to back): the warps' running top-k lists and the light curve's scalars.
    int64_t *stop = reinterpret_cast<int64_t *>(sstat + kMaxWarps * kStatWords);  // [kMaxWarps][32] x (S, q), lane-sorted list
    int64_t *sthr = stop + kMaxWarps * 64;                                       // [kMaxWarps] x (S, q) of the k-th element
    volatile double *sinfo = reinterpret_cast<volatile double *>(sthr + kMaxWarps * 2);  // [2]: dt_max, K (bits)
    uint32_t *hist = reinterpret_cast<uint32_t *>(const_cast<double *>(sinfo) + 2); // [RW][n_phi + 1][NT], 16-byte aligned
    const int hist_rows = EXT ? 2 * n_phi + 1 : n_phi + 1;  // EXT: a pair's shared floor(x) lets j reach 2 n_phi
    const uint32_t plane = (uint32_t)hist_rows * rs;                             // bytes per counter-word plane
    // shared-memory marginal (!REGM): RW planes of n_phi rows after the histogram; word (w2, j) of this thread is at
    // hb[w2] + marg_off + (j - w2) * rs
    const uint32_t marg_off = (uint32_t)RW * plane;
    const uint32_t hist_words = (uint32_t)(REGM ? RW * hist_rows : RW * (hist_rows + n_phi)) * (uint32_t)NT;
    double2 *spts = reinterpret_cast<double2 *>(hist + hist_words);              // [cap_points + 2]

    const int lc = blockIdx.x / prm.jobs_per_lc;
    const int job = blockIdx.x % prm.jobs_per_lc;
    // Tiles of a job: a contiguous range -- or, in the shared-floor kernels (EXT), the tiles job, job + J, job + 2 J, ...:
    // there a tile's cost depends on its period range (which fold mode qualifies: 4.5 to 5.25 FP64 instructions per
    // point-fold), and the stride gives every CTA the same mix so that the CTAs of the last wave end together
    // (C3: 71.0 -> 67.7 ms).  The other kernels keep the contiguous form.
    const int64_t tile_lo = EXT ? (int64_t)job : prm.tiles_per_lc * job / prm.jobs_per_lc;
    const int64_t tile_hi = prm.tiles_per_lc * (job + 1) / prm.jobs_per_lc;
    const int64_t tile_step = EXT ? (int64_t)prm.jobs_per_lc : 1;
    const int n_tiles = EXT ? (int)((prm.tiles_per_lc - job + tile_step - 1) / tile_step) : (int)(tile_hi - tile_lo);
    const int N = prm.info[lc].n;
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
    stop[2 * tid] = kInfS;
    stop[2 * tid + 1] = kInfS;
    if (tid < 2 * NW) sthr[tid] = kInfS;
    if (tid == 0) {
        sinfo[0] = prm.info[lc].dt_max;
        sinfo[1] = __longlong_as_double(prm.info[lc].K);
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        if (n_tiles > 0)
            for (int g = 0; g < 2 && g < total_seq; ++g) issue_chunk(g);
    }
    __syncthreads();

    const double nphi_d = (double)n_phi;
    const uint32_t negn = 0u - (uint32_t)n_phi;
    uint32_t hb[RW];
#pragma unroll
    for (int w2 = 0; w2 < RW; ++w2) hb[w2] = smem_u32(hist) + (uint32_t)tid * 4u + (uint32_t)w2 * plane;
    const bool ovl = prm.overlap != 0;  // N2: 2N table entries per trial
    const double ce_scale = N > 0 ? ldexp(1.0, -prm.info[lc].lshift) / (double)(ovl ? 2 * N : N) : 0.0;
    const uint32_t us = (!WIDE && (ovl ? 2 : 1) * N <= 8191) ? 3u : 0u;  // counter unit 2^us: a field is its table entry's byte offset
    const RedSink sink{1u << us, WIDE ? 1u : 0x10000u << us};
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
        const int64_t s0 = (tile_lo + tl * tile_step) * TILE + (int64_t)tid * R;  // first trial slot of this thread
        if (DUMP && single) {  // skip tiles without a listed trial (streamed tiles keep their place in the chunk sequence)
            bool any = false;
            const int64_t t0q = (tile_lo + tl * tile_step) * TILE;
            for (int64_t i = tid; i < prm.n_dump; i += NT) {
                const int64_t q = prm.trial_q[i];
                any = any || (q >= t0q && q < t0q + TILE);
            }
            if (!__syncthreads_or(any)) continue;
        }
        // ---- per-trial constants
        double invP[R], cc[R];  // SHARE_P: only invP[0] is used
        bool fast, pz;
        uint32_t orgp = 0;  // 2 bits per slot: the trial (0..R-1, relative to s0) held by slot r (EXT sorts the slots by c)
        bool pair_ok = false, quad_ok = false;
        int dpos[R];  // DUMP: position of the slot's trial in the caller's list
#pragma unroll
        for (int r = 0; r < R; ++r) dpos[r] = -1;
        {
            int64_t qv[R];
            bool valid[R];
            int org[R];
            const double dt_max = sinfo[0];
            trial_slot_constants<R, SHARE_P>(prm, s0, nphi_d, dt_max, invP, cc, qv, valid, fast, pz);
            fast = __all_sync(0xffffffffu, fast);
            pz = __all_sync(0xffffffffu, pz);
#pragma unroll
            for (int r = 0; r < R; ++r) org[r] = r;
            pair_ok = EXT && fast && !pz;
            quad_ok = pair_ok;
            if (EXT) {
                sort_slots_by_c<R>(cc, qv, valid, org, dt_max, pair_ok, quad_ok);
                pair_ok = __all_sync(0xffffffffu, pair_ok);
                quad_ok = __all_sync(0xffffffffu, quad_ok);
            }
#pragma unroll
            for (int r = 0; r < R; ++r) orgp |= (uint32_t)org[r] << (2 * r);
            if (DUMP) {
                for (int64_t i = 0; i < prm.n_dump; ++i) {
                    const int64_t q = prm.trial_q[i];
#pragma unroll
                    for (int r = 0; r < R; ++r)
                        if (valid[r] && qv[r] == q) dpos[r] = (int)i;
                }
            }
        }

        int64_t S2[R];
#pragma unroll
        for (int r = 0; r < R; ++r) S2[r] = 0;

        int seg_s = 0;  // magnitude bins finished so far, counted in this warp's (rotated) order
        for (int c = 0; c < n_chunks; ++c) {
            const int buf = single ? 0 : (g & 1);
            if (!single || tl == 0 || DUMP) mbar_wait(&full[buf], single ? 0u : (uint32_t)((g >> 1) & 1));
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
                        if (pz) fold_range<R, SHARE_P, true, 0, WSH>(sp, lo, hi, invP, cc, nphi_d, negn, rs, hb, sink);
                        else if (EXT && quad_ok) fold_range<R, SHARE_P, false, EXT ? 2 : 0, WSH>(sp, lo, hi, invP, cc, nphi_d, negn, rs, hb, sink);
                        else if (EXT && pair_ok) fold_range<R, SHARE_P, false, EXT ? 1 : 0, WSH>(sp, lo, hi, invP, cc, nphi_d, negn, rs, hb, sink);
                        else fold_range<R, SHARE_P, false, 0, WSH>(sp, lo, hi, invP, cc, nphi_d, negn, rs, hb, sink);
                    } else {
                        fold_range_generic<R, SHARE_P, WSH>(sp, lo, hi, invP, cc, n_phi, rs, hb, sink);
                    }
                }
                if (b1 > k_end) break;  // the bin continues in the next buffer
                // ---------------- S4: the bin is complete; a cell holds at most b1 - b0 points
                if (b1 > b0) {
                    // a cell of this bin holds at most b1 - b0 points (twice that with overlapping bins)
                    if constexpr (WIDE) {
                        if (!ovl) close_mag_bin<NPHI, REGM, R, DUMP, true, false, EXT, true>(n_phi, rs, marg_off, us, hb, mg, S2, sL, prm, lc, dpos, seg_i);
                        else close_mag_bin<NPHI, REGM, R, DUMP, true, true, EXT, true>(n_phi, rs, marg_off, us, hb, mg, S2, sL, prm, lc, dpos, seg_i);
                    } else if (!ovl) {
                        if (us == 3u && b1 - b0 < kLtabSmem)
                            close_mag_bin<NPHI, REGM, R, DUMP, false, false, EXT, false>(n_phi, rs, marg_off, us, hb, mg, S2, sL, prm, lc, dpos, seg_i);
                        else
                            close_mag_bin<NPHI, REGM, R, DUMP, true, false, EXT, false>(n_phi, rs, marg_off, us, hb, mg, S2, sL, prm, lc, dpos, seg_i);
                    } else {
                        if (us == 3u && 2 * (b1 - b0) < kLtabSmem)
                            close_mag_bin<NPHI, REGM, R, DUMP, false, true, EXT, false>(n_phi, rs, marg_off, us, hb, mg, S2, sL, prm, lc, dpos, seg_i);
                        else
                            close_mag_bin<NPHI, REGM, R, DUMP, true, true, EXT, false>(n_phi, rs, marg_off, us, hb, mg, S2, sL, prm, lc, dpos, seg_i);
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
                if constexpr (WIDE) {
                    S1[w2 < R ? w2 : 0] += ltab_one(sL, prm.ltab, w);
                } else {
                    int64_t v0, v1;
                    ltab_pair<decltype(big)::value>(sL, prm.ltab, w, us, v0, v1);
                    S1[(2 * w2) < R ? 2 * w2 : 0] += v0;
                    if (2 * w2 + 1 < R) S1[(2 * w2 + 1) < R ? 2 * w2 + 1 : 0] += v1;
                }
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
            S[r] = S1[r] - S2[r];  // = N * CE * 2^lshift, exact
            ce[r] = N > 0 ? (double)S[r] * ce_scale : CUDART_NAN;
        }
        if (DUMP) {
#pragma unroll
            for (int r = 0; r < R; ++r)
                if (dpos[r] >= 0 && prm.out_ce_at) prm.out_ce_at[(int64_t)lc * prm.n_dump + dpos[r]] = ce[r];
        } else {
            if (prm.out_ce) {
                const int64_t o = (int64_t)lc * prm.n_trials + s0;
                float *o32 = reinterpret_cast<float *>(prm.out_ce) + o;
                double cet[R];  // CE in trial order (EXT has sorted the slots by c)
#pragma unroll
                for (int t = 0; t < R; ++t) {
                    cet[t] = ce[t];
                    if (EXT) {
#pragma unroll
                        for (int r = 0; r < R; ++r)
                            if ((int)((orgp >> (2 * r)) & 3u) == t) cet[t] = ce[r];
                    }
                }
                if (R == 4 && !prm.ce_fp64 && s0 + R <= prm.n_trials && (reinterpret_cast<uintptr_t>(o32) & 15u) == 0) {
                    *reinterpret_cast<float4 *>(o32) = make_float4((float)cet[0], (float)cet[1 % R], (float)cet[2 % R], (float)cet[3 % R]);
                } else {
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        if (s0 + r >= prm.n_trials) continue;
                        if (prm.ce_fp64) reinterpret_cast<double *>(prm.out_ce)[o + r] = cet[r];
                        else o32[r] = (float)cet[r];
                    }
                }
            }
            // the slot's trial, recomputed here instead of being carried through the hot loop
            int64_t qv[R];
            bool valid[R];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int64_t s = s0 + (int64_t)(EXT ? ((orgp >> (2 * r)) & 3u) : (uint32_t)r);
                valid[r] = s < prm.n_trials;
                qv[r] = (valid[r] ? s : 0) + prm.q_off;
            }
            if (prm.top_k > 0) {
                volatile int64_t *vtop = stop + 2 * tid, *vthr = sthr + 2 * (tid >> 5);
                WarpTopK top;
                top.k = prm.top_k;
                top.S = vtop[0]; top.q = vtop[1]; top.thrS = vthr[0]; top.thrq = vthr[1];
#pragma unroll
                for (int r = 0; r < R; ++r) top.offer((valid[r] && N > 0) ? S[r] : kInfS, (valid[r] && N > 0) ? qv[r] : kInfS);
                vtop[0] = top.S; vtop[1] = top.q;
                if (lane == 0) { vthr[0] = top.thrS; vthr[1] = top.thrq; }
            }
            if (prm.part_stats != nullptr && N > 0) {  // Eq. 5 partial sums of this tile, warp-reduced, exact integers
                const int64_t K = __double_as_longlong(sinfo[1]);
                __int128 a = 0;
                u128_t b = 0;
                int64_t mn = kInfS, mx = INT64_MIN;
                uint32_t cnt = 0;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    if (!valid[r]) continue;
                    const int64_t d = S[r] - K;   // |d| <= max(S, K) < 2^60.1 (table_shift, gce_ce.cu)
                    a += d;
                    b += (u128_t)((__int128)d * d);
                    mn = S[r] < mn ? S[r] : mn;
                    mx = S[r] > mx ? S[r] : mx;
                    ++cnt;
                }
                u128_t au = (u128_t)a;
                for (int o = 16; o > 0; o >>= 1) {
                    au += shfl_xor_u128(au, o);
                    b += shfl_xor_u128(b, o);            // <= 32 * R * 2^120.2 < 2^128
                    const int64_t m2 = __shfl_xor_sync(0xffffffffu, mn, o), m3 = __shfl_xor_sync(0xffffffffu, mx, o);
                    mn = m2 < mn ? m2 : mn;
                    mx = m3 > mx ? m3 : mx;
                    cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
                }
                if (lane == 0) stat_add(sstat + (tid >> 5) * kStatWords, cnt, au, b, 0, mn, mx);
            }
        }
    }

    // Dump mode skips tiles without a listed trial, so a CTA may get here without ever having waited for the bulk copy
    // its prologue issued; a CTA must not exit with a copy into its own shared memory in flight (the next CTA on the SM
    // could see the late bytes or the late mbarrier transaction).  Waiting on a phase that has completed returns at once.
    if constexpr (DUMP) {
        if (tid == 0 && single && n_chunks > 0 && n_tiles > 0) mbar_wait(&full[0], 0u);
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
        __syncthreads();  // the warps' lists in shared memory are final (lanes >= K hold +inf)
        if (tid < 32) {
            WarpTopK top;
            top.reset(K);
            for (int w = 0; w < NW; ++w) top.offer(stop[2 * (w * 32 + lane)], stop[2 * (w * 32 + lane) + 1]);
            if (lane < K) {
                const int64_t o = ((int64_t)lc * prm.jobs_per_lc + job) * K + lane;
                prm.part_S[o] = top.S;
                prm.part_q[o] = top.q;
            }
        }
    }
}

// Host side of one instantiation: opt in to the dynamic shared memory once per device, then launch.
template <int NPHI, bool REGM, int R, bool SHARE_P, bool DUMP, bool EXT, int NTC, bool WIDE = false>
cudaError_t launch_search(const SearchParams &sp, const Plan &plan, int32_t n_lc, cudaStream_t st) {
    auto kern = k_search<NPHI, REGM, R, SHARE_P, DUMP, EXT, NTC, WIDE>;
    static std::mutex mu;
    static size_t smem_set[64] = {};  // largest opt-in made so far, per device
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    {
        std::lock_guard<std::mutex> lock(mu);
        if (plan.smem > smem_set[dev]) {
            e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)plan.smem);
            if (e != cudaSuccess) return e;
            smem_set[dev] = plan.smem;
        }
    }
    if (NTC > 0 && plan.nt != NTC) return cudaErrorInvalidValue;
    const unsigned grid = (unsigned)((int64_t)n_lc * plan.jobs_per_lc);
    kern<<<grid, plan.nt, plan.smem, st>>>(sp);
    return cudaGetLastError();
}

}  // namespace
