// gce_common.cuh -- constants, shared structs, TMA / mbarrier helpers, warp top-k, Eq. 5 integer sums, frozen fold arithmetic
// Included by every translation unit of the library (all compiled with -fmad=false); see the header comment of gce_ce.cu.
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>
#include <string.h>

#include <mutex>

#include "gce_ce.h"

// ---- types and entry points shared between the translation units (external linkage)
namespace gce {

struct LcInfo {
    int32_t n;
    int32_t lshift;  // fixed-point shift of this call's k ln k table (table_shift in gce_ce.cu: 42 .. 52 by table length, less beyond 2^16 entries)
    double dt_max;
    int64_t K;  // N * H(m) in 2^-lshift fixed point = L(N) - sum_i L(points in magnitude bin i): CE <= H(m), pivot of the Eq. 5 sums
};

struct SearchParams {
    const double2 *pts;        // [total_points] (dt, dt2), grouped by magnitude bin inside each light curve
    const int32_t *seg;        // [n_lc][n_m + 1] segment offsets relative to the light curve start
    const LcInfo *info;        // [n_lc]
    const int64_t *lc_offsets; // [n_lc + 1]
    const int64_t *ltab;       // [ltab_n] fixed-point k ln k
    const double *periods;
    const double *pdots;
    const int64_t *trial_q;    // DUMP only: [n_dump] flat trial indices whose count tables are written out
    int64_t n_dump;            // DUMP only
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
    uint32_t *out_counts;      // DUMP only: [n_lc][n_dump][n_phi][n_m]
    double *out_ce_at;         // DUMP only: [n_lc][n_dump] or NULL
};

// Which kernel variant runs, with how many threads, over how many CTAs: decided from sizes only (deterministic, no
// device query), so gce_ce_workspace_bytes, gce_ce_search and the debug dump agree.
struct Plan {
    int R;             // trials per thread
    bool share_p;      // the R trials of a thread share one period
    int nphi_t;        // compile-time n_phi of the kernel (15, 20, 30, 50) or 0 = generic
    bool regm;         // phase marginal in registers instead of shared memory
    bool ext;          // 2 n_phi + 1 counter rows: trials of a thread share one floor(x) (gce_search.cuh)
    bool wide;         // one 32-bit counter per trial (light curves beyond the 16-bit range), generic family only
    int nt;            // threads per CTA (multiple of 32)
    int cap_points;    // shared-memory point buffer capacity
    size_t smem;       // dynamic shared memory per CTA
    int64_t tiles_per_lc;
    int jobs_per_lc;
};

// One launcher per kernel family (compile-time n_phi) and mode, each in its own translation unit
// (gce_search_family.cu compiled with -DGCE_FAMILY=<n_phi> -DGCE_DUMP=<0|1>) so that the build runs in parallel.
// They pick the instantiation the plan names and launch it; cudaErrorInvalidValue if the plan names none.
#define GCE_DECLARE_FAMILY(N)                                                                                  \
    cudaError_t launch_search_n##N##_d0(const SearchParams &sp, const Plan &plan, int32_t n_lc, cudaStream_t st); \
    cudaError_t launch_search_n##N##_d1(const SearchParams &sp, const Plan &plan, int32_t n_lc, cudaStream_t st);
GCE_DECLARE_FAMILY(0)
GCE_DECLARE_FAMILY(15)
GCE_DECLARE_FAMILY(20)
GCE_DECLARE_FAMILY(30)
GCE_DECLARE_FAMILY(50)
#undef GCE_DECLARE_FAMILY

}  // namespace gce

namespace {

using namespace gce;

constexpr int kLtabSmem = 1024;   // entries of the L table mirrored in shared memory
constexpr int kLfixShift = 42;    // L table fixed point: at least 2^-42 for tables of up to 2^16 entries (short tables take up to 2^-52; longer ones less than 42)
constexpr double kMagic = 6755399441055744.0;  // 1.5 * 2^52: RD-add puts floor(y) in the low mantissa word
constexpr double kYSafe = 2251799813685248.0;  // 2^51: |y| below this -> the magic-add floor is exact
constexpr int64_t kInfS = INT64_MAX;
constexpr int kSmemLimit = 227 * 1024 - 8 * kLtabSmem;  // dynamic shared memory per CTA: 227 KB minus the static L table
constexpr int kStatWords = 8;     // partial Eq. 5 sums: n, sum d (i128), sum d^2 (u192), min S, max S; d = S - K
constexpr int kMaxWarps = 20;     // warps per CTA of the largest variant (640 threads)
// Threads per CTA of the register-marginal kernels (compile-time n_phi), per family.  512 threads = 4 warps per SM
// sub-partition at <= 128 registers; 384 = 3 warps at <= 168.  n_phi = 30 keeps 60 marginal registers per thread: at
// 128 the hot loop is starved of registers and at 384 threads it runs 4.6 % faster (measured on C5).
#ifndef GCE_NT_N15
#define GCE_NT_N15 512
#endif
#ifndef GCE_NT_N20
#define GCE_NT_N20 512
#endif
#ifndef GCE_NT_N30
#define GCE_NT_N30 384
#endif
#ifndef GCE_NT_N50
#define GCE_NT_N50 512
#endif
constexpr int nt_regm(int n_phi) { return n_phi == 15 ? GCE_NT_N15 : n_phi == 20 ? GCE_NT_N20 : n_phi == 30 ? GCE_NT_N30 : GCE_NT_N50; }
constexpr int kCloseGroup = 5;    // phase bins whose read-and-clear atomics are in flight together in S4

struct FalseT { static constexpr bool value = false; };
struct TrueT { static constexpr bool value = true; };

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


}  // namespace
