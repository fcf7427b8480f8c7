// gce_preprocess.cuh -- S1 (k_preprocess) and the k ln k table it builds on the side
// Part of the single translation unit gce_ce.cu (compiled with -fmad=false); see the header comment there.
#pragma once
#include "gce_common.cuh"

namespace {

// L(k) = k ln k in 2^-shift fixed point.  shift = 42 for k < 2^17 (L < 2^62, and sum_j L(n_j) <= L(N), so the sums fit in
// int64); longer tables (32-bit counters) take the smaller shift table_shift() chooses.
__device__ __forceinline__ int64_t ltab_entry(int k, int shift) {
    return k < 2 ? 0 : __double2ll_rn(ldexp((double)k * log((double)k), shift));
}

// ------------------------------------------------------------------------------------------------ S0 (optional, N4)
// The paper's normalisation (reading Q19): per light curve and per filter, u = (m - median) / sd
// with sd the population standard deviation, so that filters can be merged into one light curve; S1 then bins the
// merged u over its range.  Frozen arithmetic: the median is an order statistic (the mean of the two middle values,
// (a + b) * 0.5, when the count is even); mean and sum of squares are SEQUENTIAL sums over the filter's points in
// light-curve order, one rounding per operation (a thread per filter walks the light curve); sd == 0 -> u = 0.
// One CTA per light curve.  Order statistics by an 8-pass radix select over the order-preserving 64-bit keys.
// Cost: the sequential sums are part of the contract (they fix the rounding order the oracle also uses), so ONE thread
// per filter walks the whole light curve twice, and every filter present adds 8 radix passes over the light curve (16
// when its count is even): O(N) serial work per light curve -- microseconds at the paper's 1e3 points (DESIGN.md section
// 14), but seconds per call for a wide call near 2^26 points.  The pipelined host entry (large cubes, 8 period chunks)
// repeats S0 and S1 for each chunk.  For very long normalised light curves, normalise once outside and pass normalise = 0.
__device__ __forceinline__ unsigned long long order_key(double v) {
    const unsigned long long b = (unsigned long long)__double_as_longlong(v);
    return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}
__device__ __forceinline__ double key_value(unsigned long long k) {
    const unsigned long long b = (k >> 63) ? (k & 0x7fffffffffffffffull) : ~k;
    return __longlong_as_double((long long)b);
}

__global__ void __launch_bounds__(256) k_normalise(const double *__restrict__ mags, const int32_t *__restrict__ filt,
                                                   const int64_t *__restrict__ lc_offsets, double *__restrict__ out) {
    __shared__ unsigned int hist[256];
    __shared__ unsigned long long sh_prefix;
    __shared__ long long sh_rank;
    __shared__ int sh_cnt[GCE_CE_MAX_FILTERS];
    __shared__ double sh_med[GCE_CE_MAX_FILTERS], sh_sd[GCE_CE_MAX_FILTERS];
    const int lc = blockIdx.x, tid = threadIdx.x;
    const int64_t off = lc_offsets[lc];
    const int64_t n = lc_offsets[lc + 1] - off;
    if (n <= 0) return;
    const double *m = mags + off;
    const int32_t *f = filt ? filt + off : nullptr;
    if (tid < GCE_CE_MAX_FILTERS) sh_cnt[tid] = 0;
    __syncthreads();
    for (int64_t k = tid; k < n; k += blockDim.x) atomicAdd(&sh_cnt[(f ? f[k] : 0) & (GCE_CE_MAX_FILTERS - 1)], 1);
    __syncthreads();
    // sequential mean and standard deviation: thread g walks the light curve for filter g
    if (tid < GCE_CE_MAX_FILTERS && sh_cnt[tid] > 0) {
        const double nf = (double)sh_cnt[tid];
        double sum = 0.0;
        for (int64_t k = 0; k < n; ++k)
            if (((f ? f[k] : 0) & (GCE_CE_MAX_FILTERS - 1)) == tid) sum = __dadd_rn(sum, m[k]);
        const double mean = __ddiv_rn(sum, nf);
        double ss = 0.0;
        for (int64_t k = 0; k < n; ++k)
            if (((f ? f[k] : 0) & (GCE_CE_MAX_FILTERS - 1)) == tid) {
                const double d = __dsub_rn(m[k], mean);
                ss = __dadd_rn(ss, __dmul_rn(d, d));
            }
        sh_sd[tid] = __dsqrt_rn(__ddiv_rn(ss, nf));
    }
    // medians: radix select of the two middle order statistics, filter by filter (block-wide)
    for (int g = 0; g < GCE_CE_MAX_FILTERS; ++g) {
        const int nf = sh_cnt[g];
        if (nf == 0) continue;  // uniform
        double mid[2];
        for (int h = 0; h < 2; ++h) {
            const long long want = h == 0 ? (nf - 1) / 2 : nf / 2;
            if (h == 1 && want == (nf - 1) / 2) { mid[1] = mid[0]; break; }
            if (tid == 0) { sh_prefix = 0ull; sh_rank = want; }
            for (int pass = 7; pass >= 0; --pass) {
                hist[tid] = 0u;  // 256 threads
                __syncthreads();
                const unsigned long long prefix = sh_prefix;
                for (int64_t k = tid; k < n; k += blockDim.x) {
                    if (((f ? f[k] : 0) & (GCE_CE_MAX_FILTERS - 1)) != g) continue;
                    const unsigned long long key = order_key(m[k]);
                    if (pass == 7 || (key >> (8 * (pass + 1))) == prefix) atomicAdd(&hist[(key >> (8 * pass)) & 0xffu], 1u);
                }
                __syncthreads();
                if (tid == 0) {
                    long long r = sh_rank;
                    int b = 0;
                    while (r >= (long long)hist[b]) { r -= hist[b]; ++b; }
                    sh_rank = r;
                    sh_prefix = (prefix << 8) | (unsigned long long)b;
                }
                __syncthreads();
            }
            mid[h] = key_value(sh_prefix);
            __syncthreads();
        }
        if (tid == 0) sh_med[g] = (nf & 1) ? mid[0] : __dmul_rn(__dadd_rn(mid[0], mid[1]), 0.5);
    }
    __syncthreads();
    for (int64_t k = tid; k < n; k += blockDim.x) {
        const int g = (f ? f[k] : 0) & (GCE_CE_MAX_FILTERS - 1);
        const double sd = sh_sd[g];
        out[off + k] = sd == 0.0 ? 0.0 : __ddiv_rn(__dsub_rn(m[k], sh_med[g]), sd);
    }
}

// ------------------------------------------------------------------------------------------------ S1
// CTAs 0 .. n_lc-1: one per light curve.  Output points are permuted so equal magnitude bins are contiguous (counts do
// not depend on point order); seg[lc][i] is the first point of magnitude bin i, seg[lc][n_m] = N.
// CTAs n_lc ..: 256 entries each of the table L(k), k < ltab_n, that S4 looks up (one launch less than a kernel of its own).
// A light curve longer than max_points (the counter range of this call's k_search) is marked empty: CE = NaN, best index -1.
__global__ void __launch_bounds__(256) k_preprocess(const double *__restrict__ times, const double *__restrict__ mags,
                                                    const int64_t *__restrict__ lc_offsets, const int n_lc, const int n_m,
                                                    double2 *__restrict__ pts, int32_t *__restrict__ seg,
                                                    LcInfo *__restrict__ info, int64_t *__restrict__ ltab, const int ltab_n,
                                                    const int lshift, const int mult, const int max_points) {
    if ((int)blockIdx.x >= n_lc) {
        const int k = ((int)blockIdx.x - n_lc) * 256 + (int)threadIdx.x;
        if (k < ltab_n) ltab[k] = ltab_entry(k, lshift);
        return;
    }
    __shared__ MinMax3 sh_red[8];
    __shared__ int sh_cnt[GCE_CE_MAX_BINS + 1];
    __shared__ int sh_cur[GCE_CE_MAX_BINS];
    const int lc = blockIdx.x;
    const int64_t off = lc_offsets[lc];
    const int64_t n64 = lc_offsets[lc + 1] - off;
    if (n64 < 0 || n64 > (int64_t)max_points) {  // uniform per CTA
        for (int i = threadIdx.x; i <= n_m; i += blockDim.x) seg[(int64_t)lc * (n_m + 1) + i] = 0;
        if (threadIdx.x == 0) info[lc] = LcInfo{0, lshift, 0.0, 0};  // rejected: treated as empty
        return;
    }
    const int n = (int)n64;
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
        int64_t K = ltab_entry(mult * n, lshift);  // mult = 2 with overlapping phase bins: every point is counted twice
        for (int i = 0; i < n_m; ++i) {
            const int c = sh_cnt[i];
            seg[(int64_t)lc * (n_m + 1) + i] = acc;
            sh_cur[i] = acc;
            acc += c;
            K -= ltab_entry(mult * c, lshift);
        }
        info[lc].K = K;
        seg[(int64_t)lc * (n_m + 1) + n_m] = acc;
        info[lc].n = n;
        info[lc].lshift = lshift;
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

}  // namespace
