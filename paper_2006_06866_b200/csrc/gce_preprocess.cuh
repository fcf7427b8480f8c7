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
