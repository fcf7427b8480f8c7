// gce_preprocess.cuh -- S1 (k_preprocess), the k ln k table (k_ltab) and the test-only per-point bin dump (k_debug_bins)
// Part of the single translation unit gce_ce.cu (compiled with -fmad=false); see the header comment there.
#pragma once
#include "gce_common.cuh"

namespace {

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


}  // namespace
