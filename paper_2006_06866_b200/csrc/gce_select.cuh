// gce_select.cuh -- S5 / Eq. 5 merges (k_merge_topk, k_merge_stats): per light curve, over CTAs or caller-supplied partial blobs
// Part of the single translation unit gce_ce.cu (compiled with -fmad=false); see the header comment there.
#pragma once
#include "gce_common.cuh"

namespace {

// ---- S5 / Eq. 5 merges.  One warp per light curve.  The candidates / partial sums of light curve lc live at
// base[lc * lc_stride + p * part_stride + ...], p < n_parts: inside one call the parts are the CTAs (jobs) of k_search,
// in gce_ce_merge_partials they are the caller's partial blobs (period ranges, batches, GPUs).  Keys are
// the exact integers (S = N*CE*2^42, flat q), so the merged result does not depend on the split.
// Partial blob of one light curve (int64 words): [0,K) S ascending, [K,2K) q, [2K,2K+8) Eq. 5 sums,
// [2K+8] N in the low 32 bits and the table's fixed-point shift above them, [2K+9] pivot.
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
    const int64_t nw = info ? (int64_t)info[lc].n | ((int64_t)info[lc].lshift << 32) : npts[(int64_t)lc * npts_stride];
    const int64_t n = nw & 0xffffffffll;
    const int lshift = (int)(nw >> 32);
    out_idx[(int64_t)lc * K + lane] = have ? top.q : -1;
    if (out_ce) out_ce[(int64_t)lc * K + lane] = have ? (float)((double)top.S * (ldexp(1.0, -lshift) / (double)(mult * n))) : CUDART_NAN_F;
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
    const int64_t nw = info ? (int64_t)info[lc].n | ((int64_t)info[lc].lshift << 32) : npts[(int64_t)lc * npts_stride];
    const int64_t n_pts = nw & 0xffffffffll;
    const int lshift = (int)(nw >> 32);
    const int64_t pivot = info ? info[lc].K : npts[(int64_t)lc * npts_stride + 1];
    if (out_raw) {
        int64_t *o = out_raw + (int64_t)lc * raw_stride;
        for (int i = 0; i < kStatWords; ++i) o[i] = (int64_t)acc[i];
        o[kStatWords] = nw;
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
    const double scale = ldexp(1.0, -lshift) / (double)(mult * n_pts);
    const double mean_d = sum_d / n;
    double var = sum_d2 / n - mean_d * mean_d;
    if (var < 0.0 || acc[6] == acc[7]) var = 0.0;  // min == max: every trial has the same CE, the spread is exactly 0
    const double mn = (double)(int64_t)acc[6] * scale;
    if (acc[6] == acc[7]) { o[0] = mn; o[1] = 0.0; o[2] = mn; o[3] = CUDART_NAN; return; }  // one CE value only: mean = min exactly
    const double mean = ((double)pivot + mean_d) * scale;
    const double sd = sqrt(var) * scale;
    o[0] = mean; o[1] = sd; o[2] = mn; o[3] = (mean - mn) / sd;
}


}  // namespace
