// gce_ablation.cu -- NOT part of the product library: the histogram layout BASELINE.json's north_star sketches, built
// so that the design the product rejects has a measured number beside it (bench.py --ablation,
// profiles/r3_design_ablation.md).  Linked into its own libgce_ablation.so; libgce_ce.so never sees it.
//
// The sketch: "each warp owns a trial and keeps a private shared-memory histogram, updated with warp-aggregated
// (match_any) shared atomics; marginals and the entropy sum use warp shuffles".  Here: one CTA per (light curve, job);
// the CTA normalises and stages its light curve in shared memory (dt, dt^2, magnitude bin); each of its 16 warps takes
// trials in turn; for a trial the 32 lanes fold 32 points at a time with the frozen arithmetic of DESIGN.md section 3
// (same magic-add floors as k_search), group equal cells with __match_any_sync and let the lowest lane of each group
// add the group's size to the warp's private n_phi x n_m table with one shared atomic; then lane j closes phase bin j
// (marginal and sum of k ln k from a shared fp64 table) and the warp sums with shuffles.  CE is written as fp32.
// Same -fmad=false build as the product.
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

constexpr int kWarps = 16;
constexpr double kMagic = 6755399441055744.0;  // 1.5 * 2^52: the low word of RD(v + kMagic) is floor(v) mod 2^32

__global__ void __launch_bounds__(kWarps * 32) k_ablation_warp_per_trial(
    const double *__restrict__ times, const double *__restrict__ mags, const int64_t *__restrict__ lc_offsets,
    const double *__restrict__ periods, const double *__restrict__ pdots, int64_t n_p, int64_t n_pdot, int n_phi,
    int n_m, int jobs_per_lc, float *__restrict__ out_ce) {
    extern __shared__ __align__(16) unsigned char smem[];
    const int lc = blockIdx.x / jobs_per_lc, job = blockIdx.x % jobs_per_lc;
    const int64_t off = lc_offsets[lc];
    const int N = (int)(lc_offsets[lc + 1] - off);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    double2 *pts = reinterpret_cast<double2 *>(smem);                      // [N] (dt, dt^2)
    double *ltab = reinterpret_cast<double *>(pts + N);                    // [N + 1] k ln k
    unsigned *hist = reinterpret_cast<unsigned *>(ltab + N + 1);           // [kWarps][n_phi * n_m]
    unsigned char *mbin = reinterpret_cast<unsigned char *>(hist + kWarps * n_phi * n_m);  // [N]
    __shared__ double red[3][kWarps];
    // S1: t0, min / max magnitude by block reduction
    double t0 = 1e300, lo = 1e300, hi = -1e300;
    for (int k = tid; k < N; k += blockDim.x) {
        t0 = fmin(t0, times[off + k]); lo = fmin(lo, mags[off + k]); hi = fmax(hi, mags[off + k]);
    }
    for (int o = 16; o > 0; o >>= 1) {
        t0 = fmin(t0, __shfl_xor_sync(0xffffffffu, t0, o));
        lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
        hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
    }
    if (lane == 0) { red[0][warp] = t0; red[1][warp] = lo; red[2][warp] = hi; }
    __syncthreads();
    for (int w = 0; w < kWarps; ++w) { t0 = fmin(t0, red[0][w]); lo = fmin(lo, red[1][w]); hi = fmax(hi, red[2][w]); }
    const double r = __dsub_rn(hi, lo);
    for (int k = tid; k < N; k += blockDim.x) {
        const double dt = __dsub_rn(times[off + k], t0);
        pts[k] = make_double2(dt, __dmul_rn(dt, dt));
        int i = 0;
        if (r != 0.0) {
            i = __double2int_rd(__dmul_rn(__ddiv_rn(__dsub_rn(mags[off + k], lo), r), (double)n_m));
            i = i < n_m - 1 ? i : n_m - 1;
        }
        mbin[k] = (unsigned char)i;
    }
    for (int k = tid; k <= N; k += blockDim.x) ltab[k] = k < 2 ? 0.0 : (double)k * log((double)k);
    __syncthreads();

    unsigned *h = hist + warp * n_phi * n_m;
    const int cells = n_phi * n_m;
    const int64_t n_trials = n_p * n_pdot;
    const int64_t q_lo = n_trials * job / jobs_per_lc, q_hi = n_trials * (job + 1) / jobs_per_lc;
    const double nphi_d = (double)n_phi;
    for (int64_t q = q_lo + warp; q < q_hi; q += kWarps) {
        for (int c = lane; c < cells; c += 32) h[c] = 0u;
        __syncwarp();
        const double invP = __ddiv_rn(1.0, periods[q / n_pdot]);
        const double cc = __dmul_rn(__dmul_rn(__dmul_rn(-0.5, pdots[q % n_pdot]), invP), invP);
        for (int k0 = 0; k0 < N; k0 += 32) {
            const int k = k0 + lane;
            const bool act = k < N;
            const unsigned am = __ballot_sync(0xffffffffu, act);
            if (act) {
                const double2 p = pts[k];
                const double x = __dadd_rn(__dmul_rn(p.x, invP), __dmul_rn(p.y, cc));
                const double y = __dmul_rn(x, nphi_d);
                const int fy = __double2loint(__dadd_rd(y, kMagic)), fx = __double2loint(__dadd_rd(x, kMagic));
                int j = fy - n_phi * fx;
                j = j >= n_phi ? j - n_phi : j;   // RN(x n_phi) may reach n_phi (floor(x) + 1): that is phase bin 0
                const int cell = j * n_m + (int)mbin[k];
                const unsigned grp = __match_any_sync(am, cell);
                if ((__ffs(grp) - 1) == lane) atomicAdd(&h[cell], (unsigned)__popc(grp));
            }
        }
        __syncwarp();
        double s = 0.0;  // N * CE = sum_j L(n_j) - sum_ij L(n_ij)
        for (int j = lane; j < n_phi; j += 32) {
            unsigned nj = 0;
            double sij = 0.0;
            for (int i = 0; i < n_m; ++i) {
                const unsigned c = h[j * n_m + i];
                nj += c;
                sij += ltab[c];
            }
            s += ltab[nj] - sij;
        }
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == 0) out_ce[(int64_t)lc * n_trials + q] = (float)(s / (double)N);
        __syncwarp();
    }
}

}  // namespace

extern "C" {

// Device pointers; out_ce float[n_lc][n_p][n_pdot].  Light curves of up to max_points points (shared-memory staging);
// returns 0, or -2 for sizes this probe does not handle, or -4 with the cudaError_t in *cuda_err_host.
int gce_ablation_warp_per_trial(const double *times, const double *mags, const int64_t *lc_offsets, int32_t n_lc,
                                int32_t max_points, const double *periods, int64_t n_p, const double *pdots,
                                int64_t n_pdot, int32_t n_phi, int32_t n_m, float *out_ce, int32_t *cuda_err_host,
                                void *stream) {
    if (n_lc < 1 || max_points < 1 || n_phi < 1 || n_phi > 64 || n_m < 1 || n_m > 64 || n_p < 1 || n_pdot < 1) return -2;
    const size_t smem = (size_t)max_points * 16 + ((size_t)max_points + 1) * 8 + (size_t)kWarps * n_phi * n_m * 4 + (size_t)max_points + 16;
    if (smem > 200 * 1024) return -2;
    cudaError_t e = cudaFuncSetAttribute(k_ablation_warp_per_trial, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    // about 8 CTAs per SM over the launch, as the product's plan does
    int jobs = (int)((148 * 8 + n_lc - 1) / n_lc);
    if ((int64_t)jobs > n_p * n_pdot) jobs = (int)(n_p * n_pdot);
    if (e == cudaSuccess) {
        k_ablation_warp_per_trial<<<n_lc * jobs, kWarps * 32, smem, reinterpret_cast<cudaStream_t>(stream)>>>(
            times, mags, lc_offsets, periods, pdots, n_p, n_pdot, n_phi, n_m, jobs, out_ce);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        if (cuda_err_host) *cuda_err_host = (int)e;
        return -4;
    }
    return 0;
}

}  // extern "C"
