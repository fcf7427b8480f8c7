// gce_search_family.cu -- the k_search instantiations of ONE kernel family, compiled once per (family, mode):
//   -DGCE_FAMILY=<0|15|20|30|50>   compile-time n_phi of the family (0 = generic, any n_phi <= 64, shared-memory marginal)
//   -DGCE_DUMP=<0|1>               0: the search kernels; 1: the same kernels in dump mode (gce_ce_debug_histogram)
// so that the ten translation units build in parallel (paper_2006_06866_b200/build.py).  Every unit is compiled with
// -fmad=false.  The launcher picks the instantiation that gce_ce.cu's make_plan named.
#include "gce_search.cuh"

#ifndef GCE_FAMILY
#error "compile with -DGCE_FAMILY=<0|15|20|30|50> -DGCE_DUMP=<0|1>"
#endif
#ifndef GCE_DUMP
#error "compile with -DGCE_DUMP=<0|1>"
#endif

#define GCE_CAT3(a, b, c) a##b##c
#define GCE_LAUNCHER(n, d) GCE_CAT3(launch_search_n, n, _d##d)
#define GCE_LAUNCHER_NAME(n, d) GCE_LAUNCHER(n, d)

namespace gce {

cudaError_t GCE_LAUNCHER_NAME(GCE_FAMILY, GCE_DUMP)(const SearchParams &sp, const Plan &plan, int32_t n_lc, cudaStream_t st) {
    constexpr bool D = GCE_DUMP != 0;
    constexpr int N = GCE_FAMILY;
    if (plan.nphi_t != N) return cudaErrorInvalidValue;
    if (plan.wide && N != 0) return cudaErrorInvalidValue;
#if GCE_FAMILY == 0
    if (plan.regm || plan.ext) return cudaErrorInvalidValue;
    if (plan.wide) {  // 32-bit counters (N3: light curves of any length)
        if (plan.share_p && plan.R == 4) return launch_search<0, false, 4, true, D, false, 0, true>(sp, plan, n_lc, st);
        if (plan.share_p && plan.R == 2) return launch_search<0, false, 2, true, D, false, 0, true>(sp, plan, n_lc, st);
        if (!plan.share_p && plan.R == 4) return launch_search<0, false, 4, false, D, false, 0, true>(sp, plan, n_lc, st);
        return cudaErrorInvalidValue;
    }
    if (plan.share_p && plan.R == 4) return launch_search<0, false, 4, true, D, false, 0>(sp, plan, n_lc, st);
    if (plan.share_p && plan.R == 2) return launch_search<0, false, 2, true, D, false, 0>(sp, plan, n_lc, st);
    if (!plan.share_p && plan.R == 4) return launch_search<0, false, 4, false, D, false, 0>(sp, plan, n_lc, st);
    return cudaErrorInvalidValue;
#elif GCE_FAMILY == 50
    // 50 phase bins (the paper's production binning): R = 2, the register marginal of 4 trials would take 100 registers
    if (!plan.regm || plan.ext || plan.R != 2) return cudaErrorInvalidValue;
    if (plan.share_p) return launch_search<50, true, 2, true, D, false, nt_regm(50)>(sp, plan, n_lc, st);
    return launch_search<50, true, 2, false, D, false, nt_regm(50)>(sp, plan, n_lc, st);
#else
    if (!plan.regm) return cudaErrorInvalidValue;
#if GCE_FAMILY != 30
    if (plan.ext) {
        if (!plan.share_p || plan.R != 4) return cudaErrorInvalidValue;
        return launch_search<N, true, 4, true, D, true, nt_regm(N)>(sp, plan, n_lc, st);
    }
#else
    if (plan.ext) return cudaErrorInvalidValue;
#endif
    if (plan.share_p && plan.R == 4) return launch_search<N, true, 4, true, D, false, nt_regm(N)>(sp, plan, n_lc, st);
    if (plan.share_p && plan.R == 2) return launch_search<N, true, 2, true, D, false, nt_regm(N)>(sp, plan, n_lc, st);
    if (!plan.share_p && plan.R == 4) return launch_search<N, true, 4, false, D, false, nt_regm(N)>(sp, plan, n_lc, st);
    return cudaErrorInvalidValue;
#endif
}

}  // namespace gce
