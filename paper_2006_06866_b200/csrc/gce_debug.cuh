// gce_debug.cuh -- test-only per-point bin dump (k_debug_bins) that runs the search kernel's own fold functions
// Part of gce_ce.cu (compiled with -fmad=false); see the header comment there.
#pragma once
#include "gce_search.cuh"

namespace {

// Records, per trial slot, the histogram row the production fold (fold_bin_add / fold_bin_add_generic of
// gce_search.cuh) computes: called with row stride 1 and row base 0, the "address" it hands to the sink IS the row.
struct RowSink {
    uint32_t *rows;
    __device__ __forceinline__ void operator()(const uint32_t addr, const int r) const { rows[r] = addr; }
};

// Fold modes of the search kernel (gce_search.cuh): which of them k_search takes for a thread is decided per tile and
// warp; here it is decided for the one thread that owns trial q, or forced by the caller to cover every mode.
enum : int { kFoldAuto = 0, kFoldPlain = 1, kFoldPair = 2, kFoldQuad = 3, kFoldGeneric = 4, kFoldPdotZero = 5 };

// Phase bin and magnitude bin of every point of light curve `lc` for trial q, in the caller's point order.  The thread
// context of k_search is rebuilt exactly: trial q lives in the slot group s0 = q - q % R with its R - 1 neighbours, the
// constants come from trial_slot_constants, the slots are sorted by c when shared floors are possible, and the rows come
// from the same fold_bin_add instantiations; rows n_phi .. 2 n_phi fold back modulo n_phi as in fetch_word.
// out_mode[0] = the mode used (k_Fold*), or -1 when the forced mode's precondition does not hold (bins are then -1).
template <int R, bool SHARE_P>
__global__ void __launch_bounds__(256) k_debug_bins(const double *__restrict__ times, const double *__restrict__ mags,
                                                    const int64_t *__restrict__ lc_offsets, const SearchParams prm,
                                                    const int lc, const int64_t q, const int force_mode,
                                                    int32_t *__restrict__ out_phase, int32_t *__restrict__ out_mag,
                                                    int32_t *__restrict__ out_mode) {
    constexpr int RW = (R + 1) / 2;
    __shared__ MinMax3 sh_red[8];
    const int n_phi = prm.n_phi, n_m = prm.n_m;
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
    const double dt_max = n > 0 ? __dsub_rn(v.tmax, v.tmin) : 0.0;
    const double nphi_d = (double)n_phi;
    const uint32_t negn = 0u - (uint32_t)n_phi;

    double invP[R], cc[R];
    int64_t qv[R];
    bool valid[R];
    bool fast, pz;
    trial_slot_constants<R, SHARE_P>(prm, q - q % R, nphi_d, dt_max, invP, cc, qv, valid, fast, pz);
    int org[R];
#pragma unroll
    for (int s = 0; s < R; ++s) org[s] = s;
    constexpr bool CAN_SHARE = SHARE_P && R % 2 == 0;
    bool pair_ok = CAN_SHARE && fast && !pz, quad_ok = pair_ok;
    if (CAN_SHARE && (force_mode == kFoldAuto || force_mode == kFoldPair || force_mode == kFoldQuad))
        sort_slots_by_c<R>(cc, qv, valid, org, dt_max, pair_ok, quad_ok);
    else pair_ok = quad_ok = false;
    int mode = force_mode;
    if (mode == kFoldAuto) mode = !fast ? kFoldGeneric : pz ? kFoldPdotZero : quad_ok ? kFoldQuad : pair_ok ? kFoldPair : kFoldPlain;
    const bool ok = (mode == kFoldGeneric) || (mode == kFoldPlain && fast) || (mode == kFoldPdotZero && fast && pz) ||
                    (mode == kFoldPair && pair_ok) || (mode == kFoldQuad && quad_ok);
    if (threadIdx.x == 0 && out_mode) out_mode[0] = ok ? mode : -1;
    int slot = 0;
#pragma unroll
    for (int s = 0; s < R; ++s)
        if (valid[s] && qv[s] == q) slot = s;
    const uint32_t hb[RW] = {};
    for (int k = threadIdx.x; k < n; k += blockDim.x) {
        const double dt = __dsub_rn(t[k], v.tmin);
        const double2 p = make_double2(dt, __dmul_rn(dt, dt));
        uint32_t rows[R];
        const RowSink sink{rows};
        if (!ok) { out_phase[k] = -1; out_mag[k] = -1; continue; }
        if (mode == kFoldGeneric) fold_bin_add_generic<R, SHARE_P>(p, invP, cc, n_phi, 1u, hb, sink);
        else if (mode == kFoldPdotZero) fold_bin_add<R, SHARE_P, true, 0>(p, invP, cc, nphi_d, negn, 1u, hb, sink);
        else if (mode == kFoldPlain) fold_bin_add<R, SHARE_P, false, 0>(p, invP, cc, nphi_d, negn, 1u, hb, sink);
        else if (mode == kFoldPair) fold_bin_add<R, SHARE_P, false, CAN_SHARE ? 1 : 0>(p, invP, cc, nphi_d, negn, 1u, hb, sink);
        else fold_bin_add<R, SHARE_P, false, CAN_SHARE ? 2 : 0>(p, invP, cc, nphi_d, negn, 1u, hb, sink);
        uint32_t row = rows[0];
#pragma unroll
        for (int s = 1; s < R; ++s)
            if (s == slot) row = rows[s];
        out_phase[k] = (int32_t)(row % (uint32_t)n_phi);  // rows n_phi .. 2 n_phi fold back (fetch_word)
        out_mag[k] = mag_bin(m[k], v.mmin, r, n_m);
    }
}

}  // namespace
