// gce_probe.cuh -- diagnostic kernels behind gce_ce_probe_rate: the per-SM issue rates the roofline denominators assume
// Part of gce_ce.cu (compiled with -fmad=false); see the header comment there.
#pragma once
#include "gce_common.cuh"

namespace {

// kind 0: eight independent DADD / DMUL chains per thread (no dependent pair closer than eight instructions), 1024 threads
// per SM: FP64 lane-operations per SM per clock.  out[2 * cta] = thread-operations of the CTA, out[2 * cta + 1] = its clocks.
__global__ void __launch_bounds__(1024, 1) k_probe_fp64(double *sink, long long *out, int iters, double c) {
    double a0 = threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    __syncthreads();
    const long long t0 = clock64();
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            a0 = __dadd_rn(a0, c); a1 = __dmul_rn(a1, c); a2 = __dadd_rn(a2, c); a3 = __dmul_rn(a3, c);
            a4 = __dadd_rn(a4, c); a5 = __dmul_rn(a5, c); a6 = __dadd_rn(a6, c); a7 = __dmul_rn(a7, c);
        }
    }
    __syncthreads();
    const long long t1 = clock64();
    sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (threadIdx.x == 0) {
        out[2 * blockIdx.x] = (long long)blockDim.x * iters * 32;
        out[2 * blockIdx.x + 1] = t1 - t0;
    }
}

// kind 1: conflict-free RED.shared.add.u32 (thread t updates bank t mod 32, eight rows in turn), 1024 threads per SM:
// shared-memory wavefronts per SM per clock (one wavefront per warp instruction).  out[2 * cta] = warp instructions.
__global__ void __launch_bounds__(1024, 1) k_probe_shared(unsigned *sink, long long *out, int iters) {
    __shared__ unsigned rows[8][1024];
    for (int r = 0; r < 8; ++r) rows[r][threadIdx.x] = 0u;
    const uint32_t base = smem_u32(&rows[0][threadIdx.x]);
    __syncthreads();
    const long long t0 = clock64();
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u)
            asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(base + (uint32_t)u * 4096u), "r"(1u) : "memory");
    }
    __syncthreads();
    const long long t1 = clock64();
    unsigned s = 0;
    for (int r = 0; r < 8; ++r) s += rows[r][threadIdx.x];
    sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0) {
        out[2 * blockIdx.x] = (long long)(blockDim.x / 32) * iters * 8;
        out[2 * blockIdx.x + 1] = t1 - t0;
    }
}

}  // namespace
