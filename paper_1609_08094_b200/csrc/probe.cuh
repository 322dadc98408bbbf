// probe.cuh -- tensor-pipe peaks of the device the library runs on, measured in the process that measures the kernels.
// First: the FP64 tensor-core (mma.sync.m8n8k4.f64, SASS DMMA) peak: the roofline
// denominator of the FP64 contraction kernel, measured in the same process as the numerator
// (triples_probe_fp64_peak; bench.py roofline.peak).  Register-resident operands, 32 independent accumulator tiles
// per warp, 8 warps per SM: nothing but the DMMA pipe is exercised.
#pragma once
#include "ptx.cuh"

namespace tb {

constexpr int PROBE_ACC = 32, PROBE_THREADS = 256;

__global__ void __launch_bounds__(PROBE_THREADS)
fp64_peak_kernel(double* __restrict__ out, int iters) {
    double c[PROBE_ACC][2];
#pragma unroll
    for (int i = 0; i < PROBE_ACC; ++i) { c[i][0] = threadIdx.x * 1e-9; c[i][1] = i * 1e-9; }
    const double a = 1.0 + threadIdx.x * 1e-6, b = 1.0 - threadIdx.x * 1e-6;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < PROBE_ACC; ++i) dmma_884(c[i][0], c[i][1], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < PROBE_ACC; ++i) s += c[i][0] + c[i][1];
    out[blockIdx.x * (size_t)blockDim.x + threadIdx.x] = s;
}

// ---------------------------------------------------------------------------------------------------------------
// tcgen05.mma peak of the two kinds the packed contractions use (triples_probe_tc_peak; bench.py roofline.peak of
// gemm_f16split_kernel and gemm_emu64_kernel): the same instruction shapes, issued the same way -- CTA pairs
// (cta_group::2, M = 256), one elected lane of the leader's converged warp, operands resident in shared memory
// (128-byte swizzled rows, never re-loaded), accumulators in TMEM, no global traffic at all.
//   KIND 0: kind::f16, FP16 x FP16 -> FP32, N = 256, K = 16  (the mixed path's main and cross terms)
//   KIND 1: kind::i8,  S8 x S8 -> S32,      N = 80,  K = 32  (the emulated-FP64 path's digit products)
// The issuer works in batches of TCP_BATCH MMAs, commits each batch to one of two mbarriers and waits for the batch
// before it: one batch is always in flight, so the tensor pipe never drains.  Thread 0 of the leader reports the
// SM clocks and the nanoseconds the loop took (out[2*cluster], out[2*cluster+1]) -- the SM clock under that load.
constexpr int TCP_THREADS = 128, TCP_BATCH = 32;

template <int KIND>
__global__ void __launch_bounds__(TCP_THREADS, 1)
tc_peak_kernel(int batches, unsigned long long* __restrict__ out) {
    constexpr int N = KIND == 0 ? 256 : 80;
    __shared__ alignas(1024) uint8_t tiles[2 * 128 * 128];     // [M side: 128 rows][N side: N/2 rows], 128-byte rows
    __shared__ uint64_t bar[2];
    __shared__ uint32_t tmem_slot;
    const int warp = threadIdx.x >> 5;
    const int rank = (int)cluster_ctarank();
    for (int e = threadIdx.x; e < (int)sizeof(tiles) / 4; e += TCP_THREADS) {    // operand bits that toggle like data
        uint32_t x = (uint32_t)(e + 1) * 2654435761u + blockIdx.x * 40503u;
        x ^= x >> 15; x *= 2246822519u; x ^= x >> 13;
        if (KIND == 0) x = (x & 0x83FF83FFu) | 0x38003800u;                      // two FP16 of magnitude [0.5, 1)
        reinterpret_cast<uint32_t*>(tiles)[e] = x;
    }
    fence_proxy_async();                                    // the tensor core reads shared memory through the async proxy
    if (threadIdx.x == 0) { mbar_init(&bar[0], 1); mbar_init(&bar[1], 1); fence_barrier_init(); }
    if (warp == 1) { tmem_alloc_pair(&tmem_slot, 512); tmem_relinquish_pair(); }
    tc_fence_before_sync();
    __syncthreads();
    cluster_sync_all();
    tc_fence_after_sync();
    const uint32_t tmem_base = tmem_slot;
    if (warp == 0 && rank == 0) {
        const bool issuer = elect_one();
        const uint32_t idesc = KIND == 0 ? umma_idesc_f16_m256(N, 0, 0) : umma_idesc_s8_m256(N);
        const uint32_t a = umma_desc_lo(smem_u32(tiles)), b = umma_desc_lo(smem_u32(tiles) + 128 * 128);
        unsigned long long c0 = 0, t0 = 0;
        if (threadIdx.x == 0) {
            c0 = clock64();
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
        }
        for (int bt = 0; bt < batches; ++bt) {
            if (issuer) {
#pragma unroll
                for (int m = 0; m < TCP_BATCH / 4; ++m) {
                    const uint32_t tacc = tmem_base + (m & 1) * 256;        // two accumulators, alternating
#pragma unroll
                    for (int k = 0; k < 4; ++k)                             // four K steps of 32 bytes per 128-byte row
                        if (KIND == 0) umma_f16_pair(tacc, a + 2 * k, b + 2 * k, idesc, (m < 2 && k == 0) ? 0u : 1u);
                        else umma_i8_pair(tacc, a + 2 * k, b + 2 * k, idesc, (m < 2 && k == 0) ? 0u : 1u);
                }
                umma_commit_pair(&bar[bt & 1]);
            }
            __syncwarp();
            if (bt >= 1) mbar_wait(&bar[(bt - 1) & 1], ((bt - 1) >> 1) & 1);
        }
        if (batches > 0) mbar_wait(&bar[(batches - 1) & 1], ((batches - 1) >> 1) & 1);
        tc_fence_after_sync();
        if (threadIdx.x == 0) {
            unsigned long long t1;
            const unsigned long long c1 = clock64();
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
            out[2 * (blockIdx.x / 2)] = c1 - c0;
            out[2 * (blockIdx.x / 2) + 1] = t1 - t0;
        }
    }
    tc_fence_before_sync();
    __syncthreads();
    cluster_sync_all();
    if (warp == 1) {
        tc_fence_after_sync();
        tmem_dealloc_pair(tmem_base, 512);
    }
}

}  // namespace tb
