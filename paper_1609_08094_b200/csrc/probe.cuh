// probe.cuh -- FP64 tensor-core (mma.sync.m8n8k4.f64, SASS DMMA) peak of the device the library runs on: the roofline
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

}  // namespace tb
