// ri_slices.cuh -- RI-direct source of the (vv|vo) slices: the vvvo tensor is never
// materialised; a slice is rebuilt on the device from the RI factors whenever a batch needs it and the cache
// (plan.h build_slices) does not hold it.
//
//   (db|cr) = sum_Q B[Q,d,b] B[Q,c,r]                      (Eq. (2.1.3), applied to the (T) integrals)
//   X_r[(d,b)][c] = sum_Q Bt[(d,b)][Q] Bo[r][Q][c]         one FP64 GEMM per slice: M = v^2, N = v, K = naux
//
// Bt[(d,b)][Q] = B[Q][o+d][o+b] (K-major rows, pitch nauxp) and Bo[r][Q][c] = B[Q][o+c][r] (c-pitch vp) are repacked
// once per call.  Same DMMA tile code as the contraction kernel (gemm_f64.cuh DmmaWarp): TMA -> swizzled shared
// memory -> mma.sync.m8n8k4.f64, persistent, one CTA per SM.  Output: the natural-order slot X[slot][d][b][c]
// (c-pitch vp, pad column zero); XT and the mixed path's packed copies follow from the per-slice repack kernels.
#pragma once
#include "gemm_f64.cuh"

namespace tb {

struct alignas(64) RiMaps {
    CUtensorMap bt;   // (Q, row = (d,b))       box (16, BM)
    CUtensorMap bo;   // (c, Q, r)              box (16, 16, 1)
};

// Bt[(d,b)][Q] = B[Q][o+d][o+b]: tiled transpose of the [naux][v*v] virtual-virtual block
__global__ void __launch_bounds__(256)
ri_pack_bt_kernel(const double* __restrict__ B, int o, int v, int naux, int nauxp, double* __restrict__ Bt) {
    __shared__ double tile[32][33];
    const int n = o + v;
    const long long R = (long long)v * v;
    const long long r0 = (long long)blockIdx.x * 32;
    const int q0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int qq = ty; qq < 32; qq += 8) {
        const long long row = r0 + tx;
        if (q0 + qq < naux && row < R) {
            const int d = (int)(row / v), b = (int)(row % v);
            tile[qq][tx] = B[((size_t)(q0 + qq) * n + o + d) * n + o + b];
        }
    }
    __syncthreads();
    for (int rr = ty; rr < 32; rr += 8) {
        const long long row = r0 + rr;
        if (row < R && q0 + tx < nauxp) Bt[(size_t)row * nauxp + q0 + tx] = q0 + tx < naux ? tile[tx][rr] : 0.0;
    }
}

// Bo[r][Q][c] = B[Q][o+c][r]
__global__ void __launch_bounds__(256)
ri_pack_bo_kernel(const double* __restrict__ B, int o, int v, int naux, int vp, double* __restrict__ Bo) {
    const int n = o + v;
    const size_t total = (size_t)o * naux * vp;
    for (size_t e = blockIdx.x * (size_t)blockDim.x + threadIdx.x; e < total; e += (size_t)gridDim.x * blockDim.x) {
        const int c = (int)(e % vp);
        const int Q = (int)((e / vp) % naux);
        const int r = (int)(e / ((size_t)vp * naux));
        Bo[e] = c < v ? B[((size_t)Q * n + o + c) * n + r] : 0.0;
    }
}

// Mixed path: a bound on the largest |(ab|cr)| for the power-of-two operand scale (prepare.cuh scales_kernel) without
// building the tensor: Cauchy-Schwarz over the auxiliary index, |(ab|cr)| <= |B[:,a,b]|_2 |B[:,c,r]|_2.
// out[0] / out[1] = float bits of the largest column norm of the virtual-virtual / virtual-occupied block.
__global__ void __launch_bounds__(256)
ri_bound_kernel(const double* __restrict__ B, int o, int v, int naux, float* __restrict__ out) {
    const int n = o + v;
    const size_t nvv = (size_t)v * v, total = nvv + (size_t)v * o;
    float mvv = 0.0f, mvo = 0.0f;
    for (size_t e = blockIdx.x * (size_t)blockDim.x + threadIdx.x; e < total; e += (size_t)gridDim.x * blockDim.x) {
        const bool vv = e < nvv;
        const size_t f = vv ? e : e - nvv;
        const int p = o + (int)(vv ? f / v : f / o), q = vv ? o + (int)(f % v) : (int)(f % o);
        double s = 0.0;
        for (int Q = 0; Q < naux; ++Q) { const double x = B[((size_t)Q * n + p) * n + q]; s += x * x; }
        const float nrm = (float)sqrt(s) * 1.000001f;      // rounded up
        if (vv) mvv = fmaxf(mvv, nrm); else mvo = fmaxf(mvo, nrm);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        mvv = fmaxf(mvv, __shfl_xor_sync(0xffffffffu, mvv, off));
        mvo = fmaxf(mvo, __shfl_xor_sync(0xffffffffu, mvo, off));
    }
    if ((threadIdx.x & 31) == 0) {
        atomicMax(reinterpret_cast<unsigned int*>(out), __float_as_uint(mvv));
        atomicMax(reinterpret_cast<unsigned int*>(out) + 1, __float_as_uint(mvo));
    }
}
__global__ void ri_bound_fold_kernel(const float* __restrict__ norms, unsigned int* __restrict__ maxbits) {
    if (threadIdx.x == 0 && blockIdx.x == 0) atomicMax(maxbits, __float_as_uint(norms[0] * norms[1]));
}

// loads[n] = {r, slot}: build X_r into slot `slot` of X.
template <int WM, int WN, int NT, int STAGES>
__global__ void __launch_bounds__(GemmF64Cfg<WM, WN, NT, STAGES>::THREADS, 1)
ri_slice_kernel(const __grid_constant__ RiMaps maps, const int2* __restrict__ loads, int nloads, int v, int vp, int naux,
                int mtiles, int ntiles, double* __restrict__ X, size_t slot_elems) {
    using C = GemmF64Cfg<WM, WN, NT, STAGES>;
    constexpr int MT = C::MT;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint64_t* full = reinterpret_cast<uint64_t*>(smem + STAGES * C::STAGE_BYTES);
    uint64_t* empty = full + STAGES;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int per_slice = mtiles * ntiles;
    const long long nitems = (long long)nloads * per_slice;
    const int nch = (naux + 15) >> 4;
    const long long rows = (long long)v * v;

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], C::NCW); }
        fence_barrier_init();
    }
    __syncthreads();

    if (warp == C::NCW) {
        if (lane == 0) {
            tma_prefetch_desc(&maps.bt); tma_prefetch_desc(&maps.bo);
            uint32_t it = 0;
            for (long long w = blockIdx.x; w < nitems; w += gridDim.x) {
                const int ld = (int)(w / per_slice), tile = (int)(w % per_slice);
                const int m0 = (tile / ntiles) * C::BM, n0 = (tile % ntiles) * C::BN;
                const int r = loads[ld].x;
                for (int c = 0; c < nch; ++c, ++it) {
                    const int s = it % STAGES;
                    mbar_wait(&empty[s], ((it / STAGES) & 1) ^ 1);
                    uint8_t* sA = smem + s * C::STAGE_BYTES;
                    uint8_t* sB = sA + C::A_BYTES;
                    mbar_arrive_expect_tx(&full[s], C::STAGE_BYTES);
                    tma_load_3d(sA, &maps.bt, &full[s], c * 16, m0, 0);
                    for (int bx = 0; bx < C::BN / 16; ++bx)
                        tma_load_3d(sB + bx * 2048, &maps.bo, &full[s], n0 + bx * 16, c * 16, r);
                }
            }
        }
        return;
    }

    DmmaWarp<WM, WN, NT> dw;
    dw.init(warp, lane);
    const uint32_t smem_base = smem_u32(smem);
    uint32_t it = 0;
    for (long long w = blockIdx.x; w < nitems; w += gridDim.x) {
        const int ld = (int)(w / per_slice), tile = (int)(w % per_slice);
        const int m0 = (tile / ntiles) * C::BM, n0 = (tile % ntiles) * C::BN;
        double acc[MT][NT][2];
#pragma unroll
        for (int i = 0; i < MT; ++i)
#pragma unroll
            for (int j = 0; j < NT; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
        for (int c = 0; c < nch; ++c, ++it) {
            const int s = it % STAGES;
            const int rem = naux - c * 16;
            const int nu = rem >= 16 ? 4 : ((rem + 3) >> 2);
            mbar_wait(&full[s], (it / STAGES) & 1);
            const uint32_t sA = smem_base + s * C::STAGE_BYTES;
            dw.chunk(acc, sA, sA + C::A_BYTES, nu);
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[s]);
        }
        double* __restrict__ out = X + (size_t)loads[ld].y * slot_elems;
#pragma unroll
        for (int j = 0; j < NT; ++j) {
            const int col = n0 + dw.col(j);          // even; (col, col + 1) is one 16-byte word (vp is even)
            if (col < vp) {
#pragma unroll
                for (int i = 0; i < MT; ++i) {
                    const long long row = m0 + dw.row(i);
                    if (row < rows)
                        *reinterpret_cast<double2*>(out + (size_t)row * vp + col) = make_double2(acc[i][j][0], acc[i][j][1]);
                }
            }
        }
    }
}

}  // namespace tb
