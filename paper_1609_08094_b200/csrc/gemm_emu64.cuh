// gemm_emu64.cuh -- emulated-FP64 contraction kernel: the W build of Eq. (2.2.2)-(2.2.3)
// to FP64-class accuracy on the INTEGER tensor cores (tcgen05.mma kind::i8, cta_group::2), a third
// point of the paper's precision / throughput study (L125, L156-L158) beside the DMMA path (gemm_f64.cuh, pinned at
// the 37 TFLOP/s FP64 tensor peak) and the FP16-split path (gemm_f16split.cuh).
//
// Ozaki-style error-free slicing with ONE power-of-two scale per tensor class (as on the mixed path): every operand
// is the 47-bit fixed-point integer xi = rint(x 2^(s+32)) = sum_i d_i 256^(5-i), six balanced base-256 digits
// d_i in [-128, 127] (prepare.cuh pack_emu_store).  Then
//     sum_k xi_k yi_k = sum_{i,j} 256^(10-i-j) S_ij,   S_ij = sum_k d_i(x_k) d_j(y_k)   (an exact s8 x s8 -> s32 GEMM)
// and the pairs of one LEVEL L = i + j share a weight, so they accumulate in ONE int32 TMEM accumulator: (L+1) K 128^2
// < 2^31 for K <= 21000.  Levels L <= 5 are kept (21 digit products per 32 K elements).  What is dropped: for the x
// digit i the y digits below 5-i, i.e. y rounded to nearest (balanced digits) at the unit of its digit 5-i -- per term
// d_i 256^(5-i) * (<= 0.5 * 256^i) <= 2^46, against products of up to 2^92: ~2^-50 of (class maximum)^2 per term,
// below the 2^-46 quantisation of the operands themselves.  Integer accumulation is exact, so -- unlike the
// FP16-split kernel -- a whole work item (all four K segments) accumulates in TMEM and is read out once:
// S_L -> double, W = sum_L S_L c_L with the exact powers of two c_L = 2^(8(10-L) - (sg+st) - 64); six FMAs per
// element, rounding ~1e-16.  Measured: W within 1e-13 of the oracle on the scale of W.  (Earlier digit choices, same
// cost per product: 7 digits base 128, levels <= 6, 28 products, BN = 64: 73 TFLOP/s, W within 1e-12; 6 digits base
// 128, levels <= 5: W only within 1e-10 -- the amplitudes' dynamic range eats the 7-bit digits.)
//
// Same G job, tiling and roles as gemm_f16split.cuh (transposed: the (b,c) index is the MMA's M dimension, CTA pairs,
// 128 TMEM lanes per CTA), with BN = 80 a-columns per tile: six level accumulators of 80 columns = 480 of the 512
// TMEM columns.  K is walked in chunks of 64: per operand row three 128-byte rows of digit pairs (prepare.cuh), staged
// by TMA with SWIZZLE_128B; an MMA (K = 32) reads digit i of the M side and digit j of the N side for one half of the
// chunk through descriptors advanced by 64 bytes per digit and 32 bytes per half.  Output: the FP64 U buffers of
// ulayout.cuh, reduced by reduce_kernel<double>.
#pragma once
#include "gemm_f64.cuh"   // GemmJob, grouped_item
#include "ptx.cuh"
#include "ulayout.cuh"

namespace tb {

struct alignas(64) EmuMaps {
    CUtensorMap xk, xkt, t2k, t2kt;   // M side: (word, n = (b,c'), slot | q | r)      box (32, 128, 1)
    CUtensorMap t2a, ota;             // N side: (word, a, p*o+q | r*o+p)              box (32, 40, 1)
};

constexpr int EM_BM = 128;            // (b,c) rows per CTA tile = TMEM lanes
// a-columns per tile: template parameter BN in {80, 64, 48} (six level accumulators x BN <= 512 TMEM columns; plan.h
// picks the one that wastes the least MMA time on padded columns, charging the smaller tiles their extra feed)
constexpr int EM_DIGITS = 6;
constexpr int EM_LEVELS = 6;          // levels 0..5 kept
constexpr int EM_BK = 64;             // K elements per chunk
constexpr int EM_CW = 96;             // 4-byte words per operand row and K chunk (three 128-byte rows of digit pairs)
constexpr int EM_ROWS = 3;
constexpr int EM_THREADS = 384;
constexpr int EM_ACC_WARP0 = 4;
constexpr int EM_TMEM_COLS = 512;
constexpr int EM_STAGES = 3;
__host__ __device__ constexpr int em_tile_bytes(int bn) { return EM_ROWS * (EM_BM + bn / 2) * 128; }   // [M row 0..2][N row 0..2]
constexpr int EM_MAX_JOBS = 192;
constexpr int EM_TAIL_BYTES = 2048 + EM_MAX_JOBS * 48;
__host__ __device__ constexpr int em_smem_bytes(int bn) { return EM_STAGES * em_tile_bytes(bn) + EM_TAIL_BYTES; }

template <int EM_BN>
__global__ void __launch_bounds__(EM_THREADS, 1)
gemm_emu64_kernel(const __grid_constant__ EmuMaps maps, const GemmJob* __restrict__ gjobs, int njobs, int v, int vp, int o,
                  int mtiles, int ntiles, const float* __restrict__ scales) {
    constexpr int cs = 2;
    constexpr int EM_NPAD = EM_BN / 2;                     // N-side rows a CTA stages
    constexpr int EM_TILE_BYTES = em_tile_bytes(EM_BN);
    static_assert(EM_LEVELS * EM_BN <= EM_TMEM_COLS && EM_NPAD % 8 == 0, "level accumulators fit TMEM; whole swizzle atoms");
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* smem_tail = smem + EM_STAGES * EM_TILE_BYTES;
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_tail);   // [8] both CTAs' tiles landed (the LEADER's is used)
    uint64_t* empty = full + 8;                  // [8] tile consumed by the MMAs (per CTA, multicast commit)
    uint64_t* tfull = empty + 8;                 // the item's accumulators are complete
    uint64_t* tempty = tfull + 2;                // the accumulators are drained (the LEADER's is used)
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty + 2);
    GemmJob* jobs = reinterpret_cast<GemmJob*>(smem_tail + 256);
    for (int e = threadIdx.x; e < njobs * (int)(sizeof(GemmJob) / 4); e += EM_THREADS)
        reinterpret_cast<uint32_t*>(jobs)[e] = reinterpret_cast<const uint32_t*>(gjobs)[e];

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nrows = v * vp;
    const int rank = (int)cluster_ctarank();
    const int cid = blockIdx.x / cs, ncl = gridDim.x / cs;
    const int per_job = ((mtiles + cs - 1) / cs) * ntiles;
    const long long nitems = (long long)njobs * per_job;
    const int nch_v = (v + EM_BK - 1) / EM_BK, nch_o = (o + EM_BK - 1) / EM_BK;
    const int nch = 2 * (nch_v + nch_o);

    if (threadIdx.x == 0) {
        for (int s = 0; s < EM_STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
        mbar_init(&tfull[0], 1);
        mbar_init(&tempty[0], 8 * cs);
        fence_barrier_init();
    }
    if (warp == 2) { tmem_alloc_pair(tmem_slot, EM_TMEM_COLS); tmem_relinquish_pair(); }
    tc_fence_before_sync();
    __syncthreads();
    cluster_sync_all();
    tc_fence_after_sync();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        // ------------------------------------------------------------------------------------ TMA producer
        if (lane == 0) {
            tma_prefetch_desc(&maps.xk); tma_prefetch_desc(&maps.xkt); tma_prefetch_desc(&maps.t2k);
            tma_prefetch_desc(&maps.t2kt); tma_prefetch_desc(&maps.t2a); tma_prefetch_desc(&maps.ota);
            const uint32_t lfull0 = mapa_u32(smem_u32(&full[0]), 0);
            uint32_t it = 0;
            for (long long w = cid; w < nitems; w += ncl) {
                int jb, rem;
                grouped_item(jobs, w, per_job, jb, rem);
                const int m0 = ((rem / ntiles) * cs + rank) * EM_BM;
                const int an = (rem % ntiles) * EM_BN + rank * EM_NPAD;
                const GemmJob job = jobs[jb];
                const int p = job.p, q = job.q, r = job.r;
                for (int c = 0; c < nch; ++c, ++it) {
                    const int s = it % EM_STAGES;
                    mbar_wait(&empty[s], ((it / EM_STAGES) & 1) ^ 1);
                    uint8_t* sM = smem + s * EM_TILE_BYTES;
                    uint8_t* sN = sM + EM_ROWS * EM_BM * 128;
                    if (rank == 0) mbar_arrive_expect_tx(&full[s], 2 * EM_TILE_BYTES);
                    const CUtensorMap *mm, *nm;
                    int kk, mz, nz;
                    if (c < nch_v)                     { kk = c * EM_CW;                       mm = &maps.xk;   mz = job.xr; nm = &maps.t2a; nz = p * o + q; }
                    else if (c < 2 * nch_v)            { kk = (c - nch_v) * EM_CW;             mm = &maps.xkt;  mz = job.xq; nm = &maps.t2a; nz = p * o + r; }
                    else if (c < 2 * nch_v + nch_o)    { kk = (c - 2 * nch_v) * EM_CW;         mm = &maps.t2k;  mz = q;      nm = &maps.ota; nz = r * o + p; }
                    else                               { kk = (c - 2 * nch_v - nch_o) * EM_CW; mm = &maps.t2kt; mz = r;      nm = &maps.ota; nz = q * o + p; }
                    const uint32_t bar = lfull0 + 8u * s;
#pragma unroll
                    for (int pr = 0; pr < EM_ROWS; ++pr) {
                        tma_load_3d_pair(sM + pr * EM_BM * 128, mm, bar, kk + 32 * pr, m0, mz);
                        tma_load_3d_pair(sN + pr * EM_NPAD * 128, nm, bar, kk + 32 * pr, an, nz);
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------------------------------ MMA issuer
        if (rank == 0) {      // the whole warp walks the loop (uniform registers), one elected lane issues
            const bool issuer = elect_one();
            const uint32_t idesc = umma_idesc_s8_m256(EM_BN);
            const uint32_t smem_base = smem_u32(smem);
            uint32_t it = 0, item = 0;
            for (long long w = cid; w < nitems; w += ncl, ++item) {
                mbar_wait(&tempty[0], (item & 1) ^ 1);          // the previous item's accumulators are drained
                tc_fence_after_sync();
                for (int c = 0; c < nch; ++c, ++it) {
                    const int s = it % EM_STAGES;
                    mbar_wait(&full[s], (it / EM_STAGES) & 1);
                    tc_fence_after_sync();
                    int left;   // K elements of this chunk's segment from the chunk start
                    if (c < nch_v) left = v - c * EM_BK;
                    else if (c < 2 * nch_v) left = v - (c - nch_v) * EM_BK;
                    else if (c < 2 * nch_v + nch_o) left = o - (c - 2 * nch_v) * EM_BK;
                    else left = o - (c - 2 * nch_v - nch_o) * EM_BK;
                    const bool two = left > 32;                    // the second half of the chunk carries data
                    if (issuer) {
                        const uint32_t t0 = smem_base + s * EM_TILE_BYTES;
                        uint32_t md[EM_ROWS], nd[EM_ROWS];
#pragma unroll
                        for (int pr = 0; pr < EM_ROWS; ++pr) {
                            md[pr] = umma_desc_lo(t0 + pr * EM_BM * 128);
                            nd[pr] = umma_desc_lo(t0 + EM_ROWS * EM_BM * 128 + pr * EM_NPAD * 128);
                        }
                        const uint32_t fresh = c == 0 ? 0u : 1u;
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            if (h == 0 || two) {
#pragma unroll
                                for (int i = 0; i < EM_DIGITS; ++i) {
                                    const uint32_t ad = md[i >> 1] + 4 * (i & 1) + 2 * h;   // 64 B per digit, 32 B per half
#pragma unroll
                                    for (int j = 0; i + j < EM_LEVELS; ++j) {
                                        const uint32_t bd = nd[j >> 1] + 4 * (j & 1) + 2 * h;
                                        // level L = i + j; its first product of the item (i = 0, first half of chunk 0)
                                        // overwrites the accumulator
                                        umma_i8_pair(tmem_base + (uint32_t)(i + j) * EM_BN, ad, bd, idesc,
                                                     (i == 0 && h == 0) ? fresh : 1u);
                                    }
                                }
                            }
                        }
                        umma_commit_pair(&empty[s]);
                        if (c == nch - 1) umma_commit_pair(&tfull[0]);
                    }
                    __syncwarp();
                }
            }
        }
    } else if (warp >= EM_ACC_WARP0) {
        // ------------------------------------------------------------------------------------ accumulator warps
        const int wq = warp & 3;                            // TMEM lane quarter this warp may read
        constexpr int HC = EM_BN / 2;                       // columns per warp
        const int half = (warp - EM_ACC_WARP0) >> 2;        // columns [40*half, 40*half + 40) of every level
        const uint32_t ltempty = mapa_u32(smem_u32(&tempty[0]), 0);
        const int sexp = reinterpret_cast<const int*>(scales)[12] + reinterpret_cast<const int*>(scales)[13] + 64;
        uint32_t item = 0;
        for (long long w = cid; w < nitems; w += ncl, ++item) {
            int jb, rem;
            grouped_item(jobs, w, per_job, jb, rem);
            const int m0 = ((rem / ntiles) * cs + rank) * EM_BM, a0 = (rem % ntiles) * EM_BN + half * HC;
            double acc[HC];
#pragma unroll
            for (int j = 0; j < HC; ++j) acc[j] = 0.0;
            mbar_wait(&tfull[0], item & 1);
            tc_fence_after_sync();
            // Read-out, software-pipelined: five segments of 8 columns per level; the tcgen05.ld of segment s+1 is in
            // flight while segment s is converted, so the TMEM read port (64 B/clk), not the conversions, sets the
            // length of the serial section.  int32 -> double without the XU pipe: the bits 0x43300000'80000000 ^ x
            // are the double 2^52 + 2^31 + x (exact), one DADD removes the offset, one DFMA applies the level weight.
            {
                const uint32_t tlane = tmem_base + half * HC + ((uint32_t)(wq * 32) << 16);
                constexpr int NSEG = EM_LEVELS * (HC / 8);
                uint32_t rg[2][8];
                tmem_ld_32x32b_x8(tlane, rg[0]);
#pragma unroll
                for (int sgm = 0; sgm < NSEG; ++sgm) {
                    const int L = sgm / (HC / 8), c0 = (sgm % (HC / 8)) * 8;
                    tmem_ld_wait();
                    if (sgm + 1 < NSEG) {
                        const int Ln = (sgm + 1) / (HC / 8), cn = ((sgm + 1) % (HC / 8)) * 8;
                        tmem_ld_32x32b_x8(tlane + (uint32_t)Ln * EM_BN + cn, rg[(sgm + 1) & 1]);
                    }
                    const double cL = ldexp(1.0, 8 * (10 - L) - sexp);       // exact power of two
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        const double dv = __hiloint2double(0x43300000, (int)(rg[sgm & 1][j] ^ 0x80000000u)) - 4503601774854144.0;
                        acc[c0 + j] = fma(dv, cL, acc[c0 + j]);
                    }
                }
            }
            tc_fence_before_sync();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(ltempty);     // the leader's MMA thread may overwrite the accumulators
            // blocked + swizzled FP64 store (ulayout.cuh): this thread owns (y,z) = (b,c) = row, the columns are x = a
            const int row = m0 + wq * 32 + lane;
            const int bb = row / vp, cc = row - bb * vp;
            if (row < nrows && cc < v) {
                double* __restrict__ out = static_cast<double*>(jobs[jb].out);
                double* __restrict__ out2 = static_cast<double*>(jobs[jb].out2);
                const int nt = u_tiles(v);
                const size_t astride = (size_t)nt * nt * UCHUNK;   // one a-tile
                const size_t cb = ((size_t)(bb >> 3) * nt + (cc >> 3)) * UCHUNK + u_swz<8>(0, bb & 7, cc & 7);
#pragma unroll
                for (int j = 0; j < HC; ++j) {
                    if (a0 + j < v) {
                        const size_t off = (size_t)((a0 + j) >> 3) * astride + (cb ^ (size_t)u_swz<8>(j & 7, 0, 0));
                        out[off] = acc[j];
                        if (out2) out2[off] = acc[j];
                    }
                }
            }
        }
    }
    tc_fence_before_sync();
    __syncthreads();
    cluster_sync_all();
    if (warp == 2) {
        tc_fence_after_sync();
        tmem_dealloc_pair(tmem_base, EM_TMEM_COLS);
    }
}

}  // namespace tb
