// gemm_f16split.cuh -- mixed-precision contraction kernel (S2+S3 of DESIGN.md): TMA -> swizzled smem -> tcgen05.mma
// (cta_group::2, kind::f16) with short FP32 accumulation chains in TMEM and the running sum in registers.
//
// The paper's mixed precision runs "only the construction of the triples amplitudes" through
// sgemm.  B200 has no FP32 tensor path; an FP32-class product is recovered from a split of every operand x
// (Q13):   h = RN_fp16(x), l = RN_fp16(x - h),   x*y ~= h*h' + (h*l' + l*h').
// FP16 has the 11-bit significand of TF32 at twice the MMA rate; its narrow exponent range is handled by ONE power
// of two per tensor class (prepare.cuh scales_kernel: the largest |x| of the integrals / of t2 lands in
// [2^13, 2^14)), so every term of a contraction carries the same factor 2^(sg+st), removed exactly in the epilogue.
// h*h' is exact (11 x 11 bit products, FP32 accumulation); l <= 2^-12 |x| and its own FP16 rounding leaves 2^-23 |x|
// for elements within 2^-2 of the tensor maximum after scaling, an absolute 2^-25 * 2^-s below that (subnormal l)
// -- i.e. a 39-bit fixed-point floor relative to the tensor's largest element; the dropped l*l' is 2^-24.
// 6 MMAs (K = 16) per 32-wide K chunk where 3xTF32 needs 12.
//
// Same "G job" (p,q,r) as gemm_f64.cuh, computed TRANSPOSED so that the long flattened (b,c) index is the MMA's
// M dimension (128 TMEM lanes per CTA, no padding waste for any v) and the virtual index a is its N dimension:
//
//   G(p,q,r)[a,(b,c)] = sum_d XK_r [(b,c),d] T2A[p,q][a,d]  + sum_d XKT_q[(b,c),d] T2A[p,r][a,d]     (Eq. (2.2.2))
//                     + sum_l T2K_q[(b,c),l] OtA[r,p][a,l]  + sum_l T2KT_r[(b,c),l] OtA[q,p][a,l]
//
// Operands are K-major arrays that prepare.cuh already wrote SPLIT: per operand row and 32-wide K chunk one 128-byte
// row holding 32 FP16 of h (bytes 0..63) and 32 FP16 of l (bytes 64..127) -- 4 bytes per element, the same as one
// FP32 word, so nothing is gained by splitting inside the SM (round 1 did, with six converter warps; they and the
// shared-memory round trip of every tile are gone).  XK[s][b][c][d] = (db|cr) for the slice in cache slot s,
// XKT[s][b][c][d] = XK[s][c][b][d], T2A[p][q][a][d] = t2, OtA[r][p][a][l] = -(pa|lr), T2K[q][b][c][l] = t2[q,l,b,c],
// T2KT[r][b][c][l] = t2[l,r,b,c]; the c index has vp rows per b (row v is zero when v is odd) so that U keeps the
// pitch the reduction expects.  TMA (SWIZZLE_128B) stages the packed rows; they are the only thing the MMAs read.
//
// The kernel is persistent and runs as CTA PAIRS (thread-block clusters of 2 = the two SMs of a TPC, cta_group::2):
// a pair walks work items (job, two consecutive m-tiles of 128 (b,c) rows, n-tile of BN a-columns) as ONE
// 256 x BN MMA tile.  Each CTA stages only its own 128 M-side rows and HALF of the N-side rows (the tensor cores
// read the other half from the peer's shared memory); both CTAs' TMA loads complete on the LEADER's full barrier.
// Jobs of a launch are grouped by (q,r) so that the big XK_r / XKT_q slices come from HBM once per group
// (grouped_item, gemm_f64.cuh).
//   warp 0     : TMA producer   (K chunks of 32 = one 128-byte swizzled row per operand row, ring of FS_STAGES tiles)
//   warp 1     : MMA issuer     (one lane of the LEADER CTA; per K chunk 2+2 cross-term MMAs, then 2 main-term MMAs,
//                                all FP16 K = 16; tcgen05.commit multicasts to both CTAs' barriers)
//   warp 2     : allocates TMEM (512 columns = two 128 x 256 FP32 buffers in each CTA)
//   warps 4-11 : accumulators   (tcgen05.ld of every finished chain, packed FP32 round-to-nearest adds (FADD2) in
//                                registers, one 256-bit store per (b,c) row and a-tile of U at the end of the item)
//
// Why the running sum lives in registers and not in TMEM: the tensor core adds each MMA's result to its accumulator
// with truncation, so one long accumulation chain is biased towards zero by ~(number of MMAs) * 2^-25 (measured:
// -3.4e-6 relative on W at v = 240 for one chain over the whole K, i.e. 7e-6 on E(T), growing with v).  A TMEM buffer
// therefore only ever holds a short chain (FS_CHAIN K chunks, started with accumulate = 0, cross terms before the main
// term of each chunk); finished chains are added with FADD.RN by the accumulator warps while the tensor core fills
// the other buffer.  Chain length is set by the TMEM read port: a 128 x BN FP32 read-out costs 8*BN clk at the
// measured 64 B/clk (B300_MICROARCH.md "TMEM"), a chunk's six MMAs 3*BN clk, so chains shorter than 3 chunks leave
// the tensor pipe waiting for the read-out (round 1 ran 2).
#pragma once
#include <cuda_fp16.h>

#include "gemm_f64.cuh"   // GemmJob
#include "ptx.cuh"
#include "ulayout.cuh"

namespace tb {

struct alignas(64) SplitMaps {
    CUtensorMap xk;    // (word, n=(b,c'), slot)   box (32, 128, 1)    M side, virtual segment 1
    CUtensorMap xkt;   // (word, n, slot)          box (32, 128, 1)    M side, virtual segment 2
    CUtensorMap t2k;   // (word, n, q)             box (32, 128, 1)    M side, occupied segment 3
    CUtensorMap t2kt;  // (word, n, r)             box (32, 128, 1)    M side, occupied segment 4
    CUtensorMap t2a;   // (word, a, p*o+q)         box (32, BN/2, 1)   N side, virtual segments
    CUtensorMap ota;   // (word, a, r*o+p)         box (32, BN/2, 1)   N side, occupied segments
};

constexpr int FS_BM = 128;            // (b,c) rows per CTA tile = TMEM lanes
constexpr int FS_BK = 32;             // K elements per chunk = 4-byte words per packed row (32 h | 32 l FP16)
constexpr int FS_THREADS = 384;       // 4 service warps (TMA, MMA, TMEM allocator, idle) + 8 accumulator warps
constexpr int FS_ACC_WARP0 = 4;       // first accumulator warp (a multiple of 4: warp % 4 = its TMEM lane quarter)
constexpr int FS_CHAIN = 4;           // K chunks per TMEM accumulation chain
constexpr int FS_TMEM_COLS = 512;
constexpr int FS_SMEM_LIMIT = 227 * 1024;
constexpr int FS_MAX_JOBS = 192;        // jobs per launch (3 per triplet, plan.h: at most 4^3 triplets per batch); the
                                        // job table is copied to shared memory once (item -> job look-ups sit on the
                                        // critical path of every role, two dependent global loads each otherwise)
constexpr int FS_TAIL_BYTES = 2048 + FS_MAX_JOBS * 48;   // alignment slack + barriers, job table

// npad = N-side rows a CTA stages = bn / 2.  One shared-memory ring of (128 + npad)-row tiles with 128-byte rows.
__host__ __device__ constexpr int fs_tile_bytes(int npad) { return (FS_BM + npad) * 128; }
// as many stages as fit (at most 8); the request is always > half an SM's shared memory: exactly one CTA per SM
__host__ __device__ constexpr int fs_stages(int npad) {
    int s = (FS_SMEM_LIMIT - FS_TAIL_BYTES) / fs_tile_bytes(npad);
    return s > 8 ? 8 : s;
}
__host__ __device__ constexpr int fs_smem_bytes(int npad) {
    const int need = fs_stages(npad) * fs_tile_bytes(npad) + FS_TAIL_BYTES;
    return need > 120 * 1024 ? need : 120 * 1024;
}

__global__ void __launch_bounds__(FS_THREADS, 1)
gemm_f16split_kernel(const __grid_constant__ SplitMaps maps, const GemmJob* __restrict__ gjobs, int njobs, int v, int vp,
                     int o, int mtiles, int ntiles, int bn, int npad, const float* __restrict__ scales) {
    constexpr int cs = 2;   // CTAs per MMA tile
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    const int S = fs_stages(npad);
    const int tile_bytes = fs_tile_bytes(npad);
    uint8_t* smem_tail = smem + S * tile_bytes;
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_tail);   // [8] both CTAs' tiles landed (the LEADER's is used)
    uint64_t* empty = full + 8;                  // [8] tile consumed by the MMAs (per CTA, multicast commit)
    uint64_t* tfull = empty + 8;                 // accumulator buffer ready for the read-out
    uint64_t* tempty = tfull + 2;                // accumulator buffer drained (the LEADER's is used)
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty + 2);
    GemmJob* jobs = reinterpret_cast<GemmJob*>(smem_tail + 256);
    for (int e = threadIdx.x; e < njobs * (int)(sizeof(GemmJob) / 4); e += FS_THREADS)
        reinterpret_cast<uint32_t*>(jobs)[e] = reinterpret_cast<const uint32_t*>(gjobs)[e];

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nrows = v * vp;                                   // flattened (b,c') rows
    // a pair (cs = 2) walks two consecutive m-tiles of one (job, n-tile) as one 256-row MMA tile
    const int rank = (int)cluster_ctarank();
    const int cid = blockIdx.x / cs, ncl = gridDim.x / cs;
    const int per_job = ((mtiles + cs - 1) / cs) * ntiles;
    const long long nitems = (long long)njobs * per_job;
    const int nch_v = (v + FS_BK - 1) / FS_BK, nch_o = (o + FS_BK - 1) / FS_BK;
    const int nch = 2 * (nch_v + nch_o);

    if (threadIdx.x == 0) {
        // full / tempty are waited on by the leader's MMA thread only
        for (int s = 0; s < S; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
        for (int b = 0; b < 2; ++b) { mbar_init(&tfull[b], 1); mbar_init(&tempty[b], 8 * cs); }
        fence_barrier_init();
    }
    if (warp == 2) { tmem_alloc_pair(tmem_slot, FS_TMEM_COLS); tmem_relinquish_pair(); }
    tc_fence_before_sync();
    __syncthreads();
    cluster_sync_all();                 // every CTA's barriers are initialised before a peer's TMA / commit reaches them
    tc_fence_after_sync();
    const uint32_t tmem_base = *tmem_slot;

    if (warp < FS_ACC_WARP0) reg_dealloc<56>();
    if (warp == 0) {
        // ------------------------------------------------------------------------------------ TMA producer
        if (lane == 0) {
            tma_prefetch_desc(&maps.xk); tma_prefetch_desc(&maps.xkt); tma_prefetch_desc(&maps.t2k);
            tma_prefetch_desc(&maps.t2kt); tma_prefetch_desc(&maps.t2a); tma_prefetch_desc(&maps.ota);
            const uint32_t lfull0 = mapa_u32(smem_u32(&full[0]), 0);     // the leader's full barriers
            uint32_t it = 0;
            for (long long w = cid; w < nitems; w += ncl) {
                int jb, rem;
                grouped_item(jobs, w, per_job, jb, rem);
                const int m0 = ((rem / ntiles) * cs + rank) * FS_BM;
                const int an = (rem % ntiles) * bn + rank * npad;   // this CTA's half of the N-side rows
                const GemmJob job = jobs[jb];
                const int p = job.p, q = job.q, r = job.r;
                for (int c = 0; c < nch; ++c, ++it) {
                    const int s = it % S;
                    mbar_wait(&empty[s], ((it / S) & 1) ^ 1);
                    uint8_t* sM = smem + s * tile_bytes;            // packed rows: [M 128 rows][N npad rows]
                    uint8_t* sN = sM + FS_BM * 128;
                    // the leader announces both CTAs' bytes; the peer's copies complete on the leader's barrier too
                    if (rank == 0) mbar_arrive_expect_tx(&full[s], 2 * (FS_BM + npad) * 128);
                    const CUtensorMap *mm, *nm;
                    int kk, mz, nz;
                    if (c < nch_v)                     { kk = c * FS_BK;                       mm = &maps.xk;   mz = job.xr; nm = &maps.t2a; nz = p * o + q; }
                    else if (c < 2 * nch_v)            { kk = (c - nch_v) * FS_BK;             mm = &maps.xkt;  mz = job.xq; nm = &maps.t2a; nz = p * o + r; }
                    else if (c < 2 * nch_v + nch_o)    { kk = (c - 2 * nch_v) * FS_BK;         mm = &maps.t2k;  mz = q;      nm = &maps.ota; nz = r * o + p; }
                    else                               { kk = (c - 2 * nch_v - nch_o) * FS_BK; mm = &maps.t2kt; mz = r;      nm = &maps.ota; nz = q * o + p; }
                    tma_load_3d_pair(sM, mm, lfull0 + 8u * s, kk, m0, mz);
                    tma_load_3d_pair(sN, nm, lfull0 + 8u * s, kk, an, nz);
                }
            }
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------------------------------ MMA issuer
        // The WHOLE warp of the leader CTA walks the loop (convergent, so descriptors and loop state stay in uniform
        // registers); one elected lane issues.  With a lone thread in a divergent branch the compiler moved every
        // descriptor through ELECT + R2UR.BROADCAST -- ~26 dependent instructions per MMA, more than the 120 clk an
        // MMA takes: the issue thread, not the tensor pipe, set the pace (ncu: pipe 44 % active, no role waiting).
        if (rank == 0) {
            const bool issuer = elect_one();
            const uint32_t idesc = umma_idesc_f16_m256((uint32_t)bn, 0, 0);   // FP16 x FP16 -> FP32
            const uint32_t smem_base = smem_u32(smem);
            uint32_t it = 0, chain = 0;
            for (long long w = cid; w < nitems; w += ncl) {
                for (int c = 0; c < nch; ++c, ++it) {
                    const int s = it % S;
                    int left;   // K elements of this chunk's segment from the chunk start
                    if (c < nch_v) left = v - c * FS_BK;
                    else if (c < 2 * nch_v) left = v - (c - nch_v) * FS_BK;
                    else if (c < 2 * nch_v + nch_o) left = o - (c - 2 * nch_v) * FS_BK;
                    else left = o - (c - 2 * nch_v - nch_o) * FS_BK;
                    const bool two = left > 16;                           // K steps of 16 that carry data: 2 or 1
                    const uint32_t buf = chain & 1;
                    const bool first = (c % FS_CHAIN) == 0, last = (c % FS_CHAIN) == FS_CHAIN - 1 || c == nch - 1;
                    if (first) mbar_wait(&tempty[buf], ((chain >> 1) & 1) ^ 1);
                    mbar_wait(&full[s], (it / S) & 1);
                    tc_fence_after_sync();
                    if (issuer) {
                        const uint32_t tacc = tmem_base + buf * 256;
                        // low descriptor words of the packed M / N tiles; bytes 0..63 of a row = 32 FP16 of h,
                        // 64..127 = 32 FP16 of l; one K step = 32 bytes = 2 units of 16 bytes
                        const uint32_t m = umma_desc_lo(smem_base + s * tile_bytes);
                        const uint32_t n = umma_desc_lo(smem_base + s * tile_bytes + FS_BM * 128);
                        // cross terms l*h' + h*l' first (small), then the main term h*h'
                        umma_f16_pair(tacc, m + 4, n, idesc, first ? 0u : 1u);
                        umma_f16_pair(tacc, m, n + 4, idesc, 1u);
                        if (two) {
                            umma_f16_pair(tacc, m + 6, n + 2, idesc, 1u);
                            umma_f16_pair(tacc, m + 2, n + 6, idesc, 1u);
                        }
                        umma_f16_pair(tacc, m, n, idesc, 1u);
                        if (two) umma_f16_pair(tacc, m + 2, n + 2, idesc, 1u);
                        umma_commit_pair(&empty[s]);                       // both CTAs' ring slots
                        if (last) umma_commit_pair(&tfull[buf]);           // both CTAs' accumulator warps
                    }
                    __syncwarp();
                    if (last) ++chain;
                }
            }
        }
    } else if (warp >= FS_ACC_WARP0) {
        // ------------------------------------------------------------------------------------ accumulator warps
        reg_alloc<216>();   // 128*56 + 256*216 <= 384*168 registers
        const int wq = warp & 3;                            // TMEM lane quarter this warp may read
        const int half = (warp - FS_ACC_WARP0) >> 2;        // columns [128*half, 128*half + 128)
        const int nchain = (nch + FS_CHAIN - 1) / FS_CHAIN;
        const bool active = half * 128 < bn;
        const uint32_t ltempty0 = mapa_u32(smem_u32(&tempty[0]), 0);
        uint32_t chain = 0;
        for (long long w = cid; w < nitems; w += ncl) {
            int jb, rem;
            grouped_item(jobs, w, per_job, jb, rem);
            const int m0 = ((rem / ntiles) * cs + rank) * FS_BM, a0 = (rem % ntiles) * bn;
            uint64_t acc2[64];          // 128 FP32 running sums as 64 register pairs (packed add.rn.f32x2)
#pragma unroll
            for (int j = 0; j < 64; ++j) acc2[j] = 0ull;
            for (int ch = 0; ch < nchain; ++ch, ++chain) {
                const uint32_t buf = chain & 1;
                mbar_wait(&tfull[buf], (chain >> 1) & 1);
                tc_fence_after_sync();
                if (active) {
                    const uint32_t taddr = tmem_base + buf * 256 + half * 128 + ((uint32_t)(wq * 32) << 16);
#pragma unroll
                    for (int c0 = 0; c0 < 128; c0 += 16) {
                        uint32_t rg[16];
                        tmem_ld_32x32b_x16(taddr + c0, rg);
                        tmem_ld_wait();
#pragma unroll
                        for (int j = 0; j < 8; ++j) acc2[c0 / 2 + j] = fadd2_rn(acc2[c0 / 2 + j], rg[2 * j], rg[2 * j + 1]);
                    }
                }
                tc_fence_before_sync();
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(ltempty0 + 8u * buf);   // the leader's MMA thread owns both CTAs' buffers
            }
            // blocked + swizzled store (ulayout.cuh): this thread owns (y,z) = (b,c) = row, the columns are x = a.
            // The 8 a-values of a tile sit in one aligned 32-byte chunk at word (x ^ m), m = (z1 << 1) | (y0 << 2).
            const int row = m0 + wq * 32 + lane;
            const int bb = row / vp, cc = row - bb * vp;
            if (active && row < nrows && cc < v) {
                float* __restrict__ out = static_cast<float*>(jobs[jb].out);
                float* __restrict__ out2 = static_cast<float*>(jobs[jb].out2);
                const int nt = u_tiles(v);
                const float unscale = scales[2];             // 2^-(sg+st): exact
                const int sw = u_swz<4>(0, bb & 7, cc & 7);
                const bool s4 = (sw & 4) != 0, s2 = (sw & 2) != 0;
                const size_t astride = (size_t)nt * nt * UCHUNK;   // one a-tile
                const size_t cb = (size_t)((a0 + half * 128) >> 3) * astride +
                                  ((size_t)(bb >> 3) * nt + (cc >> 3)) * UCHUNK + (sw & ~7);
                const int acols = min(bn, v - a0) - half * 128;    // columns of this thread that exist
#pragma unroll
                for (int t = 0; t < 16; ++t) {
                    if (8 * t < acols) {
                        float acc[8], u[8], w8[8];        // the tile's 8 columns, unpacked
#pragma unroll
                        for (int j = 0; j < 4; ++j) unpack_f32x2(acc2[4 * t + j], acc[2 * j], acc[2 * j + 1]);
#pragma unroll
                        for (int j = 0; j < 8; ++j) acc[j] *= unscale;
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            u[j] = s4 ? acc[j + 4] : acc[j];
                            u[j + 4] = s4 ? acc[j] : acc[j + 4];
                        }
#pragma unroll
                        for (int j = 0; j < 8; ++j) w8[j] = s2 ? u[j ^ 2] : u[j];
                        stg_v8(out + cb + (size_t)t * astride, w8);        // one whole 32-byte sector per lane
                        if (out2) stg_v8(out2 + cb + (size_t)t * astride, w8);
                    }
                }
            }
        }
    }
    tc_fence_before_sync();
    __syncthreads();
    cluster_sync_all();                 // no CTA leaves while a peer may still write its shared memory or barriers
    if (warp == 2) {
        tc_fence_after_sync();
        tmem_dealloc_pair(tmem_base, FS_TMEM_COLS);
    }
}

}  // namespace tb
