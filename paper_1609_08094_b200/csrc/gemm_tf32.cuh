// gemm_tf32.cuh -- mixed-precision contraction kernel (S2+S3 of DESIGN.md): TMA -> swizzled smem -> in-SM operand
// split -> tcgen05.mma (cta_group::2, kind::f16) with short FP32 accumulation chains in TMEM and the running sum in
// registers.  (The file keeps its first name: the first version ran 3xTF32.)
//
// The paper's mixed precision runs "only the construction of the triples amplitudes" through
// sgemm.  B200 has no FP32 tensor path; an FP32-class product is recovered from a split of every operand x
// (Q13):   h = RN_fp16(x), l = RN_fp16(x - h),   x*y ~= h*h' + (h*l' + l*h').
// FP16 has the 11-bit significand of TF32 at twice the MMA rate; its narrow exponent range is handled by ONE power
// of two per tensor class (prepare.cuh scales_kernel: the largest |x| of the integrals / of t2 lands in
// [2^13, 2^14)), so every term of a contraction carries the same factor 2^(sg+st), removed exactly in the epilogue.
// h*h' is exact (11 x 11 bit products, FP32 accumulation); l <= 2^-12 |x| (x - h is exact in FP32) and its own
// FP16 rounding leaves 2^-23 |x| for elements within 2^-2 of the tensor maximum after scaling, an absolute
// 2^-25 * 2^-s below that (subnormal l) -- i.e. a 39-bit fixed-point floor relative to the tensor's largest
// element; the dropped l*l' is 2^-24.  6 MMAs (K = 16) per 32-wide K chunk where 3xTF32 needs 12.
// Measured on B200: W within 3e-7 of the FP64 oracle on the scale of W, E(T) within 4e-7 (chain bias, below).
//
// Same "G job" (p,q,r) as gemm_f64.cuh, computed TRANSPOSED so that the long flattened (b,c) index is the MMA's
// M dimension (128 TMEM lanes per CTA, no padding waste for any v) and the virtual index a is its N dimension:
//
//   G(p,q,r)[a,(b,c)] = sum_d XK_r [(b,c),d] T2A[p,q][a,d]  + sum_d XKT_q[(b,c),d] T2A[p,r][a,d]     (Eq. (2.2.2))
//                     + sum_l T2K_q[(b,c),l] OtA[r,p][a,l]  + sum_l T2KT_r[(b,c),l] OtA[q,p][a,l]
//
// Operands are K-major arrays of scaled FP32 values, 4 bytes per element (prepare.cuh): XK[r][b][c][d] = (db|cr),
// XKT[r][b][c][d] = XK[r][c][b][d], T2A[p][q][a][d] = t2, OtA[r][p][a][l] = -(pa|lr), T2K[q][b][c][l] = t2[q,l,b,c],
// T2KT[r][b][c][l] = t2[l,r,b,c]; the c index has vp rows per b (row v is zero when v is odd) so that U keeps the
// pitch the reduction expects.  TMA stages raw FP32 tiles; converter warps write, per 32-wide K chunk, a packed tile
// whose 128-byte rows hold 32 FP16 of h (bytes 0..63) and 32 FP16 of l (bytes 64..127) -- the only thing the MMAs
// read.  Splitting inside the SM halves the operand bytes in HBM and through L2 (with separate hi/lo arrays the loop
// was bound by the ~42 B/clk/SM L2 -> SM cap, not by the tensor pipe).
//
// The kernel is persistent and runs as CTA PAIRS (thread-block clusters of 2 = the two SMs of a TPC, cta_group::2):
// a pair walks work items (job, two consecutive m-tiles of 128 (b,c) rows, n-tile of BN a-columns) as ONE
// 256 x BN MMA tile.  Each CTA stages only its own 128 M-side rows and HALF of the N-side rows (the tensor cores
// read the other half from the peer's shared memory).  Jobs of a launch are grouped by (q,r) so that the big
// XK_r / XKT_q slices come from HBM once per group (grouped_item, gemm_f64.cuh).
//   warp 0    : TMA producer   (K chunks of 32 words = one 128-byte swizzled row per operand row, ring of 4 raw tiles)
//   warp 1    : MMA issuer     (one lane of the LEADER CTA; per K chunk 2+2 cross-term MMAs, then 2 main-term MMAs,
//                               all FP16 K = 16; tcgen05.commit multicasts to both CTAs' barriers)
//   warps 2-7 : converters     (raw tile -> packed tile, ring of 2; warp 2 also allocates TMEM: 512 columns =
//                               two 128 x 256 FP32 buffers in each CTA)
//   warps 8-15: accumulators   (tcgen05.ld of every finished chain, packed FP32 round-to-nearest adds (FADD2) in
//                               registers, one 256-bit store per (b,c) row and a-tile of U at the end of the item)
//
// Why the running sum lives in registers and not in TMEM: the tensor core adds each MMA's result to its accumulator
// with truncation, so one long accumulation chain is biased towards zero by ~(number of MMAs) * 2^-25 (measured:
// -3.4e-6 relative on W at v = 240, i.e. 7e-6 on E(T), growing with v).  A TMEM buffer therefore only ever holds a
// short chain (TF_CHAIN = 2 K chunks = 12 MMAs, started with accumulate = 0, cross terms before the main term of
// each chunk); finished chains are added with FADD.RN by the accumulator warps while the tensor core fills the
// other buffer.  Measured bias on E(T): ~2e-7 with one chunk per chain, 3e-7..5e-7 with two (8 % faster: every chain
// costs a 128 x BN TMEM read-out and the kernel runs at the 1 kW power cap); tolerance 1e-5.
#pragma once
#include <cuda_fp16.h>

#include "gemm_f64.cuh"   // GemmJob
#include "ptx.cuh"
#include "ulayout.cuh"

namespace tb {

struct alignas(64) Tf32Maps {
    CUtensorMap xk;    // (d, n=(b,c'), r)      box (32, 128, 1)    M side, virtual segment 1
    CUtensorMap xkt;   // (d, n, r)             box (32, 128, 1)    M side, virtual segment 2
    CUtensorMap t2k;   // (l, n, q)             box (32, 128, 1)    M side, occupied segment 3
    CUtensorMap t2kt;  // (l, n, r)             box (32, 128, 1)    M side, occupied segment 4
    CUtensorMap t2a;   // (d, a, p*o+q)         box (32, BN/2, 1)   N side, virtual segments
    CUtensorMap ota;   // (l, a, r*o+p)         box (32, BN/2, 1)   N side, occupied segments
};

constexpr int TF_BM = 128;            // (b,c) rows per CTA tile = TMEM lanes
constexpr int TF_BK = 32;             // floats per K chunk (128-byte rows)
constexpr int TF_THREADS = 512;         // 8 service warps (TMA, MMA, 6 converters) + 8 accumulator warps
constexpr int TF_CONV_WARPS = 6;        // warps 2..7
constexpr int TF_CHAIN = 2;             // K chunks per TMEM accumulation chain
constexpr int TF_TMEM_COLS = 512;
constexpr int TF_SMEM_LIMIT = 227 * 1024;
constexpr int TF_MAX_JOBS = 192;        // jobs per launch (3 per triplet, plan.h: at most 4^3 triplets per batch); the
                                        // job table is copied to shared memory once (item -> job look-ups sit on the
                                        // critical path of every role, two dependent global loads each otherwise)
constexpr int TF_TAIL_BYTES = 2048 + TF_MAX_JOBS * 48;   // alignment slack + barriers, job table

// npad = N-side rows a CTA stages = bn / 2.  Two shared-memory rings of (128 + npad)-row tiles with 128-byte rows:
// TF_RAW_STAGES raw FP32 tiles (TMA destination, read by the converter warps only; deep enough to cover the L2/HBM
// latency) and TF_PK_STAGES packed FP16 tiles (h | l; written by the converter warps, read by the MMAs; the conversion
// of later chunks overlaps the MMAs of chunk c).
constexpr int TF_RAW_STAGES = 4, TF_PK_STAGES = 2;
__host__ __device__ constexpr int tf32_tile_bytes(int npad) { return (TF_BM + npad) * 128; }
// the request is always > half an SM's shared memory: exactly one CTA per SM (it owns all 512 TMEM columns)
__host__ __device__ constexpr int tf32_smem_bytes(int npad) {
    return (TF_RAW_STAGES + TF_PK_STAGES) * tf32_tile_bytes(npad) + TF_TAIL_BYTES;
}

__global__ void __launch_bounds__(TF_THREADS, 1)
gemm_tf32_kernel(const __grid_constant__ Tf32Maps maps, const GemmJob* __restrict__ gjobs, int njobs, int v, int vp,
                 int o, int mtiles, int ntiles, int bn, int npad, const float* __restrict__ scales) {
    constexpr int cs = 2;   // CTAs per MMA tile
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    constexpr int RS = TF_RAW_STAGES, PS = TF_PK_STAGES;
    const int tile_bytes = tf32_tile_bytes(npad);
    uint8_t* smem_pk = smem + RS * tile_bytes;
    uint8_t* smem_tail = smem_pk + PS * tile_bytes;
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_tail);   // [RS] raw tile landed (per CTA)
    uint64_t* empty = full + RS;                 // [RS] raw tile read by this CTA's converter warps
    uint64_t* conv = empty + RS;                 // [PS] packed tile written by both CTAs' converters (leader's is used)
    uint64_t* pkempty = conv + PS;               // [PS] packed tile consumed by the MMAs
    uint64_t* tfull = pkempty + PS;              // accumulator buffer ready for the epilogue
    uint64_t* tempty = tfull + 2;                // accumulator buffer drained
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty + 2);
    GemmJob* jobs = reinterpret_cast<GemmJob*>(smem_tail + 256);
    for (int e = threadIdx.x; e < njobs * (int)(sizeof(GemmJob) / 4); e += TF_THREADS)
        reinterpret_cast<uint32_t*>(jobs)[e] = reinterpret_cast<const uint32_t*>(gjobs)[e];

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nrows = v * vp;                                   // flattened (b,c') rows
    // a pair (cs = 2) walks two consecutive m-tiles of one (job, n-tile) as one 256-row MMA tile
    const int rank = (int)cluster_ctarank();
    const int cid = blockIdx.x / cs, ncl = gridDim.x / cs;
    const int per_job = ((mtiles + cs - 1) / cs) * ntiles;
    const long long nitems = (long long)njobs * per_job;
    const int kst_v = (v + 7) >> 3, kst_o = (o + 7) >> 3;       // 8-wide k-steps per segment
    const int nch_v = (v + TF_BK - 1) / TF_BK, nch_o = (o + TF_BK - 1) / TF_BK;
    const int nch = 2 * (nch_v + nch_o);

    if (threadIdx.x == 0) {
        // conv / tempty are waited on by the leader's MMA thread only: both CTAs' converter / accumulator warps arrive
        for (int s = 0; s < RS; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], TF_CONV_WARPS); }
        for (int s = 0; s < PS; ++s) { mbar_init(&conv[s], TF_CONV_WARPS * cs); mbar_init(&pkempty[s], 1); }
        for (int b = 0; b < 2; ++b) { mbar_init(&tfull[b], 1); mbar_init(&tempty[b], 8 * cs); }
        fence_barrier_init();
    }
    if (warp == 2) { tmem_alloc_pair(tmem_slot, TF_TMEM_COLS); tmem_relinquish_pair(); }
    tc_fence_before_sync();
    __syncthreads();
    cluster_sync_all();                 // every CTA's barriers are initialised before a peer's TMA / commit reaches them
    tc_fence_after_sync();
    const uint32_t tmem_base = *tmem_slot;

    if (warp < 8) reg_dealloc<48>();
    if (warp == 0) {
        // ------------------------------------------------------------------------------------ TMA producer
        if (lane == 0) {
            tma_prefetch_desc(&maps.xk); tma_prefetch_desc(&maps.xkt); tma_prefetch_desc(&maps.t2k);
            tma_prefetch_desc(&maps.t2kt); tma_prefetch_desc(&maps.t2a); tma_prefetch_desc(&maps.ota);
            uint32_t it = 0;
            for (long long w = cid; w < nitems; w += ncl) {
                int jb, rem;
                grouped_item(jobs, w, per_job, jb, rem);
                const int m0 = ((rem / ntiles) * cs + rank) * TF_BM;
                const int an = (rem % ntiles) * bn + rank * npad;   // this CTA's half of the N-side rows
                const GemmJob job = jobs[jb];
                const int p = job.p, q = job.q, r = job.r;
                for (int c = 0; c < nch; ++c, ++it) {
                    const int s = it % RS;
                    mbar_wait(&empty[s], ((it / RS) & 1) ^ 1);
                    uint8_t* sM = smem + s * tile_bytes;            // raw FP32 words: [M 128 rows][N npad rows]
                    uint8_t* sN = sM + TF_BM * 128;
                    mbar_arrive_expect_tx(&full[s], (TF_BM + npad) * 128);
                    const CUtensorMap *mm, *nm;
                    int kk, mz, nz;
                    if (c < nch_v)                     { kk = c * TF_BK;                       mm = &maps.xk;   mz = r; nm = &maps.t2a; nz = p * o + q; }
                    else if (c < 2 * nch_v)            { kk = (c - nch_v) * TF_BK;             mm = &maps.xkt;  mz = q; nm = &maps.t2a; nz = p * o + r; }
                    else if (c < 2 * nch_v + nch_o)    { kk = (c - 2 * nch_v) * TF_BK;         mm = &maps.t2k;  mz = q; nm = &maps.ota; nz = r * o + p; }
                    else                               { kk = (c - 2 * nch_v - nch_o) * TF_BK; mm = &maps.t2kt; mz = r; nm = &maps.ota; nz = q * o + p; }
                    tma_load_3d(sM, mm, &full[s], kk, m0, mz);
                    tma_load_3d(sN, nm, &full[s], kk, an, nz);
                }
            }
        }
    } else if (warp >= 2 && warp < 8) {
        // ------------------------------------------------------------------------------------ converters
        // Operand split inside the SM (Q13): the staged word is the FP32 bit pattern of x plus 0x1000, which
        // the TF32 MMA reads as h = RN_tf32(x) (it ignores the low 13 bits).  These warps turn every 8 consecutive k of
        // a row into 8 BF16 of h (packed bytes 0..63 of the row) and 8 BF16 of l = x - h (bytes 64..127), honouring the
        // 128-byte swizzle of both tiles (16-byte unit u of row R sits at unit u ^ (R & 7)).
        const int ct = threadIdx.x - 64;
        const int rows = TF_BM + npad;
        const uint32_t smem_base = smem_u32(smem);
        const uint32_t lconv0 = mapa_u32(smem_u32(&conv[0]), 0);
        uint32_t it = 0;
        for (long long w = cid; w < nitems; w += ncl) {
            for (int c = 0; c < nch; ++c, ++it) {
                const int s = it % RS, ps = it % PS;
                mbar_wait(&pkempty[ps], ((it / PS) & 1) ^ 1);
                mbar_wait(&full[s], (it / RS) & 1);
                const uint32_t raw = smem_base + s * tile_bytes, pk = smem_base + (RS + ps) * tile_bytes;
                for (int task = ct; task < rows * 4; task += 32 * TF_CONV_WARPS) {
                    const int m = (task >> 3) & 3, R = (task & 7) | ((task >> 5) << 3);   // 8 lanes: one m, 8 rows
                    const uint32_t rb = (uint32_t)R * 128u, sw = (uint32_t)(R & 7);
                    uint32_t x[8];
                    lds_v4(raw + rb + (((2 * m) ^ sw) << 4), x[0], x[1], x[2], x[3]);
                    lds_v4(raw + rb + (((2 * m + 1) ^ sw) << 4), x[4], x[5], x[6], x[7]);
                    // h = RN_fp16(x) (11-bit significand), l = RN_fp16(x - h); packed row: 32 FP16 of h | 32 FP16 of l
                    // (kind::f16 wants A and B of one type: a BF16 x FP16 descriptor traps as an illegal instruction)
                    uint32_t hp[4], lp[4];
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const float x0 = __uint_as_float(x[2 * j]), x1 = __uint_as_float(x[2 * j + 1]);
                        const __half2 h2 = __floats2half2_rn(x0, x1);
                        const float2 hf = __half22float2(h2);
                        hp[j] = *reinterpret_cast<const uint32_t*>(&h2);
                        const __half2 l2 = __floats2half2_rn(x0 - hf.x, x1 - hf.y);
                        lp[j] = *reinterpret_cast<const uint32_t*>(&l2);
                    }
                    sts_v4(pk + rb + (((uint32_t)m ^ sw) << 4), hp[0], hp[1], hp[2], hp[3]);
                    sts_v4(pk + rb + (((uint32_t)(4 + m) ^ sw) << 4), lp[0], lp[1], lp[2], lp[3]);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[s]);       // raw tile read: the producer may refill it
                fence_proxy_async();          // generic-proxy writes -> visible to the tensor core's (async proxy) reads
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster_release(lconv0 + 8u * ps);
            }
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------------------------------ MMA issuer
        if (lane == 0 && rank == 0) {
            const uint32_t idesc = umma_idesc_f16_m256((uint32_t)bn, 0, 0);   // FP16 x FP16 -> FP32
            const uint32_t smem_base = smem_u32(smem);
            uint32_t it = 0, chain = 0;
            for (long long w = cid; w < nitems; w += ncl) {
                for (int c = 0; c < nch; ++c, ++it) {
                    const int ps = it % PS;
                    int left;   // k-steps of this chunk that carry data
                    if (c < nch_v) left = kst_v - c * 4;
                    else if (c < 2 * nch_v) left = kst_v - (c - nch_v) * 4;
                    else if (c < 2 * nch_v + nch_o) left = kst_o - (c - 2 * nch_v) * 4;
                    else left = kst_o - (c - 2 * nch_v - nch_o) * 4;
                    const int nk = left < 4 ? left : 4;
                    const uint32_t buf = chain & 1;
                    const bool first = (c % TF_CHAIN) == 0, last = (c % TF_CHAIN) == TF_CHAIN - 1 || c == nch - 1;
                    if (first) {
                        mbar_wait(&tempty[buf], ((chain >> 1) & 1) ^ 1);
                        tc_fence_after_sync();
                    }
                    mbar_wait(&conv[ps], (it / PS) & 1);
                    tc_fence_after_sync();
                    const uint32_t tacc = tmem_base + buf * 256;
                    const uint32_t pM = smem_base + (RS + ps) * tile_bytes, pN = pM + TF_BM * 128;      // packed tiles
                    const uint64_t ml = umma_desc_sw128(pM), nl = umma_desc_sw128(pN);
                    uint32_t acc = first ? 0u : 1u;
                    // packed row: bytes 0..63 = 32 FP16 of h, 64..127 = 32 FP16 of l; K = 16 per MMA.  Cross terms
                    // l*h' + h*l' first (small), then the main term h*h'
                    const int nk16 = (nk + 1) >> 1;
                    for (int k = 0; k < nk16; ++k) {
                        const uint64_t adv = (uint64_t)(k * 2);          // 32 bytes per k-step, in 16-byte units
                        umma_f16_pair(tacc, ml + 4 + adv, nl + adv, idesc, acc);   // l * h'
                        acc = 1;
                        umma_f16_pair(tacc, ml + adv, nl + 4 + adv, idesc, 1);     // h * l'
                    }
                    for (int k = 0; k < nk16; ++k) {
                        const uint64_t adv = (uint64_t)(k * 2);
                        umma_f16_pair(tacc, ml + adv, nl + adv, idesc, 1);         // h * h'
                    }
                    umma_commit_pair(&pkempty[ps]);                    // both CTAs' packed slots
                    if (last) { umma_commit_pair(&tfull[buf]); ++chain; }   // both CTAs' accumulator warps
                }
            }
        }
    } else if (warp >= 8) {
        // ------------------------------------------------------------------------------------ accumulator warps
        reg_alloc<208>();   // 256*48 + 256*208 = 64K registers
        const int wq = warp & 3;                 // TMEM lane quarter this warp may read
        const int half = (warp - 8) >> 2;        // columns [128*half, 128*half + 128)
        const int nchain = (nch + TF_CHAIN - 1) / TF_CHAIN;
        const bool active = half * 128 < bn;
        uint32_t chain = 0;
        for (long long w = cid; w < nitems; w += ncl) {
            int jb, rem;
            grouped_item(jobs, w, per_job, jb, rem);
            const int m0 = ((rem / ntiles) * cs + rank) * TF_BM, a0 = (rem % ntiles) * bn;
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
                if (lane == 0) {     // the leader's MMA thread owns the buffer hand-back of both CTAs
                    mbar_arrive_cluster(mapa_u32(smem_u32(&tempty[buf]), 0));
                }
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
                        float acc[8], u[8], w[8];        // the tile's 8 columns, unpacked
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
                        for (int j = 0; j < 8; ++j) w[j] = s2 ? u[j ^ 2] : u[j];
                        stg_v8(out + cb + (size_t)t * astride, w);        // one whole 32-byte sector per lane
                        if (out2) stg_v8(out2 + cb + (size_t)t * astride, w);
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
        tmem_dealloc_pair(tmem_base, TF_TMEM_COLS);
    }
}

}  // namespace tb
