// gemm_f64.cuh -- FP64 contraction kernel (S2+S3 of DESIGN.md): TMA -> swizzled smem -> DMMA.
//
// One launch runs a batch of "G jobs".  A job (p,q,r) is the K-concatenated GEMM
//
//   G(p,q,r)[a,(b,c)] = Y_pqr[a,b,c] + Y_prq[a,c,b]                       (two of the six images of
//                                                                          Eq. (2.2.3))
//     = sum_d t2[p,q,a,d] X_r[d,b,c] + sum_d t2[p,r,a,d] XT_q[d,b,c]      (virtual index, Eq. (2.2.2))
//     - sum_l O_pr[a,l] t2[q,l,b,c]  - sum_l O_pq[a,l] t2[l,r,b,c]        (occupied index)
//
// with X_r[d,b,c] = (db|cr) = vvvo[d,b,c,r], XT_r[d,b,c] = X_r[d,c,b], O_pr[a,l] = (pa|lr) = ovoo[p,a,l,r]
// (Ot holds -O).  M = v (rows a), N = v*vp (flat (b,c), c-pitch vp), K = 2v + 2o in four segments.
// W^abc = G(i,j,k)[a,b,c] + G(j,i,k)[b,a,c] + G(k,i,j)[c,a,b] is assembled by the reduction kernel.
//
// Tiling: CTA tile BM x BN = (40*WM) x (8*NT*WN); WM*WN compute warps, each a (5 x NT) grid of m8n8k4 DMMAs,
// plus one TMA producer warp.  K is walked in chunks of 16 (one 128-byte swizzled smem row per operand row):
//   A tile  [BM][16] doubles  (one TMA box, SWIZZLE_128B)
//   B tile  BN/16 boxes of [16 k][16 n] doubles (SWIZZLE_128B)
// Bank-conflict-free fragment reads (8-byte LDS, 16 lanes per phase) need a row permutation of the MMA's M index
// (rho) and a column permutation of its N index (nu); see DESIGN.md "contraction kernel".
#pragma once
#include "ptx.cuh"
#include "ulayout.cuh"

namespace tb {

struct GemmJob {
    int p, q, r;
    int gstart;  // jobs of a batch are sorted by (q,r); [gstart, gstart + gsize) = the jobs sharing this job's (q,r),
    void* out;   // G(p,q,r)[a][b][c] in the blocked layout of ulayout.cuh: slot base + u * UBLK
    void* out2;  // second destination (or null): a triplet with i=j or j=k uses the same G twice
    int gsize;   // i.e. the same X_r / XT_q operand slices: walked tile by tile together
    int xr, xq;  // slots of the slice cache that hold X_r and XT_q (resident run: xr = r, xq = q)
    int pad;
};
static_assert(sizeof(GemmJob) == 48, "plan.h sizes the job table with 48 bytes per job");

struct alignas(64) GemmMaps {
    CUtensorMap t2a;   // t2 as A: (d, a, pq)          box (16, BM, 1)
    CUtensorMap ota;   // -ovoo as A: (l, a, r*o+p)    box (16, BM, 1)
    CUtensorMap x;     // X:  (n, d, slot)             box (16, 16, 1)
    CUtensorMap xt;    // XT: (n, d, slot)             box (16, 16, 1)
    CUtensorMap t2bq;  // t2 as B, rows l at fixed outer index: (n, y, x) box (16, 16, 1)
    CUtensorMap t2br;  // t2 as B, rows l at fixed inner index: (n, y, x) box (16, 1, 16)
};

// Work item w -> (job, tile).  The jobs of a launch are sorted by (q,r) (triples_b200.cu); the gsize jobs of a group
// share their M-side operand slices XK_r / XKT_q / T2K_q / T2KT_r, so consecutive items are the SAME tile of the
// group's jobs: the CTAs running side by side then pull identical M-side rows, and the (vv|vo) slices come from HBM
// once per group instead of once per job (they are far larger than L2: 2 x v^3 x 8 bytes per job).
__device__ __forceinline__ void grouped_item(const GemmJob* __restrict__ jobs, long long w, int per_job, int& jb, int& rem) {
    const int any = (int)(w / per_job);                       // some job of the group item w falls in
    const int gs = jobs[any].gstart, gn = jobs[any].gsize;
    const long long local = w - (long long)gs * per_job;
    jb = gs + (int)(local % gn);
    rem = (int)(local / gn);
}

__host__ __device__ constexpr int rho_row(int g) { return 2 * (g & 3) + (g >> 2); }                 // MMA row -> tile row
__host__ __device__ constexpr int nu_col(int g) { return (g & 1) | (((g >> 2) & 1) << 1) | (((g >> 1) & 1) << 3); }

template <int WM, int WN, int NT, int STAGES>
struct GemmF64Cfg {
    static constexpr int MT = 5;
    static constexpr int BM = WM * MT * 8;
    static constexpr int BN = WN * NT * 8;
    static constexpr int NCW = WM * WN;               // compute warps
    static constexpr int THREADS = (NCW + 1) * 32;    // + producer warp
    static constexpr int A_BYTES = BM * 128;
    static constexpr int B_BYTES = BN * 128;
    static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
    static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 2 * STAGES * 8 + 1024;  // + barriers + align slack
    static_assert(NT % 2 == 0, "BN must be a multiple of 16 per warp");
    static_assert(A_BYTES % 1024 == 0 && B_BYTES % 1024 == 0, "swizzle atoms are 1 KiB");
};

// Fragment addressing and the per-chunk DMMA loop of one compute warp (shared by the contraction kernel below and the
// RI slice builder of ri_slices.cuh).  acc[i][j] = 8x8 accumulator tile (i: 5 row tiles, j: NT column tiles).
template <int WM, int WN, int NT>
struct DmmaWarp {
    static constexpr int MT = 5;
    uint32_t offA[4], offB[2][2];
    int rg, t, wm, wn;
    __device__ __forceinline__ void init(int warp, int lane) {
        const int g = lane >> 2;
        t = lane & 3;
        wm = warp % WM; wn = warp / WM;
        rg = rho_row(g);
        const int nug = nu_col(g);
        // A element (row m, k): byte = m*128 + (((k>>1) ^ (m&7)) << 4) + (k&1)*8, with k = 4u + t
#pragma unroll
        for (int u = 0; u < 4; ++u)
            offA[u] = (wm * MT * 8 + rg) * 128 + ((((2 * u + (t >> 1)) ^ rg) & 7) << 4) + (t & 1) * 8;
        // B element (k, n): box n>>4, byte = k*128 + ((((n&15)>>1) ^ (k&7)) << 4) + (n&1)*8, n&15 = nu(g) + 4*(nt&1)
#pragma unroll
        for (int ntp = 0; ntp < 2; ++ntp)
#pragma unroll
            for (int up = 0; up < 2; ++up)
                offB[ntp][up] = (wn * (NT / 2)) * 2048 + t * 128 + (((((nug >> 1) + 2 * ntp) ^ (4 * up + t)) & 7) << 4) +
                                (nug & 1) * 8;
    }
    // one staged K chunk of 16: nu = number of k4 steps that carry data
    __device__ __forceinline__ void chunk(double (&acc)[MT][NT][2], uint32_t sA, uint32_t sB, int nu) const {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (u < nu) {
                double a[MT], b[NT];
#pragma unroll
                for (int i = 0; i < MT; ++i) a[i] = lds_f64(sA + offA[u] + i * 8 * 128);
#pragma unroll
                for (int j = 0; j < NT; ++j) b[j] = lds_f64(sB + offB[j & 1][u & 1] + (j >> 1) * 2048 + u * 512);
#pragma unroll
                for (int i = 0; i < MT; ++i)
#pragma unroll
                    for (int j = 0; j < NT; ++j) dmma_884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
            }
        }
    }
    // output coordinates of acc[i][j][0..1]: row (relative to the tile), column pair (col, col + 1)
    __device__ __forceinline__ int row(int i) const { return wm * MT * 8 + i * 8 + rg; }
    __device__ __forceinline__ int col(int j) const { return (wn * (NT / 2) + (j >> 1)) * 16 + (j & 1) * 4 + nu_col(2 * t); }
};

template <int WM, int WN, int NT, int STAGES>
__global__ void __launch_bounds__(GemmF64Cfg<WM, WN, NT, STAGES>::THREADS, 1)
gemm_f64_kernel(const __grid_constant__ GemmMaps maps, const GemmJob* __restrict__ jobs, int njobs, int v, int vp,
                int o, int mtiles, int ntiles) {
    using C = GemmF64Cfg<WM, WN, NT, STAGES>;
    constexpr int MT = C::MT;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint64_t* full = reinterpret_cast<uint64_t*>(smem + STAGES * C::STAGE_BYTES);
    uint64_t* empty = full + STAGES;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // persistent: one CTA per SM walks work items (job, m-tile, n-tile), tiles of a job side by side on the SMs; the
    // producer runs ahead into the next item while the consumers store the previous one
    const int per_job = mtiles * ntiles;
    const long long nitems = (long long)njobs * per_job;
    const int N = v * vp;
    const int nchv = (v + 15) >> 4, ncho = (o + 15) >> 4;
    const int nch = 2 * (nchv + ncho);

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], C::NCW);
        }
        fence_barrier_init();
    }
    __syncthreads();

    if (warp == C::NCW) {
        // ------------------------------------------------------------ TMA producer (one lane)
        if (lane == 0) {
            tma_prefetch_desc(&maps.t2a); tma_prefetch_desc(&maps.ota); tma_prefetch_desc(&maps.x);
            tma_prefetch_desc(&maps.xt);  tma_prefetch_desc(&maps.t2bq); tma_prefetch_desc(&maps.t2br);
            uint32_t it = 0;
            for (long long w = blockIdx.x; w < nitems; w += gridDim.x) {
            int jb, tile;
            grouped_item(jobs, w, per_job, jb, tile);
            const int m0 = (tile % mtiles) * C::BM, n0 = (tile / mtiles) * C::BN;
            const int p = jobs[jb].p, q = jobs[jb].q, r = jobs[jb].r, xr = jobs[jb].xr, xq = jobs[jb].xq;
            for (int c = 0; c < nch; ++c, ++it) {
                const int s = it % STAGES;
                const uint32_t ph = (it / STAGES) & 1;
                mbar_wait(&empty[s], ph ^ 1);
                uint8_t* sA = smem + s * C::STAGE_BYTES;
                uint8_t* sB = sA + C::A_BYTES;
                mbar_arrive_expect_tx(&full[s], C::STAGE_BYTES);
                if (c < nchv) {                                   // sum_d t2[p,q,a,d] X_r[d,n]
                    const int kk = c * 16;
                    tma_load_3d(sA, &maps.t2a, &full[s], kk, m0, p * o + q);
                    for (int bx = 0; bx < C::BN / 16; ++bx)
                        tma_load_3d(sB + bx * 2048, &maps.x, &full[s], n0 + bx * 16, kk, xr);
                } else if (c < 2 * nchv) {                        // sum_d t2[p,r,a,d] XT_q[d,n]
                    const int kk = (c - nchv) * 16;
                    tma_load_3d(sA, &maps.t2a, &full[s], kk, m0, p * o + r);
                    for (int bx = 0; bx < C::BN / 16; ++bx)
                        tma_load_3d(sB + bx * 2048, &maps.xt, &full[s], n0 + bx * 16, kk, xq);
                } else if (c < 2 * nchv + ncho) {                 // -sum_l O_pr[a,l] t2[q,l,n]
                    const int kk = (c - 2 * nchv) * 16;
                    tma_load_3d(sA, &maps.ota, &full[s], kk, m0, r * o + p);
                    for (int bx = 0; bx < C::BN / 16; ++bx)
                        tma_load_3d(sB + bx * 2048, &maps.t2bq, &full[s], n0 + bx * 16, kk, q);
                } else {                                          // -sum_l O_pq[a,l] t2[l,r,n]
                    const int kk = (c - 2 * nchv - ncho) * 16;
                    tma_load_3d(sA, &maps.ota, &full[s], kk, m0, q * o + p);
                    for (int bx = 0; bx < C::BN / 16; ++bx)
                        tma_load_3d(sB + bx * 2048, &maps.t2br, &full[s], n0 + bx * 16, r, kk);
                }
            }
            }
        }
        return;
    }

    // ---------------------------------------------------------------- DMMA consumers
    DmmaWarp<WM, WN, NT> dw;
    dw.init(warp, lane);

    const uint32_t smem_base = smem_u32(smem);
    uint32_t it = 0;
    for (long long w = blockIdx.x; w < nitems; w += gridDim.x) {
    int jb, tile;
    grouped_item(jobs, w, per_job, jb, tile);
    const int m0 = (tile % mtiles) * C::BM, n0 = (tile / mtiles) * C::BN;
    double acc[MT][NT][2];
#pragma unroll
    for (int i = 0; i < MT; ++i)
#pragma unroll
        for (int j = 0; j < NT; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    for (int c = 0; c < nch; ++c, ++it) {
        const int s = it % STAGES;
        const uint32_t ph = (it / STAGES) & 1;
        int rem;  // valid k left in this segment from the chunk start
        if (c < nchv) rem = v - c * 16;
        else if (c < 2 * nchv) rem = v - (c - nchv) * 16;
        else if (c < 2 * nchv + ncho) rem = o - (c - 2 * nchv) * 16;
        else rem = o - (c - 2 * nchv - ncho) * 16;
        const int nu = rem >= 16 ? 4 : ((rem + 3) >> 2);
        mbar_wait(&full[s], ph);
        const uint32_t sA = smem_base + s * C::STAGE_BYTES;
        const uint32_t sB = sA + C::A_BYTES;
        dw.chunk(acc, sA, sB, nu);
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);
    }

    // ---------------------------------------------------------------- epilogue: blocked + swizzled store (ulayout.cuh)
    // column n = b*vp + c (c even): the pair (c, c+1) is one 16-byte word of the 8x8x8 block of (row, b, c)
    double* __restrict__ out = static_cast<double*>(jobs[jb].out);
    double* __restrict__ out2 = static_cast<double*>(jobs[jb].out2);
    const int nt = u_tiles(v);
#pragma unroll
    for (int j = 0; j < NT; ++j) {
        const int col = n0 + dw.col(j);
        const int bb = col / vp, cc = col - bb * vp;
        if (col < N && cc < v) {
            const size_t cb = ((size_t)(bb >> 3) * nt + (cc >> 3)) * UCHUNK;
#pragma unroll
            for (int i = 0; i < MT; ++i) {
                const int row = m0 + dw.row(i);
                if (row < v) {
                    const size_t off = (size_t)(row >> 3) * nt * nt * UCHUNK + cb + u_swz<8>(row & 7, bb & 7, cc & 7);
                    *reinterpret_cast<double2*>(out + off) = make_double2(acc[i][j][0], acc[i][j][1]);
                    if (out2) *reinterpret_cast<double2*>(out2 + off) = make_double2(acc[i][j][0], acc[i][j][1]);
                }
            }
        }
    }
    }   // work items
}

}  // namespace tb
