// reduce.cuh -- fused permutation-accumulate + V assembly + denominator + energy contraction (S4-S7),
// the per-triplet finalize (S8a) and the deterministic total (S8b).
//
// Per triplet (i<=j<=k) the contraction kernel left three natural-order buffers
//   U1 = G(i,j,k)[a][b][c],  U2 = G(j,i,k)[b][a][c],  U3 = G(k,i,j)[c][a][b]      (c-pitch vp)
// and W^abc = U1[a,b,c] + U2[b,a,c] + U3[c,a,b]            (Eq. (2.2.3)).
// The energy of the triplet is  e = sum_abc Z[W]^abc (W + Vd)^abc / D^abc  with
//   Z[W]^abc = 4W^abc + W^bca + W^cab - 2W^acb - 2W^cba - 2W^bac   (symmetrised Eq. (2.2.5); Q4)
//   Vd^abc   = t1[i,a] (jb|kc) + t1[j,b] (ia|kc) + t1[k,c] (ia|jb)                 (Eq. (2.2.4))
//   D^abc    = eps_i + eps_j + eps_k - eps_a - eps_b - eps_c                       (L92, L65; Q1)
//
// One CTA owns one *tile orbit* {A<=B<=C} of 8x8x8 blocks of the virtual cube: it stages W on the six
// permuted blocks in shared memory (every U element of the orbit is read from HBM once), then every thread
// walks index triples (a in A, b in B, c in C) and adds the contribution of all six permutations of (a,b,c):
//   w_pi = W at the six permutations;  E = w_abc + w_bca + w_cab (even),  O = w_acb + w_bac + w_cba (odd)
//   sum_pi Z_pi w_pi  = 3 sum w_pi^2 + (E-O)^2 - 2 E O
//   sum_pi Z_pi vd_pi = sum_pi vd_pi (3 w_pi + [same-parity sum] - 2 [other-parity sum])
// with one division per index triple (D is symmetric in abc).  Orbits with coinciding tiles visit every element
// `sym` in {2,6} times and are scaled by 1/sym.
#pragma once
#include <cstdint>

namespace tb {

template <typename T>
struct RedJob {
    int i, j, k, slot;      // slot: row of `partials` this triplet writes
    const T* u1;
    const T* u2;
    const T* u3;
};

constexpr int RT = 8;             // tile edge
constexpr int RP1 = 9;            // smem pitch of the fastest index
constexpr int RP2 = 74;           // smem pitch of the middle index (8*9 + 2)
constexpr int RBLK = RT * RP2;    // one staged block
constexpr int RED_THREADS = 256;

template <typename T> struct Vec2;
template <> struct Vec2<double> { using type = double2; };
template <> struct Vec2<float> { using type = float2; };

template <typename T>
__global__ void __launch_bounds__(RED_THREADS)
reduce_kernel(const RedJob<T>* __restrict__ jobs, const uchar4* __restrict__ orbits, int norb, int v, int vp, int o,
              const double* __restrict__ eps_o, const double* __restrict__ eps_v, const double* __restrict__ t1,
              const double* __restrict__ ovov, double2* __restrict__ partials) {
    using V2 = typename Vec2<T>::type;
    __shared__ double S[6 * RBLK];          // W on the six blocks, S[blk][x][y][z]
    __shared__ double Js[3][6][RT][RP1];    // (ov|ov) slices on the six ordered tile pairs
    __shared__ double T1s[3][3][RT];        // t1[i|j|k][tile A|B|C]
    __shared__ double Ev[3][RT];            // eps_v on tiles A,B,C
    __shared__ double red[2][RED_THREADS / 32];

    const int tid = threadIdx.x;
    const RedJob<T> job = jobs[blockIdx.y];
    const uchar4 orb = orbits[blockIdx.x];
    const int tl[3] = {orb.x * RT, orb.y * RT, orb.z * RT};   // first index of tiles A, B, C
    const size_t pa = (size_t)v * vp;                          // pitch of the slowest index of U

    // block pi holds W[x][y][z] with x in tile PX[pi], y in PY[pi], z in PZ[pi]  (0=A, 1=B, 2=C)
    constexpr int PX[6] = {0, 0, 1, 1, 2, 2};
    constexpr int PY[6] = {1, 2, 0, 2, 0, 1};
    constexpr int PZ[6] = {2, 1, 2, 0, 1, 0};

    // ---- issue all global loads of the orbit first (18 vector loads per thread in flight)
    V2 r1[6], r2[6], r3[6];
    {
        const int x = tid >> 5, y = (tid >> 2) & 7, z = (tid & 3) * 2;       // U1/U2: z pairs contiguous
        const int z3 = tid >> 5, x3 = (tid >> 2) & 7, y3 = (tid & 3) * 2;    // U3:    y pairs contiguous
#pragma unroll
        for (int b = 0; b < 6; ++b) {
            const int X0 = tl[PX[b]], Y0 = tl[PY[b]], Z0 = tl[PZ[b]];
            V2 zero; zero.x = 0; zero.y = 0;
            r1[b] = zero; r2[b] = zero; r3[b] = zero;
            if (X0 + x < v && Y0 + y < v && Z0 + z < v) {
                r1[b] = *reinterpret_cast<const V2*>(job.u1 + (size_t)(X0 + x) * pa + (size_t)(Y0 + y) * vp + Z0 + z);
                r2[b] = *reinterpret_cast<const V2*>(job.u2 + (size_t)(Y0 + y) * pa + (size_t)(X0 + x) * vp + Z0 + z);
            }
            if (Z0 + z3 < v && X0 + x3 < v && Y0 + y3 < v)
                r3[b] = *reinterpret_cast<const V2*>(job.u3 + (size_t)(Z0 + z3) * pa + (size_t)(X0 + x3) * vp + Y0 + y3);
        }
        // ---- small operands: (ov|ov) tiles, t1 rows, eps_v
        const int occ[3] = {job.i, job.j, job.k};
        for (int e = tid; e < 3 * 6 * 64; e += RED_THREADS) {
            const int yy = e & 7, xx = (e >> 3) & 7, tp = (e >> 6) % 6, s = e / 384;
            // ordered tile pairs (P,Q): (A,B),(A,C),(B,A),(B,C),(C,A),(C,B)
            const int P = tp >> 1, Q = (tp & 1) ? (P == 2 ? 1 : 2) : (P == 0 ? 1 : 0);
            const int o1 = (s == 0) ? occ[1] : occ[0];          // s=0: (j.|k.)  s=1: (i.|k.)  s=2: (i.|j.)
            const int o2 = (s == 2) ? occ[1] : occ[2];
            const int gx = tl[P] + xx, gy = tl[Q] + yy;
            double val = 0.0;
            if (gx < v && gy < v) val = ovov[(((size_t)o1 * v + gx) * o + o2) * v + gy];
            Js[s][tp][xx][yy] = val;
        }
        if (tid < 72) {
            const int xx = tid & 7, tile = (tid >> 3) % 3, s = tid / 24;
            const int gx = tl[tile] + xx;
            T1s[s][tile][xx] = gx < v ? t1[(size_t)occ[s] * v + gx] : 0.0;
        } else if (tid < 96) {
            const int xx = tid & 7, tile = (tid - 72) >> 3;
            const int gx = tl[tile] + xx;
            Ev[tile][xx] = gx < v ? eps_v[gx] : 0.0;
        }
        // ---- W = U1 + U2 (registers) -> smem, then += U3
#pragma unroll
        for (int b = 0; b < 6; ++b) {
            double* dst = S + b * RBLK + x * RP2 + y * RP1 + z;
            dst[0] = (double)r1[b].x + (double)r2[b].x;
            dst[1] = (double)r1[b].y + (double)r2[b].y;
        }
        __syncthreads();
#pragma unroll
        for (int b = 0; b < 6; ++b) {
            double* dst = S + b * RBLK + x3 * RP2 + y3 * RP1 + z3;
            dst[0] += (double)r3[b].x;
            dst[RP1] += (double)r3[b].y;
        }
        __syncthreads();
    }

    // ---- energy contraction over index triples (a in A, b in B, c in C)
    const double eo = eps_o[job.i] + eps_o[job.j] + eps_o[job.k];
    double e4 = 0.0, e5 = 0.0;
    const int c = tid & 7, b = (tid >> 3) & 7;
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const int a = (tid >> 6) + 4 * h;
        if (tl[0] + a < v && tl[1] + b < v && tl[2] + c < v) {
            const double w0 = S[0 * RBLK + a * RP2 + b * RP1 + c];   // W^abc
            const double w1 = S[1 * RBLK + a * RP2 + c * RP1 + b];   // W^acb
            const double w2 = S[2 * RBLK + b * RP2 + a * RP1 + c];   // W^bac
            const double w3 = S[3 * RBLK + b * RP2 + c * RP1 + a];   // W^bca
            const double w4 = S[4 * RBLK + c * RP2 + a * RP1 + b];   // W^cab
            const double w5 = S[5 * RBLK + c * RP2 + b * RP1 + a];   // W^cba
            const double E = w0 + w3 + w4, O = w1 + w2 + w5;
            const double q4 = 3.0 * (w0 * w0 + w1 * w1 + w2 * w2 + w3 * w3 + w4 * w4 + w5 * w5) + (E - O) * (E - O) -
                              2.0 * E * O;
            // Vd on the six permutations; Js[s][tp]: tp 0:(a,b) 1:(a,c) 2:(b,a) 3:(b,c) 4:(c,a) 5:(c,b)
            const double ti_a = T1s[0][0][a], ti_b = T1s[0][1][b], ti_c = T1s[0][2][c];
            const double tj_a = T1s[1][0][a], tj_b = T1s[1][1][b], tj_c = T1s[1][2][c];
            const double tk_a = T1s[2][0][a], tk_b = T1s[2][1][b], tk_c = T1s[2][2][c];
#define JJ(s, tp, x, y) Js[s][tp][x][y]
            const double d0 = ti_a * JJ(0, 3, b, c) + tj_b * JJ(1, 1, a, c) + tk_c * JJ(2, 0, a, b);   // abc
            const double d1 = ti_a * JJ(0, 5, c, b) + tj_c * JJ(1, 0, a, b) + tk_b * JJ(2, 1, a, c);   // acb
            const double d2 = ti_b * JJ(0, 1, a, c) + tj_a * JJ(1, 3, b, c) + tk_c * JJ(2, 2, b, a);   // bac
            const double d3 = ti_b * JJ(0, 4, c, a) + tj_c * JJ(1, 2, b, a) + tk_a * JJ(2, 3, b, c);   // bca
            const double d4 = ti_c * JJ(0, 0, a, b) + tj_a * JJ(1, 5, c, b) + tk_b * JJ(2, 4, c, a);   // cab
            const double d5 = ti_c * JJ(0, 2, b, a) + tj_b * JJ(1, 4, c, a) + tk_a * JJ(2, 5, c, b);   // cba
#undef JJ
            const double ze = E - 2.0 * O, zo = O - 2.0 * E;   // same-parity sum - 2 * other-parity sum
            const double q5 = d0 * (3.0 * w0 + ze) + d3 * (3.0 * w3 + ze) + d4 * (3.0 * w4 + ze) +
                              d1 * (3.0 * w1 + zo) + d2 * (3.0 * w2 + zo) + d5 * (3.0 * w5 + zo);
            const double rD = 1.0 / (eo - Ev[0][a] - Ev[1][b] - Ev[2][c]);
            e4 += q4 * rD;
            e5 += q5 * rD;
        }
    }
    // ---- deterministic block reduction: shuffle tree, then warp partials in index order
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        e4 += __shfl_xor_sync(0xffffffffu, e4, off);
        e5 += __shfl_xor_sync(0xffffffffu, e5, off);
    }
    if ((tid & 31) == 0) { red[0][tid >> 5] = e4; red[1][tid >> 5] = e5; }
    __syncthreads();
    if (tid == 0) {
        double s4 = 0.0, s5 = 0.0;
#pragma unroll
        for (int w = 0; w < RED_THREADS / 32; ++w) { s4 += red[0][w]; s5 += red[1][w]; }
        const double inv = orb.w == 1 ? 1.0 : (orb.w == 2 ? 0.5 : 1.0 / 6.0);
        partials[(size_t)job.slot * norb + blockIdx.x] = make_double2(s4 * inv, s5 * inv);
    }
}

// One CTA per triplet of the batch: fixed-order sum of its orbit partials, weight w = 2 - d_ij - d_jk,
// written to e_trip[3*index + {0,1,2}] = w(e4+e5), w e4, w e5.
struct FinJob { int slot; int index; double w; };

__global__ void __launch_bounds__(128)
finalize_kernel(const FinJob* __restrict__ jobs, const double2* __restrict__ partials, int norb,
                double* __restrict__ e_trip) {
    __shared__ double sh[2][128];
    const FinJob job = jobs[blockIdx.x];
    const double2* p = partials + (size_t)job.slot * norb;
    double s4 = 0.0, s5 = 0.0;
    for (int n = threadIdx.x; n < norb; n += 128) { s4 += p[n].x; s5 += p[n].y; }
    sh[0][threadIdx.x] = s4; sh[1][threadIdx.x] = s5;
    __syncthreads();
    for (int st = 64; st > 0; st >>= 1) {
        if (threadIdx.x < st) {
            sh[0][threadIdx.x] += sh[0][threadIdx.x + st];
            sh[1][threadIdx.x] += sh[1][threadIdx.x + st];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const double e4 = job.w * sh[0][0], e5 = job.w * sh[1][0];
        e_trip[3 * (size_t)job.index + 0] = e4 + e5;
        e_trip[3 * (size_t)job.index + 1] = e4;
        e_trip[3 * (size_t)job.index + 2] = e5;
    }
}

// Single CTA: E[4] = sum_n e_trip[3n+1], E[5] = sum_n e_trip[3n+2] in a fixed order, E(T) = E[4] + E[5].
__global__ void __launch_bounds__(256) total_kernel(const double* __restrict__ e_trip, long long ntrip,
                                                    double* __restrict__ result) {
    __shared__ double sh[2][256];
    double s4 = 0.0, s5 = 0.0;
    for (long long n = threadIdx.x; n < ntrip; n += 256) { s4 += e_trip[3 * n + 1]; s5 += e_trip[3 * n + 2]; }
    sh[0][threadIdx.x] = s4; sh[1][threadIdx.x] = s5;
    __syncthreads();
    for (int st = 128; st > 0; st >>= 1) {
        if (threadIdx.x < st) {
            sh[0][threadIdx.x] += sh[0][threadIdx.x + st];
            sh[1][threadIdx.x] += sh[1][threadIdx.x + st];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        result[1] = sh[0][0];
        result[2] = sh[1][0];
        result[0] = sh[0][0] + sh[1][0];
    }
}

// W_out[a][b][c] = U1[a,b,c] + U2[b,a,c] + U3[c,a,b]  (test entry point triples_w_block; not on the hot path)
template <typename T>
__global__ void assemble_w_kernel(const T* __restrict__ u1, const T* __restrict__ u2, const T* __restrict__ u3, int v,
                                  int vp, double* __restrict__ W) {
    const size_t n = (size_t)v * v * v;
    const size_t pa = (size_t)v * vp;
    for (size_t e = blockIdx.x * (size_t)blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        const int c = (int)(e % v), b = (int)((e / v) % v), a = (int)(e / ((size_t)v * v));
        W[e] = (double)u1[a * pa + (size_t)b * vp + c] + (double)u2[b * pa + (size_t)a * vp + c] +
               (double)u3[c * pa + (size_t)a * vp + b];
    }
}

}  // namespace tb
