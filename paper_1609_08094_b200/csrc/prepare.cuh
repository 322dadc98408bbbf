// prepare.cuh -- one-time operand repack (S0 of DESIGN.md; the paper's analogue is the host->device tile
// transfer).  All outputs live in the caller's workspace.
//   X [r][d][b][c] = vvvo[d][b][c][r] = (db|cr)        (c-pitch vp = v rounded up to even, pad zeroed)
//   XT[r][d][b][c] = X[r][d][c][b]
//   Ot[r][p][a][l] = -ovoo[p][a][l][r] = -(pa|lr)      (l-pitch op = o rounded up to even, pad zeroed)
//   T2[p][q][a][d] = t2[p][q][a][d]                    (d-pitch vp, pad zeroed)
// TO is the operand type of the contraction path (double; float = the mixed path's biased FP32 words).
#pragma once
#include <cstdint>

namespace tb {

// Mixed-path operands (gemm_tf32.cuh) are FP32 values scaled by ONE power of two per tensor class -- 2^sg for the
// integrals (vv|vo), (ov|oo) and 2^st for t2 -- chosen so that the largest magnitude lands in [2^13, 2^14): the main
// term of the split product then fits FP16 (11-bit significand like TF32, twice the MMA rate; 2^14 leaves a factor 4 to
// the FP16 maximum) and every contraction term carries the same factor 2^(sg+st), removed exactly in the epilogue.
//   scales[0] = 2^sg, scales[1] = 2^st, scales[2] = 2^-(sg+st)      (floats, device memory: no host round trip)
__global__ void absmax_kernel(const double* __restrict__ x, size_t n, unsigned int* __restrict__ out) {
    float m = 0.0f;
    for (size_t e = blockIdx.x * (size_t)blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x)
        m = fmaxf(m, fabsf((float)x[e]));
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, off));
    if ((threadIdx.x & 31) == 0) atomicMax(out, __float_as_uint(m));    // non-negative floats order like their bits
}
__global__ void scales_kernel(const unsigned int* __restrict__ maxbits, float* __restrict__ scales) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    int s[2];
    for (int n = 0; n < 2; ++n) {      // maxbits[0] = integrals, maxbits[1] = t2
        const float m = __uint_as_float(maxbits[n]);
        int e = 0;
        if (m > 0.0f && m < 3.0e38f) frexpf(m, &e);          // m = f * 2^e, f in [0.5, 1)
        s[n] = m > 0.0f ? 14 - e : 0;                         // m * 2^s in [2^13, 2^14)
        if (s[n] > 100) s[n] = 100;
        if (s[n] < -100) s[n] = -100;
    }
    scales[0] = ldexpf(1.0f, s[0]);
    scales[1] = ldexpf(1.0f, s[1]);
    scales[2] = ldexpf(1.0f, -(s[0] + s[1]));
}

// operand element of the contraction path: the double itself (FP64), or the mixed path's scaled FP32 value
template <typename TO> __device__ __forceinline__ TO operand_word(double x, double scale);
template <> __device__ __forceinline__ double operand_word<double>(double x, double) { return x; }
template <> __device__ __forceinline__ float operand_word<float>(double x, double scale) { return (float)(x * scale); }

// vvvo viewed as [R = v^3][o]: each CTA moves RB consecutive rows (one contiguous span) through smem.
template <typename TO>
__global__ void __launch_bounds__(256)
pack_x_kernel(const double* __restrict__ vvvo, int v, int vp, int o, int RB, TO* __restrict__ X) {
    const double scale = 1.0;   // FP64 path only
    extern __shared__ double tile[];   // [RB][o+1]
    const size_t R = (size_t)v * v * v;
    const size_t R0 = (size_t)blockIdx.x * RB;
    const int rows = (int)min((size_t)RB, R - R0);
    const int op1 = o + 1;
    for (int e = threadIdx.x; e < rows * o; e += 256) {
        const int rr = e / o, k = e % o;
        tile[rr * op1 + k] = vvvo[R0 * o + e];
    }
    __syncthreads();
    const size_t plane = (size_t)v * v * vp;   // one r-slice of X
    for (int e = threadIdx.x; e < rows * o; e += 256) {
        const int k = e / rows, rr = e % rows;
        const size_t Rg = R0 + rr;
        const size_t db = Rg / v;
        const int c = (int)(Rg % v);
        X[(size_t)k * plane + db * vp + c] = operand_word<TO>(tile[rr * op1 + k], scale);
    }
}

// XT[r][d][b][c] = X[r][d][c][b]: tile transpose of every (r,d) plane.  blockIdx.z = r*v + d.
template <typename TO>
__global__ void __launch_bounds__(256)
transpose_planes_kernel(const TO* __restrict__ X, int v, int vp, TO* __restrict__ XT) {
    __shared__ TO tile[32][33];
    const size_t base = (size_t)blockIdx.z * v * vp;
    const int x0 = blockIdx.x * 32, y0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int yy = ty; yy < 32; yy += 8)
        if (y0 + yy < v && x0 + tx < v) tile[yy][tx] = X[base + (size_t)(y0 + yy) * vp + x0 + tx];
    __syncthreads();
    for (int yy = ty; yy < 32; yy += 8)
        if (x0 + yy < v && y0 + tx < v) XT[base + (size_t)(x0 + yy) * vp + y0 + tx] = tile[tx][yy];
}

// Ot[r][p][a][l] = -ovoo[p][a][l][r]
template <typename TO>
__global__ void pack_ot_kernel(const double* __restrict__ ovoo, int v, int o, int op, TO* __restrict__ Ot,
                               const float* __restrict__ scale_ptr) {
    const double scale = scale_ptr ? (double)*scale_ptr : 1.0;
    const size_t n = (size_t)o * o * v * o;
    for (size_t e = blockIdx.x * (size_t)blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        const int l = (int)(e % o);
        const int a = (int)((e / o) % v);
        const int p = (int)((e / ((size_t)o * v)) % o);
        const int r = (int)(e / ((size_t)o * v * o));
        const double x = -ovoo[(((size_t)p * v + a) * o + l) * o + r];
        Ot[(((size_t)r * o + p) * v + a) * op + l] = operand_word<TO>(x, scale);
    }
}

// T2[p][q][a][d] (d-pitch vp) = t2[p][q][a][d]
template <typename TO>
__global__ void pack_t2_kernel(const double* __restrict__ t2, size_t rows, int v, int vp, TO* __restrict__ T2,
                               const float* __restrict__ scale_ptr) {
    const double scale = scale_ptr ? (double)*scale_ptr : 1.0;
    const size_t n = rows * v;
    for (size_t e = blockIdx.x * (size_t)blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        const size_t row = e / v;
        const int d = (int)(e % v);
        T2[row * vp + d] = operand_word<TO>(t2[e], scale);
    }
}

// ------------------------------------------------------------------------------------------------ mixed path
// K-major operands of gemm_tf32.cuh, 4 bytes per element (scaled FP32, see scales_kernel):
//   XK  [r][b][c][d] = vvvo[d][b][c][r] = (db|cr)      (c: vp rows per b, d-pitch vk = v rounded up to 4)
//   XKT [r][b][c][d] = XK[r][c][b][d]
//   T2K [q][b][c][l] = t2[q][l][b][c]                  (l-pitch ok = o rounded up to 4)
//   T2KT[r][b][c][l] = t2[l][r][b][c] = t2[r][l][c][b]
//   T2A = pack_t2_kernel with pitch vk, OtA = pack_ot_kernel with pitch ok.
// Pads are zeroed by the caller (cudaMemsetAsync) when any exists.

// vvvo viewed as [d][s = (b,c,r) flat, v*v*o]: one CTA moves a (32 d) x (PKX_SPAN s) brick through smem and writes
// rows of 32 consecutive d (128 bytes).
constexpr int PKX_SPAN = 256;
constexpr int PKX_PITCH = PKX_SPAN + 1;
constexpr int PKX_SMEM = 32 * PKX_PITCH * 8;
__global__ void __launch_bounds__(256)
pack_xk_kernel(const double* __restrict__ vvvo, int v, int vp, int vk, int o, float* __restrict__ XK,
               float* __restrict__ XKT, const float* __restrict__ scale_ptr) {
    const double scale = (double)*scale_ptr;
    extern __shared__ double tile[];                 // [32][PKX_PITCH]
    const int d0 = blockIdx.y * 32;
    const size_t S = (size_t)v * v * o;
    const size_t s0 = (size_t)blockIdx.x * PKX_SPAN;
    const int cnt = (int)min((size_t)PKX_SPAN, S - s0);
    for (int e = threadIdx.x; e < 32 * cnt; e += 256) {
        const int dd = e / cnt, s = e % cnt;
        if (d0 + dd < v) tile[dd * PKX_PITCH + s] = vvvo[(size_t)(d0 + dd) * S + s0 + s];
    }
    __syncthreads();
    const size_t plane = (size_t)v * vp * vk;        // one r-slice
    for (int e = threadIdx.x; e < 32 * cnt; e += 256) {
        const int dd = e & 31, s = e >> 5;
        if (d0 + dd >= v) continue;
        const size_t sg = s0 + s;
        const int r = (int)(sg % o);
        const size_t bc = sg / o;
        const int b = (int)(bc / v), c = (int)(bc % v);
        const double x = tile[dd * PKX_PITCH + s];
        const float wd = (float)(x * scale);
        XK[(size_t)r * plane + ((size_t)b * vp + c) * vk + d0 + dd] = wd;
        XKT[(size_t)r * plane + ((size_t)c * vp + b) * vk + d0 + dd] = wd;
    }
}

// blockIdx.x = q*v + x (x = b for T2K, x = c for T2KT), blockIdx.y = chunk of 64 along the contiguous source index y,
// blockIdx.z = chunk of 64 along l.
__global__ void __launch_bounds__(256)
pack_t2k_kernel(const double* __restrict__ t2, int v, int vp, int o, int ok, float* __restrict__ T2K,
                float* __restrict__ T2KT, const float* __restrict__ scale_ptr) {
    const double scale = (double)*scale_ptr;
    __shared__ double tile[64][65];
    const int q = blockIdx.x / v, x = blockIdx.x % v;
    const int y0 = blockIdx.y * 64, l0 = blockIdx.z * 64;
    const int ny = min(64, v - y0), nl = min(64, o - l0);
    for (int e = threadIdx.x; e < nl * ny; e += 256) {
        const int l = e / ny, yy = e % ny;
        tile[l][yy] = t2[(((size_t)q * o + l0 + l) * v + x) * v + y0 + yy];      // t2[q][l][x][y]
    }
    __syncthreads();
    for (int e = threadIdx.x; e < nl * ny; e += 256) {
        const int l = e % nl, yy = e / nl;
        const double val = tile[l][yy];
        const float wd = (float)(val * scale);
        T2K[(((size_t)q * v + x) * vp + (y0 + yy)) * ok + l0 + l] = wd;     // T2K [q][b=x][c=y][l]
        T2KT[(((size_t)q * v + (y0 + yy)) * vp + x) * ok + l0 + l] = wd;    // T2KT[q][b=y][c=x][l] = t2[q][l][x][y]
    }
}

}  // namespace tb
