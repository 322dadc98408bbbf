// prepare.cuh -- one-time operand repack (S0 of DESIGN.md; the paper's analogue is the host->device tile
// transfer).  All outputs live in the caller's workspace.
//   X [r][d][b][c] = vvvo[d][b][c][r] = (db|cr)        (c-pitch vp = v rounded up to even, pad zeroed)
//   XT[r][d][b][c] = X[r][d][c][b]
//   Ot[r][p][a][l] = -ovoo[p][a][l][r] = -(pa|lr)      (l-pitch op = o rounded up to even, pad zeroed)
//   T2[p][q][a][d] = t2[p][q][a][d]                    (d-pitch vp, pad zeroed)
// TO is the operand type of the FP64 contraction path (double).  The mixed path's operands are written pre-split
// (FP16 h | l rows, second half of this file).
#pragma once
#include <cuda_fp16.h>

#include <cstdint>

namespace tb {

// Mixed-path operands (gemm_f16split.cuh; written pre-split into FP16 h | l rows, see below) are scaled by ONE power of two per tensor class -- 2^sg for the
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
    reinterpret_cast<int*>(scales)[12] = s[0];       // the exponents themselves (emulated-FP64 path, gemm_emu64.cuh)
    reinterpret_cast<int*>(scales)[13] = s[1];
}

// vvvo viewed as [R = v^3][o]: each CTA moves RB consecutive rows (one contiguous span) through smem.
template <typename TO>
__global__ void __launch_bounds__(256)
pack_x_kernel(const double* __restrict__ vvvo, int v, int vp, int o, int RB, TO* __restrict__ X) {
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
        X[(size_t)k * plane + db * vp + c] = (TO)tile[rr * op1 + k];
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
__global__ void pack_ot_kernel(const double* __restrict__ ovoo, int v, int o, int op, TO* __restrict__ Ot) {
    const size_t n = (size_t)o * o * v * o;
    for (size_t e = blockIdx.x * (size_t)blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        const int l = (int)(e % o);
        const int a = (int)((e / o) % v);
        const int p = (int)((e / ((size_t)o * v)) % o);
        const int r = (int)(e / ((size_t)o * v * o));
        const double x = -ovoo[(((size_t)p * v + a) * o + l) * o + r];
        Ot[(((size_t)r * o + p) * v + a) * op + l] = (TO)x;
    }
}

// T2[p][q][a][d] (d-pitch vp) = t2[p][q][a][d]
template <typename TO>
__global__ void pack_t2_kernel(const double* __restrict__ t2, size_t rows, int v, int vp, TO* __restrict__ T2) {
    const size_t n = rows * v;
    for (size_t e = blockIdx.x * (size_t)blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        const size_t row = e / v;
        const int d = (int)(e % v);
        T2[row * vp + d] = (TO)t2[e];
    }
}

// ------------------------------------------------------------------------------------------------ mixed path
// K-major operands of gemm_f16split.cuh, written SPLIT (Q13): with xs = (float)(x * 2^s) the scaled value,
// h = RN_fp16(xs), l = RN_fp16(xs - h).  Per operand row and 32-wide K chunk one 128-byte row of 32 words:
// words 0..15 = the 32 FP16 of h, words 16..31 = the 32 FP16 of l (element k in the low half of word k/2 for even k).
// K pitches vk / ok = v / o rounded up to 32; K elements beyond v / o are written as zeros.
//   XK  [s][b][c][d] = (db|cr) of the slice r held in slot s   (c: vp rows per b)
//   XKT [s][b][c][d] = XK[s][c][b][d]
//   T2K [q][b][c][l] = t2[q][l][b][c]
//   T2KT[r][b][c][l] = t2[l][r][b][c] = t2[r][l][c][b]
//   T2A [p][q][a][d] = t2[p][q][a][d],  OtA[r][p][a][l] = -ovoo[p][a][l][r]
// Rows c = v (odd v only) are zeroed by the caller (cudaMemsetAsync).

// The 32 lanes of a warp hold 32 consecutive K elements (lane = k within the chunk) and write the chunk's packed row.
__device__ __forceinline__ void pack_split_store(uint32_t* __restrict__ row, float xs, int lane) {
    const __half h = __float2half_rn(xs);
    const __half l = __float2half_rn(xs - __half2float(h));
    const uint32_t hb = __half_as_ushort(h), lb = __half_as_ushort(l);
    const bool odd = (lane & 1) != 0;            // even lane 2j assembles word j (h pair), odd lane 2j+1 word 16+j (l pair)
    const uint32_t mine = odd ? lb : hb;
    const uint32_t got = __shfl_xor_sync(0xffffffffu, odd ? hb : lb, 1);
    row[(lane >> 1) + (odd ? 16 : 0)] = odd ? (got | (mine << 16)) : (mine | (got << 16));
}

// Emulated-FP64 path (gemm_emu64.cuh): the scaled value is rounded to a 47-bit fixed-point integer
// xi = rint(x * 2^(s + 32)) (|xi| < 2^46: the class maximum sits in [2^45, 2^46)) and cut into six balanced base-256
// digits d_0 (most significant, |d_0| <= 64) .. d_5 in [-128, 127], xi = sum_i d_i 256^(5-i).  K is walked in chunks of 64; per
// operand row and chunk THREE 128-byte rows (96 words): row p holds digit 2p of the 64 K elements in bytes 0..63 and
// digit 2p+1 in bytes 64..127 -- 6 bytes per element, no padding.  The 32 lanes of a warp hold 32 consecutive K
// elements = half h of a chunk.
constexpr int EMU_SHIFT = 32;
constexpr int EMU_DIGITS = 6;
constexpr int EMU_CHUNK_WORDS = 96;
__device__ __forceinline__ void pack_emu_store(uint32_t* __restrict__ chunk, int h, double x, int lane) {
    long long xi = __double2ll_rn(x);
    int8_t d[EMU_DIGITS];
#pragma unroll
    for (int i = EMU_DIGITS - 1; i >= 0; --i) {
        int r = (int)(xi & 255);
        if (r >= 128) r -= 256;
        d[i] = (int8_t)r;
        xi = (xi - r) >> 8;
    }
    int8_t* b = reinterpret_cast<int8_t*>(chunk);
#pragma unroll
    for (int i = 0; i < EMU_DIGITS; ++i) b[(i >> 1) * 128 + (i & 1) * 64 + h * 32 + lane] = d[i];
}
// K chunk ch (32 elements) of the operand row starting at `row`: MODE 0 = FP16 split (32 words per chunk),
// MODE 1 = emulated-FP64 digits (96 words per pair of chunks)
template <int MODE>
__device__ __forceinline__ void pack_store(uint32_t* __restrict__ row, int ch, double x, double scale, int lane) {
    if constexpr (MODE == 0) pack_split_store(row + (size_t)ch * 32, (float)(x * scale), lane);
    else pack_emu_store(row + (size_t)(ch >> 1) * EMU_CHUNK_WORDS, ch & 1, x * scale, lane);
}
// 32-element K chunks a row of pitch `words` holds
template <int MODE> __device__ __forceinline__ int pack_chunks(int words) {
    return MODE == 0 ? words / 32 : 2 * (words / EMU_CHUNK_WORDS);
}
// scale of a tensor class: sc = the scales block of prepare (floats 2^sg, 2^st, .. ; ints sg, st at [12], [13])
template <int MODE>
__device__ __forceinline__ double pack_scale(const float* __restrict__ sc, int cls) {
    if constexpr (MODE == 0) return (double)sc[cls];
    else return ldexp(1.0, reinterpret_cast<const int*>(sc)[12 + cls] + EMU_SHIFT);
}

// Source viewed as [d][s], s = bc * ro + r (resident vvvo: ro = o, the slice of r goes to slot r) or s = bc
// (one FP64 slice (db|c r): ro = 1, slot0 = its slot); sp = c-pitch of the source (v, or vp for a slice the RI
// builder wrote).  One CTA moves a (32 d) x (PKX_SPAN s) brick through shared memory and writes whole 128-byte
// packed rows; blockIdx.y = K chunk.
constexpr int PKX_SPAN = 256;
constexpr int PKX_PITCH = PKX_SPAN + 1;
constexpr int PKX_SMEM = 32 * PKX_PITCH * 8;
template <int MODE>
__global__ void __launch_bounds__(256)
pack_xk_kernel(const double* __restrict__ src, int v, int vp, int vk, int ro, int sp, int slot0,
               uint32_t* __restrict__ XK, uint32_t* __restrict__ XKT, const float* __restrict__ sc,
               unsigned int* __restrict__ overflow) {
    const double scale = pack_scale<MODE>(sc, 0);
    // The scale puts the class maximum in [2^13, 2^14) (FP16 split) / [2^45, 2^46) (digits).  A scaled element at or
    // beyond that bound means the maximum the scale was derived from was too small (a caller-supplied vvvo_absmax of a
    // streamed run): FP16 would overflow, the top digit would wrap.  Flagged here, turned into TRIPLES_EINVAL by the host.
    const double bound = MODE == 0 ? 16384.0 : 70368744177664.0;
    bool over = false;
    extern __shared__ double tile[];                 // [32][PKX_PITCH]
    const int d0 = blockIdx.y * 32;
    const size_t S = (size_t)v * v * ro;
    const size_t s0 = (size_t)blockIdx.x * PKX_SPAN;
    const int cnt = (int)min((size_t)PKX_SPAN, S - s0);
    const size_t Sd = (size_t)v * sp * ro;           // source elements per d
    for (int e = threadIdx.x; e < 32 * cnt; e += 256) {
        const int dd = e / cnt, s = e % cnt;
        size_t off = s0 + s;
        if (sp != v) { const size_t bc = off / ro; off = ((bc / v) * sp + bc % v) * ro + off % ro; }
        tile[dd * PKX_PITCH + s] = d0 + dd < v ? src[(size_t)(d0 + dd) * Sd + off] : 0.0;
    }
    __syncthreads();
    const size_t plane = (size_t)v * vp * vk;        // words of one slot
    const int lane = threadIdx.x & 31;
    for (int e = threadIdx.x; e < 32 * cnt; e += 256) {      // a warp = the 32 d of one s
        const int s = e >> 5;
        const size_t sg = s0 + s;
        const int r = (int)(sg % ro);
        const size_t bc = sg / ro;
        const int b = (int)(bc / v), c = (int)(bc % v);
        const double x = tile[lane * PKX_PITCH + s];
        over |= fabs(x * scale) >= bound;
        const size_t base = (size_t)(slot0 + r) * plane;
        pack_store<MODE>(XK + base + ((size_t)b * vp + c) * vk, blockIdx.y, x, scale, lane);
        pack_store<MODE>(XKT + base + ((size_t)c * vp + b) * vk, blockIdx.y, x, scale, lane);
    }
    if (over) *overflow = 1u;       // every writer stores the same value
}

// blockIdx.x = q*v + x (x = b for T2K, x = c for T2KT), blockIdx.y = chunk of 64 along the contiguous source index y,
// blockIdx.z = chunk of 64 along l (two packed rows).
template <int MODE>
__global__ void __launch_bounds__(256)
pack_t2k_kernel(const double* __restrict__ t2, int v, int vp, int o, int ok, uint32_t* __restrict__ T2K,
                uint32_t* __restrict__ T2KT, const float* __restrict__ sc) {
    const double scale = pack_scale<MODE>(sc, 1);
    __shared__ double tile[64][65];
    const int q = blockIdx.x / v, x = blockIdx.x % v;
    const int y0 = blockIdx.y * 64, l0 = blockIdx.z * 64;
    const int ny = min(64, v - y0), nl = min(64, o - l0);
    for (int e = threadIdx.x; e < 64 * ny; e += 256) {
        const int l = e / ny, yy = e % ny;
        tile[l][yy] = l < nl ? t2[(((size_t)q * o + l0 + l) * v + x) * v + y0 + yy] : 0.0;      // t2[q][l][x][y]
    }
    __syncthreads();
    const int lane = threadIdx.x & 31;
    for (int e = threadIdx.x; e < 64 * ny; e += 256) {       // a warp = 32 consecutive l of one y
        const int lh = (e >> 5) & 1, yy = e >> 6;
        const int ch = l0 / 32 + lh;                         // 32-element K chunk of the row
        if (ch >= pack_chunks<MODE>(ok)) continue;           // warp-uniform
        const double xv = tile[lh * 32 + lane][yy];
        pack_store<MODE>(T2K + (((size_t)q * v + x) * vp + (y0 + yy)) * ok, ch, xv, scale, lane);     // T2K [q][b=x][c=y][l]
        pack_store<MODE>(T2KT + (((size_t)q * v + (y0 + yy)) * vp + x) * ok, ch, xv, scale, lane);    // T2KT[q][b=y][c=x][l]
    }
}

// T2A[row][d], row = (p,q,a): one warp per (row, K chunk)
template <int MODE>
__global__ void __launch_bounds__(256)
pack_t2a_kernel(const double* __restrict__ t2, size_t rows, int v, int vk, uint32_t* __restrict__ T2A,
                const float* __restrict__ sc) {
    const double scale = pack_scale<MODE>(sc, 1);
    const int lane = threadIdx.x & 31, nch = pack_chunks<MODE>(vk);
    const size_t nw = rows * nch;
    for (size_t w = blockIdx.x * (size_t)8 + (threadIdx.x >> 5); w < nw; w += (size_t)gridDim.x * 8) {
        const size_t row = w / nch;
        const int ch = (int)(w % nch), d = ch * 32 + lane;
        const double x = d < v ? t2[row * v + d] : 0.0;
        pack_store<MODE>(T2A + row * vk, ch, x, scale, lane);
    }
}

// OtA[r][p][a][l] = -ovoo[p][a][l][r]: one warp per ((r,p,a), K chunk)
template <int MODE>
__global__ void __launch_bounds__(256)
pack_ota_kernel(const double* __restrict__ ovoo, int v, int o, int ok, uint32_t* __restrict__ OtA,
                const float* __restrict__ sc) {
    const double scale = pack_scale<MODE>(sc, 0);
    const int lane = threadIdx.x & 31, nch = pack_chunks<MODE>(ok);
    const size_t nw = (size_t)o * o * v * nch;
    for (size_t w = blockIdx.x * (size_t)8 + (threadIdx.x >> 5); w < nw; w += (size_t)gridDim.x * 8) {
        const size_t row = w / nch;                        // (r, p, a)
        const int ch = (int)(w % nch), l = ch * 32 + lane;
        const int a = (int)(row % v), p = (int)((row / v) % o), r = (int)(row / ((size_t)v * o));
        const double x = l < o ? -ovoo[(((size_t)p * v + a) * o + l) * o + r] : 0.0;
        pack_store<MODE>(OtA + row * ok, ch, x, scale, lane);
    }
}

}  // namespace tb
