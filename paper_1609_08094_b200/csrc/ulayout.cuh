// ulayout.cuh -- HBM layout of the contraction outputs U (the per-triplet v^3 blocks of DESIGN.md section 6).
//
// A U buffer holds G(p,q,r)[x][y][z] (x = GEMM row, (y,z) = flat GEMM column) cut into 8x8x8 tiles; every tile
// is one CONTIGUOUS block of 512 elements.  The three buffers U1,U2,U3 of one triplet are interleaved tile by tile:
//   slot[x/8][y/8][z/8][u = 0..2][512]          over nt = ceil(v/8) tiles per axis,
// so that the fused reduction (reduce.cuh) pulls the three blocks of a tile into shared memory with ONE
// cp.async.bulk (12 KiB FP64 / 6 KiB FP32 sequential read; the TMA unit costs ~65 clk per copy whatever its size,
// measured), and then reads every block along all three axes, because W is the sum of three
// U's at permuted indices (Eq. (2.2.3)).  To make all of those shared-memory reads bank-conflict
// free without a transposing pass, the position of (x,y,z) INSIDE a block is an XOR swizzle chosen so that the
// 16 (FP64: half-warp of 8-byte words) or 32 (FP32: warp of 4-byte words) lanes of a read hit distinct banks for
// every one of the six index permutations.  Lane bits of the reduction are (c0,c1,b0,a0[,b1]) of the index triple
// (a,b,c), i.e. {x0,y0,z0} plus one (two) of {x1,y1,z1} whatever the permutation:
//
//   FP64 (bank pair = position bits 0..3):  p = z0 | (z1^x1^y1)<<1 | (z2^x0)<<2 | y0<<3 | x0<<4 | x1<<5 | y1<<6 | x2<<7 | y2<<8
//   FP32 (bank      = position bits 0..4):  p = x0 | (x1^z1)<<1 | (x2^y0)<<2 | z0<<3 | (y1^z1)<<4 | y0<<5 | z1<<6 | y2<<7 | z2<<8
//
// FP64: the three low bits are z0, z1, z2 up to an XOR with x/y bits, so the 8 z-values of one (x,y) stay inside one
// aligned 64-byte chunk: the FP64 GEMM epilogue (a thread owns (z, z+1) column pairs) writes whole 32-byte sectors.
// FP32: the same map with the roles rotated, S(x,y,z) = S0(y,z,x) -- the reduction reads every block in all six
// arrangements, so any relabelling of the arguments is conflict free as well -- which puts the 8 x-values of one
// (y,z) into one aligned 32-byte chunk: in the mixed GEMM a thread owns one (y,z) = (b,c) row and all x = a columns
// (gemm_f16split.cuh), so its epilogue is two 16-byte stores per tile instead of eight scattered words.
// Both maps are linear over GF(2): u_swz(x,y,z) = u_swz(x,0,0) ^ u_swz(0,y,z).
// Elements with an index >= v inside the last tile of an axis are never written and never read.
#pragma once
#include <cstddef>
#include <cstdint>

namespace tb {

constexpr int UT = 8;              // tile edge
constexpr int UBLK = UT * UT * UT;   // elements per block
constexpr int UCHUNK = 3 * UBLK;     // elements per tile of a triplet slot: the blocks of U1, U2, U3

__host__ __device__ constexpr int u_tiles(int v) { return (v + UT - 1) / UT; }
// elements of ONE of the three interleaved buffers (a triplet slot has 3 * u_elems)
__host__ __device__ constexpr size_t u_elems(int v) { return (size_t)u_tiles(v) * u_tiles(v) * u_tiles(v) * UBLK; }

template <int ESZ> __host__ __device__ constexpr int u_swz(int x, int y, int z);
template <> __host__ __device__ constexpr int u_swz<8>(int x, int y, int z) {
    return (z & 1) | ((((z ^ x ^ y) >> 1) & 1) << 1) | ((((z >> 2) ^ x) & 1) << 2) | ((y & 1) << 3) | ((x & 1) << 4) |
           (((x >> 1) & 1) << 5) | (((y >> 1) & 1) << 6) | (((x >> 2) & 1) << 7) | (((y >> 2) & 1) << 8);
}
template <> __host__ __device__ constexpr int u_swz<4>(int x, int y, int z) {
    return (x & 1) | ((((x ^ z) >> 1) & 1) << 1) | ((((x >> 2) ^ y) & 1) << 2) | ((z & 1) << 3) |
           ((((y ^ z) >> 1) & 1) << 4) | ((y & 1) << 5) | (((z >> 1) & 1) << 6) | (((y >> 2) & 1) << 7) |
           (((z >> 2) & 1) << 8);
}

// element offset of (x,y,z) of buffer u = 0 relative to the slot base (buffer u starts u * UBLK further on)
template <int ESZ>
__host__ __device__ __forceinline__ size_t u_offset(int nt, int x, int y, int z) {
    return ((size_t)((x >> 3) * nt + (y >> 3)) * nt + (z >> 3)) * UCHUNK + u_swz<ESZ>(x & 7, y & 7, z & 7);
}

// (ov|ov) 8x8 tiles of the reduction's side buffer: Morton order, so that reads indexed by any ordered pair of
// (a,b,c) are conflict free with the same lane bits:  q = y0 | x0<<1 | y1<<2 | x1<<3 | y2<<4 | x2<<5.
__host__ __device__ constexpr int j_swz(int x, int y) {
    return (y & 1) | ((x & 1) << 1) | (((y >> 1) & 1) << 2) | (((x >> 1) & 1) << 3) | (((y >> 2) & 1) << 4) |
           (((x >> 2) & 1) << 5);
}

}  // namespace tb
