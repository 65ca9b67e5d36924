// md_packed.cuh -- the FRAGMENT-MAJOR PACKED layout of quarter planes inside the md_gemm workspace.
// Written by split_packed_kernel (split.cu), read by qgemm_packed_kernel (qgemm_packed.cu); internal to libmdgemm -- the
// public md_split / md_qgemm keep the plain [quarters][rows][cols] layout.
//
// An operand is seen as X groups (rows of A, axis 0 / columns of B, axis 1: the index that carries the exponent) by K
// contraction indices.  X is cut into tiles of BX (the CTA tile: BM for A, BN for B), K into slabs of BK = pack_bk(limbs); both are
// zero padded to whole tiles / slabs (zero quarters are harmless).  Memory order, slowest to fastest:
//
//     [x tile][k slab]  [quarter q][k4 = (k % BK) / 4][x8 = (x % BX) / 8]  [g = x % 8][t4 = k % 4]
//      \___ chunk ___/   \_______________ inside a chunk _______________/   \__ one DMMA fragment: 32 doubles __/
//
// so that (1) the Q * BK * BX doubles a CTA needs per k-slab are contiguous -> one cp.async.bulk; (2) consecutive slabs
// of a tile are contiguous -> a CTA streams through one region; (3) lane 4g + t4 of a warp finds its element of the
// 8x4 (A: row g, k t4) or 4x8 (B: k t4, column g) mma.m8n8k4 operand fragment at fragment base + lane.
#pragma once
#include <stddef.h>

namespace md {

// k-slab depth BK: two DMMA k-steps for double / quad double (qgemm_packed.cu), one for octo / hexa double
// (qgemm_wide.cu: 32 / 64 quarters per element make a slab of 8 too large for a multi-stage ring in 227 KB).
constexpr int PACK_BK = 8, PACK_BK_WIDE = 4;
__host__ __device__ constexpr int pack_bk(int limbs) { return limbs <= 4 ? PACK_BK : PACK_BK_WIDE; }

// CTA tile extent along the group index: BM (axis 0) or BN (axis 1) of the fused GEMM configuration for (limbs, quarters)
// (dd 64 x 32, qd 32 x 32 -- 64 x 32 with the 11 / 12 wide slices of MD_OPT_SLICE_BITS, whose accumulators leave room for
// four 8x8 tiles per warp: qgemm_packed.cu; od 32 x 16, hd 32 x 16 -- 16 x 16 in 44 wide slices: qgemm_wide.cu).
// small = the 32 x 16 tile instance of the double-double kernel that md_gemm picks when the 64 x 32 tiles would not fill the
// SMs (qgemm_packed.cu: PCfgDDS); every other format ignores it.
__host__ __device__ constexpr int pack_bx(int limbs, int quarters, int axis, bool small = false) {
  return (small && limbs == 2) ? (axis == 0 ? 32 : 16)
         : (limbs == 4 && quarters <= 10) ? (axis == 0 ? 64 : 16)  // quad double, chunked accumulation: 16 x 8 warp tile
         : (limbs == 2 || (limbs == 4 && quarters <= 12)) ? (axis == 0 ? 64 : 32)
         : limbs == 4 ? 32  // quad double with the paper's 16 (17, 18) quarters: 32 x 32 CTA tile, 8 x 16 warp tile
         : (limbs == 16 && quarters <= 44) ? 16 : (axis == 0 ? 32 : 16);  // hd with 64 quarters: 32 x 16, one order range at a time
}

// The GENERIC-Q instances of qgemm_wide.cu (runtime quarter / order counts, any (limbs, quarters, orders) md_gemm accepts
// that has no tuned kernel): 32 x 16 CTA tiles for double and quad double, 16 x 16 for octo double (two order ranges per
// tile), 16 x 8 for hexa double (four); k-slab depth 4.
__host__ __device__ constexpr int pack_bx_generic(int limbs, int axis) {
  return limbs == 16 ? (axis == 0 ? 16 : 8) : limbs == 8 ? 16 : (axis == 0 ? 32 : 16);
}

// doubles in the packed image of an operand with X groups and K contraction indices
__host__ __device__ inline size_t packed_doubles(int X, int K, int bx, int bk, int quarters) {
  const size_t xt = ((size_t)X + bx - 1) / bx, ks = ((size_t)K + bk - 1) / bk;
  return xt * ks * (size_t)quarters * bk * bx;
}

// offset (in doubles) of quarter q of element (x, k); KS = number of k slabs
__host__ __device__ inline size_t packed_offset(int x, int k, int q, int bx, int bk, int quarters, int KS) {
  const int xt = x / bx, xin = x % bx, ks = k / bk, kin = k % bk;
  const size_t chunk = ((size_t)xt * KS + ks) * ((size_t)quarters * bk * bx);
  return chunk + ((size_t)(q * (bk / 4) + kin / 4) * (bx / 8) + xin / 8) * 32 + (xin % 8) * 4 + (kin % 4);
}

}  // namespace md
