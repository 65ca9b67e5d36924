// split.cu -- steps a1 + a2 of the hot path: exponent vectors and quarter planes (include/mdgemm.h: md_split).
//   PAPER.md:47-49 (13-bit quarters with exponents 0,-13,-26,-39), :95 (balanced = exponents on an equally spaced grid),
//   :124-142 (moving bits between parts without changing the value; zeros keep the desired exponent).
// The splitters read 8*limbs and write 8*quarters bytes per element, once, and run at the HBM roofline from a few hundred MB on
// (split_kernel 0.96, split_packed_kernel 0.95-0.98 of the measured copy peak at 4096^2: profiles/r04_split_renorm_ncu.md).  What is
// NOT HBM-bound: row_exponent_kernel (134 MB in 36 us = 3.7 TB/s at 4096^2: a block per row leaves too few loads in flight;
// 0.03 % of an md_gemm step) and the cooperative prep_coop_kernel below 1024^3, which is bound by its three grid-wide barriers
// (12 us at 256^3 for 5 MB: profiles/r04_small_sizes.md section 4).
#include <cooperative_groups.h>

#include "md_common.cuh"
#include "md_kernels.h"
#include "md_packed.cuh"
#include "md_split.cuh"
#include "qgemm_pipeline.cuh"

namespace md {
namespace {

// axis 0: one block per row of the leading limb plane.
__global__ void __launch_bounds__(256) row_exponent_kernel(int rows, int cols, const double* __restrict__ lead,
                                                           int32_t* __restrict__ exps, uint32_t* flags, int exp_lo) {
  __shared__ uint32_t warp_max[8];
  for (int row = blockIdx.x; row < rows; row += gridDim.x) {
    const double* p = lead + (size_t)row * cols;
    uint32_t mx = 0;
    for (int j = threadIdx.x; j < cols; j += blockDim.x) mx = max(mx, abs_hi32(p[j]));
    mx = __reduce_max_sync(0xffffffffu, mx);
    if ((threadIdx.x & 31) == 0) warp_max[threadIdx.x >> 5] = mx;
    __syncthreads();
    if (threadIdx.x == 0) {
      uint32_t v = warp_max[0];
#pragma unroll
      for (int w = 1; w < 8; w++) v = max(v, warp_max[w]);
      exps[row] = exponent_from_hi32(v, flags, exp_lo);
    }
    __syncthreads();
  }
}

// axis 1: a thread per column walks a chunk of rows (coalesced across the warp) and folds its maximum into exps[]
// (pre-zeroed, used as uint32 scratch); the finalize kernel turns the maxima into exponents in place.
__global__ void __launch_bounds__(256) col_max_kernel(int rows, int cols, int rows_per_block,
                                                      const double* __restrict__ lead, int32_t* exps) {
  const int col = blockIdx.x * blockDim.x + threadIdx.x;
  if (col >= cols) return;
  const int r0 = blockIdx.y * rows_per_block;
  const int r1 = min(rows, r0 + rows_per_block);
  uint32_t mx = 0;
  for (int r = r0; r < r1; r++) mx = max(mx, abs_hi32(lead[(size_t)r * cols + col]));
  if (mx) atomicMax(reinterpret_cast<unsigned int*>(exps) + col, mx);
}
__global__ void col_exponent_finalize_kernel(int cols, int32_t* exps, uint32_t* flags, int exp_lo) {
  const int col = blockIdx.x * blockDim.x + threadIdx.x;
  if (col < cols) exps[col] = exponent_from_hi32((uint32_t)exps[col], flags, exp_lo);
}

// md_split: plain [quarters][rows][cols] output.  VEC elements per thread.
template <int L, int VEC>
__global__ void __launch_bounds__(256) split_kernel(size_t rows, size_t cols, int Q, int bits, int axis,
                                                    const double* __restrict__ planes, double* __restrict__ qplanes,
                                                    const int32_t* __restrict__ exps, uint32_t* flags) {
  const size_t plane = rows * cols;
  const size_t idx = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) * VEC;
  if (idx >= plane) return;
  const size_t row = idx / cols, col = idx - row * cols;  // VEC == 2 only when cols is even: both elements in one row

  double r[VEC][L];
  if (VEC == 2) {
#pragma unroll
    for (int l = 0; l < L; l++) {
      const double2 v = *reinterpret_cast<const double2*>(planes + l * plane + idx);
      r[0][l] = v.x;
      r[VEC - 1][l] = v.y;
    }
  } else {
#pragma unroll
    for (int l = 0; l < L; l++) r[0][l] = planes[l * plane + idx];
  }
  int E[VEC];
  bool bad = false;
#pragma unroll
  for (int v = 0; v < VEC; v++) {
    E[v] = axis == 0 ? exps[row] : exps[col + v];
    bad |= any_nonfinite<L>(r[v]);
  }
  if (bad && flags) atomicOr(flags, FLAG_NONFINITE);

  for (int q = 0; q < Q; q++) {
    double d[VEC];
#pragma unroll
    for (int v = 0; v < VEC; v++) d[v] = extract_digit<L>(r[v], E[v], q, bits);
    if (VEC == 2)
      *reinterpret_cast<double2*>(qplanes + (size_t)q * plane + idx) = make_double2(d[0], d[VEC - 1]);
    else
      qplanes[(size_t)q * plane + idx] = d[0];
  }
}

// 256-bit global accesses (sm_100: LDG.E.ENL2.256 / STG.E.ENL2.256); p must be 32-byte aligned.  A fragment row of the
// packed layout is 4 doubles, so one store per quarter per thread fills whole 32-byte sectors (two 16-byte stores at a
// 32-byte lane stride half-fill 32 sectors each and made the kernel L1-bound at 0.55 of the HBM peak in an earlier capture).
__device__ __forceinline__ void ldg_256(const double* p, double& a, double& b, double& c, double& d) {
  asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p));
}
__device__ __forceinline__ void stg_256(double* p, double a, double b, double c, double d) {
  asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}

// md_gemm's splitter: same digits, written in the fragment-major packed layout of md_packed.cuh (zero padded to whole
// tiles and k-slabs).  A thread owns one fragment row: group x (row of A, AXIS 0 / column of B, AXIS 1) and the four
// contraction indices k = 4*k4g .. 4*k4g+3, i.e. 32 contiguous output bytes per quarter; the 32 lanes of a warp take 32
// consecutive x, so a warp writes 1 KB contiguous per quarter (and, for B, reads 256 contiguous bytes per row).
// One fragment row of the packed layout: group x (row of A, AXIS 0 / column of B, AXIS 1), contraction indices k0 .. k0+3,
// all Q slices.  E = the group's exponent.  Zero padding outside the matrix.
template <int L, int AXIS>
__device__ __forceinline__ void split_fragment_row(int rows, int cols, int Q, int bits, int bx, int bk, int KS, int x, int k0,
                                                   int E, const double* __restrict__ planes, double* __restrict__ packed,
                                                   uint32_t* flags) {
  const int X = AXIS == 0 ? rows : cols, K = AXIS == 0 ? cols : rows;
  const size_t plane = (size_t)rows * cols;
  double r[4][L];
  const bool x_ok = x < X;
  if (AXIS == 0) {
    // rows of every limb plane 32-byte aligned -> one 256-bit load per limb (k0 is a multiple of 4)
    const bool vec = x_ok && (k0 + 4 <= K) && (cols % 4 == 0) && ((reinterpret_cast<uintptr_t>(planes) & 31) == 0);
    const double* src = planes + (size_t)(x_ok ? x : 0) * cols + k0;
#pragma unroll
    for (int l = 0; l < L; l++) {
      if (vec) {
        ldg_256(src + l * plane, r[0][l], r[1][l], r[2][l], r[3][l]);
      } else {
#pragma unroll
        for (int t = 0; t < 4; t++) r[t][l] = (x_ok && k0 + t < K) ? src[l * plane + t] : 0.0;
      }
    }
  } else {
#pragma unroll
    for (int l = 0; l < L; l++)
#pragma unroll
      for (int t = 0; t < 4; t++)
        r[t][l] = (x_ok && k0 + t < K) ? planes[l * plane + (size_t)(k0 + t) * cols + x] : 0.0;
  }
  bool bad = false;
#pragma unroll
  for (int t = 0; t < 4; t++) bad |= any_nonfinite<L>(r[t]);
  if (bad && flags) atomicOr(flags, FLAG_NONFINITE);

  // element (x, k0) of quarter 0; quarter q is q * (BK/4) * (bx/8) fragments further
  double* dst = packed + packed_offset(x, k0, 0, bx, bk, Q, KS);
  const size_t q_stride = (size_t)(bk / 4) * (bx / 8) * 32;
  for (int q = 0; q < Q; q++) {
    double d[4];
#pragma unroll
    for (int t = 0; t < 4; t++) d[t] = extract_digit<L>(r[t], E, q, bits);
    stg_256(dst + q * q_stride, d[0], d[1], d[2], d[3]);  // a fragment row; the warp writes 1 KB contiguous
  }
}

// md_gemm's splitter: same digits, written in the fragment-major packed layout of md_packed.cuh (zero padded to whole
// tiles and k-slabs).  A thread owns one fragment row: group x and the four contraction indices k = 4*k4g .. 4*k4g+3, i.e.
// 32 contiguous output bytes per quarter; the 32 lanes of a warp take 32 consecutive x, so a warp writes 1 KB contiguous
// per quarter (and, for B, reads 256 contiguous bytes per row).
template <int L, int AXIS>
__global__ void __launch_bounds__(256) split_packed_kernel(int rows, int cols, int Q, int bits, int bx, int bk, int x_blocks, int KS,
                                                           const double* __restrict__ planes,
                                                           double* __restrict__ packed,
                                                           const int32_t* __restrict__ exps, uint32_t* flags) {
  const int X = AXIS == 0 ? rows : cols;
  const int x = (blockIdx.x % x_blocks) * 32 + (threadIdx.x & 31);
  const int k4g = (blockIdx.x / x_blocks) * 8 + (threadIdx.x >> 5);  // group of four k
  const int XP = (X + bx - 1) / bx * bx;                             // padded to whole tiles
  if (k4g >= KS * (bk / 4) || x >= XP) return;
  split_fragment_row<L, AXIS>(rows, cols, Q, bits, bx, bk, KS, x, k4g * 4, x < X ? exps[x] : 0, planes, packed, flags);
}

// md_qgemm's repacking (quarter / order counts without a plain-layout kernel): plain [Q][rows][cols] quarter planes -> the packed
// layout, zero padded.  Same thread mapping as split_packed_kernel; no arithmetic.
template <int AXIS>
__global__ void __launch_bounds__(256) pack_planes_kernel(int rows, int cols, int Q, int bx, int bk, int x_blocks, int KS,
                                                          const double* __restrict__ planes, double* __restrict__ packed) {
  const int X = AXIS == 0 ? rows : cols, K = AXIS == 0 ? cols : rows;
  const int x = (blockIdx.x % x_blocks) * 32 + (threadIdx.x & 31);
  const int k4g = (blockIdx.x / x_blocks) * 8 + (threadIdx.x >> 5);
  const int XP = (X + bx - 1) / bx * bx;
  if (k4g >= KS * (bk / 4) || x >= XP) return;
  const int k0 = k4g * 4;
  const size_t plane = (size_t)rows * cols;
  double* dst = packed + packed_offset(x, k0, 0, bx, bk, Q, KS);
  const size_t q_stride = (size_t)(bk / 4) * (bx / 8) * 32;
  for (int q = 0; q < Q; q++) {
    double d[4];
#pragma unroll
    for (int t = 0; t < 4; t++) {
      const bool ok = x < X && k0 + t < K;
      d[t] = !ok ? 0.0 : AXIS == 0 ? planes[q * plane + (size_t)x * cols + k0 + t] : planes[q * plane + (size_t)(k0 + t) * cols + x];
    }
    stg_256(dst + q * q_stride, d[0], d[1], d[2], d[3]);
  }
}

// md_gemm's fused preparation: exponent vectors AND packed quarter planes of BOTH operands in ONE cooperative launch (the
// dependent launches of the separate kernels -- row maxima, column maxima, finalize, two splits, a memset -- cost a few
// microseconds each, which is a third of a 64^3 product and 2.5 % of a 1024^3 one).  Persistent blocks, three phases
// separated by grid-wide barriers: (0) clear the maxima, (1) fold the hi-32-bit maxima of the leading limb planes into
// rawA[m] / rawB[n] (the same maxima as the separate exponent kernels), (2) split, a block per (32 groups x 32 contraction
// indices) item exactly as split_packed_kernel, the exponent taken from the raw maximum on the fly.  rawA / rawB keep the
// raw maxima (md_gemm never reads the exponent vectors back).  Identical digits.
template <int L>
__global__ void __launch_bounds__(256) prep_coop_kernel(int m, int n, int k, int Q, int bits, int bxA, int bxB, int bk,
                                                        const double* __restrict__ A, const double* __restrict__ B,
                                                        double* __restrict__ Ap, double* __restrict__ Bp, uint32_t* rawA,
                                                        uint32_t* rawB, uint32_t* flags, int exp_lo, uint32_t* zero_words,
                                                        int zero_count) {
  cooperative_groups::grid_group grid = cooperative_groups::this_grid();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int gthreads = gridDim.x * blockDim.x, gtid = blockIdx.x * blockDim.x + threadIdx.x;
  for (int i = gtid; i < m; i += gthreads) rawA[i] = 0;
  for (int i = gtid; i < n; i += gthreads) rawB[i] = 0;
  // the hand-over flags of the fused GEMM that follows on the stream (qgemm_packed.cu) start at zero: cleared here instead of
  // by a memset node between the two kernels
  for (int i = gtid; i < zero_count; i += gthreads) zero_words[i] = 0;
  grid.sync();
  // phase 1a: rows of A_0 in pieces of 1024 elements, a warp per piece, lanes along the row (coalesced)
  {
    const int pieces = (k + 1023) / 1024;
    const long long items = (long long)m * pieces;
    for (long long it = (long long)blockIdx.x * 8 + warp; it < items; it += (long long)gridDim.x * 8) {
      const int row = (int)(it / pieces), k0 = (int)(it % pieces) * 1024, k1 = min(k, k0 + 1024);
      const double* p = A + (size_t)row * k;
      uint32_t mx = 0;
      for (int t = k0 + lane; t < k1; t += 32) mx = max(mx, abs_hi32(p[t]));
      mx = __reduce_max_sync(0xffffffffu, mx);
      if (lane == 0 && mx) atomicMax(&rawA[row], mx);
    }
  }
  // phase 1b: columns of B_0, 256 consecutive columns x 32 rows per block item (coalesced across the block)
  {
    const int cblocks = (n + 255) / 256, rblocks = (k + 31) / 32;
    const long long items = (long long)cblocks * rblocks;
    for (long long it = blockIdx.x; it < items; it += gridDim.x) {
      const int col = (int)(it % cblocks) * 256 + threadIdx.x, r0 = (int)(it / cblocks) * 32, r1 = min(k, r0 + 32);
      if (col < n) {
        uint32_t mx = 0;
        for (int r = r0; r < r1; r++) mx = max(mx, abs_hi32(B[(size_t)r * n + col]));
        if (mx) atomicMax(&rawB[col], mx);
      }
    }
  }
  grid.sync();
  // every block of this kernel is resident and past its last grid-wide barrier: the fused GEMM that md_gemm enqueues behind it
  // (launched with programmatic stream serialization, qgemm_packed.cu) may start its CTAs -- barrier set-up, segment tables --
  // on SMs with room; it waits for THIS grid to complete before it reads a quarter plane
  grid_launch_dependents();
  // phase 2: split, A then B
  const int KS = (k + bk - 1) / bk, k4_groups = KS * (bk / 4), k_blocks = (k4_groups + 7) / 8;
  const int XPA = (m + bxA - 1) / bxA * bxA, XPB = (n + bxB - 1) / bxB * bxB;
  const int xbA = (XPA + 31) / 32, xbB = (XPB + 31) / 32;
  const long long itemsA = (long long)xbA * k_blocks, itemsB = (long long)xbB * k_blocks;
  for (long long it = blockIdx.x; it < itemsA + itemsB; it += gridDim.x) {
    const bool isA = it < itemsA;
    const long long j = isA ? it : it - itemsA;
    const int xb = isA ? xbA : xbB;
    const int x = (int)(j % xb) * 32 + lane, kb = (int)(j / xb), k4g = kb * 8 + warp;
    const int X = isA ? m : n, XP = isA ? XPA : XPB;
    if (k4g >= k4_groups || x >= XP) continue;
    int E = 0;
    if (x < X) E = exponent_from_hi32(isA ? rawA[x] : rawB[x], kb == 0 && warp == 0 ? flags : nullptr, exp_lo);
    if (isA) split_fragment_row<L, 0>(m, k, Q, bits, bxA, bk, KS, x, k4g * 4, E, A, Ap, flags);
    else split_fragment_row<L, 1>(k, n, Q, bits, bxB, bk, KS, x, k4g * 4, E, B, Bp, flags);
  }
}

}  // namespace

// Lowest group exponent at which every kept quarter product 2^(E_i + F_j - W(s+2)), s < quarters, is still a normal
// double when both groups sit at the bound; -EXP_LIMIT for the paper's dd / qd quarter counts.
int exponent_floor(int quarters, int bits) {
  const int lo = -(1022 - bits * (quarters + 1)) / 2;
  const int pair = bits * quarters <= 13 * 24 || lo < -EXP_LIMIT ? -EXP_LIMIT : lo;
  // and every digit unit 2^(E - W (q+1)), q < quarters, must itself be a normal double (the splitter's constant c needs it)
  const int own = bits * quarters - 1022;
  return pair > own ? pair : own;
}

cudaError_t launch_exponents(int rows, int cols, int axis, int quarters, int bits, const double* lead, int32_t* exps,
                             uint32_t* flags, cudaStream_t stream, uint64_t* launches) {
  const int exp_lo = exponent_floor(quarters, bits);
  if (axis == 0) {
    const int sms = max(sm_count(), 1);
    row_exponent_kernel<<<min(rows, sms * 64), 256, 0, stream>>>(rows, cols, lead, exps, flags, exp_lo);
    *launches += 1;
    return cudaGetLastError();
  }
  cudaError_t err = cudaMemsetAsync(exps, 0, sizeof(int32_t) * (size_t)cols, stream);
  if (err != cudaSuccess) return err;
  const int col_blocks = (cols + 255) / 256;
  // enough row chunks to fill the machine, at least 16 rows each
  int chunks = max(1, min((rows + 15) / 16, (max(sm_count(), 1) * 8 + col_blocks - 1) / col_blocks));
  chunks = min(chunks, 65535);
  const int rows_per_block = (rows + chunks - 1) / chunks;
  chunks = (rows + rows_per_block - 1) / rows_per_block;
  col_max_kernel<<<dim3(col_blocks, chunks), 256, 0, stream>>>(rows, cols, rows_per_block, lead, exps);
  if ((err = cudaGetLastError()) != cudaSuccess) return err;
  col_exponent_finalize_kernel<<<col_blocks, 256, 0, stream>>>(cols, exps, flags, exp_lo);
  *launches += 2;
  return cudaGetLastError();
}

cudaError_t launch_split(int rows, int cols, int limbs, int quarters, int bits, int axis, const double* planes,
                         double* qplanes, const int32_t* exps, uint32_t* flags, cudaStream_t stream,
                         uint64_t* launches) {
  const size_t total = (size_t)rows * cols;
  const bool vec = (cols % 2 == 0) && ((reinterpret_cast<uintptr_t>(planes) | reinterpret_cast<uintptr_t>(qplanes)) % 16 == 0);
  const size_t threads = vec ? total / 2 : total;
  const unsigned blocks = (unsigned)((threads + 255) / 256);
#define MD_SPLIT(L_)                                                                                              \
  if (vec) split_kernel<L_, 2><<<blocks, 256, 0, stream>>>(rows, cols, quarters, bits, axis, planes, qplanes, exps, flags); \
  else split_kernel<L_, 1><<<blocks, 256, 0, stream>>>(rows, cols, quarters, bits, axis, planes, qplanes, exps, flags);
  switch (limbs) {
    case 1: MD_SPLIT(1) break;
    case 2: MD_SPLIT(2) break;
    case 4: MD_SPLIT(4) break;
    case 8: MD_SPLIT(8) break;
    case 16: MD_SPLIT(16) break;
    default: return cudaErrorInvalidValue;
  }
#undef MD_SPLIT
  *launches += 1;
  return cudaGetLastError();
}

cudaError_t launch_prep_packed(int m, int n, int k, int limbs, int quarters, int bits, int bxA, int bxB, int bk, const double* A,
                               const double* B, double* Ap, double* Bp, int32_t* expA, int32_t* expB, uint32_t* flags,
                               void* sk_counters, cudaStream_t stream, uint64_t* launches) {
  int exp_lo = exponent_floor(quarters, bits);
  uint32_t* zero_words = static_cast<uint32_t*>(sk_counters);
  int zero_count = sk_counters ? (int)(SK_COUNTER_BYTES / sizeof(uint32_t)) : 0;
  uint32_t* rawA = reinterpret_cast<uint32_t*>(expA);
  uint32_t* rawB = reinterpret_cast<uint32_t*>(expB);
  void* args[] = {&m, &n, &k, &quarters, &bits, &bxA, &bxB, &bk, &A, &B, &Ap, &Bp, &rawA, &rawB, &flags, &exp_lo, &zero_words, &zero_count};
  const void* kern = nullptr;
  switch (limbs) {
    case 2: kern = reinterpret_cast<const void*>(prep_coop_kernel<2>); break;
    case 4: kern = reinterpret_cast<const void*>(prep_coop_kernel<4>); break;
    case 8: kern = reinterpret_cast<const void*>(prep_coop_kernel<8>); break;
    case 16: kern = reinterpret_cast<const void*>(prep_coop_kernel<16>); break;
    default: return cudaErrorInvalidValue;
  }
  // persistent grid: as many blocks as can be co-resident (a cooperative launch needs that), at most the work there is
  static int max_blocks_dev[MD_MAX_DEVICES][17] = {};  // per device: a process may drive several
  const int dev = current_device();
  if (dev < 0 || dev >= MD_MAX_DEVICES) return cudaErrorInvalidDevice;
  int* max_blocks = max_blocks_dev[dev];
  if (max_blocks[limbs] == 0) {
    int per_sm = 0;
    const int sms = sm_count();
    cudaError_t e = sms > 0 ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, 256, 0) : cudaErrorInvalidDevice;
    if (e != cudaSuccess) return e;
    if (per_sm > 4) per_sm = 4;
    max_blocks[limbs] = sms * (per_sm > 0 ? per_sm : 1);
  }
  const long long KS = ((long long)k + bk - 1) / bk, k_blocks = (KS * (bk / 4) + 7) / 8;
  long long work = (((long long)m + bxA - 1) / bxA * bxA + 31) / 32 * k_blocks + (((long long)n + bxB - 1) / bxB * bxB + 31) / 32 * k_blocks;
  int blocks = (int)(work < max_blocks[limbs] ? (work > 0 ? work : 1) : max_blocks[limbs]);
  const cudaError_t err = cudaLaunchCooperativeKernel(kern, dim3(blocks), dim3(256), args, 0, stream);
  if (err == cudaSuccess) *launches += 1;
  return err;
}

cudaError_t launch_pack_planes(int rows, int cols, int quarters, int axis, int bx, int bk, const double* planes, double* packed,
                               cudaStream_t stream, uint64_t* launches) {
  const int X = axis == 0 ? rows : cols, K = axis == 0 ? cols : rows;
  const int KS = (K + bk - 1) / bk;
  const int x_blocks = ((X + bx - 1) / bx * bx + 31) / 32;
  const long long blocks = (long long)x_blocks * (((long long)KS * (bk / 4) + 7) / 8);
  if (blocks > 0x7fffffffLL) return cudaErrorInvalidValue;
  if (axis == 0) pack_planes_kernel<0><<<(unsigned)blocks, 256, 0, stream>>>(rows, cols, quarters, bx, bk, x_blocks, KS, planes, packed);
  else pack_planes_kernel<1><<<(unsigned)blocks, 256, 0, stream>>>(rows, cols, quarters, bx, bk, x_blocks, KS, planes, packed);
  *launches += 1;
  return cudaGetLastError();
}

cudaError_t launch_split_packed(int rows, int cols, int limbs, int quarters, int bits, int axis, int bx, int bk,
                                const double* planes, double* packed, const int32_t* exps, uint32_t* flags,
                                cudaStream_t stream, uint64_t* launches) {
  const int X = axis == 0 ? rows : cols, K = axis == 0 ? cols : rows;
  const int KS = (K + bk - 1) / bk;
  const int x_blocks = ((X + bx - 1) / bx * bx + 31) / 32;  // 32 groups per block over the padded extent
  const long long k_blocks = ((long long)KS * (bk / 4) + 7) / 8;
  const long long blocks = (long long)x_blocks * k_blocks;
  if (blocks > 0x7fffffffLL) return cudaErrorInvalidValue;
#define MD_SPLITP(L_, AX_)                                                                                           \
  split_packed_kernel<L_, AX_><<<(unsigned)blocks, 256, 0, stream>>>(rows, cols, quarters, bits, bx, bk, x_blocks, KS, planes, \
                                                                     packed, exps, flags)
  if (limbs == 2 && axis == 0) MD_SPLITP(2, 0);
  else if (limbs == 2 && axis == 1) MD_SPLITP(2, 1);
  else if (limbs == 4 && axis == 0) MD_SPLITP(4, 0);
  else if (limbs == 4 && axis == 1) MD_SPLITP(4, 1);
  else if (limbs == 8 && axis == 0) MD_SPLITP(8, 0);
  else if (limbs == 8 && axis == 1) MD_SPLITP(8, 1);
  else if (limbs == 16 && axis == 0) MD_SPLITP(16, 0);
  else if (limbs == 16 && axis == 1) MD_SPLITP(16, 1);
  else return cudaErrorInvalidValue;
#undef MD_SPLITP
  *launches += 1;
  return cudaGetLastError();
}

}  // namespace md
