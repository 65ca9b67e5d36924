// md_common.cuh -- device helpers shared by the kernels of libmdgemm (the CUDA path).  Nothing here is shared with
// oracle/ (the CPU oracle has its own, independent code).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace md {

// Status-word bits (include/mdgemm.h, md_read_flags)
constexpr uint32_t FLAG_NONFINITE = 1u;
constexpr uint32_t FLAG_EXP_RANGE = 2u;
constexpr int EXP_LIMIT = 900;

// --- error-free transformations; explicit _rn intrinsics so that nothing is ever contracted or re-associated -----------
// TwoSum (Knuth; PAPER.md refs [2],[15]): s + e == a + b exactly, s = fl(a + b).  6 flops, no branch.
__device__ __forceinline__ void two_sum(double a, double b, double& s, double& e) {
  s = __dadd_rn(a, b);
  const double bb = __dsub_rn(s, a);
  e = __dadd_rn(__dsub_rn(a, __dsub_rn(s, bb)), __dsub_rn(b, bb));
}
// FastTwoSum (Dekker): same, 3 flops, needs |a| >= |b| (or a == 0).
__device__ __forceinline__ void fast_two_sum(double a, double b, double& s, double& e) {
  s = __dadd_rn(a, b);
  e = __dsub_rn(b, __dsub_rn(s, a));
}

// 2^e as a double, e in the normal range.
__device__ __forceinline__ double pow2(int e) { return __longlong_as_double((long long)(e + 1023) << 52); }

// ----------------------------------------------------------------------------------------------------------------------
// Recombination (step a4; "summing 8 doubles into one double double for each element ... in double
// double arithmetic"; R9).  c[0..S-1] are the order values C^(s)_ij, roughly decreasing by 2^-13 per order but
// overlapping heavily.  They are added from the smallest order to the largest into an (L+1)-term accumulator by a
// TwoSum cascade (each step is error free except the last term, which is a plain add far below the L-th limb), then two
// kinds of error-free sweeps bring the accumulator to a non-overlapping expansion: limb_{l} = fl(limb_l + limb_{l+1}).
// Error: <= 2^-(53L+40) * sum|c| from the guard term + what the dropped (L+1)-th term holds (< 2^-53L |sum|).
// ----------------------------------------------------------------------------------------------------------------------
// The three pieces of renorm_orders, usable separately (the standalone kernel streams the orders from memory; the hexa
// double GEMM hands the (L+1)-term accumulator from warp to warp, qgemm_wide.cu).  r has L+1 terms, starts at zero.
template <int L>
__device__ __forceinline__ void renorm_add(double (&r)[L + 1], double x) {
#pragma unroll
  for (int l = 0; l < L; l++) two_sum(r[l], x, r[l], x);
  r[L] = __dadd_rn(r[L], x);
}
// renorm_add for the TWO elements a thread owns in a DMMA tile, interleaved (two independent dependency chains side by side:
// a cascade is 5 L dependent additions long and latency-bound on its own), and cut short once there is nothing left to carry
// down: after a group of four levels, if the carried term of BOTH elements is zero in EVERY lane of the warp, the remaining
// TwoSums would add zero to their terms and are skipped.  Same values as two calls of renorm_add (a skipped TwoSum(r, 0) returns
// (r, 0)); the orders arrive smallest first, so the early ones occupy only the top few terms of the 17-term accumulator of a
// hexa double and most of the cascade moved zeros.  All 32 lanes must call it together.
template <int L>
__device__ __forceinline__ void renorm_add2(double (&r0)[L + 1], double (&r1)[L + 1], double x0, double x1) {
#pragma unroll
  for (int g = 0; g < L; g += 4) {
#pragma unroll
    for (int l = g; l < g + 4 && l < L; l++) {
      two_sum(r0[l], x0, r0[l], x0);
      two_sum(r1[l], x1, r1[l], x1);
    }
    if (g + 4 < L && __all_sync(0xffffffffu, x0 == 0.0 && x1 == 0.0)) return;
  }
  r0[L] = __dadd_rn(r0[L], x0);
  r1[L] = __dadd_rn(r1[L], x1);
}
// N CONSECUTIVE orders (x[0] first) into both elements: order i runs i levels behind order 0 -- at step t order i adds into
// r[t - i], which order i - 1 has left one step earlier -- so every term still receives the orders in their sequence, the values
// are those of N calls of renorm_add2, and 2 N independent TwoSum chains are in flight instead of two (a TwoSum level is five
// dependent additions; the recombination of a hexa double is latency-bound on exactly that chain).  x[i][e]: order i, element e.
template <int L, int N>
__device__ __forceinline__ void renorm_add2xN(double (&r0)[L + 1], double (&r1)[L + 1], double (&x)[N][2]) {
#pragma unroll
  for (int g = 0; g < L + N - 1; g += 4) {
#pragma unroll
    for (int t = g; t < g + 4 && t < L + N - 1; t++) {
#pragma unroll
      for (int i = 0; i < N; i++) {
        const int l = t - i;
        if (l >= 0 && l < L) {
          two_sum(r0[l], x[i][0], r0[l], x[i][0]);
          two_sum(r1[l], x[i][1], r1[l], x[i][1]);
        }
      }
    }
    if (g + 4 < L + N - 1) {
      bool zero = true;
#pragma unroll
      for (int i = 0; i < N; i++) zero = zero && x[i][0] == 0.0 && x[i][1] == 0.0;
      if (__all_sync(0xffffffffu, zero)) return;
    }
  }
#pragma unroll
  for (int i = 0; i < N; i++) {
    r0[L] = __dadd_rn(r0[L], x[i][0]);
    r1[L] = __dadd_rn(r1[L], x[i][1]);
  }
}
template <int L>
__device__ __forceinline__ void renorm_finish(double (&r)[L + 1], double (&out)[L]) {
  // bottom-up: r[0] becomes fl(total), the rest the successive rounding errors
#pragma unroll
  for (int l = L; l >= 1; l--) two_sum(r[l - 1], r[l], r[l - 1], r[l]);
  // top-down sweeps: each makes r[l] = fl(r[l] + r[l+1]) and pushes the error (and interior zeros) one place down.
  // Not unrolled for the wide formats (L*L TwoSums: 1536 instructions at L = 16); same operations either way.
#pragma unroll(L <= 4 ? L : 1)
  for (int sweep = 0; sweep < L; sweep++) {
#pragma unroll
    for (int l = 0; l < L; l++) two_sum(r[l], r[l + 1], r[l], r[l + 1]);
  }
#pragma unroll
  for (int l = 0; l < L; l++) out[l] = r[l];
}

// renorm_finish for two elements, interleaved (same operations per element)
template <int L>
__device__ __forceinline__ void renorm_finish2(double (&r0)[L + 1], double (&r1)[L + 1], double (&out0)[L], double (&out1)[L]) {
#pragma unroll
  for (int l = L; l >= 1; l--) {
    two_sum(r0[l - 1], r0[l], r0[l - 1], r0[l]);
    two_sum(r1[l - 1], r1[l], r1[l - 1], r1[l]);
  }
#pragma unroll(L <= 4 ? L : 1)
  for (int sweep = 0; sweep < L; sweep++) {
#pragma unroll
    for (int l = 0; l < L; l++) {
      two_sum(r0[l], r0[l + 1], r0[l], r0[l + 1]);
      two_sum(r1[l], r1[l + 1], r1[l], r1[l + 1]);
    }
  }
#pragma unroll
  for (int l = 0; l < L; l++) out0[l] = r0[l], out1[l] = r1[l];
}

template <int L, int S>
__device__ __forceinline__ void renorm_orders(const double (&c)[S], double (&out)[L]) {
  double r[L + 1];
#pragma unroll
  for (int l = 0; l <= L; l++) r[l] = 0.0;
#pragma unroll
  for (int s = S - 1; s >= 0; s--) renorm_add<L>(r, c[s]);
  renorm_finish<L>(r, out);
}

}  // namespace md
