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
