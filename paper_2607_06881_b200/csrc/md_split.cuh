// md_split.cuh -- the per-element arithmetic of steps a1 + a2 (exponent of a group from the maximum of its leading limbs;
// Algorithm S digit extraction), shared by the stand-alone splitters (split.cu) and by the fused single-launch kernel for
// small problems (fused_small.cu), so that both produce the same bits.  CUDA path only; nothing here is shared with oracle/.
#pragma once
#include "md_common.cuh"

namespace md {

__device__ __forceinline__ uint32_t abs_hi32(double x) { return (uint32_t)(__double_as_longlong(x) >> 32) & 0x7fffffffu; }

// hi32 of the group maximum -> E = ilogb(max)+1 (0 for a zero group); flags out-of-range / non-finite maxima.
__device__ __forceinline__ int exponent_from_hi32(uint32_t hi, uint32_t* flags, int exp_lo) {
  const int biased = (int)(hi >> 20);
  if (biased == 0) return 0;  // zero group (subnormal maxima are outside the documented range and count as zero)
  const int E = biased - 1022;
  if (flags) {
    if (biased == 0x7ff) atomicOr(flags, FLAG_NONFINITE);
    else if (E < exp_lo || E > EXP_LIMIT) atomicOr(flags, FLAG_EXP_RANGE);
  }
  return E;
}

// Algorithm S, step S1 (DESIGN.md section 3 R4): digit q of the element whose remainder limbs are r[0..L-1], group exponent E:
//   c = 3*2^51 * u_q (so that ulp(c) = u_q = 2^(E - W(q+1)));  d_q = (r_0 + c) - c;  r_0 -= d_q;  carry r through the limbs.
// Every operation is exact except r_0 + c, whose rounding IS the digit selection.  W = `bits`, the slice width: 13 for the
// paper's quarters, other widths under MD_OPT_SLICE_BITS (R14).
template <int L>
__device__ __forceinline__ double extract_digit(double (&r)[L], int E, int q, int bits) {
  // c = 1.5 * 2^(E - W(q+1) + 52): exponent field + the top mantissa bit
  // (a group exponent below the documented floor would make the field non-positive: clamped, the digit is then garbage
  // but finite and the violation is flagged by the exponent kernel)
  const long long field = max(E - bits * (q + 1) + 52 + 1023, 1);
  const double c = __longlong_as_double((field << 52) | (1ll << 51));
  const double t = __dadd_rn(r[0], c);
  const double d = __dsub_rn(t, c);
  r[0] = __dsub_rn(r[0], d);
#pragma unroll
  for (int l = 0; l + 1 < L; l++) two_sum(r[l], r[l + 1], r[l], r[l + 1]);
  return d;
}

template <int L>
__device__ __forceinline__ bool any_nonfinite(const double (&r)[L]) {
  bool bad = false;
#pragma unroll
  for (int l = 0; l < L; l++) bad |= (abs_hi32(r[l]) >> 20) == 0x7ffu;
  return bad;
}

}  // namespace md
