// md_arith.cuh -- scalar multiple-double arithmetic on the regular FP64 cores, for the parts of md_qr that are not matrix
// products (column norms, reflector scalars, rank-1 updates inside a panel; qr.cu).  An L-limb multiple double is an array of L
// doubles, leading limb first.  Built from the error-free transformations of md_common.cuh (TwoSum; TwoProd by fma -- PAPER.md
// refs [2], [3], [15]) around the (L+1)-term accumulator of the recombination (renorm_add / renorm_finish): every operation
// cascades its exact pieces into such an accumulator and renormalises once.  CUDA path only; nothing here is shared with oracle/.
#pragma once
#include "md_common.cuh"

namespace md {

__device__ __forceinline__ void two_prod(double a, double b, double& p, double& e) {
  p = __dmul_rn(a, b);
  e = __fma_rn(a, b, -p);
}

template <int L>
__device__ __forceinline__ void mda_clear(double (&r)[L + 1]) {
#pragma unroll
  for (int l = 0; l <= L; l++) r[l] = 0.0;
}
// r += x (x an L-limb multiple double), smallest limb first
template <int L>
__device__ __forceinline__ void mda_acc(double (&r)[L + 1], const double (&x)[L], double sign = 1.0) {
#pragma unroll
  for (int l = L - 1; l >= 0; l--) renorm_add<L>(r, sign * x[l]);
}
// r += sign * a * b: partial products a_i b_j exact (TwoProd) for i + j < L, plain for i + j == L, dropped beyond
template <int L>
__device__ __forceinline__ void mda_mac(double (&r)[L + 1], const double (&a)[L], const double (&b)[L], double sign = 1.0) {
#pragma unroll
  for (int s = L; s >= 0; s--)
#pragma unroll
    for (int i = 0; i < L; i++) {
      const int j = s - i;
      if (j < 0 || j >= L) continue;
      if (s < L) {
        double p, e;
        two_prod(sign * a[i], b[j], p, e);
        renorm_add<L>(r, e);
        renorm_add<L>(r, p);
      } else {
        renorm_add<L>(r, __dmul_rn(sign * a[i], b[j]));
      }
    }
}
template <int L>
__device__ __forceinline__ void mda_add(const double (&a)[L], const double (&b)[L], double (&out)[L], double sign_b = 1.0) {
  double r[L + 1];
  mda_clear<L>(r);
  mda_acc<L>(r, a);
  mda_acc<L>(r, b, sign_b);
  renorm_finish<L>(r, out);
}
template <int L>
__device__ __forceinline__ void mda_mul(const double (&a)[L], const double (&b)[L], double (&out)[L]) {
  double r[L + 1];
  mda_clear<L>(r);
  mda_mac<L>(r, a, b);
  renorm_finish<L>(r, out);
}
// long division: L + 1 quotient digits q_i = r_0 / b_0, r -= q_i b
template <int L>
__device__ __forceinline__ void mda_div(const double (&a)[L], const double (&b)[L], double (&out)[L]) {
  double rem[L], q[L + 1];
#pragma unroll
  for (int l = 0; l < L; l++) rem[l] = a[l];
#pragma unroll
  for (int i = 0; i <= L; i++) {
    q[i] = __ddiv_rn(rem[0], b[0]);
    double qi[L], r[L + 1];
#pragma unroll
    for (int l = 0; l < L; l++) qi[l] = l == 0 ? q[i] : 0.0;
    mda_clear<L>(r);
    mda_acc<L>(r, rem);
    mda_mac<L>(r, qi, b, -1.0);
    renorm_finish<L>(r, rem);
  }
  double r[L + 1];
  mda_clear<L>(r);
#pragma unroll
  for (int i = L; i >= 0; i--) renorm_add<L>(r, q[i]);
  renorm_finish<L>(r, out);
}
// Heron's iteration from the double-precision root; a <= 0 gives 0
template <int L>
__device__ __forceinline__ void mda_sqrt(const double (&a)[L], double (&out)[L]) {
#pragma unroll
  for (int l = 0; l < L; l++) out[l] = 0.0;
  if (!(a[0] > 0.0)) return;
  double x[L];
#pragma unroll
  for (int l = 0; l < L; l++) x[l] = 0.0;
  x[0] = __dsqrt_rn(a[0]);
  int iters = 2;
  for (int l = 1; l < L; l *= 2) iters++;
  for (int it = 0; it < iters; it++) {
    double t[L], s[L];
    mda_div<L>(a, x, t);
    mda_add<L>(x, t, s);
#pragma unroll
    for (int l = 0; l < L; l++) x[l] = 0.5 * s[l];
  }
#pragma unroll
  for (int l = 0; l < L; l++) out[l] = x[l];
}

}  // namespace md
