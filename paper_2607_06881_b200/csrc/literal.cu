// literal.cu -- the paper's OWN balancing (section 3) as a second split mode of libmdgemm
// (include/mdgemm.h: md_split_literal, md_gemm_literal; R17-R22).
//
// md_gemm gives a row of A / a column of B a common exponent.  Section 3 of the paper works element by element instead:
//   * every double is cut into 13-bit parts relative to ITS OWN exponent;
//   * eq. (7): a low double of the opposite sign takes one ulp from the high double;
//   * eq. (8): a part with leading zeros borrows half a unit from the part above; zero parts "do nothing"
//     (PAPER.md:142);
//   * A = A_0 + ... + A_12 by the exponent of the leading quarter modulo 13, "execute many matrix multiplications"
//     (PAPER.md:120-122); optionally A = A_+ + A_- (eq. 6).
// Here: Algorithm L (the three per-element steps, the same floating-point operations as oracle_split_literal, hence the same
// bits), a statistics kernel (level range and class populations), a splitter that writes ONE class (x sign) of an operand as
// packed quarter planes on the class's common grid, the class-pair products on the fused quarter-GEMM kernels the rest of the
// library uses (a class pair is an ordinary quarter GEMM), and the accumulation of all order sums into C.
#include <cstdint>

#include "../../include/mdgemm.h"
#include "api_internal.h"
#include "md_common.cuh"
#include "md_kernels.h"
#include "md_packed.cuh"

namespace md {
namespace {

constexpr int GROUPS = 26;  // class c = e mod 13 for a positive element, 13 + c for a negative one

__device__ __forceinline__ int floor_div13(int e) { return e >= 0 ? e / 13 : -((-e + 12) / 13); }
__device__ __forceinline__ int mod13(int e) { return e - 13 * floor_div13(e); }

// Algorithm L on one element, as a stream of parts (R17-R19).  The same operations in the same order as
// oracle_split_literal_element, so the parts are bit-identical: eq. (7) by TwoSum carries, the parts by truncating what is
// left of every limb at the part's unit (ldexp / trunc: exact), eq. (8) top down with one part of look-ahead.
template <int L>
struct LiteralElement {
  double x[L];  // what is left of the limbs
  int e;        // exponent of the element = ilogb of its leading non-zero limb after eq. (7)
  bool zero, negative;
  double cur;   // part `q`, extracted and possibly topped up by eq. (8), not yet handed out
  int q;

  __device__ __forceinline__ double extract(int part) {
    const int s = e - 13 * (part + 1);
    double sum = 0.0;
#pragma unroll
    for (int l = 0; l < L; l++) {
      const double piece = ldexp(trunc(ldexp(x[l], -s)), s);  // the bits of limb l at or above 2^s
      x[l] = __dsub_rn(x[l], piece);                           // exact
      sum = __dadd_rn(sum, piece);                             // exact: multiples of 2^s below 2^(s + 14)
    }
    return sum;
  }

  __device__ __forceinline__ void init(const double (&limbs)[L]) {
#pragma unroll
    for (int l = 0; l < L; l++) x[l] = limbs[l];
    // eq. (7) (R18): b = the smallest power of two >= one ulp of the upper limb that exceeds |lower|
#pragma unroll
    for (int l = 0; l + 1 < L; l++) {
      if (x[l] == 0.0 || x[l + 1] == 0.0 || ((x[l] < 0) == (x[l + 1] < 0))) continue;
      double mag = ldexp(1.0, ilogb(x[l]) - 52);
      const double above = ldexp(1.0, ilogb(x[l + 1]) + 1);
      if (above > mag) mag = above;
      if (mag > 0.5 * fabs(x[l])) continue;
      const double b = copysign(mag, x[l]);
      x[l] = __dsub_rn(x[l], b);
      double c = b;
#pragma unroll
      for (int j = l + 1; j < L; j++) two_sum(x[j], c, x[j], c);  // what falls off the last limb is part of the remainder
    }
    double leadv = 0.0;  // the leading non-zero limb
#pragma unroll
    for (int l = 0; l < L; l++)
      if (leadv == 0.0) leadv = x[l];
    zero = leadv == 0.0;
    e = zero ? 0 : ilogb(leadv);
    negative = leadv < 0;
    q = 0;
    cur = zero ? 0.0 : extract(0);
  }

  // part q (final) and advance; Q = parts per element; eq8: apply eq. (8) with the zero rule (:142)
  __device__ __forceinline__ double next(int Q, bool eq8) {
    if (zero) return 0.0;
    double out = cur;
    if (q + 1 < Q) {
      double nxt = extract(q + 1);
      if (eq8) {
        const double top = 4096.0 * ldexp(1.0, e - 13 * (q + 2));  // 2^12 units of part q + 1 = half a unit of part q
        if (nxt != 0.0 && fabs(nxt) < top && cur != 0.0 && ((cur < 0) == (nxt < 0)) && (q == 0 || fabs(cur) > 2.0 * top * 4096.0)) {
          const double b = copysign(top, cur);
          out = __dsub_rn(cur, b);
          nxt = __dadd_rn(nxt, b);
        }
      }
      cur = nxt;
    }
    q++;
    return out;
  }
};

template <int L>
__device__ __forceinline__ bool limbs_nonfinite(const double (&r)[L]) {
  bool bad = false;
#pragma unroll
  for (int l = 0; l < L; l++) bad |= ((uint32_t)(__double_as_longlong(r[l]) >> 52) & 0x7ffu) == 0x7ffu;
  return bad;
}

// md_split_literal: plain [quarters][rows][cols] parts + one exponent per ELEMENT.
template <int L>
__global__ void __launch_bounds__(256) literal_split_kernel(size_t total, int Q, int eq8, const double* __restrict__ planes,
                                                            double* __restrict__ qplanes, int32_t* __restrict__ exps, uint32_t* flags) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= total) return;
  double r[L];
#pragma unroll
  for (int l = 0; l < L; l++) r[l] = planes[l * total + idx];
  if (flags && limbs_nonfinite<L>(r)) atomicOr(flags, FLAG_NONFINITE);
  LiteralElement<L> el;
  el.init(r);
  exps[idx] = el.e;
  for (int q = 0; q < Q; q++) qplanes[(size_t)q * total + idx] = el.next(Q, eq8 != 0);
}

// stats[0..1] = min / max level z = floor(e / 13) over the non-zero elements (pre-set to INT_MAX / INT_MIN);
// stats[2 .. 2 + 26) = elements per group
template <int L>
__global__ void __launch_bounds__(256) literal_stats_kernel(size_t total, const double* __restrict__ planes, int32_t* stats, uint32_t* flags) {
  __shared__ int s_min, s_max, s_cnt[GROUPS];
  if (threadIdx.x == 0) s_min = INT32_MAX, s_max = INT32_MIN;
  if (threadIdx.x < GROUPS) s_cnt[threadIdx.x] = 0;
  __syncthreads();
  for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
    double r[L];
#pragma unroll
    for (int l = 0; l < L; l++) r[l] = planes[l * total + idx];
    if (flags && limbs_nonfinite<L>(r)) atomicOr(flags, FLAG_NONFINITE);
    LiteralElement<L> el;
    el.init(r);
    if (el.zero) continue;
    const int z = floor_div13(el.e);
    atomicMin(&s_min, z);
    atomicMax(&s_max, z);
    atomicAdd(&s_cnt[mod13(el.e) + (el.negative ? 13 : 0)], 1);
  }
  __syncthreads();
  if (threadIdx.x == 0 && s_max >= s_min) atomicMin(&stats[0], s_min), atomicMax(&stats[1], s_max);
  if (threadIdx.x < GROUPS && s_cnt[threadIdx.x]) atomicAdd(&stats[2 + threadIdx.x], s_cnt[threadIdx.x]);
}

__device__ __forceinline__ void stg_256(double* p, double a, double b, double c, double d) {
  asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}

// One class (x sign) of an operand as NP packed quarter planes on the class's common grid (R20): part q of an
// element of level z is plane P = q + (zmax - z); every other plane of the element, and every element outside the group, is an
// "unnormalized zero with the desired exponent".  group < 13: the class, both signs; 13 + c / 39 + c: the
// positive / negative elements of class c (eq. 6).  Thread = one fragment row (group index x, four contraction indices).
template <int L, int AXIS>
__global__ void __launch_bounds__(256) literal_split_packed_kernel(int rows, int cols, int Q, int NP, int eq8, int group, int zmax,
                                                                   int bx, int bk, int x_blocks, int KS,
                                                                   const double* __restrict__ planes, double* __restrict__ packed) {
  const int X = AXIS == 0 ? rows : cols, K = AXIS == 0 ? cols : rows;
  const int x = (blockIdx.x % x_blocks) * 32 + (threadIdx.x & 31);
  const int k4g = (blockIdx.x / x_blocks) * 8 + (threadIdx.x >> 5);
  const int XP = (X + bx - 1) / bx * bx;
  if (k4g >= KS * (bk / 4) || x >= XP) return;
  const int k0 = k4g * 4;
  const size_t plane = (size_t)rows * cols;
  LiteralElement<L> el[4];
  int off[4];  // first plane of the element, or NP when it contributes nothing to this group
#pragma unroll
  for (int t = 0; t < 4; t++) {
    double r[L];
    const bool ok = x < X && k0 + t < K;
#pragma unroll
    for (int l = 0; l < L; l++)
      r[l] = !ok ? 0.0 : AXIS == 0 ? planes[l * plane + (size_t)x * cols + k0 + t] : planes[l * plane + (size_t)(k0 + t) * cols + x];
    el[t].init(r);
    const int c = mod13(el[t].e);
    const bool mine = !el[t].zero && (group < 13 ? c == group : group < 26 ? (c == group - 13 && !el[t].negative) : (c == group - 39 && el[t].negative));
    off[t] = mine ? zmax - floor_div13(el[t].e) : NP;
  }
  double* dst = packed + packed_offset(x, k0, 0, bx, bk, NP, KS);
  const size_t q_stride = (size_t)(bk / 4) * (bx / 8) * 32;
  for (int P = 0; P < NP; P++) {
    double d[4];
#pragma unroll
    for (int t = 0; t < 4; t++) d[t] = (P >= off[t] && P < off[t] + Q) ? el[t].next(Q, eq8 != 0) : 0.0;
    stg_256(dst + P * q_stride, d[0], d[1], d[2], d[3]);
  }
}

// r [L+1][m*n] (running expansions) += the S order planes of one class pair, smallest order first (R9, R16)
template <int L>
__global__ void __launch_bounds__(256) literal_accumulate_kernel(size_t total, int S, const double* __restrict__ orders, double* __restrict__ r) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= total) return;
  double acc[L + 1];
#pragma unroll
  for (int l = 0; l <= L; l++) acc[l] = r[(size_t)l * total + idx];
  for (int s = S - 1; s >= 0; s--) renorm_add<L>(acc, orders[(size_t)s * total + idx]);
#pragma unroll
  for (int l = 0; l <= L; l++) r[(size_t)l * total + idx] = acc[l];
}

template <int L>
__global__ void __launch_bounds__(256) literal_finish_kernel(size_t total, const double* __restrict__ r, double* __restrict__ C) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= total) return;
  double acc[L + 1], out[L];
#pragma unroll
  for (int l = 0; l <= L; l++) acc[l] = r[(size_t)l * total + idx];
  renorm_finish<L>(acc, out);
#pragma unroll
  for (int l = 0; l < L; l++) C[(size_t)l * total + idx] = out[l];
}

#define MD_BY_LIMBS(limbs, CALL)  \
  switch (limbs) {                \
    case 2: { CALL(2); } break;   \
    case 4: { CALL(4); } break;   \
    case 8: { CALL(8); } break;   \
    case 16: { CALL(16); } break; \
    default: return cudaErrorInvalidValue; \
  }

cudaError_t launch_literal_stats(size_t total, int limbs, const double* planes, int32_t* stats, uint32_t* flags, cudaStream_t st,
                                 uint64_t* launches) {
  const int32_t init[2 + GROUPS] = {INT32_MAX, INT32_MIN};
  cudaError_t err = cudaMemcpyAsync(stats, init, sizeof(init), cudaMemcpyHostToDevice, st);
  if (err != cudaSuccess) return err;
  const size_t want = (total + 255) / 256;
  const int cap = (sm_count() > 0 ? sm_count() : 1) * 16;
  const unsigned blocks = (unsigned)(want < (size_t)cap ? want : (size_t)cap);
#define CALL(L_) literal_stats_kernel<L_><<<blocks, 256, 0, st>>>(total, planes, stats, flags)
  MD_BY_LIMBS(limbs, CALL)
#undef CALL
  *launches += 1;
  return cudaGetLastError();
}

cudaError_t launch_literal_split_packed(int rows, int cols, int limbs, int Q, int NP, int eq8, int group, int zmax, int axis, int bx,
                                        int bk, const double* planes, double* packed, cudaStream_t st, uint64_t* launches) {
  const int X = axis == 0 ? rows : cols, K = axis == 0 ? cols : rows;
  const int KS = (K + bk - 1) / bk;
  const int x_blocks = ((X + bx - 1) / bx * bx + 31) / 32;
  const long long blocks = (long long)x_blocks * (((long long)KS * (bk / 4) + 7) / 8);
  if (blocks > 0x7fffffffLL) return cudaErrorInvalidValue;
#define CALL(L_)                                                                                                                      \
  if (axis == 0)                                                                                                                      \
    literal_split_packed_kernel<L_, 0><<<(unsigned)blocks, 256, 0, st>>>(rows, cols, Q, NP, eq8, group, zmax, bx, bk, x_blocks, KS, planes, packed); \
  else                                                                                                                                \
    literal_split_packed_kernel<L_, 1><<<(unsigned)blocks, 256, 0, st>>>(rows, cols, Q, NP, eq8, group, zmax, bx, bk, x_blocks, KS, planes, packed)
  MD_BY_LIMBS(limbs, CALL)
#undef CALL
  *launches += 1;
  return cudaGetLastError();
}

struct LiteralCarve {
  uint32_t* flags;
  int32_t *statsA, *statsB;
  double *r, *orders, *Aq, *Bq;
  void* sk;
  size_t total;
};
LiteralCarve literal_carve(void* base, int m, int n, int k, int limbs, int NP, int S, const KernelPick& pick) {
  LiteralCarve c;
  char* p = static_cast<char*>(base);
  size_t off = 0;
  c.flags = reinterpret_cast<uint32_t*>(p);
  c.statsA = reinterpret_cast<int32_t*>(p + 256);
  c.statsB = reinterpret_cast<int32_t*>(p + 512);
  off += 1024;
  c.r = reinterpret_cast<double*>(p + off);
  off += ws_round_up(sizeof(double) * (size_t)(limbs + 1) * m * n);
  c.orders = reinterpret_cast<double*>(p + off);
  off += ws_round_up(sizeof(double) * (size_t)S * m * n);
  c.Aq = reinterpret_cast<double*>(p + off);
  off += ws_round_up(sizeof(double) * packed_doubles(m, k, pick.bxA, pick.bk, NP));
  c.Bq = reinterpret_cast<double*>(p + off);
  off += ws_round_up(sizeof(double) * packed_doubles(n, k, pick.bxB, pick.bk, NP));
  c.sk = p + off;
  off += ws_round_up(sk_workspace_bytes(S, pick.bxA, pick.bxB, k, 0));
  c.total = off;
  return c;
}

inline bool limbs_ok(int limbs) { return limbs == 2 || limbs == 4 || limbs == 8 || limbs == 16; }
// parts are multiples of HALF a unit below 2^15 of them (eq. 8): products are integers below 2^30 quarter-units
constexpr int LITERAL_DIGIT_BITS = 15;

}  // namespace
}  // namespace md

using namespace md;

extern "C" {

md_status md_split_literal(int rows, int cols, int limbs, int quarters, int flags, const double* planes, double* quarter_planes,
                           int32_t* exps, md_stream stream) {
  if (rows <= 0 || cols <= 0 || !planes || !quarter_planes || !exps || (flags & ~MD_LITERAL_NO_EQ8)) return MD_ERR_BAD_ARG;
  if (!limbs_ok(limbs) || quarters < 1 || quarters > MD_MAX_QUARTERS) return MD_ERR_BAD_ARG;
  if ((reinterpret_cast<uintptr_t>(planes) | reinterpret_cast<uintptr_t>(quarter_planes)) & 7 || (reinterpret_cast<uintptr_t>(exps) & 3))
    return MD_ERR_BAD_ARG;
  DeviceState* ds = device_state();
  uint32_t* status = ds && ds->ws ? static_cast<uint32_t*>(ds->ws) : nullptr;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const size_t total = (size_t)rows * cols;
  const unsigned blocks = (unsigned)((total + 255) / 256);
  const int eq8 = (flags & MD_LITERAL_NO_EQ8) ? 0 : 1;
  switch (limbs) {
    case 2: literal_split_kernel<2><<<blocks, 256, 0, st>>>(total, quarters, eq8, planes, quarter_planes, exps, status); break;
    case 4: literal_split_kernel<4><<<blocks, 256, 0, st>>>(total, quarters, eq8, planes, quarter_planes, exps, status); break;
    case 8: literal_split_kernel<8><<<blocks, 256, 0, st>>>(total, quarters, eq8, planes, quarter_planes, exps, status); break;
    default: literal_split_kernel<16><<<blocks, 256, 0, st>>>(total, quarters, eq8, planes, quarter_planes, exps, status); break;
  }
  g_launches += 1;
  return cudaGetLastError() == cudaSuccess ? MD_OK : MD_ERR_CUDA;
}

size_t md_literal_scratch_bytes(int m, int n, int k, int limbs, int planes_per_class, int orders) {
  if (m <= 0 || n <= 0 || k <= 0 || !limbs_ok(limbs)) return 0;
  const int Q = quarters_for(limbs);
  const int NP = planes_per_class > 0 ? planes_per_class : Q, S = orders > 0 ? orders : NP;
  const KernelPick pick = pick_kernel(m, n, k, limbs, NP, S, 13, true, false);
  if (pick.family == GEMM_NONE) return 0;
  return literal_carve(nullptr, m, n, k, limbs, NP, S, pick).total;
}

md_status md_gemm_literal(int m, int n, int k, int limbs, const double* A_planes, const double* B_planes, double* C_planes,
                          void* scratch, size_t scratch_bytes, int flags, int32_t* info_host, md_stream stream) {
  if (m <= 0 || n <= 0 || k <= 0 || !A_planes || !B_planes || !C_planes || !scratch) return MD_ERR_BAD_ARG;
  if (!limbs_ok(limbs) || (flags & ~(MD_LITERAL_NO_EQ8 | MD_LITERAL_SIGN_GROUPS))) return MD_ERR_BAD_ARG;
  if ((reinterpret_cast<uintptr_t>(A_planes) | reinterpret_cast<uintptr_t>(B_planes) | reinterpret_cast<uintptr_t>(C_planes)) & 7) return MD_ERR_BAD_ARG;
  if (reinterpret_cast<uintptr_t>(scratch) % WS_ALIGN || scratch_bytes < 1024) return MD_ERR_BAD_ARG;
  if (slice_bits() != 13) return MD_ERR_UNSUPPORTED;  // the paper's 13-bit parts only
  const int Q = quarters_for(limbs);
  const int eq8 = (flags & MD_LITERAL_NO_EQ8) ? 0 : 1;
  const bool signs = (flags & MD_LITERAL_SIGN_GROUPS) != 0;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  uint64_t launches = 0;
  char* base = static_cast<char*>(scratch);
  uint32_t* status = reinterpret_cast<uint32_t*>(base);
  int32_t* statsA = reinterpret_cast<int32_t*>(base + 256);
  int32_t* statsB = reinterpret_cast<int32_t*>(base + 512);
  // 1. level range and class populations of both operands (one pass each), read back: the plane and order counts, hence the
  //    kernel and the workspace layout, depend on the data
  if (cudaMemsetAsync(status, 0, 256, st) != cudaSuccess) return MD_ERR_CUDA;
  cudaError_t err = launch_literal_stats((size_t)m * k, limbs, A_planes, statsA, status, st, &launches);
  if (err == cudaSuccess) err = launch_literal_stats((size_t)k * n, limbs, B_planes, statsB, status, st, &launches);
  int32_t hA[2 + GROUPS], hB[2 + GROUPS];
  if (err == cudaSuccess) err = cudaMemcpyAsync(hA, statsA, sizeof(hA), cudaMemcpyDeviceToHost, st);
  if (err == cudaSuccess) err = cudaMemcpyAsync(hB, statsB, sizeof(hB), cudaMemcpyDeviceToHost, st);
  g_launches += launches;
  launches = 0;
  if (err != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess) return MD_ERR_CUDA;
  if (hA[1] < hA[0]) hA[0] = hA[1] = 0;  // an all-zero operand
  if (hB[1] < hB[0]) hB[0] = hB[1] = 0;
  const int spanA = hA[1] - hA[0], spanB = hB[1] - hB[0];
  const int NP = Q + (spanA > spanB ? spanA : spanB), S = Q + spanA + spanB;
  if (info_host) {
    info_host[0] = hA[0], info_host[1] = hA[1], info_host[2] = hB[0], info_host[3] = hB[1];
    info_host[4] = NP, info_host[5] = S, info_host[6] = 0, info_host[7] = 0;
  }
  const KernelPick pick = pick_kernel(m, n, k, limbs, NP, S, 13, true, false);
  if (pick.family == GEMM_NONE) return MD_ERR_UNSUPPORTED;
  if (!k_budget_ok(k, S, LITERAL_DIGIT_BITS)) return MD_ERR_K_TOO_LARGE;
  const LiteralCarve c = literal_carve(scratch, m, n, k, limbs, NP, S, pick);
  if (c.total > scratch_bytes) return MD_ERR_WORKSPACE;  // info_host[4], [5] say what md_literal_scratch_bytes must be asked for

  // 2. the class-pair products ("execute many matrix multiplications"), every order sum of every pair added into
  //    the running expansions; empty classes are skipped
  const size_t total = (size_t)m * n;
  const unsigned eblocks = (unsigned)((total + 255) / 256);
  err = cudaMemsetAsync(c.r, 0, sizeof(double) * (size_t)(limbs + 1) * total, st);
  int pairs = 0;
  const int ngroups = signs ? 26 : 13;
  auto population = [&](const int32_t* h, int g) { return signs ? h[2 + g] : h[2 + g] + h[2 + 13 + g]; };
  for (int ga = 0; ga < ngroups && err == cudaSuccess; ga++) {
    if (population(hA, ga) == 0) continue;
    // group argument of the splitter: < 13 the whole class; 13 + c its positive, 39 + c its negative elements
    const int argA = signs ? (ga < 13 ? 13 + ga : 39 + (ga - 13)) : ga;
    err = launch_literal_split_packed(m, k, limbs, Q, NP, eq8, argA, hA[1], 0, pick.bxA, pick.bk, A_planes, c.Aq, st, &launches);
    for (int gb = 0; gb < ngroups && err == cudaSuccess; gb++) {
      if (population(hB, gb) == 0) continue;
      const int argB = signs ? (gb < 13 ? 13 + gb : 39 + (gb - 13)) : gb;
      err = launch_literal_split_packed(k, n, limbs, Q, NP, eq8, argB, hB[1], 1, pick.bxB, pick.bk, B_planes, c.Bq, st, &launches);
      if (err == cudaSuccess) err = launch_fused(m, n, k, limbs, NP, S, pick, c.Aq, c.Bq, c.orders, nullptr, c.sk, false, st, &launches);
      if (err != cudaSuccess) break;
      switch (limbs) {
        case 2: literal_accumulate_kernel<2><<<eblocks, 256, 0, st>>>(total, S, c.orders, c.r); break;
        case 4: literal_accumulate_kernel<4><<<eblocks, 256, 0, st>>>(total, S, c.orders, c.r); break;
        case 8: literal_accumulate_kernel<8><<<eblocks, 256, 0, st>>>(total, S, c.orders, c.r); break;
        default: literal_accumulate_kernel<16><<<eblocks, 256, 0, st>>>(total, S, c.orders, c.r); break;
      }
      launches += 1;
      err = cudaGetLastError();
      pairs++;
    }
  }
  if (err == cudaSuccess) {
    switch (limbs) {
      case 2: literal_finish_kernel<2><<<eblocks, 256, 0, st>>>(total, c.r, C_planes); break;
      case 4: literal_finish_kernel<4><<<eblocks, 256, 0, st>>>(total, c.r, C_planes); break;
      case 8: literal_finish_kernel<8><<<eblocks, 256, 0, st>>>(total, c.r, C_planes); break;
      default: literal_finish_kernel<16><<<eblocks, 256, 0, st>>>(total, c.r, C_planes); break;
    }
    launches += 1;
    err = cudaGetLastError();
  }
  g_launches += launches;
  if (info_host) info_host[6] = pairs, info_host[7] = (int32_t)launches;
  return err == cudaSuccess ? MD_OK : MD_ERR_CUDA;
}

}  // extern "C"
