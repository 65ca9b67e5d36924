// qgemm_wide.cu -- steps a3 + a4 for the two wider formats of the paper's Table 2: octo double
// (8 limbs, Q = S = 32 quarters / orders, T = 528 quarter products) and hexa double (16 limbs, Q = S = 64, T = 2080).
//
//   For s = 0..S-1:  C^(s) = sum_{p+q=s} A_p * B_q      (PAPER.md:66-71 eq. 3; :75-78 eq. 4: the paper's C_{s+1})
//   C = sum_s C^(s), summed error free into L limbs     (PAPER.md:88-91 steps 4-5)
//
// Same method, same packed operand layout (md_packed.cuh, k-slab depth 4), same persistent stream-K bulk-copy / mbarrier
// pipeline as qgemm_packed.cu.  What changes is where the S accumulator sets live: an 8x8 DMMA tile needs 2 doubles per
// order per thread, so 32 orders fill 128 registers and 64 orders do not fit a thread at all.  Hence
//   * a warp owns ONE 8x8 tile of C and a contiguous ORDER RANGE [S0, S1) of at most 32 orders;
//   * octo double: one range [0, 32) per tile, 8 tiles (32 x 16) per CTA;
//   * hexa double with the paper's 64 quarters: the four ranges [0,32) [32,45) [45,55) [55,64) -- 528 / 507 / 505 / 540
//     products -- are walked ONE AFTER THE OTHER by every warp on its own 8x8 tile (qgemm_hd_passes_kernel, further down): four
//     passes over the contraction, one resident k-step body at a time.  Four warps sharing a tile, each with its own range and
//     body (WCfg<.., R = 4>: what round 1 ran, still used by the GENERIC hexa-double instance), lose 4 % of the k loop to the SM's
//     instruction cache;
//   * hexa double in 44 slices of 19 bits: two ranges [0,31) [31,44) per tile, 4 tiles (16 x 16) per CTA, both warps of an SM
//     sub-partition on the same range, the upper range's k-step rolled (k_step_range_rolled) so that both bodies stay resident;
//   * inside a k-step a range walks q = 0, 1, ... and needs the A fragments p in [S0-q, S1-1-q]: a window of S1-S0 quarters
//     that slides down by one per q, kept in a register ring (one new LDS per q, issued one step ahead);
//   * the recombination of a hexa double element is a chain over its four warps: the (L+1)-term accumulator of
//     renorm_add (md_common.cuh) goes from the warp with the smallest orders to the warp with the largest through a
//     lane-private slot of shared memory, which performs exactly the operation sequence of the standalone md_renorm.
//
// GENERIC instances (WCfg<..., GENERIC = true>): the same kernel with the quarter count Q and the order count S as RUNTIME
// values below compile-time maxima (double double Q <= 16 / S <= 24, quad 24 / 32, octo 40 / 42, hexa 72 / 74, so the pruned and
// extended order sets of MD_OPT_ORDERS run here too).  Every DMMA site of the maximal triangular set stays in the code
// behind a warp-uniform predicate; the order ranges are those of the maximal set, so a smaller problem leaves the upper
// ranges short of work.  Slower than a tuned instance (one 8x8 tile per warp, predicates, k-slab depth 4), but every
// (limbs, quarters, orders) that md_plan_quarters can ask for has a kernel (R5, R15).
//
// Exactness as in qgemm_packed.cu: k * S <= 2^27 keeps every partial sum an integer below 2^53 units (PAPER.md:95-99
// eq. 5; R6), so the result does not depend on the order in which warps, slabs or the hardware add things.
#include <type_traits>

#include "md_kernels.h"
#include "md_packed.cuh"
#include "qgemm_common.cuh"
#include "qgemm_pipeline.cuh"

namespace md {
namespace {

// TM x TN 8x8 tiles per CTA, R order ranges per tile: TM * TN * R = 8 warps.  Q_, S_: the quarter / order counts of a tuned
// instance, or their MAXIMA for a GENERIC one (runtime counts in WideCtx).
template <int Q_, int L_, int TM_, int TN_, int R_, int S_ = Q_, bool GENERIC_ = false>
struct WCfg {
  static constexpr int Q = Q_, S = S_, L = L_, TM = TM_, TN = TN_, R = R_;
  static constexpr bool GENERIC = GENERIC_;
  static constexpr int BM = TM * 8, BN = TN * 8, BK = PACK_BK_WIDE;
  static constexpr int TILES = TM * TN, WARPS = TILES * R, THREADS = WARPS * 32;
  static constexpr int A_CHUNK = Q * BK * BM, B_CHUNK = Q * BK * BN;  // doubles per k-slab (GENERIC: at most)
  static constexpr int AQ = BK * BM, BQ = BK * BN;                    // doubles per quarter inside a chunk
  static constexpr int STAGE_BYTES = (A_CHUNK + B_CHUNK) * 8;
  static constexpr int BAR_BYTES = 128;
  // hand-over slots of the recombination chain: per tile, per lane, two elements of L+1 terms
  static constexpr int XCHG_BYTES = R > 1 ? TILES * 2 * (L + 1) * 32 * 8 : 0;
  static constexpr int STAGES =
      ((SMEM_LIMIT - BAR_BYTES - XCHG_BYTES) / STAGE_BYTES) < 6 ? ((SMEM_LIMIT - BAR_BYTES - XCHG_BYTES) / STAGE_BYTES) : 6;
  static constexpr int AHEAD = STAGES - 2;
  static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + BAR_BYTES + XCHG_BYTES;
  static_assert(WARPS == 8, "8 warps per CTA (2 per SM sub-partition)");
  static_assert(R == 1 || (R == 4 && (Q == 64 || Q == 72)) || (R == 2 && (Q == 44 || Q == 40)), "order ranges with a boundary table");
  static_assert(STAGES >= 3, "the non-blocking refill needs at least 3 stages");
  static_assert(2 * STAGES * 8 <= BAR_BYTES - 8, "barrier area (its last 8 bytes hold the stream-K flag)");
  static_assert(STAGE_BYTES % 128 == 0 && XCHG_BYTES % 128 == 0, "alignment");
  // order range r = [lo(r), hi(r)): boundaries that balance the product counts sum_{s in range} #{(p, q): p + q = s} --
  //   Q = 64, R = 4: 0 | 32 | 45 | 55 | 64 -> 528 / 507 / 505 / 540;   Q = 44, R = 2: 0 | 31 | 44 -> 496 / 494;
  //   generic hexa double (Q <= 72, S <= 74), R = 4: 0 | 34 | 50 | 63 | 74 -> 595 / 680 / 741 / 753 (the first range is kept
  //   at 34 orders: 37 would balance better but spills);  generic octo double (Q <= 40, S <= 42), R = 2: 0 | 30 | 42 -> 465 / 432
  __host__ __device__ static constexpr int bound(int r) {
    return R == 1   ? (r == 0 ? 0 : S)
           : R == 2 ? (Q == 40 ? (r == 0 ? 0 : r == 1 ? 30 : 42) : (r == 0 ? 0 : r == 1 ? 31 : 44))
           : Q == 72 ? (r == 0 ? 0 : r == 1 ? 34 : r == 2 ? 50 : r == 3 ? 63 : 74)
                     : (r == 0 ? 0 : r == 1 ? 32 : r == 2 ? 45 : r == 3 ? 55 : 64);
  }
  __host__ __device__ static constexpr int lo(int r) { return bound(r); }
  __host__ __device__ static constexpr int hi(int r) { return bound(r + 1); }
  // warp -> (tile, range).  Warps w and w + 4 share an SM sub-partition: R = 4 pairs ranges (0,1) and (2,3) there (1035 /
  // 1045 DMMAs per k-step), R = 2 the two ranges of one tile (990).
  // R = 2: the two warps of a sub-partition (w, w + 4) run the SAME range on different tiles (the two ranges are balanced,
  // 496 / 494 products): hd in 44 slices 0.929 -> 0.942 of the peak against one warp of each range per sub-partition.  R = 4
  // keeps mixed pairs: its ranges are unequal (528 / 507 / 505 / 540) and pairing equal ranges puts 1080 products on one
  // sub-partition against 1010 on another (measured 0.940 -> 0.913); with every warp forced onto ONE range body (a timing
  // experiment) the k loop runs at 0.99 of the peak instead of 0.96 -- profiles/r04_qgemm_hd.md
  __host__ __device__ static constexpr int tile_of(int w) { return R == 1 ? w : R == 2 ? (((w >> 2) << 1) | (w & 1)) : w / 4; }
  __host__ __device__ static constexpr int range_of(int w) {
    return R == 1 ? 0 : R == 2 ? ((w & 3) >> 1)
                      : (w < 4 ? (w == 0 ? 0 : w == 1 ? 2 : w == 2 ? 1 : 3) : (w == 4 ? 1 : w == 5 ? 3 : w == 6 ? 0 : 2));
  }
};

// What a warp needs to know about the CTA's pipeline and work list (built once in the kernel).
struct WideCtx {
  int m, n, G, cta, KS;
  int Q, S;              // quarter / order counts of this launch (GENERIC instances; the tuned ones use C::Q, C::S)
  int a_chunk, b_chunk;  // doubles of A / B per k-slab = Q * BK * BM, Q * BK * BN
  SkPlan plan;
  int g0, g1, n_sk, n_seg, total_slabs;  // this CTA's segment list (see qgemm_pipeline.cuh)
  const double *Ap, *Bp;
  double *order_planes, *C_planes, *sk_scratch;
  unsigned int* sk_counters;
  double* stages;
  uint32_t stages_u32, full_u32, empty_u32;
  volatile int* last_flag;
  double* xchg;
  __device__ __forceinline__ void segment(int i, int& tile, int& s0, int& s1) const {
    if (i < n_sk) {
      const int r = g0 / KS + i;
      tile = plan.dp_waves * G + r;
      s0 = i == 0 ? g0 - r * KS : 0;
      s1 = min(KS, g1 - r * KS);
    } else {
      tile = (i - n_sk) * G + cta;
      s0 = 0;
      s1 = KS;
    }
  }
};

// One DMMA k-step (4 contraction indices) of order range [S0, S1) on the warp's 8x8 tile: every product (p, q) with
// S0 <= p + q < S1 goes to accumulator p + q - S0.  As / Bs point at the lane's element of the quarter-0 fragment of the
// warp's row block / column block in the staged slab; quarter p of A is p * AQ doubles further, quarter q of B q * BQ.
// Fully unrolled: every register index below is a compile-time constant.
template <int Q, int S0, int S1, int AQ, int BQ>
__device__ __forceinline__ void k_step_range(double (&acc)[S1 - S0][2], const double* __restrict__ As,
                                             const double* __restrict__ Bs) {
  constexpr int W = S1 - S0;
  constexpr int RW = S0 == 0 ? W : W + 1;                   // ring slots (one spare for the fragment fetched ahead)
  constexpr int QMAX = S1 - 1 < Q - 1 ? S1 - 1 : Q - 1;     // last q with a product in the range
  double a[RW];
#pragma unroll
  for (int p = S0; p <= (S1 - 1 < Q - 1 ? S1 - 1 : Q - 1); p++) a[p % RW] = As[p * AQ];  // window of q = 0
  double b = Bs[0];
#pragma unroll
  for (int q = 0; q <= QMAX; q++) {
    double b_next = 0.0;
    if (q + 1 <= QMAX) {                                     // operands of step q + 1, issued before step q's DMMAs
      b_next = Bs[(q + 1) * BQ];
      if (S0 - (q + 1) >= 0) a[(S0 - (q + 1)) % RW] = As[(S0 - (q + 1)) * AQ];
    }
    const int lo = S0 - q > 0 ? S0 - q : 0;
    const int hi = S1 - 1 - q < Q - 1 ? S1 - 1 - q : Q - 1;
#pragma unroll
    for (int p = lo; p <= hi; p++) dmma_8x8x4(acc[p + q - S0], a[p % RW], b);
    b = b_next;
  }
}

// The same k-step for a range with S0 > 0, ROLLED over q where the range has its full width.  For q <= S0 every one of the
// W = S1 - S0 orders receives a product (p = S0 - q + j into accumulator j) and the register ring of A fragments repeats with
// period RW = W + 1 in q, so RW consecutive q-steps make one trip of a loop whose register indices are compile-time constants; only
// the remaining full-width steps (at least one) and the triangle q > S0 stay straight-line code.  Same products, same accumulators
// (exact sums, R6); the point is CODE SIZE: one fully unrolled k-step body of about 10 KB stays in the SM's instruction
// cache, two (hexa double in 44 slices: 496 + 494 DMMAs) do so only partly and were streamed from the L1.5 at 9.5 KB per
// iteration of the k loop.  With the upper range rolled (312 DMMA sites instead of 494) they fit: 0.942 -> 0.964 of the peak.
// NOT used for the four ranges of hexa double with 64 quarters: 528 + 325 + 175 + 180 sites (24 KB) still do not fit and the
// loop overhead costs more than the smaller stream saves (0.940 -> 0.935); rotating the window by register moves instead (one
// q-step per trip, 751 sites) stalls on the DMMAs that still read the registers (0.852).  profiles/r04_qgemm_hd.md.
template <int Q, int S0, int S1, int AQ, int BQ>
__device__ __forceinline__ void k_step_range_rolled(double (&acc)[S1 - S0][2], const double* __restrict__ As,
                                                    const double* __restrict__ Bs) {
  constexpr int W = S1 - S0, RW = W + 1;
  constexpr int NTRIPS = S0 / RW, Q0 = NTRIPS * RW;  // trips cover q = 0 .. Q0 - 1 (Q0 <= S0: the step q = S0 is never inside a trip)
  static_assert(S0 > 0 && S1 <= Q && S0 > RW, "a range above the first one, inside the quarter count");
  double a[RW];
#pragma unroll
  for (int p = S0; p <= S1 - 1; p++) a[p % RW] = As[p * AQ];  // window of q = 0
  double b = Bs[0];
  const double* pa = As + S0 * AQ;  // A fragment p = S0 - q0
  const double* pb = Bs;            // B fragment q0
#pragma unroll 1
  for (int trip = 0; trip < NTRIPS; trip++) {
#pragma unroll
    for (int u = 0; u < RW; u++) {  // q = trip * RW + u; fragment p = S0 - q + j sits in ring slot (S0 - u + j) % RW
      const double b_next = pb[(u + 1) * BQ];
      a[(S0 - u - 1) % RW] = pa[-(u + 1) * AQ];  // p = S0 - (q + 1) >= 0 inside the trips: the operand of the next step
#pragma unroll
      for (int j = 0; j < W; j++) dmma_8x8x4(acc[j], a[(S0 - u + j) % RW], b);
      b = b_next;
    }
    pa -= RW * AQ;
    pb += RW * BQ;
  }
#pragma unroll
  for (int q = Q0; q <= S1 - 1; q++) {  // the last full-width steps and the triangle, as in k_step_range
    double b_next = 0.0;
    if (q + 1 <= S1 - 1) {
      b_next = Bs[(q + 1) * BQ];
      if (S0 - (q + 1) >= 0) a[(S0 - (q + 1)) % RW] = As[(S0 - (q + 1)) * AQ];
    }
    const int lo = S0 - q > 0 ? S0 - q : 0;
    const int hi = S1 - 1 - q;
#pragma unroll
    for (int p = lo; p <= hi; p++) dmma_8x8x4(acc[p + q - S0], a[p % RW], b);
    b = b_next;
  }
}

// The same for a GENERIC instance: QMAX, [S0, S1) are the compile-time maxima, Qr <= QMAX and Sr the counts of this launch
// (warp-uniform).  Every site of the maximal set is predicated; for a given q the live products are a prefix
// p = lo .. min(hi, Qr - 1, Sr - 1 - q) of the compile-time range.
template <int QMAX, int S0, int S1, int AQ, int BQ>
__device__ __forceinline__ void k_step_range_rt(double (&acc)[S1 - S0][2], const double* __restrict__ As,
                                                const double* __restrict__ Bs, int Qr, int Sr) {
  constexpr int W = S1 - S0;
  constexpr int RW = S0 == 0 ? W : W + 1;
  constexpr int QTOP = S1 - 1 < QMAX - 1 ? S1 - 1 : QMAX - 1;
  if (S0 >= Sr) return;  // nothing of this range is kept
  double a[RW];
#pragma unroll
  for (int p = S0; p <= QTOP; p++) a[p % RW] = p < Qr ? As[p * AQ] : 0.0;
  double b = Bs[0];
#pragma unroll
  for (int q = 0; q <= QTOP; q++) {
    if (q >= Qr) break;
    double b_next = 0.0;
    if (q + 1 <= QTOP && q + 1 < Qr) {
      b_next = Bs[(q + 1) * BQ];
      if (S0 - (q + 1) >= 0 && S0 - (q + 1) < Qr) a[(S0 - (q + 1)) % RW] = As[(S0 - (q + 1)) * AQ];
    }
    const int lo = S0 - q > 0 ? S0 - q : 0;
    const int hi = S1 - 1 - q < QMAX - 1 ? S1 - 1 - q : QMAX - 1;
    const int pmax = min(Qr - 1, Sr - 1 - q);
    // a BRANCH out of the live prefix, not a predicate per site: a predicated-off DMMA still takes its slot in the tensor pipe
    // (measured: 83 % pipe-active at 38 % useful throughput with predication, profiles/r3d)
#pragma unroll
    for (int p = lo; p <= hi; p++) {
      if (p > pmax) break;
      dmma_8x8x4(acc[p + q - S0], a[p % RW], b);
    }
    b = b_next;
  }
}

// Producer cursor (thread 0 only): walks the CTA's flat slab sequence AHEAD slabs in front of the consumers.
template <class C>
struct WideProducer {
  int p_seg = -1, p_left = 0, p_flat = 0, pst = 0;
  const double *p_A = nullptr, *p_B = nullptr;
  __device__ __forceinline__ void produce_one(const WideCtx& x) {
    if (p_left == 0) {
      int tile, s0, s1, tm, tn;
      x.segment(++p_seg, tile, s0, s1);
      raster_tile(tile, x.plan.tiles_m, x.plan.tiles_n, tm, tn, x.plan.group_m);
      p_A = x.Ap + ((size_t)tm * x.KS + s0) * (C::GENERIC ? x.a_chunk : C::A_CHUNK);
      p_B = x.Bp + ((size_t)tn * x.KS + s0) * (C::GENERIC ? x.b_chunk : C::B_CHUNK);
      p_left = s1 - s0;
    }
    // GENERIC: a stage keeps its compile-time size and the B part its compile-time offset; only Q quarters of each arrive
    const int a_chunk = C::GENERIC ? x.a_chunk : C::A_CHUNK, b_chunk = C::GENERIC ? x.b_chunk : C::B_CHUNK;
    const uint32_t dst = x.stages_u32 + pst * C::STAGE_BYTES, bar = x.full_u32 + 8 * pst;
    mbar_expect_tx(bar, (a_chunk + b_chunk) * 8);
    bulk_g2s(dst, p_A, a_chunk * 8, bar);
    bulk_g2s(dst + C::A_CHUNK * 8, p_B, b_chunk * 8, bar);
    p_A += a_chunk;
    p_B += b_chunk;
    p_left--;
    p_flat++;
    pst = (pst + 1 == C::STAGES) ? 0 : pst + 1;
  }
  __device__ __forceinline__ void prologue(const WideCtx& x) {
#pragma unroll
    for (int j = 0; j < C::AHEAD; j++)
      if (p_flat < x.total_slabs) produce_one(x);
  }
  __device__ __forceinline__ void produce(const WideCtx& x) {  // top of a consumer iteration
    if (p_flat < x.total_slabs) {
      // the stage was last read two iterations ago: wait for its release (completed long ago)
      if (p_flat >= C::STAGES) mbar_wait(x.empty_u32 + 8 * pst, ((p_flat / C::STAGES) + 1) & 1);
      produce_one(x);
    }
  }
};

// End of a tile for the warp that owns orders [lo(RANGE), hi(RANGE)) of tile `t` of the CTA: acc[s - S0][e] is C^(s) of
// element (row, col + e), row = row_base + lane / 4, col = col_base + 2 * (lane % 4).  Writes the order planes (debug /
// parity) and / or the renormalised limb planes.  EVERY thread of the CTA must call it (block-wide barriers when R > 1).
template <class C, int RANGE>
__device__ __forceinline__ void wide_epilogue(const WideCtx& x, const double (&acc)[C::hi(RANGE) - C::lo(RANGE)][2], int t,
                                              int row_base, int col_base, int lane) {
  constexpr int S0 = C::lo(RANGE), S1 = C::hi(RANGE), L = C::L, R = C::R;
  const int row = row_base + (lane >> 2), col = col_base + 2 * (lane & 3);
  const bool inside = row < x.m && col < x.n, two = col + 1 < x.n;
  const size_t planeC = (size_t)x.m * x.n, at = (size_t)row * x.n + col;
  const bool vec_ok = (x.n % 2 == 0) && (((uintptr_t)x.C_planes | (uintptr_t)x.order_planes) % 16 == 0);
  const int Sr = C::GENERIC ? x.S : C::S;  // orders kept by this launch
  if (x.order_planes && inside) {
#pragma unroll
    for (int s = S0; s < S1; s++) {
      if (C::GENERIC && s >= Sr) break;
      if (vec_ok) {
        *reinterpret_cast<double2*>(x.order_planes + s * planeC + at) = make_double2(acc[s - S0][0], acc[s - S0][1]);
      } else {
        x.order_planes[s * planeC + at] = acc[s - S0][0];
        if (two) x.order_planes[s * planeC + at + 1] = acc[s - S0][1];
      }
    }
  }
  if (!x.C_planes) return;  // uniform over the CTA
  double out[2][L];
  // Recombination (R9): orders are added from the smallest (s = S-1) to the largest (s = 0)
  // into an (L+1)-term accumulator; with R ranges the accumulator travels range R-1 -> ... -> range 0.
#pragma unroll
  for (int rr = R - 1; rr >= 0; rr--) {
    if (rr == RANGE) {  // both elements of the thread side by side, the cascades cut short where only zeros are left (renorm_add2)
      double r0[L + 1], r1[L + 1];
      double* slot0 = x.xchg + (size_t)((t * 2 + 0) * (L + 1)) * 32 + lane;
      double* slot1 = x.xchg + (size_t)((t * 2 + 1) * (L + 1)) * 32 + lane;
#pragma unroll
      for (int l = 0; l <= L; l++) {
        r0[l] = (RANGE == R - 1) ? 0.0 : slot0[l * 32];
        r1[l] = (RANGE == R - 1) ? 0.0 : slot1[l * 32];
      }
      // a ROLLED loop over the orders, fed from a copy of the accumulators in local memory: unrolled, the recombination of a
      // hexa double was ~10 000 straight-line instructions per range executed once per tile -- every tile end re-fetched
      // 160 KB of code per warp through the instruction cache
      // (hexa double 512^3: 0.898 -> 0.931 of the peak; octo double's recombination is a quarter of the code and stays unrolled:
      // rolled it measured 0.9886 -> 0.9862)
      if constexpr (L >= 16) {
        double tmp[S1 - S0][2];
#pragma unroll
        for (int i = 0; i < S1 - S0; i++) tmp[i][0] = acc[i][0], tmp[i][1] = acc[i][1];
        const int s_top = C::GENERIC ? (Sr < S1 ? Sr : S1) : S1;
        // orders per trip, each one level behind the one before it (renorm_add2xN): 2 took hd 512^3 from 0.931 to 0.938; 4, and
        // staggering the final sweeps of renorm_finish2 the same way, measured no further gain (profiles/r04_qgemm_hd.md)
        constexpr int NW = 2;
        int s = s_top - 1;
#pragma unroll 1
        for (; s - (NW - 1) >= S0; s -= NW) {
          double xs[NW][2];
#pragma unroll
          for (int i = 0; i < NW; i++) xs[i][0] = tmp[s - i - S0][0], xs[i][1] = tmp[s - i - S0][1];
          renorm_add2xN<L, NW>(r0, r1, xs);
        }
#pragma unroll 1
        for (; s >= S0; s--) renorm_add2<L>(r0, r1, tmp[s - S0][0], tmp[s - S0][1]);
      } else {
#pragma unroll
        for (int s = S1 - 1; s >= S0; s--)
          if (!C::GENERIC || s < Sr) renorm_add2<L>(r0, r1, acc[s - S0][0], acc[s - S0][1]);
      }
      if (RANGE > 0) {
#pragma unroll
        for (int l = 0; l <= L; l++) slot0[l * 32] = r0[l], slot1[l * 32] = r1[l];
      } else {
        renorm_finish2<L>(r0, r1, out[0], out[1]);
      }
    }
    if (R > 1) __syncthreads();  // hand-over to the next range; the last one keeps the next tile's writers behind the readers
  }
  if (RANGE == 0 && inside) {
#pragma unroll
    for (int l = 0; l < L; l++) {
      if (vec_ok) {
        *reinterpret_cast<double2*>(x.C_planes + l * planeC + at) = make_double2(out[0][l], out[1][l]);
      } else {
        x.C_planes[l * planeC + at] = out[0][l];
        if (two) x.C_planes[l * planeC + at + 1] = out[1][l];
      }
    }
  }
}

// The whole life of one warp: consume the CTA's slab sequence for its (tile, order range), with thread 0 also running
// the producer cursor.  Segment ends: a whole tile goes straight to the epilogue; a stream-K part adds its partial
// order sums into the tile's scratch with fp64 red.add (exact, see the header) and the CTA that completes the slab
// count finishes the tile.
template <class C, int RANGE>
__device__ __forceinline__ void wide_consume(const WideCtx& x, int t, int lane, int tid) {
  constexpr int S0 = C::lo(RANGE), S1 = C::hi(RANGE), W = S1 - S0, STAGES = C::STAGES;
  constexpr int STAGE_DOUBLES = C::A_CHUNK + C::B_CHUNK;
  const int ti = t / C::TN, tj = t % C::TN;
  const int a_off = ti * 32 + lane, b_off = C::A_CHUNK + tj * 32 + lane;

  WideProducer<C> prod;
  if (tid == 0) prod.prologue(x);

  double acc[W][2];
#pragma unroll
  for (int s = 0; s < W; s++) acc[s][0] = acc[s][1] = 0.0;

  int c_seg = 0, c_tile, c_s0, c_s1;
  x.segment(0, c_tile, c_s0, c_s1);
  int c_left = c_s1 - c_s0;
  int st = 0;
  uint32_t phase = 0;
  for (int it = 0; it < x.total_slabs; it++) {
    if (tid == 0) prod.produce(x);
    mbar_wait(x.full_u32 + 8 * st, phase);
    const double* stage = x.stages + (size_t)st * STAGE_DOUBLES;
    if constexpr (C::GENERIC) k_step_range_rt<C::Q, S0, S1, C::AQ, C::BQ>(acc, stage + a_off, stage + b_off, x.Q, x.S);
    else if constexpr (S0 > 0 && C::R == 2) k_step_range_rolled<C::Q, S0, S1, C::AQ, C::BQ>(acc, stage + a_off, stage + b_off);
    else k_step_range<C::Q, S0, S1, C::AQ, C::BQ>(acc, stage + a_off, stage + b_off);
    __syncwarp();
    if (lane == 0) mbar_arrive(x.empty_u32 + 8 * st);  // this warp is done reading the stage
    if (++st == STAGES) {
      st = 0;
      phase ^= 1;
    }
    if (--c_left == 0) {
      int tm, tn;
      raster_tile(c_tile, x.plan.tiles_m, x.plan.tiles_n, tm, tn, x.plan.group_m);
      const int row_base = tm * C::BM + ti * 8, col_base = tn * C::BN + tj * 8;
      if (c_s1 - c_s0 == x.KS) {  // whole tile in registers
        wide_epilogue<C, RANGE>(x, acc, t, row_base, col_base, lane);
      } else {                    // partial sums of a stream-K tile
        const int r = c_tile - x.plan.dp_waves * x.G;
        const int Sr = C::GENERIC ? x.S : C::S;
        double* sc = x.sk_scratch + (size_t)r * (Sr * C::BM * C::BN) + (size_t)t * 64 + lane * 2;
#pragma unroll
        for (int s = S0; s < S1; s++) {
          if (C::GENERIC && s >= Sr) break;
          atomicAdd(sc + (size_t)s * (C::TILES * 64), acc[s - S0][0]);
          atomicAdd(sc + (size_t)s * (C::TILES * 64) + 1, acc[s - S0][1]);
        }
        __threadfence();
        __syncthreads();
        if (tid == 0) {
          const unsigned int mine = (unsigned int)(c_s1 - c_s0);
          *x.last_flag = (atomicAdd(&x.sk_counters[r], mine) + mine == (unsigned int)x.KS);
        }
        __syncthreads();
        if (*x.last_flag) {  // every slab of the tile has been added: read the totals back and finish the tile
          __threadfence();
#pragma unroll
          for (int s = S0; s < S1; s++) {
            if (C::GENERIC && s >= Sr) break;
            const double2 v = __ldcg(reinterpret_cast<const double2*>(sc + (size_t)s * (C::TILES * 64)));
            acc[s - S0][0] = v.x;
            acc[s - S0][1] = v.y;
          }
          wide_epilogue<C, RANGE>(x, acc, t, row_base, col_base, lane);
        }
      }
#pragma unroll
      for (int s = 0; s < W; s++) acc[s][0] = acc[s][1] = 0.0;
      if (++c_seg < x.n_seg) {
        x.segment(c_seg, c_tile, c_s0, c_s1);
        c_left = c_s1 - c_s0;
      }
    }
  }
}

template <class C>
__global__ void __launch_bounds__(C::THREADS, 1)
qgemm_wide_kernel(int m, int n, int Qr, int Sr, SkPlan plan, const double* __restrict__ Ap, const double* __restrict__ Bp,
                  double* __restrict__ order_planes, double* __restrict__ C_planes, double* __restrict__ sk_scratch,
                  unsigned int* __restrict__ sk_counters) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr int STAGES = C::STAGES;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

  WideCtx x;
  x.m = m, x.n = n, x.G = gridDim.x, x.cta = blockIdx.x, x.KS = plan.KS, x.plan = plan;
  x.Q = C::GENERIC ? Qr : C::Q, x.S = C::GENERIC ? Sr : C::S;
  x.a_chunk = x.Q * C::AQ, x.b_chunk = x.Q * C::BQ;
  x.Ap = Ap, x.Bp = Bp, x.order_planes = order_planes, x.C_planes = C_planes;
  x.sk_scratch = sk_scratch, x.sk_counters = sk_counters;
  x.stages = reinterpret_cast<double*>(smem_raw);
  uint64_t* const full = reinterpret_cast<uint64_t*>(smem_raw + STAGES * C::STAGE_BYTES);
  x.stages_u32 = smem_u32(x.stages);
  x.full_u32 = smem_u32(full);
  x.empty_u32 = x.full_u32 + 8 * STAGES;
  x.last_flag = reinterpret_cast<volatile int*>(smem_raw + STAGES * C::STAGE_BYTES + C::BAR_BYTES - 8);
  x.xchg = reinterpret_cast<double*>(smem_raw + STAGES * C::STAGE_BYTES + C::BAR_BYTES);

  // this CTA's segment list: its share of the stream-K slabs first, then whole tiles cta, cta + G, ...
  const int sk_total = plan.sk_tiles * plan.KS;
  x.g0 = min(x.cta * plan.sk_iters_per_cta, sk_total);
  x.g1 = min(x.g0 + plan.sk_iters_per_cta, sk_total);
  x.n_sk = x.g1 > x.g0 ? (x.g1 - 1) / plan.KS - x.g0 / plan.KS + 1 : 0;
  x.n_seg = x.n_sk + plan.dp_waves;
  x.total_slabs = (x.g1 - x.g0) + plan.dp_waves * plan.KS;

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < STAGES; s++) {
      mbar_init(x.full_u32 + 8 * s, 1);
      mbar_init(x.empty_u32 + 8 * s, C::WARPS);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (x.total_slabs == 0) return;

  const int t = C::tile_of(warp);
  if constexpr (C::R == 1) {
    wide_consume<C, 0>(x, t, lane, tid);
  } else {
    if constexpr (C::R == 2) {
      if (C::range_of(warp) == 0) wide_consume<C, 0>(x, t, lane, tid);  // warp-uniform
      else wide_consume<C, 1>(x, t, lane, tid);
    } else {
      switch (C::range_of(warp)) {  // warp-uniform
        case 0: wide_consume<C, 0>(x, t, lane, tid); break;
        case 1: wide_consume<C, 1>(x, t, lane, tid); break;
        case 2: wide_consume<C, 2>(x, t, lane, tid); break;
        default: wide_consume<C, 3>(x, t, lane, tid); break;
      }
    }
  }
}

// =====================================================================================================================
// Hexa double with the paper's 64 quarters, ONE ORDER RANGE AT A TIME (HPCfg / qgemm_hd_passes_kernel).
//
// The 64 accumulator sets of an 8x8 tile do not fit one thread.  The kernel above therefore lets four warps share a tile, each
// with its own order range and its own fully unrolled k-step body -- 45 KB of straight-line code that the SM's instruction
// cache can not hold: it is streamed from the L1.5 on every iteration of the k loop (profiles/r04_qgemm_hd.md: 96.9 M instruction
// requests against 1.07 M for octo double) and the loop runs at 0.96 of the DMMA peak where one resident body runs at 0.99.
// Here every warp owns a whole 8x8 tile (32 x 16 CTA tile, as octo double) and walks the contraction FOUR times, once per order
// range, smallest orders first: during a pass all eight warps run the same body (about 10 KB, resident), keep that range's
// <= 32 accumulator sets in registers and at the end of the pass fold them into the element's (L+1)-term expansion -- exactly
// the order-by-order sequence of the recombination (R9), so the result equals the standalone md_renorm bit for bit.
// There is no chain across warps and no block-wide barrier at a tile end any more.  Price: the operand slabs are fetched from L2
// once per pass (of pass r only the quarters 0 .. hi(r) - 1, a prefix of the packed chunk), about 3x the L2 -> SM traffic of a
// kernel that is tensor-bound by two orders of magnitude.
// Work is cut along a VIRTUAL contraction of 4 KS slabs per tile (slab v = pass v / KS, k-slab v % KS), so the persistent
// stream-K schedule above applies unchanged: a CTA that owns part of a tile adds the order sums of its slabs into the tile's
// scratch (exact, R6) and the CTA that completes the count folds the totals range by range.
struct HPCfg {
  static constexpr int Q = 64, S = 64, L = 16, TM = 4, TN = 2, TILES = 8, WARPS = 8, THREADS = 256, PASSES = 4;
  static constexpr int BM = TM * 8, BN = TN * 8, BK = PACK_BK_WIDE;
  static constexpr int AQ = BK * BM, BQ = BK * BN, A_CHUNK = Q * AQ, B_CHUNK = Q * BQ;
  static constexpr int STAGE_BYTES = (A_CHUNK + B_CHUNK) * 8, BAR_BYTES = 128, STAGES = 2;
  static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + BAR_BYTES;
  static_assert(SMEM_BYTES <= SMEM_LIMIT, "two stages of all 64 quarters");
  // pass p works on range 3 - p: [55,64) [45,55) [32,45) [0,32) -- 540 / 505 / 507 / 528 products per k-step
  __host__ __device__ static constexpr int lo(int r) { return r == 0 ? 0 : r == 1 ? 32 : r == 2 ? 45 : 55; }
  __host__ __device__ static constexpr int hi(int r) { return r == 0 ? 32 : r == 1 ? 45 : r == 2 ? 55 : 64; }
};

// fold the orders [S0, S1) held in acc (smallest first) into the two (L+1)-term expansions of the thread
template <int S0, int S1>
__device__ __forceinline__ void hp_fold(const double (&acc)[32][2], double (&r0)[HPCfg::L + 1], double (&r1)[HPCfg::L + 1]) {
  constexpr int L = HPCfg::L;
  double tmp[S1 - S0][2];  // a local-memory copy: the loop over the orders is rolled (code size, see wide_epilogue)
#pragma unroll
  for (int i = 0; i < S1 - S0; i++) tmp[i][0] = acc[i][0], tmp[i][1] = acc[i][1];
  int s = S1 - 1;
#pragma unroll 1
  for (; s - 1 >= S0; s -= 2) {
    double xs[2][2] = {{tmp[s - S0][0], tmp[s - S0][1]}, {tmp[s - 1 - S0][0], tmp[s - 1 - S0][1]}};
    renorm_add2xN<L, 2>(r0, r1, xs);
  }
  if (s == S0) renorm_add2<L>(r0, r1, tmp[0][0], tmp[0][1]);
}

__global__ void __launch_bounds__(HPCfg::THREADS, 1)
qgemm_hd_passes_kernel(int m, int n, SkPlan plan, const double* __restrict__ Ap, const double* __restrict__ Bp,
                       double* __restrict__ order_planes, double* __restrict__ C_planes, double* __restrict__ sk_scratch,
                       unsigned int* __restrict__ sk_counters) {
  using C = HPCfg;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr int L = C::L, STAGE_DOUBLES = C::A_CHUNK + C::B_CHUNK;
  double* const stages = reinterpret_cast<double*>(smem_raw);
  const uint32_t stages_u32 = smem_u32(stages);
  const uint32_t full_u32 = smem_u32(smem_raw + C::STAGES * C::STAGE_BYTES), empty_u32 = full_u32 + 8 * C::STAGES;
  volatile int* const last_flag = reinterpret_cast<volatile int*>(smem_raw + C::STAGES * C::STAGE_BYTES + C::BAR_BYTES - 8);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int G = gridDim.x, cta = blockIdx.x;
  const int KSV = plan.KS, KSR = KSV / C::PASSES;  // virtual slabs per tile (plan.KS) = 4 x the real k-slabs

  // this CTA's segment list over the virtual slabs: its share of the stream-K slabs first, then whole tiles cta, cta + G, ...
  const int sk_total = plan.sk_tiles * KSV;
  const int g0 = min(cta * plan.sk_iters_per_cta, sk_total), g1 = min(g0 + plan.sk_iters_per_cta, sk_total);
  const int n_sk = g1 > g0 ? (g1 - 1) / KSV - g0 / KSV + 1 : 0;
  const int n_seg = n_sk + plan.dp_waves, total_slabs = (g1 - g0) + plan.dp_waves * KSV;
  auto segment = [&](int i, int& tile, int& s0, int& s1) {
    if (i < n_sk) {
      const int r = g0 / KSV + i;
      tile = plan.dp_waves * G + r, s0 = i == 0 ? g0 - r * KSV : 0, s1 = min(KSV, g1 - r * KSV);
    } else {
      tile = (i - n_sk) * G + cta, s0 = 0, s1 = KSV;
    }
  };
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < C::STAGES; s++) {
      mbar_init(full_u32 + 8 * s, 1);
      mbar_init(empty_u32 + 8 * s, C::WARPS);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (total_slabs == 0) return;

  const int t = warp, ti = t / C::TN, tj = t % C::TN;
  const int a_off = ti * 32 + lane, b_off = C::A_CHUNK + tj * 32 + lane;

  // ---- producer (thread 0): one slab ahead of the consumers in a two-stage ring ------------------------------------------
  int p_seg = -1, p_v = 0, p_end = 0, p_flat = 0, pst = 0, p_tm = 0, p_tn = 0;
  auto produce_one = [&]() {
    if (p_v == p_end) {
      int tile;
      segment(++p_seg, tile, p_v, p_end);
      raster_tile(tile, plan.tiles_m, plan.tiles_n, p_tm, p_tn, plan.group_m);
    }
    const int pass = p_v / KSR, ks = p_v - pass * KSR;
    const int nq = pass == 0 ? C::hi(3) : pass == 1 ? C::hi(2) : pass == 2 ? C::hi(1) : C::hi(0);  // quarters 0 .. hi - 1: a prefix of the chunk
    const uint32_t dst = stages_u32 + pst * C::STAGE_BYTES, bar = full_u32 + 8 * pst;
    mbar_expect_tx(bar, nq * (C::AQ + C::BQ) * 8);
    bulk_g2s(dst, Ap + ((size_t)p_tm * KSR + ks) * C::A_CHUNK, nq * C::AQ * 8, bar);
    bulk_g2s(dst + C::A_CHUNK * 8, Bp + ((size_t)p_tn * KSR + ks) * C::B_CHUNK, nq * C::BQ * 8, bar);
    p_v++;
    p_flat++;
    pst ^= 1;
  };
  auto produce = [&]() {  // top of consumer iteration `it`: slab it + 1 into the stage slab it - 1 was read from
    if (p_flat < total_slabs) {
      if (p_flat >= C::STAGES) mbar_wait(empty_u32 + 8 * pst, ((p_flat / C::STAGES) + 1) & 1);
      produce_one();
    }
  };
  if (tid == 0) produce_one();

  // ---- consumers ---------------------------------------------------------------------------------------------------------
  // The two (L+1)-term expansions of the thread live in LOCAL memory between the passes (68 registers that the k loop of range 0
  // -- 128 accumulator and 64 operand registers -- does not have): ex is only ever indexed through `zoff`, a run-time zero the
  // compiler can not fold, so it is never promoted to registers; they are loaded into registers for a fold and stored back.
  double acc[32][2], ex[2 * (L + 1)];
  const int zoff = plan.flush_slabs;  // 0 (make_sk_plan)
  auto zero_acc = [&]() {
#pragma unroll
    for (int s = 0; s < 32; s++) acc[s][0] = acc[s][1] = 0.0;
  };
  auto zero_exp = [&]() {
#pragma unroll
    for (int l = 0; l < 2 * (L + 1); l++) ex[zoff + l] = 0.0;
  };
  auto load_exp = [&](double (&r0)[L + 1], double (&r1)[L + 1]) {
#pragma unroll
    for (int l = 0; l <= L; l++) r0[l] = ex[zoff + l], r1[l] = ex[zoff + L + 1 + l];
  };
  auto store_exp = [&](const double (&r0)[L + 1], const double (&r1)[L + 1]) {
#pragma unroll
    for (int l = 0; l <= L; l++) ex[zoff + l] = r0[l], ex[zoff + L + 1 + l] = r1[l];
  };
  zero_acc();
  zero_exp();
  int c_seg = 0, c_tile, c_s0, c_s1;
  segment(0, c_tile, c_s0, c_s1);
  int c_v = c_s0;
  const size_t planeC = (size_t)m * n;
  const bool vec_ok = (n % 2 == 0) && (((uintptr_t)C_planes | (uintptr_t)order_planes) % 16 == 0);
  // what is done with the accumulators of range r at the end of a pass (or of the CTA's part of it)
  auto range_done = [&](int r, bool whole, int rsk, size_t at, bool inside, bool two) {
    const int S0 = r == 0 ? C::lo(0) : r == 1 ? C::lo(1) : r == 2 ? C::lo(2) : C::lo(3);
    const int W = (r == 0 ? C::hi(0) : r == 1 ? C::hi(1) : r == 2 ? C::hi(2) : C::hi(3)) - S0;
    if (!whole) {  // stream-K part: exact fp64 reduction through the tile's scratch
      double* sc = sk_scratch + (size_t)rsk * (C::S * C::BM * C::BN) + (size_t)t * 64 + lane * 2;
#pragma unroll
      for (int i = 0; i < 32; i++)
        if (i < W) {
          atomicAdd(sc + (size_t)(S0 + i) * (C::TILES * 64), acc[i][0]);
          atomicAdd(sc + (size_t)(S0 + i) * (C::TILES * 64) + 1, acc[i][1]);
        }
      return;
    }
    if (order_planes && inside) {
#pragma unroll
      for (int i = 0; i < 32; i++)
        if (i < W) {
          if (vec_ok) {
            *reinterpret_cast<double2*>(order_planes + (size_t)(S0 + i) * planeC + at) = make_double2(acc[i][0], acc[i][1]);
          } else {
            order_planes[(size_t)(S0 + i) * planeC + at] = acc[i][0];
            if (two) order_planes[(size_t)(S0 + i) * planeC + at + 1] = acc[i][1];
          }
        }
    }
    if (C_planes) {
      double r0[L + 1], r1[L + 1];
      load_exp(r0, r1);
      switch (r) {
        case 0: hp_fold<C::lo(0), C::hi(0)>(acc, r0, r1); break;
        case 1: hp_fold<C::lo(1), C::hi(1)>(acc, r0, r1); break;
        case 2: hp_fold<C::lo(2), C::hi(2)>(acc, r0, r1); break;
        default: hp_fold<C::lo(3), C::hi(3)>(acc, r0, r1); break;
      }
      store_exp(r0, r1);
    }
  };
  auto write_C = [&](size_t at, bool inside, bool two) {  // after range 0: finish the expansions and write the limb planes once
    if (C_planes) {
      double r0[L + 1], r1[L + 1], o0[L], o1[L];
      load_exp(r0, r1);
      renorm_finish2<L>(r0, r1, o0, o1);
      if (inside) {
#pragma unroll
        for (int l = 0; l < L; l++) {
          if (vec_ok) {
            *reinterpret_cast<double2*>(C_planes + l * planeC + at) = make_double2(o0[l], o1[l]);
          } else {
            C_planes[l * planeC + at] = o0[l];
            if (two) C_planes[l * planeC + at + 1] = o1[l];
          }
        }
      }
    }
    zero_exp();
  };

  int st = 0;
  uint32_t phase = 0;
  // a RUN = the slabs of one pass inside the current segment: a tight loop with the range fixed at compile time
  auto run = [&](auto rc, int count) {
    constexpr int R_ = decltype(rc)::value;
    for (int i = 0; i < count; i++) {
      if (tid == 0) produce();
      mbar_wait(full_u32 + 8 * st, phase);
      const double* stage = stages + (size_t)st * STAGE_DOUBLES;
      k_step_range<C::Q, C::lo(R_), C::hi(R_), C::AQ, C::BQ>(reinterpret_cast<double(&)[C::hi(R_) - C::lo(R_)][2]>(acc), stage + a_off,
                                                             stage + b_off);
      __syncwarp();
      if (lane == 0) mbar_arrive(empty_u32 + 8 * st);
      st ^= 1;
      if (st == 0) phase ^= 1;
    }
  };
  for (int it = 0; it < total_slabs;) {
    const int pass = c_v / KSR, r = C::PASSES - 1 - pass;
    const int run_end = min(c_s1, (pass + 1) * KSR), count = run_end - c_v;
    switch (r) {
      case 0: run(std::integral_constant<int, 0>{}, count); break;
      case 1: run(std::integral_constant<int, 1>{}, count); break;
      case 2: run(std::integral_constant<int, 2>{}, count); break;
      default: run(std::integral_constant<int, 3>{}, count); break;
    }
    it += count;
    c_v = run_end;
    const bool seg_end = c_v == c_s1;
    {
      int tm, tn;
      raster_tile(c_tile, plan.tiles_m, plan.tiles_n, tm, tn, plan.group_m);
      const int row = tm * C::BM + ti * 8 + (lane >> 2), col = tn * C::BN + tj * 8 + 2 * (lane & 3);
      const bool inside = row < m && col < n, two = col + 1 < n, whole = c_s1 - c_s0 == KSV;
      const size_t at = (size_t)row * n + col;
      const int rsk = c_tile - plan.dp_waves * G;
      range_done(r, whole, rsk, at, inside, two);
      zero_acc();
      if (whole && r == 0) write_C(at, inside, two);
      if (seg_end) {
        if (!whole) {
          __threadfence();
          __syncthreads();
          if (tid == 0) {
            const unsigned int mine = (unsigned int)(c_s1 - c_s0);
            *last_flag = (atomicAdd(&sk_counters[rsk], mine) + mine == (unsigned int)KSV);
          }
          __syncthreads();
          if (*last_flag) {  // every virtual slab of the tile has been added: the totals, range by range, smallest orders first
            __threadfence();
            const double* sc = sk_scratch + (size_t)rsk * (C::S * C::BM * C::BN) + (size_t)t * 64 + lane * 2;
            for (int rr = C::PASSES - 1; rr >= 0; rr--) {
              const int S0 = rr == 0 ? C::lo(0) : rr == 1 ? C::lo(1) : rr == 2 ? C::lo(2) : C::lo(3);
              const int W = (rr == 0 ? C::hi(0) : rr == 1 ? C::hi(1) : rr == 2 ? C::hi(2) : C::hi(3)) - S0;
#pragma unroll
              for (int i = 0; i < 32; i++)
                if (i < W) {
                  const double2 v = __ldcg(reinterpret_cast<const double2*>(sc + (size_t)(S0 + i) * (C::TILES * 64)));
                  acc[i][0] = v.x, acc[i][1] = v.y;
                }
              range_done(rr, true, rsk, at, inside, two);
            }
            zero_acc();
            write_C(at, inside, two);
          }
        }
        if (++c_seg < n_seg) {
          segment(c_seg, c_tile, c_s0, c_s1);
          c_v = c_s0;
        }
      }
    }
  }
}

cudaError_t launch_hd_passes(int m, int n, int k, const double* Ap, const double* Bp, double* order_planes, double* C_planes,
                             void* sk_ws, cudaStream_t stream) {
  using C = HPCfg;
  const int tiles_m = (m + C::BM - 1) / C::BM, tiles_n = (n + C::BN - 1) / C::BN;
  const long long KSR = ((long long)k + C::BK - 1) / C::BK;
  if ((long long)tiles_m * tiles_n > 0x7fffffffLL || KSR * C::PASSES > 0x7fffffffLL) return cudaErrorInvalidValue;
  const int G = sk_grid();
  if (G <= 0) return cudaErrorInvalidDevice;
  const SkPlan plan = make_sk_plan(tiles_m, tiles_n, (int)(KSR * C::PASSES), G);  // the VIRTUAL slab count: four passes over k
  unsigned int* counters = static_cast<unsigned int*>(sk_ws);
  double* scratch = reinterpret_cast<double*>(static_cast<char*>(sk_ws) + SK_COUNTER_BYTES);
  cudaError_t err;
  if (plan.sk_tiles > 0) {
    err = cudaMemsetAsync(sk_ws, 0, SK_COUNTER_BYTES + sizeof(double) * (size_t)plan.sk_tiles * C::S * C::BM * C::BN, stream);
    if (err != cudaSuccess) return err;
  }
  static bool attr_done[MD_MAX_DEVICES] = {};
  const int dev = current_device();
  if (dev < 0 || dev >= MD_MAX_DEVICES || !attr_done[dev]) {
    err = cudaFuncSetAttribute(qgemm_hd_passes_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES);
    if (err != cudaSuccess) return err;
    if (dev >= 0 && dev < MD_MAX_DEVICES) attr_done[dev] = true;
  }
  qgemm_hd_passes_kernel<<<G, C::THREADS, C::SMEM_BYTES, stream>>>(m, n, plan, Ap, Bp, order_planes, C_planes, scratch, counters);
  return cudaGetLastError();
}

template <class C>
cudaError_t launch_wide_cfg(int m, int n, int k, int Q, int S, const double* Ap, const double* Bp, double* order_planes,
                            double* C_planes, void* sk_ws, cudaStream_t stream) {
  static_assert(C::GENERIC || (C::BM == pack_bx(C::L, C::Q, 0) && C::BN == pack_bx(C::L, C::Q, 1) && C::BK == pack_bk(C::L)),
                "tile shape must match the packed layout");
  static_assert(!C::GENERIC || (C::BM == pack_bx_generic(C::L, 0) && C::BN == pack_bx_generic(C::L, 1)),
                "tile shape must match the packed layout of the generic instances");
  if (C::GENERIC ? (Q < 1 || Q > C::Q || S < 1 || S > C::S || S > 2 * Q - 1) : (Q != C::Q || S != C::S)) return cudaErrorInvalidValue;
  const int tiles_m = (m + C::BM - 1) / C::BM, tiles_n = (n + C::BN - 1) / C::BN;
  if ((long long)tiles_m * tiles_n > 0x7fffffffLL) return cudaErrorInvalidValue;
  const int G = sk_grid();
  if (G <= 0) return cudaErrorInvalidDevice;
  const SkPlan plan = make_sk_plan(tiles_m, tiles_n, (k + C::BK - 1) / C::BK, G);
  unsigned int* counters = static_cast<unsigned int*>(sk_ws);
  double* scratch = reinterpret_cast<double*>(static_cast<char*>(sk_ws) + SK_COUNTER_BYTES);
  cudaError_t err;
  if (plan.sk_tiles > 0) {  // counters and the scratch tiles in use start at zero (one contiguous region)
    err = cudaMemsetAsync(sk_ws, 0, SK_COUNTER_BYTES + sizeof(double) * (size_t)plan.sk_tiles * S * C::BM * C::BN, stream);
    if (err != cudaSuccess) return err;
  }
  auto kern = qgemm_wide_kernel<C>;
  static bool attr_done[MD_MAX_DEVICES] = {};  // the shared-memory opt-in is per function and device: once, not per launch
  const int dev = current_device();
  if (dev < 0 || dev >= MD_MAX_DEVICES || !attr_done[dev]) {
    err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES);
    if (err != cudaSuccess) return err;
    if (dev >= 0 && dev < MD_MAX_DEVICES) attr_done[dev] = true;
  }
  kern<<<G, C::THREADS, C::SMEM_BYTES, stream>>>(m, n, Q, S, plan, Ap, Bp, order_planes, C_planes, scratch, counters);
  return cudaGetLastError();
}

using WCfgOD = WCfg<32, 8, 4, 2, 1>;   // octo double: 32 x 16 CTA tile, 8 tiles x 1 range
using WCfgOD22 = WCfg<22, 8, 4, 2, 1>; // octo double in 22 slices of 19 bits (MD_OPT_SLICE_BITS; R14)
using WCfgHD = WCfg<64, 16, 2, 1, 4>;  // hexa double, 16 x 8 CTA tile, 2 tiles x 4 ranges: round 1's kernel, no longer launched (qgemm_hd_passes_kernel)
using WCfgHD44 = WCfg<44, 16, 2, 2, 2>;  // hexa double in 44 slices of 19 bits: 16 x 16 CTA tile, 4 tiles x 2 ranges
// GENERIC instances: runtime (Q, S) up to these maxima
using WCfgGenDD = WCfg<GENERIC_QMAX_DD, 2, 4, 2, 1, GENERIC_SMAX_DD, true>;
using WCfgGenQD = WCfg<GENERIC_QMAX_QD, 4, 4, 2, 1, GENERIC_SMAX_QD, true>;
using WCfgGenOD = WCfg<GENERIC_QMAX_OD, 8, 2, 2, 2, GENERIC_SMAX_OD, true>;
using WCfgGenHD = WCfg<GENERIC_QMAX_HD, 16, 2, 1, 4, GENERIC_SMAX_HD, true>;

}  // namespace

bool qgemm_wide_supported(int limbs, int quarters) {
  return (limbs == 8 && (quarters == 32 || quarters == 22)) || (limbs == 16 && (quarters == 64 || quarters == 44));
}

int qgemm_generic_max_quarters(int limbs) {
  return limbs == 2 ? GENERIC_QMAX_DD : limbs == 4 ? GENERIC_QMAX_QD : limbs == 8 ? GENERIC_QMAX_OD : limbs == 16 ? GENERIC_QMAX_HD : 0;
}
int qgemm_generic_max_orders(int limbs) {
  return limbs == 2 ? GENERIC_SMAX_DD : limbs == 4 ? GENERIC_SMAX_QD : limbs == 8 ? GENERIC_SMAX_OD : limbs == 16 ? GENERIC_SMAX_HD : 0;
}
bool qgemm_generic_supported(int limbs, int quarters, int orders) {
  const int qmax = qgemm_generic_max_quarters(limbs), smax = qgemm_generic_max_orders(limbs);
  return qmax > 0 && quarters >= 1 && quarters <= qmax && orders >= 1 && orders <= smax && orders <= 2 * quarters - 1;
}

cudaError_t launch_qgemm_wide(int m, int n, int k, int limbs, int quarters, const double* Ap, const double* Bp,
                              double* order_planes, double* C_planes, void* sk_ws, cudaStream_t stream,
                              uint64_t* launches) {
  cudaError_t err = cudaErrorInvalidValue;
  const int Q = quarters;
  if (limbs == 8 && quarters == 32) err = launch_wide_cfg<WCfgOD>(m, n, k, Q, Q, Ap, Bp, order_planes, C_planes, sk_ws, stream);
  if (limbs == 8 && quarters == 22) err = launch_wide_cfg<WCfgOD22>(m, n, k, Q, Q, Ap, Bp, order_planes, C_planes, sk_ws, stream);
  if (limbs == 16 && quarters == 44) err = launch_wide_cfg<WCfgHD44>(m, n, k, Q, Q, Ap, Bp, order_planes, C_planes, sk_ws, stream);
  if (limbs == 16 && quarters == 64) err = launch_hd_passes(m, n, k, Ap, Bp, order_planes, C_planes, sk_ws, stream);
  if (err == cudaSuccess) *launches += 1;
  return err;
}

cudaError_t launch_qgemm_generic(int m, int n, int k, int limbs, int quarters, int orders, const double* Ap, const double* Bp,
                                 double* order_planes, double* C_planes, void* sk_ws, cudaStream_t stream, uint64_t* launches) {
  cudaError_t err = cudaErrorInvalidValue;
  if (!qgemm_generic_supported(limbs, quarters, orders)) return err;
  if (limbs == 2) err = launch_wide_cfg<WCfgGenDD>(m, n, k, quarters, orders, Ap, Bp, order_planes, C_planes, sk_ws, stream);
  if (limbs == 4) err = launch_wide_cfg<WCfgGenQD>(m, n, k, quarters, orders, Ap, Bp, order_planes, C_planes, sk_ws, stream);
  if (limbs == 8) err = launch_wide_cfg<WCfgGenOD>(m, n, k, quarters, orders, Ap, Bp, order_planes, C_planes, sk_ws, stream);
  if (limbs == 16) err = launch_wide_cfg<WCfgGenHD>(m, n, k, quarters, orders, Ap, Bp, order_planes, C_planes, sk_ws, stream);
  if (err == cudaSuccess) *launches += 1;
  return err;
}

}  // namespace md
