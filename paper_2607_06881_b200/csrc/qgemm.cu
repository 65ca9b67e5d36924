// qgemm.cu -- steps a3 + a4 of the hot path (include/mdgemm.h: md_qgemm; the fused kernel behind md_gemm).
//
//   For s = 0..S-1:  C^(s) = sum_{p+q=s} A_p * B_q      (PAPER.md:66-71 eq. 3; :75-78 eq. 4: the paper's C_{s+1})
//   C = sum_s C^(s), summed error free into L limbs     (PAPER.md:88-91 steps 4-5)
//
// The paper materialises Abar = [A_0 .. A_7] and the block-Toeplitz Bbar and runs one plain DGEMM, which multiplies all
// 64 blocks (zeros included) and then re-reads Cbar to add the parts.  Here the triangular set of T = S(S+1)/2 quarter
// products is issued directly: a CTA stages ALL Q quarter tiles of an A block and a B block of one k-slab in shared
// memory once (cp.async, multi-stage), every warp loads each quarter fragment once per k-step and feeds it to all the
// products that need it, each order s has its own register accumulators, and the epilogue renormalises in registers and
// writes the L limb planes of C once.
//
// FP64 tensor pipe: tcgen05.mma has no f64 kind on sm_100a (ptxas: "Unknown modifier '.kind::f64'"), so the pipe is
// reached through warp-level mma.sync.m8n8k4.f64, which is SASS DMMA.8x8x4 -- the only FP64 MMA shape sm_100a has (the
// larger PTX shapes are split into it).  Measured peak on B200: 128 flop/clk/SM (37.0 TFLOP/s at 1.955 GHz), one DMMA
// per 16 cycles per SM sub-partition, latency ~26 cycles: two independent accumulators per warp already saturate it.
//
// Exactness: quarters are integers |D| <= 2^13 times the group unit, products are <= 2^26 units, and with k*S <= 2^27 every
// partial sum stays below 2^53 units, so each fp64 FMA inside DMMA is exact and the result is independent of the
// order in which the hardware or this kernel adds things (eq. 5; R6).
#include "md_kernels.h"
#include "qgemm_common.cuh"

namespace md {
namespace {

// cp.async of BYTES (8 or 16) with zero fill when !valid (src-size 0: nothing is read).
template <int BYTES>
__device__ __forceinline__ void cp_async(void* smem_dst, const void* gmem_src, bool valid) {
  const unsigned dst = (unsigned)__cvta_generic_to_shared(smem_dst);
  const int src_size = valid ? BYTES : 0;
  if (BYTES == 16)
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(gmem_src), "r"(src_size) : "memory");
  else
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(dst), "l"(gmem_src), "r"(src_size) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// Tile configuration.  A warp owns an (8*MT) x (8*NT) block of C and Q (= S) accumulator sets for it.
//   shared memory, per stage:  As[Q][BM][LDA]  (k contiguous, as in the row-major A planes)
//                              Bs[Q][BK][LDB]  (n contiguous, as in the row-major B planes)
//   LDA, LDB == 4 (mod 16) doubles (or LDA == 12): the 16 lanes of a half warp (4 rows x 4 k, or 4 k x 4 columns) then
//   hit 16 different 8-byte bank pairs -> conflict-free LDS.64 fragment loads.
template <int Q_, int L_, int BM_, int BN_, int BK_, int WM_, int WN_>
struct Cfg {
  static constexpr int Q = Q_, S = Q_, L = L_, BM = BM_, BN = BN_, BK = BK_, WM = WM_, WN = WN_;
  static constexpr int THREADS = WM * WN * 32;
  static constexpr int MT = BM / WM / 8, NT = BN / WN / 8;
  static constexpr int LDA = BK + 4, LDB = BN + 4;
  static constexpr int A_STAGE = Q * BM * LDA, B_STAGE = Q * BK * LDB;  // doubles
  static constexpr int STAGE_BYTES = (A_STAGE + B_STAGE) * 8;
  static constexpr int STAGES = (SMEM_LIMIT / STAGE_BYTES) < 4 ? (SMEM_LIMIT / STAGE_BYTES) : 4;
  static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES;
  static_assert(BM % (WM * 8) == 0 && BN % (WN * 8) == 0 && BK % 4 == 0, "tile shape");
  static_assert(LDA % 16 == 4 || LDA % 16 == 12, "A fragment loads would bank-conflict");
  static_assert(LDB % 16 == 4 || LDB % 16 == 12, "B fragment loads would bank-conflict");
  static_assert(STAGES >= 2, "not enough shared memory for double buffering");
};

// One k-slab (BK deep) of all Q quarter planes of the A block and the B block -> shared memory stage.
// CH = doubles per cp.async (2 when rows are 16-byte aligned, else 1).  Out-of-range rows / columns / k are zero filled:
// zero quarters are harmless.
template <class C, int CH>
__device__ __forceinline__ void load_stage(double* As, double* Bs, const double* __restrict__ Aq,
                                           const double* __restrict__ Bq, int m, int n, int k, int m0, int n0, int k0,
                                           int tid) {
  constexpr int KC = C::BK / CH;            // chunks per A row
  constexpr int A_CHUNKS = C::BM * KC;      // per plane
  constexpr int NC = C::BN / CH;            // chunks per B row
  constexpr int B_CHUNKS = C::BK * NC;      // per plane
  const size_t planeA = (size_t)m * k, planeB = (size_t)k * n;
#pragma unroll
  for (int c = tid; c < C::Q * A_CHUNKS; c += C::THREADS) {
    const int p = c / A_CHUNKS, rem = c % A_CHUNKS;
    const int row = rem / KC, kc = (rem % KC) * CH;
    const bool valid = (m0 + row < m) && (k0 + kc < k);  // CH == 2 implies k even: both doubles valid together
    const double* src = valid ? Aq + p * planeA + (size_t)(m0 + row) * k + (k0 + kc) : Aq;
    cp_async<CH * 8>(As + (p * C::BM + row) * C::LDA + kc, src, valid);
  }
#pragma unroll
  for (int c = tid; c < C::Q * B_CHUNKS; c += C::THREADS) {
    const int q = c / B_CHUNKS, rem = c % B_CHUNKS;
    const int kk = rem / NC, nc = (rem % NC) * CH;
    const bool valid = (k0 + kk < k) && (n0 + nc < n);
    const double* src = valid ? Bq + q * planeB + (size_t)(k0 + kk) * n + (n0 + nc) : Bq;
    cp_async<CH * 8>(Bs + (q * C::BK + kk) * C::LDB + nc, src, valid);
  }
}

template <class C, int CH>
__global__ void __launch_bounds__(C::THREADS, 1)
qgemm_kernel(int m, int n, int k, int tiles_m, int tiles_n, const double* __restrict__ Aq,
             const double* __restrict__ Bq, double* __restrict__ order_planes, double* __restrict__ C_planes) {
  extern __shared__ __align__(16) double smem[];
  constexpr int Q = C::Q, S = C::S, L = C::L, MT = C::MT, NT = C::NT;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp / C::WN, wn = warp % C::WN;
  const int g = lane >> 2, t4 = lane & 3;  // DMMA fragment coordinates: A[g][t4], B[t4][g], C[g][2*t4 + {0,1}]

  int tm, tn;
  raster_tile(blockIdx.x, tiles_m, tiles_n, tm, tn);
  const int m0 = tm * C::BM, n0 = tn * C::BN;

  double acc[S][MT][NT][2];
#pragma unroll
  for (int s = 0; s < S; s++)
#pragma unroll
    for (int i = 0; i < MT; i++)
#pragma unroll
      for (int j = 0; j < NT; j++) acc[s][i][j][0] = acc[s][i][j][1] = 0.0;

  const int KT = (k + C::BK - 1) / C::BK;
  auto stage_A = [&](int st) { return smem + st * (C::A_STAGE + C::B_STAGE); };
  auto stage_B = [&](int st) { return smem + st * (C::A_STAGE + C::B_STAGE) + C::A_STAGE; };

#pragma unroll
  for (int st = 0; st < C::STAGES - 1; st++) {
    if (st < KT) load_stage<C, CH>(stage_A(st), stage_B(st), Aq, Bq, m, n, k, m0, n0, st * C::BK, tid);
    cp_async_commit();
  }

  for (int kt = 0; kt < KT; kt++) {
    cp_async_wait<C::STAGES - 2>();  // slab kt has landed (for this thread's copies) ...
    __syncthreads();                 // ... and for everyone's; also: everyone is done reading slab kt-1
    {
      const int nxt = kt + C::STAGES - 1;  // refill the stage that slab kt-1 occupied
      if (nxt < KT) load_stage<C, CH>(stage_A(nxt % C::STAGES), stage_B(nxt % C::STAGES), Aq, Bq, m, n, k, m0, n0, nxt * C::BK, tid);
      cp_async_commit();
    }
    const double* As = stage_A(kt % C::STAGES) + (wm * MT * 8 + g) * C::LDA + t4;
    const double* Bs = stage_B(kt % C::STAGES) + t4 * C::LDB + wn * NT * 8 + g;
#pragma unroll
    for (int k4 = 0; k4 < C::BK / 4; k4++) {
      double a[Q][MT];
#pragma unroll
      for (int p = 0; p < Q; p++)
#pragma unroll
        for (int i = 0; i < MT; i++) a[p][i] = As[(p * C::BM + i * 8) * C::LDA + k4 * 4];
#pragma unroll
      for (int q = 0; q < Q; q++) {
        double b[NT];
#pragma unroll
        for (int j = 0; j < NT; j++) b[j] = Bs[(q * C::BK + k4 * 4) * C::LDB + j * 8];
#pragma unroll
        for (int p = 0; p + q < S; p++)  // product (p, q) goes to order s = p + q: consecutive DMMAs hit different accumulators
#pragma unroll
          for (int i = 0; i < MT; i++)
#pragma unroll
            for (int j = 0; j < NT; j++) dmma_8x8x4(acc[p + q][i][j], a[p][i], b[j]);
      }
    }
  }
  cp_async_wait<0>();

  qgemm_epilogue<S, L, MT, NT>(acc, m, n, m0 + wm * MT * 8, n0 + wn * NT * 8, lane, order_planes, C_planes);
}

template <class C>
cudaError_t launch_cfg(int m, int n, int k, const double* Aq, const double* Bq, double* order_planes,
                       double* C_planes, cudaStream_t stream) {
  const int tiles_m = (m + C::BM - 1) / C::BM, tiles_n = (n + C::BN - 1) / C::BN;
  const long long tiles = (long long)tiles_m * tiles_n;
  if (tiles > 0x7fffffffLL) return cudaErrorInvalidValue;
  const bool aligned = (k % 2 == 0) && (n % 2 == 0) && (((uintptr_t)Aq | (uintptr_t)Bq) % 16 == 0);
  auto kern = aligned ? qgemm_kernel<C, 2> : qgemm_kernel<C, 1>;
  cudaError_t err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES);
  if (err != cudaSuccess) return err;
  kern<<<(unsigned)tiles, C::THREADS, C::SMEM_BYTES, stream>>>(m, n, k, tiles_m, tiles_n, Aq, Bq, order_planes, C_planes);
  return cudaGetLastError();
}

// double double: 64 x 32 CTA tile, 8 warps (4 x 2), 16 x 16 warp tile.  quad double: 32 x 16 CTA tile, 8 x 8 warp tile
// (16 orders x 2 registers per 8x8 tile: one tile per warp keeps the accumulators in registers).
template <int Q> using CfgDD = Cfg<Q, 2, 64, 32, 8, 4, 2>;
template <int Q> using CfgQD = Cfg<Q, 4, 32, 16, 8, 4, 2>;

}  // namespace

bool qgemm_supported(int limbs, int quarters) {
  // 8-10 / 16-18: the paper's 13-bit quarters (R5); 6, 7 / 11, 12: wider slices (MD_OPT_SLICE_BITS, R14)
  return (limbs == 2 && quarters >= 6 && quarters <= 10) || (limbs == 4 && ((quarters >= 16 && quarters <= 18) || quarters == 11 || quarters == 12));
}

// md_plan_quarters: W~ = X * Y for two plain fp64 matrices (|A_0|, |B_0|) on the same DMMA kernel with one "quarter" and
// one order (no exactness needed there: all terms are non-negative, the relative error is k 2^-53).
cudaError_t launch_plain_dgemm(int m, int n, int k, const double* X, const double* Y, double* XY, cudaStream_t stream,
                               uint64_t* launches) {
  const cudaError_t err = launch_cfg<CfgDD<1>>(m, n, k, X, Y, XY, nullptr, stream);
  if (err == cudaSuccess) *launches += 1;
  return err;
}

cudaError_t launch_qgemm(int m, int n, int k, int limbs, int quarters, const double* Aq, const double* Bq,
                         double* order_planes, double* C_planes, cudaStream_t stream, uint64_t* launches) {
  cudaError_t err = cudaErrorInvalidValue;
  if (limbs == 2) {
    if (quarters == 6) err = launch_cfg<CfgDD<6>>(m, n, k, Aq, Bq, order_planes, C_planes, stream);
    if (quarters == 7) err = launch_cfg<CfgDD<7>>(m, n, k, Aq, Bq, order_planes, C_planes, stream);
    if (quarters == 8) err = launch_cfg<CfgDD<8>>(m, n, k, Aq, Bq, order_planes, C_planes, stream);
    if (quarters == 9) err = launch_cfg<CfgDD<9>>(m, n, k, Aq, Bq, order_planes, C_planes, stream);
    if (quarters == 10) err = launch_cfg<CfgDD<10>>(m, n, k, Aq, Bq, order_planes, C_planes, stream);
  } else if (limbs == 4) {
    if (quarters == 11) err = launch_cfg<CfgQD<11>>(m, n, k, Aq, Bq, order_planes, C_planes, stream);
    if (quarters == 12) err = launch_cfg<CfgQD<12>>(m, n, k, Aq, Bq, order_planes, C_planes, stream);
    if (quarters == 16) err = launch_cfg<CfgQD<16>>(m, n, k, Aq, Bq, order_planes, C_planes, stream);
    if (quarters == 17) err = launch_cfg<CfgQD<17>>(m, n, k, Aq, Bq, order_planes, C_planes, stream);
    if (quarters == 18) err = launch_cfg<CfgQD<18>>(m, n, k, Aq, Bq, order_planes, C_planes, stream);
  }
  if (err == cudaSuccess) *launches += 1;
  return err;
}

}  // namespace md
