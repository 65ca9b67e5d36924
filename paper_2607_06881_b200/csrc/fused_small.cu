// fused_small.cu -- the WHOLE hot path (steps a1-a4) in ONE launch, for problems too small to amortise the separate
// preparation: exponent vectors, Algorithm S and the quarter products of a tile all happen inside the CTA that owns the tile,
// the quarter planes never leave shared memory ("no quarter planes in HBM"; PAPER.md:82-89 five steps).
//
//   a1  E_i / F_j of the tile's 32 rows of A / 16 columns of B: maxima of the leading limbs over the WHOLE contraction, read by
//       every CTA of the tile's cluster for itself (a few KB from L2: cheaper than a cluster barrier)  (R2, R11)
//   a2  Algorithm S on the CTA's operand slabs, digits written straight into the fragment-major stage the DMMA warps read
//       (md_split.cuh: the same operations as split.cu, hence the same bits)          (R1-R4)
//   a3  the triangular set of quarter products on DMMA.8x8x4, one accumulator set per order   (eq. 3-4)
//   a4  partial order sums of the cluster's CTAs added through distributed shared memory (exact: DESIGN.md R6) -- CTA r of the
//       cluster collects and finishes 8 / Z of the eight 8x8 tiles of the 32 x 16 tile, so the reads and the renormalising
//       epilogue of qgemm_common.cuh are spread over the cluster
//
// Decomposition: a CTA tile is 32 x 16 of C (8 warps, one 8x8 DMMA tile each); a cluster of Z in {1, 2, 4, 8} CTAs shares a
// tile and cuts the contraction into Z runs of k-slabs, so that a 64^3 product occupies 64 SMs instead of 8.  Every CTA splits
// its own slabs (the A rows of a tile are split once per tile column: redundant arithmetic, but no workspace traffic, no second
// launch, no grid-wide barrier).  Chunks of two k-slabs are double buffered: the limbs of chunk c+1 are loaded into registers
// before the DMMAs of chunk c issue and split into the other buffer after them, one block barrier per chunk.
#include <cooperative_groups.h>

#include "md_kernels.h"
#include "md_split.cuh"
#include "qgemm_common.cuh"

namespace md {
namespace {

namespace cg = cooperative_groups;

template <int L_, int Q_, int S_ = Q_>
struct FCfg {
  static constexpr int L = L_, Q = Q_, S = S_;
  static constexpr int BM = 32, BN = 16, BK = 8, CS = 2, THREADS = 256;
  static constexpr int A_SLAB = Q * BK * BM, B_SLAB = Q * BK * BN, SLAB = A_SLAB + B_SLAB;  // doubles
  static constexpr int CHUNK = CS * SLAB;
  static constexpr int SMEM_BYTES = 2 * CHUNK * 8;
  static_assert(S * 2 * THREADS <= 2 * CHUNK, "the hand-over area of the cluster reduction reuses the stage buffers");
  static_assert(SMEM_BYTES <= SMEM_LIMIT, "two chunk buffers must fit");
};

template <class C>
__global__ void __launch_bounds__(C::THREADS, 1)
fused_small_kernel(int m, int n, int k, int bits, int exp_lo, int tiles_n, int KS, const double* __restrict__ A,
                   const double* __restrict__ B, double* __restrict__ order_planes, double* __restrict__ C_planes, uint32_t* flags) {
  constexpr int L = C::L, Q = C::Q, S = C::S;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double* const buf = reinterpret_cast<double*>(smem_raw);
  __shared__ uint32_t pmaxA[C::BM], pmaxB[C::BN];
  __shared__ int expA[C::BM], expB[C::BN];

  cg::cluster_group cluster = cg::this_cluster();
  const int Z = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
  const int tile = blockIdx.x / Z, tm = tile / tiles_n, tn = tile % tiles_n;
  const int row0 = tm * C::BM, col0 = tn * C::BN;
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5, wm = warp >> 1, wn = warp & 1;
  const int s0 = (int)((long long)rank * KS / Z), s1 = (int)((long long)(rank + 1) * KS / Z);  // this CTA's k-slabs
  const int k1 = min(k, s1 * C::BK);
  const size_t planeA = (size_t)m * k, planeB = (size_t)k * n;

  // ---- a2 + a3: chunks of CS = 2 slabs ---------------------------------------------------------------------------------------
  // Split assignment per chunk: A -- slab j = 0, 1: element (row x8*8+g, k kin = k4*4+t4) with (k4, x8) = (warp / 4, warp % 4),
  // digit q at A part + q*256 + t; B -- one element: slab jb = t / 128, (k4, x8) from (t % 128) / 32, digit q at B part + q*128 +
  // t % 128.  Both are the fragment-major order of md_packed.cuh, so lane 4g + t4 of a DMMA warp finds its operand at base + lane.
  const int g = lane >> 2, t4 = lane & 3;
  const int a_row = (warp & 3) * 8 + g, a_kin = (warp >> 2) * 4 + t4;
  const int tb = t & 127, jb = t >> 7, wb = tb >> 5;
  const int b_col = (wb & 1) * 8 + g, b_kin = (wb >> 1) * 4 + t4;
  const bool a_ok = row0 + a_row < m, b_ok = col0 + b_col < n;
  const double* a_src = A + (size_t)(a_ok ? row0 + a_row : 0) * k;
  const double* b_src = B + (b_ok ? col0 + b_col : 0);

  double ra[C::CS][L], rb[L];
  auto load_chunk = [&](int c) {
#pragma unroll
    for (int j = 0; j < C::CS; j++) {
      const int kk = (s0 + c * C::CS + j) * C::BK + a_kin;
      const bool ok = a_ok && kk < k1;
#pragma unroll
      for (int l = 0; l < L; l++) ra[j][l] = ok ? a_src[l * planeA + kk] : 0.0;
    }
    const int kk = (s0 + c * C::CS + jb) * C::BK + b_kin;
    const bool ok = b_ok && kk < k1;
#pragma unroll
    for (int l = 0; l < L; l++) rb[l] = ok ? b_src[l * planeB + (size_t)kk * n] : 0.0;
  };
  const int my_slabs = s1 - s0, nchunks = (my_slabs + C::CS - 1) / C::CS;
  if (nchunks > 0) load_chunk(0);  // in flight under the maxima

  // ---- a1: maxima of the leading limbs over the whole contraction -> exponents (every CTA of the cluster for itself) -------
  if (t < C::BN) pmaxB[t] = 0;
  __syncthreads();
  {
    const int row = t >> 3, sub = t & 7;
    uint32_t mx = 0;
    if (row0 + row < m) {
      const double* p = A + (size_t)(row0 + row) * k;
      for (int kk = sub; kk < k; kk += 8) mx = max(mx, abs_hi32(p[kk]));
    }
    mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, 1));
    mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, 2));
    mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, 4));
    if (sub == 0) pmaxA[row] = mx;
    const int col = t & 15, kr = t >> 4;
    mx = 0;
    if (col0 + col < n)
      for (int kk = kr; kk < k; kk += 16) mx = max(mx, abs_hi32(B[(size_t)kk * n + col0 + col]));
    if (mx) atomicMax(&pmaxB[col], mx);
  }
  __syncthreads();
  if (t < C::BM + C::BN) {
    const bool isA = t < C::BM;
    const uint32_t v = isA ? pmaxA[t] : pmaxB[t - C::BM];
    // range / non-finite flags once per group: from the first tile column (rows of A) / tile row (columns of B), rank 0
    const bool valid = isA ? row0 + t < m : col0 + (t - C::BM) < n;
    const bool report = rank == 0 && (isA ? tn == 0 : tm == 0);
    const int E = valid ? exponent_from_hi32(v, report ? flags : nullptr, exp_lo) : 0;
    if (isA) expA[t] = E;
    else expB[t - C::BM] = E;
  }
  __syncthreads();

  const int EA = expA[a_row], EB = expB[b_col];
  auto split_chunk = [&](double* dst) {
    bool bad = any_nonfinite<L>(rb);
#pragma unroll
    for (int j = 0; j < C::CS; j++) bad |= any_nonfinite<L>(ra[j]);
    if (bad && flags) atomicOr(flags, FLAG_NONFINITE);
#pragma unroll
    for (int q = 0; q < Q; q++) {
#pragma unroll
      for (int j = 0; j < C::CS; j++) dst[j * C::SLAB + q * 256 + t] = extract_digit<L>(ra[j], EA, q, bits);
      dst[jb * C::SLAB + C::A_SLAB + q * 128 + tb] = extract_digit<L>(rb, EB, q, bits);
    }
  };

  double acc[S][1][1][2];
#pragma unroll
  for (int s = 0; s < S; s++) acc[s][0][0][0] = acc[s][0][0][1] = 0.0;
  auto dmma_chunk = [&](const double* src, int slabs) {
    for (int j = 0; j < slabs; j++) {
      const double* As = src + j * C::SLAB + wm * 32 + lane;
      const double* Bs = src + j * C::SLAB + C::A_SLAB + wn * 32 + lane;
#pragma unroll
      for (int k4 = 0; k4 < 2; k4++) {
        double a[Q];
#pragma unroll
        for (int p = 0; p < Q; p++) a[p] = As[(p * 2 + k4) * 128];
#pragma unroll
        for (int q = 0; q < Q; q++) {
          const double b = Bs[(q * 2 + k4) * 64];
#pragma unroll
          for (int p = 0; p + q < S && p < Q; p++) dmma_8x8x4(acc[p + q][0][0], a[p], b);
        }
      }
    }
  };

  if (nchunks > 0) split_chunk(buf);
  __syncthreads();
  for (int c = 0; c < nchunks; c++) {
    const bool more = c + 1 < nchunks;
    if (more) load_chunk(c + 1);  // global loads in flight under the DMMAs
    dmma_chunk(buf + (c & 1) * C::CHUNK, min(C::CS, my_slabs - c * C::CS));
    if (more) split_chunk(buf + ((c + 1) & 1) * C::CHUNK);
    __syncthreads();
  }

  // ---- a4: the cluster's partial order sums (exact integers in units of the order: any order of addition), the epilogue ----
  if (Z > 1) {
    // every CTA publishes its accumulators: value (s, e) of warp w, lane l at buf[((w * S + s) * 2 + e) * 32 + l]
#pragma unroll
    for (int s = 0; s < S; s++) {
      buf[((warp * S + s) * 2) * 32 + lane] = acc[s][0][0][0];
      buf[((warp * S + s) * 2 + 1) * 32 + lane] = acc[s][0][0][1];
    }
    cluster.sync();
    // CTA `rank` finishes 8 / Z of the eight 8x8 tiles, one per warp: warp j < 8 / Z collects tile rank * (8 / Z) + j from all Z
    // CTAs.  The Z remote reads of one value are independent loads; the sums are exact (R6).
    const int per = 8 / Z;  // tiles per CTA
    if (warp < per) {
      const int w = rank * per + warp;
#pragma unroll
      for (int s = 0; s < S; s++) acc[s][0][0][0] = acc[s][0][0][1] = 0.0;
      for (int r = 0; r < Z; r++) {
        const double* other = cluster.map_shared_rank(buf, r) + (size_t)w * S * 64 + lane;
#pragma unroll
        for (int s = 0; s < S; s++) {
          acc[s][0][0][0] += other[(2 * s) * 32];
          acc[s][0][0][1] += other[(2 * s + 1) * 32];
        }
      }
      qgemm_epilogue<S, L, 1, 1>(acc, m, n, row0 + (w >> 1) * 8, col0 + (w & 1) * 8, lane, order_planes, C_planes);
    }
    cluster.sync();  // nobody leaves while its shared memory is still being read
    return;
  }
  qgemm_epilogue<S, L, 1, 1>(acc, m, n, row0 + wm * 8, col0 + wn * 8, lane, order_planes, C_planes);
}

template <class C>
cudaError_t launch_fs(int m, int n, int k, int bits, int exp_lo, int Z, const double* A, const double* B, double* order_planes,
                      double* C_planes, uint32_t* flags, cudaStream_t stream) {
  const int tiles_m = (m + C::BM - 1) / C::BM, tiles_n = (n + C::BN - 1) / C::BN, KS = (k + C::BK - 1) / C::BK;
  const long long blocks = (long long)tiles_m * tiles_n * Z;
  if (blocks > 0x7fffffffLL) return cudaErrorInvalidValue;
  auto kern = fused_small_kernel<C>;
  static bool attr_done[MD_MAX_DEVICES] = {};  // the shared-memory opt-in is per function and device: once, not per launch
  const int dev = current_device();
  if (dev < 0 || dev >= MD_MAX_DEVICES || !attr_done[dev]) {
    cudaError_t err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES);
    if (err != cudaSuccess) return err;
    if (dev >= 0 && dev < MD_MAX_DEVICES) attr_done[dev] = true;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)blocks);
  cfg.blockDim = dim3(C::THREADS);
  cfg.dynamicSmemBytes = C::SMEM_BYTES;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)Z;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, m, n, k, bits, exp_lo, tiles_n, KS, A, B, order_planes, C_planes, flags);
}

}  // namespace

bool fused_small_supported(int limbs, int quarters, int orders) {
  return (limbs == 2 && quarters == 8 && orders == 8) || (limbs == 4 && quarters == 16 && orders == 16);
}

// CTAs per cluster: as many k-runs per tile as keep the grid within one wave of the SMs (a power of two, at most 8, at most
// one per k-slab); 1 when the tiles alone fill the machine.
int fused_small_cluster(int m, int n, int k) {
  const long long tiles = (((long long)m + 31) / 32) * (((long long)n + 15) / 16);
  const int G = sk_grid(), KS = (k + 7) / 8;
  int Z = 8;
  while (Z > 1 && (tiles * Z > G || Z > KS)) Z >>= 1;
  return Z;
}

cudaError_t launch_fused_small(int m, int n, int k, int limbs, int quarters, int orders, int bits, const double* A, const double* B,
                               double* order_planes, double* C_planes, uint32_t* flags, cudaStream_t stream, uint64_t* launches) {
  if (!fused_small_supported(limbs, quarters, orders)) return cudaErrorInvalidValue;
  const int exp_lo = exponent_floor(quarters, bits), Z = fused_small_cluster(m, n, k);
  cudaError_t err = cudaErrorInvalidValue;
  if (limbs == 2) err = launch_fs<FCfg<2, 8>>(m, n, k, bits, exp_lo, Z, A, B, order_planes, C_planes, flags, stream);
  if (limbs == 4) err = launch_fs<FCfg<4, 16>>(m, n, k, bits, exp_lo, Z, A, B, order_planes, C_planes, flags, stream);
  if (err == cudaSuccess) *launches += 1;
  return err;
}

}  // namespace md
