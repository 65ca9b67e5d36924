// qgemm_common.cuh -- pieces shared by the two fused quarter-GEMM kernels of libmdgemm (qgemm.cu: plain quarter planes,
// cp.async staging; qgemm_packed.cu: fragment-major packed planes, bulk-copy + mbarrier pipeline): the DMMA wrapper,
// the order in which the triangular set of quarter products is issued, and the epilogue (steps a3 + a4,
// PAPER.md:66-78 eq. 3-4 and :88-91).  CUDA path only; nothing here is shared with oracle/.
#pragma once
#include "md_common.cuh"

namespace md {

constexpr int SMEM_LIMIT = 232448;  // 227 KB usable per CTA on sm_100a

// mma.sync.m8n8k4.f64 == SASS DMMA.8x8x4, the only FP64 tensor instruction of sm_100a (tcgen05.mma has no f64 kind).
// Fragment coordinates for lane = 4*g + t4:  A[g][t4], B[t4][g], C[g][2*t4 + {0,1}].
__device__ __forceinline__ void dmma_8x8x4(double (&c)[2], double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
      : "+d"(c[0]), "+d"(c[1])
      : "d"(a), "d"(b));
}

// Epilogue of one warp: acc[s][i][j][0..1] holds, for the 8x8 tile (i, j) of the warp's block of C whose top-left
// element is (row_base, col_base), the S order values of C[row][col], C[row][col+1] with row = row_base + 8i + g,
// col = col_base + 8j + 2*t4.  Writes the order planes C^(s) (debug / parity) and / or the renormalised limb planes.
template <int S, int L, int MT, int NT>
__device__ __forceinline__ void qgemm_epilogue(const double (&acc)[S][MT][NT][2], int m, int n, int row_base,
                                               int col_base, int lane, double* __restrict__ order_planes,
                                               double* __restrict__ C_planes) {
  const int g = lane >> 2, t4 = lane & 3;
  const size_t planeC = (size_t)m * n;
  const bool vec_ok = (n % 2 == 0) && (((uintptr_t)C_planes | (uintptr_t)order_planes) % 16 == 0);
#pragma unroll
  for (int i = 0; i < MT; i++) {
    const int row = row_base + i * 8 + g;
#pragma unroll
    for (int j = 0; j < NT; j++) {
      const int col = col_base + j * 8 + 2 * t4;
      if (row >= m || col >= n) continue;
      const size_t at = (size_t)row * n + col;
      const bool two = col + 1 < n;
      if (order_planes) {
#pragma unroll
        for (int s = 0; s < S; s++) {
          if (vec_ok) {
            *reinterpret_cast<double2*>(order_planes + s * planeC + at) = make_double2(acc[s][i][j][0], acc[s][i][j][1]);
          } else {
            order_planes[s * planeC + at] = acc[s][i][j][0];
            if (two) order_planes[s * planeC + at + 1] = acc[s][i][j][1];
          }
        }
      }
      if (C_planes) {
        double c0[S], c1[S], o0[L], o1[L];
#pragma unroll
        for (int s = 0; s < S; s++) {
          c0[s] = acc[s][i][j][0];
          c1[s] = acc[s][i][j][1];
        }
        renorm_orders<L, S>(c0, o0);
        renorm_orders<L, S>(c1, o1);
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
  }
}

// Epilogue of one warp in chunked mode (qgemm_packed.cu, R16): r[i][j][e] is the (L+1)-term expansion that has
// received every order value of every chunk; finish it (renorm_finish) and write the L limb planes.
template <int L, int MT, int NT>
__device__ __forceinline__ void chunk_epilogue(double (&r)[MT][NT][2][L + 1], int m, int n, int row_base, int col_base,
                                               int lane, double* __restrict__ C_planes) {
  const int g = lane >> 2, t4 = lane & 3;
  const size_t planeC = (size_t)m * n;
  const bool vec_ok = (n % 2 == 0) && ((uintptr_t)C_planes % 16 == 0);
#pragma unroll
  for (int i = 0; i < MT; i++) {
    const int row = row_base + i * 8 + g;
#pragma unroll
    for (int j = 0; j < NT; j++) {
      const int col = col_base + j * 8 + 2 * t4;
      if (row >= m || col >= n) continue;
      const size_t at = (size_t)row * n + col;
      double o0[L], o1[L];
      renorm_finish<L>(r[i][j][0], o0);
      renorm_finish<L>(r[i][j][1], o1);
#pragma unroll
      for (int l = 0; l < L; l++) {
        if (vec_ok) {
          *reinterpret_cast<double2*>(C_planes + l * planeC + at) = make_double2(o0[l], o1[l]);
        } else {
          C_planes[l * planeC + at] = o0[l];
          if (col + 1 < n) C_planes[l * planeC + at + 1] = o1[l];
        }
      }
    }
  }
}

// Tile rasterisation shared by both kernels: groups of GROUP_M tile rows are swept along n, so that the ~148 CTAs in
// flight cover a near-square patch of C and share their A / B slabs through L2.
__device__ __forceinline__ void raster_tile(int bid, int tiles_m, int tiles_n, int& tm, int& tn, int GROUP_M = 8) {
  const int per_group = GROUP_M * tiles_n;
  const int first_m = (bid / per_group) * GROUP_M;
  const int gsize = min(tiles_m - first_m, GROUP_M);
  tm = first_m + (bid % per_group) % gsize;
  tn = (bid % per_group) / gsize;
}

}  // namespace md
