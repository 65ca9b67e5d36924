// qr.cu -- md_qr (include/mdgemm.h): blocked Householder QR of a multiple-double matrix with the trailing updates running through
// the multiple-double matrix product of this library.  PAPER.md:213 (conclusions): "Future work will apply this multiple double
// tensor core matrix multiplication to accelerate the blocked Householder QR, extending [18]" (ref [18]: least squares
// on GPUs in multiple double precision).  SURVEY.md 8(f) NEXT-4.
//
// A = Q R, A m x n (m >= n).  Panels of QR_NB = 32 columns:
//   1. qr_panel_kernel: the reflections of one panel, column by column, on the regular FP64 cores in multiple-double arithmetic
//      (md_arith.cuh).  ONE cooperative launch per panel; a CTA owns a slab of rows of the panel in shared memory, the column dot
//      products are reduced block -> grid through a double-buffered partial array, one grid-wide barrier per column.
//   2. the panel's reflectors as a block reflector I - V T V^T (compact WY): S = V^T V through md_gemm, T from S by a triangular
//      recurrence (qr_build_T_kernel).
//   3. the trailing columns: A2 <- A2 - V (T^T (V^T A2)) -- three md_gemm calls (gemm_impl: split, fused quarter GEMM on DMMA,
//      renormalising epilogue) and one multiple-double subtraction.  Sub-matrices are compacted into contiguous limb planes first
//      (md_gemm has no leading dimension; the copies are < 1 % of the time).
//   4. Q = H_0 ... H_{n-1} I_{m x n}, panel by panel backwards with the same three products; R = the upper triangle; rows of R /
//      columns of Q are negated where R_jj < 0, so that diag(R) >= 0 (unique for a full-rank A, comparable with the oracle).
#include <cooperative_groups.h>
#include <cstdint>
#include <vector>

#include "../../include/mdgemm.h"
#include "api_internal.h"
#include "md_arith.cuh"
#include "md_kernels.h"

namespace md {
namespace {

constexpr int QR_NB = 32;        // panel width
constexpr int QR_THREADS = 256;  // 8 row groups x 32 columns
constexpr int QR_RG = QR_THREADS / QR_NB;

template <int L>
__device__ __forceinline__ void ld_md(const double* p, size_t stride, double (&x)[L]) {
#pragma unroll
  for (int l = 0; l < L; l++) x[l] = p[l * stride];
}
template <int L>
__device__ __forceinline__ void st_md(double* p, size_t stride, const double (&x)[L]) {
#pragma unroll
  for (int l = 0; l < L; l++) p[l * stride] = x[l];
}

// The reflections of panel columns [j0, j0 + nbw) on rows [j0, m) of A [L][m][n], in place: R on and above the diagonal, the
// reflector vectors v (v_j = 1 implied) below it, tau[(j0 + j) * L ..].  Textbook reflections (Golub & Van Loan alg. 5.1.1 / LAPACK
// dgeqr2): alpha = a_jj, sigma = sum_{r>j} a_rj^2, beta = -sign(alpha) sqrt(alpha^2 + sigma), tau = (beta - alpha) / beta,
// v = a_{>j,j} / (alpha - beta); a_c <- a_c - tau (v^T a_c) v for the columns c > j of the panel.
// Shared memory: P[l][r][c] = the CTA's slab (RPB rows x QR_NB columns per limb), then red[QR_RG][QR_NB][L], fc[QR_NB][L],
// tw[QR_NB][L], sc[3][L] (1 / (alpha - beta), beta, tau).
template <int L>
__global__ void __launch_bounds__(QR_THREADS) qr_panel_kernel(int m, int n, int j0, int nbw, int RPB, double* __restrict__ A,
                                                              double* __restrict__ tau, double* partial, double* diagrow) {
  cooperative_groups::grid_group grid = cooperative_groups::this_grid();
  extern __shared__ double qr_smem[];
  const int t = threadIdx.x, c = t % QR_NB, rg = t / QR_NB, b = blockIdx.x, G = gridDim.x;
  const size_t planeA = (size_t)m * n;
  const int slab = RPB * QR_NB;
  double* P = qr_smem;                       // [L][RPB][QR_NB]
  double* red = P + (size_t)L * slab;        // [QR_RG][QR_NB][L]
  double* fc = red + QR_RG * QR_NB * L;      // [QR_NB][L]
  double* tw = fc + QR_NB * L;               // [QR_NB][L]
  double* sc = tw + QR_NB * L;               // [3][L]
  const int row0 = b * RPB;                  // first row of this slab, relative to j0
  const int rows_here = max(0, min(RPB, m - j0 - row0));
  for (int i = t; i < L * slab; i += QR_THREADS) {
    const int l = i / slab, r = (i % slab) / QR_NB, cc = i % QR_NB;
    P[i] = (r < rows_here && cc < nbw) ? A[l * planeA + (size_t)(j0 + row0 + r) * n + (j0 + cc)] : 0.0;
  }
  __syncthreads();

  for (int j = 0; j < nbw; j++) {
    const int par = j & 1;
    double* part = partial + (size_t)par * G * QR_NB * L;
    double* drow = diagrow + (size_t)par * QR_NB * L;
    const int owner = j / RPB, jr = j % RPB;  // the slab and local row of the diagonal element
    // ---- phase A: this slab's share of the dot products a_j^T a_c over the rows below the diagonal, c = j .. nbw-1
    {
      double acc[L + 1];
      mda_clear<L>(acc);
      if (c >= j && c < nbw)
        for (int r = rg; r < rows_here; r += QR_RG)
          if (row0 + r > j) {
            double x[L], y[L];
            ld_md<L>(P + r * QR_NB + j, slab, x);
            ld_md<L>(P + r * QR_NB + c, slab, y);
            mda_mac<L>(acc, x, y);
          }
      double out[L];
      renorm_finish<L>(acc, out);
#pragma unroll
      for (int l = 0; l < L; l++) red[(rg * QR_NB + c) * L + l] = out[l];
    }
    __syncthreads();
    if (rg == 0 && c >= j && c < nbw) {
      double acc[L + 1];
      mda_clear<L>(acc);
      for (int g2 = 0; g2 < QR_RG; g2++) {
        double x[L];
#pragma unroll
        for (int l = 0; l < L; l++) x[l] = red[(g2 * QR_NB + c) * L + l];
        mda_acc<L>(acc, x);
      }
      double out[L];
      renorm_finish<L>(acc, out);
#pragma unroll
      for (int l = 0; l < L; l++) part[((size_t)b * QR_NB + c) * L + l] = out[l];
      if (b == owner) {
#pragma unroll
        for (int l = 0; l < L; l++) drow[c * L + l] = P[l * slab + jr * QR_NB + c];
      }
    }
    grid.sync();
    // ---- phase B (every CTA, redundantly): the reflector scalars and, per column c > j, tau w_c and tau w_c / (alpha - beta)
    if (rg == 0 && c >= j && c < nbw) {
      double acc[L + 1], dot[L], sigma[L], alpha[L], ajc[L];
      mda_clear<L>(acc);
      for (int g2 = 0; g2 < G; g2++) {
        double x[L];
#pragma unroll
        for (int l = 0; l < L; l++) x[l] = __ldcg(part + ((size_t)g2 * QR_NB + c) * L + l);
        mda_acc<L>(acc, x);
      }
      renorm_finish<L>(acc, dot);
      mda_clear<L>(acc);
      for (int g2 = 0; g2 < G; g2++) {
        double x[L];
#pragma unroll
        for (int l = 0; l < L; l++) x[l] = __ldcg(part + ((size_t)g2 * QR_NB + j) * L + l);
        mda_acc<L>(acc, x);
      }
      renorm_finish<L>(acc, sigma);
#pragma unroll
      for (int l = 0; l < L; l++) alpha[l] = __ldcg(drow + j * L + l), ajc[l] = __ldcg(drow + c * L + l);
      double beta[L], tj[L], inv[L], twc[L], fcc[L];
      if (sigma[0] == 0.0) {  // nothing below the diagonal: H = I
#pragma unroll
        for (int l = 0; l < L; l++) beta[l] = alpha[l], tj[l] = 0.0, inv[l] = 0.0, twc[l] = 0.0, fcc[l] = 0.0;
      } else {
        double r2[L + 1], nrm2[L], nrm[L], den[L], one[L], num[L], w[L];
        mda_clear<L>(r2);
        mda_acc<L>(r2, sigma);
        mda_mac<L>(r2, alpha, alpha);
        renorm_finish<L>(r2, nrm2);
        mda_sqrt<L>(nrm2, nrm);
        const double sgn = alpha[0] >= 0.0 ? -1.0 : 1.0;
#pragma unroll
        for (int l = 0; l < L; l++) beta[l] = sgn * nrm[l], one[l] = l == 0 ? 1.0 : 0.0;
        mda_add<L>(beta, alpha, num, -1.0);   // beta - alpha
        mda_div<L>(num, beta, tj);            // tau
        mda_add<L>(alpha, beta, den, -1.0);   // alpha - beta
        mda_div<L>(one, den, inv);
        // w_c = a_jc + (a_{>j,j}^T a_{>j,c}) / (alpha - beta)
        mda_clear<L>(r2);
        mda_acc<L>(r2, ajc);
        mda_mac<L>(r2, inv, dot);
        renorm_finish<L>(r2, w);
        mda_mul<L>(tj, w, twc);
        mda_mul<L>(twc, inv, fcc);
      }
#pragma unroll
      for (int l = 0; l < L; l++) fc[c * L + l] = fcc[l], tw[c * L + l] = twc[l];
      if (c == j) {
#pragma unroll
        for (int l = 0; l < L; l++) sc[l] = inv[l], sc[L + l] = beta[l], sc[2 * L + l] = tj[l];
        if (b == 0) {
#pragma unroll
          for (int l = 0; l < L; l++) tau[(size_t)(j0 + j) * L + l] = tj[l];
        }
      }
    }
    __syncthreads();
    const bool reflect = sc[2 * L] != 0.0;  // tau != 0
    // ---- update of the panel columns c > j: a_rc -= (tau w_c / (alpha - beta)) a_rj below the diagonal, a_jc -= tau w_c on it
    if (reflect && c > j && c < nbw) {
      double f[L];
#pragma unroll
      for (int l = 0; l < L; l++) f[l] = fc[c * L + l];
      for (int r = rg; r < rows_here; r += QR_RG) {
        const int gr = row0 + r;
        if (gr < j) continue;
        double acc[L + 1], y[L], out[L];
        ld_md<L>(P + r * QR_NB + c, slab, y);
        mda_clear<L>(acc);
        mda_acc<L>(acc, y);
        if (gr == j) {
          double x[L];
#pragma unroll
          for (int l = 0; l < L; l++) x[l] = tw[c * L + l];
          mda_acc<L>(acc, x, -1.0);
        } else {
          double x[L];
          ld_md<L>(P + r * QR_NB + j, slab, x);
          mda_mac<L>(acc, f, x, -1.0);
        }
        renorm_finish<L>(acc, out);
        st_md<L>(P + r * QR_NB + c, slab, out);
      }
    }
    __syncthreads();
    // ---- column j itself: v below the diagonal, beta on it
    if (reflect)
      for (int r = t; r < rows_here; r += QR_THREADS) {
        const int gr = row0 + r;
        if (gr < j) continue;
        double out[L];
        if (gr == j) {
#pragma unroll
          for (int l = 0; l < L; l++) out[l] = sc[L + l];
        } else {
          double x[L], inv[L];
          ld_md<L>(P + r * QR_NB + j, slab, x);
#pragma unroll
          for (int l = 0; l < L; l++) inv[l] = sc[l];
          mda_mul<L>(x, inv, out);
        }
        st_md<L>(P + r * QR_NB + j, slab, out);
      }
    __syncthreads();
  }
  for (int i = t; i < L * slab; i += QR_THREADS) {
    const int l = i / slab, r = (i % slab) / QR_NB, cc = i % QR_NB;
    if (r < rows_here && cc < nbw) A[l * planeA + (size_t)(j0 + row0 + r) * n + (j0 + cc)] = P[i];
  }
}

// V [L][mp][nbw] (unit lower trapezoid of the factored panel) and its transpose VT [L][nbw][mp]
template <int L>
__global__ void qr_extract_V_kernel(int m, int n, int j0, int nbw, const double* __restrict__ A, double* __restrict__ V, double* __restrict__ VT) {
  const int mp = m - j0;
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)mp * nbw) return;
  const int r = (int)(idx / nbw), c = (int)(idx % nbw);
#pragma unroll
  for (int l = 0; l < L; l++) {
    const double v = r > c ? A[(size_t)l * m * n + (size_t)(j0 + r) * n + (j0 + c)] : (r == c && l == 0 ? 1.0 : 0.0);
    V[(size_t)l * mp * nbw + idx] = v;
    VT[(size_t)l * mp * nbw + (size_t)c * mp + r] = v;
  }
}

// T of the block reflector I - V T V^T from S = V^T V: T_jj = tau_j, T_{0:j,j} = -tau_j T_{0:j,0:j} S_{0:j,j}.  Row i of T depends
// on row i only: one thread per row.  Writes T [L][nbw][nbw] and its transpose.
template <int L>
__global__ void qr_build_T_kernel(int nbw, const double* __restrict__ S, const double* __restrict__ tau, double* __restrict__ T, double* __restrict__ Tt) {
  const int i = threadIdx.x;
  const size_t plane = (size_t)nbw * nbw;
  if (i >= nbw) return;
  for (int j = 0; j < nbw; j++) {
    double out[L];
    if (j < i) {
#pragma unroll
      for (int l = 0; l < L; l++) out[l] = 0.0;
    } else if (j == i) {
#pragma unroll
      for (int l = 0; l < L; l++) out[l] = tau[(size_t)j * L + l];
    } else {
      double acc[L + 1], z[L], tj[L];
      mda_clear<L>(acc);
      for (int q = i; q < j; q++) {
        double a[L], s[L];
        ld_md<L>(T + (size_t)i * nbw + q, plane, a);
        ld_md<L>(S + (size_t)q * nbw + j, plane, s);
        mda_mac<L>(acc, a, s);
      }
      renorm_finish<L>(acc, z);
#pragma unroll
      for (int l = 0; l < L; l++) tj[l] = -tau[(size_t)j * L + l];
      mda_mul<L>(tj, z, out);
    }
    st_md<L>(T + (size_t)i * nbw + j, plane, out);
    st_md<L>(Tt + (size_t)j * nbw + i, plane, out);
  }
}

// compact copy of the sub-matrix X[r0 : r0 + rows, c0 : c0 + cols] of X [L][m][n]
template <int L>
__global__ void qr_copy_sub_kernel(int m, int n, int r0, int c0, int rows, int cols, const double* __restrict__ X, double* __restrict__ out) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)rows * cols) return;
  const int r = (int)(idx / cols), c = (int)(idx % cols);
#pragma unroll
  for (int l = 0; l < L; l++) out[(size_t)l * rows * cols + idx] = X[(size_t)l * m * n + (size_t)(r0 + r) * n + (c0 + c)];
}
// X[r0 : r0 + rows, c0 : c0 + cols] = Xc - P in multiple-double arithmetic (Xc, P compact [L][rows][cols])
template <int L>
__global__ void qr_sub_update_kernel(int m, int n, int r0, int c0, int rows, int cols, const double* __restrict__ Xc, const double* __restrict__ P,
                                     double* __restrict__ X) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)rows * cols) return;
  const int r = (int)(idx / cols), c = (int)(idx % cols);
  const size_t plane = (size_t)rows * cols;
  double a[L], b2[L], out[L];
  ld_md<L>(Xc + idx, plane, a);
  ld_md<L>(P + idx, plane, b2);
  mda_add<L>(a, b2, out, -1.0);
#pragma unroll
  for (int l = 0; l < L; l++) X[(size_t)l * m * n + (size_t)(r0 + r) * n + (c0 + c)] = out[l];
}
// Q <- I (m x n);  R <- upper triangle of the factored A
template <int L>
__global__ void qr_init_QR_kernel(int m, int n, const double* __restrict__ A, double* __restrict__ Q, double* __restrict__ R) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)m * n) return;
  const int r = (int)(idx / n), c = (int)(idx % n);
#pragma unroll
  for (int l = 0; l < L; l++) {
    Q[(size_t)l * m * n + idx] = (r == c && l == 0) ? 1.0 : 0.0;
    if (r < n) R[(size_t)l * n * n + (size_t)r * n + c] = c >= r ? A[(size_t)l * m * n + idx] : 0.0;
  }
}
// diag(R) >= 0: negate row j of R and column j of Q where R_jj < 0
template <int L>
__global__ void qr_fix_signs_kernel(int m, int n, double* __restrict__ Q, double* __restrict__ R) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)m * n) return;
  const int r = (int)(idx / n), c = (int)(idx % n);
  const bool flip_col = R[(size_t)c * n + c] < 0.0;                // column c of Q
  const bool flip_row = r < n && c >= r && R[(size_t)r * n + r] < 0.0 && r != c;  // off-diagonal entries of row r of R
  if (flip_col) {
#pragma unroll
    for (int l = 0; l < L; l++) Q[(size_t)l * m * n + idx] = -Q[(size_t)l * m * n + idx];
  }
  if (flip_row) {
#pragma unroll
    for (int l = 0; l < L; l++) R[(size_t)l * n * n + (size_t)r * n + c] = -R[(size_t)l * n * n + (size_t)r * n + c];
  }
}
// ... and the diagonal itself, once nobody reads its sign any more
template <int L>
__global__ void qr_fix_diag_kernel(int n, double* __restrict__ R) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n || !(R[(size_t)j * n + j] < 0.0)) return;
#pragma unroll
  for (int l = 0; l < L; l++) R[(size_t)l * n * n + (size_t)j * n + j] = -R[(size_t)l * n * n + (size_t)j * n + j];
}

struct QrCarve {
  double *Aw, *tau, *partial, *diagrow, *V, *VT, *S, *T, *Tt, *Tall, *Xc, *P, *W, *W2;
  void* ws;
  size_t ws_bytes, total;
};
size_t qr_gemm_ws_bytes(int m, int n, int limbs) {
  const int Q = quarters_for(limbs), S = orders_for(limbs);
  size_t best = 0;
  const int shapes[4][3] = {{QR_NB, QR_NB, m}, {QR_NB, n, m}, {QR_NB, n, QR_NB}, {m, n, QR_NB}};
  for (auto& s : shapes) {
    const size_t b = workspace_bytes_for(s[0], s[1], s[2], limbs, Q, S);
    if (b == 0) return 0;
    if (b > best) best = b;
  }
  return best;
}
int qr_rows_per_block(int m, int limbs) {
  // slab of the panel per CTA: at most ~150 KB of shared memory, at least 64 rows; few enough CTAs to be co-resident
  int rpb = 64;
  const int sms = sm_count() > 0 ? sm_count() : 1;
  while ((m + rpb - 1) / rpb > sms) rpb *= 2;
  return rpb;
}
size_t qr_panel_smem(int rpb, int limbs) {
  return sizeof(double) * ((size_t)limbs * rpb * QR_NB + (QR_RG + 2) * QR_NB * limbs + 3 * limbs);
}
QrCarve qr_carve(void* base, int m, int n, int limbs) {
  QrCarve c;
  char* p = static_cast<char*>(base);
  size_t off = 0;
  auto take = [&](size_t doubles) {
    double* q = reinterpret_cast<double*>(p + off);
    off += ws_round_up(sizeof(double) * doubles);
    return q;
  };
  const size_t L = limbs;
  const int panels = (n + QR_NB - 1) / QR_NB;
  const int G = (m + qr_rows_per_block(m, limbs) - 1) / qr_rows_per_block(m, limbs);
  c.Aw = take(L * m * n);
  c.tau = take(L * n);
  c.partial = take(2 * (size_t)G * QR_NB * L);
  c.diagrow = take(2 * QR_NB * L);
  c.V = take(L * m * QR_NB);
  c.VT = take(L * m * QR_NB);
  c.S = take(L * QR_NB * QR_NB);
  c.T = take(L * QR_NB * QR_NB);
  c.Tt = take(L * QR_NB * QR_NB);
  c.Tall = take((size_t)panels * L * QR_NB * QR_NB);
  c.Xc = take(L * m * n);
  c.P = take(L * m * n);
  c.W = take(L * QR_NB * n);
  c.W2 = take(L * QR_NB * n);
  c.ws = p + off;
  c.ws_bytes = qr_gemm_ws_bytes(m, n, limbs);
  off += ws_round_up(c.ws_bytes);
  c.total = off;
  return c;
}

template <int L>
md_status qr_run(int m, int n, const double* A, double* Q, double* R, const QrCarve& c, float* times_ms_host, cudaStream_t st) {
  const int Qc = quarters_for(L), Sc = orders_for(L);
  const int rpb = qr_rows_per_block(m, L);
  const size_t smem = qr_panel_smem(rpb, L);
  if (smem > 200 * 1024) return MD_ERR_UNSUPPORTED;
  static bool attr_done[MD_MAX_DEVICES] = {};
  const int dev = current_device();
  if (dev < 0 || dev >= MD_MAX_DEVICES || !attr_done[dev]) {
    if (cudaFuncSetAttribute(qr_panel_kernel<L>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024) != cudaSuccess) return MD_ERR_CUDA;
    if (dev >= 0 && dev < MD_MAX_DEVICES) attr_done[dev] = true;
  }
  uint64_t launches = 0;
  std::vector<cudaEvent_t> ev;  // pairs around every md_gemm call, when timing is asked for
  cudaEvent_t ev_all[2] = {nullptr, nullptr};
  auto cleanup = [&]() {
    for (cudaEvent_t e : ev) cudaEventDestroy(e);
    for (cudaEvent_t e : ev_all)
      if (e) cudaEventDestroy(e);
  };
  if (times_ms_host) {
    if (cudaEventCreate(&ev_all[0]) != cudaSuccess || cudaEventCreate(&ev_all[1]) != cudaSuccess) return cleanup(), MD_ERR_CUDA;
    cudaEventRecord(ev_all[0], st);
  }
  md_status status = MD_OK;
  auto gemm = [&](int gm, int gn, int gk, const double* X, const double* Y, double* Z) {
    if (status != MD_OK) return;
    cudaEvent_t a = nullptr, b = nullptr;
    if (times_ms_host && cudaEventCreate(&a) == cudaSuccess && cudaEventCreate(&b) == cudaSuccess) {
      ev.push_back(a), ev.push_back(b);
      cudaEventRecord(a, st);
    }
    status = gemm_impl(gm, gn, gk, L, Qc, Sc, X, Y, Z, nullptr, c.ws, c.ws_bytes, st, true);
    if (b) cudaEventRecord(b, st);
  };
  auto blocks_for = [](size_t items) { return (unsigned)((items + 255) / 256); };
#define QR_CHECK() \
  if (cudaGetLastError() != cudaSuccess) status = status == MD_OK ? MD_ERR_CUDA : status

  if (cudaMemsetAsync(c.ws, 0, WS_ALIGN, st) != cudaSuccess) return cleanup(), MD_ERR_CUDA;
  if (cudaMemcpyAsync(c.Aw, A, sizeof(double) * (size_t)L * m * n, cudaMemcpyDeviceToDevice, st) != cudaSuccess) return cleanup(), MD_ERR_CUDA;
  const int panels = (n + QR_NB - 1) / QR_NB;
  // the block reflector of the panel at j0 applied to X[j0:, c0 : c0 + cols] (X = the working copy of A, or Q): X2 -= V (Tm (V^T X2))
  auto apply_block = [&](double* X, int j0, int nbw, int c0, int cols, const double* Tm) {
    const int mp = m - j0;
    qr_copy_sub_kernel<L><<<blocks_for((size_t)mp * cols), 256, 0, st>>>(m, n, j0, c0, mp, cols, X, c.Xc);
    launches++;
    QR_CHECK();
    gemm(nbw, cols, mp, c.VT, c.Xc, c.W);     // W = V^T X2
    gemm(nbw, cols, nbw, Tm, c.W, c.W2);      // W2 = Tm W
    gemm(mp, cols, nbw, c.V, c.W2, c.P);      // P = V W2
    if (status != MD_OK) return;
    qr_sub_update_kernel<L><<<blocks_for((size_t)mp * cols), 256, 0, st>>>(m, n, j0, c0, mp, cols, c.Xc, c.P, X);
    launches++;
    QR_CHECK();
  };
  for (int p = 0; p < panels && status == MD_OK; p++) {
    const int j0 = p * QR_NB, nbw = n - j0 < QR_NB ? n - j0 : QR_NB, mp = m - j0;
    int G = (mp + rpb - 1) / rpb;
    int mm = m, nn = n, jj = j0, nb2 = nbw, rr = rpb;
    double *Aw = c.Aw, *tau = c.tau, *partial = c.partial, *diagrow = c.diagrow;
    void* args[] = {&mm, &nn, &jj, &nb2, &rr, &Aw, &tau, &partial, &diagrow};
    if (cudaLaunchCooperativeKernel(reinterpret_cast<const void*>(qr_panel_kernel<L>), dim3(G), dim3(QR_THREADS), args, smem, st) != cudaSuccess) {
      status = MD_ERR_CUDA;
      break;
    }
    launches++;
    qr_extract_V_kernel<L><<<blocks_for((size_t)mp * nbw), 256, 0, st>>>(m, n, j0, nbw, c.Aw, c.V, c.VT);
    launches++;
    QR_CHECK();
    gemm(nbw, nbw, mp, c.VT, c.V, c.S);        // S = V^T V
    if (status != MD_OK) break;
    double* Tp = c.Tall + (size_t)p * L * QR_NB * QR_NB;  // T of this panel, kept for Q ([L][nbw][nbw])
    qr_build_T_kernel<L><<<1, QR_NB, 0, st>>>(nbw, c.S, c.tau + (size_t)j0 * L, Tp, c.Tt);
    launches++;
    QR_CHECK();
    if (j0 + nbw < n) apply_block(c.Aw, j0, nbw, j0 + nbw, n - j0 - nbw, c.Tt);  // Q_p^T A2 = (I - V T^T V^T) A2
  }
  if (status == MD_OK) {
    qr_init_QR_kernel<L><<<blocks_for((size_t)m * n), 256, 0, st>>>(m, n, c.Aw, Q, R);
    launches++;
    QR_CHECK();
  }
  for (int p = panels - 1; p >= 0 && status == MD_OK; p--) {
    const int j0 = p * QR_NB, nbw = n - j0 < QR_NB ? n - j0 : QR_NB, mp = m - j0;
    qr_extract_V_kernel<L><<<blocks_for((size_t)mp * nbw), 256, 0, st>>>(m, n, j0, nbw, c.Aw, c.V, c.VT);
    launches++;
    QR_CHECK();
    apply_block(Q, j0, nbw, j0, n - j0, c.Tall + (size_t)p * L * QR_NB * QR_NB);  // Q[j0:, j0:] <- (I - V T V^T) Q[j0:, j0:]
  }
  if (status == MD_OK) {
    qr_fix_signs_kernel<L><<<blocks_for((size_t)m * n), 256, 0, st>>>(m, n, Q, R);
    qr_fix_diag_kernel<L><<<blocks_for((size_t)n), 256, 0, st>>>(n, R);
    launches += 2;
    QR_CHECK();
  }
#undef QR_CHECK
  g_launches += launches;
  if (times_ms_host) {
    cudaEventRecord(ev_all[1], st);
    if (cudaStreamSynchronize(st) != cudaSuccess) status = status == MD_OK ? MD_ERR_CUDA : status;
    float total = 0.f, in_gemm = 0.f;
    if (status == MD_OK) {
      cudaEventElapsedTime(&total, ev_all[0], ev_all[1]);
      for (size_t i = 0; i + 1 < ev.size(); i += 2) {
        float t = 0.f;
        cudaEventElapsedTime(&t, ev[i], ev[i + 1]);
        in_gemm += t;
      }
    }
    times_ms_host[0] = total;
    times_ms_host[1] = in_gemm;
  }
  cleanup();
  return status;
}

inline bool qr_limbs_ok(int limbs) { return limbs == 2 || limbs == 4; }

}  // namespace
}  // namespace md

using namespace md;

extern "C" {

size_t md_qr_scratch_bytes(int m, int n, int limbs) {
  if (m <= 0 || n <= 0 || m < n || !qr_limbs_ok(limbs)) return 0;
  if (qr_gemm_ws_bytes(m, n, limbs) == 0) return 0;
  return qr_carve(nullptr, m, n, limbs).total;
}

md_status md_qr(int m, int n, int limbs, const double* A_planes, double* Q_planes, double* R_planes, void* scratch,
                size_t scratch_bytes, float* times_ms_host, md_stream stream) {
  if (m <= 0 || n <= 0 || m < n || !A_planes || !Q_planes || !R_planes || !scratch) return MD_ERR_BAD_ARG;
  if (!qr_limbs_ok(limbs)) return MD_ERR_BAD_ARG;
  if ((reinterpret_cast<uintptr_t>(A_planes) | reinterpret_cast<uintptr_t>(Q_planes) | reinterpret_cast<uintptr_t>(R_planes)) & 7) return MD_ERR_BAD_ARG;
  if (reinterpret_cast<uintptr_t>(scratch) % WS_ALIGN) return MD_ERR_BAD_ARG;
  const size_t need = md_qr_scratch_bytes(m, n, limbs);
  if (need == 0) return MD_ERR_UNSUPPORTED;
  if (scratch_bytes < need) return MD_ERR_WORKSPACE;
  if (!k_budget_ok(m, orders_for(limbs), slice_bits())) return MD_ERR_K_TOO_LARGE;
  const QrCarve c = qr_carve(scratch, m, n, limbs);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  return limbs == 2 ? qr_run<2>(m, n, A_planes, Q_planes, R_planes, c, times_ms_host, st)
                    : qr_run<4>(m, n, A_planes, Q_planes, R_planes, c, times_ms_host, st);
}

}  // extern "C"
