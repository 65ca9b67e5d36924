// compare.cu -- libmdcompare (include/mdcompare.h): the paper's own two paths on B200, as comparison beside md_gemm
// (SURVEY.md section 8(f) NEXT-2).  Not part of the product path: libmdgemm never calls into this file.
//   * top-down / materialised: PAPER.md:73-89 eq. 4, :192-207 Table 2 -- quarter, STORE Atil (A convoluted: block lower
//     triangular Toeplitz) and Bstk (B stacked), ONE plain DGEMM (cuBLAS), extract and add the parts;
//   * CUDA-core classical multiple-double GEMM: PAPER.md:166, one thread per inner product on the regular FP64 cores.
#include <cublas_v2.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../../include/mdcompare.h"
#include "../../../include/mdgemm.h"

namespace {

constexpr size_t ALIGN = 256;
inline size_t round_up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }

// Atil[(s*m + i) * (Q*k) + p*k + t] = Aq[s-p][i][t] for p <= s, else 0.  One thread per element, grid-stride, coalesced.
__global__ void __launch_bounds__(256) build_atil_kernel(int m, int k, int Q, const double* __restrict__ Aq,
                                                         double* __restrict__ Atil) {
  const size_t row_len = (size_t)Q * k;
  const size_t total = (size_t)Q * m * row_len;
  for (size_t at = (size_t)blockIdx.x * blockDim.x + threadIdx.x; at < total; at += (size_t)gridDim.x * blockDim.x) {
    const size_t row = at / row_len, col = at - row * row_len;
    const int s = (int)(row / m), i = (int)(row - (size_t)s * m);
    const int p = (int)(col / k), t = (int)(col - (size_t)p * k);
    Atil[at] = p <= s ? Aq[((size_t)(s - p) * m + i) * k + t] : 0.0;
  }
}

cublasHandle_t g_handle = nullptr;

// --- classical multiple-double arithmetic on the regular cores (textbook error-free transformations) -------------------
__device__ __forceinline__ void two_sum(double a, double b, double& s, double& e) {
  s = __dadd_rn(a, b);
  const double bb = __dsub_rn(s, a);
  e = __dadd_rn(__dsub_rn(a, __dsub_rn(s, bb)), __dsub_rn(b, bb));
}
__device__ __forceinline__ void two_prod(double a, double b, double& p, double& e) {
  p = __dmul_rn(a, b);
  e = __fma_rn(a, b, -p);
}
template <int T>
__device__ __forceinline__ void cascade_add(double (&acc)[T], double x) {
#pragma unroll
  for (int l = 0; l < T; l++) two_sum(acc[l], x, acc[l], x);
}
template <int T>
__device__ __forceinline__ void renormalise(double (&acc)[T]) {
#pragma unroll
  for (int l = T - 1; l > 0; l--) two_sum(acc[l - 1], acc[l], acc[l - 1], acc[l]);
#pragma unroll
  for (int l = 0; l + 1 < T; l++) two_sum(acc[l], acc[l + 1], acc[l], acc[l + 1]);
}

// One thread per element of C.  Every partial product a_la * b_lb with la + lb < L exactly by TwoProd,
// those with la + lb == L in plain fp64, each term added into an (L+1)-term accumulator by a TwoSum cascade, a
// renormalising sweep per k.  A warp covers 32 consecutive columns of one row: B loads coalesce, A loads broadcast.
template <int L>
__global__ void __launch_bounds__(256) classic_gemm_kernel(int m, int n, int k, const double* __restrict__ A,
                                                           const double* __restrict__ B, double* __restrict__ C) {
  const int j = blockIdx.x * 32 + (threadIdx.x & 31);
  const int i = blockIdx.y * 8 + (threadIdx.x >> 5);
  if (i >= m || j >= n) return;
  const size_t pa = (size_t)m * k, pb = (size_t)k * n, pc = (size_t)m * n;
  double acc[L + 1];
#pragma unroll
  for (int l = 0; l <= L; l++) acc[l] = 0.0;
  for (int kk = 0; kk < k; kk++) {
    double a[L], b[L];
#pragma unroll
    for (int l = 0; l < L; l++) {
      a[l] = A[l * pa + (size_t)i * k + kk];
      b[l] = B[l * pb + (size_t)kk * n + j];
    }
#pragma unroll
    for (int la = 0; la < L; la++)
#pragma unroll
      for (int lb = 0; lb < L; lb++) {
        if (la + lb > L) continue;
        if (la + lb < L) {
          double p, e;
          two_prod(a[la], b[lb], p, e);
          cascade_add<L + 1>(acc, p);
          cascade_add<L + 1>(acc, e);
        } else {
          cascade_add<L + 1>(acc, __dmul_rn(a[la], b[lb]));
        }
      }
    renormalise<L + 1>(acc);
  }
#pragma unroll
  for (int l = 0; l < L; l++) C[l * pc + (size_t)i * n + j] = acc[l];
}

struct Carve {
  double *Aq, *Atil, *Bstk, *Cbar;
  int32_t *expA, *expB;
  size_t total;
};
Carve carve(void* base, int m, int n, int k, int Q) {
  Carve c;
  char* p = static_cast<char*>(base);
  size_t off = 0;
  c.expA = reinterpret_cast<int32_t*>(p + off);
  off += round_up(sizeof(int32_t) * (size_t)m);
  c.expB = reinterpret_cast<int32_t*>(p + off);
  off += round_up(sizeof(int32_t) * (size_t)n);
  c.Aq = reinterpret_cast<double*>(p + off);
  off += round_up(sizeof(double) * (size_t)Q * m * k);
  c.Bstk = reinterpret_cast<double*>(p + off);
  off += round_up(sizeof(double) * (size_t)Q * k * n);
  c.Cbar = reinterpret_cast<double*>(p + off);
  off += round_up(sizeof(double) * (size_t)Q * m * n);
  c.Atil = reinterpret_cast<double*>(p + off);
  off += round_up(sizeof(double) * (size_t)Q * m * Q * k);
  c.total = off;
  return c;
}

}  // namespace

extern "C" {

size_t mdc_topdown_workspace_bytes(int m, int n, int k, int limbs, int quarters) {
  if (m <= 0 || n <= 0 || k <= 0 || (limbs != 2 && limbs != 4) || quarters < 1 || quarters > 24) return 0;
  return carve(nullptr, m, n, k, quarters).total;
}

int mdc_topdown_gemm(int m, int n, int k, int limbs, int quarters, const double* A_planes, const double* B_planes,
                     double* C_planes, double* order_planes_out, void* ws, size_t ws_bytes, void* stream,
                     float* stage_ms_host) {
  if (m <= 0 || n <= 0 || k <= 0 || !A_planes || !B_planes || !C_planes || !ws) return MD_ERR_BAD_ARG;
  if ((limbs != 2 && limbs != 4) || quarters < 1 || quarters > 24) return MD_ERR_BAD_ARG;
  if (reinterpret_cast<uintptr_t>(ws) % ALIGN) return MD_ERR_BAD_ARG;
  const int Q = quarters;
  if ((long long)Q * m > 0x7fffffffLL || (long long)Q * k > 0x7fffffffLL) return MD_ERR_BAD_ARG;
  const Carve c = carve(ws, m, n, k, Q);
  if (c.total > ws_bytes) return MD_ERR_WORKSPACE;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (!g_handle && cublasCreate(&g_handle) != CUBLAS_STATUS_SUCCESS) return MD_ERR_CUDA;
  if (cublasSetStream(g_handle, st) != CUBLAS_STATUS_SUCCESS) return MD_ERR_CUDA;
  cudaEvent_t ev[5] = {};
  if (stage_ms_host)
    for (auto& e : ev)
      if (cudaEventCreate(&e) != cudaSuccess) return MD_ERR_CUDA;
  auto mark = [&](int i) {
    if (stage_ms_host) cudaEventRecord(ev[i], st);
  };
  mark(0);
  // step 1: quarter both operands.  B's quarter planes [Q][k][n] ARE the stacked Bstk (Q*k x n).
  md_status s1 = md_split(m, k, limbs, Q, 0, A_planes, c.Aq, c.expA, stream);
  if (s1 != MD_OK) return s1;
  s1 = md_split(k, n, limbs, Q, 1, B_planes, c.Bstk, c.expB, stream);
  if (s1 != MD_OK) return s1;
  mark(1);
  // step 2 (eq. 4): store the convoluted A
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0)
    return MD_ERR_CUDA;
  build_atil_kernel<<<sms * 16, 256, 0, st>>>(m, k, Q, c.Aq, c.Atil);
  if (cudaGetLastError() != cudaSuccess) return MD_ERR_CUDA;
  mark(2);
  // step 3: one plain double-precision GEMM.  Row-major Cbar (Qm x n) = Atil (Qm x Qk) * Bstk (Qk x n) is the
  // column-major product Cbar^T (n x Qm) = Bstk^T (n x Qk) * Atil^T (Qk x Qm).
  const double one = 1.0, zero = 0.0;
  if (cublasDgemm(g_handle, CUBLAS_OP_N, CUBLAS_OP_N, n, Q * m, Q * k, &one, c.Bstk, n, c.Atil, Q * k, &zero, c.Cbar, n) !=
      CUBLAS_STATUS_SUCCESS)
    return MD_ERR_CUDA;
  mark(3);
  // steps 4-5: the parts C_1..C_Q are the m x n row blocks of Cbar; add them in multiple double arithmetic
  s1 = md_renorm(m, n, limbs, Q, c.Cbar, C_planes, stream);
  if (s1 != MD_OK) return s1;
  mark(4);
  if (order_planes_out &&
      cudaMemcpyAsync(order_planes_out, c.Cbar, sizeof(double) * (size_t)Q * m * n, cudaMemcpyDeviceToDevice, st) != cudaSuccess)
    return MD_ERR_CUDA;
  if (stage_ms_host) {
    if (cudaStreamSynchronize(st) != cudaSuccess) return MD_ERR_CUDA;
    for (int i = 0; i < 4; i++) cudaEventElapsedTime(&stage_ms_host[i], ev[i], ev[i + 1]);
    for (auto& e : ev) cudaEventDestroy(e);
  }
  return MD_OK;
}

int mdc_classic_gemm(int m, int n, int k, int limbs, const double* A_planes, const double* B_planes, double* C_planes,
                     void* stream) {
  if (m <= 0 || n <= 0 || k <= 0 || !A_planes || !B_planes || !C_planes) return MD_ERR_BAD_ARG;
  if (limbs != 2 && limbs != 4) return MD_ERR_BAD_ARG;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const dim3 grid((n + 31) / 32, (m + 7) / 8);
  if (grid.y > 65535) return MD_ERR_BAD_ARG;
  if (limbs == 2) classic_gemm_kernel<2><<<grid, 256, 0, st>>>(m, n, k, A_planes, B_planes, C_planes);
  else classic_gemm_kernel<4><<<grid, 256, 0, st>>>(m, n, k, A_planes, B_planes, C_planes);
  return cudaGetLastError() == cudaSuccess ? MD_OK : MD_ERR_CUDA;
}

}  // extern "C"
