/* mdcompare.h -- C-ABI of libmdcompare: the PAPER'S OWN two ways of multiplying multiple-double matrices, on B200, as
 * comparison paths beside the product.  Nothing in libmdgemm / md_gemm uses this library;
 * it exists so that the numbers of the paper's Table 1 (t_TC, t_CUDA) have B200 counterparts measured
 * on the same inputs as the fused path.
 *
 *   1. TOP-DOWN / materialised (PAPER.md:73-89 eq. 4, :192-207 section 4.3 and Table 2): quarter the matrices, STORE the
 *      stacked / convoluted quarter matrices, run ONE plain double-precision GEMM on them -- here cuBLAS DGEMM, the
 *      library counterpart of the paper's modified dmmaTensorCoreGemm -- then extract the parts and add them in multiple
 *      double arithmetic.  Table 2 (a 1024 x 512 double double A becomes 8192 x 4096 doubles) fixes which
 *      operand is convoluted: A.  So
 *          Atil  (S*m) x (Q*k), block lower triangular Toeplitz:  Atil[s*m + i][p*k + t] = A_{s-p}[i][t]  (0 for p > s)
 *          Bstk  (Q*k) x n, stacked:                              Bstk[p*k + t][j]       = B_p[t][j]
 *          Cbar  (S*m) x n = Atil * Bstk:                         Cbar[s*m + i][j]       = C^(s)[i][j] = sum_{p+q=s} A_q B_p
 *      which multiplies all Q*S blocks, zeros included (64 for double double against the 36 of the triangular set).
 *      Every accumulation is exact, so Cbar equals the oracle's order matrices BIT FOR BIT
 *      whatever cuBLAS does inside, and C equals md_gemm's C bit for bit.
 *   2. CUDA-CORE CLASSICAL ("a single thread executes an inner product"; the paper's C_CUDA of eq. 9 and t_CUDA
 *      of Table 1): one thread per element of C runs the multiple-double dot product with the textbook error-free
 *      transformations (TwoSum, TwoProd by fma; refs [2], [3], [15]) on the regular FP64 cores -- operation for operation
 *      the oracle's O5 (oracle_classic_gemm), so the result matches it bit for bit.
 *
 * Conventions as in mdgemm.h: plain DEVICE pointers unless "host" is said, limb planes [limbs][rows][cols] row-major fp64,
 * `stream` a cudaStream_t, calls enqueue and return (no sync) unless stated, return value 0 or a negative md_status.
 * cuBLAS keeps a handle (created on first use) and may allocate its own workspace: this is a comparison path, not the
 * product.
 */
#ifndef MDCOMPARE_H_
#define MDCOMPARE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Device bytes mdc_topdown_gemm needs for (m, n, k, limbs, quarters): quarter planes of A, Atil, Bstk, Cbar, exponents.
 * 0 on bad arguments.  At double double 4096^3: 8 GiB for Atil + 1 + 1 + 1 GiB. */
size_t mdc_topdown_workspace_bytes(int m, int n, int k, int limbs, int quarters);

/* The top-down path.  quarters = orders = Q (4 * limbs reproduces the paper).  ws: device, 256-byte aligned,
 * mdc_topdown_workspace_bytes bytes.  order_planes_out (device, [Q][m][n]) may be NULL; when given it receives a copy of
 * Cbar.  stage_ms_host (HOST, 4 floats) may be NULL; when given the call SYNCHRONISES the stream and stores the CUDA-event
 * times of: split (both operands), construction of Atil, the DGEMM, recombination.  limbs in {2, 4}. */
int mdc_topdown_gemm(int m, int n, int k, int limbs, int quarters, const double* A_planes, const double* B_planes,
                     double* C_planes, double* order_planes_out, void* ws, size_t ws_bytes, void* stream,
                     float* stage_ms_host);

/* The CUDA-core classical multiple-double GEMM, one thread per inner product.  limbs in {2, 4}. */
int mdc_classic_gemm(int m, int n, int k, int limbs, const double* A_planes, const double* B_planes, double* C_planes,
                     void* stream);

#ifdef __cplusplus
}
#endif
#endif /* MDCOMPARE_H_ */
