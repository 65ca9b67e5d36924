// md_kernels.h -- internal launcher declarations of libmdgemm (host side).  Each launcher enqueues on `stream`, returns
// the cudaError_t of the launch, and adds the number of kernels it launched to *launches.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace md {

// `bits` = slice width W (13 = the paper's quarter; R14).  In launch_exponents `quarters` and `bits` only set
// the lower bound of the exponent range that is flagged (exponent_floor).
cudaError_t launch_exponents(int rows, int cols, int axis, int quarters, int bits, const double* lead_plane,
                             int32_t* exps, uint32_t* flags, cudaStream_t stream, uint64_t* launches);
int exponent_floor(int quarters, int bits);
cudaError_t launch_split(int rows, int cols, int limbs, int quarters, int bits, int axis, const double* planes,
                         double* quarter_planes, const int32_t* exps, uint32_t* flags, cudaStream_t stream,
                         uint64_t* launches);
cudaError_t launch_renorm(int m, int n, int limbs, int orders, const double* order_planes, double* C_planes,
                          cudaStream_t stream, uint64_t* launches);
// returns cudaErrorInvalidValue when (limbs, quarters) has no instantiation
cudaError_t launch_qgemm(int m, int n, int k, int limbs, int quarters, const double* Aq, const double* Bq,
                         double* order_planes, double* C_planes, cudaStream_t stream, uint64_t* launches);
bool qgemm_supported(int limbs, int quarters);
// md_plan_quarters (plan.cu): plain fp64 product of two non-negative matrices on the DMMA kernel of qgemm.cu; absolute
// values of a plane; D = max over W~ > 0 of E_i + F_j - ilogb(W~_ij) folded into *spread (pre-set to INT32_MIN)
cudaError_t launch_plain_dgemm(int m, int n, int k, const double* X, const double* Y, double* XY, cudaStream_t stream,
                               uint64_t* launches);
cudaError_t launch_abs(size_t count, const double* in, double* out, cudaStream_t stream, uint64_t* launches);
cudaError_t launch_spread(int m, int n, const double* W, const int32_t* expA, const int32_t* expB, int32_t* spread,
                          cudaStream_t stream, uint64_t* launches);
// md_gemm's internal pair: splitter writing the fragment-major packed layout (md_packed.cuh) and the bulk-copy /
// mbarrier pipelined fused GEMM reading it.  Same (limbs, quarters) support as launch_qgemm.
// bx, bk: the CTA tile extent along the group index and the k-slab depth of the fused kernel that will read the planes
// (md_packed.cuh pack_bx / pack_bx_generic; api.cu pick_kernel): splitter and GEMM must agree
cudaError_t launch_split_packed(int rows, int cols, int limbs, int quarters, int bits, int axis, int bx, int bk,
                                const double* planes, double* packed, const int32_t* exps, uint32_t* flags,
                                cudaStream_t stream, uint64_t* launches);
// plain [quarters][rows][cols] planes -> the packed layout (no arithmetic): md_qgemm for counts without a plain-layout kernel
cudaError_t launch_pack_planes(int rows, int cols, int quarters, int axis, int bx, int bk, const double* planes, double* packed,
                               cudaStream_t stream, uint64_t* launches);
bool qgemm_small_supported(int limbs, int quarters, int orders);
// exponent vectors + packed quarter planes of BOTH operands in one launch (small and medium problems: md_gemm's fused prep)
cudaError_t launch_prep_packed(int m, int n, int k, int limbs, int quarters, int bits, int bxA, int bxB, int bk, const double* A,
                               const double* B, double* Ap, double* Bp, int32_t* expA, int32_t* expB, uint32_t* flags,
                               void* sk_counters, cudaStream_t stream, uint64_t* launches);  // sk_counters != nullptr: also clears the
                               // SK_COUNTER_BYTES counter / flag words of the fused GEMM's stream-K scratch
// sk_ws: sk_workspace_bytes(limbs, quarters) bytes of device scratch for the stream-K tail (slab counters + one
// order-plane tile per stream-K tile); zeroed by the launcher (a memset node on `stream`) as far as it is used.
constexpr int SK_MAX_TILES = 256;
constexpr size_t SK_COUNTER_BYTES = 2048;  // 512 unsigned ints: slab counters of the stream-K tiles (red.add hand-in) or one hand-over
                                           // flag per CTA at [0, SK_MAX_TILES), the work-queue counter of the dynamic schedule at
                                           // SK_QUEUE_INDEX
constexpr int SK_QUEUE_INDEX = SK_MAX_TILES;
// chunk > 0: the chunked kernel's stream-K tail keeps one slot per (tile, chunk of the contraction) while that fits
// SK_CHUNK_CAP_BYTES; beyond, the chunked kernel runs whole tiles only
constexpr size_t SK_CHUNK_CAP_BYTES = (size_t)512 << 20;
inline bool sk_chunk_scratch_fits(size_t nchunks, int S, int BM, int BN) {
  return sizeof(double) * (size_t)SK_MAX_TILES * nchunks * S * BM * BN <= SK_CHUNK_CAP_BYTES;
}
size_t sk_workspace_bytes(int orders, int bxA, int bxB, int k, int chunk);
int sk_grid();
// fused_small.cu: steps a1-a4 in one launch for single-wave problems (quarter planes only in shared memory)
bool fused_small_supported(int limbs, int quarters, int orders);
int fused_small_cluster(int m, int n, int k);
cudaError_t launch_fused_small(int m, int n, int k, int limbs, int quarters, int orders, int bits, const double* A, const double* B,
                               double* order_planes, double* C_planes, uint32_t* flags, cudaStream_t stream, uint64_t* launches);
// chunk = 0: exact orders over the whole k.  chunk > 0 (R16; a multiple of 8, qgemm_chunk_supported instances
// only, C_planes only): the accumulators are folded into the elements' expansions every `chunk` contraction indices.
bool qgemm_chunk_supported(int limbs, int quarters);
bool qgemm_packed_supported(int limbs, int quarters, int orders);
// counters_clear: the SK_COUNTER_BYTES words at sk_ws are already zero on `stream` (launch_prep_packed cleared them), so a launch
// that needs nothing else zeroed (the hand-over schedule) enqueues no memset node
cudaError_t launch_qgemm_packed(int m, int n, int k, int limbs, int quarters, int orders, int chunk, bool small, const double* Ap,
                                const double* Bp, double* order_planes, double* C_planes, void* sk_ws, bool counters_clear,
                                cudaStream_t stream, uint64_t* launches);
// octo / hexa double (qgemm_wide.cu): same packed operands (k-slab depth 4), same stream-K scratch convention
bool qgemm_wide_supported(int limbs, int quarters);
cudaError_t launch_qgemm_wide(int m, int n, int k, int limbs, int quarters, const double* Ap, const double* Bp,
                              double* order_planes, double* C_planes, void* sk_ws, cudaStream_t stream,
                              uint64_t* launches);
// GENERIC instances of the same kernel (qgemm_wide.cu): quarter and order counts are runtime values up to these maxima (and
// orders <= 2 quarters - 1); packed operands with the tile shape of pack_bx_generic and k-slab depth 4.  Double and quad double
// keep 8 orders beyond the quarter maximum: the class-pair products of the literal mode (literal.cu) need quarters + spans.
constexpr int GENERIC_QMAX_DD = 16, GENERIC_QMAX_QD = 24, GENERIC_QMAX_OD = 40, GENERIC_QMAX_HD = 72;
constexpr int GENERIC_SMAX_DD = 24, GENERIC_SMAX_QD = 32, GENERIC_SMAX_OD = 42, GENERIC_SMAX_HD = 74;
int qgemm_generic_max_quarters(int limbs);
int qgemm_generic_max_orders(int limbs);
bool qgemm_generic_supported(int limbs, int quarters, int orders);
cudaError_t launch_qgemm_generic(int m, int n, int k, int limbs, int quarters, int orders, const double* Ap, const double* Bp,
                                 double* order_planes, double* C_planes, void* sk_ws, cudaStream_t stream, uint64_t* launches);
// per-device bookkeeping shared by the launchers (api.cu): the current device (-1 on error) and its SM count
constexpr int MD_MAX_DEVICES = 64;
int current_device();
int sm_count();
// calibration (probe.cu): register-only DMMA loop; *flops receives the FP64 flops the launch issues
cudaError_t launch_dmma_probe(int blocks, int warps_per_block, int iters, double* sink, cudaStream_t stream,
                              uint64_t* launches, uint64_t* flops);

}  // namespace md
