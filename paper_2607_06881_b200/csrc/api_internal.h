// api_internal.h -- host-side state and helpers shared by the translation units that implement the C-ABI of libmdgemm
// (api.cu: the md_gemm family; literal.cu: the per-element-exponent balancing mode; qr.cu: md_geqrf).  Host code only.
#pragma once
#include <atomic>
#include <cstdint>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/mdgemm.h"
#include "md_kernels.h"

namespace md {

// Options are process-wide (include/mdgemm.h: md_set_option); 0 = default everywhere.
struct Options {
  int quarters = 0;      // 0 = 4 * limbs
  int orders = 0;        // 0 = quarters
  int bits = 0;          // 0 = 13, the paper's quarter
  int tile = 0;          // 0 = automatic, 1 = the 32 x 16 tile instance wherever it exists, 2 = never
  int fused_prep = 0;    // 0 = automatic (small / medium operands), 1 = always, 2 = never
  int one_launch = 0;    // 0 = automatic (single-wave problems), 1 = wherever the kernel exists, 2 = never
  int tile_schedule = 0; // 0 = automatic (hybrid from many whole-tile waves on), 1 = hybrid wherever possible, 2 = tile queue only, 3 = static lists
  int k_chunk = 0;       // 0 = chunked accumulation only when k exceeds the exactness budget; else the chunk length to force
  int host_blocks = 0;   // md_gemm_host: 0 = automatic panel plan, else the number of blocks of C (1 = no pipelining)
  int raster_group = 0;  // tile rows per raster group of the fused GEMM (0 = default 8)
};
extern Options g_opt;

// Everything the library keeps per DEVICE (a process may drive several GPUs): the registered workspace, the SM count, the
// profile events, md_gemm_host's copy streams and events, and the status bits host-side calls have brought back.
struct DeviceState {
  void* ws = nullptr;
  size_t ws_bytes = 0;
  int sms = 0;
  std::vector<cudaEvent_t> prof_ev;  // md_profile_*: three events per recorded call (start, before the fused GEMM, end)
  int prof_capacity = 0, prof_count = 0;
  cudaStream_t host_in = nullptr, host_out = nullptr;
  std::vector<cudaEvent_t> host_ev;
  uint32_t host_flags = 0;  // status words of md_gemm_host / md_gemm_auto calls since the last md_set_workspace
  bool host_flags_valid = false;
};
DeviceState* device_state();  // of the current device; nullptr when it cannot be determined
extern std::atomic<uint64_t> g_launches;

constexpr size_t WS_ALIGN = 256;
constexpr int MD_MAX_QUARTERS = 72;  // md_split accepts up to 4 * 16 + 8 quarters; md_renorm up to twice as many orders
constexpr int MD_MIN_BITS = 4, MD_MAX_BITS = 24;
inline size_t ws_round_up(size_t x) { return (x + WS_ALIGN - 1) / WS_ALIGN * WS_ALIGN; }

inline int quarters_for(int limbs) { return g_opt.quarters ? g_opt.quarters : 4 * limbs; }
inline int orders_for(int limbs) { return g_opt.orders ? g_opt.orders : quarters_for(limbs); }
inline int slice_bits() { return g_opt.bits ? g_opt.bits : 13; }
// the tolerance each format is held to: north_star for double / quad double, R13 for octo / hexa double
inline double format_tolerance(int limbs) {
  return limbs == 1 ? 0x1p-50 : limbs == 2 ? 1e-28 : limbs == 4 ? 1e-58 : limbs == 8 ? 1e-120 : 1e-245;
}
// Exactness budget (eq. 5 generalised; R6, R14): order s adds at most min(s + 1, Q) <= S products per
// k, each an integer of at most 2^(2W) units, so every partial sum is exactly representable while k * S * 2^(2W) <= 2^53.
// W = 13: k * S <= 2^27.
inline bool k_budget_ok(long long k, int S, int bits) { return k * S <= (1ll << (53 - 2 * bits)); }
int chunk_for(int k, int limbs, int Q, int S, int bits);

// Which fused kernel runs a problem, and the packed layout (CTA tile extents bxA x bxB, k-slab depth bk) the splitter must
// write for it.  chunk > 0: the chunked instance of the packed kernel with that chunk length (R16).
enum GemmFamily { GEMM_NONE = 0, GEMM_PACKED, GEMM_PACKED_SMALL, GEMM_WIDE, GEMM_GENERIC };
struct KernelPick {
  int family;
  int bxA, bxB, bk;
  int chunk;
};
KernelPick pick_kernel(int m, int n, int k, int limbs, int Q, int S, int bits, bool want_orders, bool allow_small);

// Workspace layout: [status word | expA int32[m] | expB int32[n] | Aq | Bq | stream-K scratch], Aq / Bq = the packed quarter
// planes of A / B (md_packed.cuh: zero padded to whole CTA tiles and k-slabs)
struct Carve {
  uint32_t* flags;
  int32_t* expA;
  int32_t* expB;
  double* Aq;
  double* Bq;
  void* sk;
  size_t total;
};
Carve carve(void* base, int m, int n, int k, int Q, int S, const KernelPick& pick);
size_t workspace_bytes_for(int m, int n, int k, int limbs, int Q, int S);

md_status check_gemm_args(int m, int n, int k, int limbs, const void* A, const void* B, const void* C, bool want_orders);
cudaError_t launch_fused(int m, int n, int k, int limbs, int Q, int S, const KernelPick& pick, const double* Aq, const double* Bq,
                         double* order_planes, double* C_planes, void* sk, bool counters_clear, cudaStream_t stream,
                         uint64_t* launches);
// a1-a4 on device-resident operands with explicit (Q, S) and workspace: what md_gemm / md_gemm_orders / md_gemm_host /
// md_gemm_auto and md_geqrf's trailing updates all run
md_status gemm_impl(int m, int n, int k, int limbs, int Q, int S, const double* A, const double* B, double* C_planes,
                    double* order_planes, void* ws, size_t ws_bytes, cudaStream_t stream, bool allow_small);

}  // namespace md
