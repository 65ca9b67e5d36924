// api.cu -- the C-ABI of libmdgemm (include/mdgemm.h): argument checking, options, workspace carving, and the sequence
// of kernel launches of the hot path.  No arithmetic of the method lives here.
#include <atomic>
#include <cstdint>
#include <vector>

#include "../../include/mdgemm.h"
#include "md_common.cuh"
#include "md_kernels.h"
#include "md_packed.cuh"

namespace {

struct State {
  int opt_quarters = 0;  // 0 = default (4 * limbs)
  int opt_orders = 0;    // 0 = default (= quarters)
  int opt_bits = 0;      // 0 = default (13, the paper's quarter)
  void* ws = nullptr;
  size_t ws_bytes = 0;
};
State g_state;

// md_profile_*: three events per recorded call (start, before the fused GEMM kernel, end)
struct Profile {
  std::vector<cudaEvent_t> ev;
  int capacity = 0, count = 0;
};
Profile g_prof;
std::atomic<uint64_t> g_launches{0};

constexpr size_t ALIGN = 256;
constexpr int MD_MAX_QUARTERS = 72;  // md_split accepts up to 4 * 16 + 8 quarters; md_renorm up to twice as many orders
inline size_t round_up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }

inline int quarters_for(int limbs) { return g_state.opt_quarters ? g_state.opt_quarters : 4 * limbs; }
inline int orders_for(int limbs) { return g_state.opt_orders ? g_state.opt_orders : quarters_for(limbs); }
inline int slice_bits() { return g_state.opt_bits ? g_state.opt_bits : 13; }
constexpr int MD_MIN_BITS = 4, MD_MAX_BITS = 24;
// Exactness budget (eq. 5 generalised; R6, R13): order s adds (s+1) <= S products per k, each an
// integer of at most 2^(2W) units, so every partial sum is exactly representable while k * S * 2^(2W) <= 2^53.
// W = 13: k * S <= 2^27.
inline bool k_budget_ok(long long k, int S, int bits) { return k * S <= (1ll << (53 - 2 * bits)); }

// Workspace layout: [status word | expA int32[m] | expB int32[n] | Aq | Bq], Aq / Bq = the packed quarter planes of A / B
// (md_packed.cuh: zero padded to whole CTA tiles and k-slabs), then the stream-K scratch of the fused GEMM
struct Carve {
  uint32_t* flags;
  int32_t* expA;
  int32_t* expB;
  double* Aq;
  double* Bq;
  void* sk;  // stream-K scratch of the fused GEMM
  size_t total;
};
Carve carve(void* base, int m, int n, int k, int limbs, int quarters) {
  Carve c;
  size_t off = 0;
  char* p = static_cast<char*>(base);
  c.flags = reinterpret_cast<uint32_t*>(p + off);
  off += ALIGN;
  c.expA = reinterpret_cast<int32_t*>(p + off);
  off += round_up(sizeof(int32_t) * (size_t)m);
  c.expB = reinterpret_cast<int32_t*>(p + off);
  off += round_up(sizeof(int32_t) * (size_t)n);
  c.Aq = reinterpret_cast<double*>(p + off);
  off += round_up(sizeof(double) * md::packed_doubles(m, k, md::pack_bx(limbs, 0), md::pack_bk(limbs), quarters));
  c.Bq = reinterpret_cast<double*>(p + off);
  off += round_up(sizeof(double) * md::packed_doubles(n, k, md::pack_bx(limbs, 1), md::pack_bk(limbs), quarters));
  c.sk = p + off;
  off += round_up(md::sk_workspace_bytes(limbs, quarters));
  c.total = off;
  return c;
}

inline bool aligned8(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 7) == 0; }

md_status check_gemm_args(int m, int n, int k, int limbs, const void* A, const void* B, const void* C) {
  if (m <= 0 || n <= 0 || k <= 0 || !A || !B || !C) return MD_ERR_BAD_ARG;
  if (!aligned8(A) || !aligned8(B) || !aligned8(C)) return MD_ERR_BAD_ARG;
  if (limbs != 2 && limbs != 4 && limbs != 8 && limbs != 16) return MD_ERR_BAD_ARG;
  const int Q = quarters_for(limbs), S = orders_for(limbs);
  if (S != Q || !(md::qgemm_supported(limbs, Q) || md::qgemm_wide_supported(limbs, Q))) return MD_ERR_UNSUPPORTED;
  if (!k_budget_ok(k, S, slice_bits())) return MD_ERR_K_TOO_LARGE;
  return MD_OK;
}

// split A (rows) and B (columns) into the packed quarter planes of the carved workspace, then the fused quarter GEMM.
md_status gemm_impl(int m, int n, int k, int limbs, const double* A, const double* B, double* C_planes,
                    double* order_planes, void* ws, size_t ws_bytes, cudaStream_t stream) {
  const int Q = quarters_for(limbs), W = slice_bits();
  if (!ws) return MD_ERR_WORKSPACE;
  const Carve c = carve(ws, m, n, k, limbs, Q);
  if (c.total > ws_bytes) return MD_ERR_WORKSPACE;
  uint64_t launches = 0;
  cudaEvent_t* ev = (g_prof.count < g_prof.capacity) ? &g_prof.ev[3 * (size_t)g_prof.count] : nullptr;
  if (ev) cudaEventRecord(ev[0], stream);
  cudaError_t err = md::launch_exponents(m, k, 0, Q, W, A, c.expA, c.flags, stream, &launches);
  if (err == cudaSuccess) err = md::launch_exponents(k, n, 1, Q, W, B, c.expB, c.flags, stream, &launches);
  if (err == cudaSuccess) err = md::launch_split_packed(m, k, limbs, Q, W, 0, A, c.Aq, c.expA, c.flags, stream, &launches);
  if (err == cudaSuccess) err = md::launch_split_packed(k, n, limbs, Q, W, 1, B, c.Bq, c.expB, c.flags, stream, &launches);
  if (ev) cudaEventRecord(ev[1], stream);
  if (err == cudaSuccess)
    err = limbs <= 4 ? md::launch_qgemm_packed(m, n, k, limbs, Q, c.Aq, c.Bq, order_planes, C_planes, c.sk, stream, &launches)
                     : md::launch_qgemm_wide(m, n, k, limbs, Q, c.Aq, c.Bq, order_planes, C_planes, c.sk, stream, &launches);
  if (ev) {
    cudaEventRecord(ev[2], stream);
    if (err == cudaSuccess) g_prof.count++;
  }
  g_launches += launches;
  return err == cudaSuccess ? MD_OK : MD_ERR_CUDA;
}

}  // namespace

extern "C" {

md_status md_set_option(int key, int value) {
  if (value < 0 || value > MD_MAX_QUARTERS) return MD_ERR_BAD_ARG;
  switch (key) {
    case MD_OPT_SLICE_BITS:
      if (value != 0 && (value < MD_MIN_BITS || value > MD_MAX_BITS)) return MD_ERR_BAD_ARG;
      g_state.opt_bits = value;
      return MD_OK;
    case MD_OPT_QUARTERS: g_state.opt_quarters = value; return MD_OK;
    case MD_OPT_ORDERS: g_state.opt_orders = value; return MD_OK;
    default: return MD_ERR_BAD_ARG;
  }
}

int md_get_option(int key) {
  switch (key) {
    case MD_OPT_QUARTERS: return g_state.opt_quarters;
    case MD_OPT_ORDERS: return g_state.opt_orders;
    case MD_OPT_SLICE_BITS: return g_state.opt_bits;
    default: return -1;
  }
}

md_status md_split(int rows, int cols, int limbs, int quarters, int axis, const double* planes, double* quarter_planes,
                   int32_t* exps, md_stream stream) {
  if (rows <= 0 || cols <= 0 || !planes || !quarter_planes || !exps) return MD_ERR_BAD_ARG;
  if (limbs != 1 && limbs != 2 && limbs != 4 && limbs != 8 && limbs != 16) return MD_ERR_BAD_ARG;
  if (quarters < 1 || quarters > MD_MAX_QUARTERS || (axis != 0 && axis != 1)) return MD_ERR_BAD_ARG;
  if (!aligned8(planes) || !aligned8(quarter_planes) || (reinterpret_cast<uintptr_t>(exps) & 3)) return MD_ERR_BAD_ARG;
  uint32_t* flags = g_state.ws ? static_cast<uint32_t*>(g_state.ws) : nullptr;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  uint64_t launches = 0;
  const int W = slice_bits();
  cudaError_t err = md::launch_exponents(rows, cols, axis, quarters, W, planes, exps, flags, st, &launches);
  if (err == cudaSuccess)
    err = md::launch_split(rows, cols, limbs, quarters, W, axis, planes, quarter_planes, exps, flags, st, &launches);
  g_launches += launches;
  return err == cudaSuccess ? MD_OK : MD_ERR_CUDA;
}

md_status md_qgemm(int m, int n, int k, int limbs, int quarters, int orders, const double* Aq, const double* Bq,
                   double* order_planes, double* C_planes, md_stream stream) {
  if (m <= 0 || n <= 0 || k <= 0 || !Aq || !Bq || (!order_planes && !C_planes)) return MD_ERR_BAD_ARG;
  if (!aligned8(Aq) || !aligned8(Bq) || !aligned8(order_planes) || !aligned8(C_planes)) return MD_ERR_BAD_ARG;
  if (limbs != 2 && limbs != 4 && limbs != 8 && limbs != 16) return MD_ERR_BAD_ARG;
  // plain-layout quarter planes: double / quad double only (octo / hexa double go through md_gemm's packed operands)
  if (orders != quarters || !md::qgemm_supported(limbs, quarters)) return MD_ERR_UNSUPPORTED;
  if (!k_budget_ok(k, orders, slice_bits())) return MD_ERR_K_TOO_LARGE;
  uint64_t launches = 0;
  cudaError_t err = md::launch_qgemm(m, n, k, limbs, quarters, Aq, Bq, order_planes, C_planes,
                                     static_cast<cudaStream_t>(stream), &launches);
  g_launches += launches;
  return err == cudaSuccess ? MD_OK : MD_ERR_CUDA;
}

md_status md_renorm(int m, int n, int limbs, int orders, const double* order_planes, double* C_planes,
                    md_stream stream) {
  if (m <= 0 || n <= 0 || !order_planes || !C_planes) return MD_ERR_BAD_ARG;
  if (limbs != 1 && limbs != 2 && limbs != 4 && limbs != 8 && limbs != 16) return MD_ERR_BAD_ARG;
  if (orders < 1 || orders > 2 * MD_MAX_QUARTERS || !aligned8(order_planes) || !aligned8(C_planes)) return MD_ERR_BAD_ARG;
  uint64_t launches = 0;
  cudaError_t err = md::launch_renorm(m, n, limbs, orders, order_planes, C_planes, static_cast<cudaStream_t>(stream), &launches);
  g_launches += launches;
  return err == cudaSuccess ? MD_OK : MD_ERR_CUDA;
}

size_t md_workspace_bytes(int m, int n, int k, int limbs) {
  if (m <= 0 || n <= 0 || k <= 0 || (limbs != 2 && limbs != 4 && limbs != 8 && limbs != 16)) return 0;
  return carve(nullptr, m, n, k, limbs, quarters_for(limbs)).total;
}

md_status md_set_workspace(void* dev_ptr, size_t bytes) {
  if ((dev_ptr == nullptr) != (bytes == 0)) return MD_ERR_BAD_ARG;
  if (reinterpret_cast<uintptr_t>(dev_ptr) % ALIGN) return MD_ERR_BAD_ARG;
  if (dev_ptr && bytes < ALIGN) return MD_ERR_WORKSPACE;
  if (dev_ptr && cudaMemset(dev_ptr, 0, ALIGN) != cudaSuccess) return MD_ERR_CUDA;  // clear the status word
  g_state.ws = dev_ptr;
  g_state.ws_bytes = bytes;
  return MD_OK;
}

md_status md_read_flags(uint32_t* flags_host, md_stream stream) {
  if (!flags_host) return MD_ERR_BAD_ARG;
  if (!g_state.ws) return MD_ERR_WORKSPACE;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (cudaMemcpyAsync(flags_host, g_state.ws, sizeof(uint32_t), cudaMemcpyDeviceToHost, st) != cudaSuccess) return MD_ERR_CUDA;
  return cudaStreamSynchronize(st) == cudaSuccess ? MD_OK : MD_ERR_CUDA;
}

md_status md_gemm(int m, int n, int k, int limbs, const double* A_planes, const double* B_planes, double* C_planes,
                  md_stream stream) {
  const md_status st = check_gemm_args(m, n, k, limbs, A_planes, B_planes, C_planes);
  if (st != MD_OK) return st;
  return gemm_impl(m, n, k, limbs, A_planes, B_planes, C_planes, nullptr, g_state.ws, g_state.ws_bytes,
                   static_cast<cudaStream_t>(stream));
}

md_status md_gemm_orders(int m, int n, int k, int limbs, const double* A_planes, const double* B_planes,
                         double* order_planes, md_stream stream) {
  const md_status st = check_gemm_args(m, n, k, limbs, A_planes, B_planes, order_planes);
  if (st != MD_OK) return st;
  return gemm_impl(m, n, k, limbs, A_planes, B_planes, nullptr, order_planes, g_state.ws, g_state.ws_bytes,
                   static_cast<cudaStream_t>(stream));
}

md_status md_plan_slices(int k, int limbs, int* bits_out, int* quarters_out) {
  if (k <= 0 || !bits_out || !quarters_out) return MD_ERR_BAD_ARG;
  if (limbs != 2 && limbs != 4 && limbs != 8 && limbs != 16) return MD_ERR_BAD_ARG;
  // the fewest slices Q with a kernel, at the widest W the exactness budget allows for (k, Q), whose window W * Q covers
  // the paper's 13 * 4 * limbs bits; the paper's own (13, 4 * limbs) when nothing better qualifies
  for (int Q = 1; Q < 4 * limbs; Q++) {
    if (!(md::qgemm_supported(limbs, Q) || md::qgemm_wide_supported(limbs, Q))) continue;
    int W = MD_MAX_BITS;
    while (W >= MD_MIN_BITS && !k_budget_ok(k, Q, W)) W--;
    if (W >= MD_MIN_BITS && W * Q >= 52 * limbs) {
      *bits_out = W;
      *quarters_out = Q;
      return MD_OK;
    }
  }
  if (!k_budget_ok(k, 4 * limbs, 13)) return MD_ERR_K_TOO_LARGE;
  *bits_out = 13;
  *quarters_out = 4 * limbs;
  return MD_OK;
}

size_t md_host_scratch_bytes(int m, int n, int k, int limbs) {
  const size_t ws = md_workspace_bytes(m, n, k, limbs);
  if (!ws) return 0;
  return round_up(sizeof(double) * (size_t)limbs * m * k) + round_up(sizeof(double) * (size_t)limbs * k * n) +
         round_up(sizeof(double) * (size_t)limbs * m * n) + ws;
}

md_status md_gemm_host(int m, int n, int k, int limbs, const double* A_host, const double* B_host, double* C_host,
                       void* dev_scratch, size_t scratch_bytes, md_stream stream) {
  const md_status chk = check_gemm_args(m, n, k, limbs, A_host, B_host, C_host);
  if (chk != MD_OK) return chk;
  if (!dev_scratch || reinterpret_cast<uintptr_t>(dev_scratch) % ALIGN) return MD_ERR_BAD_ARG;
  if (scratch_bytes < md_host_scratch_bytes(m, n, k, limbs)) return MD_ERR_WORKSPACE;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const size_t a_bytes = sizeof(double) * (size_t)limbs * m * k, b_bytes = sizeof(double) * (size_t)limbs * k * n,
               c_bytes = sizeof(double) * (size_t)limbs * m * n;
  char* p = static_cast<char*>(dev_scratch);
  double* dA = reinterpret_cast<double*>(p);
  double* dB = reinterpret_cast<double*>(p + round_up(a_bytes));
  double* dC = reinterpret_cast<double*>(p + round_up(a_bytes) + round_up(b_bytes));
  char* ws = p + round_up(a_bytes) + round_up(b_bytes) + round_up(c_bytes);
  const size_t ws_bytes = scratch_bytes - (size_t)(ws - p);
  if (cudaMemsetAsync(ws, 0, ALIGN, st) != cudaSuccess) return MD_ERR_CUDA;
  if (cudaMemcpyAsync(dA, A_host, a_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return MD_ERR_CUDA;
  if (cudaMemcpyAsync(dB, B_host, b_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return MD_ERR_CUDA;
  const md_status run = gemm_impl(m, n, k, limbs, dA, dB, dC, nullptr, ws, ws_bytes, st);
  if (run != MD_OK) return run;
  if (cudaMemcpyAsync(C_host, dC, c_bytes, cudaMemcpyDeviceToHost, st) != cudaSuccess) return MD_ERR_CUDA;
  return cudaStreamSynchronize(st) == cudaSuccess ? MD_OK : MD_ERR_CUDA;
}

md_status md_profile_enable(int capacity) {
  if (capacity < 0 || capacity > (1 << 20)) return MD_ERR_BAD_ARG;
  for (cudaEvent_t e : g_prof.ev) cudaEventDestroy(e);
  g_prof.ev.clear();
  g_prof.capacity = g_prof.count = 0;
  g_prof.ev.resize(3 * (size_t)capacity);
  for (size_t i = 0; i < g_prof.ev.size(); i++)
    if (cudaEventCreate(&g_prof.ev[i]) != cudaSuccess) {
      for (size_t j = 0; j < i; j++) cudaEventDestroy(g_prof.ev[j]);
      g_prof.ev.clear();
      return MD_ERR_CUDA;
    }
  g_prof.capacity = capacity;
  return MD_OK;
}

int md_profile_read(float* split_ms_host, float* gemm_ms_host, int capacity) {
  if (capacity < g_prof.count) return MD_ERR_BAD_ARG;
  for (int i = 0; i < g_prof.count; i++) {
    cudaEvent_t* ev = &g_prof.ev[3 * (size_t)i];
    float a = 0.f, b = 0.f;
    if (cudaEventSynchronize(ev[2]) != cudaSuccess) return MD_ERR_CUDA;
    if (cudaEventElapsedTime(&a, ev[0], ev[1]) != cudaSuccess) return MD_ERR_CUDA;
    if (cudaEventElapsedTime(&b, ev[1], ev[2]) != cudaSuccess) return MD_ERR_CUDA;
    if (split_ms_host) split_ms_host[i] = a;
    if (gemm_ms_host) gemm_ms_host[i] = b;
  }
  return g_prof.count;
}

md_status md_probe_dmma(int blocks, int warps_per_block, int iters, double* sink, uint64_t* flops_host, md_stream stream) {
  if (blocks < 1 || warps_per_block < 1 || warps_per_block > 32 || iters < 1 || iters >= (1 << 25) || !flops_host)
    return MD_ERR_BAD_ARG;
  if (!aligned8(sink)) return MD_ERR_BAD_ARG;
  uint64_t launches = 0;
  cudaError_t err = md::launch_dmma_probe(blocks, warps_per_block, iters, sink, static_cast<cudaStream_t>(stream),
                                          &launches, flops_host);
  g_launches += launches;
  return err == cudaSuccess ? MD_OK : MD_ERR_CUDA;
}

uint64_t md_launch_count(void) { return g_launches.load(); }

const char* md_status_string(md_status status) {
  switch (status) {
    case MD_OK: return "MD_OK";
    case MD_ERR_BAD_ARG: return "MD_ERR_BAD_ARG: null/misaligned pointer, bad dimension, or unsupported limbs/quarters/orders value";
    case MD_ERR_K_TOO_LARGE: return "MD_ERR_K_TOO_LARGE: k * orders * 2^(2 * slice bits) exceeds 2^53 (k * orders > 2^27 for 13-bit quarters), fp64 accumulation would not be exact";
    case MD_ERR_WORKSPACE: return "MD_ERR_WORKSPACE: workspace missing or too small (md_workspace_bytes / md_host_scratch_bytes)";
    case MD_ERR_CUDA: return "MD_ERR_CUDA: a CUDA call failed (see cudaGetLastError)";
    case MD_ERR_UNSUPPORTED: return "MD_ERR_UNSUPPORTED: no kernel for this (limbs, quarters, orders)";
    default: return "unknown md_status";
  }
}

}  // extern "C"
