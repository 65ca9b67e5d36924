// api.cu -- the C-ABI of libmdgemm (include/mdgemm.h): argument checking, options, workspace carving, and the sequence
// of kernel launches of the hot path.  No arithmetic of the method lives here.
#include <atomic>
#include <cmath>
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
  int opt_tile = 0;        // 0 = automatic, 1 = the 32 x 16 tile instance wherever it exists, 2 = never
  int opt_fused_prep = 0;  // 0 = automatic (small / medium operands), 1 = always, 2 = never
  int opt_k_chunk = 0;   // 0 = chunked accumulation only when k exceeds the exactness budget; else the chunk length to force
  int opt_host_blocks = 0;  // md_gemm_host: 0 = automatic panel plan, else the number of blocks of C (1 = no pipelining)
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
// Exactness budget (eq. 5 generalised; R6, R14): order s adds (s+1) <= S products per k, each an
// integer of at most 2^(2W) units, so every partial sum is exactly representable while k * S * 2^(2W) <= 2^53.
// W = 13: k * S <= 2^27.
inline bool k_budget_ok(long long k, int S, int bits) { return k * S <= (1ll << (53 - 2 * bits)); }
// Chunked accumulation (R16): the budget is kept per chunk of the contraction; the chunk md_gemm uses for
// (limbs, S, W), a multiple of the k-slab depth 8, or 0 when the path stays unchunked / cannot be chunked.
inline int chunk_for(int k, int limbs, int S, int bits) {
  if (!md::qgemm_chunk_supported(limbs, S)) return 0;
  long long c = (1ll << (53 - 2 * bits)) / S;
  if (g_state.opt_k_chunk > 0 && g_state.opt_k_chunk < c) c = g_state.opt_k_chunk;
  c = c / md::PACK_BK * md::PACK_BK;
  if (c < md::PACK_BK) return 0;
  const bool needed = !k_budget_ok(k, S, bits) || !md::qgemm_supported(limbs, S) || (g_state.opt_k_chunk > 0 && k > c);
  return needed ? (int)(c > 0x40000000 ? 0x40000000 : c) : 0;
}

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
Carve carve(void* base, int m, int n, int k, int limbs, int quarters, bool small = false) {
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
  off += round_up(sizeof(double) * md::packed_doubles(m, k, md::pack_bx(limbs, quarters, 0, small), md::pack_bk(limbs), quarters));
  c.Bq = reinterpret_cast<double*>(p + off);
  off += round_up(sizeof(double) * md::packed_doubles(n, k, md::pack_bx(limbs, quarters, 1, small), md::pack_bk(limbs), quarters));
  c.sk = p + off;
  off += round_up(md::sk_workspace_bytes(limbs, quarters, k, chunk_for(k, limbs, quarters, slice_bits())));
  c.total = off;
  return c;
}

inline bool aligned8(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 7) == 0; }

md_status check_gemm_args(int m, int n, int k, int limbs, const void* A, const void* B, const void* C,
                          bool want_orders = false) {
  if (m <= 0 || n <= 0 || k <= 0 || !A || !B || !C) return MD_ERR_BAD_ARG;
  if (!aligned8(A) || !aligned8(B) || !aligned8(C)) return MD_ERR_BAD_ARG;
  if (limbs != 2 && limbs != 4 && limbs != 8 && limbs != 16) return MD_ERR_BAD_ARG;
  const int Q = quarters_for(limbs), S = orders_for(limbs);
  // order planes need the order sums of the WHOLE contraction to be exact doubles: no chunking there
  const int chunk = want_orders ? 0 : chunk_for(k, limbs, S, slice_bits());
  if (S != Q || !(md::qgemm_supported(limbs, Q) || md::qgemm_wide_supported(limbs, Q) || chunk > 0)) return MD_ERR_UNSUPPORTED;
  if (chunk == 0 && !k_budget_ok(k, S, slice_bits())) return MD_ERR_K_TOO_LARGE;
  return MD_OK;
}

// Fused preparation (one cooperative launch for both exponent vectors and both packed splits) where the latencies of five
// dependent launches show: measured faster up to 2048^3, equal at 4096^3
inline bool use_fused_prep(int m, int n, int k) {
  if (g_state.opt_fused_prep == 1) return true;
  if (g_state.opt_fused_prep == 2) return false;
  return ((long long)m + n) * k <= (1ll << 23);
}

// The 32 x 16 tile instance of the double-double kernel: where the 64 x 32 tiles would not fill the SMs (at most one tile
// per SM), every tile would be cut along k and each CTA would flush a whole tile of partial sums through L2 atomics; four
// times the tiles avoid most of that (measured).  Splitter and GEMM must agree on the answer.
inline bool use_small_tiles(int m, int n, int k, int limbs, int Q, int W) {
  if (!md::qgemm_small_supported(limbs, Q) || chunk_for(k, limbs, Q, W) > 0 || g_state.opt_tile == 2) return false;
  if (g_state.opt_tile == 1) return true;
  const int G = md::sk_grid();
  const long long tiles = ((long long)m + 63) / 64 * (((long long)n + 31) / 32);
  return G > 0 && 3 * tiles <= 2 * G;  // measured on dd n^3: faster up to n = 448 (98 tiles), slower from n = 512 (128 tiles)
}

// the fused quarter GEMM of one (block of a) problem on packed operands: double / quad double (chunked when md_gemm asks
// for C of a contraction beyond the exactness budget), octo / hexa double
cudaError_t launch_fused(int m, int n, int k, int limbs, int Q, int W, bool small, const double* Aq, const double* Bq,
                         double* order_planes, double* C_planes, void* sk, cudaStream_t stream, uint64_t* launches) {
  if (limbs > 4) return md::launch_qgemm_wide(m, n, k, limbs, Q, Aq, Bq, order_planes, C_planes, sk, stream, launches);
  const int chunk = order_planes ? 0 : chunk_for(k, limbs, Q, W);
  return md::launch_qgemm_packed(m, n, k, limbs, Q, chunk, small, Aq, Bq, order_planes, C_planes, sk, stream, launches);
}

// split A (rows) and B (columns) into the packed quarter planes of the carved workspace, then the fused quarter GEMM.
md_status gemm_impl(int m, int n, int k, int limbs, const double* A, const double* B, double* C_planes,
                    double* order_planes, void* ws, size_t ws_bytes, cudaStream_t stream) {
  const int Q = quarters_for(limbs), W = slice_bits();
  if (!ws) return MD_ERR_WORKSPACE;
  const bool small = use_small_tiles(m, n, k, limbs, Q, W);
  const Carve c = carve(ws, m, n, k, limbs, Q, small);
  if (c.total > ws_bytes) return MD_ERR_WORKSPACE;
  uint64_t launches = 0;
  cudaEvent_t* ev = (g_prof.count < g_prof.capacity) ? &g_prof.ev[3 * (size_t)g_prof.count] : nullptr;
  if (ev) cudaEventRecord(ev[0], stream);
  cudaError_t err = cudaErrorUnknown;
  if (use_fused_prep(m, n, k)) {  // one launch instead of five: what matters below ~2048^3
    err = md::launch_prep_packed(m, n, k, limbs, Q, W, small, A, B, c.Aq, c.Bq, c.expA, c.expB, c.flags, stream, &launches);
    if (err != cudaSuccess) cudaGetLastError();  // a cooperative launch the context cannot take: the separate kernels do the same
  }
  if (err != cudaSuccess) {
    err = md::launch_exponents(m, k, 0, Q, W, A, c.expA, c.flags, stream, &launches);
    if (err == cudaSuccess) err = md::launch_exponents(k, n, 1, Q, W, B, c.expB, c.flags, stream, &launches);
    if (err == cudaSuccess) err = md::launch_split_packed(m, k, limbs, Q, W, 0, small, A, c.Aq, c.expA, c.flags, stream, &launches);
    if (err == cudaSuccess) err = md::launch_split_packed(k, n, limbs, Q, W, 1, small, B, c.Bq, c.expB, c.flags, stream, &launches);
  }
  if (ev) cudaEventRecord(ev[1], stream);
  if (err == cudaSuccess) err = launch_fused(m, n, k, limbs, Q, W, small, c.Aq, c.Bq, order_planes, C_planes, c.sk, stream, &launches);
  if (ev) {
    cudaEventRecord(ev[2], stream);
    if (err == cudaSuccess) g_prof.count++;
  }
  g_launches += launches;
  return err == cudaSuccess ? MD_OK : MD_ERR_CUDA;
}


// ---- md_gemm_host: panel plan and the library's two copy streams ------------------------------------------------------
struct HostPanels {
  int PR, PC;  // row panels of A / C, column panels of B / C
  int mp, np;  // rows / columns per panel (multiples of the CTA tile; the last panel takes what is left)
};
// About one wave of CTA tiles per block, at most 32 blocks (the stream-K tail keeps a short block efficient; measured on
// dd 4096^3: 8 x 4 blocks 138.4 ms, 4 x 2 140.0 ms, 1 block 150.2 ms against 135.1 ms of kernels alone); four column
// panels from 16 blocks up, two from 4, so that the first kernel waits for a fraction of B only.
HostPanels plan_host_panels(int m, int n, int limbs, int quarters) {
  const int bxA = md::pack_bx(limbs, quarters, 0), bxB = md::pack_bx(limbs, quarters, 1);
  const long long tm = (m + bxA - 1) / bxA, tn = (n + bxB - 1) / bxB;
  int G = md::sk_grid();
  if (G <= 0) G = 148;
  long long blocks = (tm * tn + G - 1) / G;
  if (g_state.opt_host_blocks > 0) blocks = g_state.opt_host_blocks;
  blocks = blocks < 1 ? 1 : blocks > 32 ? 32 : blocks;
  HostPanels hp;
  hp.PC = blocks >= 16 ? 4 : blocks >= 4 ? 2 : 1;
  hp.PR = (int)(blocks / hp.PC);
  if (g_state.opt_host_blocks >= 256) hp.PR = g_state.opt_host_blocks >> 8, hp.PC = g_state.opt_host_blocks & 255;  // PR * 256 + PC
  if (hp.PR < 1) hp.PR = 1;
  if (hp.PC < 1) hp.PC = 1;
  if (hp.PC > tn) hp.PC = (int)tn;
  if (hp.PR > tm) hp.PR = (int)tm;
  hp.mp = (int)((tm + hp.PR - 1) / hp.PR) * bxA;
  hp.np = (int)((tn + hp.PC - 1) / hp.PC) * bxB;
  hp.PR = (m + hp.mp - 1) / hp.mp;
  hp.PC = (n + hp.np - 1) / hp.np;
  return hp;
}

struct HostPipeline {
  cudaStream_t in = nullptr, out = nullptr;
  std::vector<cudaEvent_t> ev;
};
HostPipeline g_host;
// streams and events are created on first use and kept (no device memory is allocated)
bool host_pipeline_ready(int events) {
  if (!g_host.in && cudaStreamCreateWithFlags(&g_host.in, cudaStreamNonBlocking) != cudaSuccess) return false;
  if (!g_host.out && cudaStreamCreateWithFlags(&g_host.out, cudaStreamNonBlocking) != cudaSuccess) return false;
  while ((int)g_host.ev.size() < events) {
    cudaEvent_t e;
    if (cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) return false;
    g_host.ev.push_back(e);
  }
  return true;
}

}  // namespace

extern "C" {

md_status md_set_option(int key, int value) {
  if (key == MD_OPT_K_CHUNK) {  // 0 = automatic, else a chunk length: a multiple of 8
    if (value < 0 || value % md::PACK_BK) return MD_ERR_BAD_ARG;
    g_state.opt_k_chunk = value;
    return MD_OK;
  }
  if (key == MD_OPT_TILE) {
    if (value < 0 || value > 2) return MD_ERR_BAD_ARG;
    g_state.opt_tile = value;
    return MD_OK;
  }
  if (key == MD_OPT_FUSED_PREP) {
    if (value < 0 || value > 2) return MD_ERR_BAD_ARG;
    g_state.opt_fused_prep = value;
    return MD_OK;
  }
  if (key == MD_OPT_HOST_BLOCKS) {  // 0 = automatic, 1..32 blocks, or PR * 256 + PC (explicit panel counts, each <= 64)
    if (value < 0 || (value > 32 && (value < 256 || (value >> 8) > 64 || (value & 255) > 64))) return MD_ERR_BAD_ARG;
    g_state.opt_host_blocks = value;
    return MD_OK;
  }
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
    case MD_OPT_HOST_BLOCKS: return g_state.opt_host_blocks;
    case MD_OPT_K_CHUNK: return g_state.opt_k_chunk;
    case MD_OPT_FUSED_PREP: return g_state.opt_fused_prep;
    case MD_OPT_TILE: return g_state.opt_tile;
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
  const md_status st = check_gemm_args(m, n, k, limbs, A_planes, B_planes, order_planes, true);
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

md_status md_plan_slices_chunked(int k, int limbs, int min_chunk, int* bits_out, int* quarters_out, int* chunk_out) {
  if (k <= 0 || min_chunk < md::PACK_BK || !bits_out || !quarters_out || !chunk_out) return MD_ERR_BAD_ARG;
  if (limbs != 2 && limbs != 4 && limbs != 8 && limbs != 16) return MD_ERR_BAD_ARG;
  // as md_plan_slices, but the budget only has to hold for a chunk of at least min_chunk contraction indices where a
  // chunked kernel exists: the fewest slices, then the widest width
  for (int Q = 1; Q < 4 * limbs; Q++) {
    const bool whole = md::qgemm_supported(limbs, Q) || md::qgemm_wide_supported(limbs, Q);
    const bool chunked = md::qgemm_chunk_supported(limbs, Q);
    if (!whole && !chunked) continue;
    for (int W = MD_MAX_BITS; W >= MD_MIN_BITS && W * Q >= 52 * limbs; W--) {
      if (whole && k_budget_ok(k, Q, W)) {
        *bits_out = W, *quarters_out = Q, *chunk_out = 0;
        return MD_OK;
      }
      const long long c = (1ll << (53 - 2 * W)) / Q / md::PACK_BK * md::PACK_BK;
      if (chunked && c >= min_chunk) {
        *bits_out = W, *quarters_out = Q, *chunk_out = (int)(c < k ? c : 0);
        return MD_OK;
      }
    }
  }
  *chunk_out = 0;
  return md_plan_slices(k, limbs, bits_out, quarters_out);
}

size_t md_plan_scratch_bytes(int m, int n, int k) {
  if (m <= 0 || n <= 0 || k <= 0) return 0;
  return ALIGN + round_up(sizeof(int32_t) * (size_t)m) + round_up(sizeof(int32_t) * (size_t)n) +
         round_up(sizeof(double) * (size_t)m * k) + round_up(sizeof(double) * (size_t)k * n) +
         round_up(sizeof(double) * (size_t)m * n);
}

md_status md_plan_quarters(int m, int n, int k, int limbs, const double* A_planes, const double* B_planes, void* scratch,
                           size_t scratch_bytes, double rel_tol, int* quarters_out, int* spread_out, md_stream stream) {
  if (m <= 0 || n <= 0 || k <= 0 || !A_planes || !B_planes || !scratch || !quarters_out) return MD_ERR_BAD_ARG;
  if (limbs != 1 && limbs != 2 && limbs != 4 && limbs != 8 && limbs != 16) return MD_ERR_BAD_ARG;
  if (!aligned8(A_planes) || !aligned8(B_planes) || reinterpret_cast<uintptr_t>(scratch) % ALIGN) return MD_ERR_BAD_ARG;
  if (scratch_bytes < md_plan_scratch_bytes(m, n, k)) return MD_ERR_WORKSPACE;
  if (rel_tol == 0.0) rel_tol = limbs == 1 ? 0x1p-50 : limbs == 2 ? 1e-28 : limbs == 4 ? 1e-58 : limbs == 8 ? 1e-120 : 1e-245;
  if (!(rel_tol > 0.0)) return MD_ERR_BAD_ARG;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int W = slice_bits();
  char* p = static_cast<char*>(scratch);
  int32_t* spread = reinterpret_cast<int32_t*>(p);
  int32_t* expA = reinterpret_cast<int32_t*>(p + ALIGN);
  int32_t* expB = reinterpret_cast<int32_t*>(p + ALIGN + round_up(sizeof(int32_t) * (size_t)m));
  double* absA = reinterpret_cast<double*>(reinterpret_cast<char*>(expB) + round_up(sizeof(int32_t) * (size_t)n));
  double* absB = reinterpret_cast<double*>(reinterpret_cast<char*>(absA) + round_up(sizeof(double) * (size_t)m * k));
  double* Wt = reinterpret_cast<double*>(reinterpret_cast<char*>(absB) + round_up(sizeof(double) * (size_t)k * n));
  const int32_t none = INT32_MIN;
  uint64_t launches = 0;
  cudaError_t err = cudaMemcpyAsync(spread, &none, sizeof(none), cudaMemcpyHostToDevice, st);
  // exponent vectors of the leading limb planes, |A_0| |B_0| on the DMMA kernel, then the spread D
  if (err == cudaSuccess) err = md::launch_exponents(m, k, 0, 4 * limbs, W, A_planes, expA, nullptr, st, &launches);
  if (err == cudaSuccess) err = md::launch_exponents(k, n, 1, 4 * limbs, W, B_planes, expB, nullptr, st, &launches);
  if (err == cudaSuccess) err = md::launch_abs((size_t)m * k, A_planes, absA, st, &launches);
  if (err == cudaSuccess) err = md::launch_abs((size_t)k * n, B_planes, absB, st, &launches);
  if (err == cudaSuccess) err = md::launch_plain_dgemm(m, n, k, absA, absB, Wt, st, &launches);
  if (err == cudaSuccess) err = md::launch_spread(m, n, Wt, expA, expB, spread, st, &launches);
  g_launches += launches;
  int32_t D = 0;
  if (err == cudaSuccess) err = cudaMemcpyAsync(&D, spread, sizeof(D), cudaMemcpyDeviceToHost, st);
  if (err != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess) return MD_ERR_CUDA;
  if (spread_out) *spread_out = D;
  // the smallest Q >= ceil(52 limbs / W) with k (Q+1) 2^(D - W Q - 2) <= rel_tol (R15; the left side is exact)
  int Q = (52 * limbs + W - 1) / W;
  if (D != INT32_MIN)
    while (Q < 4096 && ldexp((double)k * (Q + 1), D - W * Q - 2) > rel_tol) Q++;
  *quarters_out = Q;
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
  const int Q = quarters_for(limbs), W = slice_bits();
  const size_t a_bytes = sizeof(double) * (size_t)limbs * m * k, b_bytes = sizeof(double) * (size_t)limbs * k * n,
               c_bytes = sizeof(double) * (size_t)limbs * m * n;
  char* p = static_cast<char*>(dev_scratch);
  double* dA = reinterpret_cast<double*>(p);
  double* dB = reinterpret_cast<double*>(p + round_up(a_bytes));
  double* dC = reinterpret_cast<double*>(p + round_up(a_bytes) + round_up(b_bytes));
  char* ws = p + round_up(a_bytes) + round_up(b_bytes) + round_up(c_bytes);
  const Carve c = carve(ws, m, n, k, limbs, Q);

  // Panels: C is cut into PR x PC blocks (rows of A x columns of B).  A row's exponent and quarters depend on that row of A
  // only, a column's on that column of B only, so every block is an independent md_gemm on COMPACT
  // device copies of its operands: panel i of A is [limbs][mi][k] at dA + limbs * row0 * k, panel j of B is [limbs][k][nj]
  // at dB + limbs * k * col0, block (i, j) of C is [limbs][mi][nj].  Three streams: copies in (in order of first use),
  // the kernels (the caller's stream), copies out; the first kernel starts after A_0 and B_0 have arrived and the last
  // copy out is one block of C, instead of the whole of A, B before and the whole of C after.
  const HostPanels hp = plan_host_panels(m, n, limbs, Q);
  if (hp.PR == 1 && hp.PC == 1) {  // one block: nothing to overlap -- copy in, the device path as md_gemm runs it, copy out
    if (cudaMemsetAsync(ws, 0, ALIGN, st) != cudaSuccess) return MD_ERR_CUDA;
    if (cudaMemcpyAsync(dA, A_host, a_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return MD_ERR_CUDA;
    if (cudaMemcpyAsync(dB, B_host, b_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return MD_ERR_CUDA;
    const md_status run = gemm_impl(m, n, k, limbs, dA, dB, dC, nullptr, ws, scratch_bytes - (size_t)(ws - p), st);
    if (run != MD_OK) return run;
    if (cudaMemcpyAsync(C_host, dC, c_bytes, cudaMemcpyDeviceToHost, st) != cudaSuccess) return MD_ERR_CUDA;
    return cudaStreamSynchronize(st) == cudaSuccess ? MD_OK : MD_ERR_CUDA;
  }
  if (!host_pipeline_ready(hp.PR + hp.PC + hp.PR * hp.PC + 2)) return MD_ERR_CUDA;
  cudaStream_t s_in = g_host.in, s_out = g_host.out;
  cudaEvent_t* ev = g_host.ev.data();
  cudaEvent_t ev_start = ev[0], ev_done = ev[1];
  cudaEvent_t* ev_A = ev + 2;
  cudaEvent_t* ev_B = ev_A + hp.PR;
  cudaEvent_t* ev_C = ev_B + hp.PC;
#define MD_TRY(call) \
  if ((call) != cudaSuccess) return MD_ERR_CUDA
  MD_TRY(cudaMemsetAsync(ws, 0, ALIGN, st));  // the status word
  MD_TRY(cudaEventRecord(ev_start, st));
  MD_TRY(cudaStreamWaitEvent(s_in, ev_start, 0));
  MD_TRY(cudaStreamWaitEvent(s_out, ev_start, 0));
  auto rows_of = [&](int i, int& r0, int& mi) { r0 = i * hp.mp, mi = (r0 + hp.mp <= m ? hp.mp : m - r0); };
  auto cols_of = [&](int j, int& c0, int& nj) { c0 = j * hp.np, nj = (c0 + hp.np <= n ? hp.np : n - c0); };
  auto copy_in_A = [&](int i) -> cudaError_t {
    int r0, mi;
    rows_of(i, r0, mi);
    double* dst = dA + (size_t)limbs * r0 * k;
    for (int l = 0; l < limbs; l++) {
      cudaError_t e = cudaMemcpyAsync(dst + (size_t)l * mi * k, A_host + (size_t)l * m * k + (size_t)r0 * k,
                                      sizeof(double) * (size_t)mi * k, cudaMemcpyHostToDevice, s_in);
      if (e != cudaSuccess) return e;
    }
    return cudaEventRecord(ev_A[i], s_in);
  };
  auto copy_in_B = [&](int j) -> cudaError_t {
    int c0, nj;
    cols_of(j, c0, nj);
    double* dst = dB + (size_t)limbs * k * c0;
    // all limb planes at once: limbs * k rows of nj doubles out of rows of n
    cudaError_t e = cudaMemcpy2DAsync(dst, sizeof(double) * (size_t)nj, B_host + c0, sizeof(double) * (size_t)n,
                                      sizeof(double) * (size_t)nj, (size_t)limbs * k, cudaMemcpyHostToDevice, s_in);
    if (e != cudaSuccess) return e;
    return cudaEventRecord(ev_B[j], s_in);
  };
  // copies in, in the order the blocks (column panel outer, row panel inner) first touch them
  MD_TRY(copy_in_A(0));
  MD_TRY(copy_in_B(0));
  for (int i = 1; i < hp.PR; i++) MD_TRY(copy_in_A(i));
  for (int j = 1; j < hp.PC; j++) MD_TRY(copy_in_B(j));

  const int bxA = md::pack_bx(limbs, Q, 0), bxB = md::pack_bx(limbs, Q, 1), bk = md::pack_bk(limbs);
  const size_t KS = ((size_t)k + bk - 1) / bk;
  const size_t chunkA = (size_t)Q * bk * bxA, chunkB = (size_t)Q * bk * bxB;  // doubles per (tile, k slab)
  uint64_t launches = 0;
  cudaError_t err = cudaSuccess;
  for (int j = 0; j < hp.PC && err == cudaSuccess; j++) {
    int c0, nj;
    cols_of(j, c0, nj);
    const double* Bj = dB + (size_t)limbs * k * c0;
    double* Bq = c.Bq + (size_t)(c0 / bxB) * KS * chunkB;  // panel boundaries are multiples of the CTA tile
    MD_TRY(cudaStreamWaitEvent(st, ev_B[j], 0));
    err = md::launch_exponents(k, nj, 1, Q, W, Bj, c.expB + c0, c.flags, st, &launches);
    if (err == cudaSuccess) err = md::launch_split_packed(k, nj, limbs, Q, W, 1, false, Bj, Bq, c.expB + c0, c.flags, st, &launches);
    for (int i = 0; i < hp.PR && err == cudaSuccess; i++) {
      int r0, mi;
      rows_of(i, r0, mi);
      const double* Ai = dA + (size_t)limbs * r0 * k;
      double* Aq = c.Aq + (size_t)(r0 / bxA) * KS * chunkA;
      if (j == 0) {
        MD_TRY(cudaStreamWaitEvent(st, ev_A[i], 0));
        err = md::launch_exponents(mi, k, 0, Q, W, Ai, c.expA + r0, c.flags, st, &launches);
        if (err == cudaSuccess) err = md::launch_split_packed(mi, k, limbs, Q, W, 0, false, Ai, Aq, c.expA + r0, c.flags, st, &launches);
        if (err != cudaSuccess) break;
      }
      // block (i, j): compact [limbs][mi][nj] at the position its elements have in a row-panel-major walk of C
      double* Cb = dC + (size_t)limbs * ((size_t)r0 * n + (size_t)mi * c0);
      err = launch_fused(mi, nj, k, limbs, Q, W, false, Aq, Bq, nullptr, Cb, c.sk, st, &launches);  // the host path keeps the 64 x 32 tiles its panels are cut to
      if (err != cudaSuccess) break;
      cudaEvent_t done = ev_C[j * hp.PR + i];
      MD_TRY(cudaEventRecord(done, st));
      MD_TRY(cudaStreamWaitEvent(s_out, done, 0));
      for (int l = 0; l < limbs; l++)
        MD_TRY(cudaMemcpy2DAsync(C_host + (size_t)l * m * n + (size_t)r0 * n + c0, sizeof(double) * (size_t)n,
                                 Cb + (size_t)l * mi * nj, sizeof(double) * (size_t)nj, sizeof(double) * (size_t)nj,
                                 (size_t)mi, cudaMemcpyDeviceToHost, s_out));
    }
  }
  g_launches += launches;
  // join: the caller's stream waits for the last copy out (and, on an error path, for whatever was enqueued)
  MD_TRY(cudaEventRecord(ev_done, s_out));
  MD_TRY(cudaStreamWaitEvent(st, ev_done, 0));
#undef MD_TRY
  if (cudaStreamSynchronize(st) != cudaSuccess || err != cudaSuccess) return MD_ERR_CUDA;
  return MD_OK;
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
