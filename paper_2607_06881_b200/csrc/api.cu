// api.cu -- the C-ABI of libmdgemm (include/mdgemm.h): argument checking, options, workspace carving, and the sequence
// of kernel launches of the hot path.  No arithmetic of the method lives here.
#include <atomic>
#include <cmath>
#include <cstdint>
#include <vector>

#include "../../include/mdgemm.h"
#include "api_internal.h"
#include "md_common.cuh"
#include "md_kernels.h"
#include "md_packed.cuh"

namespace md {

Options g_opt;
DeviceState g_dev[MD_MAX_DEVICES];
std::atomic<uint64_t> g_launches{0};

int current_device() {
  int dev = -1;
  return cudaGetDevice(&dev) == cudaSuccess ? dev : -1;
}

// SM count of the current device, cached per device (a process may drive several GPUs)
int sm_count() {
  const int dev = current_device();
  if (dev < 0) return -1;
  if (dev >= MD_MAX_DEVICES) {
    int v = 0;
    return cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess ? v : -1;
  }
  if (g_dev[dev].sms == 0) {
    int v = 0;
    if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -1;
    g_dev[dev].sms = v;
  }
  return g_dev[dev].sms;
}

DeviceState* device_state() {
  const int dev = current_device();
  if (dev < 0) return &g_dev[0];  // no usable device: argument checks still work, the first CUDA call reports the failure
  return dev < MD_MAX_DEVICES ? &g_dev[dev] : nullptr;
}

int raster_group() { return g_opt.raster_group ? g_opt.raster_group : 8; }
int tile_schedule() { return g_opt.tile_schedule; }

// Chunked accumulation (R16): the budget is kept per chunk of the contraction; the chunk md_gemm uses for
// (limbs, S, W), a multiple of the k-slab depth 8, or 0 when the path stays unchunked / cannot be chunked.
int chunk_for(int k, int limbs, int Q, int S, int bits) {
  if (S != Q || !qgemm_chunk_supported(limbs, S)) return 0;
  long long c = (1ll << (53 - 2 * bits)) / S;
  if (g_opt.k_chunk > 0 && g_opt.k_chunk < c) c = g_opt.k_chunk;
  c = c / PACK_BK * PACK_BK;
  if (c < PACK_BK) return 0;
  const bool needed = !k_budget_ok(k, S, bits) || !qgemm_packed_supported(limbs, Q, S) || (g_opt.k_chunk > 0 && k > c);
  return needed ? (int)(c > 0x40000000 ? 0x40000000 : c) : 0;
}

// The 32 x 16 tile instance of the double-double kernel: where the 64 x 32 tiles would not fill the SMs (at most one tile
// per SM), every tile would be cut along k and each CTA would flush a whole tile of partial sums through L2 atomics; four
// times the tiles avoid most of that (measured).
static bool use_small_tiles(int m, int n, int limbs, int Q, int S) {
  if (!qgemm_small_supported(limbs, Q, S) || g_opt.tile == 2) return false;
  if (g_opt.tile == 1) return true;
  const int G = sk_grid();
  const long long tiles = ((long long)m + 63) / 64 * (((long long)n + 31) / 32);
  // measured on dd n^3 with the stream-K hand-over in place (profiles/r04_small_sizes.md section 8): the small tile is faster up
  // to n = 352 (66 large tiles: 0.80 against 0.75 of the peak), even at 368 and slower from n = 384 (72 tiles: 0.82 against 0.85).
  // (Before the hand-over, when every cut tile went through L2 atomics, it won up to 448.)
  return G > 0 && 20 * tiles <= 9 * G;
}

// Which fused kernel runs (limbs, Q, S) on an m x n x k problem, and hence the packed layout the splitter writes for it:
// a tuned instance where one exists, else the generic kernel (runtime Q, S; qgemm_wide.cu).
KernelPick pick_kernel(int m, int n, int k, int limbs, int Q, int S, int bits, bool want_orders, bool allow_small) {
  KernelPick p{GEMM_NONE, 0, 0, 0, 0};
  const int chunk = want_orders ? 0 : chunk_for(k, limbs, Q, S, bits);
  if (limbs <= 4 && chunk > 0) {
    p = {GEMM_PACKED, pack_bx(limbs, Q, 0), pack_bx(limbs, Q, 1), PACK_BK, chunk};
  } else if (limbs <= 4 && qgemm_packed_supported(limbs, Q, S)) {
    const bool small = allow_small && use_small_tiles(m, n, limbs, Q, S);
    p = {small ? GEMM_PACKED_SMALL : GEMM_PACKED, pack_bx(limbs, Q, 0, small), pack_bx(limbs, Q, 1, small), PACK_BK, 0};
  } else if (limbs > 4 && S == Q && qgemm_wide_supported(limbs, Q)) {
    p = {GEMM_WIDE, pack_bx(limbs, Q, 0), pack_bx(limbs, Q, 1), PACK_BK_WIDE, 0};
  } else if (qgemm_generic_supported(limbs, Q, S)) {
    p = {GEMM_GENERIC, pack_bx_generic(limbs, 0), pack_bx_generic(limbs, 1), PACK_BK_WIDE, 0};
  }
  return p;
}

Carve carve(void* base, int m, int n, int k, int Q, int S, const KernelPick& pick) {
  Carve c;
  size_t off = 0;
  char* p = static_cast<char*>(base);
  c.flags = reinterpret_cast<uint32_t*>(p + off);
  off += WS_ALIGN;
  c.expA = reinterpret_cast<int32_t*>(p + off);
  off += ws_round_up(sizeof(int32_t) * (size_t)m);
  c.expB = reinterpret_cast<int32_t*>(p + off);
  off += ws_round_up(sizeof(int32_t) * (size_t)n);
  c.Aq = reinterpret_cast<double*>(p + off);
  off += ws_round_up(sizeof(double) * packed_doubles(m, k, pick.bxA, pick.bk, Q));
  c.Bq = reinterpret_cast<double*>(p + off);
  off += ws_round_up(sizeof(double) * packed_doubles(n, k, pick.bxB, pick.bk, Q));
  c.sk = p + off;
  off += ws_round_up(sk_workspace_bytes(S, pick.bxA, pick.bxB, k, pick.chunk));
  c.total = off;
  return c;
}

static inline bool aligned8(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 7) == 0; }
static inline bool limbs_ok(int limbs) { return limbs == 2 || limbs == 4 || limbs == 8 || limbs == 16; }

md_status check_gemm_args(int m, int n, int k, int limbs, const void* A, const void* B, const void* C, bool want_orders) {
  if (m <= 0 || n <= 0 || k <= 0 || !A || !B || !C) return MD_ERR_BAD_ARG;
  if (!aligned8(A) || !aligned8(B) || !aligned8(C)) return MD_ERR_BAD_ARG;
  if (!limbs_ok(limbs)) return MD_ERR_BAD_ARG;
  const int Q = quarters_for(limbs), S = orders_for(limbs);
  // order planes need the order sums of the WHOLE contraction to be exact doubles: no chunking there
  const KernelPick pick = pick_kernel(m, n, k, limbs, Q, S, slice_bits(), want_orders, true);
  if (pick.family == GEMM_NONE) return MD_ERR_UNSUPPORTED;
  if (pick.chunk == 0 && !k_budget_ok(k, S, slice_bits())) return MD_ERR_K_TOO_LARGE;
  return MD_OK;
}

// Fused preparation (one cooperative launch for both exponent vectors and both packed splits) where the latencies of five
// dependent launches show: measured faster up to 2048^3, equal at 4096^3
static inline bool use_fused_prep(int m, int n, int k) {
  if (g_opt.fused_prep == 1) return true;
  if (g_opt.fused_prep == 2) return false;
  return ((long long)m + n) * k <= (1ll << 23);
}

// The whole path in ONE launch (fused_small.cu): where the 32 x 16 tiles of C number at most the SMs, so that a tile per CTA
// (times the k-runs of its cluster) is a single wave, and a CTA's run of the contraction is short (at most 16 k-slabs: the CTA
// splits its own operand slabs, which costs about 0.6 of the DMMA time of the slab -- measured: faster than prepare + multiply
// up to 192^3 and slower from 224^3 on, where a tile's contraction is no longer shared by a cluster).
constexpr int ONE_LAUNCH_MAX_SLABS = 16;
static bool use_one_launch(int m, int n, int k, int limbs, int Q, int S, int bits) {
  if (g_opt.one_launch == 2 || !fused_small_supported(limbs, Q, S) || chunk_for(k, limbs, Q, S, bits) > 0) return false;
  if (g_opt.one_launch == 1) return true;
  const long long tiles = (((long long)m + 31) / 32) * (((long long)n + 15) / 16);
  const int G = sk_grid();
  if (G <= 0 || tiles > G) return false;
  const int KS = (k + 7) / 8;
  return (KS + fused_small_cluster(m, n, k) - 1) / fused_small_cluster(m, n, k) <= ONE_LAUNCH_MAX_SLABS;
}

// the fused quarter GEMM of one (block of a) problem on packed operands
cudaError_t launch_fused(int m, int n, int k, int limbs, int Q, int S, const KernelPick& pick, const double* Aq, const double* Bq,
                         double* order_planes, double* C_planes, void* sk, bool counters_clear, cudaStream_t stream,
                         uint64_t* launches) {
  switch (pick.family) {
    case GEMM_PACKED:
    case GEMM_PACKED_SMALL:
      return launch_qgemm_packed(m, n, k, limbs, Q, S, order_planes ? 0 : pick.chunk, pick.family == GEMM_PACKED_SMALL, Aq, Bq,
                                 order_planes, C_planes, sk, counters_clear, stream, launches);
    case GEMM_WIDE: return launch_qgemm_wide(m, n, k, limbs, Q, Aq, Bq, order_planes, C_planes, sk, stream, launches);
    case GEMM_GENERIC: return launch_qgemm_generic(m, n, k, limbs, Q, S, Aq, Bq, order_planes, C_planes, sk, stream, launches);
    default: return cudaErrorInvalidValue;
  }
}

// split A (rows) and B (columns) into the packed quarter planes of the carved workspace, then the fused quarter GEMM.
md_status gemm_impl(int m, int n, int k, int limbs, int Q, int S, const double* A, const double* B, double* C_planes,
                    double* order_planes, void* ws, size_t ws_bytes, cudaStream_t stream, bool allow_small) {
  const int W = slice_bits();
  if (!ws) return MD_ERR_WORKSPACE;
  const KernelPick pick = pick_kernel(m, n, k, limbs, Q, S, W, order_planes != nullptr, allow_small);
  if (pick.family == GEMM_NONE) return MD_ERR_UNSUPPORTED;
  const Carve c = carve(ws, m, n, k, Q, S, pick);
  if (c.total > ws_bytes) return MD_ERR_WORKSPACE;
  uint64_t launches = 0;
  DeviceState* ds = device_state();
  cudaEvent_t* ev = (ds && ds->prof_count < ds->prof_capacity) ? &ds->prof_ev[3 * (size_t)ds->prof_count] : nullptr;
  if (ev) cudaEventRecord(ev[0], stream);
  cudaError_t err = cudaErrorUnknown;
  if (allow_small && use_one_launch(m, n, k, limbs, Q, S, W)) {  // a1-a4 in one kernel, no quarter planes in HBM
    if (ev) cudaEventRecord(ev[1], stream);
    err = launch_fused_small(m, n, k, limbs, Q, S, W, A, B, order_planes, C_planes, c.flags, stream, &launches);
    if (err == cudaSuccess) {
      if (ev) {
        cudaEventRecord(ev[2], stream);
        ds->prof_count++;
      }
      g_launches += launches;
      return MD_OK;
    }
    cudaGetLastError();  // a cluster launch the context cannot take: the two-launch path does the same work
    err = cudaErrorUnknown;
  }
  bool counters_clear = false;
  if (use_fused_prep(m, n, k)) {  // one launch instead of five: what matters below ~2048^3
    err = launch_prep_packed(m, n, k, limbs, Q, W, pick.bxA, pick.bxB, pick.bk, A, B, c.Aq, c.Bq, c.expA, c.expB, c.flags, c.sk, stream, &launches);
    if (err != cudaSuccess) cudaGetLastError();  // a cooperative launch the context cannot take: the separate kernels do the same
    else counters_clear = true;                  // the preparation kernel has also cleared the fused kernel's counter / flag words
  }
  if (err != cudaSuccess) {
    err = launch_exponents(m, k, 0, Q, W, A, c.expA, c.flags, stream, &launches);
    if (err == cudaSuccess) err = launch_exponents(k, n, 1, Q, W, B, c.expB, c.flags, stream, &launches);
    if (err == cudaSuccess) err = launch_split_packed(m, k, limbs, Q, W, 0, pick.bxA, pick.bk, A, c.Aq, c.expA, c.flags, stream, &launches);
    if (err == cudaSuccess) err = launch_split_packed(k, n, limbs, Q, W, 1, pick.bxB, pick.bk, B, c.Bq, c.expB, c.flags, stream, &launches);
  }
  if (ev) cudaEventRecord(ev[1], stream);
  if (err == cudaSuccess) err = launch_fused(m, n, k, limbs, Q, S, pick, c.Aq, c.Bq, order_planes, C_planes, c.sk, counters_clear, stream, &launches);
  if (ev) {
    cudaEventRecord(ev[2], stream);
    if (err == cudaSuccess) ds->prof_count++;
  }
  g_launches += launches;
  return err == cudaSuccess ? MD_OK : MD_ERR_CUDA;
}

size_t workspace_bytes_for(int m, int n, int k, int limbs, int Q, int S) {
  // the pick may choose the small-tile instance, whose padding differs: size for the larger of the layouts in question
  const KernelPick a = pick_kernel(m, n, k, limbs, Q, S, slice_bits(), false, false);
  const KernelPick b = pick_kernel(m, n, k, limbs, Q, S, slice_bits(), false, true);
  const KernelPick o = pick_kernel(m, n, k, limbs, Q, S, slice_bits(), true, true);  // md_gemm_orders never chunks
  size_t best = 0;
  for (const KernelPick* p : {&a, &b, &o})
    if (p->family != GEMM_NONE) {
      const size_t t = carve(nullptr, m, n, k, Q, S, *p).total;
      if (t > best) best = t;
    }
  return best;
}

// ---- md_gemm_host: panel plan and the library's two copy streams ------------------------------------------------------
struct HostPanels {
  int PR, PC;  // row panels of A / C, column panels of B / C
  int mp, np;  // rows / columns per panel (multiples of the CTA tile; the last panel takes what is left)
};
// About one wave of CTA tiles per block, at most 32 blocks (the stream-K tail keeps a short block efficient; measured on
// dd 4096^3: 8 x 4 blocks 138.4 ms, 4 x 2 140.0 ms, 1 block 150.2 ms against 135.1 ms of kernels alone); four column
// panels from 16 blocks up, two from 4, so that the first kernel waits for a fraction of B only.
static HostPanels plan_host_panels(int m, int n, int bxA, int bxB) {
  const long long tm = (m + bxA - 1) / bxA, tn = (n + bxB - 1) / bxB;
  int G = sk_grid();
  if (G <= 0) G = 1;
  long long blocks = (tm * tn + G - 1) / G;
  if (g_opt.host_blocks > 0) blocks = g_opt.host_blocks;
  blocks = blocks < 1 ? 1 : blocks > 32 ? 32 : blocks;
  HostPanels hp;
  hp.PC = blocks >= 16 ? 4 : blocks >= 4 ? 2 : 1;
  hp.PR = (int)(blocks / hp.PC);
  if (g_opt.host_blocks >= 256) hp.PR = g_opt.host_blocks >> 8, hp.PC = g_opt.host_blocks & 255;  // PR * 256 + PC
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

// streams and events are created on first use and kept, per device (no device memory is allocated)
static bool host_pipeline_ready(DeviceState* ds, int events) {
  if (!ds->host_in && cudaStreamCreateWithFlags(&ds->host_in, cudaStreamNonBlocking) != cudaSuccess) return false;
  if (!ds->host_out && cudaStreamCreateWithFlags(&ds->host_out, cudaStreamNonBlocking) != cudaSuccess) return false;
  while ((int)ds->host_ev.size() < events) {
    cudaEvent_t e;
    if (cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) return false;
    ds->host_ev.push_back(e);
  }
  return true;
}

}  // namespace md

using namespace md;

extern "C" {

md_status md_set_option(int key, int value) {
  switch (key) {
    case MD_OPT_K_CHUNK:  // 0 = automatic, else a chunk length: a multiple of 8
      if (value < 0 || value % PACK_BK) return MD_ERR_BAD_ARG;
      g_opt.k_chunk = value;
      return MD_OK;
    case MD_OPT_TILE:
      if (value < 0 || value > 2) return MD_ERR_BAD_ARG;
      g_opt.tile = value;
      return MD_OK;
    case MD_OPT_RASTER_GROUP:
      if (value < 0 || value > 1024) return MD_ERR_BAD_ARG;
      g_opt.raster_group = value;
      return MD_OK;
    case MD_OPT_FUSED_PREP:
      if (value < 0 || value > 2) return MD_ERR_BAD_ARG;
      g_opt.fused_prep = value;
      return MD_OK;
    case MD_OPT_ONE_LAUNCH:
      if (value < 0 || value > 2) return MD_ERR_BAD_ARG;
      g_opt.one_launch = value;
      return MD_OK;
    case MD_OPT_TILE_SCHEDULE:
      if (value < 0 || value > 3) return MD_ERR_BAD_ARG;
      g_opt.tile_schedule = value;
      return MD_OK;
    case MD_OPT_HOST_BLOCKS:  // 0 = automatic, 1..32 blocks, or PR * 256 + PC (explicit panel counts, each <= 64)
      if (value < 0 || (value > 32 && (value < 256 || (value >> 8) > 64 || (value & 255) > 64))) return MD_ERR_BAD_ARG;
      g_opt.host_blocks = value;
      return MD_OK;
    case MD_OPT_SLICE_BITS:
      if (value != 0 && (value < MD_MIN_BITS || value > MD_MAX_BITS)) return MD_ERR_BAD_ARG;
      g_opt.bits = value;
      return MD_OK;
    case MD_OPT_QUARTERS:
      if (value < 0 || value > MD_MAX_QUARTERS) return MD_ERR_BAD_ARG;
      g_opt.quarters = value;
      return MD_OK;
    case MD_OPT_ORDERS:
      if (value < 0 || value > MD_MAX_QUARTERS + 2) return MD_ERR_BAD_ARG;
      g_opt.orders = value;
      return MD_OK;
    default: return MD_ERR_BAD_ARG;
  }
}

int md_get_option(int key) {
  switch (key) {
    case MD_OPT_QUARTERS: return g_opt.quarters;
    case MD_OPT_ORDERS: return g_opt.orders;
    case MD_OPT_SLICE_BITS: return g_opt.bits;
    case MD_OPT_HOST_BLOCKS: return g_opt.host_blocks;
    case MD_OPT_K_CHUNK: return g_opt.k_chunk;
    case MD_OPT_FUSED_PREP: return g_opt.fused_prep;
    case MD_OPT_ONE_LAUNCH: return g_opt.one_launch;
    case MD_OPT_TILE_SCHEDULE: return g_opt.tile_schedule;
    case MD_OPT_TILE: return g_opt.tile;
    case MD_OPT_RASTER_GROUP: return g_opt.raster_group;
    default: return -1;
  }
}

md_status md_split(int rows, int cols, int limbs, int quarters, int axis, const double* planes, double* quarter_planes,
                   int32_t* exps, md_stream stream) {
  if (rows <= 0 || cols <= 0 || !planes || !quarter_planes || !exps) return MD_ERR_BAD_ARG;
  if (limbs != 1 && !limbs_ok(limbs)) return MD_ERR_BAD_ARG;
  if (quarters < 1 || quarters > MD_MAX_QUARTERS || (axis != 0 && axis != 1)) return MD_ERR_BAD_ARG;
  if (!aligned8(planes) || !aligned8(quarter_planes) || (reinterpret_cast<uintptr_t>(exps) & 3)) return MD_ERR_BAD_ARG;
  DeviceState* ds = device_state();
  uint32_t* flags = ds && ds->ws ? static_cast<uint32_t*>(ds->ws) : nullptr;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  uint64_t launches = 0;
  const int W = slice_bits();
  cudaError_t err = launch_exponents(rows, cols, axis, quarters, W, planes, exps, flags, st, &launches);
  if (err == cudaSuccess)
    err = launch_split(rows, cols, limbs, quarters, W, axis, planes, quarter_planes, exps, flags, st, &launches);
  g_launches += launches;
  return err == cudaSuccess ? MD_OK : MD_ERR_CUDA;
}

md_status md_qgemm(int m, int n, int k, int limbs, int quarters, int orders, const double* Aq, const double* Bq,
                   double* order_planes, double* C_planes, md_stream stream) {
  if (m <= 0 || n <= 0 || k <= 0 || !Aq || !Bq || (!order_planes && !C_planes)) return MD_ERR_BAD_ARG;
  if (!aligned8(Aq) || !aligned8(Bq) || !aligned8(order_planes) || !aligned8(C_planes)) return MD_ERR_BAD_ARG;
  if (!limbs_ok(limbs) || quarters < 1 || orders < 1) return MD_ERR_BAD_ARG;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  uint64_t launches = 0;
  cudaError_t err;
  if (orders == quarters && qgemm_supported(limbs, quarters)) {  // a tuned kernel on the plain quarter planes
    if (!k_budget_ok(k, orders, slice_bits())) return MD_ERR_K_TOO_LARGE;
    err = launch_qgemm(m, n, k, limbs, quarters, Aq, Bq, order_planes, C_planes, st, &launches);
  } else {
    // any other (limbs, quarters, orders): repack the planes into the registered workspace and run the kernel md_gemm would
    const KernelPick pick = pick_kernel(m, n, k, limbs, quarters, orders, slice_bits(), true, true);
    if (pick.family == GEMM_NONE) return MD_ERR_UNSUPPORTED;
    if (!k_budget_ok(k, orders, slice_bits())) return MD_ERR_K_TOO_LARGE;
    DeviceState* ds = device_state();
    if (!ds || !ds->ws) return MD_ERR_WORKSPACE;
    const Carve c = carve(ds->ws, m, n, k, quarters, orders, pick);
    if (c.total > ds->ws_bytes) return MD_ERR_WORKSPACE;
    err = launch_pack_planes(m, k, quarters, 0, pick.bxA, pick.bk, Aq, c.Aq, st, &launches);
    if (err == cudaSuccess) err = launch_pack_planes(k, n, quarters, 1, pick.bxB, pick.bk, Bq, c.Bq, st, &launches);
    if (err == cudaSuccess)
      err = launch_fused(m, n, k, limbs, quarters, orders, pick, c.Aq, c.Bq, order_planes, C_planes, c.sk, false, st, &launches);
  }
  g_launches += launches;
  return err == cudaSuccess ? MD_OK : MD_ERR_CUDA;
}

md_status md_renorm(int m, int n, int limbs, int orders, const double* order_planes, double* C_planes,
                    md_stream stream) {
  if (m <= 0 || n <= 0 || !order_planes || !C_planes) return MD_ERR_BAD_ARG;
  if (limbs != 1 && !limbs_ok(limbs)) return MD_ERR_BAD_ARG;
  if (orders < 1 || orders > 2 * MD_MAX_QUARTERS || !aligned8(order_planes) || !aligned8(C_planes)) return MD_ERR_BAD_ARG;
  uint64_t launches = 0;
  cudaError_t err = launch_renorm(m, n, limbs, orders, order_planes, C_planes, static_cast<cudaStream_t>(stream), &launches);
  g_launches += launches;
  return err == cudaSuccess ? MD_OK : MD_ERR_CUDA;
}

size_t md_workspace_bytes(int m, int n, int k, int limbs) {
  if (m <= 0 || n <= 0 || k <= 0 || !limbs_ok(limbs)) return 0;
  return workspace_bytes_for(m, n, k, limbs, quarters_for(limbs), orders_for(limbs));
}

md_status md_set_workspace(void* dev_ptr, size_t bytes) {
  if ((dev_ptr == nullptr) != (bytes == 0)) return MD_ERR_BAD_ARG;
  if (reinterpret_cast<uintptr_t>(dev_ptr) % WS_ALIGN) return MD_ERR_BAD_ARG;
  if (dev_ptr && bytes < WS_ALIGN) return MD_ERR_WORKSPACE;
  DeviceState* ds = device_state();
  if (!ds) return MD_ERR_CUDA;
  if (dev_ptr && cudaMemset(dev_ptr, 0, WS_ALIGN) != cudaSuccess) return MD_ERR_CUDA;  // clear the status word (synchronous: header)
  ds->ws = dev_ptr;
  ds->ws_bytes = bytes;
  ds->host_flags = 0;
  ds->host_flags_valid = false;
  return MD_OK;
}

md_status md_read_flags(uint32_t* flags_host, md_stream stream) {
  if (!flags_host) return MD_ERR_BAD_ARG;
  DeviceState* ds = device_state();
  if (!ds) return MD_ERR_CUDA;
  if (!ds->ws) {  // no workspace registered: what md_gemm_host / md_gemm_auto calls have recorded since the last md_set_workspace
    *flags_host = ds->host_flags;
    return ds->host_flags_valid ? MD_OK : MD_ERR_WORKSPACE;
  }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  uint32_t word = 0;
  if (cudaMemcpyAsync(&word, ds->ws, sizeof(uint32_t), cudaMemcpyDeviceToHost, st) != cudaSuccess) return MD_ERR_CUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return MD_ERR_CUDA;
  *flags_host = word | ds->host_flags;
  return MD_OK;
}

md_status md_gemm(int m, int n, int k, int limbs, const double* A_planes, const double* B_planes, double* C_planes,
                  md_stream stream) {
  const md_status st = check_gemm_args(m, n, k, limbs, A_planes, B_planes, C_planes, false);
  if (st != MD_OK) return st;
  DeviceState* ds = device_state();
  if (!ds) return MD_ERR_CUDA;
  return gemm_impl(m, n, k, limbs, quarters_for(limbs), orders_for(limbs), A_planes, B_planes, C_planes, nullptr, ds->ws,
                   ds->ws_bytes, static_cast<cudaStream_t>(stream), true);
}

md_status md_gemm_orders(int m, int n, int k, int limbs, const double* A_planes, const double* B_planes,
                         double* order_planes, md_stream stream) {
  const md_status st = check_gemm_args(m, n, k, limbs, A_planes, B_planes, order_planes, true);
  if (st != MD_OK) return st;
  DeviceState* ds = device_state();
  if (!ds) return MD_ERR_CUDA;
  return gemm_impl(m, n, k, limbs, quarters_for(limbs), orders_for(limbs), A_planes, B_planes, nullptr, order_planes, ds->ws,
                   ds->ws_bytes, static_cast<cudaStream_t>(stream), true);
}

md_status md_plan_slices(int k, int limbs, int* bits_out, int* quarters_out) {
  if (k <= 0 || !bits_out || !quarters_out) return MD_ERR_BAD_ARG;
  if (!limbs_ok(limbs)) return MD_ERR_BAD_ARG;
  // the fewest slices Q with a TUNED kernel, at the widest W the exactness budget allows for (k, Q), whose window W * Q covers
  // the paper's 13 * 4 * limbs bits; the paper's own (13, 4 * limbs) when nothing better qualifies
  for (int Q = 1; Q < 4 * limbs; Q++) {
    if (!(qgemm_supported(limbs, Q) || qgemm_wide_supported(limbs, Q))) continue;
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
  if (k <= 0 || min_chunk < PACK_BK || !bits_out || !quarters_out || !chunk_out) return MD_ERR_BAD_ARG;
  if (!limbs_ok(limbs)) return MD_ERR_BAD_ARG;
  // as md_plan_slices, but the budget only has to hold for a chunk of at least min_chunk contraction indices where a
  // chunked kernel exists: the fewest slices, then the widest width
  for (int Q = 1; Q < 4 * limbs; Q++) {
    const bool whole = qgemm_supported(limbs, Q) || qgemm_wide_supported(limbs, Q);
    const bool chunked = qgemm_chunk_supported(limbs, Q);
    if (!whole && !chunked) continue;
    for (int W = MD_MAX_BITS; W >= MD_MIN_BITS && W * Q >= 52 * limbs; W--) {
      if (whole && k_budget_ok(k, Q, W)) {
        *bits_out = W, *quarters_out = Q, *chunk_out = 0;
        return MD_OK;
      }
      const long long c = (1ll << (53 - 2 * W)) / Q / PACK_BK * PACK_BK;
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
  return WS_ALIGN + ws_round_up(sizeof(int32_t) * (size_t)m) + ws_round_up(sizeof(int32_t) * (size_t)n) +
         ws_round_up(sizeof(double) * (size_t)m * k) + ws_round_up(sizeof(double) * (size_t)k * n) +
         ws_round_up(sizeof(double) * (size_t)m * n);
}

md_status md_plan_quarters(int m, int n, int k, int limbs, const double* A_planes, const double* B_planes, void* scratch,
                           size_t scratch_bytes, double rel_tol, int* quarters_out, int* spread_out, md_stream stream) {
  if (m <= 0 || n <= 0 || k <= 0 || !A_planes || !B_planes || !scratch || !quarters_out) return MD_ERR_BAD_ARG;
  if (limbs != 1 && !limbs_ok(limbs)) return MD_ERR_BAD_ARG;
  if (!aligned8(A_planes) || !aligned8(B_planes) || reinterpret_cast<uintptr_t>(scratch) % WS_ALIGN) return MD_ERR_BAD_ARG;
  if (scratch_bytes < md_plan_scratch_bytes(m, n, k)) return MD_ERR_WORKSPACE;
  if (rel_tol == 0.0) rel_tol = format_tolerance(limbs);
  if (!(rel_tol > 0.0)) return MD_ERR_BAD_ARG;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int W = slice_bits();
  char* p = static_cast<char*>(scratch);
  int32_t* spread = reinterpret_cast<int32_t*>(p);
  int32_t* expA = reinterpret_cast<int32_t*>(p + WS_ALIGN);
  int32_t* expB = reinterpret_cast<int32_t*>(p + WS_ALIGN + ws_round_up(sizeof(int32_t) * (size_t)m));
  double* absA = reinterpret_cast<double*>(reinterpret_cast<char*>(expB) + ws_round_up(sizeof(int32_t) * (size_t)n));
  double* absB = reinterpret_cast<double*>(reinterpret_cast<char*>(absA) + ws_round_up(sizeof(double) * (size_t)m * k));
  double* Wt = reinterpret_cast<double*>(reinterpret_cast<char*>(absB) + ws_round_up(sizeof(double) * (size_t)k * n));
  const int32_t none = INT32_MIN;
  uint64_t launches = 0;
  cudaError_t err = cudaMemcpyAsync(spread, &none, sizeof(none), cudaMemcpyHostToDevice, st);
  // exponent vectors of the leading limb planes, |A_0| |B_0| on the DMMA kernel, then the spread D
  if (err == cudaSuccess) err = launch_exponents(m, k, 0, 4 * limbs, W, A_planes, expA, nullptr, st, &launches);
  if (err == cudaSuccess) err = launch_exponents(k, n, 1, 4 * limbs, W, B_planes, expB, nullptr, st, &launches);
  if (err == cudaSuccess) err = launch_abs((size_t)m * k, A_planes, absA, st, &launches);
  if (err == cudaSuccess) err = launch_abs((size_t)k * n, B_planes, absB, st, &launches);
  if (err == cudaSuccess) err = launch_plain_dgemm(m, n, k, absA, absB, Wt, st, &launches);
  if (err == cudaSuccess) err = launch_spread(m, n, Wt, expA, expB, spread, st, &launches);
  g_launches += launches;
  int32_t D = 0;
  if (err == cudaSuccess) err = cudaMemcpyAsync(&D, spread, sizeof(D), cudaMemcpyDeviceToHost, st);
  if (err != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess) return MD_ERR_CUDA;
  if (spread_out) *spread_out = D;
  // the smallest Q >= ceil(52 limbs / W) with k (Q+3) 2^(D - W Q - 2) <= rel_tol (R15; the left side is exact)
  int Q = (52 * limbs + W - 1) / W;
  if (D != INT32_MIN)
    while (Q < 4096 && ldexp((double)k * (Q + 3), D - W * Q - 2) > rel_tol) Q++;
  *quarters_out = Q;
  return MD_OK;
}

size_t md_auto_scratch_bytes(int m, int n, int k, int limbs, int quarters) {
  if (m <= 0 || n <= 0 || k <= 0 || !limbs_ok(limbs) || quarters < 0 || quarters > MD_MAX_QUARTERS) return 0;
  const int Q = quarters ? quarters : 4 * limbs;
  const size_t ws = workspace_bytes_for(m, n, k, limbs, Q, Q);
  if (!ws) return 0;
  const size_t plan = ws_round_up(md_plan_scratch_bytes(m, n, k));
  return ws > plan ? ws : plan;  // the plan's scratch is dead before the split starts: the two share the buffer
}

md_status md_gemm_auto(int m, int n, int k, int limbs, const double* A_planes, const double* B_planes, double* C_planes,
                       void* scratch, size_t scratch_bytes, double rel_tol, int* quarters_used, md_stream stream) {
  if (m <= 0 || n <= 0 || k <= 0 || !A_planes || !B_planes || !C_planes || !scratch) return MD_ERR_BAD_ARG;
  if (!aligned8(A_planes) || !aligned8(B_planes) || !aligned8(C_planes) || reinterpret_cast<uintptr_t>(scratch) % WS_ALIGN) return MD_ERR_BAD_ARG;
  if (!limbs_ok(limbs)) return MD_ERR_BAD_ARG;
  if (scratch_bytes < md_plan_scratch_bytes(m, n, k)) return MD_ERR_WORKSPACE;
  int Q = 0, D = 0;
  md_status st = md_plan_quarters(m, n, k, limbs, A_planes, B_planes, scratch, scratch_bytes, rel_tol, &Q, &D, stream);
  if (st != MD_OK) return st;
  const int W = slice_bits();
  if (quarters_used) *quarters_used = Q;
  if (pick_kernel(m, n, k, limbs, Q, Q, W, false, true).family == GEMM_NONE) return MD_ERR_UNSUPPORTED;
  if (!k_budget_ok(k, Q, W) && chunk_for(k, limbs, Q, Q, W) == 0) return MD_ERR_K_TOO_LARGE;
  if (workspace_bytes_for(m, n, k, limbs, Q, Q) > scratch_bytes) return MD_ERR_WORKSPACE;  // *quarters_used says what to size for
  cudaStream_t cs = static_cast<cudaStream_t>(stream);
  if (cudaMemsetAsync(scratch, 0, WS_ALIGN, cs) != cudaSuccess) return MD_ERR_CUDA;  // the status word of this call
  st = gemm_impl(m, n, k, limbs, Q, Q, A_planes, B_planes, C_planes, nullptr, scratch, scratch_bytes, cs, true);
  if (st != MD_OK) return st;
  // the status word of this call is kept for md_read_flags (the call has synchronised once already, for the plan)
  DeviceState* ds = device_state();
  uint32_t word = 0;
  if (!ds || cudaMemcpyAsync(&word, scratch, sizeof(word), cudaMemcpyDeviceToHost, cs) != cudaSuccess ||
      cudaStreamSynchronize(cs) != cudaSuccess)
    return MD_ERR_CUDA;
  ds->host_flags |= word;
  ds->host_flags_valid = true;
  return MD_OK;
}

size_t md_host_scratch_bytes(int m, int n, int k, int limbs) {
  if (m <= 0 || n <= 0 || k <= 0 || !limbs_ok(limbs)) return 0;
  const int Q = quarters_for(limbs), S = orders_for(limbs);
  const size_t ws = workspace_bytes_for(m, n, k, limbs, Q, S);
  if (!ws) return 0;
  return ws_round_up(sizeof(double) * (size_t)limbs * m * k) + ws_round_up(sizeof(double) * (size_t)limbs * k * n) +
         ws_round_up(sizeof(double) * (size_t)limbs * m * n) + ws;
}

md_status md_gemm_host(int m, int n, int k, int limbs, const double* A_host, const double* B_host, double* C_host,
                       void* dev_scratch, size_t scratch_bytes, md_stream stream) {
  const md_status chk = check_gemm_args(m, n, k, limbs, A_host, B_host, C_host, false);
  if (chk != MD_OK) return chk;
  if (!dev_scratch || reinterpret_cast<uintptr_t>(dev_scratch) % WS_ALIGN) return MD_ERR_BAD_ARG;
  if (scratch_bytes < md_host_scratch_bytes(m, n, k, limbs)) return MD_ERR_WORKSPACE;
  DeviceState* ds = device_state();
  if (!ds) return MD_ERR_CUDA;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int Q = quarters_for(limbs), S = orders_for(limbs), W = slice_bits();
  const size_t a_bytes = sizeof(double) * (size_t)limbs * m * k, b_bytes = sizeof(double) * (size_t)limbs * k * n,
               c_bytes = sizeof(double) * (size_t)limbs * m * n;
  char* p = static_cast<char*>(dev_scratch);
  double* dA = reinterpret_cast<double*>(p);
  double* dB = reinterpret_cast<double*>(p + ws_round_up(a_bytes));
  double* dC = reinterpret_cast<double*>(p + ws_round_up(a_bytes) + ws_round_up(b_bytes));
  char* ws = p + ws_round_up(a_bytes) + ws_round_up(b_bytes) + ws_round_up(c_bytes);
  // the multi-panel path keeps the large tiles its panels are cut to
  const KernelPick pick = pick_kernel(m, n, k, limbs, Q, S, W, false, false);
  const Carve c = carve(ws, m, n, k, Q, S, pick);
  uint32_t flags_word = 0;
  // the status word of this call travels back with the result: md_read_flags reports it (ORed into the device's record)
  auto finish = [&](md_status result) -> md_status {
    const bool copied = cudaMemcpyAsync(&flags_word, ws, sizeof(uint32_t), cudaMemcpyDeviceToHost, st) == cudaSuccess;
    const bool synced = cudaStreamSynchronize(st) == cudaSuccess;
    if (copied && synced) ds->host_flags |= flags_word, ds->host_flags_valid = true;
    return synced ? result : MD_ERR_CUDA;
  };

  // Panels: C is cut into PR x PC blocks (rows of A x columns of B).  A row's exponent and quarters depend on that row of A
  // only, a column's on that column of B only, so every block is an independent md_gemm on COMPACT
  // device copies of its operands: panel i of A is [limbs][mi][k] at dA + limbs * row0 * k, panel j of B is [limbs][k][nj]
  // at dB + limbs * k * col0, block (i, j) of C is [limbs][mi][nj].  Three streams: copies in (in order of first use),
  // the kernels (the caller's stream), copies out; the first kernel starts after A_0 and B_0 have arrived and the last
  // copy out is one block of C, instead of the whole of A, B before and the whole of C after.
  const HostPanels hp = plan_host_panels(m, n, pick.bxA, pick.bxB);
  if (hp.PR == 1 && hp.PC == 1) {  // one block: nothing to overlap -- copy in, the device path as md_gemm runs it, copy out
    if (cudaMemsetAsync(ws, 0, WS_ALIGN, st) != cudaSuccess) return MD_ERR_CUDA;
    if (cudaMemcpyAsync(dA, A_host, a_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return finish(MD_ERR_CUDA);
    if (cudaMemcpyAsync(dB, B_host, b_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return finish(MD_ERR_CUDA);
    const md_status run = gemm_impl(m, n, k, limbs, Q, S, dA, dB, dC, nullptr, ws, scratch_bytes - (size_t)(ws - p), st, true);
    if (run != MD_OK) return finish(run);
    if (cudaMemcpyAsync(C_host, dC, c_bytes, cudaMemcpyDeviceToHost, st) != cudaSuccess) return finish(MD_ERR_CUDA);
    return finish(MD_OK);
  }
  if (!host_pipeline_ready(ds, hp.PR + hp.PC + hp.PR * hp.PC + 2)) return MD_ERR_CUDA;
  cudaStream_t s_in = ds->host_in, s_out = ds->host_out;
  cudaEvent_t* ev = ds->host_ev.data();
  cudaEvent_t ev_start = ev[0], ev_done = ev[1];
  cudaEvent_t* ev_A = ev + 2;
  cudaEvent_t* ev_B = ev_A + hp.PR;
  cudaEvent_t* ev_C = ev_B + hp.PC;
  // on any failure: nothing the library enqueued on its own streams may still be in flight when the call returns
  auto fail = [&]() -> md_status {
    cudaStreamSynchronize(s_in);
    cudaStreamSynchronize(s_out);
    cudaStreamSynchronize(st);
    return MD_ERR_CUDA;
  };
#define MD_TRY(call) \
  if ((call) != cudaSuccess) return fail()
  MD_TRY(cudaMemsetAsync(ws, 0, WS_ALIGN, st));  // the status word
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

  const int bxA = pick.bxA, bxB = pick.bxB, bk = pick.bk;
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
    err = launch_exponents(k, nj, 1, Q, W, Bj, c.expB + c0, c.flags, st, &launches);
    if (err == cudaSuccess) err = launch_split_packed(k, nj, limbs, Q, W, 1, bxB, bk, Bj, Bq, c.expB + c0, c.flags, st, &launches);
    for (int i = 0; i < hp.PR && err == cudaSuccess; i++) {
      int r0, mi;
      rows_of(i, r0, mi);
      const double* Ai = dA + (size_t)limbs * r0 * k;
      double* Aq = c.Aq + (size_t)(r0 / bxA) * KS * chunkA;
      if (j == 0) {
        MD_TRY(cudaStreamWaitEvent(st, ev_A[i], 0));
        err = launch_exponents(mi, k, 0, Q, W, Ai, c.expA + r0, c.flags, st, &launches);
        if (err == cudaSuccess) err = launch_split_packed(mi, k, limbs, Q, W, 0, bxA, bk, Ai, Aq, c.expA + r0, c.flags, st, &launches);
        if (err != cudaSuccess) break;
      }
      // block (i, j): compact [limbs][mi][nj] at the position its elements have in a row-panel-major walk of C
      double* Cb = dC + (size_t)limbs * ((size_t)r0 * n + (size_t)mi * c0);
      err = launch_fused(mi, nj, k, limbs, Q, S, pick, Aq, Bq, nullptr, Cb, c.sk, false, st, &launches);
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
  if (err != cudaSuccess) return fail();
  // join: the caller's stream waits for the last copy out
  MD_TRY(cudaEventRecord(ev_done, s_out));
  MD_TRY(cudaStreamWaitEvent(st, ev_done, 0));
#undef MD_TRY
  return finish(MD_OK);
}

md_status md_profile_enable(int capacity) {
  if (capacity < 0 || capacity > (1 << 20)) return MD_ERR_BAD_ARG;
  DeviceState* ds = device_state();
  if (!ds) return MD_ERR_CUDA;
  for (cudaEvent_t e : ds->prof_ev) cudaEventDestroy(e);
  ds->prof_ev.clear();
  ds->prof_capacity = ds->prof_count = 0;
  ds->prof_ev.resize(3 * (size_t)capacity);
  for (size_t i = 0; i < ds->prof_ev.size(); i++)
    if (cudaEventCreate(&ds->prof_ev[i]) != cudaSuccess) {
      for (size_t j = 0; j < i; j++) cudaEventDestroy(ds->prof_ev[j]);
      ds->prof_ev.clear();
      return MD_ERR_CUDA;
    }
  ds->prof_capacity = capacity;
  return MD_OK;
}

int md_profile_read(float* split_ms_host, float* gemm_ms_host, int capacity) {
  DeviceState* ds = device_state();
  if (!ds) return MD_ERR_CUDA;
  if (capacity < ds->prof_count) return MD_ERR_BAD_ARG;
  for (int i = 0; i < ds->prof_count; i++) {
    cudaEvent_t* ev = &ds->prof_ev[3 * (size_t)i];
    float a = 0.f, b = 0.f;
    if (cudaEventSynchronize(ev[2]) != cudaSuccess) return MD_ERR_CUDA;
    if (cudaEventElapsedTime(&a, ev[0], ev[1]) != cudaSuccess) return MD_ERR_CUDA;
    if (cudaEventElapsedTime(&b, ev[1], ev[2]) != cudaSuccess) return MD_ERR_CUDA;
    if (split_ms_host) split_ms_host[i] = a;
    if (gemm_ms_host) gemm_ms_host[i] = b;
  }
  return ds->prof_count;
}

md_status md_probe_dmma(int blocks, int warps_per_block, int iters, double* sink, uint64_t* flops_host, md_stream stream) {
  if (blocks < 1 || warps_per_block < 1 || warps_per_block > 32 || iters < 1 || iters >= (1 << 25) || !flops_host)
    return MD_ERR_BAD_ARG;
  if (!aligned8(sink)) return MD_ERR_BAD_ARG;
  uint64_t launches = 0;
  cudaError_t err = launch_dmma_probe(blocks, warps_per_block, iters, sink, static_cast<cudaStream_t>(stream),
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
    case MD_ERR_STATIC_LIMIT: return "MD_ERR_STATIC_LIMIT: the problem needs more than the 64 MiB built-in scratch of md_gemm_static (md_gemm_static_bytes > md_static_scratch_bytes); use md_gemm with a workspace";
    default: return "unknown md_status";
  }
}

}  // extern "C"
