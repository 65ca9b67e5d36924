// qgemm_pipeline.cuh -- what the two persistent fused quarter-GEMM kernels (qgemm_packed.cu: double / quad double;
// qgemm_wide.cu: octo / hexa double) share: mbarrier and bulk-copy wrappers, and the stream-K work plan.
// CUDA path only; nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace md {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// mbarrier / bulk-copy wrappers; barriers and shared destinations are passed as 32-bit shared-window addresses that the
// kernel computes once (a generic->shared conversion inside the k loop costs an S2R + LEA chain per slab).
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}" ::"r"(bar), "r"(parity)
      : "memory");
}
// global -> shared bulk copy (bytes % 16 == 0, both addresses 16-byte aligned); completion = complete_tx on `bar`.
__device__ __forceinline__ void bulk_g2s(uint32_t smem_dst, const void* gmem_src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_dst),
               "l"(gmem_src), "r"(bytes), "r"(bar)
               : "memory");
}

// Programmatic dependent launch (sm_90+): a kernel launched with cudaLaunchAttributeProgrammaticStreamSerialization may start
// while its predecessor on the stream still runs -- once every block of the predecessor has executed launch_dependents (or exited)
// -- and must execute grid_dependency_wait before it touches anything the predecessor wrote.  Both are no-ops in a plain launch.
__device__ __forceinline__ void grid_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void grid_dependency_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// Persistent kernel: gridDim.x = G CTAs (one per SM), each walks a private list of SEGMENTS = (tile, slab range):
//   * dp_waves whole tiles, ids b, b + G, b + 2G, ... (tile ids are rasterised, so at any time the G CTAs cover a compact patch
//     of C), accumulated and renormalised entirely in registers;
//   * the stream-K part: the sk_tiles tiles that do not fill a whole wave of G CTAs are cut along k into G nearly equal runs of
//     slabs (CTA b owns global slab iterations [b*ipc, (b+1)*ipc) of the sk_tiles * KS), so that the last wave costs
//     sk_tiles*KS/G slab-times instead of KS.  The partial order sums of the CTAs that share a tile are combined EXACTLY --
//     every partial sum is an integer below 2^53 units (R6), so the result is bit-identical whatever the order --
//     either by fp64 red.global.add into the tile's scratch (whoever completes the slab count runs the epilogue; nobody waits)
//     or by a hand-over through per-CTA slots and flags (qgemm_packed.cu says which and why).
// The stage ring runs straight through segment boundaries: the refill thread is AHEAD slabs ahead, possibly already in the
// next tile, so the pipeline never drains between tiles.
struct SkPlan {
  int KS;                // k slabs per tile
  int tiles_m, tiles_n;
  int dp_waves;          // whole tiles per CTA
  int sk_tiles;          // tiles dp_waves*G .. dp_waves*G + sk_tiles - 1 are processed stream-K
  int sk_iters_per_cta;  // ipc
  int dp_tail;           // CTAs 0 .. dp_tail-1 own a tile in the LAST of the dp_waves (all G of them unless chunked, below)
  int flush_slabs;       // chunked accumulation (qgemm_packed.cu, R16): slabs between two flushes; 0 = never
  int group_m;           // tile rows per raster group (raster_tile; MD_OPT_RASTER_GROUP, default 8)
  // DYNAMIC schedule (qgemm_packed.cu, MODE 2): CTAs claim work items from a queue counter in item order --
  // items [0, dyn_whole) are whole tiles (tile id = item), the others cut the remaining tiles along k into units of dyn_unit slabs
  int dyn_whole;         // whole-tile items
  int dyn_unit;          // slabs per unit of a cut tile
  int dyn_upt;           // units per cut tile = ceil(KS / dyn_unit)
  int dyn_items;         // all items
  int dyn_static;        // the first dyn_static whole tiles of CTA b are b, b + G, ... without a claim; the queue starts at item dyn_static * G
};

// Plan for `tiles` output tiles of KS slabs each on a grid of G persistent CTAs.
int raster_group();  // api.cu: MD_OPT_RASTER_GROUP (default 8)
int tile_schedule();  // api.cu: MD_OPT_TILE_SCHEDULE (0 = automatic, 1 = hybrid, 2 = tile queue only, 3 = static lists)
inline SkPlan make_sk_plan(int tiles_m, int tiles_n, int KS, int G) {
  const long long tiles = (long long)tiles_m * tiles_n;
  SkPlan plan;
  plan.KS = KS;
  plan.tiles_m = tiles_m;
  plan.tiles_n = tiles_n;
  plan.dp_waves = (int)(tiles / G);
  plan.sk_tiles = (int)(tiles % G);
  plan.sk_iters_per_cta = (int)(((long long)plan.sk_tiles * KS + G - 1) / G);
  plan.dp_tail = G;
  plan.flush_slabs = 0;
  plan.group_m = raster_group();
  plan.dyn_whole = plan.dyn_unit = plan.dyn_upt = plan.dyn_items = plan.dyn_static = 0;
  return plan;
}

}  // namespace md
