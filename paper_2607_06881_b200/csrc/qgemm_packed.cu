// qgemm_packed.cu -- steps a3 + a4 of the hot path, the kernel behind md_gemm / md_gemm_orders.
//
//   For s = 0..S-1:  C^(s) = sum_{p+q=s} A_p * B_q      (PAPER.md:66-71 eq. 3; :75-78 eq. 4: the paper's C_{s+1})
//   C = sum_s C^(s), summed error free into L limbs     (PAPER.md:88-91 steps 4-5)
//
// Same arithmetic as qgemm.cu (all T = S(S+1)/2 quarter products of a tile issued on DMMA.8x8x4 from one staging of the
// Q quarter tiles, one register accumulator set per order, renormalising epilogue), but fed from the FRAGMENT-MAJOR
// PACKED quarter planes the splitter writes for md_gemm (md_packed.cuh):
//   * everything a CTA needs for one k-slab of its A block (all Q quarters) is ONE contiguous chunk of global memory, and
//     so is its B block: a slab is staged with two cp.async.bulk copies (SASS UBLKCP) issued by one thread, completing
//     on an mbarrier -- no per-thread address arithmetic, no LDGSTS, no register traffic in the DMMA stream;
//   * inside a chunk every 8x4 (A) / 4x8 (B) DMMA operand fragment is 32 consecutive doubles in lane order, so a
//     fragment load is one conflict-free LDS.64 at base + 8*lane with an immediate offset, no padding;
//   * stages are handed back through per-stage "empty" mbarriers (one arrive per warp) instead of a block-wide
//     __syncthreads, so the two warps of an SM sub-partition drift apart and one's LDS / barrier latency hides behind
//     the other's DMMA stream.  The refill of a stage is issued two slabs after its last read, when its empty barrier
//     has long completed, so the issuing thread never actually waits.
// The first ncu capture of the cp.async kernel of qgemm.cu (round 1) showed exactly these three costs as the gap
// between 88 % and the DMMA peak.
//
// Exactness (eq. 5; R6): quarters are integers |D| <= 2^13 times the group unit and
// k*S <= 2^27, so every partial sum is an integer below 2^53 units: each FMA inside DMMA is exact and the result does not
// depend on the order in which warps, slabs or the hardware add things.  Zero padding is harmless.
#include "md_kernels.h"
#include "md_packed.cuh"
#include "qgemm_common.cuh"
#include "qgemm_pipeline.cuh"

namespace md {
namespace {

// A warp owns an (8*MT) x (8*NT) block of C and S accumulator sets for it (S = Q, the paper's C_1..C_Q, unless MD_OPT_ORDERS
// asks for a pruned or extended order set); WM x WN warps tile the CTA block.
template <int Q_, int L_, int WM_, int WN_, int MT_, int NT_, int S_ = Q_>
struct PCfg {
  static constexpr int Q = Q_, S = S_, L = L_, WM = WM_, WN = WN_, MT = MT_, NT = NT_;
  static constexpr int BM = WM * MT * 8, BN = WN * NT * 8, BK = PACK_BK;
  static constexpr int WARPS = WM * WN, THREADS = WARPS * 32;
  static constexpr int K4 = BK / 4, R8 = BM / 8, N8 = BN / 8;
  static constexpr int A_CHUNK = Q * BK * BM, B_CHUNK = Q * BK * BN;  // doubles per k-slab
  static constexpr int STAGE_BYTES = (A_CHUNK + B_CHUNK) * 8;
  static constexpr int BAR_BYTES = 128;
  static constexpr int STAGES = ((SMEM_LIMIT - BAR_BYTES) / STAGE_BYTES) < 6 ? ((SMEM_LIMIT - BAR_BYTES) / STAGE_BYTES) : 6;
  static constexpr int AHEAD = STAGES - 2;  // slabs in flight beyond the one being consumed
  // second register set of operand fragments (software pipelining across k-steps and slabs) where 255 registers allow
  static constexpr bool PREFETCH = (S * MT * NT * 4 + 2 * (Q * MT + NT) * 2) <= 200;
  static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + BAR_BYTES;
  static_assert(STAGES >= 3, "the non-blocking refill needs at least 3 stages");
  static_assert(2 * STAGES * 8 <= BAR_BYTES - 8, "barrier area (its last 8 bytes hold the stream-K flag)");
  static_assert(STAGE_BYTES % 128 == 0, "stage alignment");
};

// CHUNK (R16): the exactness budget k S 2^(2W) <= 2^53 is kept PER CHUNK of plan.flush_slabs slabs instead of
// for the whole contraction.  Chunks are the slab ranges [c * flush_slabs, (c+1) * flush_slabs) of a tile.  Whole tile: at
// the end of a chunk every order accumulator (still an exact sum) is added into the element's (L+1)-term expansion by
// the TwoSum cascade of the recombination (renorm_add) and cleared; the expansion carries over the chunks and the
// epilogue only finishes it.  Stream-K part of a tile: the sums of each chunk are added into THAT CHUNK's slot of the
// tile's scratch (exact, like the unchunked stream-K: the total of a chunk is within the budget whoever contributes), and
// the CTA that completes the slab count runs the same renorm_add sequence over the chunks' totals -- so the result is
// bit-identical to a whole-tile run whatever the split.  No order planes (the order sums of the whole k are not doubles).
// HANDOVER: how the CTAs that share a stream-K tile combine their partial order sums (both exact, R6, hence the same
// bits): false -- fp64 red.global.add into the tile's zeroed scratch, whoever completes the slab count re-reads the totals and
// runs the epilogue, nobody waits (large problems: the stream-K tail is one wave in dozens); true -- per-CTA slots and flags, the
// CTA that owns a tile's last slabs collects the others' sums (small problems, where every tile is cut and 16 KB of atomics per
// warp through L2 were the critical path: 256^3 0.55 -> 0.66, 512^3 0.88 -> 0.92 of the peak).  Two instantiations rather than
// one: at 254 registers the DMMA loop's schedule is sensitive to the code around it.
// MODE: SCHED_STATIC (0) the static segment lists above with the red.add hand-in; SCHED_HANDOVER (1) static lists, hand-over;
// SCHED_DYNAMIC (2) -- the segments are CLAIMED from a queue counter in global memory instead of computed from the CTA index:
// first every whole tile in raster order, then the remaining tiles (the last partial wave plus, when that is short, one more
// wave) cut along k into units of plan.dyn_unit slabs, red.add hand-in.  An SM that runs ahead simply claims more, and the run
// ends within one unit's time on every SM (under the static lists the SMs of the quad-double run finish up to 1.3 % apart).
// An OPTION, not the default: launch_cfg says what it costs.
// Thread 0 claims one item ahead of the segment it is producing and publishes the descriptors through a ring in shared
// memory; a descriptor is written before the bulk copies of the PRECEDING segment's first slab are issued, so any warp that
// has passed that slab's full barrier (release / acquire through the mbarrier) may read it -- no extra synchronisation in the loop.
constexpr int SCHED_STATIC = 0, SCHED_HANDOVER = 1, SCHED_DYNAMIC = 2;
constexpr int DYN_RING = 8;  // > STAGES + 1: a descriptor is not overwritten while a warp may still read it
template <class C, bool CHUNK, int MODE = SCHED_STATIC>
__global__ void __launch_bounds__(C::THREADS, 1)
qgemm_packed_kernel(int m, int n, SkPlan plan, const double* __restrict__ Ap, const double* __restrict__ Bp,
                    double* __restrict__ order_planes, double* __restrict__ C_planes, double* __restrict__ sk_scratch,
                    unsigned int* __restrict__ sk_counters) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr int Q = C::Q, S = C::S, L = C::L, MT = C::MT, NT = C::NT, STAGES = C::STAGES;
  double* const stages = reinterpret_cast<double*>(smem_raw);
  uint64_t* const full = reinterpret_cast<uint64_t*>(smem_raw + STAGES * C::STAGE_BYTES);
  uint64_t* const empty = full + STAGES;
  volatile int* const last_flag = reinterpret_cast<volatile int*>(smem_raw + STAGES * C::STAGE_BYTES + C::BAR_BYTES - 8);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp / C::WN, wn = warp % C::WN;
  const int G = gridDim.x, cta = blockIdx.x, KS = plan.KS;
  constexpr bool HANDOVER = MODE == SCHED_HANDOVER, DYN = MODE == SCHED_DYNAMIC;
  static_assert(!(CHUNK && MODE != SCHED_STATIC), "the chunked kernel keeps the static lists");
  static_assert(DYN_RING > STAGES + 1, "descriptor ring");

  // ---- this CTA's segment list ---------------------------------------------------------------------------------------
  const int sk_total = plan.sk_tiles * KS;
  const int g0 = min(cta * plan.sk_iters_per_cta, sk_total), g1 = min(g0 + plan.sk_iters_per_cta, sk_total);
  const int n_sk = g1 > g0 ? (g1 - 1) / KS - g0 / KS + 1 : 0;
  const int dp_mine = plan.dp_waves - (cta >= plan.dp_tail ? 1 : 0);  // whole tiles of this CTA
  const int n_seg = n_sk + dp_mine;
  const int total_slabs = DYN ? 1 : (g1 - g0) + dp_mine * KS;
  const int sk_base = DYN ? plan.dyn_whole : plan.dp_waves * G;  // first tile that is cut along k
  // Segment list.  Without hand-over: the stream-K segments in slab order, then the whole tiles.
  // With hand-over: a CTA's share of stream-K slabs is at most one tile long (sk_tiles < G), so it has at most TWO stream-K
  // segments -- in slab order the TAIL of a tile begun by the CTAs before it (it ends at the tile's last slab) and / or the HEAD
  // (or a middle part) of a tile that a later CTA finishes.  Thread 0 writes them to shared memory in PROCESSING order: head,
  // whole tiles, tail.  A tile that is cut along k is FINISHED by the CTA that owns its last slabs; every other contributor
  // stores its partial sums to its own scratch slot and raises a flag.  Running the head first and the tail last means (1) the
  // partial sums a tail needs were written long before it asks for them -- the flag wait rarely spins -- and (2) a CTA only ever
  // waits for CTAs of LOWER index, none of which waits before raising its own flag: no deadlock even if the grid were not fully
  // resident.
  __shared__ int sk_tab[8];  // HANDOVER: [0..2], [3..5] = tile, s0, s1 of the stream-K segments in processing order; [6] = 1 if the first is a head
  if constexpr (HANDOVER) {
    if (tid == 0) {
      int seg[2][3] = {{0, 0, 0}, {0, 0, 0}};
      for (int i = 0; i < n_sk && i < 2; i++) {
        const int r = g0 / KS + i;
        seg[i][0] = plan.dp_waves * G + r;
        seg[i][1] = i == 0 ? g0 - r * KS : 0;
        seg[i][2] = min(KS, g1 - r * KS);
      }
      const bool swap = n_sk == 2;  // the head is the last one in slab order
#pragma unroll
      for (int e = 0; e < 3; e++) sk_tab[e] = seg[swap ? 1 : 0][e], sk_tab[3 + e] = seg[swap ? 0 : 1][e];
      sk_tab[6] = (n_sk > 0 && sk_tab[2] < KS) ? 1 : 0;
    }
  }
  __shared__ int dyn_tab[DYN ? DYN_RING : 1][4];  // DYNAMIC: descriptor of segment j at [j % DYN_RING] = tile (-1: no more work), s0, s1
  auto dyn_claim = [&](int j) {  // thread 0: claim the next item of the queue and publish it as segment j
    // the first dyn_static segments of a CTA are the whole tiles cta, cta + G, ... (no claim): the CTAs stay in lock-step on
    // neighbouring tiles and share operand slabs through L2 for most of the run; only what follows is claimed from the queue
    const int x = j < plan.dyn_static ? j * G + cta : plan.dyn_static * G + (int)atomicAdd(&sk_counters[SK_QUEUE_INDEX], 1u);
    int tile = -1, s0 = 0, s1 = 0;
    if (x < plan.dyn_whole) {
      tile = x, s1 = KS;
    } else if (x < plan.dyn_items) {
      // unit `part` of EVERY cut tile before unit part + 1 of any: the CTAs that run at the same time then work on the same
      // k-range of neighbouring tiles and share their operand slabs through L2, as in the whole-tile phase (with the 16 units
      // of one tile claimed together nothing was shared and the tail ran at DRAM speed: dd 4096^3 137.5 against 134.4 ms)
      const int cut = plan.dyn_items - plan.dyn_whole, u = x - plan.dyn_whole;
      const int cut_tiles = cut / plan.dyn_upt, part = u / cut_tiles;
      tile = plan.dyn_whole + (u - part * cut_tiles);
      s0 = part * plan.dyn_unit;
      s1 = min(KS, s0 + plan.dyn_unit);
    }
    volatile int* d = dyn_tab[j % DYN_RING];
    d[0] = tile, d[1] = s0, d[2] = s1;
  };
  auto segment = [&](int i, int& tile, int& s0, int& s1) {
    if constexpr (DYN) {
      const volatile int* d = dyn_tab[i % DYN_RING];
      tile = d[0], s0 = d[1], s1 = d[2];
    } else if constexpr (HANDOVER) {
      const int pre = sk_tab[6];  // the whole tiles come after the head
      if (i >= pre && i < pre + dp_mine) {
        tile = (i - pre) * G + cta, s0 = 0, s1 = KS;
        return;
      }
      if (i >= pre) i -= dp_mine;
      tile = sk_tab[3 * i], s0 = sk_tab[3 * i + 1], s1 = sk_tab[3 * i + 2];
    } else {
      if (i < n_sk) {
        const int r = g0 / KS + i;
        tile = plan.dp_waves * G + r;
        s0 = i == 0 ? g0 - r * KS : 0;
        s1 = min(KS, g1 - r * KS);
      } else {
        tile = (i - n_sk) * G + cta;
        s0 = 0;
        s1 = KS;
      }
    }
  };

  const uint32_t stages_u32 = smem_u32(stages);
  const uint32_t full_u32 = smem_u32(full), empty_u32 = smem_u32(empty);  // barrier s at + 8 * s
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < STAGES; s++) {
      mbar_init(full_u32 + 8 * s, 1);
      mbar_init(empty_u32 + 8 * s, C::WARPS);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    if constexpr (DYN) dyn_claim(0);
  }
  __syncthreads();
  grid_dependency_wait();  // (programmatic dependent launch behind the preparation kernel: nothing it wrote has been touched so far)
  if (total_slabs == 0) return;
  if constexpr (DYN) {
    if (dyn_tab[0][0] < 0) return;  // the queue was empty before this CTA's first claim
  }

  // ---- producer side (thread 0): a cursor over the flat slab sequence, AHEAD slabs ahead of the consumers -------------
  int p_seg = -1, p_left = 0, p_flat = 0, pst = 0;
  bool p_done = false;  // DYNAMIC: the producer has met the end of the queue
  const double *p_A = nullptr, *p_B = nullptr;
  auto produce_one = [&]() {  // issue the bulk copies of flat slab p_flat into stage pst (its empty barrier has completed)
    if (p_left == 0) {
      int tile, s0, s1, tm, tn;
      segment(++p_seg, tile, s0, s1);
      if constexpr (DYN) {
        if (tile < 0) {
          p_done = true;
          return;
        }
        dyn_claim(p_seg + 1);  // published before this segment's first slab is issued
      }
      raster_tile(tile, plan.tiles_m, plan.tiles_n, tm, tn, plan.group_m);
      p_A = Ap + ((size_t)tm * KS + s0) * C::A_CHUNK;
      p_B = Bp + ((size_t)tn * KS + s0) * C::B_CHUNK;
      p_left = s1 - s0;
    }
    const uint32_t dst = stages_u32 + pst * C::STAGE_BYTES, bar = full_u32 + 8 * pst;
    mbar_expect_tx(bar, C::STAGE_BYTES);
    bulk_g2s(dst, p_A, C::A_CHUNK * 8, bar);
    bulk_g2s(dst + C::A_CHUNK * 8, p_B, C::B_CHUNK * 8, bar);
    p_A += C::A_CHUNK;
    p_B += C::B_CHUNK;
    p_left--;
    p_flat++;
    pst = (pst + 1 == STAGES) ? 0 : pst + 1;
  };
  if (tid == 0) {
#pragma unroll
    for (int j = 0; j < C::AHEAD; j++)
      if (DYN ? !p_done : p_flat < total_slabs) produce_one();
  }
  auto produce = [&]() {  // top of consumer iteration `it`: refill for flat slab it + AHEAD
    if (DYN ? !p_done : p_flat < total_slabs) {
      // the stage was last read for flat slab (p_flat - STAGES) = it - 2: wait for its release (completed long ago)
      if (p_flat >= STAGES) mbar_wait(empty_u32 + 8 * pst, ((p_flat / STAGES) + 1) & 1);
      produce_one();
    }
  };

  double acc[S][MT][NT][2];
  auto zero_acc = [&]() {
#pragma unroll
    for (int s = 0; s < S; s++)
#pragma unroll
      for (int i = 0; i < MT; i++)
#pragma unroll
        for (int j = 0; j < NT; j++) acc[s][i][j][0] = acc[s][i][j][1] = 0.0;
  };
  zero_acc();
  // CHUNK: the running (L+1)-term expansion of every element this thread owns
  double rexp[CHUNK ? MT : 1][CHUNK ? NT : 1][2][L + 1];
  auto zero_rexp = [&]() {
#pragma unroll
    for (int i = 0; i < (CHUNK ? MT : 1); i++)
#pragma unroll
      for (int j = 0; j < (CHUNK ? NT : 1); j++)
#pragma unroll
        for (int e = 0; e < 2; e++)
#pragma unroll
          for (int l = 0; l <= L; l++) rexp[i][j][e][l] = 0.0;
  };
  auto flush_chunk = [&]() {  // orders from the smallest to the largest, as in renorm_orders (R9)
    if constexpr (CHUNK) {
      // order by order across ALL elements of the thread (each element still receives its orders from the smallest to the largest):
      // the TwoSum cascade of one element is a chain of dependent additions, 2 * MT * NT independent chains side by side hide it
#pragma unroll
      for (int s = S - 1; s >= 0; s--)
#pragma unroll
        for (int i = 0; i < MT; i++)
#pragma unroll
          for (int j = 0; j < NT; j++)
#pragma unroll
            for (int e = 0; e < 2; e++) renorm_add<L>(rexp[i][j][e], acc[s][i][j][e]);
      zero_acc();
    }
  };
  // CHUNK, stream-K: chunk c of stream-K tile r has its own S * BM * BN slot in the scratch
  auto chunk_slot = [&](int r, int c) -> double* {
    const int nchunks = (KS + plan.flush_slabs - 1) / plan.flush_slabs;
    return sk_scratch + ((size_t)r * nchunks + c) * (S * C::BM * C::BN) + (size_t)warp * (S * MT * NT * 64) + lane * 2;
  };
  auto flush_partial = [&](int r, int c) {  // exact fp64 red.add of this run's share of chunk c, then clear
    if constexpr (CHUNK) {
      double* sc = chunk_slot(r, c);
#pragma unroll
      for (int s = 0; s < S; s++)
#pragma unroll
        for (int i = 0; i < MT; i++)
#pragma unroll
          for (int j = 0; j < NT; j++) {
            atomicAdd(sc + ((s * MT + i) * NT + j) * 64, acc[s][i][j][0]);
            atomicAdd(sc + ((s * MT + i) * NT + j) * 64 + 1, acc[s][i][j][1]);
          }
      zero_acc();
    }
  };
  if constexpr (CHUNK) zero_rexp();
  int c_chunk = 0, to_flush = 0;  // CHUNK: the chunk the slab being consumed belongs to; slabs left in that chunk

  // Operand fragments of one DMMA k-step held in registers: all Q quarters of the warp's MT row blocks of A, and the
  // quarter-0 fragments of its NT column blocks of B (the B fragments of quarters 1.. are loaded inside the step).
  // Two sets: while the DMMAs of one k-step issue, the next step's set is already being loaded -- across the slab
  // boundary too, so no LDS latency is exposed at the hand-over between stages.
  struct Frags {
    double a[Q][MT];
    double b0[NT];
  };
  auto load_frags = [&](Frags& f, const double* As, const double* Bs, int k4) {
#pragma unroll
    for (int p = 0; p < Q; p++)
#pragma unroll
      for (int i = 0; i < MT; i++) f.a[p][i] = As[((p * C::K4 + k4) * C::R8 + i) * 32];
#pragma unroll
    for (int j = 0; j < NT; j++) f.b0[j] = Bs[(k4 * C::N8 + j) * 32];
  };
  auto k_step = [&](const Frags& f, const double* Bs, int k4) {
#pragma unroll
    for (int q = 0; q < Q; q++) {
      double b[NT];
#pragma unroll
      for (int j = 0; j < NT; j++) b[j] = q == 0 ? f.b0[j] : Bs[((q * C::K4 + k4) * C::N8 + j) * 32];
#pragma unroll
      for (int p = 0; p + q < S && p < Q; p++)  // product (p, q) goes to order s = p + q: consecutive DMMAs hit different accumulators
#pragma unroll
        for (int i = 0; i < MT; i++)
#pragma unroll
          for (int j = 0; j < NT; j++) dmma_8x8x4(acc[p + q][i][j], f.a[p][i], b[j]);
    }
  };
  static_assert(C::K4 == 2, "the k loop below is written for two DMMA k-steps per slab");
  const int a_off = (wm * MT) * 32 + lane, b_off = C::A_CHUNK + (wn * NT) * 32 + lane;

  // ---- consumer side: segment bookkeeping and the end-of-segment epilogue ----------------------------------------------
  int c_seg = 0, c_tile, c_s0, c_s1;
  segment(0, c_tile, c_s0, c_s1);
  int c_left = c_s1 - c_s0;
  // slabs this CTA is known to consume.  DYNAMIC (two fragment sets): the segments up to the one AFTER the current one -- its
  // descriptor is readable once the current segment's first slab has arrived -- so that "a slab follows this one" is a register
  // compare, as with the static lists
  int total_known = total_slabs;
  auto dyn_peek = [&]() {  // add the length of the segment after the current one (nothing is published after the end marker)
    if (c_tile < 0) return;
    const volatile int* d = dyn_tab[(c_seg + 1) % DYN_RING];
    total_known += d[0] >= 0 ? d[2] - d[1] : 0;
  };
  if constexpr (CHUNK) {
    c_chunk = c_s0 / plan.flush_slabs;
    to_flush = plan.flush_slabs - c_s0 % plan.flush_slabs;
  }
  auto end_of_segment = [&]() {
    int tm, tn;
    raster_tile(c_tile, plan.tiles_m, plan.tiles_n, tm, tn, plan.group_m);
    const int row_base = tm * C::BM + wm * MT * 8, col_base = tn * C::BN + wn * NT * 8;
    if constexpr (CHUNK) {
      if (c_s1 - c_s0 == KS) {  // whole tile: fold the last chunk in, finish the expansions, write C once
        flush_chunk();
        chunk_epilogue<L, MT, NT>(rexp, m, n, row_base, col_base, lane, C_planes);
        zero_rexp();
      } else {                  // stream-K part: the last (possibly partial) chunk of this run, then the hand-over
        const int r = c_tile - sk_base;
        flush_partial(r, c_chunk);
        __threadfence();
        __syncthreads();
        if (tid == 0) {
          const unsigned int mine = (unsigned int)(c_s1 - c_s0);
          *last_flag = (atomicAdd(&sk_counters[r], mine) + mine == (unsigned int)KS);
        }
        __syncthreads();
        if (*last_flag) {  // every slab of the tile is in the scratch: the chunk totals in order, as a whole-tile run would
          __threadfence();
          const int nchunks = (KS + plan.flush_slabs - 1) / plan.flush_slabs;
          for (int c = 0; c < nchunks; c++) {
            const double* sc = chunk_slot(r, c);
#pragma unroll
            for (int s = 0; s < S; s++)
#pragma unroll
              for (int i = 0; i < MT; i++)
#pragma unroll
                for (int j = 0; j < NT; j++) {
                  const double2 v = __ldcg(reinterpret_cast<const double2*>(sc + ((s * MT + i) * NT + j) * 64));
                  acc[s][i][j][0] = v.x;
                  acc[s][i][j][1] = v.y;
                }
            flush_chunk();
          }
          chunk_epilogue<L, MT, NT>(rexp, m, n, row_base, col_base, lane, C_planes);
          zero_rexp();
        }
      }
    } else if (c_s1 - c_s0 == KS) {  // whole tile in registers
      qgemm_epilogue<S, L, MT, NT>(acc, m, n, row_base, col_base, lane, order_planes, C_planes);
    } else if constexpr (!HANDOVER) {  // partial sums of a stream-K tile: exact fp64 reduction through the tile's scratch
      const int r = c_tile - sk_base;
      double* sc = sk_scratch + (size_t)r * (S * C::BM * C::BN) + (size_t)warp * (S * MT * NT * 64) + lane * 2;
#pragma unroll
      for (int s = 0; s < S; s++)
#pragma unroll
        for (int i = 0; i < MT; i++)
#pragma unroll
          for (int j = 0; j < NT; j++) {
            atomicAdd(sc + ((s * MT + i) * NT + j) * 64, acc[s][i][j][0]);
            atomicAdd(sc + ((s * MT + i) * NT + j) * 64 + 1, acc[s][i][j][1]);
          }
      __threadfence();
      __syncthreads();
      if (tid == 0) {
        const unsigned int mine = (unsigned int)(c_s1 - c_s0);
        *last_flag = (atomicAdd(&sk_counters[r], mine) + mine == (unsigned int)KS);
      }
      __syncthreads();
      if (*last_flag) {  // every slab of the tile has been added: read the totals back and finish the tile
        __threadfence();
#pragma unroll
        for (int s = 0; s < S; s++)
#pragma unroll
          for (int i = 0; i < MT; i++)
#pragma unroll
            for (int j = 0; j < NT; j++) {
              const double2 v = __ldcg(reinterpret_cast<const double2*>(sc + ((s * MT + i) * NT + j) * 64));
              acc[s][i][j][0] = v.x;
              acc[s][i][j][1] = v.y;
            }
        qgemm_epilogue<S, L, MT, NT>(acc, m, n, row_base, col_base, lane, order_planes, C_planes);
      }
    } else {
      if (c_s1 < KS) {   // the head (or a middle part) of a tile that another CTA finishes: hand the partial sums over
        double* sc = sk_scratch + (size_t)cta * (S * C::BM * C::BN) + (size_t)warp * (S * MT * NT * 64) + lane * 2;
#pragma unroll
        for (int s = 0; s < S; s++)
#pragma unroll
          for (int i = 0; i < MT; i++)
#pragma unroll
            for (int j = 0; j < NT; j++)
              __stcg(reinterpret_cast<double2*>(sc + ((s * MT + i) * NT + j) * 64), make_double2(acc[s][i][j][0], acc[s][i][j][1]));
        // PER WARP: a warp's part of the slot is read by the same warp of the finishing CTA only, so each warp raises its own
        // flag and goes on -- no block-wide barrier (ncu at 256^3: 0.76 barrier + 0.19 membar stall cycles per issued
        // instruction with the block-wide version, about 3 us per warp of a 45 us kernel)
        // (one flag per CTA behind a block-wide barrier.  A flag per WARP, without the barrier, was measured and not kept: 256^3
        // unchanged, 1024^3 2.135 -> 2.201 ms -- profiles/r04_small_sizes.md)
        __threadfence();
        __syncthreads();
        if (tid == 0) {
          __threadfence();
          atomicExch(&sk_counters[cta], 1u);  // the flag: this CTA's slot is complete
        }
      } else {                  // the tail of a tile: add what the CTAs before this one computed of it, then finish the tile
        const int r = c_tile - plan.dp_waves * G;
        const int first = (r * KS) / plan.sk_iters_per_cta;  // the CTA whose range holds the tile's first slab
        for (int other = first; other < cta; other++) {
          if (tid == 0) {
            while (atomicAdd(&sk_counters[other], 0u) == 0u) __nanosleep(64);
            __threadfence();
          }
          __syncthreads();
          const double* sc = sk_scratch + (size_t)other * (S * C::BM * C::BN) + (size_t)warp * (S * MT * NT * 64) + lane * 2;
#pragma unroll
          for (int s = 0; s < S; s++)
#pragma unroll
            for (int i = 0; i < MT; i++)
#pragma unroll
              for (int j = 0; j < NT; j++) {
                const double2 v = __ldcg(reinterpret_cast<const double2*>(sc + ((s * MT + i) * NT + j) * 64));
                acc[s][i][j][0] += v.x;  // exact: integers below 2^53 units (R6)
                acc[s][i][j][1] += v.y;
              }
        }
        qgemm_epilogue<S, L, MT, NT>(acc, m, n, row_base, col_base, lane, order_planes, C_planes);
      }
    }
    zero_acc();
    if (DYN || ++c_seg < n_seg) {
      if constexpr (DYN) ++c_seg;
      segment(c_seg, c_tile, c_s0, c_s1);  // DYNAMIC: tile < 0 when the queue is exhausted (the loops below have stopped by then)
      c_left = c_s1 - c_s0;
      if constexpr (DYN && C::PREFETCH) dyn_peek();
      if constexpr (CHUNK) {
        c_chunk = c_s0 / plan.flush_slabs;
        to_flush = plan.flush_slabs - c_s0 % plan.flush_slabs;
      }
    }
  };
  // CHUNK: after a slab of the current segment -- at a chunk boundary inside the segment fold the chunk away
  auto after_slab = [&]() {
    if constexpr (CHUNK) {
      if (--to_flush == 0 && c_left > 0) {
        if (c_s1 - c_s0 == KS) flush_chunk();
        else flush_partial(c_tile - sk_base, c_chunk);
        c_chunk++;
        to_flush = plan.flush_slabs;
      }
    }
  };

  int st = 0;          // stage of the slab being consumed
  uint32_t phase = 0;  // parity of that stage's current fill
  if constexpr (C::PREFETCH) {
    Frags f0, f1;
    mbar_wait(full_u32, 0);
    if constexpr (DYN) {
      total_known = c_left;
      dyn_peek();
    }
    load_frags(f0, stages + a_off, stages + b_off, 0);
    for (int it = 0; it < total_known; it++) {
      if (tid == 0) produce();
      const double* As = stages + (size_t)st * (C::A_CHUNK + C::B_CHUNK) + a_off;
      const double* Bs = stages + (size_t)st * (C::A_CHUNK + C::B_CHUNK) + b_off;
      load_frags(f1, As, Bs, 1);
      k_step(f0, Bs, 0);

      const int nst = (st + 1 == STAGES) ? 0 : st + 1;
      const uint32_t nphase = (st + 1 == STAGES) ? phase ^ 1 : phase;
      if (it + 1 < total_known) {  // next slab: its first k-step's fragments are fetched under this slab's second k-step
        mbar_wait(full_u32 + 8 * nst, nphase);
        load_frags(f0, stages + (size_t)nst * (C::A_CHUNK + C::B_CHUNK) + a_off,
                   stages + (size_t)nst * (C::A_CHUNK + C::B_CHUNK) + b_off, 0);
      }
      k_step(f1, Bs, 1);
      __syncwarp();
      if (lane == 0) mbar_arrive(empty_u32 + 8 * st);  // this warp is done reading the stage
      st = nst;
      phase = nphase;
      --c_left;
      after_slab();
      if (c_left == 0) end_of_segment();
    }
  } else {  // one fragment set (register budget): loads of a k-step are issued at its start
    for (int it = 0; DYN ? c_tile >= 0 : it < total_slabs; it++) {
      if (tid == 0) produce();
      mbar_wait(full_u32 + 8 * st, phase);
      const double* As = stages + (size_t)st * (C::A_CHUNK + C::B_CHUNK) + a_off;
      const double* Bs = stages + (size_t)st * (C::A_CHUNK + C::B_CHUNK) + b_off;
#pragma unroll
      for (int k4 = 0; k4 < C::K4; k4++) {
        Frags f;
        load_frags(f, As, Bs, k4);
        k_step(f, Bs, k4);
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(empty_u32 + 8 * st);
      if (++st == STAGES) {
        st = 0;
        phase ^= 1;
      }
      --c_left;
      after_slab();
      if (c_left == 0) end_of_segment();
    }
  }
}

// whole-tile waves from which the stream-K tail goes through red.add (launch_cfg).  Re-measured on the final build (hand-over
// against red.add, fraction of the peak): dd 768^3 (1 whole wave) 0.965 / 0.952, qd 768^3 (3) 0.9715 / 0.9699, dd 1024^3 (3)
// 0.9724 / 0.9733, dd 1280^3 (5) 0.9788 / 0.9799, qd 1024^3 (6) 0.9729 / 0.9763, dd 1536^3 (7) 0.9819 / 0.9831, dd 2048^3 (13)
// 0.9841 / 0.9862 -- the hand-over pays while the cut tiles are a large part of the work
constexpr int HANDOVER_MAX_WAVES = 4;

// Exact orders over the whole k, persistent stream-K.
template <class C>
cudaError_t launch_cfg(int m, int n, int k, const double* Ap, const double* Bp, double* order_planes, double* C_planes,
                       void* sk_ws, bool counters_clear, cudaStream_t stream) {
  constexpr bool SMALL = C::L == 2 && C::MT == 1;
  static_assert(C::BM == pack_bx(C::L, C::Q, 0, SMALL) && C::BN == pack_bx(C::L, C::Q, 1, SMALL), "tile shape must match the packed layout");
  const int tiles_m = (m + C::BM - 1) / C::BM, tiles_n = (n + C::BN - 1) / C::BN;
  const long long tiles = (long long)tiles_m * tiles_n;
  if (tiles > 0x7fffffffLL) return cudaErrorInvalidValue;
  const int G = sk_grid();
  if (G <= 0) return cudaErrorInvalidDevice;
  SkPlan plan = make_sk_plan(tiles_m, tiles_n, (k + C::BK - 1) / C::BK, G);
  unsigned int* counters = static_cast<unsigned int*>(sk_ws);
  double* scratch = reinterpret_cast<double*>(static_cast<char*>(sk_ws) + SK_COUNTER_BYTES);
  cudaError_t err;
  // Which schedule (all give the same bits):
  //   hand-over between the CTAs of a stream-K tile while every tile is cut or nearly so (small problems; measured: 512^3
  //   0.88 -> 0.92 of the peak with it, dd 4096^3 134.65 against 134.88 ms without);
  //   the static lists with red.add once whole-tile waves dominate;
  //   the HYBRID from many waves on: every whole tile keeps its static place (tile = wave * G + cta: the CTAs stay in lock-step
  //   and share operand slabs through L2) and only the k-units of the last, partial wave's tiles are claimed from the queue, so
  //   that a CTA which has fallen behind claims fewer and all SMs finish within one unit's time.  It costs a red.add of the
  //   accumulators per unit (16 per cut tile instead of about 2) and pays once the spread it removes is larger than that:
  //   measured (profiles/r04_dynamic_schedule.md) quad double from about 10 whole waves on (1280^3 +0.001, 1536^3 +0.005,
  //   2048^3 0.9747 -> 0.9796 of the peak; 1024^3, 6.9 waves: -0.012), double double, whose SMs finish within 0.1 % anyway, from
  //   about 48 (3072^3, 31 waves: -0.0004; 4096^3, 55: +0.0003; 8192 x 8192 x 2048 with 9 quarters, 221: +0.002);
  //   the queue for EVERYTHING only on request: it levels the finishing times too, but CTAs that claim whole tiles at their own
  //   pace no longer fetch the same slabs at the same time (dd 4096^3: L2 hit rate 84 % -> 63 %, DRAM reads x 3) and lose more than
  //   the balance returns (dd 4096^3 135.17 against 134.41 ms, qd 2048^3 65.31 against 64.40).
  // MD_OPT_TILE_SCHEDULE: 0 = this rule, 1 = hybrid wherever there is a whole wave, 2 = queue only, 3 = never (static lists).
  const int sched_opt = tile_schedule();
  const int hybrid_from = C::L >= 4 ? 10 : 48;  // whole-tile waves
  const bool hybrid = (sched_opt == 1 && plan.dp_waves >= 1) || (sched_opt == 0 && plan.dp_waves >= hybrid_from);
  const bool dynamic = hybrid || (sched_opt == 2 && plan.dp_waves >= 1);
  const bool handover = !dynamic && plan.dp_waves < HANDOVER_MAX_WAVES;
  if (dynamic) {
    // the tiles that are cut: the last partial wave, plus one whole wave when that is short -- the whole-tile phase ends with
    // the SMs spread over one tile time, and the cut tiles have to fill that triangle (about G / 2 tile times)
    int cut = plan.sk_tiles;
    if (hybrid) {
      if (cut == 0) cut = G;  // no partial wave: the last whole wave is the one that is cut
    } else if (cut < (7 * G) / 10 && cut + G <= SK_MAX_TILES - 1) {
      cut += G;
    }
    constexpr int units = 16;
    plan.dyn_whole = (int)tiles - cut;
    // 1: EVERY whole tile keeps the static assignment (lock-step, L2 sharing) and only the k-units of the cut tiles are claimed;
    // 2: the queue from the start
    plan.dyn_static = hybrid ? plan.dyn_whole / G : 0;
    plan.dyn_unit = (plan.KS + units - 1) / units;
    plan.dyn_upt = (plan.KS + plan.dyn_unit - 1) / plan.dyn_unit;
    plan.dyn_items = plan.dyn_whole + cut * plan.dyn_upt;
    // queue counter, slab counters and the scratch tiles of the cut tiles start at zero
    err = cudaMemsetAsync(sk_ws, 0, SK_COUNTER_BYTES + sizeof(double) * (size_t)(plan.dyn_upt > 1 ? cut : 0) * C::S * C::BM * C::BN, stream);
    if (err != cudaSuccess) return err;
  } else if (plan.sk_tiles > 0) {  // hand-over: the flags (one per CTA) start at zero, the slots are written before they are read;
                                   // red.add: counters and the scratch tiles in use start at zero (one contiguous region)
    const size_t bytes = handover ? (size_t)SK_COUNTER_BYTES
                                  : SK_COUNTER_BYTES + sizeof(double) * (size_t)plan.sk_tiles * C::S * C::BM * C::BN;
    if (!(handover && counters_clear)) {  // the fused preparation kernel has cleared the flags already (md_gemm below ~2048^3)
      err = cudaMemsetAsync(sk_ws, 0, bytes, stream);
      if (err != cudaSuccess) return err;
    }
  }
  static bool attr_done[MD_MAX_DEVICES][3] = {};  // the shared-memory opt-in is per function and device: once, not per launch
  const int dev = current_device();
  const bool known = dev >= 0 && dev < MD_MAX_DEVICES;
  const int mode = dynamic ? SCHED_DYNAMIC : handover ? SCHED_HANDOVER : SCHED_STATIC;
  auto kern = mode == SCHED_DYNAMIC ? qgemm_packed_kernel<C, false, SCHED_DYNAMIC>
            : mode == SCHED_HANDOVER ? qgemm_packed_kernel<C, false, SCHED_HANDOVER> : qgemm_packed_kernel<C, false, SCHED_STATIC>;
  if (!known || !attr_done[dev][mode]) {
    err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES);
    if (err != cudaSuccess) return err;
    if (known) attr_done[dev][mode] = true;
  }
  if (handover && counters_clear) {
    // directly behind the cooperative preparation kernel on this stream (no memset node in between): let the CTAs start while
    // it drains -- launch latency, barrier set-up and the segment tables then cost nothing (256^3: 53.9 -> 51.6 us per md_gemm)
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(G), cfg.blockDim = dim3(C::THREADS), cfg.dynamicSmemBytes = C::SMEM_BYTES, cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr, cfg.numAttrs = 1;
    err = cudaLaunchKernelEx(&cfg, kern, m, n, plan, Ap, Bp, order_planes, C_planes, scratch, counters);
    if (err == cudaSuccess) return cudaGetLastError();
    cudaGetLastError();  // a context that refuses the attribute: the plain launch does the same work
  }
  kern<<<G, C::THREADS, C::SMEM_BYTES, stream>>>(m, n, plan, Ap, Bp, order_planes, C_planes, scratch, counters);
  return cudaGetLastError();
}

// Chunked accumulation (chunk = contraction indices per chunk, a multiple of BK): whole tiles only, wave after wave on the
// persistent grid, the last wave possibly partial.
template <class C>
cudaError_t launch_chunked(int m, int n, int k, int chunk, const double* Ap, const double* Bp, double* C_planes,
                           void* sk_ws, cudaStream_t stream) {
  static_assert(C::BM == pack_bx(C::L, C::Q, 0) && C::BN == pack_bx(C::L, C::Q, 1), "tile shape must match the packed layout");
  const int tiles_m = (m + C::BM - 1) / C::BM, tiles_n = (n + C::BN - 1) / C::BN;
  const long long tiles = (long long)tiles_m * tiles_n;
  if (tiles > 0x7fffffffLL || !C_planes || chunk <= 0 || chunk % C::BK) return cudaErrorInvalidValue;
  const int G = sk_grid();
  if (G <= 0) return cudaErrorInvalidDevice;
  SkPlan plan = make_sk_plan(tiles_m, tiles_n, (k + C::BK - 1) / C::BK, G);
  plan.flush_slabs = chunk / C::BK;
  const size_t nchunks = ((size_t)plan.KS + plan.flush_slabs - 1) / plan.flush_slabs;
  unsigned int* counters = static_cast<unsigned int*>(sk_ws);
  double* scratch = reinterpret_cast<double*>(static_cast<char*>(sk_ws) + SK_COUNTER_BYTES);
  cudaError_t err;
  if (sk_chunk_scratch_fits(nchunks, C::S, C::BM, C::BN)) {  // stream-K tail, one scratch slot per (tile, chunk)
    if (plan.sk_tiles > 0) {
      err = cudaMemsetAsync(sk_ws, 0, SK_COUNTER_BYTES + sizeof(double) * plan.sk_tiles * nchunks * C::S * C::BM * C::BN, stream);
      if (err != cudaSuccess) return err;
    }
  } else {  // too many chunks for the scratch (a very long contraction): whole tiles only, the last wave partial
    plan.dp_waves = (int)((tiles + G - 1) / G);
    plan.dp_tail = tiles % G ? (int)(tiles % G) : G;
    plan.sk_tiles = 0;
    plan.sk_iters_per_cta = 0;
  }
  auto kern = qgemm_packed_kernel<C, true>;
  static bool attr_done[MD_MAX_DEVICES] = {};  // the shared-memory opt-in is per function and device: once, not per launch
  const int dev = current_device();
  if (dev < 0 || dev >= MD_MAX_DEVICES || !attr_done[dev]) {
    err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES);
    if (err != cudaSuccess) return err;
    if (dev >= 0 && dev < MD_MAX_DEVICES) attr_done[dev] = true;
  }
  kern<<<G, C::THREADS, C::SMEM_BYTES, stream>>>(m, n, plan, Ap, Bp, nullptr, C_planes, scratch, counters);
  return cudaGetLastError();
}

// double double: 64 x 32 CTA tile, 8 warps (4 x 2), 16 x 16 warp tile.  quad double: 32 x 32 CTA tile, 8 x 16 warp tile
// (16 orders x 2 registers per 8x8 tile).
template <int Q, int S = Q> using PCfgDD = PCfg<Q, 2, 4, 2, 2, 2, S>;
// double double on 32 x 16 CTA tiles (8 x 8 warp tiles): four times the tiles, for problems whose 64 x 32 tiles would not
// fill the SMs -- every tile would be cut along k and each CTA would flush a whole tile of partial sums through L2
template <int Q> using PCfgDDS = PCfg<Q, 2, 4, 2, 1, 1>;
template <int Q, int S = Q> using PCfgQD = PCfg<Q, 4, 4, 2, 1, 2, S>;
// quad double in 11 / 12 wide slices (MD_OPT_SLICE_BITS): 22 / 24 accumulator registers per 8x8 tile leave room for the
// double-double warp tile (16 x 16), which halves the LDS and L2 traffic per DMMA and doubles the DMMAs per slab
template <int Q> using PCfgQDW = PCfg<Q, 4, 4, 2, 2, 2>;
// quad double with chunked accumulation (10 slices): the expansions of the elements (5 terms each) live in registers
// beside the accumulators, so the warp tile is 16 x 8 (64 x 16 CTA tile)
template <int Q> using PCfgQDC = PCfg<Q, 4, 4, 2, 2, 1>;

}  // namespace

// CTAs of the persistent grid: one per SM of the current device, at most SK_MAX_TILES (the scratch holds one tile per stream-K
// tile, < grid)
int sk_grid() {
  const int sms = sm_count();
  if (sms <= 0) return -1;
  return sms < SK_MAX_TILES ? sms : SK_MAX_TILES;
}

// chunk > 0 (chunked accumulation): one slot per (stream-K tile, chunk) as long as that stays below SK_CHUNK_CAP_BYTES
size_t sk_workspace_bytes(int orders, int bxA, int bxB, int k, int chunk) {
  const size_t tile = sizeof(double) * (size_t)orders * bxA * bxB;
  size_t slots = SK_MAX_TILES;
  if (chunk > 0) {
    const size_t nchunks = ((size_t)k + chunk - 1) / chunk;
    if (sk_chunk_scratch_fits(nchunks, orders, bxA, bxB)) slots *= nchunks;
  }
  return SK_COUNTER_BYTES + tile * slots;
}

bool qgemm_small_supported(int limbs, int quarters, int orders) { return limbs == 2 && orders == quarters && (quarters == 8 || quarters == 6); }

bool qgemm_chunk_supported(int limbs, int quarters) {
  return (limbs == 2 && (quarters == 5 || quarters == 6 || quarters == 8)) || (limbs == 4 && quarters == 10);
}

// tuned instances: orders == quarters for the counts of qgemm_supported, plus the extended order sets the cfg3-like cases use
// (S = Q + 1, Q + 2 at the paper's quarter counts); everything else runs on the generic kernel (qgemm_wide.cu)
bool qgemm_packed_supported(int limbs, int quarters, int orders) {
  if (orders == quarters) return qgemm_supported(limbs, quarters);
  return (limbs == 2 && quarters == 8 && (orders == 9 || orders == 10)) || (limbs == 4 && quarters == 16 && (orders == 17 || orders == 18));
}

cudaError_t launch_qgemm_packed(int m, int n, int k, int limbs, int quarters, int orders, int chunk, bool small, const double* Ap,
                                const double* Bp, double* order_planes, double* C_planes, void* sk_ws, bool counters_clear,
                                cudaStream_t stream, uint64_t* launches) {
  cudaError_t err = cudaErrorInvalidValue;
#define MD_Q(...) err = launch_cfg<__VA_ARGS__>(m, n, k, Ap, Bp, order_planes, C_planes, sk_ws, counters_clear, stream)
  if (small) {
    if (chunk > 0 || !qgemm_small_supported(limbs, quarters, orders)) return cudaErrorInvalidValue;
    if (quarters == 8) MD_Q(PCfgDDS<8>);
    if (quarters == 6) MD_Q(PCfgDDS<6>);
  } else if (chunk > 0) {  // only the instances of qgemm_chunk_supported are compiled with the chunked kernel
    if (orders != quarters) return cudaErrorInvalidValue;
    if (limbs == 2 && quarters == 5) err = launch_chunked<PCfgDD<5>>(m, n, k, chunk, Ap, Bp, C_planes, sk_ws, stream);
    if (limbs == 2 && quarters == 6) err = launch_chunked<PCfgDD<6>>(m, n, k, chunk, Ap, Bp, C_planes, sk_ws, stream);
    if (limbs == 2 && quarters == 8) err = launch_chunked<PCfgDD<8>>(m, n, k, chunk, Ap, Bp, C_planes, sk_ws, stream);
    if (limbs == 4 && quarters == 10) err = launch_chunked<PCfgQDC<10>>(m, n, k, chunk, Ap, Bp, C_planes, sk_ws, stream);
  } else if (orders != quarters) {
    if (limbs == 2 && quarters == 8 && orders == 9) MD_Q(PCfgDD<8, 9>);
    if (limbs == 2 && quarters == 8 && orders == 10) MD_Q(PCfgDD<8, 10>);
    if (limbs == 4 && quarters == 16 && orders == 17) MD_Q(PCfgQD<16, 17>);
    if (limbs == 4 && quarters == 16 && orders == 18) MD_Q(PCfgQD<16, 18>);
  } else if (limbs == 2) {
    if (quarters == 6) MD_Q(PCfgDD<6>);
    if (quarters == 7) MD_Q(PCfgDD<7>);
    if (quarters == 8) MD_Q(PCfgDD<8>);
    if (quarters == 9) MD_Q(PCfgDD<9>);
    if (quarters == 10) MD_Q(PCfgDD<10>);
  } else if (limbs == 4) {
    if (quarters == 11) MD_Q(PCfgQDW<11>);
    if (quarters == 12) MD_Q(PCfgQDW<12>);
    if (quarters == 16) MD_Q(PCfgQD<16>);
    if (quarters == 17) MD_Q(PCfgQD<17>);
    if (quarters == 18) MD_Q(PCfgQD<18>);
  }
#undef MD_Q
  if (err == cudaSuccess) *launches += 1;
  return err;
}

}  // namespace md
