/* mdgemm.h -- C-ABI boundary of the B200 (sm_100a) multiple-double matrix multiplication library.
 *
 * Hot path of "Multiple Double Arithmetic on NVIDIA Tensor Cores" (Chen & Verschelde, arxiv/paper_2607_06881):
 *   C = A * B for matrices whose elements are multiple doubles (Definition 1.1: an unevaluated sum of
 *   non-overlapping doubles), stored as `limbs` fp64 LIMB PLANES (double-double: A_hi, A_lo; quad-double:
 *   4 planes).  The five steps of PAPER.md:82-89 are:
 *     1. split every element into 13-bit "quarters"                                   -> md_split      (a1 + a2)
 *     2./3. multiply the quarter matrices on the FP64 tensor pipe, exactly            -> md_qgemm      (a3)
 *     4./5. extract the parts C_1..C_S and add them into a multiple-double matrix     -> md_renorm     (a4)
 *   and md_gemm runs all of them (steps 3-5 fused in one kernel: the stacked matrices Abar, Bbar of eq. (4),
 *   PAPER.md:75, are never built).  Citations "PAPER.md:<line>" refer to /root/reference/PAPER.md; "DESIGN.md Rn" to
 *   the readings of the paper listed in DESIGN.md section 3.
 *
 * Conventions for every entry point
 *   - No torch / C++ types: plain pointers and sizes.  Unless a parameter says "host", every data pointer is a DEVICE
 *     pointer (cudaMalloc'ed or a torch CUDA tensor's data_ptr) on the current device, 8-byte aligned (16-byte
 *     alignment together with even column counts enables the vectorised paths; anything else still works).
 *   - Matrices are dense, row-major planes: a multiple-double matrix X (rows x cols) with `limbs` limbs is
 *     limbs * rows * cols doubles, plane l at X + l*rows*cols, element (i,j) of plane l at X[l*rows*cols + i*cols + j]
 *     (a contiguous torch tensor [limbs, rows, cols]).  Plane 0 is the leading (high) double.
 *   - `stream` is a cudaStream_t passed as an opaque pointer (NULL = the legacy default stream).  Calls ENQUEUE work on
 *     it and return without synchronising (md_gemm_host and md_read_flags excepted); they are safe to capture in a
 *     CUDA graph.  The library never allocates device memory; the caller owns every buffer, and must keep it alive until
 *     the stream has run the work.  Inputs are read-only; outputs must not alias inputs or the workspace.
 *   - Return value: MD_OK (0) or a negative md_status.  Errors are detected from the ARGUMENTS only, synchronously,
 *     and nothing has been enqueued when one is returned (MD_ERR_CUDA: a launch failed; cudaGetLastError is preserved).
 *   - Data preconditions (cannot be seen without a sync, so they are not return codes): inputs finite; the leading limb
 *     is the largest in magnitude and |limb_{l+1}| <= ulp(limb_l); every group exponent E (below) within [-900, 900] and
 *     E >= W * quarters - 1022 (every digit unit a normal double).  Violations set bits in a device status word
 *     (md_read_flags) and give unspecified values, never a fault.  For a PRODUCT the conditions are pairwise: with E_i the
 *     exponent of row i of A and F_j of column j of B, exactness needs E_i + F_j <= 1023 and E_i + F_j - W (orders + 1) >= -1022
 *     (the smallest kept order unit a normal double).  The first shows in C itself (an overflow gives +-inf / NaN there);
 *     the second is NOT flagged per pair: below it the lowest orders lose bits silently.  |E| <= 450 on both sides is always
 *     safe for double and quad double.
 *   - ACCURACY IS RELATIVE TO 2^(E_i + F_j), NOT TO (|A||B|)_ij (see md_gemm): on data whose rows / columns span many binades
 *     the default quarter count can miss the format's tolerance relative to (|A||B|)_ij without any flag.  md_plan_quarters
 *     measures what the data needs, md_gemm_auto runs the plan and the product in one call, and every count the plan can
 *     return (up to 16 / 24 / 40 / 72 quarters for 2 / 4 / 8 / 16 limbs) has a kernel.
 *   - Options (md_set_option) are process-wide; the registered workspace, the profile record and md_gemm_host's copy streams
 *     are per DEVICE (the current device of the calling thread).  All calls of the md_gemm family that share a workspace
 *     (including its stream-K scratch) must be serialised on ONE stream; two md_gemm_host calls on one device must not run
 *     concurrently; md_set_option / md_set_workspace / md_profile_* must not race with anything.  Distinct devices are
 *     independent.
 */
#ifndef MDGEMM_H_
#define MDGEMM_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef int md_status;
enum {
  MD_OK = 0,
  MD_ERR_BAD_ARG = -1,      /* null pointer, dimension <= 0, misaligned pointer, limbs/quarters/orders unsupported */
  MD_ERR_K_TOO_LARGE = -2,  /* k exceeds the exactness budget k * orders <= 2^27 (eq. 5; R6) and the
                               call cannot chunk the contraction (md_gemm_orders, md_qgemm, quad double and wider) */
  MD_ERR_WORKSPACE = -3,    /* no workspace registered, or it is too small (md_workspace_bytes) */
  MD_ERR_CUDA = -4,         /* a CUDA call failed */
  MD_ERR_UNSUPPORTED = -5,  /* combination of (limbs, quarters, orders) that has no kernel instantiation */
  MD_ERR_STATIC_LIMIT = -6  /* md_gemm_static: the problem needs more than the built-in scratch (md_static_scratch_bytes) */
};

typedef void* md_stream;    /* a cudaStream_t */

/* Options (process-wide).  value 0 restores the default. */
enum {
  MD_OPT_QUARTERS = 1,  /* quarters per element used by md_gemm / md_gemm_orders / md_gemm_host.  Default 4*limbs, the
                           paper's count (8 for double double, 16 for quad double).  Any count up to 16
                           (limbs=2), 24 (4), 40 (8), 72 (16) runs.  Tuned kernels: limbs=2: 8, 9, 10; limbs=4: 16, 17, 18
                           (R5); limbs=8: 32; limbs=16: 64 (octo / hexa double, Table 2,
                           DESIGN.md R13); with MD_OPT_SLICE_BITS also 6, 7 / 11, 12 / 22 / 44.  Every other count runs on
                           the generic kernel (runtime counts; slower, same bits). */
  MD_OPT_ORDERS = 2,    /* kept product orders S: C^(s) for s = 0..S-1 (the paper's C_1..C_S).  Default = quarters
                           (the paper keeps C_1..C_8 of 8 quarters).  1 <= S <= min(2*quarters - 1, 24 / 32 / 42 / 74 for limbs 2 / 4 / 8 / 16): S < quarters
                           is a PRUNED set (fewer products, larger error), S > quarters an EXTENDED one -- order Q adds the Q - 1
                           products p + q = Q that the paper's set drops, for less work than another quarter (R5).
                           Tuned kernels for (8, 9), (8, 10), (16, 17), (16, 18); the generic kernel otherwise.  Error bound:
                           see md_gemm. */
  MD_OPT_SLICE_BITS = 3, /* width W of a slice in bits, used by md_split and the md_gemm family.  Default 13: the paper's
                           quarter ("4 parts ... each of 13 bits").  Other widths (4..24) are the k-adaptive
                           variant of DESIGN.md R14 / SURVEY.md 8(f) NEXT-3 -- NOT the paper's quarters: a slice of W
                           bits sits on the unit 2^(E_g - W(q+1)), |D| <= 2^W (q = 0), 2^(W-1) (q > 0), and the
                           exactness budget becomes k * orders * 2^(2W) <= 2^53.  With wider slices fewer are needed:
                           set MD_OPT_QUARTERS to the slice count (limbs=2: 6, 7; limbs=4: 11, 12; limbs=8: 22; limbs=16: 44), or
                           take both from md_plan_slices. */
  MD_OPT_K_CHUNK = 5,    /* md_gemm / md_gemm_host, double double (5, 6, 8 slices) and quad double (10 slices) (R16): length of the chunks of the
                            contraction over which the accumulations are kept exact.  Default 0 = automatic: chunking is
                            used only when k exceeds the exactness budget k * orders * 2^(2W) <= 2^53, with the largest
                            chunk the budget allows; a value (a multiple of 8) forces a shorter chunk.  Within a chunk
                            every order sum is exact; at its end the sums are added into the element's expansion by the
                            TwoSum cascade of md_renorm.  md_gemm_orders never chunks (MD_ERR_K_TOO_LARGE as before). */
  MD_OPT_FUSED_PREP = 6, /* md_gemm / md_gemm_orders: 0 = automatic -- exponent vectors and packed quarter planes of both operands
                            in ONE cooperative launch when (m + n) * k <= 2^23 elements, five launches otherwise; 1 = always; 2 = never.
                            Same bits either way. */
  MD_OPT_TILE = 7,       /* md_gemm / md_gemm_orders, double double with 8 or 6 slices: 0 = automatic -- the 32 x 16 CTA tile
                            instance of the fused kernel when the 64 x 32 tiles would number at most 0.45 of the SMs
                            (up to about 352^3), 64 x 32 otherwise; 1 = 32 x 16 wherever it exists; 2 = never.  Same bits. */
  MD_OPT_RASTER_GROUP = 8, /* fused quarter GEMM: tile rows per raster group (the CTAs in flight cover GROUP x (SMs / GROUP) tiles of C and
                            share their operand slabs through L2).  0 = default 8 (the best of the measured 4 / 8 / 16 / 32,
                            profiles/).  Same bits for any value. */
  MD_OPT_ONE_LAUNCH = 9,  /* md_gemm / md_gemm_orders, double double (8 quarters) and quad double (16): 0 = automatic -- when the
                            32 x 16 tiles of C number at most the SMs and a CTA's run of the contraction is at most 16 k-slabs (cubes: up to 192^3) the WHOLE path runs in ONE launch: each
                            CTA derives the exponents of its rows / columns, splits its operand slabs into shared memory and
                            issues the quarter products; a thread-block cluster shares a tile along k (no quarter planes in
                            HBM); 1 = wherever that kernel exists (any size); 2 = never.  Same bits. */
  MD_OPT_TILE_SCHEDULE = 10, /* fused quarter GEMM of double / quad double (the persistent kernel), problems of at least one whole wave
                            of tiles.  The static stream-K lists keep the CTAs in lock-step on neighbouring tiles (they share operand
                            slabs through L2); a queue lets a CTA that has fallen behind take less.  0 = automatic: HYBRID -- every
                            whole tile keeps its static place, only the k-units (16 per tile) of the last, partial wave's tiles
                            are claimed from a queue, partial order sums combined by exact fp64 red.add -- from about 10 whole waves
                            on for quad double and 48 for double double, the static lists below; 1 = hybrid wherever there is a
                            whole wave; 2 = the queue for every tile; 3 = static lists always.  Same bits for all (every partial
                            sum is exact, R6).  Measured: profiles/r04_dynamic_schedule.md. */
  MD_OPT_HOST_BLOCKS = 4 /* md_gemm_host only: number of blocks C is cut into for overlapping copies and kernels.
                            Default 0 = automatic (about one wave of CTA tiles per block, at most 32); 1 = no overlap;
                            PR * 256 + PC = explicit numbers of row panels and column panels (each <= 64). */
};
md_status md_set_option(int key, int value);
int md_get_option(int key); /* current value (0 = default), or -1 for an unknown key */

/* Host-only helper for MD_OPT_SLICE_BITS: the fewest slices with a kernel for `limbs`, at the widest width W whose
 * exactness budget k * Q * 2^(2W) <= 2^53 holds (eq. 5 generalised), such that the window W * Q is at least
 * the paper's 13 * 4 * limbs bits.  Stores W in *bits_out and Q in *quarters_out (host pointers); (13, 4*limbs), the paper's
 * own split, when nothing wider qualifies.  Launches nothing and changes no option. */
md_status md_plan_slices(int k, int limbs, int* bits_out, int* quarters_out);
/* The same with chunked accumulation allowed (MD_OPT_K_CHUNK, R16): the budget only has to hold for a chunk of at
 * least min_chunk (>= 8) contraction indices where a chunked kernel exists (double double: 5, 6, 8 slices; quad double: 10), which admits
 * wider and fewer slices: double double at k = 4096 gets 5 slices of 21 bits in chunks of 408 (15 products instead of 21).
 * *chunk_out = the chunk md_gemm will use, 0 when this k needs none.  md_gemm_orders is not available beyond the budget. */
md_status md_plan_slices_chunked(int k, int limbs, int min_chunk, int* bits_out, int* quarters_out, int* chunk_out);

/* ---------------------------------------------------------------------------------------------------------------------
 * md_split -- steps a1 + a2: exponent vectors ("balancing") and quarter planes.
 *   PAPER.md:47-49 (section 2): the bits of a double are distributed over parts of 13 bits, the QUARTERS, doubles with
 *   exponents 0, -13, -26, -39; a double double gives 8 quarter matrices; exactness needs the
 *   exponents on an equally spaced grid; PAPER.md:124-142 (section 3): bits are moved between parts, value unchanged,
 *   until they are; zeros are "unnormalized zeros with the desired exponent".  Reading (R1-R4): one exponent
 *   per ROW (axis = 0, use for A) or per COLUMN (axis = 1, use for B):
 *       exps[g]  = E_g = ilogb(max over the group of |leading limb|) + 1   (0 for an all-zero group)
 *       quarter q of an element of group g = D * 2^(E_g - 13(q+1)), D an integer, |D| <= 2^13 (q = 0), 2^12 (q > 0),
 *       chosen nearest to what is left of the element after quarters 0..q-1 (ties to even on the leading remainder
 *       limb).  The element equals the sum of its quarters plus a remainder of at most 2^(E_g - 13*quarters - 1)
 *       (1 + 2^-27) in magnitude; the remainder is zero when the element fits the 13*quarters-bit window below 2^E_g.
 *   planes          in   [limbs][rows][cols]
 *   quarter_planes  out  [quarters][rows][cols]  true-valued quarters (not the integers D)
 *   exps            out  int32[rows] (axis 0) / int32[cols] (axis 1)
 *   limbs in {1, 2, 4, 8, 16}; 1 <= quarters <= 72; rows, cols >= 1.  Bit-exact against the oracle's Algorithm S.
 *   With MD_OPT_SLICE_BITS = W the 13 above reads W (R14).
 * ------------------------------------------------------------------------------------------------------------------ */
md_status md_split(int rows, int cols, int limbs, int quarters, int axis, const double* planes,
                   double* quarter_planes, int32_t* exps, md_stream stream);

/* ---------------------------------------------------------------------------------------------------------------------
 * md_qgemm -- steps a3 (+ a4): the triangular set of quarter products on the FP64 tensor pipe (DMMA).
 *   PAPER.md:66-71 eq. (3) and :75-78 eq. (4): C^(s) = sum_{p+q=s} A_p * B_q for s = 0..orders-1 (the paper's C_{s+1}),
 *   orders*(orders+1)/2 quarter GEMMs (36 for double double) instead of the 64 blocks of Abar*Bbar.  Every fp64
 *   accumulation is exact, so the result does not depend on any summation order.
 *   Aq            in   [quarters][m][k]  quarter planes of A (md_split axis 0)
 *   Bq            in   [quarters][k][n]  quarter planes of B (md_split axis 1)
 *   order_planes  out  [orders][m][n] fp64, C^(s) true-valued; may be NULL
 *   C_planes      out  [limbs][m][n]: the orders summed error-free into `limbs` limbs in the kernel's epilogue
 *                      (same arithmetic as md_renorm); may be NULL.  Not both NULL.
 *   k * orders * 2^(2W) <= 2^53 (W = 13: k * orders <= 2^27).  limbs in {2, 4} with orders == quarters in {6..10} / {11, 12,
 *   16, 17, 18} run a kernel that reads the plain planes directly; every other (limbs, quarters, orders) md_gemm accepts is
 *   repacked into the REGISTERED WORKSPACE (md_set_workspace, sized by md_workspace_bytes with MD_OPT_QUARTERS / MD_OPT_ORDERS
 *   set to these counts) and runs the kernel md_gemm would (MD_ERR_WORKSPACE without one).
 * ------------------------------------------------------------------------------------------------------------------ */
md_status md_qgemm(int m, int n, int k, int limbs, int quarters, int orders, const double* Aq, const double* Bq,
                   double* order_planes, double* C_planes, md_stream stream);

/* ---------------------------------------------------------------------------------------------------------------------
 * md_renorm -- step a4: recombination.  PAPER.md:88-91 steps 4-5: "summing 8 doubles into one double double for each
 *   element of the product ... in double double arithmetic ... on regular cores".
 *   order_planes  in   [orders][m][n]
 *   C_planes      out  [limbs][m][n]:  sum_s C^(s) as `limbs` non-overlapping doubles (|limb_{l+1}| <= ulp(limb_l)/2),
 *                      within 2^-(53*limbs - 3) * sum_s |C^(s)| of the exact sum (R9).
 *   limbs in {1, 2, 4, 8, 16}; 1 <= orders <= 144.
 * ------------------------------------------------------------------------------------------------------------------ */
md_status md_renorm(int m, int n, int limbs, int orders, const double* order_planes, double* C_planes,
                    md_stream stream);

/* ---------------------------------------------------------------------------------------------------------------------
 * md_gemm -- the whole hot path: C = A * B (all five steps), A: m x k, B: k x n, C: m x n, each with
 *   `limbs` limb planes.  Splits A by rows and B by columns into the registered workspace, then one fused kernel does
 *   the quarter products and writes the renormalised C once.  limbs in {2, 4, 8, 16} (double double, quad double, and the
 *   octo / hexa double of PAPER.md:196-205 Table 2).
 *   Accuracy: |C - A*B|_ij <= k (Q+3) 2^(E_i + F_j - 13Q - 2) + 2^-(53*limbs - 3) |C|_ij for any input (Q = quarters = orders;
 *   E, F the exponent vectors of A's rows and B's columns).  THE BOUND IS RELATIVE TO 2^(E_i + F_j), NOT TO (|A||B|)_ij: on the
 *   BASELINE.json workloads it is within 1e-28 (|A||B|)_ij (double double; configs[3] with 9 quarters) and 1e-58 (quad
 *   double), but a row such as [2^60, 1 + 2^-70] loses the low limb of its small element -- no flag is raised; use
 *   md_plan_quarters / md_gemm_auto when the data is not known to be well scaled.  The Q + 3 units are: 2 + 2 from what the
 *   split leaves of a and of b, Q - 1 from the dropped products of order Q.  With orders S > Q the last becomes
 *   (2Q - 1 - S) 2^(-13 (S - Q)): about 4 units in all; with S < Q the bound is that of Q = S (R5).
 *   md_gemm_orders is the debug/parity variant: same split, then writes the order matrices C^(s) [orders][m][n] instead.
 * ------------------------------------------------------------------------------------------------------------------ */
md_status md_gemm(int m, int n, int k, int limbs, const double* A_planes, const double* B_planes, double* C_planes,
                  md_stream stream);
md_status md_gemm_orders(int m, int n, int k, int limbs, const double* A_planes, const double* B_planes,
                         double* order_planes, md_stream stream);

/* ---------------------------------------------------------------------------------------------------------------------
 * md_plan_quarters -- how many quarters THIS data needs (R15; SURVEY.md 8(f) NEXT-1 "exponent-spread-driven quarter
 *   count").  With one exponent per row of A / column of B the error of md_gemm is bounded relative to 2^(E_i + F_j), not to
 *   (|A||B|)_ij (see md_gemm below): |C - A*B|_ij <= k (Q+3) 2^(E_i + F_j - W Q - 2) + renormalisation, W = slice width (13).
 *   This call measures D = max over positions with (|A_0||B_0|)_ij > 0 of E_i + F_j - ilogb((|A_0||B_0|)_ij) -- the leading
 *   limb planes multiplied in plain fp64 on the same DMMA kernel, 1/36 of a double-double md_gemm -- and returns the
 *   smallest Q >= ceil(52 limbs / W) with k (Q+3) 2^(D - W Q - 2) <= rel_tol: with MD_OPT_QUARTERS = Q the first term of
 *   the bound is below rel_tol (|A||B|)_ij at EVERY position, for any input.  It is a worst-case guarantee (all dropped
 *   digit products at their bound with one sign); measured errors are 2-3 orders of magnitude below it.
 *   scratch        device, 256-byte aligned, md_plan_scratch_bytes(m, n, k) bytes (|A_0|, |B_0|, their product, exponents)
 *   rel_tol        0 = the tolerance of the format: 1e-28 (limbs 2), 1e-58 (4), 1e-120 (8), 1e-245 (16), 2^-50 (1)
 *   quarters_out   HOST: Q (not limited to the counts that have a kernel: md_gemm returns MD_ERR_UNSUPPORTED for those)
 *   spread_out     HOST, may be NULL: D (INT32_MIN when |A||B| is zero everywhere)
 *   SYNCHRONISES `stream`.  Launches 8 kernels.  Bit-exact against the oracle's plan up to the rounding of the fp64 sums
 *   (D can differ by one where a sum sits on a power of two).
 * ------------------------------------------------------------------------------------------------------------------ */
size_t md_plan_scratch_bytes(int m, int n, int k);
md_status md_plan_quarters(int m, int n, int k, int limbs, const double* A_planes, const double* B_planes, void* scratch,
                           size_t scratch_bytes, double rel_tol, int* quarters_out, int* spread_out, md_stream stream);

/* ---------------------------------------------------------------------------------------------------------------------
 * md_gemm_auto -- md_plan_quarters and md_gemm in one call: measures the spread D of THIS data, takes the smallest quarter
 *   count Q whose bound meets rel_tol (|A||B|)_ij at every position (0 = the format's tolerance), and runs the product with
 *   Q = S = that count (the tuned kernel where one exists, the generic one otherwise), ignoring MD_OPT_QUARTERS / MD_OPT_ORDERS.
 *   scratch        device, 256-byte aligned, caller-owned: the plan's scratch and then the workspace of the product.
 *                  md_auto_scratch_bytes(m, n, k, limbs, quarters) sizes it for a given count (0 = 4 * limbs, the paper's);
 *                  if the plan needs more, the call returns MD_ERR_WORKSPACE with the needed count in *quarters_used and has
 *                  enqueued nothing but the plan: size again and repeat.
 *   quarters_used  HOST, may be NULL: the count the product ran with (or needs)
 *   Returns MD_ERR_UNSUPPORTED when the plan exceeds the generic maxima (16 / 24 / 40 / 72).  SYNCHRONISES `stream` (the plan
 *   returns Q to the host, and the status word of the call is read back for md_read_flags); not capturable in a CUDA graph.
 * ------------------------------------------------------------------------------------------------------------------ */
size_t md_auto_scratch_bytes(int m, int n, int k, int limbs, int quarters);
md_status md_gemm_auto(int m, int n, int k, int limbs, const double* A_planes, const double* B_planes, double* C_planes,
                       void* scratch, size_t scratch_bytes, double rel_tol, int* quarters_used, md_stream stream);

/* ---------------------------------------------------------------------------------------------------------------------
 * The paper's OWN balancing, element by element (section 3; R17-R22) -- a second
 * split mode beside md_split / md_gemm, measured against them in profiles/ (it is far more work).
 *
 * md_split_literal -- Algorithm L on every element of a multiple-double matrix:
 *   (1) eq. (7): where a limb and the next have opposite signs, the upper gives b (one ulp of it; in general the
 *       smallest power of two >= that ulp above |lower|) to the lower; rounding errors travel down by TwoSum ("the last bit should
 *       then be added to the next double");
 *   (2) the element's exponent e = ilogb of its leading non-zero limb ("the exponent of the leading quarter");
 *   (3) part q = the bits of the element on the unit 2^(e - 13 (q+1)) (13-bit parts with exponents 0, -13, -26,
 *       -39, here of the ELEMENT and continued through all its limbs); the leading part also holds the hidden bit (14 bits);
 *   (4) eq. (8), top down: a part below 2^12 of its units borrows b = 2^12 units (half a unit of the part above,
 *       the paper's 2^-14) from the part above, provided that part keeps its own exponent; zero parts "do nothing".
 *   planes          in   [limbs][rows][cols]
 *   quarter_planes  out  [quarters][rows][cols]  true-valued parts, all of the element's sign, multiples of HALF their unit
 *   exps            out  int32[rows * cols]      e per ELEMENT (0 for a zero element)
 *   flags           MD_LITERAL_NO_EQ8: skip step (4)
 *   The element equals the sum of its parts plus a remainder below limbs * 2^(e - 13 quarters).  limbs in {2, 4, 8, 16};
 *   bit-exact against the oracle's Algorithm L.
 *
 * md_gemm_literal -- C = A * B through the exponent classes of PAPER.md:120-122: A = A_0 + ... + A_12 by e mod 13 (B likewise);
 *   inside a class every part of every element lies on the grid 2^(c + 13 Z), so part q of an element of level z = floor(e / 13)
 *   is plane q + (zmax - z) of the class matrix, a class pair A_c B_d is an ORDINARY quarter GEMM (md_gemm's kernels) with exact
 *   accumulations, and all order sums of all non-empty pairs are added error free into C.  Planes per class matrix: quarters +
 *   max(spanA, spanB); orders kept: quarters + spanA + spanB (span = zmax - zmin of an operand).  MD_LITERAL_SIGN_GROUPS adds the
 *   sign groups of eq. (6): 26 groups per operand, four sign-pair products per class pair, same C (every
 *   accumulation being exact, grouping by sign changes nothing but the cost).
 *   Error: relative to (|A||B|)_ij term by term -- about (quarters + 3) 2^(-13 quarters + 2) -- whatever the dynamic range.
 *   scratch      device, 256-byte aligned, caller-owned; md_literal_scratch_bytes(m, n, k, limbs, planes, orders) for given counts
 *                (0, 0 = no spread: quarters planes and orders).  If the data needs more, MD_ERR_WORKSPACE with the counts in
 *                info_host[4], [5]: size again and repeat.
 *   info_host    HOST int32[8], may be NULL: zminA, zmaxA, zminB, zmaxB, planes, orders, class pairs run, kernels launched
 *   MD_ERR_UNSUPPORTED when planes / orders exceed the generic kernel's maxima (16 / 24 for double double, 24 / 32 for quad
 *   double: level spans up to 8, i.e. elements over about 2^+-50); uses MD_OPT_QUARTERS, needs MD_OPT_SLICE_BITS = 13.
 *   SYNCHRONISES `stream` once (the counts come back to the host); not capturable in a CUDA graph.
 * ------------------------------------------------------------------------------------------------------------------ */
enum { MD_LITERAL_NO_EQ8 = 1, MD_LITERAL_SIGN_GROUPS = 2 };
md_status md_split_literal(int rows, int cols, int limbs, int quarters, int flags, const double* planes, double* quarter_planes,
                           int32_t* exps, md_stream stream);
size_t md_literal_scratch_bytes(int m, int n, int k, int limbs, int planes_per_class, int orders);
md_status md_gemm_literal(int m, int n, int k, int limbs, const double* A_planes, const double* B_planes, double* C_planes,
                          void* scratch, size_t scratch_bytes, int flags, int32_t* info_host, md_stream stream);

/* ---------------------------------------------------------------------------------------------------------------------
 * md_qr -- blocked Householder QR of a multiple-double matrix on top of md_gemm: the application the paper announces.
 *   PAPER.md:213 (conclusions): "Future work will apply this multiple double tensor core matrix multiplication to accelerate the
 *   blocked Householder QR, extending [18]" (ref [18]: least squares on GPUs in multiple double precision).
 *   A = Q R with A m x n (m >= n), Q m x n with orthonormal columns, R n x n upper triangular with diag(R) >= 0.
 *   Panels of 32 columns are factored on the regular FP64 cores in multiple-double arithmetic (one cooperative launch per panel);
 *   every trailing update and the accumulation of Q are products of limb-plane matrices through the SAME path as md_gemm
 *   (split, fused quarter GEMM on the FP64 tensor pipe, renormalising epilogue; MD_OPT_QUARTERS / MD_OPT_ORDERS apply).
 *   A_planes   in   [limbs][m][n]
 *   Q_planes   out  [limbs][m][n]
 *   R_planes   out  [limbs][n][n]
 *   scratch    device, 256-byte aligned, md_qr_scratch_bytes(m, n, limbs) bytes, caller-owned (working copy of A, block reflectors,
 *              compacted sub-matrices, the workspace of the products)
 *   times_ms_host  HOST float[2] or NULL: when given the call records CUDA events, SYNCHRONISES `stream`, and stores the device
 *              time of the whole factorisation and the part of it spent inside the md_gemm path (for bench.py)
 *   limbs in {2, 4}.  Backward error: |A - Q R| and |Q^T Q - I| of the order n 2^-(52 limbs) (norm-wise; tests/test_gpu_qr.py).
 *   Asynchronous unless times_ms_host is given; not capturable in a CUDA graph (cooperative launches).
 * ------------------------------------------------------------------------------------------------------------------ */
size_t md_qr_scratch_bytes(int m, int n, int limbs);
md_status md_qr(int m, int n, int limbs, const double* A_planes, double* Q_planes, double* R_planes, void* scratch,
                size_t scratch_bytes, float* times_ms_host, md_stream stream);

/* Workspace for md_gemm / md_gemm_orders: quarter planes of A and B, exponent vectors and the status word, for the
 * CURRENT option values.  The caller allocates (device memory, 256-byte aligned) and registers it FOR THE CURRENT DEVICE; the
 * library keeps the pointer until it is replaced (ptr = NULL, bytes = 0 unregisters).  md_workspace_bytes returns 0 on bad
 * arguments.  md_set_workspace clears the status word with a SYNCHRONOUS cudaMemset (it is a set-up call, not capturable). */
size_t md_workspace_bytes(int m, int n, int k, int limbs);
md_status md_set_workspace(void* dev_ptr, size_t bytes);

/* Device status word of the registered workspace, ORed with the status words md_gemm_host / md_gemm_auto calls on this device
 * have brought back (they run in caller scratch, not in the registered workspace), copied to *flags_host (host pointer);
 * SYNCHRONISES `stream`.  bit 0: a non-finite input was seen; bit 1: a group exponent outside its range (see the conventions
 * at the top).  Cleared by md_set_workspace, accumulates until then.  Without a registered workspace: the host-side record
 * alone, MD_ERR_WORKSPACE if there is none yet. */
md_status md_read_flags(uint32_t* flags_host, md_stream stream);

/* ---------------------------------------------------------------------------------------------------------------------
 * md_gemm_host -- md_gemm on HOST buffers (end-to-end path).  A_host, B_host, C_host are HOST pointers (pinned memory
 *   makes the copies asynchronous and fast; pageable works, without overlap).  dev_scratch is DEVICE memory of at least
 *   md_host_scratch_bytes(m,n,k,limbs) bytes, 256-byte aligned, owned by the caller; it receives the device copies of
 *   A, B, C and the workspace.  C is cut into blocks (row panels of A x column panels of B; a row's / column's exponent
 *   depends on that row / column only, so each block is an independent md_gemm with bit-identical results) and the
 *   copies in, the kernels and the copies out of successive blocks overlap: kernels run on `stream`, the copies on two
 *   streams the library creates on first use and keeps (the only resources it ever creates).  Work already enqueued on
 *   `stream` is waited for first; the call SYNCHRONISES `stream` before returning: C_host is complete on return.
 * ------------------------------------------------------------------------------------------------------------------ */
size_t md_host_scratch_bytes(int m, int n, int k, int limbs);
md_status md_gemm_host(int m, int n, int k, int limbs, const double* A_host, const double* B_host, double* C_host,
                       void* dev_scratch, size_t scratch_bytes, md_stream stream);

/* Per-call device timing of md_gemm / md_gemm_orders / md_gemm_host, for roofline accounting (bench.py).
 * md_profile_enable(capacity > 0): each following call on this device records CUDA events on its stream before its first
 * kernel, before the fused quarter-GEMM kernel and after it, for up to `capacity` calls (further calls are not recorded);
 * calling it again restarts the record; capacity = 0 disables and frees the events.  Do not enable while capturing a CUDA
 * graph (the timing events would become graph nodes).  md_gemm_host is recorded only when it runs as ONE block (small
 * problems); its multi-panel pipeline interleaves splits and products and records nothing.
 * md_profile_read synchronises the recorded events and returns how many calls were recorded (<= capacity, or a negative
 * md_status); for call i it stores the split time (exponent + split kernels) in split_ms_host[i] and the fused GEMM
 * kernel time in gemm_ms_host[i] (HOST arrays of at least `capacity` floats; either may be NULL). */
md_status md_profile_enable(int capacity);
int md_profile_read(float* split_ms_host, float* gemm_ms_host, int capacity);

/* ---------------------------------------------------------------------------------------------------------------------
 * md_probe_dmma -- calibration, not a step of the path: enqueues ONE kernel in which `blocks` CTAs of `warps_per_block`
 *   warps each issue iters * 8 register-only mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4, the instruction md_qgemm computes
 *   with; "double precision tensor cores").  Timed by the caller with CUDA events it gives the FP64
 *   tensor peak of this device, the roofline denominator of md_qgemm.
 *   sink            out  device, blocks * warps_per_block * 32 doubles, or NULL (nothing is written)
 *   flops_host      out  HOST pointer: FP64 flops the launch issues = blocks * warps_per_block * iters * 8 * 512
 *   1 <= blocks; 1 <= warps_per_block <= 32; 1 <= iters < 2^25.
 * ------------------------------------------------------------------------------------------------------------------ */
md_status md_probe_dmma(int blocks, int warps_per_block, int iters, double* sink, uint64_t* flops_host, md_stream stream);

/* ---------------------------------------------------------------------------------------------------------------------
 * md_gemm_static -- md_gemm (steps a1-a4: split, triangular quarter GEMM, recombination) for callers that can
 *   NOT allocate device memory: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The
 *   workspace md_gemm takes from md_set_workspace is a file-scope device array inside the library here (md_static_scratch_bytes()
 *   = 64 MiB); the call allocates nothing (no cudaMalloc / cudaFree / allocating library routine), needs no md_set_workspace, and
 *   runs the same kernels as md_gemm: the result is bit-identical.
 *   A_planes / B_planes / C_planes, limbs, stream, options (MD_OPT_QUARTERS, ...): as md_gemm.
 *   Limit: md_gemm_static_bytes(m, n, k, limbs) -- what this problem needs of the array with the current options, 0 for bad
 *   arguments -- must not exceed md_static_scratch_bytes(): with the default options cubes up to 496^3 (double double), 352^3
 *   (quad double), 192^3 (octo double); hexa double never fits (its stream-K scratch alone is 64 MiB).  Otherwise
 *   MD_ERR_STATIC_LIMIT, with nothing enqueued.
 *   Every GPU on which the library is used holds the 64 MiB until the process exits.  ALL calls on a device share the array, and
 *   it keeps the last call's contents (each call clears what must start at zero, on `stream`): two calls that overlap on the
 *   GPU -- different streams with no ordering between them -- RACE; serialise them.  The status word of the LAST call
 *   (md_read_flags's bits) is read with md_gemm_static_read_flags, which synchronises `stream`.
 * ------------------------------------------------------------------------------------------------------------------ */
size_t md_static_scratch_bytes(void);
size_t md_gemm_static_bytes(int m, int n, int k, int limbs);
md_status md_gemm_static(int m, int n, int k, int limbs, const double* A_planes, const double* B_planes, double* C_planes,
                         md_stream stream);
md_status md_gemm_static_read_flags(uint32_t* flags_host, md_stream stream);

/* Number of kernels this library has launched since load (all entry points), for launch accounting. */
uint64_t md_launch_count(void);

const char* md_status_string(md_status status);

#ifdef __cplusplus
}
#endif
#endif /* MDGEMM_H_ */
