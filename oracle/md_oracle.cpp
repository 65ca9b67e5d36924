// md_oracle.cpp -- CPU ORACLE for the multiple-double GEMM hot path of arxiv/paper_2607_06881
// ("Multiple Double Arithmetic on NVIDIA Tensor Cores", Chen & Verschelde).
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
// cpu_baseline / --impl reference legs of bench.py may load it.  It shares no code, header,
// table or helper with paper_2607_06881_b200/csrc (the CUDA path) and neither includes the other.
// It is deliberately plain and slow: straight loops in the paper's order and notation, fp64
// with contraction disabled (-ffp-contract=off), exact arithmetic done with a long accumulator.
// The only parallelism is an OpenMP `parallel for` over output rows (no blocking, no fusion).
//
// Citations are "PAPER.md:<line>" plus section / equation; "DESIGN.md Rn"
// names a reading of the paper listed in DESIGN.md section 3.
//
// Parts (all pinned by tests/test_oracle_*.py against things other than themselves -- exact
// rational arithmetic in Python, closed forms, hand-derived special cases, the paper's constants):
//   O1  oracle_exact_*      exact product  C = A*B of multiple-double matrices (plain definition)
//   O2  oracle_split        Algorithm S: exponent vectors + 13-bit quarters
//       oracle_*_w          the same with the slice width as a parameter (R14; 13 = the paper's quarter)
//   O3  oracle_orders_*     order matrices C^(s) = sum_{p+q=s} A_p B_q  (eq. 3-4)
//   O4  oracle_renorm       sum of the S order values -> L non-overlapping limbs
//   O5  oracle_classic_gemm classical multiple-double GEMM on "regular cores", cross-check
//   --  oracle_md_gemm      O2 -> O3 (fp64 route) -> O4, the paper's 5-step algorithm
//   --  oracle_md_gemm_rows_chunked_w   the same with the order sums formed exactly per chunk of k (R16)
//   --  oracle_plan_quarters            the quarter count a given input needs for a tolerance (R15)
//   O7  oracle_md_qr                   unblocked Householder QR in multiple-double arithmetic (PAPER.md:213 future work; ref [18])
//   O6  oracle_split_literal, oracle_md_gemm_literal   the paper's own section-3 balancing, element by element: eq. 7, eq. 8,
//                                       exponent classes A_0..A_12, sign groups of eq. 6 (R17-R22)
// Parity status: every function above has an independent pin (tests/test_oracle_*.py: accumulator, split, orders,
// renorm_exact, wide, slices, plan); none is "parity unpinned".

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>

#ifdef _OPENMP
#include <omp.h>
#endif

typedef unsigned __int128 u128;

// =====================================================================================================
// Long accumulator: an exact fixed-point two's-complement integer of NW 32-bit digits (stored in int64
// words with deferred carries).  Bit 0 has weight 2^-BIAS.  Every finite double and every product of two
// finite doubles is an integer multiple of 2^-2148 below 2^2048, so with BIAS = 2240 and 4608 bits nothing
// is ever rounded: sums of such terms are exact (a Kulisch accumulator).
// =====================================================================================================
namespace {

const int BIAS = 2240;
const int NW = 144;  // 144 * 32 = 4608 bits

struct LongAcc {
  int64_t w[NW];
  int pending;  // additions since the last carry propagation

  LongAcc() { clear(); }
  void clear() {
    std::memset(w, 0, sizeof(w));
    pending = 0;
  }

  // Carry propagation: afterwards every word except the top one is in [0, 2^32); the top word carries the sign.
  void normalize() {
    int64_t carry = 0;
    for (int i = 0; i < NW; i++) {
      int64_t v = w[i] + carry;
      int64_t lo = v & 0xffffffffLL;
      carry = (v - lo) >> 32;  // arithmetic shift: floor division by 2^32
      w[i] = lo;
    }
    w[NW - 1] += carry * 4294967296LL;  // carry * 2^32 (a multiplication: << of a negative carry is undefined before C++20); keeps the sign in the top word
    pending = 0;
  }

  // Add sign * mag * 2^e, with mag < 2^106.
  void add_scaled(u128 mag, int e, int sign) {
    if (mag == 0) return;
    int pos = e + BIAS;  // bit position of mag's bit 0
    int idx = pos >> 5, sh = pos & 31;
    // mag << sh spans at most 138 bits: three 64-bit words {v2, v1, v0}, i.e. five 32-bit digits.
    const uint64_t lo = (uint64_t)mag, hi = (uint64_t)(mag >> 64);  // hi < 2^42
    const u128 low = (u128)lo << sh;                                // < 2^95, weight 2^0
    const u128 mid = (low >> 64) + ((u128)hi << sh);                // < 2^74, weight 2^64
    const uint64_t v0 = (uint64_t)low, v1 = (uint64_t)mid, v2 = (uint64_t)(mid >> 64);
    uint64_t d[5];
    d[0] = v0 & 0xffffffffULL;
    d[1] = v0 >> 32;
    d[2] = v1 & 0xffffffffULL;
    d[3] = v1 >> 32;
    d[4] = v2 & 0xffffffffULL;
    for (int t = 0; t < 5; t++) {
      if (sign > 0)
        w[idx + t] += (int64_t)d[t];
      else
        w[idx + t] -= (int64_t)d[t];
    }
    if (++pending >= (1 << 28)) normalize();
  }

  // Decompose a finite double: x = sign * mant * 2^e with mant < 2^53 an integer.
  static void decompose(double x, uint64_t* mant, int* e, int* sign) {
    uint64_t b;
    std::memcpy(&b, &x, 8);
    *sign = (b >> 63) ? -1 : 1;
    int be = (int)((b >> 52) & 0x7ff);
    uint64_t f = b & 0xfffffffffffffULL;
    if (be == 0) {
      *mant = f;
      *e = -1074;
    } else {
      *mant = f | (1ULL << 52);
      *e = be - 1075;
    }
  }

  void add_double(double x, int sgn = 1) {
    uint64_t m;
    int e, s;
    decompose(x, &m, &e, &s);
    add_scaled((u128)m, e, s * sgn);
  }

  void add_product(double a, double b, int sgn = 1) {
    uint64_t ma, mb;
    int ea, eb, sa, sb;
    decompose(a, &ma, &ea, &sa);
    decompose(b, &mb, &eb, &sb);
    add_scaled((u128)ma * (u128)mb, ea + eb, sa * sb * sgn);
  }

  // sign of the value (-1, 0, +1); normalises first.
  int signum() {
    normalize();
    if (w[NW - 1] < 0) return -1;
    for (int i = 0; i < NW; i++)
      if (w[i] != 0) return 1;
    return 0;
  }

  // Round to nearest double, ties to even (the value must be within double range).  Does not modify *this
  // except for normalisation.
  double to_double() {
    normalize();
    bool neg = w[NW - 1] < 0;
    // magnitude digits
    uint32_t mag[NW];
    if (!neg) {
      for (int i = 0; i < NW; i++) mag[i] = (uint32_t)w[i];
    } else {
      // two's complement negate of the NW-digit number (top word holds sign-extended value)
      uint64_t carry = 1;
      for (int i = 0; i < NW; i++) {
        uint32_t digit = (uint32_t)(w[i] & 0xffffffffLL);
        uint64_t v = (uint64_t)(uint32_t)(~digit) + carry;
        mag[i] = (uint32_t)v;
        carry = v >> 32;
      }
    }
    int top = -1;
    for (int i = NW - 1; i >= 0 && top < 0; i--)
      if (mag[i]) {
        int b = 31;
        while (!((mag[i] >> b) & 1)) b--;
        top = i * 32 + b;
      }
    if (top < 0) return 0.0;
    // lowest bit position we keep: 53 significant bits, but never below the subnormal grid 2^-1074
    int low = top - 52;
    int min_low = -1074 + BIAS;
    if (low < min_low) low = min_low;
    auto bit = [&](int p) -> int { return p < 0 ? 0 : (int)((mag[p >> 5] >> (p & 31)) & 1); };
    uint64_t m = 0;
    for (int p = top; p >= low; p--) m = (m << 1) | (uint64_t)bit(p);
    int round_bit = bit(low - 1);
    bool sticky = false;
    for (int p = low - 2; p >= 0 && !sticky; p--) {
      if ((p & 31) == 31 && mag[p >> 5] == 0) {
        p -= 31;
        continue;
      }
      if (bit(p)) sticky = true;
    }
    if (round_bit && (sticky || (m & 1))) m++;
    double r = std::ldexp((double)m, low - BIAS);  // exact: m <= 2^53, result representable
    return neg ? -r : r;
  }
};

// --- error-free transformations (textbook: Knuth TwoSum, Dekker FastTwoSum, TwoProd by fma; PAPER.md refs [2],[15]) ---
inline void two_sum(double a, double b, double* s, double* e) {
  double sum = a + b;
  double bb = sum - a;
  double err = (a - (sum - bb)) + (b - bb);
  *s = sum;
  *e = err;
}
inline void fast_two_sum(double a, double b, double* s, double* e) {  // needs |a| >= |b| or a == 0
  double sum = a + b;
  *e = b - (sum - a);
  *s = sum;
}
inline void two_prod(double a, double b, double* p, double* e) {
  double prod = a * b;
  *e = std::fma(a, b, -prod);
  *p = prod;
}

}  // namespace

extern "C" {

// =====================================================================================================
// O2 -- Algorithm S: exponent vectors and quarters.
//   PAPER.md:47-49 (section 2): the bits of a double are distributed over 13-bit parts, the quarters, with
//   exponents 0, -13, -26, -39 relative to the number; a double double gives 8 quarter matrices, the
//   quarters of the high double first; the exponents must lie on an equally spaced grid ("balanced");
//   PAPER.md:124-142 (section 3, eq. 7-8): bits are moved between neighbouring parts, without changing the value,
//   until every part sits on the grid; a zero part is an "unnormalized zero with the desired exponent".
//   Reading (R1, R2, R4; BASELINE.json north_star): the grid is common to a row of A (axis 0) or a column
//   of B (axis 1): E_g = ilogb(max |leading limb| over the group) + 1 and quarter q of every element of the group is
//   an integer multiple of u_q = 2^(E_g - 13(q+1)), the nearest one to what is left of the element (ties to even on
//   the leading remainder limb), so |digit| <= 2^13 for q = 0 and <= 2^12 after.  All operations are error free.
//
//   planes          [limbs][rows][cols]  fp64, input
//   quarter_planes  [quarters][rows][cols] fp64, output, true-valued quarters d_q = D_q * u_q
//   exps            int32[rows] (axis 0) or int32[cols] (axis 1), output
//   remainder       [limbs][rows][cols] or NULL: what is left after the last quarter (sum of quarters + remainder
//                   == element, exactly)
// =====================================================================================================
//   oracle_split_w: the same procedure with `bits` in place of 13 (R14: a slice of `bits` bits per part,
//   unit u_q = 2^(E_g - bits*(q+1)); the paper's quarter is bits = 13 = 52/4).
void oracle_split_w(int rows, int cols, int limbs, int quarters, int bits, int axis, const double* planes,
                    double* quarter_planes, int32_t* exps, double* remainder) {
  const size_t plane = (size_t)rows * cols;
  const int groups = axis == 0 ? rows : cols;
  // S0: the exponent of each scale group, from the leading limb only.
  for (int g = 0; g < groups; g++) {
    double M = 0.0;
    const int len = axis == 0 ? cols : rows;
    for (int t = 0; t < len; t++) {
      size_t at = axis == 0 ? (size_t)g * cols + t : (size_t)t * cols + g;
      double v = std::fabs(planes[at]);
      if (v > M) M = v;
    }
    exps[g] = (M == 0.0) ? 0 : std::ilogb(M) + 1;  // 2^(E-1) <= M < 2^E
  }
  // S1: per element, peel off one quarter at a time.
#pragma omp parallel for schedule(static)
  for (int i = 0; i < rows; i++) {
    std::vector<double> r(limbs);
    for (int j = 0; j < cols; j++) {
      const size_t at = (size_t)i * cols + j;
      const int E = exps[axis == 0 ? i : j];
      for (int l = 0; l < limbs; l++) r[l] = planes[l * plane + at];
      for (int q = 0; q < quarters; q++) {
        const double u = std::ldexp(1.0, E - bits * (q + 1));  // the unit of quarter q
        const double c = 6755399441055744.0 * u;            // 3 * 2^51 * u: ulp(c) == u, so r0 + c rounds r0 to a multiple of u
        const double t = r[0] + c;
        const double d = t - c;   // exact; the quarter
        r[0] = r[0] - d;          // exact; |r0| <= u/2 now
        for (int l = 0; l + 1 < limbs; l++) two_sum(r[l], r[l + 1], &r[l], &r[l + 1]);  // carry into the next limbs
        quarter_planes[(size_t)q * plane + at] = d;
      }
      if (remainder)
        for (int l = 0; l < limbs; l++) remainder[l * plane + at] = r[l];
    }
  }
}

void oracle_split(int rows, int cols, int limbs, int quarters, int axis, const double* planes,
                  double* quarter_planes, int32_t* exps, double* remainder) {
  oracle_split_w(rows, cols, limbs, quarters, 13, axis, planes, quarter_planes, exps, remainder);  // 13 bits
}

// =====================================================================================================
// O3 -- order matrices C^(s)[i,j] = sum_k sum_{p+q=s} A_p[i,k] * B_q[k,j], s = 0..orders-1 (the paper's C_{s+1}).
//   PAPER.md:66-71 eq. (3): "the convolutions with the sum of the last two indices ... equal to the index of the
//   quarter"; eq. (4): Cbar = [C_1 ... C_8] = Abar * Bbar with Bbar block upper triangular Toeplitz.
//   Two routes that must agree bit for bit (that IS the exactness claim of PAPER.md:51-54 and :95-99):
//   * oracle_orders_int: on the integer digits D = d / u in int64, scaled by 2^(E_i + F_j - 13(s+2)) at the end;
//   * oracle_orders_fp64: the same sums in plain fp64, k innermost, products in the order p = 0..s.
//   Aq [quarters][m][k], Bq [quarters][k][n], order_planes [orders][m][n] (true values).
// =====================================================================================================
//   The _w variants take the slice width `bits` (13 in the paper): unit of order s = 2^(E_i + F_j - bits*(s+2)).
void oracle_orders_int_w(int m, int n, int k, int quarters, int orders, int bits, const double* Aq, const int32_t* expA,
                         const double* Bq, const int32_t* expB, double* order_planes, int64_t* raw_sums) {
  const size_t pa = (size_t)m * k, pb = (size_t)k * n, pc = (size_t)m * n;
  // integer digits
  std::vector<int32_t> DA((size_t)quarters * pa), DB((size_t)quarters * pb);
  for (int q = 0; q < quarters; q++) {
    for (int i = 0; i < m; i++)
      for (int t = 0; t < k; t++)
        DA[q * pa + (size_t)i * k + t] = (int32_t)std::ldexp(Aq[q * pa + (size_t)i * k + t], -(expA[i] - bits * (q + 1)));
    for (int t = 0; t < k; t++)
      for (int j = 0; j < n; j++)
        DB[q * pb + (size_t)t * n + j] = (int32_t)std::ldexp(Bq[q * pb + (size_t)t * n + j], -(expB[j] - bits * (q + 1)));
  }
#pragma omp parallel for schedule(static)
  for (int i = 0; i < m; i++)
    for (int j = 0; j < n; j++)
      for (int s = 0; s < orders; s++) {
        int64_t acc = 0;
        for (int p = 0; p <= s; p++) {
          const int q = s - p;
          if (p >= quarters || q >= quarters) continue;
          for (int t = 0; t < k; t++)
            acc += (int64_t)DA[p * pa + (size_t)i * k + t] * (int64_t)DB[q * pb + (size_t)t * n + j];
        }
        if (raw_sums) raw_sums[s * pc + (size_t)i * n + j] = acc;
        // |acc| < 2^53 under the k-budget (R6), so the conversion and the scaling are exact.
        order_planes[s * pc + (size_t)i * n + j] = std::ldexp((double)acc, expA[i] + expB[j] - bits * (s + 2));
      }
}

void oracle_orders_int(int m, int n, int k, int quarters, int orders, const double* Aq, const int32_t* expA,
                       const double* Bq, const int32_t* expB, double* order_planes, int64_t* raw_sums) {
  oracle_orders_int_w(m, n, k, quarters, orders, 13, Aq, expA, Bq, expB, order_planes, raw_sums);
}

// The same integer route at sampled output positions only (for full-size matrices): out[t*orders + s] = C^(s)[si[t], sj[t]].
void oracle_orders_int_samples_w(int m, int n, int k, int quarters, int orders, int bits, const double* Aq,
                                 const int32_t* expA, const double* Bq, const int32_t* expB, int64_t nsamples,
                                 const int64_t* si, const int64_t* sj, double* out) {
  const size_t pa = (size_t)m * k, pb = (size_t)k * n;
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t t = 0; t < nsamples; t++) {
    const int64_t i = si[t], j = sj[t];
    for (int s = 0; s < orders; s++) {
      int64_t acc = 0;
      for (int p = 0; p <= s; p++) {
        const int q = s - p;
        if (p >= quarters || q >= quarters) continue;
        for (int kk = 0; kk < k; kk++) {
          const int64_t da = (int64_t)std::ldexp(Aq[p * pa + (size_t)i * k + kk], -(expA[i] - bits * (p + 1)));
          const int64_t db = (int64_t)std::ldexp(Bq[q * pb + (size_t)kk * n + j], -(expB[j] - bits * (q + 1)));
          acc += da * db;
        }
      }
      out[t * orders + s] = std::ldexp((double)acc, expA[i] + expB[j] - bits * (s + 2));
    }
  }
}

void oracle_orders_int_samples(int m, int n, int k, int quarters, int orders, const double* Aq, const int32_t* expA,
                               const double* Bq, const int32_t* expB, int64_t nsamples, const int64_t* si,
                               const int64_t* sj, double* out) {
  oracle_orders_int_samples_w(m, n, k, quarters, orders, 13, Aq, expA, Bq, expB, nsamples, si, sj, out);
}

void oracle_orders_fp64(int m, int n, int k, int quarters, int orders, const double* Aq, const double* Bq,
                        double* order_planes) {
  const size_t pa = (size_t)m * k, pb = (size_t)k * n, pc = (size_t)m * n;
#pragma omp parallel for schedule(static)
  for (int i = 0; i < m; i++)
    for (int j = 0; j < n; j++)
      for (int s = 0; s < orders; s++) {
        double acc = 0.0;
        for (int p = 0; p <= s; p++) {
          const int q = s - p;
          if (p >= quarters || q >= quarters) continue;
          for (int t = 0; t < k; t++) acc += Aq[p * pa + (size_t)i * k + t] * Bq[q * pb + (size_t)t * n + j];
        }
        order_planes[s * pc + (size_t)i * n + j] = acc;
      }
}

// =====================================================================================================
// O4 -- recombination.  PAPER.md:88-91 steps 4-5: "Add the parts of the product into a double double matrix ...
//   summing 8 doubles into one double double for each element".  The oracle's result is the plain definition: the
//   exact sum of the `orders` values, rounded to `limbs` limbs one after another, limb_l = RN(sum - limb_0 - ... -
//   limb_{l-1}).  Several results are acceptable for an implementation (R9); this one is the best possible.
// =====================================================================================================
void oracle_renorm(int m, int n, int limbs, int orders, const double* order_planes, double* C_planes) {
  const size_t pc = (size_t)m * n;
#pragma omp parallel for schedule(static)
  for (int i = 0; i < m; i++) {
    LongAcc acc;
    for (int j = 0; j < n; j++) {
      const size_t at = (size_t)i * n + j;
      acc.clear();
      for (int s = 0; s < orders; s++) acc.add_double(order_planes[s * pc + at]);
      for (int l = 0; l < limbs; l++) {
        const double v = acc.to_double();
        C_planes[l * pc + at] = v;
        acc.add_double(v, -1);
      }
    }
  }
}

// =====================================================================================================
// O1 -- the exact product (the plain definition of what the whole path must reach).
//   a_ik = sum_l A_l[i,k], b_kj = sum_l B_l[k,j] (Definition 1.1: a multiple double is the unevaluated
//   sum of its doubles); C_exact[i,j] = sum_k a_ik * b_kj, W[i,j] = sum_k |a_ik| |b_kj| = (|A||B|)_ij, all exact.
//   For each sampled position (si[t], sj[t]):
//     Cexact_limbs[t*out_limbs + l]  the exact value rounded to out_limbs limbs (if not NULL)
//     W[t]                            (|A||B|)_ij rounded to double (if not NULL)
//     err[t]                          | sum_l C_l[i,j] - C_exact[i,j] | evaluated exactly, then rounded (if C not NULL)
//   A [limbs][m][k], B [limbs][k][n], C [limbs][m][n].
// =====================================================================================================
void oracle_exact_samples(int m, int n, int k, int limbs, const double* A, const double* B, const double* C,
                          int64_t nsamples, const int64_t* si, const int64_t* sj, double* err, double* W,
                          double* Cexact_limbs, int out_limbs) {
  const size_t pa = (size_t)m * k, pb = (size_t)k * n, pc = (size_t)m * n;
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t t = 0; t < nsamples; t++) {
    const int64_t i = si[t], j = sj[t];
    LongAcc acc, wacc, aabs, babs;
    for (int kk = 0; kk < k; kk++) {
      for (int la = 0; la < limbs; la++)
        for (int lb = 0; lb < limbs; lb++)
          acc.add_product(A[la * pa + (size_t)i * k + kk], B[lb * pb + (size_t)kk * n + j]);
      if (W) {
        // |a_ik| * |b_kj| = sign(a) sign(b) * a * b with the signs of the exact sums of limbs
        aabs.clear();
        babs.clear();
        for (int la = 0; la < limbs; la++) aabs.add_double(A[la * pa + (size_t)i * k + kk]);
        for (int lb = 0; lb < limbs; lb++) babs.add_double(B[lb * pb + (size_t)kk * n + j]);
        const int sg = aabs.signum() * babs.signum();
        if (sg != 0)
          for (int la = 0; la < limbs; la++)
            for (int lb = 0; lb < limbs; lb++)
              wacc.add_product(A[la * pa + (size_t)i * k + kk], B[lb * pb + (size_t)kk * n + j], sg);
      }
    }
    if (W) W[t] = wacc.to_double();
    if (Cexact_limbs) {
      LongAcc tmp = acc;
      for (int l = 0; l < out_limbs; l++) {
        const double v = tmp.to_double();
        Cexact_limbs[t * out_limbs + l] = v;
        tmp.add_double(v, -1);
      }
    }
    if (C && err) {
      for (int l = 0; l < limbs; l++) acc.add_double(C[l * pc + (size_t)i * n + j], -1);
      err[t] = std::fabs(acc.to_double());
    }
  }
}

// Exact sum of `count` doubles rounded to `limbs` limbs (used by tests to examine the accumulator itself).
void oracle_exact_sum(int count, const double* x, int limbs, double* out) {
  LongAcc acc;
  for (int i = 0; i < count; i++) acc.add_double(x[i]);
  for (int l = 0; l < limbs; l++) {
    out[l] = acc.to_double();
    acc.add_double(out[l], -1);
  }
}

// Exact dot product sum_i x[i]*y[i] rounded to `limbs` limbs.
void oracle_exact_dot(int count, const double* x, const double* y, int limbs, double* out) {
  LongAcc acc;
  for (int i = 0; i < count; i++) acc.add_product(x[i], y[i]);
  for (int l = 0; l < limbs; l++) {
    out[l] = acc.to_double();
    acc.add_double(out[l], -1);
  }
}

// =====================================================================================================
// O5 -- classical multiple-double GEMM, "a single thread executes an inner product" in multiple-double arithmetic on
//   regular cores (the paper's C_CUDA of eq. 9).  Built from the textbook error-free transformations
//   only (refs [2], [3], [15]: TwoSum, FastTwoSum, TwoProd): every partial product a_la * b_lb with la + lb < limbs
//   is formed exactly by TwoProd, those with la + lb == limbs in plain fp64, and each term is added into a
//   (limbs+1)-term accumulator by a TwoSum cascade, followed by a renormalising sweep.  Its own error is about
//   k * 2^-(53*limbs - 2) * (|A||B|)_ij, so it is a cross-check with that threshold, not the ground truth.
// =====================================================================================================
static void md_cascade_add(double* acc, int terms, double x) {
  for (int l = 0; l < terms; l++) two_sum(acc[l], x, &acc[l], &x);  // what is left in x is below the last term
}
static void md_renormalise(double* acc, int terms) {
  // bottom-up then top-down sweep of FastTwoSum/TwoSum: leaves a non-overlapping, decreasing expansion
  for (int l = terms - 1; l > 0; l--) two_sum(acc[l - 1], acc[l], &acc[l - 1], &acc[l]);
  for (int l = 0; l + 1 < terms; l++) two_sum(acc[l], acc[l + 1], &acc[l], &acc[l + 1]);
}

void oracle_classic_gemm(int m, int n, int k, int limbs, const double* A, const double* B, double* C) {
  const size_t pa = (size_t)m * k, pb = (size_t)k * n, pc = (size_t)m * n;
  const int terms = limbs + 1;
#pragma omp parallel for schedule(static)
  for (int i = 0; i < m; i++) {
    std::vector<double> acc(terms);
    for (int j = 0; j < n; j++) {
      for (int l = 0; l < terms; l++) acc[l] = 0.0;
      for (int kk = 0; kk < k; kk++) {
        for (int la = 0; la < limbs; la++)
          for (int lb = 0; la + lb <= limbs && lb < limbs; lb++) {
            const double a = A[la * pa + (size_t)i * k + kk], b = B[lb * pb + (size_t)kk * n + j];
            if (la + lb < limbs) {
              double p, e;
              two_prod(a, b, &p, &e);
              md_cascade_add(acc.data(), terms, p);
              md_cascade_add(acc.data(), terms, e);
            } else {
              md_cascade_add(acc.data(), terms, a * b);
            }
          }
        md_renormalise(acc.data(), terms);
      }
      for (int l = 0; l < limbs; l++) C[l * pc + (size_t)i * n + j] = acc[l];
    }
  }
}

// =====================================================================================================
// The paper's five steps end to end: split -> (rewrite) -> quarter products -> (extract) -> add the
// parts.  Steps 2 and 4 are index bookkeeping only (Abar/Bbar are never stored).  Computes rows [row0,row1) of C
// into C_rows [limbs][row1-row0][n]; B's quarters are computed for the whole of B every call.
// =====================================================================================================
void oracle_md_gemm_rows_w(int m, int n, int k, int limbs, int quarters, int orders, int bits, const double* A,
                           const double* B, int row0, int row1, double* C_rows) {
  const int mr = row1 - row0;
  std::vector<double> Arows((size_t)limbs * mr * k);
  for (int l = 0; l < limbs; l++)
    std::memcpy(&Arows[(size_t)l * mr * k], &A[(size_t)l * m * k + (size_t)row0 * k], sizeof(double) * (size_t)mr * k);
  std::vector<double> Aq((size_t)quarters * mr * k), Bq((size_t)quarters * k * n), ord((size_t)orders * mr * n);
  std::vector<int32_t> eA(mr), eB(n);
  oracle_split_w(mr, k, limbs, quarters, bits, 0, Arows.data(), Aq.data(), eA.data(), nullptr);
  oracle_split_w(k, n, limbs, quarters, bits, 1, B, Bq.data(), eB.data(), nullptr);
  oracle_orders_fp64(mr, n, k, quarters, orders, Aq.data(), Bq.data(), ord.data());
  oracle_renorm(mr, n, limbs, orders, ord.data(), C_rows);
}

void oracle_md_gemm_rows(int m, int n, int k, int limbs, int quarters, int orders, const double* A, const double* B,
                         int row0, int row1, double* C_rows) {
  oracle_md_gemm_rows_w(m, n, k, limbs, quarters, orders, 13, A, B, row0, row1, C_rows);
}

// Chunked accumulation (R16): the contraction is cut into chunks of `chunk` indices; inside a chunk the order sums
// are formed exactly as above (the budget k S 2^(2 bits) <= 2^53 now only has to hold for chunk in place of k), and the
// parts of ALL chunks -- orders * ceil(k / chunk) doubles per element -- are added into the multiple-double result
// (here by the exact sum of oracle_renorm).  chunk >= k is oracle_md_gemm_rows_w.
void oracle_md_gemm_rows_chunked_w(int m, int n, int k, int limbs, int quarters, int orders, int bits, int chunk,
                                   const double* A, const double* B, int row0, int row1, double* C_rows) {
  const int mr = row1 - row0;
  std::vector<double> Arows((size_t)limbs * mr * k);
  for (int l = 0; l < limbs; l++)
    std::memcpy(&Arows[(size_t)l * mr * k], &A[(size_t)l * m * k + (size_t)row0 * k], sizeof(double) * (size_t)mr * k);
  std::vector<double> Aq((size_t)quarters * mr * k), Bq((size_t)quarters * k * n);
  std::vector<int32_t> eA(mr), eB(n);
  oracle_split_w(mr, k, limbs, quarters, bits, 0, Arows.data(), Aq.data(), eA.data(), nullptr);
  oracle_split_w(k, n, limbs, quarters, bits, 1, B, Bq.data(), eB.data(), nullptr);
  const int nchunks = (k + chunk - 1) / chunk;
  std::vector<double> ord((size_t)nchunks * orders * mr * n);
  for (int c = 0; c < nchunks; c++) {
    const int k0 = c * chunk, kc = (k0 + chunk <= k ? chunk : k - k0);
    // the quarter planes of this chunk: columns [k0, k0 + kc) of A's, rows [k0, k0 + kc) of B's
    std::vector<double> Ac((size_t)quarters * mr * kc), Bc((size_t)quarters * kc * n);
    for (int q = 0; q < quarters; q++) {
      for (int i = 0; i < mr; i++)
        std::memcpy(&Ac[((size_t)q * mr + i) * kc], &Aq[((size_t)q * mr + i) * k + k0], sizeof(double) * (size_t)kc);
      std::memcpy(&Bc[(size_t)q * kc * n], &Bq[((size_t)q * k + k0) * n], sizeof(double) * (size_t)kc * n);
    }
    oracle_orders_fp64(mr, n, kc, quarters, orders, Ac.data(), Bc.data(), &ord[(size_t)c * orders * mr * n]);
  }
  oracle_renorm(mr, n, limbs, nchunks * orders, ord.data(), C_rows);
}

// =====================================================================================================
// O6 -- the paper's OWN balancing, element by element (section 3; R17-R22).
//   The path of O2 gives a row of A / a column of B a common exponent (BASELINE.json north_star).  Section 3 of the paper
//   instead works on single numbers and on the whole matrix:
//     * PAPER.md:47-49   each double is cut into 4 parts of 13 bits relative to ITS OWN exponent          (R17)
//     * PAPER.md:124-131 eq. (7): hi and lo of opposite sign -> take one ulp from hi and give it to lo     (R18)
//     * PAPER.md:133-140 eq. (8): a part with leading zeros borrows half a unit of the part above it       (R19)
//     * PAPER.md:142     a zero part keeps "the desired exponent": do nothing                              (R19)
//     * PAPER.md:120-122 A = A_0 + ... + A_12 by the exponent of the leading quarter (mod 13), "execute many
//                        matrix multiplications"                                                           (R20)
//     * PAPER.md:107-118 eq. (6): A = A_+ + A_-, four sign-pair products                                   (R21)
//   Everything below follows those passages step by step; every move is value invariant (pinned in exact rationals).
// =====================================================================================================

// R17: x = +-2^e (1.f0 f1 f2 f3), four fields of 13 bits; quarters x_0 = +-2^e (1 + f0 2^-13),
// x_t = +-f_t 2^(e - 13 (t+1)), t = 1, 2, 3 -- "exponents 0, -13, -26, -39".  Plain bit fields; x_0 + x_1 + x_2 + x_3 == x.
void oracle_quarter_double(double x, double* out4) {
  out4[0] = out4[1] = out4[2] = out4[3] = 0.0;
  if (x == 0.0) return;
  int ex;
  const double mant = std::frexp(std::fabs(x), &ex);      // |x| = mant 2^ex, mant in [1/2, 1)
  const uint64_t M = (uint64_t)std::ldexp(mant, 53);        // 53-bit integer, bit 52 = the hidden bit
  const int e = ex - 1;                                     // |x| = 2^e (1.f)
  const uint64_t f = M - (1ULL << 52);
  const double sign = x < 0 ? -1.0 : 1.0;
  out4[0] = sign * std::ldexp((double)((1ULL << 13) + (f >> 39)), e - 13);
  out4[1] = sign * std::ldexp((double)((f >> 26) & 8191), e - 26);
  out4[2] = sign * std::ldexp((double)((f >> 13) & 8191), e - 39);
  out4[3] = sign * std::ldexp((double)(f & 8191), e - 52);
}

static inline double ulp_of(double x) { return std::ldexp(1.0, std::ilogb(x) - 52); }

// R18, eq. (7) for a multiple double x[0..limbs-1]: wherever a limb and the next one have opposite signs,
// b := one ulp of the upper limb (with its sign); upper -= b; lower += b.  The paper's b = 2^-52 assumes |lower| below one ulp
// of upper; after a borrow further up a limb can have shrunk by cancellation, so in general b = the smallest power of two that
// is at least one ulp of upper AND exceeds |lower| (one ulp for a normalised pair), which makes lower + b take upper's sign.
// "the last bit should then be added to the next double in the sequence ... using multiple double arithmetic": the rounding
// error of lower + b is carried down by TwoSum; what falls off the last limb is returned in carry[l] (exact).  Value
// invariant: sum x + sum carry is unchanged.  A pair that is not even weakly normalised (b would exceed |upper| / 2) is left.
void oracle_eq7(int limbs, double* x, double* carry) {
  for (int l = 0; l < limbs; l++) carry[l] = 0.0;
  for (int l = 0; l + 1 < limbs; l++) {
    if (x[l] == 0.0 || x[l + 1] == 0.0 || ((x[l] < 0) == (x[l + 1] < 0))) continue;
    double mag = ulp_of(x[l]);
    const double above = std::ldexp(1.0, std::ilogb(x[l + 1]) + 1);  // the power of two just above |lower|
    if (above > mag) mag = above;
    if (mag > 0.5 * std::fabs(x[l])) continue;
    const double b = std::copysign(mag, x[l]);
    x[l] = x[l] - b;  // exact: x[l] is a multiple of its ulp, b a multiple of that ulp below |x[l]|
    double c = b;
    for (int j = l + 1; j < limbs; j++) two_sum(x[j], c, &x[j], &c);
    carry[l] = c;
  }
}

// R19, eq. (8) on the quarters d[0..Q-1] of ONE element whose quarter q sits on the unit u_q = 2^(e - 13 (q+1)):
// top down, if quarter q+1 has leading zeros (|d_{q+1}| < 2^12 u_{q+1}: its exponent is below the grid) it borrows
// b = 2^12 u_{q+1} (the paper's b = 2^-14 for q = 0, e = 0) from quarter q: d_q -= b; d_{q+1} += b.  A zero quarter "keeps the
// desired exponent: do nothing"; a quarter lends only if that "does not alter [its] exponent" (PAPER.md:137:
// q = 0, or more than 2^12 units).  Afterwards d_q is a multiple of u_q / 2.  Value invariant.
void oracle_eq8(int Q, int e, double* d) {
  for (int q = 0; q + 1 < Q; q++) {
    const double u_next = std::ldexp(1.0, e - 13 * (q + 2));
    const double top = 4096.0 * u_next;  // 2^12 u_{q+1} = u_q / 2
    if (d[q + 1] == 0.0 || std::fabs(d[q + 1]) >= top) continue;
    if (d[q] == 0.0 || ((d[q] < 0) != (d[q + 1] < 0))) continue;
    if (q > 0 && std::fabs(d[q]) <= 2.0 * top * 4096.0) continue;  // lender must keep its top bit: more than 2^12 units of u_q
    const double b = std::copysign(top, d[q]);
    d[q] -= b;
    d[q + 1] += b;
  }
}

// Algorithm L: the literal split of one element (limbs x[0..limbs-1]) into `quarters` parts on the element's OWN grid.
//   L1  eq. (7): all limbs get one sign (oracle_eq7)
//   L2  e = ilogb of the leading non-zero limb: the element's exponent (the paper's "exponent of the leading quarter")
//   L3  for q = 0 .. quarters-1: u_q = 2^(e - 13 (q+1)); part q = sum over the limbs of the bits of that limb at or above u_q
//       (truncation toward zero of what is left of each limb: the paper's bit fields, R17, re-cut on the element's grid),
//       and those bits are taken off the limbs.  Exact: every piece is a multiple of u_q below 2^14 u_q.
//   L4  eq. (8) (oracle_eq8), if apply_eq8
//   d[q] = the quarters (true values); rem[0..limbs-1] = what is left of the limbs, rem[limbs..2 limbs-1] = eq. (7) carries:
//   sum d + sum rem == sum x exactly.  Returns e (0 for a zero element).
int oracle_split_literal_element(int limbs, int quarters, int apply_eq8, const double* x_in, double* d, double* rem) {
  std::vector<double> x(x_in, x_in + limbs), carry(limbs);
  oracle_eq7(limbs, x.data(), carry.data());
  int lead = 0;
  while (lead < limbs && x[lead] == 0.0) lead++;
  for (int q = 0; q < quarters; q++) d[q] = 0.0;
  int e = 0;
  if (lead < limbs) {
    e = std::ilogb(x[lead]);
    for (int q = 0; q < quarters; q++) {
      const int s = e - 13 * (q + 1);
      double part = 0.0;
      for (int l = 0; l < limbs; l++) {
        const double piece = std::ldexp(std::trunc(std::ldexp(x[l], -s)), s);  // the bits of limb l at or above 2^s
        x[l] -= piece;                                                            // exact
        part += piece;                                                            // exact: multiples of 2^s below 2^(s+14)
      }
      d[q] = part;
    }
    if (apply_eq8) oracle_eq8(quarters, e, d);
  }
  if (rem) {
    for (int l = 0; l < limbs; l++) rem[l] = x[l];
    for (int l = 0; l < limbs; l++) rem[limbs + l] = carry[l];
  }
  return e;
}

// The whole matrix: quarter_planes [quarters][rows][cols], exps int32[rows*cols] (per ELEMENT), remainder [2*limbs][rows][cols] or NULL.
void oracle_split_literal(int rows, int cols, int limbs, int quarters, int apply_eq8, const double* planes,
                          double* quarter_planes, int32_t* exps, double* remainder) {
  const size_t plane = (size_t)rows * cols;
#pragma omp parallel for schedule(static)
  for (int i = 0; i < rows; i++) {
    std::vector<double> x(limbs), d(quarters), rem(2 * limbs);
    for (int j = 0; j < cols; j++) {
      const size_t at = (size_t)i * cols + j;
      for (int l = 0; l < limbs; l++) x[l] = planes[l * plane + at];
      exps[at] = oracle_split_literal_element(limbs, quarters, apply_eq8, x.data(), d.data(), rem.data());
      for (int q = 0; q < quarters; q++) quarter_planes[(size_t)q * plane + at] = d[q];
      if (remainder)
        for (int l = 0; l < 2 * limbs; l++) remainder[(size_t)l * plane + at] = rem[l];
    }
  }
}

static inline int floor_div13(int e) { return (e >= 0) ? e / 13 : -((-e + 12) / 13); }

// R20-R22: the literal product.  Every element has its class c = e mod 13 ("the index is the exponent of the
// leading quarter", 13 possible values on a grid of spacing 13) and its level z = floor(e / 13); A = A_0 + ... + A_12,
// B likewise, and A B = sum over the 169 class pairs of A_c B_d ("execute many matrix multiplications").  Inside a class all
// parts of all elements lie on ONE grid 2^(c + 13 Z), so part q of an element of level z is part P = q + (zmax - z) of its
// class matrix on the common grid anchored at zmax (R20), and the class-pair product is an ordinary quarter product whose
// order t = P + P' collects terms of ONE unit 2^(c + d + 13 (zmaxA + zmaxB) - 13 (t + 2)): exact accumulations, as in
// PAPER.md:95-99.  Kept orders: t < quarters + spanA + spanB (span = zmax - zmin over the non-zero elements), i.e. every
// product p + q < quarters of every element pair and whatever else shares its order.  With sign_groups (eq. 6)
// every class is further cut into its positive and its negative elements: four sign-pair products per class pair, each a sum of
// terms of one sign.  C = all order sums of all pairs added into `limbs` limbs (here: exactly, then rounded limb by limb).
//   info[0..5] (if not NULL) = zminA, zmaxA, zminB, zmaxB, planes per class matrix of A / of B is quarters + span.
void oracle_md_gemm_literal(int m, int n, int k, int limbs, int quarters, int apply_eq8, int sign_groups, const double* A,
                            const double* B, double* C, int32_t* info) {
  const size_t pa = (size_t)m * k, pb = (size_t)k * n, pc = (size_t)m * n;
  std::vector<double> Aq((size_t)quarters * pa), Bq((size_t)quarters * pb);
  std::vector<int32_t> eA(pa), eB(pb);
  oracle_split_literal(m, k, limbs, quarters, apply_eq8, A, Aq.data(), eA.data(), nullptr);
  oracle_split_literal(k, n, limbs, quarters, apply_eq8, B, Bq.data(), eB.data(), nullptr);
  auto nonzero = [&](const std::vector<double>& Xq, size_t plane, size_t at) {
    for (int q = 0; q < quarters; q++)
      if (Xq[(size_t)q * plane + at] != 0.0) return true;
    return false;
  };
  int zminA = 1 << 30, zmaxA = -(1 << 30), zminB = 1 << 30, zmaxB = -(1 << 30);
  for (size_t at = 0; at < pa; at++)
    if (nonzero(Aq, pa, at)) zminA = std::min(zminA, floor_div13(eA[at])), zmaxA = std::max(zmaxA, floor_div13(eA[at]));
  for (size_t at = 0; at < pb; at++)
    if (nonzero(Bq, pb, at)) zminB = std::min(zminB, floor_div13(eB[at])), zmaxB = std::max(zmaxB, floor_div13(eB[at]));
  if (zmaxA < zminA) zminA = zmaxA = 0;
  if (zmaxB < zminB) zminB = zmaxB = 0;
  if (info) info[0] = zminA, info[1] = zmaxA, info[2] = zminB, info[3] = zmaxB;
  const int orders = quarters + (zmaxA - zminA) + (zmaxB - zminB);
  const int groups = sign_groups ? 26 : 13;  // group id = class (+ 13 for a negative element)
#pragma omp parallel for schedule(static)
  for (int i = 0; i < m; i++) {
    std::vector<int64_t> acc((size_t)groups * groups * orders);
    LongAcc sum;
    for (int j = 0; j < n; j++) {
      std::fill(acc.begin(), acc.end(), 0);
      for (int t = 0; t < k; t++) {
        const size_t aa = (size_t)i * k + t, bb = (size_t)t * n + j;
        const int ea = eA[aa], eb = eB[bb];
        const int ca = ((ea % 13) + 13) % 13, cb = ((eb % 13) + 13) % 13;
        const int za = floor_div13(ea), zb = floor_div13(eb);
        int ga = ca, gb = cb;
        if (sign_groups) {  // the sign of an element = the sign of its parts (all equal after eq. 7)
          for (int q = 0; q < quarters; q++)
            if (Aq[(size_t)q * pa + aa] != 0.0) { if (Aq[(size_t)q * pa + aa] < 0) ga += 13; break; }
          for (int q = 0; q < quarters; q++)
            if (Bq[(size_t)q * pb + bb] != 0.0) { if (Bq[(size_t)q * pb + bb] < 0) gb += 13; break; }
        }
        for (int p = 0; p < quarters; p++) {
          // integer digit of part p in HALF units (eq. 8 leaves multiples of u / 2): D = d / 2^(e - 13 (p+1) - 1)
          const int64_t Da = (int64_t)std::ldexp(Aq[(size_t)p * pa + aa], -(ea - 13 * (p + 1) - 1));
          if (Da == 0) continue;
          const int P = p + (zmaxA - za);
          for (int q = 0; q < quarters; q++) {
            const int ord = P + q + (zmaxB - zb);
            if (ord >= orders) break;
            const int64_t Db = (int64_t)std::ldexp(Bq[(size_t)q * pb + bb], -(eb - 13 * (q + 1) - 1));
            acc[((size_t)ga * groups + gb) * orders + ord] += Da * Db;
          }
        }
      }
      // every order sum is an exact double (|acc| < 2^53 under the budget k * orders * 2^30 <= 2^53); add them all, exactly
      sum.clear();
      for (int ga = 0; ga < groups; ga++)
        for (int gb = 0; gb < groups; gb++)
          for (int ord = 0; ord < orders; ord++) {
            const int64_t v = acc[((size_t)ga * groups + gb) * orders + ord];
            if (v == 0) continue;
            // unit of the sum: 2^(ca + cb + 13 (zmaxA + zmaxB) - 13 (ord + 2)) / 4
            const int ex = (ga % 13) + (gb % 13) + 13 * (zmaxA + zmaxB) - 13 * (ord + 2) - 2;
            sum.add_double(std::ldexp((double)v, ex));
          }
      for (int l = 0; l < limbs; l++) {
        const double v = sum.to_double();
        C[l * pc + (size_t)i * n + j] = v;
        sum.add_double(v, -1);
      }
    }
  }
}

// =====================================================================================================
// O7 -- Householder QR in multiple-double arithmetic, the "second workload" the paper names as future work
//   ("apply this multiple double tensor core matrix multiplication to accelerate the blocked Householder QR,
//   extending [18]"; ref [18] PAPER.md:235, least squares on GPUs in multiple double precision).
//   The oracle is the plain UNBLOCKED algorithm (one reflection per column, applied column by column), every scalar operation
//   in multiple-double arithmetic built from the textbook error-free transformations of O5 (refs [2], [3], [15]):
//     mdx_add   (L+1)-term TwoSum cascade, renormalised
//     mdx_mul   partial products a_i b_j with i + j < L by TwoProd, those with i + j = L in plain fp64, cascaded
//     mdx_div   long division: L + 1 quotient digits q_i = r_0 / b_0, r -= q_i b
//     mdx_sqrt  Heron's iteration x <- (x + a / x) / 2 from the double-precision root
//   A = Q R, A m x n (m >= n), Q m x n with orthonormal columns, R n x n upper triangular with diag(R) >= 0 (the sign of every
//   row of R / column of Q is fixed that way, which makes the factorisation of a full-rank A unique).
// =====================================================================================================
namespace {

void mdx_renorm(int terms, double* acc) {
  for (int l = terms - 1; l > 0; l--) two_sum(acc[l - 1], acc[l], &acc[l - 1], &acc[l]);
  for (int sweep = 0; sweep + 1 < terms; sweep++)
    for (int l = 0; l + 1 < terms; l++) two_sum(acc[l], acc[l + 1], &acc[l], &acc[l + 1]);
}
void mdx_add(int L, const double* a, const double* b, double* out, double sign_b = 1.0) {
  std::vector<double> acc(L + 1, 0.0);
  for (int l = 0; l < L; l++) acc[l] = a[l];
  for (int l = L - 1; l >= 0; l--) md_cascade_add(acc.data(), L + 1, sign_b * b[l]);
  mdx_renorm(L + 1, acc.data());
  for (int l = 0; l < L; l++) out[l] = acc[l];
}
void mdx_mul(int L, const double* a, const double* b, double* out) {
  std::vector<double> acc(L + 1, 0.0);
  for (int s = L; s >= 0; s--)  // smallest partial products first
    for (int la = 0; la < L; la++) {
      const int lb = s - la;
      if (lb < 0 || lb >= L) continue;
      if (s < L) {
        double p, e;
        two_prod(a[la], b[lb], &p, &e);
        md_cascade_add(acc.data(), L + 1, e);
        md_cascade_add(acc.data(), L + 1, p);
      } else {
        md_cascade_add(acc.data(), L + 1, a[la] * b[lb]);
      }
    }
  mdx_renorm(L + 1, acc.data());
  for (int l = 0; l < L; l++) out[l] = acc[l];
}
void mdx_div(int L, const double* a, const double* b, double* out) {
  std::vector<double> r(a, a + L), q(L + 1, 0.0), qb(L), t(L);
  for (int i = 0; i <= L; i++) {
    q[i] = r[0] / b[0];
    std::fill(t.begin(), t.end(), 0.0);
    t[0] = q[i];
    mdx_mul(L, t.data(), b, qb.data());
    mdx_add(L, r.data(), qb.data(), r.data(), -1.0);
  }
  mdx_renorm(L + 1, q.data());
  for (int l = 0; l < L; l++) out[l] = q[l];
}
void mdx_sqrt(int L, const double* a, double* out) {
  std::fill(out, out + L, 0.0);
  if (a[0] <= 0.0) return;
  std::vector<double> x(L, 0.0), t(L);
  x[0] = std::sqrt(a[0]);
  int iters = 2;
  for (int l = 1; l < L; l *= 2) iters++;
  for (int it = 0; it < iters; it++) {
    mdx_div(L, a, x.data(), t.data());
    mdx_add(L, x.data(), t.data(), x.data());
    for (int l = 0; l < L; l++) x[l] *= 0.5;
  }
  for (int l = 0; l < L; l++) out[l] = x[l];
}

}  // namespace

// test access to the four scalar operations (a, b, out: `limbs` doubles each); op: 0 add, 1 sub, 2 mul, 3 div, 4 sqrt(a)
void oracle_mdx_op(int limbs, int op, const double* a, const double* b, double* out) {
  switch (op) {
    case 0: mdx_add(limbs, a, b, out); break;
    case 1: mdx_add(limbs, a, b, out, -1.0); break;
    case 2: mdx_mul(limbs, a, b, out); break;
    case 3: mdx_div(limbs, a, b, out); break;
    default: mdx_sqrt(limbs, a, out); break;
  }
}

// A [limbs][m][n] -> Q [limbs][m][n], R [limbs][n][n].  Reflections as in the textbook (Golub & Van Loan alg. 5.1.1 / LAPACK
// dgeqr2): for column j, alpha = A_jj, sigma = sum_{i>j} A_ij^2, beta = -sign(alpha) sqrt(alpha^2 + sigma), tau = (beta - alpha) /
// beta, v = (1, A_{j+1:,j} / (alpha - beta)); H_j = I - tau v v^T; R_jj = beta.  Q = H_0 H_1 ... H_{n-1} applied to the first n
// columns of I, backwards.  Finally the signs: R_jj < 0 => row j of R and column j of Q are negated.
void oracle_md_qr(int m, int n, int limbs, const double* A, double* Q, double* R) {
  const int L = limbs;
  const size_t pa = (size_t)m * n, pr = (size_t)n * n;
  std::vector<double> W((size_t)L * pa);  // working copy: R above the diagonal, v below
  std::memcpy(W.data(), A, sizeof(double) * (size_t)L * pa);
  std::vector<double> tau((size_t)n * L, 0.0);
  auto get = [&](const std::vector<double>& X, size_t plane, size_t at, double* out) {
    for (int l = 0; l < L; l++) out[l] = X[l * plane + at];
  };
  auto put = [&](std::vector<double>& X, size_t plane, size_t at, const double* in) {
    for (int l = 0; l < L; l++) X[l * plane + at] = in[l];
  };
  std::vector<double> a(L), b(L), c(L), d(L), alpha(L), beta(L), sigma(L), w(L), one(L, 0.0), zero(L, 0.0);
  one[0] = 1.0;
  for (int j = 0; j < n; j++) {
    get(W, pa, (size_t)j * n + j, alpha.data());
    std::fill(sigma.begin(), sigma.end(), 0.0);
    for (int i = j + 1; i < m; i++) {
      get(W, pa, (size_t)i * n + j, a.data());
      mdx_mul(L, a.data(), a.data(), b.data());
      mdx_add(L, sigma.data(), b.data(), sigma.data());
    }
    double* tj = &tau[(size_t)j * L];
    if (sigma[0] == 0.0) {  // nothing below the diagonal: H = I (the sign of R_jj is fixed at the end)
      std::fill(tj, tj + L, 0.0);
      continue;
    }
    mdx_mul(L, alpha.data(), alpha.data(), b.data());
    mdx_add(L, b.data(), sigma.data(), b.data());
    mdx_sqrt(L, b.data(), beta.data());
    if (alpha[0] >= 0.0)
      for (int l = 0; l < L; l++) beta[l] = -beta[l];
    mdx_add(L, beta.data(), alpha.data(), c.data(), -1.0);  // beta - alpha
    mdx_div(L, c.data(), beta.data(), tj);                  // tau
    mdx_add(L, alpha.data(), beta.data(), c.data(), -1.0);  // alpha - beta
    for (int i = j + 1; i < m; i++) {
      get(W, pa, (size_t)i * n + j, a.data());
      mdx_div(L, a.data(), c.data(), b.data());
      put(W, pa, (size_t)i * n + j, b.data());
    }
    put(W, pa, (size_t)j * n + j, beta.data());
    // apply H_j to the columns to the right: w = v^T a_c, a_c -= tau w v
#pragma omp parallel for schedule(static) firstprivate(a, b, c, d, w)
    for (int col = j + 1; col < n; col++) {
      get(W, pa, (size_t)j * n + col, w.data());
      for (int i = j + 1; i < m; i++) {
        get(W, pa, (size_t)i * n + j, a.data());
        get(W, pa, (size_t)i * n + col, b.data());
        mdx_mul(L, a.data(), b.data(), c.data());
        mdx_add(L, w.data(), c.data(), w.data());
      }
      mdx_mul(L, tj, w.data(), d.data());  // tau w
      get(W, pa, (size_t)j * n + col, b.data());
      mdx_add(L, b.data(), d.data(), b.data(), -1.0);
      put(W, pa, (size_t)j * n + col, b.data());
      for (int i = j + 1; i < m; i++) {
        get(W, pa, (size_t)i * n + j, a.data());
        mdx_mul(L, a.data(), d.data(), c.data());
        get(W, pa, (size_t)i * n + col, b.data());
        mdx_add(L, b.data(), c.data(), b.data(), -1.0);
        put(W, pa, (size_t)i * n + col, b.data());
      }
    }
  }
  // R
  std::vector<double> Rv((size_t)L * pr, 0.0), Qv((size_t)L * pa, 0.0);
  for (int i = 0; i < n; i++)
    for (int col = i; col < n; col++)
      for (int l = 0; l < L; l++) Rv[l * pr + (size_t)i * n + col] = W[l * pa + (size_t)i * n + col];
  // Q = H_0 ... H_{n-1} I_{m x n}: apply the reflections backwards to the identity
  for (int i = 0; i < n; i++) Qv[(size_t)i * n + i] = 1.0;
  for (int j = n - 1; j >= 0; j--) {
    const double* tj = &tau[(size_t)j * L];
    if (tj[0] == 0.0) continue;
#pragma omp parallel for schedule(static) firstprivate(a, b, c, d, w)
    for (int col = j; col < n; col++) {
      get(Qv, pa, (size_t)j * n + col, w.data());
      for (int i = j + 1; i < m; i++) {
        get(W, pa, (size_t)i * n + j, a.data());
        get(Qv, pa, (size_t)i * n + col, b.data());
        mdx_mul(L, a.data(), b.data(), c.data());
        mdx_add(L, w.data(), c.data(), w.data());
      }
      mdx_mul(L, tj, w.data(), d.data());
      get(Qv, pa, (size_t)j * n + col, b.data());
      mdx_add(L, b.data(), d.data(), b.data(), -1.0);
      put(Qv, pa, (size_t)j * n + col, b.data());
      for (int i = j + 1; i < m; i++) {
        get(W, pa, (size_t)i * n + j, a.data());
        mdx_mul(L, a.data(), d.data(), c.data());
        get(Qv, pa, (size_t)i * n + col, b.data());
        mdx_add(L, b.data(), c.data(), b.data(), -1.0);
        put(Qv, pa, (size_t)i * n + col, b.data());
      }
    }
  }
  // signs: diag(R) >= 0
  for (int j = 0; j < n; j++) {
    if (Rv[(size_t)j * n + j] >= 0.0) continue;
    for (int l = 0; l < L; l++) {
      for (int col = j; col < n; col++) Rv[l * pr + (size_t)j * n + col] = -Rv[l * pr + (size_t)j * n + col];
      for (int i = 0; i < m; i++) Qv[l * pa + (size_t)i * n + j] = -Qv[l * pa + (size_t)i * n + j];
    }
  }
  std::memcpy(Q, Qv.data(), sizeof(double) * (size_t)L * pa);
  std::memcpy(R, Rv.data(), sizeof(double) * (size_t)L * pr);
}

int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}


// =====================================================================================================
// Planning the quarter count from the data (R15; SURVEY.md 8(f) NEXT-1 "exponent-spread-driven quarter count").
//   With one exponent per row of A / column of B (R2) the error of the path is bounded relative to
//   2^(E_i + F_j), not to (|A||B|)_ij (R5):
//       |C - A*B|_ij <= k (Q+3) 2^(E_i + F_j - bits*Q - 2)  +  (renormalisation, 2^-(53 limbs - 1) |C|_ij).
//   The first term stays below rel_tol * W_ij, W = |A||B|, at every position iff
//       k (Q+3) 2^(D - bits*Q - 2) <= rel_tol,     D >= log2 max_ij 2^(E_i + F_j) / W_ij.
//   Plain definition, written out: W~_ij = sum_k |A_0[i,k]| |B_0[k,j]| on the leading limbs in fp64 (k innermost),
//   D = max over positions with W~_ij > 0 of E_i + F_j - ilogb(W~_ij) (an integer upper bound of the log2 above), and
//   Q = the smallest Q >= ceil(52 limbs / bits) that satisfies the inequality.  Positions with W~_ij = 0 have C_ij = 0
//   exactly and need nothing.  Returns Q; *spread_out = D (INT32_MIN when W~ == 0 everywhere, then Q is the minimum).
// =====================================================================================================
int oracle_plan_quarters(int m, int n, int k, int limbs, int bits, const double* A, const double* B, double rel_tol,
                         int32_t* spread_out) {
  std::vector<int32_t> E(m), F(n);
  for (int i = 0; i < m; i++) {
    double M = 0.0;
    for (int t = 0; t < k; t++) M = std::fmax(M, std::fabs(A[(size_t)i * k + t]));
    E[i] = (M == 0.0) ? 0 : std::ilogb(M) + 1;
  }
  for (int j = 0; j < n; j++) {
    double M = 0.0;
    for (int t = 0; t < k; t++) M = std::fmax(M, std::fabs(B[(size_t)t * n + j]));
    F[j] = (M == 0.0) ? 0 : std::ilogb(M) + 1;
  }
  int32_t D = INT32_MIN;
  for (int i = 0; i < m; i++)
    for (int j = 0; j < n; j++) {
      double w = 0.0;
      for (int t = 0; t < k; t++) w += std::fabs(A[(size_t)i * k + t]) * std::fabs(B[(size_t)t * n + j]);
      if (w > 0.0) {
        const int32_t d = E[i] + F[j] - std::ilogb(w);
        if (d > D) D = d;
      }
    }
  if (spread_out) *spread_out = D;
  int Q = (52 * limbs + bits - 1) / bits;
  if (D == INT32_MIN) return Q;
  // k (Q+3) 2^(D - bits*Q - 2) <= rel_tol: the left side is exact in fp64 (an integer below 2^53 times a power of two)
  while (Q < 4096 && std::ldexp((double)k * (Q + 3), D - bits * Q - 2) > rel_tol) Q++;
  return Q;
}

}  // extern "C"
