/*
 * emugemm_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU restatement of what the EmuGEMM hot path
 * computes (arxiv/paper_2606_25453, text in /root/reference/PAPER.md at build
 * time; cited below as PAPER.md:<line>).  Written from the paper, before and
 * independently of the CUDA path: it shares no code, header, table or constant
 * generator with paper_2606_25453_b200/csrc, and neither imports the other.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference leg may load this library.
 *
 * The method is an approximation with an exact integer core (slicing /
 * truncation loses low bits by design; everything between the slices or
 * residues and the integer reconstruction is exact; only the last conversion
 * rounds).  So this file follows the algorithm step by step in the paper's
 * order and notation; the exact product in __float128 (bf128_*) is the brute
 * force that tests use to check the error bound.
 *
 * Readings of the paper where it is silent or ambiguous are the R-numbers of
 * DESIGN.md ("Readings"), repeated at each use.  Arithmetic: int64 for slice
 * and residue products, unsigned 256-bit integers (4 x 64-bit limbs, schoolbook)
 * for CRT, __float128 (libquadmath) for the final scaling and rounding.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): slice re-sum invariant and an
 * independent FP64 digit recurrence; textbook integer matmul; identity / small
 * integer special cases; __float128 brute force within the closed-form error
 * bound; moduli pairwise coprime and first three = the paper's; CRT constants
 * against Python big integers; CRT round trip; X == sum a'b' exactly; 3M vs the
 * four-product complex integer matmul.  No function here is "parity unpinned".
 *
 * Layout conventions (row-major everywhere, strides in elements):
 *   A is m x k (lda >= k), B is k x n (ldb >= n), C is m x n (ldc >= n).
 *   "Canonical slice view": int8 [p][rows][k]; for B, "rows" are the COLUMNS j
 *   of B (so both operands are indexed [t][row-or-col][h]).
 */
#include <math.h>
#include <quadmath.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_BETA 7 /* beta = 7: every slice is a signed INT8 value ("signed-slice method supports beta <= 7") */

/* Slice-digit mode of Scheme I (R24 / R1 / R23).  The caller selects it with one code:
 *   7      (default; R24): 7-bit two's-complement digits -- a signed leading slice d_0 in [-128, 127] and non-negative
 *          remaining slices d_t in [0, 127], the slice form the paper's own implementation uses ("a signed
 *          leading slice with unsigned remaining slices"), here at beta = 7 so that every slice is an INT8 value
 *          ("signed-slice method supports beta <= 7").
 *   0x207  (R1): 7-bit sign-magnitude digits d_t = sign(x) * field_t(|X|) in [-127, 127], the reading of round 1; the SAME
 *          integer X = trunc(x 2^(7p)) as the default form, spelled with other digits.
 *   8      (R23): balanced signed base-256 digits, d_t in [-128, 127], two guard bits: x = a 2^-(e+2)
 *          in (-1/4, 1/4) so that X + sum_j 128 256^j stays inside [0, 256^p).
 * Internally g_slice_bits holds 0x107 (two's complement), 7 (sign-magnitude) or 8. */
#define ORACLE_DIGITS_TWOS 0x107
#define ORACLE_DIGITS_SIGNMAG_CODE 0x207
static int g_slice_bits = ORACLE_DIGITS_TWOS;
void oracle_set_slice_bits(int code) { g_slice_bits = (code == 8) ? 8 : (code == ORACLE_DIGITS_SIGNMAG_CODE) ? 7 : ORACLE_DIGITS_TWOS; }
int oracle_get_slice_bits(void) { return g_slice_bits == 8 ? 8 : g_slice_bits == 7 ? ORACLE_DIGITS_SIGNMAG_CODE : 7; }
#define ORACLE_MAX_MODULI 24

typedef __int128 i128;
typedef unsigned __int128 u128;

int oracle_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
void oracle_set_threads(int t) {
#ifdef _OPENMP
  if (t > 0) omp_set_num_threads(t);
#else
  (void)t;
#endif
}

/* ------------------------------------------------------------------------- */
/* Exponents ("each row of A is scaled by a power-of-two factor   */
/* mu_i to align exponents"; R2: frexp exponent of the row/col max magnitude, */
/* zero row => 0).                                                            */
/* ------------------------------------------------------------------------- */

/* e with |a| in [2^(e-1), 2^e); subnormals handled by frexp; 0 -> INT32_MIN. */
static int exp_of(double a) {
  if (a == 0.0) return INT32_MIN;
  int e;
  (void)frexp(a, &e);
  return e;
}

/* eA[i] = max_h exp(a_ih) over nonzero entries, 0 for an all-zero row. */
void oracle_row_exponents(int64_t m, int64_t k, const double *A, int64_t lda, int32_t *eA) {
  for (int64_t i = 0; i < m; ++i) {
    int e = INT32_MIN;
    for (int64_t h = 0; h < k; ++h) {
      int x = exp_of(A[i * lda + h]);
      if (x > e) e = x;
    }
    eA[i] = (e == INT32_MIN) ? 0 : e;
  }
}

/* eB[j] = max_h exp(b_hj) over column j of B. */
void oracle_col_exponents(int64_t k, int64_t n, const double *B, int64_t ldb, int32_t *eB) {
  for (int64_t j = 0; j < n; ++j) {
    int e = INT32_MIN;
    for (int64_t h = 0; h < k; ++h) {
      int x = exp_of(B[h * ldb + j]);
      if (x > e) e = x;
    }
    eB[j] = (e == INT32_MIN) ? 0 : e;
  }
}

/* 3M (R16): one exponent per row from max(exp(re), exp(im)); Z is complex,
 * stored as (re, im) pairs, ldz in complex elements. */
void oracle_row_exponents_z(int64_t m, int64_t k, const double *Z, int64_t ldz, int32_t *e_out) {
  for (int64_t i = 0; i < m; ++i) {
    int e = INT32_MIN;
    for (int64_t h = 0; h < k; ++h)
      for (int c = 0; c < 2; ++c) {
        int x = exp_of(Z[2 * (i * ldz + h) + c]);
        if (x > e) e = x;
      }
    e_out[i] = (e == INT32_MIN) ? 0 : e;
  }
}
void oracle_col_exponents_z(int64_t k, int64_t n, const double *Z, int64_t ldz, int32_t *e_out) {
  for (int64_t j = 0; j < n; ++j) {
    int e = INT32_MIN;
    for (int64_t h = 0; h < k; ++h)
      for (int c = 0; c < 2; ++c) {
        int x = exp_of(Z[2 * (h * ldz + j) + c]);
        if (x > e) e = x;
      }
    e_out[j] = (e == INT32_MIN) ? 0 : e;
  }
}

/* ------------------------------------------------------------------------- */
/* Scheme I slicing (Eq. 1; R1, R3: truncation toward zero).  */
/* x = a * 2^-e in (-1, 1) exactly; X = trunc(|x| * 2^(beta p)); digit t      */
/* (t = 0 most significant) d_t = (X >> beta (p-1-t)) & (2^beta - 1);         */
/* slice value = sign(a) * d_t in [-127, 127].                                */
/* ------------------------------------------------------------------------- */
static void slice_one_balanced(double a, int e, int p, int8_t *digits /* [p] */) {
  /* X = trunc(a 2^(8p - e - 2)) toward zero (R3), |X| < 2^(8p-2); Y = X + C, C = sum_{j<p} 128 256^j: every byte of
   * Y minus 128 is a balanced digit, sum_t d_t 256^(p-1-t) == X exactly. */
  __float128 sc = scalbnq((__float128)a, 8 * p - e - 2);
  int64_t X = (int64_t)truncq(sc);
  uint64_t Cc = 0;
  for (int j = 0; j < p; ++j) Cc |= (uint64_t)128 << (8 * j);
  uint64_t Y = (uint64_t)(X + (int64_t)Cc); /* 0 < Y < 256^p (p = 8: wraps mod 2^64 only if violated) */
  for (int t = 0; t < p; ++t) digits[t] = (int8_t)((int)((Y >> (8 * (p - 1 - t))) & 255u) - 128);
}

/* R24 ("a signed leading slice with unsigned remaining slices", here with beta = 7 so that every slice is
 * an INT8 value): the SAME integer as R1, X = trunc(a 2^(beta p - e)) toward zero, |X| < 2^(beta p), written in two's
 * complement: d_0 = floor(X / 2^(beta (p-1))) in [-128, 127], d_t = floor(X / 2^(beta (p-1-t))) mod 2^beta in [0, 127]
 * for t >= 1, so that sum_t d_t 2^(beta (p-1-t)) == X exactly. */
static void slice_one_twos(double a, int e, int p, int8_t *digits /* [p] */) {
  __float128 sc = scalbnq((__float128)a, ORACLE_BETA * p - e);
  int64_t X = (int64_t)truncq(sc); /* |X| < 2^56 */
  for (int t = 0; t < p; ++t) {
    const int sh = ORACLE_BETA * (p - 1 - t);
    /* floor division by a power of two of a possibly negative X, written out (no reliance on >> of negatives) */
    int64_t q = X / ((int64_t)1 << sh);
    if (X % ((int64_t)1 << sh) < 0) q -= 1;
    if (t == 0) digits[t] = (int8_t)q;                      /* in [-128, 127] */
    else digits[t] = (int8_t)(((q % 128) + 128) % 128);     /* in [0, 127] */
  }
}

static void slice_one(double a, int e, int p, int8_t *digits /* [p] */) {
  if (g_slice_bits == 8) { slice_one_balanced(a, e, p, digits); return; }
  if (g_slice_bits == ORACLE_DIGITS_TWOS) { slice_one_twos(a, e, p, digits); return; }
  /* |a| * 2^(beta p - e): a power-of-two scaling, exact in __float128. */
  __float128 sc = scalbnq(fabsq((__float128)a), ORACLE_BETA * p - e);
  uint64_t X = (uint64_t)truncq(sc); /* X < 2^(beta p) <= 2^56 */
  int sgn = (a < 0.0) ? -1 : 1;
  for (int t = 0; t < p; ++t) {
    int d = (int)((X >> (ORACLE_BETA * (p - 1 - t))) & ((1u << ORACLE_BETA) - 1u));
    digits[t] = (int8_t)(sgn * d);
  }
}

/* SA[t][i][h], t < p: slices of the rows of A with the row exponents eA. */
void oracle_oz1_slices_rows(int64_t m, int64_t k, const double *A, int64_t lda, const int32_t *eA,
                            int p, int8_t *SA) {
  int8_t d[8];
  for (int64_t i = 0; i < m; ++i)
    for (int64_t h = 0; h < k; ++h) {
      slice_one(A[i * lda + h], eA[i], p, d);
      for (int t = 0; t < p; ++t) SA[((int64_t)t * m + i) * k + h] = d[t];
    }
}

/* SB[t][j][h], t < p: slices of the columns of B with the column exponents. */
void oracle_oz1_slices_cols(int64_t k, int64_t n, const double *B, int64_t ldb, const int32_t *eB,
                            int p, int8_t *SB) {
  int8_t d[8];
  for (int64_t j = 0; j < n; ++j)
    for (int64_t h = 0; h < k; ++h) {
      slice_one(B[h * ldb + j], eB[j], p, d);
      for (int t = 0; t < p; ++t) SB[((int64_t)t * n + j) * k + h] = d[t];
    }
}

/* ------------------------------------------------------------------------- */
/* Scheme I accumulators (Eq. 2): C_s = sum_{t=0..s} A'_t B'_{s-t}*/
/* in int64, s < p.  Pairs with t + u >= p are never computed (R5).           */
/* CS[s][i][j].                                                               */
/* ------------------------------------------------------------------------- */
static int64_t acc_one(const int8_t *SA, const int8_t *SB, int64_t m, int64_t n, int64_t k, int s,
                       int64_t i, int64_t j) {
  int64_t c = 0;
  for (int t = 0; t <= s; ++t) {
    const int8_t *a = SA + ((int64_t)t * m + i) * k;
    const int8_t *b = SB + ((int64_t)(s - t) * n + j) * k;
    for (int64_t h = 0; h < k; ++h) c += (int64_t)a[h] * (int64_t)b[h];
  }
  return c;
}

void oracle_oz1_accumulators(int64_t m, int64_t n, int64_t k, int p, const int8_t *SA,
                             const int8_t *SB, int64_t *CS) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < m; ++i)
    for (int64_t j = 0; j < n; ++j)
      for (int s = 0; s < p; ++s) CS[((int64_t)s * m + i) * n + j] = acc_one(SA, SB, m, n, k, s, i, j);
}

/* ------------------------------------------------------------------------- */
/* Shift-reduce and output (Eq. 3; R4, R6, R9):                   */
/*   S = sum_s C_s 2^(beta (p-1-s))           exact integer (<= 81 bits)       */
/*   v = S * 2^(eA_i + eB_j - beta (p+1))     exact in __float128              */
/*   C = round( alpha v + beta_ C_in )        evaluated in __float128          */
/* beta_ == 0 => C_in is not read (BLAS rule).                                 */
/* ------------------------------------------------------------------------- */
static __float128 oz1_value(const int64_t *cs /* [p] */, int p, int eAi, int eBj) {
  if (g_slice_bits == 8) { /* balanced base 256: v = S 2^(eA + eB + 4 - 8 (p+1)), the +4 are the guard bits */
    i128 S8 = 0;
    for (int s = 0; s < p; ++s) S8 += (i128)cs[s] * ((i128)1 << (8 * (p - 1 - s)));
    return scalbnq((__float128)S8, eAi + eBj + 4 - 8 * (p + 1));
  }
  i128 S = 0;
  for (int s = 0; s < p; ++s) S += (i128)cs[s] * ((i128)1 << (ORACLE_BETA * (p - 1 - s)));
  return scalbnq((__float128)S, eAi + eBj - ORACLE_BETA * (p + 1));
}

static double finish_d(double alpha, __float128 v, double beta_, const double *cin) {
  __float128 r = (__float128)alpha * v;
  if (beta_ != 0.0) r += (__float128)beta_ * (__float128)(*cin);
  return (double)r;
}

void oracle_oz1_reduce(int64_t m, int64_t n, int p, const int64_t *CS, const int32_t *eA,
                       const int32_t *eB, double alpha, double beta_, double *C, int64_t ldc) {
  int64_t cs[8];
  for (int64_t i = 0; i < m; ++i)
    for (int64_t j = 0; j < n; ++j) {
      for (int s = 0; s < p; ++s) cs[s] = CS[((int64_t)s * m + i) * n + j];
      C[i * ldc + j] = finish_d(alpha, oz1_value(cs, p, eA[i], eB[j]), beta_, &C[i * ldc + j]);
    }
}

/* Whole Scheme I DGEMM, C = alpha A B + beta C with p slices. Returns 0. */
int oracle_dgemm_oz1(int64_t m, int64_t n, int64_t k, double alpha, const double *A, int64_t lda,
                     const double *B, int64_t ldb, double beta_, double *C, int64_t ldc, int p) {
  if (p < 1 || p > 8 || m < 0 || n < 0 || k < 0) return -1;
  if (m == 0 || n == 0) return 0;
  int32_t *eA = malloc(sizeof(int32_t) * (size_t)m), *eB = malloc(sizeof(int32_t) * (size_t)n);
  int8_t *SA = malloc((size_t)p * m * (k ? k : 1)), *SB = malloc((size_t)p * n * (k ? k : 1));
  int64_t *CS = malloc(sizeof(int64_t) * (size_t)p * m * n);
  oracle_row_exponents(m, k, A, lda, eA);
  oracle_col_exponents(k, n, B, ldb, eB);
  oracle_oz1_slices_rows(m, k, A, lda, eA, p, SA);
  oracle_oz1_slices_cols(k, n, B, ldb, eB, p, SB);
  oracle_oz1_accumulators(m, n, k, p, SA, SB, CS);
  oracle_oz1_reduce(m, n, p, CS, eA, eB, alpha, beta_, C, ldc);
  free(eA); free(eB); free(SA); free(SB); free(CS);
  return 0;
}

/* FP32 entry point (north_star "emugemm_sgemm_oz1"): same algorithm on 24-bit
 * inputs, one rounding to float.  Inputs are widened exactly to double. */
int oracle_sgemm_oz1(int64_t m, int64_t n, int64_t k, float alpha, const float *A, int64_t lda,
                     const float *B, int64_t ldb, float beta_, float *C, int64_t ldc, int p) {
  if (p < 1 || p > 8 || m < 0 || n < 0 || k < 0) return -1;
  if (m == 0 || n == 0) return 0;
  double *Ad = malloc(sizeof(double) * (size_t)m * (k ? k : 1));
  double *Bd = malloc(sizeof(double) * (size_t)(k ? k : 1) * n);
  for (int64_t i = 0; i < m; ++i) for (int64_t h = 0; h < k; ++h) Ad[i * k + h] = A[i * lda + h];
  for (int64_t h = 0; h < k; ++h) for (int64_t j = 0; j < n; ++j) Bd[h * n + j] = B[h * ldb + j];
  int32_t *eA = malloc(sizeof(int32_t) * (size_t)m), *eB = malloc(sizeof(int32_t) * (size_t)n);
  int8_t *SA = malloc((size_t)p * m * (k ? k : 1)), *SB = malloc((size_t)p * n * (k ? k : 1));
  int64_t *CS = malloc(sizeof(int64_t) * (size_t)p * m * n);
  oracle_row_exponents(m, k, Ad, k, eA);
  oracle_col_exponents(k, n, Bd, n, eB);
  oracle_oz1_slices_rows(m, k, Ad, k, eA, p, SA);
  oracle_oz1_slices_cols(k, n, Bd, n, eB, p, SB);
  oracle_oz1_accumulators(m, n, k, p, SA, SB, CS);
  int64_t cs[8];
  for (int64_t i = 0; i < m; ++i)
    for (int64_t j = 0; j < n; ++j) {
      for (int s = 0; s < p; ++s) cs[s] = CS[((int64_t)s * m + i) * n + j];
      __float128 r = (__float128)alpha * oz1_value(cs, p, eA[i], eB[j]);
      if (beta_ != 0.0f) r += (__float128)beta_ * (__float128)C[i * ldc + j];
      C[i * ldc + j] = (float)r;
    }
  free(Ad); free(Bd); free(eA); free(eB); free(SA); free(SB); free(CS);
  return 0;
}

/* Sampled Scheme I output for large sizes: out[r][c] for the given row and
 * column index lists (beta_ = 0).  Same per-element arithmetic as above; only
 * rows rows[r] of A and columns cols[c] of B are touched.  is_f32 != 0: the
 * value is rounded once to float and returned widened. */
void oracle_oz1_sampled(int64_t m, int64_t n, int64_t k, double alpha, const double *A, int64_t lda,
                        const double *B, int64_t ldb, int p, int64_t nr, const int64_t *rows,
                        int64_t nc, const int64_t *cols, int is_f32, double *out /* [nr][nc] */) {
  (void)m; (void)n;
  int32_t *eA = malloc(sizeof(int32_t) * (size_t)nr), *eB = malloc(sizeof(int32_t) * (size_t)nc);
  double *Ar = malloc(sizeof(double) * (size_t)nr * k), *Bc = malloc(sizeof(double) * (size_t)k * nc);
  for (int64_t r = 0; r < nr; ++r) memcpy(Ar + r * k, A + rows[r] * lda, sizeof(double) * (size_t)k);
  for (int64_t h = 0; h < k; ++h) for (int64_t c = 0; c < nc; ++c) Bc[h * nc + c] = B[h * ldb + cols[c]];
  int8_t *SA = malloc((size_t)p * nr * k), *SB = malloc((size_t)p * nc * k);
  oracle_row_exponents(nr, k, Ar, k, eA);
  oracle_col_exponents(k, nc, Bc, nc, eB);
  oracle_oz1_slices_rows(nr, k, Ar, k, eA, p, SA);
  oracle_oz1_slices_cols(k, nc, Bc, nc, eB, p, SB);
#pragma omp parallel for schedule(static)
  for (int64_t r = 0; r < nr; ++r)
    for (int64_t c = 0; c < nc; ++c) {
      int64_t cs[8];
      for (int s = 0; s < p; ++s) cs[s] = acc_one(SA, SB, nr, nc, k, s, r, c);
      __float128 v = (__float128)alpha * oz1_value(cs, p, eA[r], eB[c]);
      out[r * nc + c] = is_f32 ? (double)(float)v : (double)v;
    }
  free(eA); free(eB); free(Ar); free(Bc); free(SA); free(SB);
}

/* ------------------------------------------------------------------------- */
/* Scheme I complex GEMM by the 4M formulation ("EmuGEMM-I uses  */
/* the 4M formulation"), written as FOUR SEPARATE REAL     */
/* slice products:                                                            */
/*   Re(A B) = ReA ReB + (-ImA) ImB,   Im(A B) = ImA ReB + ReA ImB,           */
/* i.e. the real embedding A' = [[ReA, -ImA], [ImA, ReA]], B' = [[ReB], [ImB]] */
/* taken product by product: the minus sign is carried by the OPERAND (-ImA is */
/* sliced), which matters for the balanced 8-bit digits (R23), whose digits of */
/* -x are not the negated digits of x; with sign-magnitude digits (R1) it is   */
/* the same as subtracting the product.                                        */
/* Real and imaginary part of a row of A (column of B) share ONE exponent, the */
/* maximum over both (R16 applied to 4M: a real diagonal scaling must commute */
/* with the complex product).  Per s < p the four int64 accumulators          */
/* P1..P4 (Eq. 2 on the slices of the parts) give                             */
/*   C_s^re = P1_s + P2_s,   C_s^im = P3_s + P4_s     exactly,                */
/* Eq. 3 and the scaling are exact in __float128 and each component T_re,     */
/* T_im is rounded ONCE to double (a real Scheme I result each); then          */
/*   C = alpha (T_re + i T_im) + beta C_in   in __float128, rounded once per  */
/* component (to float first when is_f32: the CGEMM entry point).             */
/* A, B, C: (re, im) pairs, strides in complex elements.                      */
/* ------------------------------------------------------------------------- */
int oracle_zgemm_oz1_4m(int64_t m, int64_t n, int64_t k, const double *alpha, const double *A, int64_t lda,
                        const double *B, int64_t ldb, const double *beta_, double *C, int64_t ldc, int p,
                        int is_f32) {
  if (p < 1 || p > 8 || m < 0 || n < 0 || k < 0) return -1;
  if (m == 0 || n == 0) return 0;
  const int64_t kk = k ? k : 1;
  int32_t *eA = malloc(sizeof(int32_t) * (size_t)m), *eB = malloc(sizeof(int32_t) * (size_t)n);
  double *Ar = malloc(sizeof(double) * (size_t)m * kk), *Ai = malloc(sizeof(double) * (size_t)m * kk);
  double *An = malloc(sizeof(double) * (size_t)m * kk); /* -Im A */
  double *Br = malloc(sizeof(double) * (size_t)kk * n), *Bi = malloc(sizeof(double) * (size_t)kk * n);
  for (int64_t i = 0; i < m; ++i)
    for (int64_t h = 0; h < k; ++h) {
      Ar[i * k + h] = A[2 * (i * lda + h)];
      Ai[i * k + h] = A[2 * (i * lda + h) + 1];
      An[i * k + h] = -A[2 * (i * lda + h) + 1];
    }
  for (int64_t h = 0; h < k; ++h)
    for (int64_t j = 0; j < n; ++j) { Br[h * n + j] = B[2 * (h * ldb + j)]; Bi[h * n + j] = B[2 * (h * ldb + j) + 1]; }
  oracle_row_exponents_z(m, k, A, lda, eA);
  oracle_col_exponents_z(k, n, B, ldb, eB);
  int8_t *SAr = malloc((size_t)p * m * kk), *SAi = malloc((size_t)p * m * kk), *SAn = malloc((size_t)p * m * kk);
  int8_t *SBr = malloc((size_t)p * n * kk), *SBi = malloc((size_t)p * n * kk);
  oracle_oz1_slices_rows(m, k, Ar, k, eA, p, SAr);
  oracle_oz1_slices_rows(m, k, Ai, k, eA, p, SAi);
  oracle_oz1_slices_rows(m, k, An, k, eA, p, SAn);
  oracle_oz1_slices_cols(k, n, Br, n, eB, p, SBr);
  oracle_oz1_slices_cols(k, n, Bi, n, eB, p, SBi);
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < m; ++i)
    for (int64_t j = 0; j < n; ++j) {
      int64_t cre[8], cim[8];
      for (int s = 0; s < p; ++s) {
        const int64_t p1 = acc_one(SAr, SBr, m, n, k, s, i, j), p2 = acc_one(SAn, SBi, m, n, k, s, i, j);
        const int64_t p3 = acc_one(SAi, SBr, m, n, k, s, i, j), p4 = acc_one(SAr, SBi, m, n, k, s, i, j);
        cre[s] = p1 + p2;
        cim[s] = p3 + p4;
      }
      const double tre = (double)oz1_value(cre, p, eA[i], eB[j]), tim = (double)oz1_value(cim, p, eA[i], eB[j]);
      __float128 re = (__float128)alpha[0] * tre - (__float128)alpha[1] * tim;
      __float128 im = (__float128)alpha[0] * tim + (__float128)alpha[1] * tre;
      double *c = C + 2 * (i * ldc + j);
      if (beta_[0] != 0.0 || beta_[1] != 0.0) {
        re += (__float128)beta_[0] * c[0] - (__float128)beta_[1] * c[1];
        im += (__float128)beta_[0] * c[1] + (__float128)beta_[1] * c[0];
      }
      c[0] = is_f32 ? (double)(float)re : (double)re;
      c[1] = is_f32 ? (double)(float)im : (double)im;
    }
  free(eA); free(eB); free(Ar); free(Ai); free(An); free(Br); free(Bi); free(SAr); free(SAi); free(SAn); free(SBr); free(SBi);
  return 0;
}

/* ------------------------------------------------------------------------- */
/* Brute force: exact-ish product of the ORIGINAL operands in __float128      */
/* (113-bit significand; each product of two doubles is exact, the sum rounds */
/* at 2^-113 relative) -- used only to check error bounds.                    */
/* out128 (optional) receives the unrounded value as two doubles hi+lo.       */
/* ------------------------------------------------------------------------- */
void oracle_bf128_dgemm(int64_t m, int64_t n, int64_t k, const double *A, int64_t lda,
                        const double *B, int64_t ldb, double *C, int64_t ldc, double *absAB) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < m; ++i)
    for (int64_t j = 0; j < n; ++j) {
      __float128 s = 0, sa = 0;
      for (int64_t h = 0; h < k; ++h) {
        __float128 t = (__float128)A[i * lda + h] * (__float128)B[h * ldb + j];
        s += t;
        sa += fabsq(t);
      }
      C[i * ldc + j] = (double)s;
      if (absAB) absAB[i * n + j] = (double)sa;
    }
}

/* complex: Z = X * Y, (re, im) pairs; absZ (optional, [m][n]) receives
 * sum_h (|x_re|+|x_im|)(|y_re|+|y_im|), the scale the 3M tolerance uses. */
void oracle_bf128_zgemm(int64_t m, int64_t n, int64_t k, const double *X, int64_t ldx,
                        const double *Y, int64_t ldy, double *Z, int64_t ldz, double *absZ) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < m; ++i)
    for (int64_t j = 0; j < n; ++j) {
      __float128 sr = 0, si = 0, sa = 0;
      for (int64_t h = 0; h < k; ++h) {
        __float128 xr = X[2 * (i * ldx + h)], xi = X[2 * (i * ldx + h) + 1];
        __float128 yr = Y[2 * (h * ldy + j)], yi = Y[2 * (h * ldy + j) + 1];
        sr += xr * yr - xi * yi;
        si += xr * yi + xi * yr;
        sa += (fabsq(xr) + fabsq(xi)) * (fabsq(yr) + fabsq(yi));
      }
      Z[2 * (i * ldz + j)] = (double)sr;
      Z[2 * (i * ldz + j) + 1] = (double)si;
      if (absZ) absZ[i * n + j] = (double)sa;
    }
}

/* ========================================================================= */
/* Scheme II                                                                  */
/* ========================================================================= */

/* -- tiny unsigned 256-bit integers: 4 little-endian 64-bit limbs ---------- */
typedef struct { uint64_t w[4]; } u256;

static u256 u256_from_u64(uint64_t x) { u256 r = {{x, 0, 0, 0}}; return r; }
static int u256_cmp(const u256 *a, const u256 *b) {
  for (int i = 3; i >= 0; --i) {
    if (a->w[i] < b->w[i]) return -1;
    if (a->w[i] > b->w[i]) return 1;
  }
  return 0;
}
static u256 u256_add(const u256 *a, const u256 *b) {
  u256 r; u128 c = 0;
  for (int i = 0; i < 4; ++i) { c += (u128)a->w[i] + b->w[i]; r.w[i] = (uint64_t)c; c >>= 64; }
  return r;
}
static u256 u256_sub(const u256 *a, const u256 *b) { /* a >= b */
  u256 r; i128 c = 0;
  for (int i = 0; i < 4; ++i) {
    i128 d = (i128)a->w[i] - (i128)b->w[i] + c;
    r.w[i] = (uint64_t)d;
    c = (d < 0) ? -1 : 0;
  }
  return r;
}
static u256 u256_mul_small(const u256 *a, uint64_t s) {
  u256 r; u128 c = 0;
  for (int i = 0; i < 4; ++i) { c += (u128)a->w[i] * s; r.w[i] = (uint64_t)c; c >>= 64; }
  return r;
}
static u256 u256_div_small(const u256 *a, uint64_t s, uint64_t *rem) {
  u256 q; u128 r = 0;
  for (int i = 3; i >= 0; --i) {
    u128 cur = (r << 64) | a->w[i];
    q.w[i] = (uint64_t)(cur / s);
    r = cur % s;
  }
  if (rem) *rem = (uint64_t)r;
  return q;
}
static u256 u256_shl(const u256 *a, int sh) { /* 0 <= sh < 256 */
  u256 r = {{0, 0, 0, 0}};
  int ws = sh / 64, bs = sh % 64;
  for (int i = 3; i >= ws; --i) {
    uint64_t v = a->w[i - ws] << bs;
    if (bs && i - ws - 1 >= 0) v |= a->w[i - ws - 1] >> (64 - bs);
    r.w[i] = v;
  }
  return r;
}
/* a mod P for a < 2^9 * P: binary shift-and-subtract. */
static u256 u256_mod_near(u256 a, const u256 *P) {
  for (int b = 9; b >= 0; --b) {
    u256 Pb = u256_shl(P, b);
    if (u256_cmp(&a, &Pb) >= 0) a = u256_sub(&a, &Pb);
  }
  return a;
}
static __float128 u256_to_q(const u256 *a) {
  __float128 r = 0;
  for (int i = 3; i >= 0; --i) r = r * 18446744073709551616.0Q + (__float128)a->w[i];
  return r; /* exact below 2^113, else rounded at <= 3 * 2^-113 relative (<< FP64 ulp) */
}

/* Moduli ("pairwise co-prime ... e.g. {256, 255, 253, ...}";
 * R10): scan 256, 255, ... downward, keep m if coprime to all kept. */
static uint32_t gcd_u32(uint32_t a, uint32_t b) { while (b) { uint32_t t = a % b; a = b; b = t; } return a; }
int oracle_oz2_moduli(int N, int32_t *mod /* [N] */) {
  if (N < 1 || N > ORACLE_MAX_MODULI) return -1;
  int cnt = 0;
  for (uint32_t c = 256; c >= 2 && cnt < N; --c) {
    int ok = 1;
    for (int i = 0; i < cnt; ++i) if (gcd_u32(c, (uint32_t)mod[i]) != 1) { ok = 0; break; }
    if (ok) mod[cnt++] = (int32_t)c;
  }
  return cnt == N ? 0 : -1;
}

static u256 oz2_P(int N, const int32_t *mod) {
  u256 P = u256_from_u64(1);
  for (int l = 0; l < N; ++l) P = u256_mul_small(&P, (uint64_t)mod[l]);
  return P;
}
void oracle_oz2_P_limbs(int N, uint64_t *limbs /* [4] */) {
  int32_t mod[ORACLE_MAX_MODULI];
  oracle_oz2_moduli(N, mod);
  u256 P = oz2_P(N, mod);
  memcpy(limbs, P.w, 32);
}

/* Bit budget (PAPER.md:132 exactness condition "2 sum |a'||b'| < P"; R12):
 * T = max{T : k 2^(T+2) <= P} (3M: k 2^(T+3) <= P), tA = T - floor(T/2),
 * tB = floor(T/2).  Returns T (or < 0 if none). */
int oracle_oz2_budget(int N, int64_t k, int is3m, int32_t *tA, int32_t *tB) {
  int32_t mod[ORACLE_MAX_MODULI];
  if (oracle_oz2_moduli(N, mod) != 0 || k < 1) return -1;
  u256 P = oz2_P(N, mod);
  int guard = is3m ? 3 : 2, T = -1;
  for (int t = 0; t + guard < 200; ++t) {
    u256 kk = u256_from_u64((uint64_t)k);
    u256 lhs = u256_shl(&kk, t + guard);
    if (u256_cmp(&lhs, &P) <= 0) T = t; else break;
  }
  if (T < 0) return -1;
  *tB = T / 2;
  *tA = T - T / 2;
  return T;
}

/* sym(x, m) (R11, R13): r = x - m floor(x/m) in [0, m); if r >= ceil(m/2)
 * then r -= m.  Range [-128,127] for 256, [-(m-1)/2,(m-1)/2] for odd m. */
static int sym_i128(i128 x, int m) {
  i128 r = x % m; /* C remainder: sign of x */
  if (r < 0) r += m;
  int ri = (int)r;
  if (ri >= (m + 1) / 2) ri -= m;
  return ri;
}

/* a' = trunc(a 2^(t - e)) toward zero (R3), |a'| < 2^t <= 2^70. */
static i128 oz2_int(double a, int t, int e) {
  return (i128)truncq(scalbnq((__float128)a, t - e));
}

/* RA[l][i][h] = sym(trunc(a_ih 2^(tA - eA_i)), m_l)   (Eq. 5) */
void oracle_oz2_residues_rows(int64_t m, int64_t k, const double *A, int64_t lda, const int32_t *eA,
                              int tA, int N, int8_t *RA) {
  int32_t mod[ORACLE_MAX_MODULI];
  oracle_oz2_moduli(N, mod);
  for (int64_t i = 0; i < m; ++i)
    for (int64_t h = 0; h < k; ++h) {
      i128 ai = oz2_int(A[i * lda + h], tA, eA[i]);
      for (int l = 0; l < N; ++l) RA[((int64_t)l * m + i) * k + h] = (int8_t)sym_i128(ai, mod[l]);
    }
}
/* RB[l][j][h] = sym(trunc(b_hj 2^(tB - eB_j)), m_l) */
void oracle_oz2_residues_cols(int64_t k, int64_t n, const double *B, int64_t ldb, const int32_t *eB,
                              int tB, int N, int8_t *RB) {
  int32_t mod[ORACLE_MAX_MODULI];
  oracle_oz2_moduli(N, mod);
  for (int64_t j = 0; j < n; ++j)
    for (int64_t h = 0; h < k; ++h) {
      i128 bi = oz2_int(B[h * ldb + j], tB, eB[j]);
      for (int l = 0; l < N; ++l) RB[((int64_t)l * n + j) * k + h] = (int8_t)sym_i128(bi, mod[l]);
    }
}

/* 3M operand planes (R15): for complex Z (rows = rows of A or
 * columns of B), R3[part][l][row][h], part 0 = re, 1 = im, 2 = Sigma with
 * r_Sigma = sym(r_re + r_im, m_l).  by_cols != 0: Z is k x rows, read
 * column-wise (operand B). */
void oracle_oz2_residues_z(int64_t rows, int64_t k, const double *Z, int64_t ldz, int by_cols,
                           const int32_t *e, int t, int N, int8_t *R3) {
  int32_t mod[ORACLE_MAX_MODULI];
  oracle_oz2_moduli(N, mod);
  int64_t plane = (int64_t)N * rows * k;
  for (int64_t r = 0; r < rows; ++r)
    for (int64_t h = 0; h < k; ++h) {
      const double *z = by_cols ? Z + 2 * (h * ldz + r) : Z + 2 * (r * ldz + h);
      i128 zr = oz2_int(z[0], t, e[r]), zi = oz2_int(z[1], t, e[r]);
      for (int l = 0; l < N; ++l) {
        int rr = sym_i128(zr, mod[l]), ri = sym_i128(zi, mod[l]);
        int64_t o = ((int64_t)l * rows + r) * k + h;
        R3[o] = (int8_t)rr;
        R3[plane + o] = (int8_t)ri;
        R3[2 * plane + o] = (int8_t)sym_i128((i128)(rr + ri), mod[l]);
      }
    }
}

/* Per-modulus product + reduction (Eq. 6-7):
 * acc_l[i][j] = sum_h RA_l[i][h] RB_l[j][h] (int64; caller may request it),
 * CR[l][i][j] = sym(acc_l, m_l).  Returns the max |acc| seen (must be < 2^31
 * for the INT32 accumulation the paper prescribes; R7). */
int64_t oracle_oz2_modprod(int64_t m, int64_t n, int64_t k, int N, const int8_t *RA, const int8_t *RB,
                           int8_t *CR, int64_t *ACC /* optional [N][m][n] */) {
  int32_t mod[ORACLE_MAX_MODULI];
  oracle_oz2_moduli(N, mod);
  int64_t maxabs = 0;
  for (int l = 0; l < N; ++l) {
#pragma omp parallel for schedule(static) reduction(max : maxabs)
    for (int64_t i = 0; i < m; ++i)
      for (int64_t j = 0; j < n; ++j) {
        const int8_t *a = RA + ((int64_t)l * m + i) * k, *b = RB + ((int64_t)l * n + j) * k;
        int64_t c = 0;
        for (int64_t h = 0; h < k; ++h) c += (int64_t)a[h] * (int64_t)b[h];
        if (ACC) ACC[((int64_t)l * m + i) * n + j] = c;
        int64_t ab = c < 0 ? -c : c;
        if (ab > maxabs) maxabs = ab;
        CR[((int64_t)l * m + i) * n + j] = (int8_t)sym_i128((i128)c, mod[l]);
      }
  }
  return maxabs;
}

/* 3M per-modulus products (Eq. 16; R15): T1 = sym(re.re),
 * T2 = sym(im.im), T3 = sym(Sig.Sig); c_re = sym(T1 - T2), c_im = sym(T3 - T1 - T2).
 * RA3/RB3 are the [3][N][rows][k] planes above; CZ[part][l][i][j], part 0 = re, 1 = im. */
void oracle_oz2_modprod_3m(int64_t m, int64_t n, int64_t k, int N, const int8_t *RA3, const int8_t *RB3,
                           int8_t *CZ) {
  int32_t mod[ORACLE_MAX_MODULI];
  oracle_oz2_moduli(N, mod);
  int64_t pa = (int64_t)N * m * k, pb = (int64_t)N * n * k, pc = (int64_t)N * m * n;
  for (int l = 0; l < N; ++l) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < m; ++i)
      for (int64_t j = 0; j < n; ++j) {
        int T[3];
        for (int part = 0; part < 3; ++part) {
          const int8_t *a = RA3 + part * pa + ((int64_t)l * m + i) * k;
          const int8_t *b = RB3 + part * pb + ((int64_t)l * n + j) * k;
          int64_t c = 0;
          for (int64_t h = 0; h < k; ++h) c += (int64_t)a[h] * (int64_t)b[h];
          T[part] = sym_i128((i128)c, mod[l]);
        }
        int64_t o = ((int64_t)l * m + i) * n + j;
        CZ[o] = (int8_t)sym_i128((i128)(T[0] - T[1]), mod[l]);
        CZ[pc + o] = (int8_t)sym_i128((i128)(T[2] - T[0] - T[1]), mod[l]);
      }
  }
}

/* CRT constants (Eq. 8): w_l = (P/m_l) q_l with q_l the
 * inverse of P/m_l modulo m_l (q_l < m_l so w_l < P already). limbs [N][4]. */
static void oz2_weights(int N, const int32_t *mod, const u256 *P, u256 *w) {
  for (int l = 0; l < N; ++l) {
    uint64_t rem;
    u256 Pl = u256_div_small(P, (uint64_t)mod[l], &rem); /* rem == 0 */
    uint64_t plm;
    (void)u256_div_small(&Pl, (uint64_t)mod[l], &plm); /* (P/m_l) mod m_l */
    uint64_t q = 0;
    for (uint64_t c = 1; c < (uint64_t)mod[l]; ++c) if ((plm * c) % (uint64_t)mod[l] == 1) { q = c; break; }
    w[l] = u256_mul_small(&Pl, q);
  }
}
void oracle_oz2_weights_limbs(int N, uint64_t *limbs /* [N][4] */) {
  int32_t mod[ORACLE_MAX_MODULI];
  oracle_oz2_moduli(N, mod);
  u256 P = oz2_P(N, mod), w[ORACLE_MAX_MODULI];
  oz2_weights(N, mod, &P, w);
  for (int l = 0; l < N; ++l) memcpy(limbs + 4 * l, w[l].w, 32);
}

/* X = (sum_l w_l c_l) mod P mapped to (-P/2, P/2] (R14), exact.  Returns the
 * magnitude in *mag and the sign (+1/-1/0). */
static int oz2_crt_one(int N, const int32_t *mod, const u256 *P, const u256 *w, const int *c, u256 *mag) {
  u256 acc = u256_from_u64(0);
  for (int l = 0; l < N; ++l) {
    int cu = c[l] % mod[l];
    if (cu < 0) cu += mod[l]; /* representative in [0, m) */
    u256 t = u256_mul_small(&w[l], (uint64_t)cu); /* < 2^8 P */
    t = u256_mod_near(t, P);
    acc = u256_add(&acc, &t);
    if (u256_cmp(&acc, P) >= 0) acc = u256_sub(&acc, P);
  }
  /* symmetric representative: X in (-P/2, P/2]  <=>  if 2 acc > P then acc - P */
  u256 twice = u256_add(&acc, &acc);
  if (u256_cmp(&twice, P) > 0) { *mag = u256_sub(P, &acc); return -1; }
  *mag = acc;
  return (acc.w[0] | acc.w[1] | acc.w[2] | acc.w[3]) ? 1 : 0;
}

/* Test hook: CRT of one residue vector -> sign and 4 magnitude limbs. */
int oracle_oz2_crt_limbs(int N, const int32_t *c, uint64_t *mag_limbs) {
  int32_t mod[ORACLE_MAX_MODULI];
  oracle_oz2_moduli(N, mod);
  u256 P = oz2_P(N, mod), w[ORACLE_MAX_MODULI], mag;
  oz2_weights(N, mod, &P, w);
  int cc[ORACLE_MAX_MODULI];
  for (int l = 0; l < N; ++l) cc[l] = c[l];
  int s = oz2_crt_one(N, mod, &P, w, cc, &mag);
  memcpy(mag_limbs, mag.w, 32);
  return s;
}

/* CRT + inverse scaling: for every (i, j),
 *   X = crt(CR[.][i][j]);  v = X 2^(eA_i + eB_j - tA - tB)  in __float128;
 *   C = round(alpha v + beta_ C_in).   X128 (optional, [m][n][5] uint64) receives X exactly for tests: the sign
 *   (0, 1 or 2^64 - 1) followed by the four 64-bit limbs of |X| (no truncation: |X| < P/2 < 2^256). */
void oracle_oz2_crt(int64_t m, int64_t n, int N, const int8_t *CR, const int32_t *eA, const int32_t *eB,
                    int tA, int tB, double alpha, double beta_, double *C, int64_t ldc, int64_t cstride,
                    int64_t *X128) {
  int32_t mod[ORACLE_MAX_MODULI];
  oracle_oz2_moduli(N, mod);
  u256 P = oz2_P(N, mod), w[ORACLE_MAX_MODULI];
  oz2_weights(N, mod, &P, w);
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < m; ++i)
    for (int64_t j = 0; j < n; ++j) {
      int c[ORACLE_MAX_MODULI];
      for (int l = 0; l < N; ++l) c[l] = CR[((int64_t)l * m + i) * n + j];
      u256 mag;
      int sg = oz2_crt_one(N, mod, &P, w, c, &mag);
      if (X128) {
        int64_t *xo = X128 + 5 * (i * n + j);
        xo[0] = sg;
        for (int q = 0; q < 4; ++q) xo[1 + q] = (int64_t)mag.w[q];
      }
      __float128 v = scalbnq(u256_to_q(&mag), eA[i] + eB[j] - tA - tB);
      if (sg < 0) v = -v;
      double *dst = C + (i * ldc + j) * cstride;
      __float128 r = (__float128)alpha * v;
      if (beta_ != 0.0) r += (__float128)beta_ * (__float128)(*dst);
      *dst = (double)r;
    }
}

/* Whole Scheme II DGEMM with N moduli. Returns 0, -1 bad args, -2 no budget. */
int oracle_dgemm_oz2(int64_t m, int64_t n, int64_t k, double alpha, const double *A, int64_t lda,
                     const double *B, int64_t ldb, double beta_, double *C, int64_t ldc, int N) {
  if (N < 2 || N > ORACLE_MAX_MODULI || m < 0 || n < 0 || k < 1) return -1;
  if (m == 0 || n == 0) return 0;
  int32_t tA, tB;
  if (oracle_oz2_budget(N, k, 0, &tA, &tB) < 2) return -2;
  int32_t *eA = malloc(sizeof(int32_t) * (size_t)m), *eB = malloc(sizeof(int32_t) * (size_t)n);
  int8_t *RA = malloc((size_t)N * m * k), *RB = malloc((size_t)N * n * k), *CR = malloc((size_t)N * m * n);
  oracle_row_exponents(m, k, A, lda, eA);
  oracle_col_exponents(k, n, B, ldb, eB);
  oracle_oz2_residues_rows(m, k, A, lda, eA, tA, N, RA);
  oracle_oz2_residues_cols(k, n, B, ldb, eB, tB, N, RB);
  (void)oracle_oz2_modprod(m, n, k, N, RA, RB, CR, NULL);
  oracle_oz2_crt(m, n, N, CR, eA, eB, tA, tB, alpha, beta_, C, ldc, 1, NULL);
  free(eA); free(eB); free(RA); free(RB); free(CR);
  return 0;
}

/* Whole Scheme II ZGEMM via 3M (R15, R16).  alpha, beta_ are
 * complex (re, im); A, B, C complex (re, im) pairs, strides in complex elements. */
/* FP32 entry point of Scheme II ("EmuGEMM-II SGEMM (p8-p11)"): the same
 * algorithm on 24-bit inputs widened exactly to double, one rounding to float from the __float128 value. */
int oracle_sgemm_oz2(int64_t m, int64_t n, int64_t k, float alpha, const float *A, int64_t lda, const float *B,
                     int64_t ldb, float beta_, float *C, int64_t ldc, int N) {
  if (N < 2 || N > ORACLE_MAX_MODULI || m < 0 || n < 0 || k < 1) return -1;
  if (m == 0 || n == 0) return 0;
  int32_t tA, tB;
  if (oracle_oz2_budget(N, k, 0, &tA, &tB) < 2) return -2;
  double *Ad = malloc(sizeof(double) * (size_t)m * k), *Bd = malloc(sizeof(double) * (size_t)k * n);
  for (int64_t i = 0; i < m; ++i) for (int64_t h = 0; h < k; ++h) Ad[i * k + h] = A[i * lda + h];
  for (int64_t h = 0; h < k; ++h) for (int64_t j = 0; j < n; ++j) Bd[h * n + j] = B[h * ldb + j];
  int32_t *eA = malloc(sizeof(int32_t) * (size_t)m), *eB = malloc(sizeof(int32_t) * (size_t)n);
  int8_t *RA = malloc((size_t)N * m * k), *RB = malloc((size_t)N * n * k), *CR = malloc((size_t)N * m * n);
  oracle_row_exponents(m, k, Ad, k, eA);
  oracle_col_exponents(k, n, Bd, n, eB);
  oracle_oz2_residues_rows(m, k, Ad, k, eA, tA, N, RA);
  oracle_oz2_residues_cols(k, n, Bd, n, eB, tB, N, RB);
  (void)oracle_oz2_modprod(m, n, k, N, RA, RB, CR, NULL);
  int32_t mod[ORACLE_MAX_MODULI];
  oracle_oz2_moduli(N, mod);
  u256 P = oz2_P(N, mod), w[ORACLE_MAX_MODULI];
  oz2_weights(N, mod, &P, w);
  for (int64_t i = 0; i < m; ++i)
    for (int64_t j = 0; j < n; ++j) {
      int c[ORACLE_MAX_MODULI];
      for (int l = 0; l < N; ++l) c[l] = CR[((int64_t)l * m + i) * n + j];
      u256 mag;
      int sg = oz2_crt_one(N, mod, &P, w, c, &mag);
      __float128 v = scalbnq(u256_to_q(&mag), eA[i] + eB[j] - tA - tB);
      if (sg < 0) v = -v;
      __float128 r = (__float128)alpha * v;
      if (beta_ != 0.0f) r += (__float128)beta_ * (__float128)C[i * ldc + j];
      C[i * ldc + j] = (float)r;
    }
  free(Ad); free(Bd); free(eA); free(eB); free(RA); free(RB); free(CR);
  return 0;
}

int oracle_zgemm_oz2_3m(int64_t m, int64_t n, int64_t k, const double *alpha, const double *A, int64_t lda,
                        const double *B, int64_t ldb, const double *beta_, double *C, int64_t ldc, int N) {
  if (N < 2 || N > ORACLE_MAX_MODULI || m < 0 || n < 0 || k < 1) return -1;
  if (m == 0 || n == 0) return 0;
  int32_t tA, tB;
  if (oracle_oz2_budget(N, k, 1, &tA, &tB) < 2) return -2;
  int32_t *eA = malloc(sizeof(int32_t) * (size_t)m), *eB = malloc(sizeof(int32_t) * (size_t)n);
  int8_t *RA3 = malloc((size_t)3 * N * m * k), *RB3 = malloc((size_t)3 * N * n * k);
  int8_t *CZ = malloc((size_t)2 * N * m * n);
  double *X = malloc(sizeof(double) * 2 * (size_t)m * n); /* unit-scaled re, im before alpha/beta */
  oracle_row_exponents_z(m, k, A, lda, eA);
  oracle_col_exponents_z(k, n, B, ldb, eB);
  oracle_oz2_residues_z(m, k, A, lda, 0, eA, tA, N, RA3);
  oracle_oz2_residues_z(n, k, B, ldb, 1, eB, tB, N, RB3);
  oracle_oz2_modprod_3m(m, n, k, N, RA3, RB3, CZ);
  /* CRT each part, then complex alpha/beta in __float128 with one rounding per part. */
  int32_t mod[ORACLE_MAX_MODULI];
  oracle_oz2_moduli(N, mod);
  u256 P = oz2_P(N, mod), w[ORACLE_MAX_MODULI];
  oz2_weights(N, mod, &P, w);
  int64_t pc = (int64_t)N * m * n;
  (void)X;
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < m; ++i)
    for (int64_t j = 0; j < n; ++j) {
      __float128 v[2];
      for (int part = 0; part < 2; ++part) {
        int c[ORACLE_MAX_MODULI];
        for (int l = 0; l < N; ++l) c[l] = CZ[part * pc + ((int64_t)l * m + i) * n + j];
        u256 mag;
        int sg = oz2_crt_one(N, mod, &P, w, c, &mag);
        v[part] = scalbnq(u256_to_q(&mag), eA[i] + eB[j] - tA - tB);
        if (sg < 0) v[part] = -v[part];
      }
      __float128 ar = alpha[0], ai = alpha[1];
      __float128 rr = ar * v[0] - ai * v[1], ri = ar * v[1] + ai * v[0];
      double *dst = C + 2 * (i * ldc + j);
      if (beta_[0] != 0.0 || beta_[1] != 0.0) {
        __float128 br = beta_[0], bi = beta_[1], cr = dst[0], ci = dst[1];
        rr += br * cr - bi * ci;
        ri += br * ci + bi * cr;
      }
      dst[0] = (double)rr;
      dst[1] = (double)ri;
    }
  free(eA); free(eB); free(RA3); free(RB3); free(CZ); free(X);
  return 0;
}

/* Sampled Scheme II outputs for large sizes (beta_ = 0): real (is3m = 0, out
 * [nr][nc]) or complex 3M (is3m = 1, out [nr][nc][2]).  A/B are real or complex
 * accordingly.  Only the sampled rows of A and columns of B are touched. */
int oracle_oz2_sampled(int64_t k, const double *alpha, const double *A, int64_t lda, const double *B,
                       int64_t ldb, int N, int is3m, int64_t nr, const int64_t *rows, int64_t nc,
                       const int64_t *cols, double *out) {
  int cw = is3m ? 2 : 1;
  double *Ar = malloc(sizeof(double) * cw * (size_t)nr * k), *Bc = malloc(sizeof(double) * cw * (size_t)k * nc);
  for (int64_t r = 0; r < nr; ++r) memcpy(Ar + cw * r * k, A + cw * rows[r] * lda, sizeof(double) * cw * (size_t)k);
  for (int64_t h = 0; h < k; ++h)
    for (int64_t c = 0; c < nc; ++c)
      for (int q = 0; q < cw; ++q) Bc[cw * (h * nc + c) + q] = B[cw * (h * ldb + cols[c]) + q];
  int rc;
  if (is3m) {
    double beta0[2] = {0.0, 0.0};
    rc = oracle_zgemm_oz2_3m(nr, nc, k, alpha, Ar, k, Bc, nc, beta0, out, nc, N);
  } else {
    rc = oracle_dgemm_oz2(nr, nc, k, alpha[0], Ar, k, Bc, nc, 0.0, out, nc, N);
  }
  free(Ar); free(Bc);
  return rc;
}
