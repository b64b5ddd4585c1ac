// crt_dev.cuh -- device side of the exact FP64 CRT (Eq. 8; R17), shared by the
// stand-alone reconstruction kernel (crt.cu) and the fused Scheme II kernel (gemm_oz2.cu).
//
//   1. Moduli are combined in PAIRS on the integer pipe (an odd last modulus stays alone).  With the signed INT8
//      residues c1, c2 of the pair (m1, m2), M = m1 m2 and the two-modulus CRT weights K1 = m2 (m2^-1 mod m1),
//      K2 = m1 (m1^-1 mod m2) (both < 2^16):
//        s = K1 c1 + K2 c2 + C0          one IDP.2A (C0 = a multiple of M above 2^24 keeps s positive)
//        x = s mod M  in [0, M)          multiply-high by floor(2^32 / M) (quotient at most one too small), one
//                                        multiply-add, one fused add-min;   x == c1 mod m1,  x == c2 mod m2
//      so the FP64 part sees ceil(N/2) residues of 16 bits.
//   2. Every pair weight W_q = (P/M_q)((P/M_q)^-1 mod M_q) and P are written in BALANCED base-2^g digits
//      (|digit| <= 2^(g-1), g chosen on the host so that 2^g (sum_q (M_q - 1) + 2) <= 2^52).  x_q enters the FMAs as
//      the SUBNORMAL double whose bit pattern is the integer itself (no int -> double conversion instruction); the
//      digits carry the compensating power of two, so every accumulator holds (integer) 2^SC, |integer| < 2^52:
//        acc_j = sum_q W_qj x_q                                  -- exact
//        Q     = rint(sum_j acc_j 2^(jg) / P)  (two top digits)  -- |true C'| < P/4 (R12) keeps it 1/4 from a tie
//        T_j   = acc_j - Q P_j                                   -- exact (one FMA each)
//      and C' = sum_j T_j 2^(jg) exactly.
//   3. The T_j are carry-normalised to balanced digits (exact), summed from the top with a compensated Horner
//      scheme (Fast2Sum is valid because a nonzero leading digit dominates everything below it) and hi + lo is
//      rounded ONCE: C' is the correctly rounded big integer for EVERY residue vector.
//   4. 2^(eA_i + eB_j - tA - tB) is applied as two factors, the first clamped so that it can neither overflow nor
//      underflow: results down to the subnormal range are rounded once.
#pragma once
#include "common.cuh"

namespace emu {

constexpr int kMaxPairs = (kMaxModuli + 1) / 2;
constexpr int kCrtMaxJ = 5;
constexpr int kCrtSC = -94;  // accumulators hold integer * 2^kCrtSC: x enters as x 2^-1074, digits carry 2^(1074 + kCrtSC)

struct CrtConst {
  double wd[kMaxPairs][kCrtMaxJ];  // balanced digits of W_q times 2^(1074 + SC)
  double pd[kCrtMaxJ];             // balanced digits of P times 2^SC
  double qc[kCrtMaxJ];             // 2^(j g - SC) / P: Q = rint(sum_j acc_j qc_j)
  double c_norm;                   // 2^(-g - SC): T_j -> carry estimate at scale 1
  double c_g;                      // 2^g
  double c_gsc;                    // 2^(g + SC)
  double c_sc;                     // 2^SC
  unsigned kpack[kMaxPairs];       // K1 | K2 << 16
  unsigned c0[kMaxPairs];          // multiple of M_q in [2^24, 2^24 + M_q)
  unsigned magic[kMaxPairs];       // floor(2^32 / M_q)
  unsigned mq[kMaxPairs];          // M_q
  int NP, N, J, g;
};

// host (crt.cu): pair moduli, digit width, digit count and all constants for n_moduli = N; false for an unsupported N
bool crt_constants_host(int N, CrtConst &c);

// d = a.lo16 * (signed byte 0 of b) + a.hi16 * (signed byte 1 of b) + c   (a: unsigned halves)
__device__ __forceinline__ int dp2a_lo_u16_s8(unsigned a, unsigned b, int c) {
  int d;
  asm("dp2a.lo.u32.s32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
  return d;
}
__device__ __forceinline__ int dp2a_hi_u16_s8(unsigned a, unsigned b, int c) {  // bytes 2, 3 of b
  int d;
  asm("dp2a.hi.u32.s32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
  return d;
}

// pair residue x in [0, M) of the signed bytes (c1, c2) held in bytes (0, 1) [HI = false] or (2, 3) [HI = true] of w
template <bool HI>
__device__ __forceinline__ unsigned crt_pair_residue(unsigned w, unsigned kpack, unsigned c0, unsigned magic, unsigned mq) {
  const unsigned s = static_cast<unsigned>(HI ? dp2a_hi_u16_s8(kpack, w, static_cast<int>(c0)) : dp2a_lo_u16_s8(kpack, w, static_cast<int>(c0)));
  const unsigned x = s - __umulhi(s, magic) * mq;  // in [0, 2M): the quotient estimate is at most one too small
  return min(x, x - mq);                           // unsigned: x - M wraps above x when x < M
}

__device__ __forceinline__ double crt_round_nearest(double x) {  // |x| < 2^51: round to nearest even without F2F (XU pipe)
  const double big = 6755399441055744.0;  // 1.5 * 2^52
  return (x + big) - big;
}

// acc[e][j] += W_qj x for the four columns e whose residues are the bytes of wa (modulus 2q) and wb (modulus 2q + 1)
// (first = true: acc is initialised with the product instead of being added to)
template <int J>
__device__ __forceinline__ void crt_accumulate_pair(const CrtConst &k, int q, unsigned wa, unsigned wb, double (&acc)[4][J],
                                                    bool first = false) {
  const unsigned kp = k.kpack[q], c0 = k.c0[q], mg = k.magic[q], mq = k.mq[q];
  const unsigned w01 = __byte_perm(wa, wb, 0x5140);  // (c1, c2) of column 0, (c1, c2) of column 1
  const unsigned w23 = __byte_perm(wa, wb, 0x7362);
  const unsigned x[4] = {crt_pair_residue<false>(w01, kp, c0, mg, mq), crt_pair_residue<true>(w01, kp, c0, mg, mq),
                         crt_pair_residue<false>(w23, kp, c0, mg, mq), crt_pair_residue<true>(w23, kp, c0, mg, mq)};
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    const double xd = __hiloint2double(0, static_cast<int>(x[e]));  // the subnormal x 2^-1074: no conversion instruction
#pragma unroll
    for (int j = 0; j < J; ++j) acc[e][j] = first ? k.wd[q][j] * xd : fma(k.wd[q][j], xd, acc[e][j]);
  }
}

// t (exact digits of sum_q W_q x_q, scaled by 2^SC) -> the correctly rounded C' 2^SC
template <int J>
__device__ __forceinline__ double crt_finish(const CrtConst &k, double (&t)[J]) {
  // quotient from the two leading digits: the rest contributes < 2^(54 - 3g) of a unit
  double v = t[J - 1] * k.qc[J - 1];
  if (J > 1) v = fma(t[J - 2], k.qc[J - 2], v);
  const double Q = crt_round_nearest(v);
#pragma unroll
  for (int j = 0; j < J; ++j) t[j] = fma(-Q, k.pd[j], t[j]);  // exact: |T_j| < 2^52 2^SC
  // carry normalisation to balanced digits (all operations exact)
#pragma unroll
  for (int j = 0; j + 1 < J; ++j) {
    const double big = 6755399441055744.0;  // 1.5 * 2^52: rint of the exactly scaled digit
    const double c = fma(t[j], k.c_norm, big) - big;
    t[j] = fma(-c, k.c_gsc, t[j]);
    t[j + 1] = fma(c, k.c_sc, t[j + 1]);
  }
  // compensated Horner from the top: (hi, lo) <- (hi, lo) 2^g + t_j; Fast2Sum is valid because |hi 2^g| >= 2^g 2^SC
  // > |t_j| whenever hi != 0, and hi == 0 gives s = t_j, err = 0
  double hi = t[J - 1], lo = 0.0;
#pragma unroll
  for (int j = J - 2; j >= 0; --j) {
    const double s = fma(hi, k.c_g, t[j]);
    const double err = fma(hi, k.c_g, -s) + t[j];
    lo = (j == J - 2) ? err : fma(lo, k.c_g, err);
    hi = s;
  }
  return hi + lo;
}

// 2^e for -1022 <= e <= 1023
__device__ __forceinline__ double crt_pow2(int e) { return __hiloint2double((1023 + e) << 20, 0); }
// v * 2^E for |v| in [2^-100, 2^90] or v == 0, rounded once: the first factor is clamped so that v 2^h1 stays a normal
// number, the second (clamped to the exponent range) takes the result to zero / subnormal / infinity when it must
__device__ __forceinline__ double crt_scale_pow2(double v, int E) {
  const int h1 = max(min(E, 930), -920);
  const int h2 = max(min(E - h1, 1023), -1022);
  return (v * crt_pow2(h1)) * crt_pow2(h2);
}

}  // namespace emu
