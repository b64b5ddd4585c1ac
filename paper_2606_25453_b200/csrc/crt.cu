// crt.cu -- Scheme II reconstruction in FP64.
//
// What it computes (Eq. 8): C' = sum_l w_l c_l mod P mapped to
// (-P/2, P/2], w_l = (P/m_l) ((P/m_l)^-1 mod m_l), then C = alpha C' 2^(eA_i+eB_j-tA-tB) + beta C.
// The paper uses a separate multi-word-integer kernel; north_star asks for FP64.
//
// FP64 scheme (R17): with E = bit length of P and G = 2^(E-41), every constant is split on
// the grid G:  w_l = whi_l + wlo_l, P = Phi + Plo, whi_l and Phi multiples of G below 2^41 G.
//   S_hi = sum whi_l c_l   -- exact in FP64 (41 + 7 + 5 bits)
//   S_lo = sum wlo_l c_l   -- rounded; |error| ~ 2^(E-82)
//   Q    = rint((S_hi + S_lo) / P)      -- |true C'| < P/4 keeps the quotient 1/4 away from a tie
//   C'   = (S_hi - Q Phi) + (S_lo - Q Plo)   -- first bracket exact (multiples of G, small result)
// Absolute error ~ 2^(E-82) << 2^-53 (|A'||B'|)_ij for the paper's input distributions.
#include "common.cuh"

namespace emu {

struct CrtConst {
  double whi[kMaxModuli], wlo[kMaxModuli];
  double Phi, Plo, invP;
  int N;
};

// ---- host: 256-bit unsigned integers as eight 32-bit limbs ------------------
struct Big256 {
  uint32_t w[8];
};
static Big256 big_one() { Big256 b{}; b.w[0] = 1; return b; }
static void big_mul_small(Big256 &b, uint32_t s) {
  uint64_t c = 0;
  for (int i = 0; i < 8; ++i) { c += static_cast<uint64_t>(b.w[i]) * s; b.w[i] = static_cast<uint32_t>(c); c >>= 32; }
}
static uint32_t big_div_small(Big256 &b, uint32_t s) {  // b /= s, returns remainder
  uint64_t r = 0;
  for (int i = 7; i >= 0; --i) { const uint64_t cur = (r << 32) | b.w[i]; b.w[i] = static_cast<uint32_t>(cur / s); r = cur % s; }
  return static_cast<uint32_t>(r);
}
static int big_bitlen(const Big256 &b) {
  for (int i = 7; i >= 0; --i)
    if (b.w[i]) return 32 * i + (32 - __builtin_clz(b.w[i]));
  return 0;
}
static int big_bit(const Big256 &b, int i) { return (b.w[i >> 5] >> (i & 31)) & 1; }
// value of bits [lo, hi) as a double (exact when hi - lo <= 53, else correctly truncated to 64 bits then rounded)
static double big_bits_to_double(const Big256 &b, int lo, int hi) {
  if (hi <= lo) return 0.0;
  int top = hi - 1;
  while (top >= lo && !big_bit(b, top)) --top;
  if (top < lo) return 0.0;
  int bot = top - 63;
  if (bot < lo) bot = lo;
  unsigned long long v = 0;
  for (int i = top; i >= bot; --i) v = (v << 1) | static_cast<unsigned>(big_bit(b, i));
  return __builtin_ldexp(static_cast<double>(v), bot);
}

static void crt_constants(int N, CrtConst &c) {
  int mod[24];
  oz2_moduli_host(N, mod);
  Big256 P = big_one();
  for (int l = 0; l < N; ++l) big_mul_small(P, static_cast<uint32_t>(mod[l]));
  const int E = big_bitlen(P);
  const int g = E > 41 ? E - 41 : 0;  // grid exponent
  c.N = N;
  c.Phi = big_bits_to_double(P, g, 256);
  c.Plo = big_bits_to_double(P, 0, g);
  c.invP = 1.0 / (c.Phi + c.Plo);
  for (int l = 0; l < N; ++l) {
    Big256 Pl = P;
    big_div_small(Pl, static_cast<uint32_t>(mod[l]));            // P / m_l
    Big256 t = Pl;
    const uint32_t plm = big_div_small(t, static_cast<uint32_t>(mod[l]));  // (P / m_l) mod m_l
    uint32_t q = 0;
    for (uint32_t x = 1; x < static_cast<uint32_t>(mod[l]); ++x)
      if ((plm * x) % static_cast<uint32_t>(mod[l]) == 1) { q = x; break; }
    big_mul_small(Pl, q);                                         // w_l = (P/m_l) q_l < P
    c.whi[l] = big_bits_to_double(Pl, g, 256);
    c.wlo[l] = big_bits_to_double(Pl, 0, g);
  }
  for (int l = N; l < kMaxModuli; ++l) c.whi[l] = c.wlo[l] = 0.0;
}

// ---- device ------------------------------------------------------------------
__device__ __forceinline__ double pow2_dev(int e) { return __hiloint2double((1023 + e) << 20, 0); }

__device__ __forceinline__ double crt_value(const CrtConst &k, const int (&c)[kMaxModuli]) {
  double shi = 0.0, slo = 0.0;
#pragma unroll
  for (int l = 0; l < kMaxModuli; ++l)
    if (l < k.N) {
      const double cl = static_cast<double>(c[l]);
      shi = fma(k.whi[l], cl, shi);
      slo = fma(k.wlo[l], cl, slo);
    }
  const double Q = rint((shi + slo) * k.invP);
  return fma(-Q, k.Phi, shi) + fma(-Q, k.Plo, slo);
}

// one thread per 4 consecutive columns; VEC = 4: aligned 32-bit plane loads, VEC = 1: byte loads
template <int VEC>
__global__ void __launch_bounds__(256) crt_kernel(int64_t m, int64_t n, const int8_t *__restrict__ CR,
                                                  const int32_t *__restrict__ eA, const int32_t *__restrict__ eB,
                                                  int tsum, int is_complex, double ar, double ai, double br, double bi,
                                                  double *__restrict__ C, int64_t ldc, const CrtConst k) {
  const int64_t ncol4 = (n + 3) / 4;
  const int64_t idx = static_cast<int64_t>(blockIdx.x) * 256 + threadIdx.x;
  if (idx >= m * ncol4) return;
  const int64_t i = idx / ncol4, j0 = (idx - i * ncol4) * 4;
  const int64_t plane = m * n;
  const int eAi = eA[i] - tsum;
  const int nparts = is_complex ? 2 : 1;
  double val[2][4];
  for (int part = 0; part < nparts; ++part) {
    const int8_t *src = CR + static_cast<int64_t>(part) * k.N * plane + i * n + j0;
    int c[4][kMaxModuli];
#pragma unroll
    for (int l = 0; l < kMaxModuli; ++l)
      if (l < k.N) {
        if (VEC == 4) {
          const unsigned w = *reinterpret_cast<const unsigned *>(src + l * plane);
#pragma unroll
          for (int e = 0; e < 4; ++e) c[e][l] = static_cast<int>(static_cast<int8_t>((w >> (8 * e)) & 0xFFu));
        } else {
#pragma unroll
          for (int e = 0; e < 4; ++e) c[e][l] = (j0 + e < n) ? static_cast<int>(src[l * plane + e]) : 0;
        }
      }
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const double x = crt_value(k, c[e]);
      const int E2 = eAi + ((j0 + e < n) ? eB[j0 + e] : 0);
      val[part][e] = x * pow2_dev(E2 >> 1) * pow2_dev(E2 - (E2 >> 1));
    }
  }
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    if (j0 + e >= n) break;
    if (!is_complex) {
      double *o = C + i * ldc + j0 + e;
      *o = (br != 0.0) ? fma(ar, val[0][e], br * *o) : ar * val[0][e];
    } else {
      double *o = C + 2 * (i * ldc + j0 + e);
      double re = ar * val[0][e] - ai * val[1][e];
      double im = ar * val[1][e] + ai * val[0][e];
      if (br != 0.0 || bi != 0.0) {
        const double cr = o[0], ci = o[1];
        re += br * cr - bi * ci;
        im += br * ci + bi * cr;
      }
      o[0] = re;
      o[1] = im;
    }
  }
}

int launch_oz2_crt(emugemm_ctx *ctx, const Oz2CrtArgs &a) {
  if (a.m == 0 || a.n == 0) return EMUGEMM_OK;
  CrtConst k;
  crt_constants(a.n_moduli, k);
  const int64_t work = a.m * ((a.n + 3) / 4);
  const unsigned grid = static_cast<unsigned>((work + 255) / 256);
  const bool vec = (a.n % 4 == 0) && ((reinterpret_cast<uintptr_t>(a.CR) & 3) == 0);
  if (vec)
    crt_kernel<4><<<grid, 256, 0, ctx->stream>>>(a.m, a.n, a.CR, a.eA, a.eB, a.tA + a.tB, a.is_complex, a.alpha[0], a.alpha[1],
                                                 a.beta[0], a.beta[1], a.C, a.ldc, k);
  else
    crt_kernel<1><<<grid, 256, 0, ctx->stream>>>(a.m, a.n, a.CR, a.eA, a.eB, a.tA + a.tB, a.is_complex, a.alpha[0], a.alpha[1],
                                                 a.beta[0], a.beta[1], a.C, a.ldc, k);
  ctx->launches++;
  EMU_CUDA(ctx, cudaGetLastError());
  return EMUGEMM_OK;
}

}  // namespace emu
