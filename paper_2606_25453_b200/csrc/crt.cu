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
// Integer -> double conversions (I2F.F64) and rint (F2F) run on the XU pipe, which ncu showed saturated
// (108 %) by the first version of this kernel at 1 conversion / clk / SM; both are replaced by exponent-bias
// additions on the FP64 pipe (profiles/).
__device__ __forceinline__ double pow2_dev(int e) { return __hiloint2double((1023 + e) << 20, 0); }
// exact double of residue byte i of wx, where wx = w ^ 0x80808080 holds c + 128 in [0, 255] per byte:
// one byte permute + one FP64 addition: (2^52 + c + 128) - (2^52 + 128)
__device__ __forceinline__ double residue_to_double(unsigned wx, int i) {
  const unsigned biased = __byte_perm(wx, 0u, 0x4440u | static_cast<unsigned>(i));
  return __hiloint2double(0x43300000, static_cast<int>(biased)) - 4503599627370624.0;
}
__device__ __forceinline__ double round_nearest(double x) {  // |x| < 2^51: round to nearest even without F2F
  const double big = 6755399441055744.0;  // 1.5 * 2^52
  return (x + big) - big;
}

// columns per thread: 8 (one 8-byte load per residue plane) for real outputs, 4 for complex ones, whose second
// accumulation pass otherwise pushes the kernel to 153 registers / 12 % occupancy (profiles/r1_prepass_v2.md)

template <bool VEC, int kCrtVec>
__device__ __forceinline__ void crt_accumulate(const CrtConst &k, const int8_t *__restrict__ src, int64_t plane, int64_t j0,
                                               int64_t n, double (&shi)[kCrtVec], double (&slo)[kCrtVec]) {
  // all residue planes are requested before any is consumed: up to 20 independent 8-byte loads in flight per
  // thread (the first version interleaved load and use and stalled on the long scoreboard, ncu)
  unsigned w0[kMaxModuli], w1[kMaxModuli];
#pragma unroll
  for (int l = 0; l < kMaxModuli; ++l) {
    w0[l] = w1[l] = 0x80808080u;
    if (l < k.N) {
      if (VEC && kCrtVec == 8) {
        const uint2 w = __ldg(reinterpret_cast<const uint2 *>(src + l * plane));
        w0[l] = w.x; w1[l] = w.y;
      } else if (VEC) {
        w0[l] = __ldg(reinterpret_cast<const unsigned *>(src + l * plane));
      } else {
        unsigned a = 0, b = 0;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          if (j0 + e < n) a |= static_cast<unsigned>(static_cast<uint8_t>(src[l * plane + e])) << (8 * e);
          if (kCrtVec == 8 && j0 + 4 + e < n) b |= static_cast<unsigned>(static_cast<uint8_t>(src[l * plane + 4 + e])) << (8 * e);
        }
        w0[l] = a; w1[l] = b;
      }
    }
  }
#pragma unroll
  for (int e = 0; e < kCrtVec; ++e) { shi[e] = 0.0; slo[e] = 0.0; }
#pragma unroll
  for (int l = 0; l < kMaxModuli; ++l) {
    if (l < k.N) {
      const unsigned x0 = w0[l] ^ 0x80808080u, x1 = w1[l] ^ 0x80808080u;
#pragma unroll
      for (int e = 0; e < kCrtVec; ++e) {
        const double cl = residue_to_double(e < 4 ? x0 : x1, e & 3);
        shi[e] = fma(k.whi[l], cl, shi[e]);
        slo[e] = fma(k.wlo[l], cl, slo[e]);
      }
    }
  }
}

__device__ __forceinline__ double crt_finish(const CrtConst &k, double shi, double slo) {
  const double Q = round_nearest((shi + slo) * k.invP);
  return fma(-Q, k.Phi, shi) + fma(-Q, k.Plo, slo);
}

// one thread per 8 consecutive columns of one row
// KIND: 0 = FP64 C, 1 = complex128 C, 2 = FP32 C (SGEMM), 3 = complex64 C (CGEMM); 2 and 3 round once more to float
template <bool VEC, int KIND, int kCrtVec>
__global__ void __launch_bounds__(256) crt_kernel(int64_t m, int64_t n, const int8_t *__restrict__ CR,
                                                  const int32_t *__restrict__ eA, const int32_t *__restrict__ eB,
                                                  int tsum, double ar, double ai, double br, double bi,
                                                  double *__restrict__ C, int64_t ldc, const CrtConst k,
                                                  int64_t c_entry_bytes) {
  const int64_t ncolv = (n + kCrtVec - 1) / kCrtVec;
  const int64_t idx = static_cast<int64_t>(blockIdx.x) * 256 + threadIdx.x;
  if (idx >= m * ncolv) return;
  const int64_t i = idx / ncolv, j0 = (idx - i * ncolv) * kCrtVec;
  // batch entry blockIdx.y: CR is [N][batch][m][n], the exponents are stacked entry-major
  const int64_t plane = m * n * gridDim.y;
  CR += static_cast<int64_t>(blockIdx.y) * m * n;
  eA += static_cast<int64_t>(blockIdx.y) * m;
  eB += static_cast<int64_t>(blockIdx.y) * n;
  C = reinterpret_cast<double *>(reinterpret_cast<char *>(C) + static_cast<int64_t>(blockIdx.y) * c_entry_bytes);
  const int eAi = eA[i] - tsum;
  double sc1[kCrtVec], sc2[kCrtVec];
#pragma unroll
  for (int e = 0; e < kCrtVec; ++e) {
    const int E2 = eAi + ((j0 + e < n) ? __ldg(eB + j0 + e) : 0);
    sc1[e] = pow2_dev(E2 >> 1);
    sc2[e] = pow2_dev(E2 - (E2 >> 1));
  }
  double shi[kCrtVec], slo[kCrtVec], vr[kCrtVec];
  crt_accumulate<VEC, kCrtVec>(k, CR + i * n + j0, plane, j0, n, shi, slo);
#pragma unroll
  for (int e = 0; e < kCrtVec; ++e) vr[e] = crt_finish(k, shi[e], slo[e]) * sc1[e] * sc2[e];
  if (KIND == 2) {
    float *o = reinterpret_cast<float *>(C) + i * ldc + j0;
    float f[kCrtVec];
#pragma unroll
    for (int e = 0; e < kCrtVec; ++e) {
      double x = ar * vr[e];
      if (br != 0.0 && j0 + e < n) x = fma(br, static_cast<double>(o[e]), x);
      f[e] = static_cast<float>(x);
    }
    if (VEC && (ldc % 4 == 0) && ((reinterpret_cast<uintptr_t>(C) & 15) == 0)) {
#pragma unroll
      for (int e = 0; e < kCrtVec; e += 4) reinterpret_cast<float4 *>(o)[e / 4] = make_float4(f[e], f[e + 1], f[e + 2], f[e + 3]);
    } else {
#pragma unroll
      for (int e = 0; e < kCrtVec; ++e)
        if (j0 + e < n) o[e] = f[e];
    }
  } else if (KIND == 0) {
    double *o = C + i * ldc + j0;
    if (br != 0.0) {
#pragma unroll
      for (int e = 0; e < kCrtVec; ++e)
        if (j0 + e < n) vr[e] = fma(ar, vr[e], br * o[e]);
    } else {
#pragma unroll
      for (int e = 0; e < kCrtVec; ++e) vr[e] *= ar;
    }
    if (VEC && (ldc % 2 == 0) && ((reinterpret_cast<uintptr_t>(C) & 15) == 0)) {
#pragma unroll
      for (int e = 0; e < kCrtVec; e += 2) *reinterpret_cast<double2 *>(o + e) = make_double2(vr[e], vr[e + 1]);
    } else {
#pragma unroll
      for (int e = 0; e < kCrtVec; ++e)
        if (j0 + e < n) o[e] = vr[e];
    }
  } else {
    double vi[kCrtVec];
    crt_accumulate<VEC, kCrtVec>(k, CR + static_cast<int64_t>(k.N) * plane + i * n + j0, plane, j0, n, shi, slo);
#pragma unroll
    for (int e = 0; e < kCrtVec; ++e) vi[e] = crt_finish(k, shi[e], slo[e]) * sc1[e] * sc2[e];
    const bool has_beta = (br != 0.0 || bi != 0.0);
    if (KIND == 3) {  // complex64 C: float pairs
      float *o = reinterpret_cast<float *>(C) + 2 * (i * ldc + j0);
#pragma unroll
      for (int e = 0; e < kCrtVec; ++e) {
        if (j0 + e >= n) break;
        double re = ar * vr[e] - ai * vi[e];
        double im = ar * vi[e] + ai * vr[e];
        if (has_beta) {
          const double cr = o[2 * e], ci = o[2 * e + 1];
          re += br * cr - bi * ci;
          im += br * ci + bi * cr;
        }
        *reinterpret_cast<float2 *>(o + 2 * e) = make_float2(static_cast<float>(re), static_cast<float>(im));
      }
    } else {
      double *o = C + 2 * (i * ldc + j0);
#pragma unroll
      for (int e = 0; e < kCrtVec; ++e) {
        if (j0 + e >= n) break;
        double re = ar * vr[e] - ai * vi[e];
        double im = ar * vi[e] + ai * vr[e];
        if (has_beta) {
          const double cr = o[2 * e], ci = o[2 * e + 1];
          re += br * cr - bi * ci;
          im += br * ci + bi * cr;
        }
        if ((reinterpret_cast<uintptr_t>(C) & 15) == 0) *reinterpret_cast<double2 *>(o + 2 * e) = make_double2(re, im);
        else { o[2 * e] = re; o[2 * e + 1] = im; }
      }
    }
  }
}

int launch_oz2_crt(emugemm_ctx *ctx, const Oz2CrtArgs &a) {
  if (a.m == 0 || a.n == 0) return EMUGEMM_OK;
  CrtConst k;
  crt_constants(a.n_moduli, k);
  const int kind = a.is_complex ? (a.out_f32 ? 3 : 1) : (a.out_f32 ? 2 : 0);
  const int V = a.is_complex ? 4 : 8;  // columns per thread (real outputs with 4: 0.524 -> 0.551 ms, measured)
  const int64_t work = a.m * ((a.n + V - 1) / V);
  const unsigned grid = static_cast<unsigned>((work + 255) / 256);
  const bool vec = (a.n % V == 0) && ((reinterpret_cast<uintptr_t>(a.CR) & (V - 1)) == 0);
  const int tsum = a.tA + a.tB;
  const int batch = a.batch > 0 ? a.batch : 1;
  if (batch > 65535) return EMUGEMM_ERR_ARG;
  // bytes between the C matrices of consecutive batch entries (element = float / double, x2 for complex)
  const int64_t c_entry_bytes = a.batch_stride_c * (a.out_f32 ? 4 : 8) * (a.is_complex ? 2 : 1);
#define EMU_CRT_LAUNCH(V_, Z, W_)                                                                                              \
  crt_kernel<V_, Z, W_><<<dim3(grid, static_cast<unsigned>(batch)), 256, 0, ctx->stream>>>(a.m, a.n, a.CR, a.eA, a.eB, tsum, a.alpha[0], a.alpha[1], a.beta[0], \
                                                   a.beta[1], a.C, a.ldc, k, c_entry_bytes)
  if (vec && kind == 3) EMU_CRT_LAUNCH(true, 3, 4);
  else if (kind == 3) EMU_CRT_LAUNCH(false, 3, 4);
  else if (vec && kind == 1) EMU_CRT_LAUNCH(true, 1, 4);
  else if (vec && kind == 2) EMU_CRT_LAUNCH(true, 2, 8);
  else if (vec) EMU_CRT_LAUNCH(true, 0, 8);
  else if (kind == 1) EMU_CRT_LAUNCH(false, 1, 4);
  else if (kind == 2) EMU_CRT_LAUNCH(false, 2, 8);
  else EMU_CRT_LAUNCH(false, 0, 8);
#undef EMU_CRT_LAUNCH
  ctx->launches++;
  EMU_CUDA(ctx, cudaGetLastError());
  return EMUGEMM_OK;
}

}  // namespace emu
