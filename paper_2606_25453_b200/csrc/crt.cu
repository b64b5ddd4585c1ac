// crt.cu -- Scheme II reconstruction in FP64, EXACT for every residue vector.
//
// What it computes (Eq. 8): C' = sum_l w_l c_l mod P mapped to
// (-P/2, P/2], w_l = (P/m_l) ((P/m_l)^-1 mod m_l), then C = alpha C' 2^(eA_i+eB_j-tA-tB) + beta C.
// The paper uses a separate multi-word-integer kernel; north_star asks for FP64.
//
// Round 1 split every weight in a 41-bit head and a ROUNDED tail, which left an absolute error of ~2^(E-82) (E = bit
// length of P) whatever the size of C': outside the 2-ulp tolerance as soon as (|A'||B'|)_ij is far below P.  The
// scheme of crt_dev.cuh never rounds before the final conversion (pairs of moduli on the integer pipe, balanced-digit
// FP64 accumulators that stay exact, one rounding of the carry-normalised digits).  This file: the host-side constants
// (256-bit integers) and the stand-alone kernel; the fused Scheme II kernel (gemm_oz2.cu) uses the same device code.
#include "common.cuh"
#include "crt_dev.cuh"

namespace emu {

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
static int big_bit(const Big256 &b, int i) { return i < 256 ? static_cast<int>((b.w[i >> 5] >> (i & 31)) & 1u) : 0; }
// balanced base-2^g digits of v (v < 2^(J g - 1)): v = sum_j d_j 2^(j g), |d_j| <= 2^(g-1); returns false if v does not fit
static bool big_balanced_digits(const Big256 &v, int g, int J, long long *d) {
  long long carry = 0;
  for (int j = 0; j < J; ++j) {
    long long x = 0;
    for (int b = g - 1; b >= 0; --b) x = (x << 1) | big_bit(v, j * g + b);
    x += carry;
    carry = 0;
    if (j + 1 < J && x >= (1LL << (g - 1))) { x -= (1LL << g); carry = 1; }
    d[j] = x;
  }
  if (big_bitlen(v) > J * g) return false;
  return d[J - 1] <= (1LL << (g - 1)) && d[J - 1] >= 0;
}
static long long inv_mod(long long a, long long m) {  // a^-1 mod m (gcd(a, m) = 1), m > 1
  long long g0 = m, g1 = a % m, s0 = 0, s1 = 1;
  while (g1) {
    const long long q = g0 / g1;
    long long t = g0 - q * g1; g0 = g1; g1 = t;
    t = s0 - q * s1; s0 = s1; s1 = t;
  }
  return ((s0 % m) + m) % m;
}

// Pair moduli, digit width, digit count and all constants for n_moduli = N.  Returns false for an unsupported N.
bool crt_constants_host(int N, CrtConst &c) {
  if (N < 1 || N > kMaxModuli) return false;
  int mod[24];
  oz2_moduli_host(N, mod);
  Big256 P = big_one();
  for (int l = 0; l < N; ++l) big_mul_small(P, static_cast<uint32_t>(mod[l]));
  const int E = big_bitlen(P);
  const int NP = (N + 1) / 2;
  // sum of the largest pair residues: x_q <= M_q - 1
  long long xsum = 2;
  for (int q = 0; q < NP; ++q) {
    const long long m1 = mod[2 * q], m2 = (2 * q + 1 < N) ? mod[2 * q + 1] : 1;
    xsum += m1 * m2 - 1;
  }
  int g = 40;
  while (g > 8 && (static_cast<unsigned __int128>(xsum) << g) > (static_cast<unsigned __int128>(1) << 52)) --g;
  const int J = (E + 1 + g - 1) / g;  // J g >= E + 1: the top digit of anything below P stays within 2^(g-1)
  if (J > kCrtMaxJ) return false;
  c.NP = NP; c.N = N; c.J = J; c.g = g;
  const int SC = kCrtSC;
  long long d[kCrtMaxJ];
  if (!big_balanced_digits(P, g, J, d)) return false;
  // 1 / P as a double (53 correct bits are far more than the quotient needs): from the top 64 bits of P
  unsigned long long top = 0;
  const int sh = E > 64 ? E - 64 : 0;
  for (int b = 63; b >= 0; --b) top = (top << 1) | static_cast<unsigned>(big_bit(P, sh + b));
  const double Pd = __builtin_ldexp(static_cast<double>(top), sh);
  for (int j = 0; j < kCrtMaxJ; ++j) {
    c.pd[j] = j < J ? __builtin_ldexp(static_cast<double>(d[j]), SC) : 0.0;
    c.qc[j] = j < J ? __builtin_ldexp(1.0 / Pd, j * g - SC) : 0.0;
  }
  for (int q = 0; q < kMaxPairs; ++q) {
    for (int j = 0; j < kCrtMaxJ; ++j) c.wd[q][j] = 0.0;
    c.kpack[q] = 0; c.c0[q] = 0; c.magic[q] = 0; c.mq[q] = 1;
    if (q >= NP) continue;
    const uint32_t m1 = static_cast<uint32_t>(mod[2 * q]);
    const uint32_t m2 = (2 * q + 1 < N) ? static_cast<uint32_t>(mod[2 * q + 1]) : 1u;
    const uint32_t Mq = m1 * m2;
    // two-modulus CRT weights: K1 == 1 mod m1, == 0 mod m2; K2 the other way round (a single modulus: K1 = 1, K2 = 0)
    const uint32_t K1 = m2 > 1 ? m2 * static_cast<uint32_t>(inv_mod(m2 % m1, m1)) : 1u;
    const uint32_t K2 = m2 > 1 ? m1 * static_cast<uint32_t>(inv_mod(m1 % m2, m2)) : 0u;
    c.kpack[q] = K1 | (K2 << 16);
    c.c0[q] = ((1u << 24) + Mq - 1u) / Mq * Mq;                // |K1 c1 + K2 c2| < 2^24
    c.magic[q] = static_cast<unsigned>((1ull << 32) / Mq);     // floor: the quotient estimate never exceeds the quotient
    c.mq[q] = Mq;
    Big256 W = P;
    big_div_small(W, Mq);                        // P / M_q
    Big256 t = W;
    const uint32_t r = big_div_small(t, Mq);     // (P / M_q) mod M_q
    const uint32_t inv = Mq > 1 ? static_cast<uint32_t>(inv_mod(r, Mq)) : 1u;
    big_mul_small(W, inv);                       // W_q = (P / M_q) ((P / M_q)^-1 mod M_q) < P
    if (!big_balanced_digits(W, g, J, d)) return false;
    for (int j = 0; j < J; ++j) c.wd[q][j] = __builtin_ldexp(static_cast<double>(d[j]), 1074 + SC);
  }
  c.c_norm = __builtin_ldexp(1.0, -g - SC);
  c.c_g = __builtin_ldexp(1.0, g);
  c.c_gsc = __builtin_ldexp(1.0, g + SC);
  c.c_sc = __builtin_ldexp(1.0, SC);
  return true;
}

// Host-only test hook (emugemm_dbg_crt_constants): the integers behind the constants, for the CPU-side check against
// Python big integers.  digits: [(NP + 1)][J] int64, row q < NP = W_q, row NP = P; pair: [NP][5] = M_q, K1, K2, C0, magic.
int crt_constants_dump(int N, int *NP, int *J, int *g, long long *digits, unsigned *pair) {
  CrtConst c;
  if (!crt_constants_host(N, c)) return -1;
  *NP = c.NP; *J = c.J; *g = c.g;
  for (int q = 0; q <= c.NP; ++q)
    for (int j = 0; j < c.J; ++j) {
      const double v = q < c.NP ? __builtin_ldexp(c.wd[q][j], -(1074 + kCrtSC)) : __builtin_ldexp(c.pd[j], -kCrtSC);
      digits[q * c.J + j] = static_cast<long long>(v);
    }
  for (int q = 0; q < c.NP; ++q) {
    pair[5 * q] = c.mq[q]; pair[5 * q + 1] = c.kpack[q] & 0xFFFFu; pair[5 * q + 2] = c.kpack[q] >> 16;
    pair[5 * q + 3] = c.c0[q]; pair[5 * q + 4] = c.magic[q];
  }
  return 0;
}

// ---- device ------------------------------------------------------------------
constexpr int kCrtVec = 4;  // columns per thread: one 32-bit load per residue plane

// Exact accumulators acc[e][j] (e = column, j = digit) of kCrtVec consecutive columns of one row from the N residue
// planes starting at src (plane stride `plane`).  NP = ceil(N / 2) is a template parameter (the digit count follows
// from it: J = ceil(NP / 2) for the moduli list of R10, checked on the host), so the plane loop, the pair loop and every
// constant index are resolved at compile time; all plane words are requested before the first is consumed.
template <int NP, int J>
__device__ __forceinline__ void crt_accumulate(const CrtConst &k, const int8_t *__restrict__ src, int64_t plane, int64_t j0,
                                               int64_t n, bool vec, double (&acc)[kCrtVec][J]) {
  unsigned w[2 * NP];
#pragma unroll
  for (int l = 0; l < 2 * NP; ++l) {
    w[l] = 0u;
    if (l < 2 * NP - 1 || l < k.N) {  // only the last plane of the last pair can be absent (odd N): uniform
      if (vec) {
        w[l] = __ldg(reinterpret_cast<const unsigned *>(src));
      } else {
        unsigned a = 0;
#pragma unroll
        for (int e = 0; e < 4; ++e)
          if (j0 + e < n) a |= static_cast<unsigned>(static_cast<uint8_t>(src[e])) << (8 * e);
        w[l] = a;
      }
    }
    if (l + 1 < 2 * NP) src += plane;
  }
#pragma unroll
  for (int q = 0; q < NP; ++q) crt_accumulate_pair<J>(k, q, w[2 * q], w[2 * q + 1], acc, q == 0);
}

// one thread per kCrtVec consecutive columns of one row
// KIND: 0 = FP64 C, 1 = complex128 C, 2 = FP32 C (SGEMM), 3 = complex64 C (CGEMM); 2 and 3 round once more to float
template <int NP, int KIND>
__global__ void __launch_bounds__(256) crt_kernel(int64_t m, int64_t n, const int8_t *__restrict__ CR,
                                                  const int32_t *__restrict__ eA, const int32_t *__restrict__ eB,
                                                  int tsum, double ar, double ai, double br, double bi,
                                                  double *__restrict__ C, int64_t ldc, const __grid_constant__ CrtConst k,
                                                  int64_t c_entry_bytes, int vec_flag) {
  constexpr int J = (NP + 1) / 2;
  const bool VEC = vec_flag != 0;  // n % 4 == 0 and the residue planes 4-byte aligned: one 32-bit load per plane
  const int64_t ncolv = (n + kCrtVec - 1) / kCrtVec;
  const int64_t idx = static_cast<int64_t>(blockIdx.x) * 256 + threadIdx.x;
  if (idx >= m * ncolv) return;
  int64_t i, j0;
  if (m * ncolv < (1LL << 32)) {  // uniform: 32-bit division (the 64-bit one is ~50 instructions per thread)
    const unsigned iu = static_cast<unsigned>(idx) / static_cast<unsigned>(ncolv);
    i = iu;
    j0 = static_cast<int64_t>(static_cast<unsigned>(idx) - iu * static_cast<unsigned>(ncolv)) * kCrtVec;
  } else {
    i = idx / ncolv;
    j0 = (idx - i * ncolv) * kCrtVec;
  }
  // batch entry blockIdx.y: CR is [N][batch][m][n], the exponents are stacked entry-major
  const int64_t plane = m * n * gridDim.y;
  CR += static_cast<int64_t>(blockIdx.y) * m * n;
  eA += static_cast<int64_t>(blockIdx.y) * m;
  eB += static_cast<int64_t>(blockIdx.y) * n;
  C = reinterpret_cast<double *>(reinterpret_cast<char *>(C) + static_cast<int64_t>(blockIdx.y) * c_entry_bytes);
  const int eAi = __ldg(eA + i) - tsum - kCrtSC;
  int E2[kCrtVec];
#pragma unroll
  for (int e = 0; e < kCrtVec; ++e) E2[e] = eAi + ((j0 + e < n) ? __ldg(eB + j0 + e) : 0);
  double acc[kCrtVec][J], vr[kCrtVec];
  crt_accumulate<NP, J>(k, CR + i * n + j0, plane, j0, n, VEC, acc);
#pragma unroll
  for (int e = 0; e < kCrtVec; ++e) vr[e] = crt_scale_pow2(crt_finish<J>(k, acc[e]), E2[e]);
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
      *reinterpret_cast<float4 *>(o) = make_float4(f[0], f[1], f[2], f[3]);
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
    } else if (ar != 1.0) {
#pragma unroll
      for (int e = 0; e < kCrtVec; ++e) vr[e] *= ar;
    }
    if (VEC && (ldc % 4 == 0) && ((reinterpret_cast<uintptr_t>(C) & 31) == 0)) {
      asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(o), "d"(vr[0]), "d"(vr[1]), "d"(vr[2]), "d"(vr[3]) : "memory");
    } else if (VEC && (ldc % 2 == 0) && ((reinterpret_cast<uintptr_t>(C) & 15) == 0)) {
      *reinterpret_cast<double2 *>(o) = make_double2(vr[0], vr[1]);
      *reinterpret_cast<double2 *>(o + 2) = make_double2(vr[2], vr[3]);
    } else {
#pragma unroll
      for (int e = 0; e < kCrtVec; ++e)
        if (j0 + e < n) o[e] = vr[e];
    }
  } else {
    double vi[kCrtVec];
    crt_accumulate<NP, J>(k, CR + static_cast<int64_t>(k.N) * plane + i * n + j0, plane, j0, n, VEC, acc);
#pragma unroll
    for (int e = 0; e < kCrtVec; ++e) vi[e] = crt_scale_pow2(crt_finish<J>(k, acc[e]), E2[e]);
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

template <int NP>
static void crt_launch_np(dim3 grid, cudaStream_t st, bool vec, int kind, const Oz2CrtArgs &a, int tsum, const CrtConst &k,
                          int64_t c_entry_bytes) {
#define EMU_CRT_LAUNCH(K_)                                                                                                \
  crt_kernel<NP, K_><<<grid, 256, 0, st>>>(a.m, a.n, a.CR, a.eA, a.eB, tsum, a.alpha[0], a.alpha[1], a.beta[0], a.beta[1], a.C, \
                                           a.ldc, k, c_entry_bytes, vec ? 1 : 0)
  switch (kind) {
    case 0: EMU_CRT_LAUNCH(0); break;
    case 1: EMU_CRT_LAUNCH(1); break;
    case 2: EMU_CRT_LAUNCH(2); break;
    default: EMU_CRT_LAUNCH(3); break;
  }
#undef EMU_CRT_LAUNCH
}

int launch_oz2_crt(emugemm_ctx *ctx, const Oz2CrtArgs &a) {
  if (a.m == 0 || a.n == 0) return EMUGEMM_OK;
  CrtConst k;
  if (!crt_constants_host(a.n_moduli, k)) return EMUGEMM_ERR_ARG;
  const int kind = a.is_complex ? (a.out_f32 ? 3 : 1) : (a.out_f32 ? 2 : 0);
  const int64_t work = a.m * ((a.n + kCrtVec - 1) / kCrtVec);
  const unsigned gx = static_cast<unsigned>((work + 255) / 256);
  const bool vec = (a.n % kCrtVec == 0) && ((reinterpret_cast<uintptr_t>(a.CR) & (kCrtVec - 1)) == 0);
  const int tsum = a.tA + a.tB;
  const int batch = a.batch > 0 ? a.batch : 1;
  if (batch > 65535) return EMUGEMM_ERR_ARG;
  // bytes between the C matrices of consecutive batch entries (element = float / double, x2 for complex)
  const int64_t c_entry_bytes = a.batch_stride_c * (a.out_f32 ? 4 : 8) * (a.is_complex ? 2 : 1);
  const dim3 grid(gx, static_cast<unsigned>(batch));
  if (k.J != (k.NP + 1) / 2) return EMUGEMM_ERR_ARG;  // the kernels derive the digit count from the pair count
  switch (k.NP) {
    case 1: crt_launch_np<1>(grid, ctx->stream, vec, kind, a, tsum, k, c_entry_bytes); break;
    case 2: crt_launch_np<2>(grid, ctx->stream, vec, kind, a, tsum, k, c_entry_bytes); break;
    case 3: crt_launch_np<3>(grid, ctx->stream, vec, kind, a, tsum, k, c_entry_bytes); break;
    case 4: crt_launch_np<4>(grid, ctx->stream, vec, kind, a, tsum, k, c_entry_bytes); break;
    case 5: crt_launch_np<5>(grid, ctx->stream, vec, kind, a, tsum, k, c_entry_bytes); break;
    case 6: crt_launch_np<6>(grid, ctx->stream, vec, kind, a, tsum, k, c_entry_bytes); break;
    case 7: crt_launch_np<7>(grid, ctx->stream, vec, kind, a, tsum, k, c_entry_bytes); break;
    case 8: crt_launch_np<8>(grid, ctx->stream, vec, kind, a, tsum, k, c_entry_bytes); break;
    case 9: crt_launch_np<9>(grid, ctx->stream, vec, kind, a, tsum, k, c_entry_bytes); break;
    default: crt_launch_np<10>(grid, ctx->stream, vec, kind, a, tsum, k, c_entry_bytes); break;
  }
  ctx->launches++;
  EMU_CUDA(ctx, cudaGetLastError());
  return EMUGEMM_OK;
}

}  // namespace emu
