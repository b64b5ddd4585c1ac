// prepass.cu -- decomposition kernels: one pass over the operand, one write of
// the planes; the digit kernels end up bound by the ALU pipe, the residue kernels by the integer multiplier
// (profiles/r1_prepass_v2.md).
//
//  * exponent scan: max |x| bit pattern per row of A / per column of B -> frexp
//    exponent ("each row of A is scaled by a power-of-two factor";
//    DESIGN.md R2).
//  * Scheme I slicing (Eq. 1): p signed 7-bit digits per element,
//    integer work on the FP bit pattern only (shift / mask / sign).
//  * Scheme II residues (Eq. 5): a' = trunc(a 2^(t-e)) as a
//    <= 70-bit integer held in three 32-bit words, a' mod m_l by byte dot products
//    against (256^j mod m_l) + one multiply-high reduction, symmetric INT8 range.
//
// Output layout (library-private): int8 planes
// [plane][row][kpad], k contiguous, zero padded to kpad (multiple of 128) so the
// fused GEMMs fetch K-major 128-byte rows with TMA for BOTH operands; operand B
// (k x n row-major) is therefore transposed on the fly through shared memory.
#include "common.cuh"

namespace emu {

// ----------------------------------------------------------------------------
// element decode: |x| = M * 2^ex2 with integer M
// ----------------------------------------------------------------------------
__device__ __forceinline__ void decode_bits(double v, unsigned long long &M, int &ex2, bool &neg) {
  const unsigned long long b = static_cast<unsigned long long>(__double_as_longlong(v));
  neg = (b >> 63) != 0;
  const int E = static_cast<int>((b >> 52) & 0x7FF);
  const unsigned long long frac = b & 0xFFFFFFFFFFFFFull;
  M = E ? (frac | (1ull << 52)) : frac;
  ex2 = (E ? E : 1) - 1075;
}
__device__ __forceinline__ void decode_bits(float v, unsigned long long &M, int &ex2, bool &neg) {
  const unsigned int b = __float_as_uint(v);
  neg = (b >> 31) != 0;
  const int E = static_cast<int>((b >> 23) & 0xFF);
  const unsigned int frac = b & 0x7FFFFFu;
  M = E ? (frac | (1u << 23)) : frac;
  ex2 = (E ? E : 1) - 150;
}
__device__ __forceinline__ unsigned long long abs_bits(double v) {
  return static_cast<unsigned long long>(__double_as_longlong(v)) & 0x7FFFFFFFFFFFFFFFull;
}
__device__ __forceinline__ unsigned long long abs_bits(float v) { return __float_as_uint(v) & 0x7FFFFFFFu; }

// ----------------------------------------------------------------------------
// exponent scan
// ----------------------------------------------------------------------------
template <typename T, int W /* scalars per element: 1 real, 2 complex */>
__global__ void __launch_bounds__(256) rowmax_kernel(const T *__restrict__ X, int64_t ldx, int64_t k,
                                                     unsigned long long *__restrict__ maxbits) {
  const int64_t row = blockIdx.x;
  const T *src = X + row * ldx * W;
  unsigned long long mx = 0;
  for (int64_t h = threadIdx.x; h < k * W; h += 256) {
    const unsigned long long b = abs_bits(src[h]);
    mx = b > mx ? b : mx;
  }
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned long long y = __shfl_xor_sync(0xffffffffu, mx, o);
    mx = y > mx ? y : mx;
  }
  __shared__ unsigned long long red[8];
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = mx;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < 8; ++w) mx = red[w] > mx ? red[w] : mx;
    maxbits[row] = mx;
  }
}

// X is k x rows (ldx), one thread per column, grid.y splits k; atomicMax merges.
template <typename T, int W>
__global__ void __launch_bounds__(256) colmax_kernel(const T *__restrict__ X, int64_t ldx, int64_t rows, int64_t k,
                                                     int64_t kseg, unsigned long long *__restrict__ maxbits,
                                                     int64_t xstride) {
  const int64_t j = static_cast<int64_t>(blockIdx.x) * 256 + threadIdx.x;
  if (j >= rows) return;
  X += static_cast<int64_t>(blockIdx.z) * xstride * W;  // batch entry (strided batched calls)
  maxbits += static_cast<int64_t>(blockIdx.z) * rows;
  const int64_t h0 = static_cast<int64_t>(blockIdx.y) * kseg;
  const int64_t h1 = (h0 + kseg < k) ? h0 + kseg : k;
  unsigned long long mx = 0;
#pragma unroll 4
  for (int64_t h = h0; h < h1; ++h) {
#pragma unroll
    for (int c = 0; c < W; ++c) {
      const unsigned long long b = abs_bits(X[(h * ldx + j) * W + c]);
      mx = b > mx ? b : mx;
    }
  }
  if (mx) atomicMax(&maxbits[j], mx);
}

// Non-finite inputs ("result unspecified, no fault"; the pre-pass raises a device-side flag): the row /
// column maximum of the |x| bit patterns has an all-ones exponent field exactly when the row / column holds an Inf or NaN.
template <typename T>
__device__ __forceinline__ void flag_nonfinite(unsigned long long maxbits, unsigned long long *flag) {
  const unsigned long long inf = sizeof(T) == 8 ? 0x7FF0000000000000ull : 0x7F800000ull;
  if (flag && maxbits >= inf) atomicOr(flag, 1ull);
}

// frexp exponent of the magnitude whose bit pattern is b (the row / column maximum); zero row -> 0 (R2)
template <typename T>
__device__ __forceinline__ int exponent_of_maxbits(unsigned long long b) {
  unsigned long long M;
  int ex2;
  bool neg;
  if (sizeof(T) == 8) decode_bits(__longlong_as_double(static_cast<long long>(b)), M, ex2, neg);
  else decode_bits(__uint_as_float(static_cast<unsigned int>(b)), M, ex2, neg);
  return M ? ex2 + (64 - __clzll(static_cast<long long>(M))) : 0;
}

template <typename T>
__global__ void bits_to_exponent_kernel(const unsigned long long *__restrict__ maxbits, int64_t rows,
                                        int32_t *__restrict__ e_out) {
  const int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (i < rows) e_out[i] = exponent_of_maxbits<T>(maxbits[i]);
}

// Column maxima of X (k x rows, ldx) as |x| bit patterns -> maxbits[rows] (zeroed here); the column kernels turn them
// into exponents.
int launch_colmax(emugemm_ctx *ctx, int elem, int64_t rows, int64_t k, const void *X, int64_t ldx,
                  unsigned long long *maxbits, int batch, int64_t xstride) {
  if (rows == 0 || batch == 0) return EMUGEMM_OK;
  cudaStream_t st = ctx->stream;
  EMU_CUDA(ctx, cudaMemsetAsync(maxbits, 0, sizeof(unsigned long long) * rows * batch, st));
  if (k == 0) return EMUGEMM_OK;
  // enough k-segments to fill the machine: ~8 CTAs per SM
  const int64_t gx = (rows + 255) / 256;
  int64_t segs = (static_cast<int64_t>(ctx->num_sms) * 8 + gx * batch - 1) / (gx * batch);
  if (segs > (k + 63) / 64) segs = (k + 63) / 64;
  if (segs < 1) segs = 1;
  const int64_t kseg = (k + segs - 1) / segs;
  const dim3 grid(static_cast<unsigned>(gx), static_cast<unsigned>((k + kseg - 1) / kseg), static_cast<unsigned>(batch));
  if (elem == kF64) colmax_kernel<double, 1><<<grid, 256, 0, st>>>(static_cast<const double *>(X), ldx, rows, k, kseg, maxbits, xstride);
  else if (elem == kF32) colmax_kernel<float, 1><<<grid, 256, 0, st>>>(static_cast<const float *>(X), ldx, rows, k, kseg, maxbits, xstride);
  else if (elem == kC64) colmax_kernel<float, 2><<<grid, 256, 0, st>>>(static_cast<const float *>(X), ldx, rows, k, kseg, maxbits, xstride);
  else colmax_kernel<double, 2><<<grid, 256, 0, st>>>(static_cast<const double *>(X), ldx, rows, k, kseg, maxbits, xstride);
  ctx->launches++;
  EMU_CUDA(ctx, cudaGetLastError());
  return EMUGEMM_OK;
}

// Exponents alone (test hook emugemm_dbg_exponents): row scan or column scan + bit pattern -> exponent.
int launch_exponent_scan(emugemm_ctx *ctx, int elem, int by_cols, int64_t rows, int64_t k, const void *X,
                         int64_t ldx, unsigned long long *maxbits, int32_t *e_out) {
  if (rows == 0) return EMUGEMM_OK;
  cudaStream_t st = ctx->stream;
  if (by_cols) {
    EMU_TRY(launch_colmax(ctx, elem, rows, k, X, ldx, maxbits));
  } else {
    EMU_CUDA(ctx, cudaMemsetAsync(maxbits, 0, sizeof(unsigned long long) * rows, st));
    if (k > 0) {
      const unsigned grid = static_cast<unsigned>(rows);
      if (elem == kF64) rowmax_kernel<double, 1><<<grid, 256, 0, st>>>(static_cast<const double *>(X), ldx, k, maxbits);
      else if (elem == kF32) rowmax_kernel<float, 1><<<grid, 256, 0, st>>>(static_cast<const float *>(X), ldx, k, maxbits);
      else rowmax_kernel<double, 2><<<grid, 256, 0, st>>>(static_cast<const double *>(X), ldx, k, maxbits);
      ctx->launches++;
    }
  }
  const unsigned g2 = static_cast<unsigned>((rows + 255) / 256);
  if (elem == kF32) bits_to_exponent_kernel<float><<<g2, 256, 0, st>>>(maxbits, rows, e_out);
  else bits_to_exponent_kernel<double><<<g2, 256, 0, st>>>(maxbits, rows, e_out);
  ctx->launches++;
  EMU_CUDA(ctx, cudaGetLastError());
  return EMUGEMM_OK;
}

// ----------------------------------------------------------------------------
// digitizers.  MODE 0: Scheme I digits (PARAM = p, compile-time so that every digit is one funnel shift + mask),
// MODE 1: Scheme II residues (PARAM = words of |a'|: 2 when t <= 64, else 3).
// ----------------------------------------------------------------------------
// |v| = (M / 2^63) 2^ex with the leading mantissa bit of a normal number at bit 63 (subnormals: no hidden bit)
__device__ __forceinline__ void decode_top(double v, unsigned long long &M, int &ex, bool &neg) {
  const unsigned long long b = static_cast<unsigned long long>(__double_as_longlong(v));
  neg = (b >> 63) != 0;
  const int E = static_cast<int>((b >> 52) & 0x7FF);
  M = ((b & 0xFFFFFFFFFFFFFull) | (E ? (1ull << 52) : 0ull)) << 11;
  ex = (E ? E : 1) - 1023;
}
__device__ __forceinline__ void decode_top(float v, unsigned long long &M, int &ex, bool &neg) {
  const unsigned int b = __float_as_uint(v);
  neg = (b >> 31) != 0;
  const int E = static_cast<int>((b >> 23) & 0xFF);
  M = static_cast<unsigned long long>((b & 0x7FFFFFu) | (E ? (1u << 23) : 0u)) << 40;
  ex = (E ? E : 1) - 127;
}

struct Prep {            // one scalar prepared for plane extraction
  unsigned int w0, w1, w2;  // magnitude: OZ1 X (<= 56 bits) in w0,w1; OZ2 |a'| (<= 70 bits) in w0..w2
  bool neg;
};

// trunc(|v| 2^(scale_bits - e_row)) (R3: toward zero).  |v| < 2^e_row, so the right shift rs >= 64 - scale_bits.
template <typename T, int NW>
__device__ __forceinline__ Prep prepare(T v, int e_row, int scale_bits) {
  unsigned long long M;
  int ex;
  Prep r;
  decode_top(v, M, ex, r.neg);
  const int rs = 63 - ex - scale_bits + e_row;
  if (NW == 2) {  // scale_bits <= 64: rs >= 0, result < 2^64
    const unsigned long long X = (rs >= 64) ? 0ull : (M >> rs);
    r.w0 = static_cast<unsigned int>(X);
    r.w1 = static_cast<unsigned int>(X >> 32);
    r.w2 = 0u;
  } else {        // scale_bits <= 95: 96-bit value (M : 0) >> (rs + 32), rs + 32 >= 96 - scale_bits > 0
    const int W = rs + 32;
    const unsigned int mh = static_cast<unsigned int>(M >> 32), ml = static_cast<unsigned int>(M);
    const int q = W >> 5, b = W & 31;
    const unsigned int hi = (q == 0) ? mh : 0u;
    const unsigned int mid = (q == 0) ? ml : (q == 1) ? mh : 0u;
    const unsigned int lo = (q == 0) ? 0u : (q == 1) ? ml : (q == 2) ? mh : 0u;
    r.w0 = __funnelshift_r(lo, mid, b);
    r.w1 = __funnelshift_r(mid, hi, b);
    r.w2 = hi >> b;
  }
  return r;
}

// moduli: greedy pairwise-coprime list descending from 256 (R10)
__device__ __constant__ int c_moduli[24] = {256, 255, 253, 251, 247, 241, 239, 233, 229, 227, 223, 217,
                                            211, 199, 197, 193, 191, 181, 179, 173, 167, 163, 157, 151};
constexpr int h_moduli[24] = {256, 255, 253, 251, 247, 241, 239, 233, 229, 227, 223, 217,
                              211, 199, 197, 193, 191, 181, 179, 173, 167, 163, 157, 151};

__host__ __device__ constexpr unsigned int pow256_mod(int j, int m) {
  unsigned int r = 1u % static_cast<unsigned int>(m);
  for (int i = 0; i < j; ++i) r = (r * 256u) % static_cast<unsigned int>(m);
  return r;
}
__host__ __device__ constexpr unsigned int pack_w(int word, int m) {  // bytes 256^(4 word + b) mod m
  return pow256_mod(4 * word, m) | (pow256_mod(4 * word + 1, m) << 8) | (pow256_mod(4 * word + 2, m) << 16) |
         (pow256_mod(4 * word + 3, m) << 24);
}
__host__ __device__ constexpr unsigned int magic32(int m) {  // ceil(2^32 / m)
  return static_cast<unsigned int>(((1ull << 32) + static_cast<unsigned long long>(m) - 1ull) /
                                   static_cast<unsigned long long>(m));
}

// ----------------------------------------------------------------------------
// plane emission.  Each thread owns 4 consecutive k of one row/column ("quad")
// and emits one packed 32-bit word per plane through `sink(plane, word)`.
// ----------------------------------------------------------------------------
// Balanced base-256 digits (R23): X = +-|X| (|X| < 2^(8P-2)), Y = X + sum_j 128 256^j; digit t = byte (P-1-t) of Y
// minus 128 = that byte XOR 0x80 as int8.  One 64-bit add per element, then byte permutes only.
template <int P, typename Sink>
__device__ __forceinline__ void emit_oz1_b8(const Prep (&q)[4], Sink sink) {
  constexpr unsigned long long kC = (P == 8) ? 0x8080808080808080ull : ((0x8080808080808080ull) & ((1ull << (8 * (P & 7))) - 1ull));
  unsigned int lo[4], hi[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const long long mag = static_cast<long long>((static_cast<unsigned long long>(q[i].w1) << 32) | q[i].w0);
    const unsigned long long Y = (static_cast<unsigned long long>(q[i].neg ? -mag : mag) + kC) ^ kC;  // bytes = int8 digits
    lo[i] = static_cast<unsigned int>(Y);
    hi[i] = static_cast<unsigned int>(Y >> 32);
  }
#pragma unroll
  for (int t = 0; t < P; ++t) {
    const int byte = P - 1 - t;  // byte index inside Y
    // selector: result byte 0 = byte (byte & 3) of the first operand, result byte 1 = the same byte of the second
    const unsigned int sel = static_cast<unsigned int>(byte & 3) | (static_cast<unsigned int>(4 + (byte & 3)) << 4);
    const unsigned int w = (byte < 4)
        ? __byte_perm(__byte_perm(lo[0], lo[1], sel), __byte_perm(lo[2], lo[3], sel), 0x5410)
        : __byte_perm(__byte_perm(hi[0], hi[1], sel), __byte_perm(hi[2], hi[3], sel), 0x5410);
    sink(t, w);
  }
}

// Two's-complement 7-bit digits (R24; PAPER.md:345 at beta = 7): X = +-|X| (|X| < 2^(7P)) as a 64-bit two's-complement integer;
// digit 0 = the low BYTE of X >> 7 (P - 1) (in [-128, 127]), digit t >= 1 = the 7-bit field (X >> 7 (P - 1 - t)) & 127 in [0, 127]:
// per plane one funnel shift per element, three byte permutes, one AND; no sign fix-up.  Every slice but the leading one is
// sign-free, which is what the tensor pipe's power likes (profiles/r2_operand_sign_power.md).
template <int P, typename Sink>
__device__ __forceinline__ void emit_oz1_tc(const Prep (&q)[4], Sink sink) {
  unsigned int lo[4], hi[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const long long mag = static_cast<long long>((static_cast<unsigned long long>(q[i].w1) << 32) | q[i].w0);
    const unsigned long long Y = static_cast<unsigned long long>(q[i].neg ? -mag : mag);
    lo[i] = static_cast<unsigned int>(Y);
    hi[i] = static_cast<unsigned int>(Y >> 32);
  }
#pragma unroll
  for (int t = 0; t < P; ++t) {
    const int sh = kBeta * (P - 1 - t);  // compile-time after unrolling
    unsigned int b[4];
#pragma unroll
    for (int i = 0; i < 4; ++i)  // low byte of the arithmetic shift: for sh >= 32 the bits above come from hi's sign extension
      b[i] = (sh == 0) ? lo[i] : (sh < 32) ? __funnelshift_r(lo[i], hi[i], sh) : (sh == 32) ? hi[i]
                                           : static_cast<unsigned int>(static_cast<int>(hi[i]) >> (sh - 32));
    const unsigned int w = __byte_perm(__byte_perm(b[0], b[1], 0x0040), __byte_perm(b[2], b[3], 0x0040), 0x5410);
    sink(t, t == 0 ? w : (w & 0x7F7F7F7Fu));
  }
}

// Sign-magnitude 7-bit digits (R1) of four elements, one packed word per plane.  Per plane: one funnel shift per
// element brings digit t to byte 0, three byte permutes gather the four bytes, one AND keeps 7 bits, and the signs
// are applied to the whole word at once: for a byte d in [0, 127] of a negative element
// ((d ^ 0x7F) + 1) ^ 0x80 = (128 - d) ^ 0x80 = -d (mod 256) without a carry into the next byte ((d ^ 0x7F) + 1 <= 128).
// 11 integer instructions per word instead of 19 (shift + mask + negate + select per digit, then the pack).
template <int P, typename Sink>
__device__ __forceinline__ void emit_oz1(const Prep (&q)[4], Sink sink) {
  const unsigned int m1 = (q[0].neg ? 0x1u : 0u) | (q[1].neg ? 0x100u : 0u) | (q[2].neg ? 0x10000u : 0u) | (q[3].neg ? 0x1000000u : 0u);
  const unsigned int m7 = m1 * 0x7Fu, m8 = m1 << 7;
#pragma unroll
  for (int t = 0; t < P; ++t) {
    const int sh = kBeta * (P - 1 - t);  // compile-time after unrolling
    unsigned int b[4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
      b[i] = (sh == 0) ? q[i].w0 : (sh < 32) ? __funnelshift_r(q[i].w0, q[i].w1, sh) : (sh == 32) ? q[i].w1 : (q[i].w1 >> (sh - 32));
    const unsigned int w = __byte_perm(__byte_perm(b[0], b[1], 0x0040), __byte_perm(b[2], b[3], 0x0040), 0x5410) & 0x7F7F7F7Fu;
    sink(t, ((w ^ m7) + m1) ^ m8);
  }
}

// Scheme II residues of real operands (Eq. 5; R11 / R13).  The element is first turned into its
// two's complement over NW words (U = a' + neg 2^(32 NW), neg only for a nonzero negative a'), then per modulus
//   t = sum_j byte_j(U) (256^j mod m) + hm + neg ((-2^(32 NW)) mod m)  ==  a' + hm (mod m),   t < 2^20,
//   u = t - floor(t / m) m in [0, m): q = floor(t / m) by ONE multiply-high with ceil(2^32 / m) (exact:
//       t (M m - 2^32) / (m 2^32) < 2^-12 < 1/m), hm = (m - 1) / 2,
// so u - hm in [-hm, hm] is the symmetric residue of the SIGNED value.  The four u of a quad are packed and hm is
// subtracted from all four bytes at once: (u + (128 - hm)) ^ 0x80 is u - hm as int8 (u + 128 - hm lies in [1, 255]:
// no carry).  m = 256: the low byte of U.  6.25 integer instructions per residue (first version: sign-magnitude
// residue, negate / select and -hm per element: 7.75).
struct PrepS {
  unsigned int w0, w1, w2;
  unsigned int neg;  // all ones for a nonzero negative value, else 0
};
template <int NW>
__device__ __forceinline__ PrepS twos_complement(const Prep &q) {
  PrepS r;
  const bool nz = (q.w0 | q.w1 | (NW == 3 ? q.w2 : 0u)) != 0u;
  r.neg = (q.neg && nz) ? 0xFFFFFFFFu : 0u;
  if (NW == 2) {
    const unsigned long long X = (static_cast<unsigned long long>(q.w1) << 32) | q.w0;
    const unsigned long long U = r.neg ? 0ull - X : X;
    r.w0 = static_cast<unsigned int>(U);
    r.w1 = static_cast<unsigned int>(U >> 32);
    r.w2 = 0u;
  } else {
    // 96-bit negate: ~x + 1
    const unsigned int n0 = ~q.w0 + 1u;
    const unsigned int c0 = (q.w0 == 0u) ? 1u : 0u;
    const unsigned int n1 = ~q.w1 + c0;
    const unsigned int c1 = (c0 && q.w1 == 0u) ? 1u : 0u;
    const unsigned int n2 = ~q.w2 + c1;
    r.w0 = r.neg ? n0 : q.w0;
    r.w1 = r.neg ? n1 : q.w1;
    r.w2 = r.neg ? n2 : q.w2;
  }
  return r;
}
__host__ __device__ constexpr unsigned int neg_pow_mod(int nw, int m) {  // (-2^(32 nw)) mod m
  const unsigned int r = pow256_mod(4 * nw, m);
  return r == 0u ? 0u : static_cast<unsigned int>(m) - r;
}
template <int L, int NW, typename Sink>
__device__ __forceinline__ void emit_oz2_real_lean(const PrepS (&q)[4], int N, Sink sink) {
  if constexpr (L < kMaxModuli) {
    if (L < N) {
      constexpr int m = h_moduli[L];
      if constexpr (m == 256) {
        sink(L, __byte_perm(__byte_perm(q[0].w0, q[1].w0, 0x0040), __byte_perm(q[2].w0, q[3].w0, 0x0040), 0x5410));
      } else {
        constexpr unsigned int c0 = pack_w(0, m), c1 = pack_w(1, m), c2 = pack_w(2, m), mg = magic32(m);
        constexpr unsigned int hm = (m - 1) / 2, kneg = neg_pow_mod(NW, m);
        unsigned int u[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          unsigned int t = __dp4a(q[i].w0, c0, (q[i].neg & kneg) + hm);
          t = __dp4a(q[i].w1, c1, t);
          if (NW == 3) t = __dp4a(q[i].w2, c2, t);
          u[i] = t - __umulhi(t, mg) * static_cast<unsigned int>(m);
        }
        const unsigned int w = __byte_perm(__byte_perm(u[0], u[1], 0x0040), __byte_perm(u[2], u[3], 0x0040), 0x5410);
        sink(L, (w + (128u - hm) * 0x01010101u) ^ 0x80808080u);
      }
      emit_oz2_real_lean<L + 1, NW>(q, N, sink);
    }
  }
}
// Complex operands (3M): residues of re, im and the Sigma plane sym(r_re + r_im) (R15), four elements
// per word.  The moduli are walked by a run-time loop over a constant-memory table (the compile-time recursion of
// the first version kept the addresses and constants of all 3N planes live: 252 registers, 12.5 % occupancy).  With
// u_re == re + hm, u_im == im + hm (as in emit_oz2_real_lean; hm = floor(m / 2), so m = 256 runs through the same
// code), t = u_re + u_im + (m - hm) == re + im + hm (mod m) and one more multiply-high reduction gives the Sigma
// residue: no compares.
struct ModC {
  unsigned int c0, c1, c2, mg, negm, hm, kneg2, kneg3;  // negm = -m (mod 2^32)
};
#define EMU_MODC(L)                                                                                              \
  {pack_w(0, h_moduli[L]), pack_w(1, h_moduli[L]), pack_w(2, h_moduli[L]), magic32(h_moduli[L]),                  \
   0u - static_cast<unsigned int>(h_moduli[L]), static_cast<unsigned int>(h_moduli[L] / 2), neg_pow_mod(2, h_moduli[L]), \
   neg_pow_mod(3, h_moduli[L])}
__device__ __constant__ ModC c_modc[24] = {EMU_MODC(0),  EMU_MODC(1),  EMU_MODC(2),  EMU_MODC(3),  EMU_MODC(4),  EMU_MODC(5),
                                           EMU_MODC(6),  EMU_MODC(7),  EMU_MODC(8),  EMU_MODC(9),  EMU_MODC(10), EMU_MODC(11),
                                           EMU_MODC(12), EMU_MODC(13), EMU_MODC(14), EMU_MODC(15), EMU_MODC(16), EMU_MODC(17),
                                           EMU_MODC(18), EMU_MODC(19), EMU_MODC(20), EMU_MODC(21), EMU_MODC(22), EMU_MODC(23)};
#undef EMU_MODC

// The integer multiplier ("fmaheavy": IDP.4A, IMAD, IMAD.HI) is the pipe these kernels saturate (ncu: 85 %), so the
// reduction spends exactly NW + 2 instructions there: the start constant is added by ONE three-input add on the ALU
// pipe (a two-input add tends to be emitted as IMAD.IADD) and t - q m is one multiply-add with -m.
template <int NW>
__device__ __forceinline__ unsigned int oz2_u(const PrepS &q, const ModC &mc) {  // (value + hm) mod m in [0, m)
  unsigned int t = __dp4a(q.w0, mc.c0, 0u);
  t = __dp4a(q.w1, mc.c1, t);
  if (NW == 3) t = __dp4a(q.w2, mc.c2, t);
  t = t + mc.hm + (q.neg & (NW == 2 ? mc.kneg2 : mc.kneg3));
  return __umulhi(t, mc.mg) * mc.negm + t;
}
__device__ __forceinline__ unsigned int pack4u(const unsigned int (&u)[4]) {
  return __byte_perm(__byte_perm(u[0], u[1], 0x0040), __byte_perm(u[2], u[3], 0x0040), 0x5410);
}
template <int NW, typename Sink>
__device__ __forceinline__ void emit_oz2_cplx_lean(const PrepS (&re)[4], const PrepS (&im)[4], int N, Sink sink) {
#pragma unroll 1
  for (int L = 0; L < N; ++L) {
    const ModC mc = c_modc[L];
    const unsigned int mhm = 0u - mc.negm - mc.hm;  // m - hm
    unsigned int ua[4], ub[4], us[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      ua[i] = oz2_u<NW>(re[i], mc);
      ub[i] = oz2_u<NW>(im[i], mc);
      const unsigned int t = ua[i] + ub[i] + mhm;
      us[i] = __umulhi(t, mc.mg) * mc.negm + t;
    }
    const unsigned int bias = (128u - mc.hm) * 0x01010101u;  // (u + 128 - hm) ^ 0x80 = u - hm as int8, all four bytes at once
    sink(L, (pack4u(ua) + bias) ^ 0x80808080u);
    sink(N + L, (pack4u(ub) + bias) ^ 0x80808080u);
    sink(2 * N + L, (pack4u(us) + bias) ^ 0x80808080u);
  }
}

// MODE 0: OZ1 (PARAM = p, scale_bits = 7p); MODE 1: OZ2 (PARAM = words, param = N, scale_bits = t)
template <typename T, int W, int MODE, int PARAM, typename Sink>
__device__ __forceinline__ void emit_quad(const T (&v)[4][W], int e_row, int param, int scale_bits, Sink sink) {
  constexpr int NW = (MODE == 0) ? 2 : PARAM;
  Prep a[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) a[i] = prepare<T, NW>(v[i][0], e_row, scale_bits);
  if constexpr (MODE == 0) {
    if constexpr (PARAM >= 32) emit_oz1_tc<PARAM - 32>(a, sink);       // PARAM = 32 + p: two's-complement 7-bit digits (R24)
    else if constexpr (PARAM >= 16) emit_oz1_b8<PARAM - 16>(a, sink);  // PARAM = 16 + p: balanced 8-bit digits
    else emit_oz1<PARAM>(a, sink);
  } else if constexpr (W == 1) {
    PrepS u[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) u[i] = twos_complement<NW>(a[i]);
    emit_oz2_real_lean<0, NW>(u, param, sink);
  } else {
    PrepS re[4], im[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      re[i] = twos_complement<NW>(a[i]);
      im[i] = twos_complement<NW>(prepare<T, NW>(v[i][W - 1], e_row, scale_bits));
    }
    emit_oz2_cplx_lean<NW>(re, im, param, sink);
  }
}

// ---- rows: X is rows x k (ldx); out[plane][row][kpad] --------------------------
// One CTA per row, two phases: (1) max |x| bit pattern of the row -> exponent (written to e_out), (2) the row is
// read again -- it was just fetched by this CTA, so it comes from L1 / L2 -- and every thread digitises quads of 4
// consecutive k.  One DRAM read of A, no separate scan / exponent launches.
template <typename T, int W, int MODE, int PARAM>
__global__ void __launch_bounds__(256) planes_rows_kernel(const T *__restrict__ X, int64_t ldx, int64_t rows,
                                                          int64_t k, int64_t kpad, int32_t *__restrict__ e_out,
                                                          int param, int scale_bits, int8_t *__restrict__ out,
                                                          int64_t xstride, int64_t plane_rows, unsigned long long *nf_flag) {
  // batch entry b = blockIdx.y (strided batched calls: entry b of X starts xstride elements further; its planes are
  // rows [b rows, (b + 1) rows) of planes that hold plane_rows rows)
  const int64_t row = static_cast<int64_t>(blockIdx.y) * rows + blockIdx.x;
  const T *src = X + (static_cast<int64_t>(blockIdx.y) * xstride + static_cast<int64_t>(blockIdx.x) * ldx) * W;
  unsigned long long mx = 0;
  for (int64_t h = static_cast<int64_t>(threadIdx.x) * 4; h < k; h += 1024) {
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int c = 0; c < W; ++c)
        if (h + i < k) {
          const unsigned long long b = abs_bits(src[(h + i) * W + c]);
          mx = b > mx ? b : mx;
        }
  }
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned long long y = __shfl_xor_sync(0xffffffffu, mx, o);
    mx = y > mx ? y : mx;
  }
  __shared__ unsigned long long red[8];
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = mx;
  __syncthreads();
#pragma unroll
  for (int w = 0; w < 8; ++w) mx = red[w] > mx ? red[w] : mx;
  const int e_row = exponent_of_maxbits<T>(mx);
  if (threadIdx.x == 0) { e_out[row] = e_row; flag_nonfinite<T>(mx, nf_flag); }

  const int64_t plane_stride = plane_rows * kpad;
  for (int64_t h0 = static_cast<int64_t>(threadIdx.x) * 4; h0 < kpad; h0 += 1024) {
    T v[4][W];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int c = 0; c < W; ++c) v[i][c] = (h0 + i < k) ? src[(h0 + i) * W + c] : T(0);
    int8_t *dst = out + row * kpad + h0;
    emit_quad<T, W, MODE, PARAM>(v, e_row, param, scale_bits, [&](int plane, unsigned int word) {
      *reinterpret_cast<unsigned int *>(dst + plane * plane_stride) = word;
    });
  }
}


// 4 * W consecutive scalars from a 32-byte (double) / 16-byte (float) aligned address: 256-bit / 128-bit loads
template <int W>
__device__ __forceinline__ void load_quad_vec(const double *p, double (&v)[4][W]) {
  double f[4 * W];
#pragma unroll
  for (int i = 0; i < W; ++i)
    asm("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(f[4 * i]), "=d"(f[4 * i + 1]), "=d"(f[4 * i + 2]), "=d"(f[4 * i + 3]) : "l"(p + 4 * i));
#pragma unroll
  for (int i = 0; i < 4 * W; ++i) v[i / W][i % W] = f[i];
}
template <int W>
__device__ __forceinline__ void load_quad_vec(const float *p, float (&v)[4][W]) {
#pragma unroll
  for (int i = 0; i < W; ++i) {
    const float4 t = __ldg(reinterpret_cast<const float4 *>(p) + i);
    const float f[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
    for (int j = 0; j < 4; ++j) v[(4 * i + j) / W][(4 * i + j) % W] = f[j];
  }
}

// ---- rows, register-resident (kpad * W <= 32 NT): ONE read of X -------------------
// One CTA per row; every thread loads its 8 / W quads (32 scalars) once with vector loads, the row maximum is
// reduced from the registers, and the digits / residues are computed from the same registers: X is requested from
// memory exactly once (the two-phase kernel above re-reads the row, which misses L2 at 8192^2: 1.0 GB of DRAM reads
// for a 0.5 GB operand, profiles/).  Longer rows keep the two-phase kernel.
template <typename T, int W, int MODE, int PARAM, int NT>
__global__ void __launch_bounds__(NT) planes_rows_reg_kernel(const T *__restrict__ X, int64_t ldx, int64_t rows,
                                                              int64_t k, int64_t kpad, int32_t *__restrict__ e_out,
                                                              int param, int scale_bits, int8_t *__restrict__ out,
                                                              int64_t xstride, int64_t plane_rows, unsigned long long *nf_flag) {
  constexpr int R = 8 / W;
  const int64_t row = static_cast<int64_t>(blockIdx.y) * rows + blockIdx.x;
  const T *src = X + (static_cast<int64_t>(blockIdx.y) * xstride + static_cast<int64_t>(blockIdx.x) * ldx) * W;
  const bool vec = (reinterpret_cast<uintptr_t>(src) & (sizeof(T) == 8 ? 31 : 15)) == 0;
  const int kk = static_cast<int>(k);
  T v[R][4][W];
  unsigned long long mx = 0;
#pragma unroll
  for (int q = 0; q < R; ++q) {
    const int h0 = (static_cast<int>(threadIdx.x) + q * NT) * 4;
    if (vec && h0 + 4 <= kk) {
      load_quad_vec<W>(src + static_cast<int64_t>(h0) * W, v[q]);
    } else {
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int c = 0; c < W; ++c) v[q][i][c] = (h0 + i < kk) ? src[static_cast<int64_t>(h0 + i) * W + c] : T(0);
    }
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int c = 0; c < W; ++c) {
        const unsigned long long b = abs_bits(v[q][i][c]);
        mx = b > mx ? b : mx;
      }
  }
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned long long y = __shfl_xor_sync(0xffffffffu, mx, o);
    mx = y > mx ? y : mx;
  }
  __shared__ unsigned long long red[NT / 32];
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = mx;
  __syncthreads();
#pragma unroll
  for (int w = 0; w < NT / 32; ++w) mx = red[w] > mx ? red[w] : mx;
  const int e_row = exponent_of_maxbits<T>(mx);
  if (threadIdx.x == 0) { e_out[row] = e_row; flag_nonfinite<T>(mx, nf_flag); }

  const int64_t plane_stride = plane_rows * kpad;
#pragma unroll
  for (int q = 0; q < R; ++q) {
    const int h0 = (static_cast<int>(threadIdx.x) + q * NT) * 4;
    if (h0 < kpad) {
      int8_t *dst = out + row * kpad + h0;
      emit_quad<T, W, MODE, PARAM>(v[q], e_row, param, scale_bits, [&](int plane, unsigned int word) {
        *reinterpret_cast<unsigned int *>(dst + plane * plane_stride) = word;
      });
    }
  }
}

// ---- columns: X is k x rows (ldx); transposed through shared memory ----------
// tile = 32 columns x TH k; thread (lane = column, warp = k-quad index).
template <typename T, int W, int MODE, int PARAM, int TH>
__global__ void __launch_bounds__(256) planes_cols_kernel(const T *__restrict__ X, int64_t ldx, int64_t rows,
                                                          int64_t k, int64_t kpad,
                                                          const unsigned long long *__restrict__ maxbits,
                                                          int32_t *__restrict__ e_out, int param, int scale_bits, int nplanes,
                                                          int8_t *__restrict__ out, int64_t xstride, int64_t plane_rows,
                                                          unsigned long long *nf_flag) {
  extern __shared__ unsigned int tile[];  // [plane][32][TH/4 + 1]
  // batch entry blockIdx.z (see planes_rows_kernel)
  X += static_cast<int64_t>(blockIdx.z) * xstride * W;
  maxbits += static_cast<int64_t>(blockIdx.z) * rows;
  e_out += static_cast<int64_t>(blockIdx.z) * rows;
  out += static_cast<int64_t>(blockIdx.z) * rows * kpad;
  constexpr int PW = TH / 4 + 1;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int64_t j = static_cast<int64_t>(blockIdx.x) * 32 + lane;
  const int64_t hb = static_cast<int64_t>(blockIdx.y) * TH;
  // column exponent from the column-max bit pattern (colmax_kernel ran before); the first k-block publishes it
  const int e_row = (j < rows) ? exponent_of_maxbits<T>(maxbits[j]) : 0;
  if (blockIdx.y == 0 && warp == 0 && j < rows) { e_out[j] = e_row; flag_nonfinite<T>(maxbits[j], nf_flag); }
  for (int hw = warp; hw < TH / 4; hw += 8) {
    const int64_t h0 = hb + hw * 4;
    T v[4][W];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int c = 0; c < W; ++c) v[i][c] = (j < rows && h0 + i < k) ? X[((h0 + i) * ldx + j) * W + c] : T(0);
    emit_quad<T, W, MODE, PARAM>(v, e_row, param, scale_bits, [&](int plane, unsigned int word) {
      tile[(plane * 32 + lane) * PW + hw] = word;
    });
  }
  __syncthreads();
  // write-out: rows of TH bytes, (TH/4) lanes per row
  constexpr int LPR = TH / 4;          // lanes per row
  constexpr int RPW = 32 / LPR;        // rows per warp pass
  const int nrows = nplanes * 32;
  for (int r = warp * RPW + lane / LPR; r < nrows; r += 8 * RPW) {
    const int plane = r >> 5, jj = r & 31;
    const int64_t jg = static_cast<int64_t>(blockIdx.x) * 32 + jj;
    if (jg < rows) {
      const int wd = lane % LPR;
      *reinterpret_cast<unsigned int *>(out + (static_cast<int64_t>(plane) * plane_rows + jg) * kpad + hb + wd * 4) =
          tile[(plane * 32 + jj) * PW + wd];
    }
  }
}


// by_cols = 0: fused scan + planes of the rows of X, exponents written to e.
// by_cols = 1: column maxima (launch_colmax into the scratch maxbits[rows]) + planes of the columns of X, exponents written to e.
template <typename T, int W, int MODE, int PARAM>
static int launch_planes(emugemm_ctx *ctx, int elem, int by_cols, int64_t rows, int64_t k, int64_t kpad, const void *X,
                         int64_t ldx, unsigned long long *maxbits, int32_t *e, int param, int scale_bits, int nplanes,
                         int8_t *out, int batch = 1, int64_t xstride = 0) {
  if (rows == 0 || kpad == 0 || batch == 0) return EMUGEMM_OK;
  if (batch > 65535) return EMUGEMM_ERR_ARG;  // grid.y / grid.z
  const int64_t plane_rows = rows * batch;
  cudaStream_t st = ctx->stream;
  const T *x = static_cast<const T *>(X);
  if (!by_cols) {
    const dim3 grid(static_cast<unsigned>(rows), static_cast<unsigned>(batch));
    const bool two_phase = EMU_PROBE_FLAG(ctx->dbg_flags, 32) != 0;  // dbg bit 5: the two-phase kernels (A/B timing)
    // Scheme I digits: the register-resident single-read kernel when the row fits (p = 2: 0.159 -> 0.111 ms, p = 8: 0.246 ->
    // 0.218 ms at 8192^2).  Scheme II residues are bound by the integer pipes, not by the second read: there the 80
    // registers of the resident row cost occupancy (N = 16: 0.431 -> 0.475 ms, 3M N = 18: 1.81 -> 2.89 ms), so they keep
    // the two-phase kernel.
    bool done = false;
    if constexpr (MODE == 0) {
      if (!two_phase && kpad * W <= 32 * 256) {
        planes_rows_reg_kernel<T, W, MODE, PARAM, 256><<<grid, 256, 0, st>>>(x, ldx, rows, k, kpad, e, param, scale_bits, out,
                                                                              xstride, plane_rows, ctx->nf_flag);
        done = true;
      } else if (!two_phase && kpad * W <= 32 * 512) {
        planes_rows_reg_kernel<T, W, MODE, PARAM, 512><<<grid, 512, 0, st>>>(x, ldx, rows, k, kpad, e, param, scale_bits, out,
                                                                              xstride, plane_rows, ctx->nf_flag);
        done = true;
      }
    }
    if (!done)
      planes_rows_kernel<T, W, MODE, PARAM><<<grid, 256, 0, st>>>(x, ldx, rows, k, kpad, e, param, scale_bits, out, xstride,
                                                                   plane_rows, ctx->nf_flag);
    ctx->launches++;
  } else {
    // The column maxima are a true dependency: a separate launch reads X once more.  A single-read variant (tile kept in
    // registers, per-panel arrival counters, tickets) measured SLOWER: the panel barrier re-synchronises the CTAs of
    // a wave, so the load phase and the digit phase no longer overlap (p = 2: 0.207 -> 0.215 ms, p = 8: 0.30 -> 0.34 ms,
    // N = 16: 0.64 -> 0.70 ms at 8192^2).
    EMU_TRY(launch_colmax(ctx, elem, rows, k, X, ldx, maxbits, batch, xstride));
    if (nplanes <= 20) {
      constexpr int TH = 128;
      const size_t smem = static_cast<size_t>(nplanes) * 32 * (TH / 4 + 1) * 4;
      auto kern = planes_cols_kernel<T, W, MODE, PARAM, TH>;
      EMU_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 20 * 32 * (TH / 4 + 1) * 4));
      const dim3 grid(static_cast<unsigned>((rows + 31) / 32), static_cast<unsigned>(kpad / TH), static_cast<unsigned>(batch));
      kern<<<grid, 256, smem, st>>>(x, ldx, rows, k, kpad, maxbits, e, param, scale_bits, nplanes, out, xstride, plane_rows, ctx->nf_flag);
    } else {
      constexpr int TH = 32;
      const size_t smem = static_cast<size_t>(nplanes) * 32 * (TH / 4 + 1) * 4;
      auto kern = planes_cols_kernel<T, W, MODE, PARAM, TH>;
      EMU_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 60 * 32 * (TH / 4 + 1) * 4));
      const dim3 grid(static_cast<unsigned>((rows + 31) / 32), static_cast<unsigned>(kpad / TH), static_cast<unsigned>(batch));
      kern<<<grid, 256, smem, st>>>(x, ldx, rows, k, kpad, maxbits, e, param, scale_bits, nplanes, out, xstride, plane_rows, ctx->nf_flag);
    }
    ctx->launches++;
  }
  EMU_CUDA(ctx, cudaGetLastError());
  return EMUGEMM_OK;
}

template <typename T, int P>
static int slice_p(emugemm_ctx *ctx, int by_cols, int64_t rows, int64_t k, int64_t kpad, const void *X, int64_t ldx,
                   unsigned long long *maxbits, int32_t *e, int slice_bits, int8_t *out, int batch, int64_t xstride) {
  if (slice_bits == kDigitsTwos)  // the same X as R1, two's-complement fields
    return launch_planes<T, 1, 0, 32 + P>(ctx, sizeof(T) == 8 ? kF64 : kF32, by_cols, rows, k, kpad, X, ldx, maxbits, e, P, kBeta * P, P, out, batch, xstride);
  if (slice_bits == 8)  // |X| = trunc(|x| 2^(8p - 2 - e)): two guard bits
    return launch_planes<T, 1, 0, 16 + P>(ctx, sizeof(T) == 8 ? kF64 : kF32, by_cols, rows, k, kpad, X, ldx, maxbits, e, P, 8 * P - 2, P, out, batch, xstride);
  return launch_planes<T, 1, 0, P>(ctx, sizeof(T) == 8 ? kF64 : kF32, by_cols, rows, k, kpad, X, ldx, maxbits, e, P, kBeta * P, P, out, batch, xstride);
}

int launch_oz1_slice(emugemm_ctx *ctx, int elem, int by_cols, int64_t rows, int64_t k, int64_t kpad,
                     const void *X, int64_t ldx, unsigned long long *maxbits, int32_t *e, int p, int slice_bits,
                     int8_t *out, int batch, int64_t xstride) {
#define EMU_SLICE_CASE(T, PP) case PP: return slice_p<T, PP>(ctx, by_cols, rows, k, kpad, X, ldx, maxbits, e, slice_bits, out, batch, xstride)
  if (elem == kF64) {
    switch (p) {
      EMU_SLICE_CASE(double, 1); EMU_SLICE_CASE(double, 2); EMU_SLICE_CASE(double, 3); EMU_SLICE_CASE(double, 4);
      EMU_SLICE_CASE(double, 5); EMU_SLICE_CASE(double, 6); EMU_SLICE_CASE(double, 7); EMU_SLICE_CASE(double, 8);
      default: return EMUGEMM_ERR_ARG;
    }
  }
  if (elem == kF32) {  // 24-bit inputs: more than 4 slices add nothing (API range), the test hook allows up to 8
    switch (p) {
      EMU_SLICE_CASE(float, 1); EMU_SLICE_CASE(float, 2); EMU_SLICE_CASE(float, 3); EMU_SLICE_CASE(float, 4);
      EMU_SLICE_CASE(float, 5); EMU_SLICE_CASE(float, 6); EMU_SLICE_CASE(float, 7); EMU_SLICE_CASE(float, 8);
      default: return EMUGEMM_ERR_ARG;
    }
  }
#undef EMU_SLICE_CASE
  return EMUGEMM_ERR_ARG;
}

int launch_oz2_residues(emugemm_ctx *ctx, int elem, int by_cols, int64_t rows, int64_t k, int64_t kpad,
                        const void *X, int64_t ldx, unsigned long long *maxbits, int32_t *e, int n_moduli, int t_bits,
                        int8_t *out, int batch, int64_t xstride) {
  if (t_bits < 1 || t_bits > 95) return EMUGEMM_ERR_ARG;  // three 32-bit words hold |a'| < 2^t (t = 77 at most: N = 20, k = 1)
  const bool two = t_bits <= 64;  // |a'| < 2^t fits two 32-bit words: one byte dot product less per residue
  if (elem == kF64)
    return two ? launch_planes<double, 1, 1, 2>(ctx, kF64, by_cols, rows, k, kpad, X, ldx, maxbits, e, n_moduli, t_bits, n_moduli, out, batch, xstride)
               : launch_planes<double, 1, 1, 3>(ctx, kF64, by_cols, rows, k, kpad, X, ldx, maxbits, e, n_moduli, t_bits, n_moduli, out, batch, xstride);
  if (elem == kF32)  // 24-bit inputs (Scheme II SGEMM)
    return two ? launch_planes<float, 1, 1, 2>(ctx, kF32, by_cols, rows, k, kpad, X, ldx, maxbits, e, n_moduli, t_bits, n_moduli, out, batch, xstride)
               : launch_planes<float, 1, 1, 3>(ctx, kF32, by_cols, rows, k, kpad, X, ldx, maxbits, e, n_moduli, t_bits, n_moduli, out, batch, xstride);
  if (elem == kC64)
    return two ? launch_planes<float, 2, 1, 2>(ctx, kC64, by_cols, rows, k, kpad, X, ldx, maxbits, e, n_moduli, t_bits, 3 * n_moduli, out, batch, xstride)
               : launch_planes<float, 2, 1, 3>(ctx, kC64, by_cols, rows, k, kpad, X, ldx, maxbits, e, n_moduli, t_bits, 3 * n_moduli, out, batch, xstride);
  if (elem == kZ128)
    return two ? launch_planes<double, 2, 1, 2>(ctx, kZ128, by_cols, rows, k, kpad, X, ldx, maxbits, e, n_moduli, t_bits, 3 * n_moduli, out, batch, xstride)
               : launch_planes<double, 2, 1, 3>(ctx, kZ128, by_cols, rows, k, kpad, X, ldx, maxbits, e, n_moduli, t_bits, 3 * n_moduli, out, batch, xstride);
  return EMUGEMM_ERR_ARG;
}

// ---- Scheme I complex (4M): digit planes of the REAL EMBEDDING ------------
//   A' = [[Re A, -Im A], [Im A, Re A]] (2m x 2k),  B' = [[Re B], [Im B]] (2k x n)
// written directly from the complex operands: every digit word of Re A / Im A is stored twice (rows i and m + i),
// the negated imaginary part is digitised from the sign-flipped value (exact in both digit formats).
// Embedded k index: [0, kpad) = first half, [kpad, 2 kpad) = second half (each half zero-padded to kpad).
template <int PARAM, typename Sink>
__device__ __forceinline__ void emit_oz1_any(const Prep (&q)[4], Sink sink) {
  if constexpr (PARAM >= 32) emit_oz1_tc<PARAM - 32>(q, sink);
  else if constexpr (PARAM >= 16) emit_oz1_b8<PARAM - 16>(q, sink);
  else emit_oz1<PARAM>(q, sink);
}

template <typename T, int PARAM>
__global__ void __launch_bounds__(256) oz1_4m_rows_kernel(const T *__restrict__ X, int64_t ldx, int64_t m, int64_t k,
                                                          int64_t kpad, int32_t *__restrict__ e_out, int scale_bits,
                                                          int8_t *__restrict__ out, unsigned long long *nf_flag) {
  const int64_t row = blockIdx.x;
  const T *src = X + row * ldx * 2;
  unsigned long long mx = 0;
  for (int64_t h = static_cast<int64_t>(threadIdx.x) * 4; h < 2 * k; h += 1024)
#pragma unroll
    for (int i = 0; i < 4; ++i)
      if (h + i < 2 * k) {
        const unsigned long long b = abs_bits(src[h + i]);
        mx = b > mx ? b : mx;
      }
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned long long y = __shfl_xor_sync(0xffffffffu, mx, o);
    mx = y > mx ? y : mx;
  }
  __shared__ unsigned long long red[8];
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = mx;
  __syncthreads();
#pragma unroll
  for (int w = 0; w < 8; ++w) mx = red[w] > mx ? red[w] : mx;
  const int e_row = exponent_of_maxbits<T>(mx);
  if (threadIdx.x == 0) { e_out[row] = e_row; e_out[m + row] = e_row; flag_nonfinite<T>(mx, nf_flag); }

  const int64_t kk = 2 * kpad, plane_stride = 2 * m * kk;
  for (int64_t h0 = static_cast<int64_t>(threadIdx.x) * 4; h0 < kpad; h0 += 1024) {
    Prep re[4], im[4], nim[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const bool in = h0 + i < k;
      re[i] = prepare<T, 2>(in ? src[(h0 + i) * 2] : T(0), e_row, scale_bits);
      im[i] = prepare<T, 2>(in ? src[(h0 + i) * 2 + 1] : T(0), e_row, scale_bits);
      nim[i] = im[i];
      nim[i].neg = !im[i].neg;
    }
    int8_t *top = out + row * kk + h0, *bot = out + (m + row) * kk + h0;
    emit_oz1_any<PARAM>(re, [&](int t, unsigned int w) {
      *reinterpret_cast<unsigned int *>(top + t * plane_stride) = w;
      *reinterpret_cast<unsigned int *>(bot + t * plane_stride + kpad) = w;
    });
    emit_oz1_any<PARAM>(im, [&](int t, unsigned int w) { *reinterpret_cast<unsigned int *>(bot + t * plane_stride) = w; });
    emit_oz1_any<PARAM>(nim, [&](int t, unsigned int w) { *reinterpret_cast<unsigned int *>(top + t * plane_stride + kpad) = w; });
  }
}

// B (k x n complex, ldx in complex elements): planes out[t][j][2 kpad] = [digits of Re B(:, j) | digits of Im B(:, j)];
// tile = 32 columns x 128 k, transposed through shared memory ("virtual plane" P + t = imaginary half).
template <typename T, int PARAM>
__global__ void __launch_bounds__(256) oz1_4m_cols_kernel(const T *__restrict__ X, int64_t ldx, int64_t n, int64_t k,
                                                          int64_t kpad, const unsigned long long *__restrict__ maxbits,
                                                          int32_t *__restrict__ e_out, int scale_bits, int P,
                                                          int8_t *__restrict__ out, unsigned long long *nf_flag) {
  extern __shared__ unsigned int tile[];  // [2 P][32][33]
  constexpr int TH = 128, PW = TH / 4 + 1;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int64_t j = static_cast<int64_t>(blockIdx.x) * 32 + lane;
  const int64_t hb = static_cast<int64_t>(blockIdx.y) * TH;
  const int e_row = (j < n) ? exponent_of_maxbits<T>(maxbits[j]) : 0;
  if (blockIdx.y == 0 && warp == 0 && j < n) { e_out[j] = e_row; flag_nonfinite<T>(maxbits[j], nf_flag); }
  for (int hw = warp; hw < TH / 4; hw += 8) {
    const int64_t h0 = hb + hw * 4;
    Prep re[4], im[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const bool in = j < n && h0 + i < k;
      re[i] = prepare<T, 2>(in ? X[((h0 + i) * ldx + j) * 2] : T(0), e_row, scale_bits);
      im[i] = prepare<T, 2>(in ? X[((h0 + i) * ldx + j) * 2 + 1] : T(0), e_row, scale_bits);
    }
    emit_oz1_any<PARAM>(re, [&](int t, unsigned int w) { tile[(t * 32 + lane) * PW + hw] = w; });
    emit_oz1_any<PARAM>(im, [&](int t, unsigned int w) { tile[((P + t) * 32 + lane) * PW + hw] = w; });
  }
  __syncthreads();
  const int64_t kk = 2 * kpad;
  for (int r = warp; r < 2 * P * 32; r += 8) {  // one warp writes one 128-byte row segment
    const int vp = r >> 5, jj = r & 31;
    const int64_t jg = static_cast<int64_t>(blockIdx.x) * 32 + jj;
    if (jg < n) {
      const int t = vp % P, halfsel = vp / P;
      *reinterpret_cast<unsigned int *>(out + (static_cast<int64_t>(t) * n + jg) * kk + halfsel * kpad + hb + lane * 4) =
          tile[(vp * 32 + jj) * PW + lane];
    }
  }
}

template <typename T, int P>
static int slice4m_p(emugemm_ctx *ctx, int is_b, int64_t rows, int64_t k, int64_t kpad, const void *X, int64_t ldx,
                     const unsigned long long *maxbits, int32_t *e, int slice_bits, int8_t *out) {
  cudaStream_t st = ctx->stream;
  const T *x = static_cast<const T *>(X);
  const int scale_bits = slice_bits == 8 ? 8 * P - 2 : kBeta * P;
  if (!is_b) {
    if (slice_bits == 8) oz1_4m_rows_kernel<T, 16 + P><<<static_cast<unsigned>(rows), 256, 0, st>>>(x, ldx, rows, k, kpad, e, scale_bits, out, ctx->nf_flag);
    else if (slice_bits == kDigitsTwos) oz1_4m_rows_kernel<T, 32 + P><<<static_cast<unsigned>(rows), 256, 0, st>>>(x, ldx, rows, k, kpad, e, scale_bits, out, ctx->nf_flag);
    else oz1_4m_rows_kernel<T, P><<<static_cast<unsigned>(rows), 256, 0, st>>>(x, ldx, rows, k, kpad, e, scale_bits, out, ctx->nf_flag);
  } else {
    const size_t smem = static_cast<size_t>(2 * P) * 32 * 33 * 4;
    const dim3 grid(static_cast<unsigned>((rows + 31) / 32), static_cast<unsigned>(kpad / 128));
    if (slice_bits == 8) {
      auto kern = oz1_4m_cols_kernel<T, 16 + P>;
      EMU_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 16 * 32 * 33 * 4));
      kern<<<grid, 256, smem, st>>>(x, ldx, rows, k, kpad, maxbits, e, scale_bits, P, out, ctx->nf_flag);
    } else if (slice_bits == kDigitsTwos) {
      auto kern = oz1_4m_cols_kernel<T, 32 + P>;
      EMU_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 16 * 32 * 33 * 4));
      kern<<<grid, 256, smem, st>>>(x, ldx, rows, k, kpad, maxbits, e, scale_bits, P, out, ctx->nf_flag);
    } else {
      auto kern = oz1_4m_cols_kernel<T, P>;
      EMU_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 16 * 32 * 33 * 4));
      kern<<<grid, 256, smem, st>>>(x, ldx, rows, k, kpad, maxbits, e, scale_bits, P, out, ctx->nf_flag);
    }
  }
  ctx->launches++;
  EMU_CUDA(ctx, cudaGetLastError());
  return EMUGEMM_OK;
}

// is_b = 0: A (rows x k complex) -> out[p][2 rows][2 kpad], e[2 rows];  is_b = 1: B (k x rows complex) ->
// out[p][rows][2 kpad], e[rows], maxbits from launch_colmax.  elem: kZ128 (complex128) or kC64 (complex64, p <= 4).
int launch_oz1_4m_slice(emugemm_ctx *ctx, int elem, int is_b, int64_t rows, int64_t k, int64_t kpad, const void *X, int64_t ldx,
                        const unsigned long long *maxbits, int32_t *e, int p, int slice_bits, int8_t *out) {
  if (rows == 0 || kpad == 0) return EMUGEMM_OK;
#define EMU_4M_CASE(T, PP) case PP: return slice4m_p<T, PP>(ctx, is_b, rows, k, kpad, X, ldx, maxbits, e, slice_bits, out)
  if (elem == kC64) {
    switch (p) {
      EMU_4M_CASE(float, 1); EMU_4M_CASE(float, 2); EMU_4M_CASE(float, 3); EMU_4M_CASE(float, 4);
      default: return EMUGEMM_ERR_ARG;
    }
  }
  switch (p) {
    EMU_4M_CASE(double, 1); EMU_4M_CASE(double, 2); EMU_4M_CASE(double, 3); EMU_4M_CASE(double, 4);
    EMU_4M_CASE(double, 5); EMU_4M_CASE(double, 6); EMU_4M_CASE(double, 7); EMU_4M_CASE(double, 8);
    default: return EMUGEMM_ERR_ARG;
  }
#undef EMU_4M_CASE
}

// ---- host helpers -----------------------------------------------------------
int oz2_moduli_host(int n, int *mod) {
  if (n < 1 || n > 24) return -1;
  for (int i = 0; i < n; ++i) mod[i] = h_moduli[i];
  return 0;
}

// T = max{T : k 2^(T+guard) <= P}, guard = 2 (real) / 3 (3M) (R12), with P as a
// 192-bit integer (three 64-bit limbs are enough: P < 2^156 for 20 moduli).
int oz2_budget_host(int n, int64_t k, int is3m, int *tA, int *tB) {
  if (n < 2 || n > kMaxModuli || k < 1) return -1;
  unsigned long long P[3] = {1, 0, 0};
  for (int l = 0; l < n; ++l) {
    unsigned __int128 c = 0;
    for (int i = 0; i < 3; ++i) {
      c += static_cast<unsigned __int128>(P[i]) * static_cast<unsigned>(h_moduli[l]);
      P[i] = static_cast<unsigned long long>(c);
      c >>= 64;
    }
  }
  const int guard = is3m ? 3 : 2;
  int T = -1;
  for (int t = 0; t + guard < 190; ++t) {
    // lhs = k << (t + guard) as 192 bits
    unsigned long long L[3] = {0, 0, 0};
    const int sh = t + guard, ws = sh / 64, bs = sh % 64;
    const unsigned long long kk = static_cast<unsigned long long>(k);
    if (ws < 3) L[ws] = kk << bs;
    if (bs && ws + 1 < 3) L[ws + 1] = kk >> (64 - bs);
    if (bs && ws + 1 >= 3 && (kk >> (64 - bs))) break;  // overflowed 192 bits
    int cmp = 0;
    for (int i = 2; i >= 0; --i) {
      if (L[i] != P[i]) { cmp = L[i] < P[i] ? -1 : 1; break; }
    }
    if (cmp <= 0) T = t; else break;
  }
  if (T < 0) return -1;
  *tB = T / 2;
  *tA = T - T / 2;
  return T;
}

}  // namespace emu
