// gemm_oz1.cu -- fused Ozaki Scheme I GEMM for sm_100a.
//
// What it computes (Eq. 2-3; Alg. 1): for one
// 128 x NT output tile, the p INT32 accumulators C_s = sum_{t+u=s} A'_t B'_u
// (s < p, only the p(p+1)/2 pairs with t + u < p), kept in tensor memory for the
// whole k-chunk, then C = alpha 2^(eA_i+eB_j-7(p+1)) sum_s 2^(7(p-1-s)) C_s + beta C
// in the epilogue.  INT32 never reaches global memory.
//
// B200-first design (differs from the paper's DeepGEMM kernel):
//  * Operands are slice-major K-major planes [p][rows][kpad]; one 3-D TMA box
//    brings ALL p slices of a 128-byte k-block of B into shared memory as one
//    contiguous (p*NT) x 128 B operand, A slices stream through their own ring
//    (A_t is needed only against B_0..B_{p-1-t}).
//  * "N-concatenation": the accumulators C_0..C_{p-1} are consecutive NT-column
//    blocks of TMEM and the B slices are consecutive NT-row blocks of one SMEM
//    operand, so A_t x [B_0 | ... | B_{p-1-t}] is ONE tcgen05.mma of width
//    (p-t) NT (two near-equal halves when > 256) writing columns [t NT, p NT):
//    exactly the products A_t B_u -> C_{t+u}.  A_t is fetched from shared memory
//    once per (t, k32) (A-operand collector across the two halves) instead of once
//    per product (12 instead of 36 MMAs per k32 at p = 8).
//  * A ring of slice PAIRS (j, p-1-j): every stage carries the same MMA time;
//    the issuing thread probes the next stage's barrier before issuing.
//  * Warp-specialised persistent CTA: warp 0 = TMA producer, warp 1 = MMA issuer
//    (one elected thread) + TMEM allocator, warps 2-9 = epilogue (accumulator
//    triples folded into exact int64, exponent-bias conversion, FP64 scaling).
//  * Clusters of 2: p >= 4 one tile per CTA, two N-adjacent tiles share A by TMA
//    multicast; p <= 3 a cta_group::2 pair owns one 256 x NT tile (one MMA per
//    product).  k-chunks that cannot overflow INT32 are work items of the same
//    launch.
#include "common.cuh"
#include "ptx.cuh"
#include "gemm_common.cuh"

namespace emu {


constexpr bool kUseCollector = true;  // A-operand collector reuse across the MMAs of one (t, ks)

template <int P, bool PAIR = false>
struct Oz1Cfg {
  // NT: tile width; P * NT <= 512 TMEM columns, every MMA width a multiple of 16
  static constexpr int NT = (P <= 2) ? 256 : (P == 3) ? 160 : (P == 4) ? 128 : (P == 5) ? 96 : (P == 6) ? 80 : 64;
  // PAIR (cta_group::2, P <= 3): a CTA pair owns a 256 x NT tile; each CTA stages only NT/2 rows of every B slice
  static constexpr int kBRows = PAIR ? NT / 2 : NT;
  static constexpr int kBStageBytes = P * kBRows * kBlockK;
  // B ring depth.  A k-block of B is released only when all P slices have used it, so its refill has one k-block of
  // MMA time to arrive: 4,608 clk at P = 8 but 1,536 clk at P = 2 -- pairs (small P, small stages) get three stages.
  static constexpr int SB = PAIR ? 3 : 2;
  // A ring: one stage = the slice PAIR (j, P-1-j) of a k-block (2 x 16 KB).  Pairing the widest with the
  // narrowest slice gives every stage the same MMA time ((P+1) NT/2 clk per k32), so the single issuing thread
  // pays one barrier wait + one commit per ~constant amount of tensor work and the MMA queue never drains
  // on the narrow slices (measured: +11 % tensor-pipe activity over one barrier per slice).
  static constexpr int NPAIR = (P + 1) / 2;
  static constexpr int kAPairBytes = 2 * kAStageBytes;
  static constexpr int kSAMax = 4;
  static constexpr int SA = (kSmemLimit - 2048 - SB * kBStageBytes) / kAPairBytes > kSAMax
                                ? kSAMax
                                : (kSmemLimit - 2048 - SB * kBStageBytes) / kAPairBytes;
  static constexpr int kTmemCols = (P * NT <= 256) ? 256 : 512;
  static constexpr int kSmemBytes = SB * kBStageBytes + SA * kAPairBytes + 1024 /*align*/ + 256 /*barriers*/;
  static_assert(P * NT <= 512, "TMEM budget");
  static_assert(kSmemBytes <= kSmemLimit, "SMEM budget");
  static_assert(SA >= 2, "A ring too shallow");
};

// MMAs of slice t for one 128-byte k-block: A_t x [B_0 | ... | B_{P-1-t}] -> TMEM columns [t NT, P NT), split at 256
// columns, four k32 sub-blocks.  `accumulate` = false only for the very first MMAs of a tile (t = 0, ks = 0).
template <int P, bool COLL>
__device__ __forceinline__ void oz1_issue_slice(int t, uint32_t tmem_base, uint32_t a_base, uint32_t b_base, bool accumulate,
                                                uint32_t imask = ~0u /* probes: clears the operand signedness bits */) {
  constexpr int NT = Oz1Cfg<P>::NT;
  // (P - t) NT columns: one MMA if <= 256, else two of near-equal width (multiples of 16).  An even split keeps
  // both above the ~112-column width below which an MMA is bound by its fixed cost (256 + 32 at p = 5, t = 2 would
  // run the 32-wide one at a third of the rate; 256 + 64 at p = 6, 7, 8 at two thirds).
  const int cols = (P - t) * NT;
  const int n0 = (cols <= 256) ? cols : ((cols / 2 + 15) / 16) * 16;
  const int n1 = cols - n0;
  const uint32_t a_lo = sdesc_lo(a_base), b_lo = sdesc_lo(b_base);  // per MMA: one add on the address field
#pragma unroll
  for (int ks = 0; ks < kBlockK / 32; ++ks) {
    const uint64_t adesc = sdesc_from_lo(a_lo + ((ks * 32) >> 4));
    const uint32_t acc = (accumulate || ks != 0) ? 1u : 0u;
    const uint32_t d = tmem_base + t * NT;
    const uint64_t bdesc0 = sdesc_from_lo(b_lo + ((ks * 32) >> 4));
    if (n1 == 0) {
      umma_i8<0>(d, adesc, bdesc0, make_idesc_i8(kTileM, n0) & imask, acc);
    } else {
      // the two MMAs share A_t: the first keeps it in the collector, the second drops it
      const uint64_t bdesc1 = sdesc_from_lo(b_lo + ((n0 * kBlockK + ks * 32) >> 4));
      if (COLL) {
        umma_i8<1>(d, adesc, bdesc0, make_idesc_i8(kTileM, n0) & imask, acc);
        umma_i8<3>(d + n0, adesc, bdesc1, make_idesc_i8(kTileM, n1) & imask, acc);
      } else {
        umma_i8<0>(d, adesc, bdesc0, make_idesc_i8(kTileM, n0) & imask, acc);
        umma_i8<0>(d + n0, adesc, bdesc1, make_idesc_i8(kTileM, n1) & imask, acc);
      }
    }
  }
}

// CTA-pair schedule (cta_group::2, used for P <= 3; needs NT >= 128): one 256 x NT x 32 MMA per product, issued by the leader
// CTA for both SMs; CTA r supplies rows 128 r .. of A_t and rows NT/2 r .. of B_u from its own shared memory, so the
// columns of D come out in natural order and land on C_{t+u}.  A_t stays in the collector across its P - t MMAs.
template <int P>
__device__ __forceinline__ void oz1_issue_slice_pair(int t, uint32_t tmem_base, uint32_t a_base, uint32_t b_base, bool accumulate) {
  constexpr int NT = Oz1Cfg<P, true>::NT;
  constexpr uint32_t idesc = make_idesc_i8(2 * kTileM, NT);
  const uint32_t a_lo = sdesc_lo(a_base), b_lo = sdesc_lo(b_base);
#pragma unroll
  for (int ks = 0; ks < kBlockK / 32; ++ks) {
    const uint64_t adesc = sdesc_from_lo(a_lo + ((ks * 32) >> 4));
#pragma unroll
    for (int u = 0; u < P; ++u) {
      if (u < P - t) {
        const uint32_t acc = (accumulate || ks != 0) ? 1u : 0u;
        const uint32_t d = tmem_base + (t + u) * NT;
        const uint64_t bdesc = sdesc_from_lo(b_lo + ((u * (NT / 2) * kBlockK + ks * 32) >> 4));
        const bool first = (u == 0), last = (u == P - t - 1);
        if (first && !last) umma_i8_cg2<1>(d, adesc, bdesc, idesc, acc);
        else if (!first && last) umma_i8_cg2<3>(d, adesc, bdesc, idesc, acc);
        else if (!first && !last) umma_i8_cg2<2>(d, adesc, bdesc, idesc, acc);
        else umma_i8_cg2<0>(d, adesc, bdesc, idesc, acc);
      }
    }
  }
}

struct Oz1Dev {
  int64_t m, n;
  int kb0, kb1;       // k-blocks [kb0, kb1) of 128
  int chunk_kb, nch;  // overflow-safe k-chunks of chunk_kb k-blocks each: a work item is (chunk, tile)
  int64_t chunk_stride;  // bytes between the outputs of consecutive chunks (OUT = 2 dump, OUT = 3 partials)
  int mt, nt_tiles;   // tile grid
  int nbatch;         // strided batched call: entry b uses plane rows [b m, (b+1) m) / [b n, (b+1) n), exponents likewise
  int64_t batch_stride_c;  // bytes between the C matrices of consecutive entries
  const int32_t *eA, *eB;
  int out_kind;
  double alpha, beta;
  void *C;
  int64_t ldc;
  unsigned long long *cycles;
  int slice_bits;  // 7 or 8
  int group_m;     // rasterisation group (tile_coords)
  int serp;        // 1: every other tile of a CTA walks k downwards, so the k-blocks its L2 neighbourhood used last come first
  unsigned long long *wave_ctr;  // wave barrier (null: none): all CTAs start their w-th tile together, so that the CTAs
                                 // sharing an A or B panel ask for the same k-block at the same time (one DRAM read)
  int n_waves;                   // ceil(items / workers): every CTA arrives that many times
  int dbg;  // experiment flags (emugemm_dbg_set_flags): 1 = no TMA after the ring is first filled, 2 = no epilogue math
};

__device__ __forceinline__ double pow2d(int e) {  // 2^e for -1022 <= e <= 1023
  return __hiloint2double((1023 + e) << 20, 0);
}
// exact double of x * 2^sh (x int32) without I2F: bit pattern 2^(52+sh) + (x + 2^31) 2^sh, minus that offset
__device__ __forceinline__ double i32_scaled(uint32_t x, int sh) {
  const double magic = __hiloint2double((0x433 + sh) << 20, static_cast<int>(x ^ 0x80000000u));
  const double off = __hiloint2double((0x433 + sh) << 20, 0) + __hiloint2double((0x3FF + 31 + sh) << 20, 0);
  return magic - off;
}

// exact double of G * 2^sh for an int64 |G| < 2^51 that already carries the bias magic_bias(sh): the bits are the
// double (2^52 + 2^51 + G) 2^sh; subtracting 1.5 * 2^(52+sh) is exact.
__device__ __forceinline__ constexpr long long magic_bias(int sh) { return (static_cast<long long>(0x433 + sh) << 52) + (1LL << 51); }
__device__ __forceinline__ double unbias(long long biased, int sh) {
  return __longlong_as_double(biased) - __longlong_as_double((static_cast<long long>(0x433 + sh) << 52) + (1LL << 51));
}

// Epilogue arithmetic (Eq. 3 + scaling) for one row x 8 columns x P accumulators.
// The accumulators are folded three at a time into exact 64-bit integers G_g = C_s 2^14 + C_{s+1} 2^7 + C_{s+2}
// (|G| < 2^46, integer multiply-adds), each converted exactly with the exponent-bias trick, so only
// ceil(P/3) - 1 FP64 additions round.
// OUT: 0 final FP64 C, 1 final FP32 C, 2 INT32 accumulator dump (test hook), 3 exact double-double k-chunk partial.
template <int P, int OUT>
struct Oz1Epi {
  static constexpr int NG = (P + 2) / 3;  // groups, most significant first; the last may hold 1 or 2 accumulators
  bool vec_c, vec_e;
  int w1, w2;             // 2^bits, 2^(2 bits): weights inside a group (bits = 7 or 8, run-time: same code for R1 and R23)
  long long bias[NG];     // exponent-bias constants per group
  double unb[NG];
  int e_off;              // exponent of the scaling besides eA_i + eB_j
  // vector access flags of the current work item (its C and column exponents may start anywhere in a batch)
  __device__ __forceinline__ void set_item(const Oz1Dev &a) {
    vec_c = (a.ldc % 4 == 0) && ((reinterpret_cast<uintptr_t>(a.C) & 31) == 0);
    vec_e = (reinterpret_cast<uintptr_t>(a.eB) & 15) == 0;
  }
  __device__ __forceinline__ void init(const Oz1Dev &a) {
    set_item(a);
    const int bits = a.slice_bits & 0xFF;  // kDigitsTwos: 7-bit weights like R1
    w1 = 1 << bits;
    w2 = 1 << (2 * bits);
#pragma unroll
    for (int g = 0; g < NG; ++g) {
      const int s1 = (3 * g + 2 < P - 1) ? 3 * g + 2 : P - 1;
      const int sh = bits * (P - 1 - s1);
      bias[g] = (static_cast<long long>(0x433 + sh) << 52) + (1LL << 51);
      unb[g] = __longlong_as_double(bias[g]);
    }
    e_off = (bits == 8 ? 4 : 0) - bits * (P + 1);  // R23: two guard bits per operand
  }
  // group g covers accumulators s = 3g .. min(3g+2, P-1); its weight is 2^(bits (P-1-last)); |G| < 2^49 < 2^51
  __device__ __forceinline__ double group(const uint32_t (&v)[P][8], int c, int g) const {
    const int s0 = 3 * g, s1 = (3 * g + 2 < P - 1) ? 3 * g + 2 : P - 1;
    long long G = bias[g];
#pragma unroll
    for (int s = s0; s <= s1; ++s) {  // IMAD.WIDE: sign-extending 32 x 32 -> 64 multiply-add
      const int w = (s1 - s == 0) ? 1 : (s1 - s == 1) ? w1 : w2;
      G += static_cast<long long>(static_cast<int32_t>(v[s][c])) * static_cast<long long>(w);
    }
    return __longlong_as_double(G) - unb[g];
  }
  // column exponents of one 8-column chunk (issued one chunk ahead of their use: the load latency is hidden)
  __device__ __forceinline__ void load_eb(const Oz1Dev &a, int64_t gcol, int (&eb)[8]) const {
    if constexpr (OUT != 2) {
      if (gcol + 8 <= a.n && vec_e) {
        const int4 e0 = __ldg(reinterpret_cast<const int4 *>(a.eB + gcol)), e1 = __ldg(reinterpret_cast<const int4 *>(a.eB + gcol) + 1);
        eb[0] = e0.x; eb[1] = e0.y; eb[2] = e0.z; eb[3] = e0.w; eb[4] = e1.x; eb[5] = e1.y; eb[6] = e1.z; eb[7] = e1.w;
      } else {
#pragma unroll
        for (int c = 0; c < 8; ++c) eb[c] = (gcol + c < a.n) ? __ldg(a.eB + gcol + c) : 0;
      }
    }
  }
  __device__ __forceinline__ void chunk(const Oz1Dev &a, const uint32_t (&v)[P][8], const int (&eb)[8], int64_t grow, bool row_ok,
                                        int eArow, int64_t gcol) const {
    if constexpr (OUT == 2) {
      if (row_ok) {
        int32_t *o = static_cast<int32_t *>(a.C);
#pragma unroll
        for (int s = 0; s < P; ++s)
#pragma unroll
          for (int c = 0; c < 8; ++c)
            if (gcol + c < a.n) o[(static_cast<int64_t>(s) * a.m + grow) * a.n + gcol + c] = static_cast<int32_t>(v[s][c]);
      }
      return;
    } else {
      const bool full = gcol + 8 <= a.n;
      double r[8], rlo[8];
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        // least significant group first; every group value is exact, each addition rounds at most 1/2 ulp of a
        // partial sum bounded by (|A'||B'|)_ij
        double acc = group(v, c, NG - 1), lo = 0.0;
        if constexpr (OUT != 3) {
#pragma unroll
          for (int g = NG - 2; g >= 0; --g) acc += group(v, c, g);
        } else {  // exact double-double (TwoSum): hi + lo == S exactly (S < 2^82, the error terms are small integers)
#pragma unroll
          for (int g = NG - 2; g >= 0; --g) {
            const double t = group(v, c, g);
            const double sum = acc + t;
            const double bb = sum - acc;
            lo += (acc - (sum - bb)) + (t - bb);
            acc = sum;
          }
        }
        // power-of-two scaling 2^E, E = eA_i + eB_j - 7 (p+1), as two factors: the first is clamped so that acc 2^h1
        // (|acc| an integer below 2^83, or 0) stays a normal number, the second (clamped to the exponent range) takes the
        // result to zero / subnormal / infinity when it must: one rounding for every finite input (operands
        // near DBL_MIN made E >> 1 fall below -1022 and the exponent field wrap)
        const int E = eArow + eb[c];
        const int h1 = max(min(E, 930), -1000);
        const int h2 = max(min(E - h1, 1023), -1022);
        const double d1 = pow2d(h1), d2 = pow2d(h2);
        r[c] = acc * d1 * d2;
        if constexpr (OUT == 3) rlo[c] = lo * d1 * d2;
      }
      if (!row_ok || EMU_PROBE_FLAG(a.dbg, 4)) return;
      if constexpr (OUT == 3) {  // k-chunk partial as double-double [m][n][2]
        double *o = static_cast<double *>(a.C) + (grow * a.n + gcol) * 2;
#pragma unroll
        for (int c = 0; c < 8; ++c)
          if (gcol + c < a.n) { o[2 * c] = r[c]; o[2 * c + 1] = rlo[c]; }
      } else if constexpr (OUT == 0) {
        double *o = static_cast<double *>(a.C) + grow * a.ldc + gcol;
        if (a.beta != 0.0) {
#pragma unroll
          for (int c = 0; c < 8; ++c)
            if (gcol + c < a.n) r[c] = fma(a.alpha, r[c], a.beta * o[c]);
        } else if (a.alpha != 1.0) {
#pragma unroll
          for (int c = 0; c < 8; ++c) r[c] *= a.alpha;
        }
        if (full && vec_c) {
          asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(o), "d"(r[0]), "d"(r[1]), "d"(r[2]), "d"(r[3]) : "memory");
          asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(o + 4), "d"(r[4]), "d"(r[5]), "d"(r[6]), "d"(r[7]) : "memory");
        } else {
#pragma unroll
          for (int c = 0; c < 8; ++c)
            if (gcol + c < a.n) o[c] = r[c];
        }
      } else {  // OUT == 1: FP32 C, one rounding to float
        float *o = static_cast<float *>(a.C) + grow * a.ldc + gcol;
        float f[8];
#pragma unroll
        for (int c = 0; c < 8; ++c) {
          double x = a.alpha * r[c];
          if (a.beta != 0.0 && gcol + c < a.n) x = fma(a.beta, static_cast<double>(o[c]), x);
          f[c] = static_cast<float>(x);
        }
        if (full && vec_c) {
          *reinterpret_cast<float4 *>(o) = make_float4(f[0], f[1], f[2], f[3]);
          *reinterpret_cast<float4 *>(o + 4) = make_float4(f[4], f[5], f[6], f[7]);
        } else {
#pragma unroll
          for (int c = 0; c < 8; ++c)
            if (gcol + c < a.n) o[c] = f[c];
        }
      }
    }
  }
};

// MC (one-CTA tiles, P >= 5): a cluster of 2 CTAs works on two N-adjacent tiles of the same 128-row block; each CTA
// fetches half of the rows of every A slice and TMA-multicasts them to both, so A crosses L2 -> SM once per
// cluster (-33 % operand traffic at NT = 64; operand movement costs clock through the power cap).
template <int P, int OUT, bool PAIR, bool MC>
__global__ void __launch_bounds__(kGemmThreads, 1)
oz1_gemm_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const Oz1Dev a) {
  using Cfg = Oz1Cfg<P, PAIR>;
  constexpr int NT = Cfg::NT, SA = Cfg::SA, SB = Cfg::SB;
  extern __shared__ uint8_t smem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t *sB = smem;
  uint8_t *sA = smem + SB * Cfg::kBStageBytes;
  uint64_t *bars = reinterpret_cast<uint64_t *>(sA + SA * Cfg::kAPairBytes);
  uint64_t *bfull = bars, *bempty = bars + SB, *afull = bars + 2 * SB, *aempty = bars + 2 * SB + SA;
  uint64_t *tfull = bars + 2 * SB + 2 * SA, *tempty = tfull + 1;
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(tempty + 1);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int num_tiles = a.mt * a.nt_tiles;
  const int per_entry = num_tiles * a.nch;  // chunk-major: consecutive items share the k-range of their operands
  const int num_items = per_entry * a.nbatch;  // entry-major: item = (batch entry, chunk, tile)
  // PAIR: the two CTAs of a cluster work on one 256-row tile; rank 0 (leader) issues the MMAs for both
  static_assert(!(PAIR && MC), "pairs already share operands");
  constexpr bool CL2 = PAIR || MC;  // launched as clusters of 2
  const uint32_t cta = CL2 ? cluster_ctarank() : 0u;
  const int work_id = CL2 ? static_cast<int>(blockIdx.x >> 1) : static_cast<int>(blockIdx.x);
  const int num_workers = CL2 ? static_cast<int>(gridDim.x >> 1) : static_cast<int>(gridDim.x);
  constexpr int kTileRows = PAIR ? 2 * kTileM : kTileM;
  constexpr uint32_t kTxMul = PAIR ? 2u : 1u;  // the leader's "full" barriers collect the bytes of both CTAs

  if (threadIdx.x == 0) {
    for (int i = 0; i < SB; ++i) { mbar_init(&bfull[i], 1); mbar_init(&bempty[i], 1); }
    // MC: a stage is refilled (in BOTH CTAs, by multicast) only after both CTAs' MMAs have read it
    for (int i = 0; i < SA; ++i) { mbar_init(&afull[i], 1); mbar_init(&aempty[i], MC ? 2 : 1); }
    mbar_init(tfull, 1);
    mbar_init(tempty, PAIR ? 2 * kEpiWarps : kEpiWarps);
    fence_mbar_init();
    tma_prefetch_desc(&tmA);
    tma_prefetch_desc(&tmB);
  }
  if (warp == 1) {
    if constexpr (PAIR) { tmem_alloc_cg2(tmem_slot, Cfg::kTmemCols); tmem_relinquish_cg2(); }
    else { tmem_alloc(tmem_slot, Cfg::kTmemCols); tmem_relinquish(); }
  }
  tc_fence_before();
  if constexpr (CL2) cluster_sync_all(); else __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const long long t_start = clock64();

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (lane == 0) {
      int sa = 0, sb = 0, nloada = 0, nloadb = 0;
      uint32_t pa = 0, pb = 0;
      // L2 eviction hints were measured and dropped twice: without the wave barrier EVICT_LAST on A changes nothing (15.1 vs
      // 15.2 GB) and EVICT_FIRST on B raises the DRAM reads to 21.9 GB; with the barrier A EVICT_LAST / B EVICT_FIRST /
      // B EVICT_LAST all time within noise of the plain policy (11.98-12.24 against 11.88-12.00 ms at 8192^3 p = 8)
      // (probes build: 0x200000 = A EVICT_LAST, 0x400000 = B EVICT_FIRST, 0x800000 = B EVICT_LAST, for the DRAM-byte captures)
      const uint64_t polA = EMU_PROBE_FLAG(a.dbg, 0x200000) ? kEvictLast : kEvictNormal;
      const uint64_t polB = EMU_PROBE_FLAG(a.dbg, 0x400000) ? kEvictFirst : EMU_PROBE_FLAG(a.dbg, 0x800000) ? kEvictLast : kEvictNormal;
      int wave = 0;
      bool wave_off = false;  // a barrier wait ran into its bound: stop waiting (keep arriving) for the rest of the launch
      for (int item = work_id; item < num_items; item += num_workers, ++wave) {
        // static round-robin keeps the tiles of a wave adjacent, but CTAs drift apart by whole tiles over a launch (the
        // per-SM speed differs by a few per cent) and then every CTA streams its own copy of the panels from DRAM
        // (13.7 GB instead of ~7 GB per 8192^3 p = 8 launch, ncu): re-align the producers at every tile
        if (a.wave_ctr && wave > 0 && !wave_off) wave_off = !grid_wait(a.wave_ctr, static_cast<unsigned long long>(wave) * gridDim.x);
        const int bidx = item / per_entry, rem = item - bidx * per_entry;
        const int chunk = rem / num_tiles, tile = rem - chunk * num_tiles;
        const int kb0 = a.kb0 + chunk * a.chunk_kb, kb1 = (kb0 + a.chunk_kb < a.kb1) ? kb0 + a.chunk_kb : a.kb1;
        int mb, nb;
        tile_coords(tile, a.mt, a.nt_tiles, mb, nb, a.group_m);
        if (EMU_PROBE_FLAG(a.dbg, 64)) { mb = 0; nb = 0; }  // probe: every CTA loads tile (0, 0): no DRAM traffic, same L2 -> SM traffic
        if constexpr (MC) nb = 2 * nb + static_cast<int>(cta);  // a.nt_tiles counts PAIRS of N-tiles
        const int rowA0 = static_cast<int>(bidx * a.m), rowB0 = static_cast<int>(bidx * a.n);  // this entry's plane rows
        // integer accumulation is exact in any order: odd tiles of this CTA walk k downwards (serpentine), so the k-blocks
        // the previous tile (and its L2 neighbours) touched last are the first ones asked for again
        const bool rev = a.serp && (((item - work_id) / num_workers) & 1);
        const int nkb = kb1 - kb0;
        auto load_b = [&](int kbx) {
          mbar_wait(&bempty[sb], pb ^ 1);
          if constexpr (PAIR) {
            if (cta == 0) mbar_arrive_expect_tx(&bfull[sb], kTxMul * Cfg::kBStageBytes);
            tma_load_3d_cg2(sB + sb * Cfg::kBStageBytes, &tmB, mapa_u32(&bfull[sb], 0), kbx * kBlockK,
                            rowB0 + nb * NT + static_cast<int>(cta) * Cfg::kBRows, 0, polB);
          } else if (EMU_PROBE_FLAG(a.dbg, 1) && nloadb >= SB) {
            mbar_arrive(&bfull[sb]);
          } else {
            mbar_arrive_expect_tx(&bfull[sb], Cfg::kBStageBytes);
            tma_load_3d(sB + sb * Cfg::kBStageBytes, &tmB, &bfull[sb], kbx * kBlockK, rowB0 + nb * NT, 0, polB);
          }
          ++nloadb;
          if (++sb == SB) { sb = 0; pb ^= 1; }
        };
        // B of k-block kb + 1 goes into the stage k-block kb - 1 used, which is released together with the A stage that
        // (kb, 2) refills: with four pair stages per k-block (P = 7, 8) the B load is issued there, one A stage earlier than
        // at the top of its own k-block, so that its 56-64 KB are not in the way of the next k-block's first A stages
        // (p = 7: 0.884 -> 0.913 per clock, p = 8: 0.941 -> 0.946; with three stages per k-block the two places coincide)
        constexpr bool early_b = !PAIR && Cfg::NPAIR >= 4;
        // the arrival on the wave barrier is signalled kWaveLead k-blocks before the last load of the tile: the slowest CTA
        // then releases the others while it still has that much of its tile to go, so the fast ones do not idle at the
        // barrier, and the drift stays within a few k-blocks (the panels of that window are a few MB of L2)
        constexpr int kWaveLead = 6;
        const int lead = EMU_PROBE_FLAG(a.dbg, 0x0F000000) ? 2 * ((EMU_PROBE_FLAG(a.dbg, 0x0F000000) >> 24) - 1) : kWaveLead;  // probe: 0, 2, ... 28
        const int arrive_it = nkb - 1 - lead > 0 ? nkb - 1 - lead : 0;
        for (int it = 0; it < nkb; ++it) {
          const int kb = rev ? kb1 - 1 - it : kb0 + it;
          const int kb_next = rev ? kb - 1 : kb + 1;
          if (a.wave_ctr && it == arrive_it) grid_arrive(a.wave_ctr);
          if (!early_b || it == 0) load_b(kb);
#pragma unroll 1
          for (int j = 0; j < Cfg::NPAIR; ++j) {
            const int lo = j, hi = P - 1 - j;
            mbar_wait(&aempty[sa], pa ^ 1);
            uint8_t *dst = sA + sa * Cfg::kAPairBytes;
            if constexpr (PAIR) {
              const uint32_t bar = mapa_u32(&afull[sa], 0);
              const int arow = rowA0 + mb * kTileRows + static_cast<int>(cta) * kTileM;
              if (cta == 0) mbar_arrive_expect_tx(&afull[sa], kTxMul * (lo == hi ? kAStageBytes : Cfg::kAPairBytes));
              tma_load_3d_cg2(dst, &tmA, bar, kb * kBlockK, arow, lo, polA);
              if (hi != lo) tma_load_3d_cg2(dst + kAStageBytes, &tmA, bar, kb * kBlockK, arow, hi, polA);
            } else if constexpr (MC) {
              // this CTA fetches rows [64 cta, 64 cta + 64) of both slices and multicasts them to the pair
              constexpr int kHalf = kAStageBytes / 2;
              const int arow = rowA0 + mb * kTileM + static_cast<int>(cta) * (kTileM / 2);
              mbar_arrive_expect_tx(&afull[sa], lo == hi ? kAStageBytes : Cfg::kAPairBytes);
              tma_load_3d_mc(dst + cta * kHalf, &tmA, &afull[sa], kb * kBlockK, arow, lo, 3, polA);
              if (hi != lo) tma_load_3d_mc(dst + kAStageBytes + cta * kHalf, &tmA, &afull[sa], kb * kBlockK, arow, hi, 3, polA);
            } else if (EMU_PROBE_FLAG(a.dbg, 1) && nloada >= SA) {
              mbar_arrive(&afull[sa]);
            } else {
              mbar_arrive_expect_tx(&afull[sa], lo == hi ? kAStageBytes : Cfg::kAPairBytes);
              tma_load_3d(dst, &tmA, &afull[sa], kb * kBlockK, rowA0 + mb * kTileM, lo, polA);
              if (hi != lo) tma_load_3d(dst + kAStageBytes, &tmA, &afull[sa], kb * kBlockK, rowA0 + mb * kTileM, hi, polA);
            }
            ++nloada;
            if (++sa == SA) { sa = 0; pa ^= 1; }
            if (early_b && j == 2 && it + 1 < nkb) load_b(kb_next);
          }
        }
      }
      if (a.wave_ctr)
        for (; wave < a.n_waves; ++wave) grid_arrive(a.wave_ctr);  // no tile in the last wave(s): the others must not wait for us
    }
    __syncwarp();
  } else if (warp == 1) {
    // ===================== MMA issuer (PAIR: leader CTA only) =====================
    if (lane == 0 && (!PAIR || cta == 0)) {
      int sa = 0, sb = 0;
      uint32_t pa = 0, pb = 0, pt = 0;
      // look-ahead: the barrier of the NEXT stage is probed (non-blocking) before the MMAs of the current stage are
      // issued, so the ~90-cycle try_wait latency overlaps tensor work instead of draining the MMA queue
      bool a_ready = false, b_ready = false;
      for (int item = work_id; item < num_items; item += num_workers) {
        const int bidx = item / per_entry, rem = item - bidx * per_entry;
        const int chunk = rem / num_tiles, tile = rem - chunk * num_tiles;
        const int kb0 = a.kb0 + chunk * a.chunk_kb, kb1 = (kb0 + a.chunk_kb < a.kb1) ? kb0 + a.chunk_kb : a.kb1;
        mbar_wait(tempty, pt ^ 1);  // epilogue has drained the accumulators of the previous tile
        tc_fence_after();
        for (int kb = kb0; kb < kb1; ++kb) {
          if (!b_ready) mbar_wait(&bfull[sb], pb);
          const uint32_t b_base = smem_u32(sB + sb * Cfg::kBStageBytes);
          const int sb_next = (sb + 1 == SB) ? 0 : sb + 1;
          const uint32_t pb_next = (sb + 1 == SB) ? pb ^ 1 : pb;
#pragma unroll
          for (int j = 0; j < Cfg::NPAIR; ++j) {
            const int lo = j, hi = P - 1 - j;
            if (!a_ready) mbar_wait(&afull[sa], pa);
            tc_fence_after();
            const uint32_t a_base = smem_u32(sA + sa * Cfg::kAPairBytes);
            const int sa_cur = sa;
            if (++sa == SA) { sa = 0; pa ^= 1; }
            a_ready = mbar_try_wait(&afull[sa], pa);
            if (j == Cfg::NPAIR - 1) b_ready = mbar_try_wait(&bfull[sb_next], pb_next);
            if constexpr (PAIR) {
              oz1_issue_slice_pair<P>(lo, tmem_base, a_base, b_base, kb != kb0 || lo != 0);
              if (hi != lo) oz1_issue_slice_pair<P>(hi, tmem_base, a_base + kAStageBytes, b_base, true);
              umma_commit_cg2(&aempty[sa_cur], 3);  // both CTAs' stages reusable once these MMAs have read them
            } else {
              // probes build, 0x40000000: the MMAs treat both operands as UNSIGNED bytes (results wrong): all products
              // non-negative, same bytes -- what operand / accumulator signs cost in clock under the power cap
              const uint32_t imask = EMU_PROBE_FLAG(a.dbg, 0x40000000) ? ~((1u << 7) | (1u << 10)) : ~0u;
              oz1_issue_slice<P, kUseCollector>(lo, tmem_base, a_base, b_base, kb != kb0 || lo != 0, imask);
              if (hi != lo) oz1_issue_slice<P, kUseCollector>(hi, tmem_base, a_base + kAStageBytes, b_base, true, imask);
              if constexpr (MC) umma_commit_mc(&aempty[sa_cur], 3);  // both CTAs must be done before either refills
              else umma_commit(&aempty[sa_cur]);                     // stage reusable once these MMAs have read it
            }
          }
          if constexpr (PAIR) umma_commit_cg2(&bempty[sb], 3); else umma_commit(&bempty[sb]);
          sb = sb_next; pb = pb_next;
        }
        if constexpr (PAIR) umma_commit_cg2(tfull, 3); else umma_commit(tfull);  // accumulators complete
        pt ^= 1;
      }
    }
    __syncwarp();
  } else {
    // ===================== epilogue =====================
    const int ew = warp - 2;
    const int quad = warp & 3;     // TMEM lane quadrant this warp may read
    const int half = ew >> 2;      // column half
    const int row = quad * 32 + lane;
    const uint32_t trow = tmem_base + (static_cast<uint32_t>(quad * 32) << 16);
    uint32_t pt = 0;
    Oz1Epi<P, OUT> epi;
    epi.init(a);
    constexpr int kChunks = NT / 2 / 8;  // 8-column chunks per thread
    constexpr bool kDoubleBuffer = (P <= 6);  // two register sets of P x 8 accumulator values fit without spilling
    Oz1Dev ac = a;  // per-item copy: the output of chunk c starts c * chunk_stride bytes further
    for (int item = work_id; item < num_items; item += num_workers) {
      const int bidx = item / per_entry, rem = item - bidx * per_entry;
      const int chunk = rem / num_tiles, tile = rem - chunk * num_tiles;
      ac.C = static_cast<char *>(a.C) + chunk * a.chunk_stride + bidx * a.batch_stride_c;
      ac.eA = a.eA + bidx * a.m;
      ac.eB = a.eB + bidx * a.n;
      epi.set_item(ac);
      int mb, nb;
      tile_coords(tile, a.mt, a.nt_tiles, mb, nb, a.group_m);
      if constexpr (MC) nb = 2 * nb + static_cast<int>(cta);
      const int64_t grow = static_cast<int64_t>(mb) * kTileRows + (PAIR ? cta * kTileM : 0u) + row;
      const bool row_ok = grow < a.m;
      const int eArow = row_ok ? __ldg(ac.eA + grow) + epi.e_off : 0;
      const int64_t gcol0 = static_cast<int64_t>(nb) * NT + half * (NT / 2);
      int ea[8], eb[8];
      epi.load_eb(ac, gcol0, ea);  // first chunk's column exponents: in flight while the tile's MMAs finish
      mbar_wait(tfull, pt);
      tc_fence_after();
      if (!EMU_PROBE_FLAG(a.dbg, 2)) {
        const uint32_t tcol = trow + half * (NT / 2);
        if constexpr (kDoubleBuffer) {
          // software pipeline: the TMEM loads and column exponents of chunk i+1 are in flight while chunk i is
          // converted and stored
          uint32_t va[P][8], vb[P][8];
#pragma unroll
          for (int s = 0; s < P; ++s) tmem_ld8(tcol + s * NT, va[s]);
#pragma unroll 1
          for (int i = 0; i < kChunks; i += 2) {
            tmem_ld_wait();
            if (i + 1 < kChunks) {
#pragma unroll
              for (int s = 0; s < P; ++s) tmem_ld8(tcol + s * NT + (i + 1) * 8, vb[s]);
              epi.load_eb(ac, gcol0 + (i + 1) * 8, eb);
            }
            epi.chunk(ac, va, ea, grow, row_ok, eArow, gcol0 + i * 8);
            if (i + 1 < kChunks) {
              tmem_ld_wait();
              if (i + 2 < kChunks) {
#pragma unroll
                for (int s = 0; s < P; ++s) tmem_ld8(tcol + s * NT + (i + 2) * 8, va[s]);
                epi.load_eb(ac, gcol0 + (i + 2) * 8, ea);
              }
              epi.chunk(ac, vb, eb, grow, row_ok, eArow, gcol0 + (i + 1) * 8);
            }
          }
        } else {
          // P >= 7: one register set; only the column exponents are prefetched a chunk ahead
          uint32_t v[P][8];
#pragma unroll 1
          for (int i = 0; i < kChunks; i += 2) {
#pragma unroll
            for (int s = 0; s < P; ++s) tmem_ld8(tcol + s * NT + i * 8, v[s]);
            if (i + 1 < kChunks) epi.load_eb(ac, gcol0 + (i + 1) * 8, eb);
            tmem_ld_wait();
            epi.chunk(ac, v, ea, grow, row_ok, eArow, gcol0 + i * 8);
            if (i + 1 < kChunks) {
#pragma unroll
              for (int s = 0; s < P; ++s) tmem_ld8(tcol + s * NT + (i + 1) * 8, v[s]);
              if (i + 2 < kChunks) epi.load_eb(ac, gcol0 + (i + 2) * 8, ea);
              tmem_ld_wait();
              epi.chunk(ac, v, eb, grow, row_ok, eArow, gcol0 + (i + 1) * 8);
            }
          }
        }
      }
      // all TMEM reads of this tile are complete (tcgen05.wait::ld above): release the accumulators
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        if constexpr (PAIR) mbar_arrive_remote(mapa_u32(tempty, 0)); else mbar_arrive(tempty);
      }
      pt ^= 1;
    }
  }

  tc_fence_before();
  if constexpr (CL2) cluster_sync_all(); else __syncthreads();
  if (warp == 1) {
    if constexpr (PAIR) tmem_dealloc_cg2(tmem_base, Cfg::kTmemCols); else tmem_dealloc(tmem_base, Cfg::kTmemCols);
  }
  if (blockIdx.x == 0 && threadIdx.x == 0 && a.cycles) atomicAdd(a.cycles, static_cast<unsigned long long>(clock64() - t_start));
}

// P <= 3 runs as CTA pairs (cta_group::2, one MMA per product, NT >= 160); P >= 4 uses N-concatenated MMAs, whose
// columns a pair would split between the two CTAs' B halves, so it stays one CTA per tile, two N-adjacent tiles per
// cluster sharing A by TMA multicast.  Same-run A/B at 8192^3: p = 3 pairs +6 %, p = 4 one-CTA +4 %.
template <int P, bool PAIR, bool MC>
static int launch_pp(emugemm_ctx *ctx, const Oz1GemmArgs &g) {
  using Cfg = Oz1Cfg<P, PAIR>;
  constexpr int kTileRows = PAIR ? 2 * kTileM : kTileM;
  CUtensorMap tmA, tmB;
  const int batch = g.batch > 0 ? g.batch : 1;
  if (batch > 1 && g.n_chunks > 1) return EMUGEMM_ERR_ARG;  // the API runs chunked entries one by one
  EMU_TRY(encode_planes_tmap(ctx, &tmA, g.SA, g.kpad, g.m * batch, P, MC ? kTileM / 2 : kTileM, 1));
  EMU_TRY(encode_planes_tmap(ctx, &tmB, g.SB, g.kpad, g.n * batch, P, Cfg::kBRows, P));
  Oz1Dev d;
  d.m = g.m; d.n = g.n;
  d.kb0 = static_cast<int>(g.k0 / kBlockK);
  d.kb1 = static_cast<int>(g.k1 / kBlockK);
  d.nch = g.n_chunks > 0 ? g.n_chunks : 1;
  d.chunk_kb = g.n_chunks > 1 ? static_cast<int>(g.chunk_k / kBlockK) : d.kb1 - d.kb0;
  d.chunk_stride = g.chunk_stride;
  d.mt = static_cast<int>((g.m + kTileRows - 1) / kTileRows);
  d.nt_tiles = static_cast<int>((g.n + Cfg::NT - 1) / Cfg::NT);
  if (MC) d.nt_tiles = (d.nt_tiles + 1) / 2;  // pairs of N-adjacent tiles, one per CTA of the cluster
  d.nbatch = batch; d.batch_stride_c = g.batch_stride_c;
  d.eA = g.eA; d.eB = g.eB;
  d.out_kind = g.out_kind; d.alpha = g.alpha; d.beta = g.beta; d.C = g.C; d.ldc = g.ldc;
  d.cycles = g.cycles;
  d.slice_bits = g.slice_bits;
  d.group_m = pick_group_m(ctx->dbg_flags, kGroupM);
  d.wave_ctr = nullptr;
  d.n_waves = 0;
  d.serp = EMU_PROBE_FLAG(ctx->dbg_flags, 128) ? 0 : 1;
  d.dbg = ctx->dbg_flags;
  constexpr bool CL2 = PAIR || MC;
  const int64_t tiles = static_cast<int64_t>(d.mt) * d.nt_tiles * d.nch * batch;
  if (tiles >= (1LL << 31)) return EMUGEMM_ERR_ARG;
  const int workers = CL2 ? ctx->num_sms / 2 : ctx->num_sms;
  const int grid = (CL2 ? 2 : 1) * static_cast<int>(tiles < workers ? tiles : workers);
  void (*kern)(CUtensorMap, CUtensorMap, Oz1Dev) = nullptr;
  switch (g.out_kind) {
    case 0: kern = oz1_gemm_kernel<P, 0, PAIR, MC>; break;
    case 1: kern = oz1_gemm_kernel<(P <= 4 ? P : 4), 1, PAIR, MC>; break;  // FP32 entry point: p <= 4 (checked by the API)
    case 2: kern = oz1_gemm_kernel<P, 2, PAIR, MC>; break;
    default: kern = oz1_gemm_kernel<P, 3, PAIR, MC>; break;
  }
  if (g.out_kind == 1 && P > 4) return EMUGEMM_ERR_ARG;
  EMU_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::kSmemBytes));
#ifdef EMUGEMM_PROBES
  // probe 0x20000000: give the L2 a persisting carve-out (with 0x200000 = A EVICT_LAST) -- does the hint need one?
  if (ctx->dbg_flags & 0x20000000) {
    int maxp = 0, dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&maxp, cudaDevAttrMaxPersistingL2CacheSize, dev);
    size_t want = static_cast<size_t>(80) << 20;
    if (want > static_cast<size_t>(maxp)) want = static_cast<size_t>(maxp);
    cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, want);
    static bool said = false;
    if (!said) { printf("emugemm probe: persisting L2 max %d bytes, set %zu\n", maxp, want); said = true; }
  }
#endif
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(static_cast<unsigned>(grid));
  cfg.blockDim = dim3(kGemmThreads);
  cfg.dynamicSmemBytes = Cfg::kSmemBytes;
  cfg.stream = ctx->stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = CL2 ? 2 : 1;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  // Wave barrier: only when every CTA is certainly co-resident (grid <= the clusters the device can hold at once), there
  // are at least two waves, and the panels are long: measured (A/B, profiles/r2_wave_barrier.md) +18-19 % at 16384^3
  // (p = 8, FP32 p = 4: the SM clock goes 1.16 -> 1.40 GHz), +1-3 % at 8192^3 p = 8, -0.3 ... -1.9 % at 8192^3 p <= 7 and at
  // 4096^3 (the re-alignment costs ~1 % of the tensor pipe per clock), so it is on for >= 64 KB of slices per operand row
  // or k >= 16384.  Probes build: flag 0x10000 switches it off, 0x40000 forces it on.
  const int workers_used = grid / (CL2 ? 2 : 1);
  const bool long_panels = static_cast<int64_t>(d.chunk_kb) * kBlockK * P >= 65536 || static_cast<int64_t>(d.chunk_kb) * kBlockK >= 16384;
  if (g.wave_ctr && tiles > workers_used && d.chunk_kb >= 16 && (long_panels || EMU_PROBE_FLAG(ctx->dbg_flags, 0x40000)) &&
      !EMU_PROBE_FLAG(ctx->dbg_flags, 0x10000)) {
    int max_clusters = 0;
    if (cudaOccupancyMaxActiveClusters(&max_clusters, kern, &cfg) == cudaSuccess && max_clusters >= workers_used) {
      d.wave_ctr = g.wave_ctr;
      d.n_waves = static_cast<int>((tiles + workers_used - 1) / workers_used);
    }
  }
  // plain launch: the barrier's wait is bounded and gives up (ptx.cuh), so CTAs that are not co-resident after all (a
  // second handle launching on another stream, a profiler) cost time, never progress
  EMU_CUDA(ctx, cudaLaunchKernelEx(&cfg, kern, tmA, tmB, d));
  ctx->launches++;
  EMU_CUDA(ctx, cudaGetLastError());
  return EMUGEMM_OK;
}

template <int P>
static int launch_p(emugemm_ctx *ctx, const Oz1GemmArgs &g) {
  if constexpr (P <= 3) {
    if (!EMU_PROBE_FLAG(ctx->dbg_flags, 8)) return launch_pp<P, true, false>(ctx, g);  // dbg bit 3: force the one-CTA N-concatenated kernel (A/B timing)
  }
  // A multicast: +2-4 % at p = 8 (NT = 64, A dominates the operand traffic), +2 % at p = 4, within noise at p = 5, 6
  if (P >= 4 && !EMU_PROBE_FLAG(ctx->dbg_flags, 16)) return launch_pp<P, false, true>(ctx, g);  // dbg bit 4: no multicast clusters (A/B timing)
  return launch_pp<P, false, false>(ctx, g);
}

int launch_oz1_gemm(emugemm_ctx *ctx, const Oz1GemmArgs &g) {
  if (g.m == 0 || g.n == 0 || g.k1 <= g.k0) return EMUGEMM_OK;
  switch (g.p) {
    case 1: return launch_p<1>(ctx, g);
    case 2: return launch_p<2>(ctx, g);
    case 3: return launch_p<3>(ctx, g);
    case 4: return launch_p<4>(ctx, g);
    case 5: return launch_p<5>(ctx, g);
    case 6: return launch_p<6>(ctx, g);
    case 7: return launch_p<7>(ctx, g);
    case 8: return launch_p<8>(ctx, g);
    default: return EMUGEMM_ERR_ARG;
  }
}

// Overflow-safe k-chunk (R7): the fullest accumulator C_{p-1} sums p products of k_c
// terms each bounded by 127^2, so p k_c 127^2 <= 2^31 - 1; rounded down to a multiple of 128.
int64_t oz1_chunk_k_host(int p, int slice_bits) {
  if (slice_bits == kDigitsTwos) {
    // R24: leading digit in [-128, 127], the others in [0, 127]; the fullest accumulator C_(p-1) sums the pairs (0, p-1),
    // (p-1, 0) with |d d'| <= 128 * 127 and p - 2 pairs <= 127^2 (p = 1: one pair <= 128^2)
    const int64_t per_k = p == 1 ? 128 * 128 : 2 * 128 * 127 + static_cast<int64_t>(p - 2) * 127 * 127;
    return (2147483647LL / per_k) / kBlockK * kBlockK;
  }
  const int64_t dmax = (slice_bits == 8) ? 128 : 127;  // largest digit magnitude
  const int64_t bound = 2147483647LL / (static_cast<int64_t>(p) * dmax * dmax);
  return bound / kBlockK * kBlockK;
}

int64_t oz1_cluster_tiles_host(int p, int64_t m, int64_t n) {
  auto cdiv = [](int64_t a, int64_t b) { return (a + b - 1) / b; };
  switch (p) {  // the NT table of Oz1Cfg; p <= 3: 256-row pair tiles, p >= 4: two N-adjacent 128-row tiles per cluster
    case 1: case 2: return cdiv(m, 2 * kTileM) * cdiv(n, Oz1Cfg<2, true>::NT);
    case 3: return cdiv(m, 2 * kTileM) * cdiv(n, Oz1Cfg<3, true>::NT);
    case 4: return cdiv(m, kTileM) * cdiv(cdiv(n, Oz1Cfg<4>::NT), 2);
    case 5: return cdiv(m, kTileM) * cdiv(cdiv(n, Oz1Cfg<5>::NT), 2);
    case 6: return cdiv(m, kTileM) * cdiv(cdiv(n, Oz1Cfg<6>::NT), 2);
    default: return cdiv(m, kTileM) * cdiv(cdiv(n, Oz1Cfg<8>::NT), 2);  // p = 7, 8: NT = 64
  }
}

// ---- k-chunk reduction: C = alpha * sum_c (hi_c + lo_c) + beta C, double-double sum ----
__global__ void __launch_bounds__(256) oz1_chunk_reduce_kernel(int64_t m, int64_t n, int n_chunks,
                                                               const double *__restrict__ part, int out_kind,
                                                               double alpha, double beta, void *C, int64_t ldc) {
  const int64_t idx = static_cast<int64_t>(blockIdx.x) * 256 + threadIdx.x;
  if (idx >= m * n) return;
  const int64_t i = idx / n, j = idx - i * n;
  double hi = 0.0, lo = 0.0;
  for (int c = 0; c < n_chunks; ++c) {
    const double2 v = *reinterpret_cast<const double2 *>(part + (static_cast<int64_t>(c) * m * n + idx) * 2);
    const double sum = hi + v.x;
    const double bb = sum - hi;
    lo += (hi - (sum - bb)) + (v.x - bb) + v.y;
    hi = sum;
  }
  const double s = hi + lo;
  if (out_kind == 0) {
    double *o = static_cast<double *>(C) + i * ldc + j;
    *o = (beta != 0.0) ? fma(alpha, s, beta * *o) : alpha * s;
  } else {
    float *o = static_cast<float *>(C) + i * ldc + j;
    double x = alpha * s;
    if (beta != 0.0) x = fma(beta, static_cast<double>(*o), x);
    *o = static_cast<float>(x);
  }
}

int launch_oz1_chunk_reduce(emugemm_ctx *ctx, int64_t m, int64_t n, int n_chunks, const double *part,
                            int out_kind, double alpha, double beta, void *C, int64_t ldc) {
  if (m * n == 0) return EMUGEMM_OK;
  const unsigned grid = static_cast<unsigned>((m * n + 255) / 256);
  oz1_chunk_reduce_kernel<<<grid, 256, 0, ctx->stream>>>(m, n, n_chunks, part, out_kind, alpha, beta, C, ldc);
  ctx->launches++;
  EMU_CUDA(ctx, cudaGetLastError());
  return EMUGEMM_OK;
}

#ifdef EMUGEMM_PROBES
// Same products, ONE MMA per product (width NT): A_t stays in the collector across its P - t consecutive MMAs.
// This is the schedule a cta_group::2 pair needs (an N-concatenated MMA would split its columns between the
// two CTAs' B halves); probed with cta_group::1: MMAs narrower than ~112 columns hit a ~55-cycle
// per-instruction floor (p = 8, NT = 64: 0.56 of peak), so it only pays for NT >= 128.
template <int P, bool COLL>
__device__ __forceinline__ void oz1_issue_slice_per_product(int t, uint32_t tmem_base, uint32_t a_base, uint32_t b_base,
                                                            bool accumulate) {
  constexpr int NT = Oz1Cfg<P>::NT;
  constexpr uint32_t idesc = make_idesc_i8(kTileM, NT);
  const uint32_t a_lo = sdesc_lo(a_base), b_lo = sdesc_lo(b_base);
#pragma unroll
  for (int ks = 0; ks < kBlockK / 32; ++ks) {
    const uint64_t adesc = sdesc_from_lo(a_lo + ((ks * 32) >> 4));
#pragma unroll
    for (int u = 0; u < P; ++u) {
      if (u < P - t) {
        const uint32_t acc = (accumulate || ks != 0) ? 1u : 0u;
        const uint32_t d = tmem_base + (t + u) * NT;
        const uint64_t bdesc = sdesc_from_lo(b_lo + ((u * NT * kBlockK + ks * 32) >> 4));
        const bool first = (u == 0), last = (u == P - t - 1);
        if (COLL && first && !last) umma_i8<1>(d, adesc, bdesc, idesc, acc);
        else if (COLL && !first && last) umma_i8<3>(d, adesc, bdesc, idesc, acc);
        else if (COLL && !first && !last) umma_i8<2>(d, adesc, bdesc, idesc, acc);
        else umma_i8<0>(d, adesc, bdesc, idesc, acc);
      }
    }
  }
}

// ---- issue-bound INT8 tensor-core probe (third denominator) ----
// One CTA per SM; operands are whatever bytes sit in shared memory; no loads in the loop.  The host passes a
// schedule of up to 64 MMAs (TMEM column, width N, A slot, B row offset); one "iteration" issues the whole
// schedule once, the k32 sub-block rotating with the iteration like the real kernels.
// cycles_out[0] = SM cycles block 0 spent between the first issue and the completion of the last MMA.
struct ProbeSched {
  int n_ops;
  uint16_t col[64], n[64], aslot[64], brow[64], coll[64];
};
__global__ void __launch_bounds__(128, 1) i8_probe_kernel(const ProbeSched sc, int iters, long long *cycles_out) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  __shared__ uint64_t bar;
  __shared__ uint32_t slot;
  // pseudo-random operand bytes: the multiplier arrays toggle like on real slices (power-realistic)
  for (int i = threadIdx.x; i < (8 * 16384 + 65536) / 4; i += 128) {
    uint32_t x = static_cast<uint32_t>(i) * 2654435761u + blockIdx.x * 40503u;
    x ^= x >> 15; x *= 2246822519u; x ^= x >> 13;
    reinterpret_cast<uint32_t *>(smem)[i] = x;
  }
  if (threadIdx.x == 0) { mbar_init(&bar, 1); fence_mbar_init(); }
  fence_proxy_async_smem();
  if (threadIdx.x < 32) { tmem_alloc(&slot, 512); tmem_relinquish(); }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tb = slot;
  if (threadIdx.x == 0) {
    const uint32_t abase = smem_u32(smem), bbase = smem_u32(smem + 8 * 16384);
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
      const int ks = it & 3;
      for (int o = 0; o < sc.n_ops; ++o) {
        const uint32_t d = tb + sc.col[o], idesc = make_idesc_i8(128, sc.n[o]);
        const uint64_t ad = make_sdesc_sw128(abase + sc.aslot[o] * 16384 + ks * 32);
        const uint64_t bd = make_sdesc_sw128(bbase + sc.brow[o] * kBlockK + ks * 32);
        switch (sc.coll[o]) {
          case 1: umma_i8<1>(d, ad, bd, idesc, it > 0); break;
          case 2: umma_i8<2>(d, ad, bd, idesc, it > 0); break;
          case 3: umma_i8<3>(d, ad, bd, idesc, it > 0); break;
          default: umma_i8<0>(d, ad, bd, idesc, it > 0); break;
        }
      }
    }
    umma_commit(&bar);
    mbar_wait(&bar, 0);
    if (blockIdx.x == 0 && cycles_out) *cycles_out = clock64() - t0;
  }
  tc_fence_before();
  __syncthreads();
  if (threadIdx.x < 32) tmem_dealloc(tb, 512);
}

int launch_i8_probe(emugemm_ctx *ctx, int n_ops, const int *ops, int iters, float *ms, int *ctas, long long *cycles) {
  if (iters < 1 || n_ops < 1 || n_ops > 64 || !ops) return EMUGEMM_ERR_ARG;
  ProbeSched sc;
  sc.n_ops = n_ops;
  for (int o = 0; o < n_ops; ++o) {
    const int col = ops[5 * o], n = ops[5 * o + 1], as = ops[5 * o + 2], br = ops[5 * o + 3], cl = ops[5 * o + 4];
    if (n < 16 || n > 256 || n % 16 || col < 0 || col + n > 512 || as < 0 || as > 7 || br < 0 || br + n > 512 || cl < 0 || cl > 3) return EMUGEMM_ERR_ARG;
    sc.col[o] = col; sc.n[o] = n; sc.aslot[o] = as; sc.brow[o] = br; sc.coll[o] = cl;
  }
  if (!ctx->ws || ctx->ws_bytes < 8) return EMUGEMM_ERR_WORKSPACE;
  const int smem = 8 * 16384 + 65536 + 1024;
  EMU_CUDA(ctx, cudaFuncSetAttribute(i8_probe_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  cudaEvent_t e0, e1;
  EMU_CUDA(ctx, cudaEventCreate(&e0));
  EMU_CUDA(ctx, cudaEventCreate(&e1));
  long long *dcyc = static_cast<long long *>(ctx->ws);
  i8_probe_kernel<<<ctx->num_sms, 128, smem, ctx->stream>>>(sc, iters / 8 + 1, nullptr);  // warm-up
  EMU_CUDA(ctx, cudaEventRecord(e0, ctx->stream));
  i8_probe_kernel<<<ctx->num_sms, 128, smem, ctx->stream>>>(sc, iters, dcyc);
  EMU_CUDA(ctx, cudaEventRecord(e1, ctx->stream));
  EMU_CUDA(ctx, cudaEventSynchronize(e1));
  EMU_CUDA(ctx, cudaEventElapsedTime(ms, e0, e1));
  if (cycles) EMU_CUDA(ctx, cudaMemcpy(cycles, dcyc, sizeof(long long), cudaMemcpyDeviceToHost));
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  *ctas = ctx->num_sms;
  ctx->launches += 2;
  return EMUGEMM_OK;
}

// ---- compiled-schedule probe: the exact MMA issue code of the fused kernel on SMEM-resident operands ----
template <int P, bool COLL, bool PERPROD>
__global__ void __launch_bounds__(128, 1) oz1_issue_probe_kernel(int iters, long long *cycles_out) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  __shared__ uint64_t bar;
  __shared__ uint32_t slot;
  for (int i = threadIdx.x; i < (8 * 16384 + 65536) / 4; i += 128) {
    uint32_t x = static_cast<uint32_t>(i) * 2654435761u + blockIdx.x * 40503u;
    x ^= x >> 15; x *= 2246822519u; x ^= x >> 13;
    reinterpret_cast<uint32_t *>(smem)[i] = x;
  }
  if (threadIdx.x == 0) { mbar_init(&bar, 1); fence_mbar_init(); }
  fence_proxy_async_smem();
  if (threadIdx.x < 32) { tmem_alloc(&slot, 512); tmem_relinquish(); }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tb = slot;
  if (threadIdx.x == 0) {
    const uint32_t abase = smem_u32(smem), bbase = smem_u32(smem + 8 * 16384);
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int t = 0; t < P; ++t) {
        if (PERPROD) oz1_issue_slice_per_product<P, COLL>(t, tb, abase + t * 16384, bbase, it > 0 || t > 0);
        else oz1_issue_slice<P, COLL>(t, tb, abase + t * 16384, bbase, it > 0 || t > 0);
      }
    }
    umma_commit(&bar);
    mbar_wait(&bar, 0);
    if (blockIdx.x == 0 && cycles_out) *cycles_out = clock64() - t0;
  }
  tc_fence_before();
  __syncthreads();
  if (threadIdx.x < 32) tmem_dealloc(tb, 512);
}

template <int P>
static int issue_probe_p(emugemm_ctx *ctx, int coll, int iters, float *ms, long long *cycles) {
  const int smem = 8 * 16384 + 65536 + 1024;
  auto kern = (coll & 2) ? ((coll & 1) ? oz1_issue_probe_kernel<P, true, true> : oz1_issue_probe_kernel<P, false, true>)
                         : ((coll & 1) ? oz1_issue_probe_kernel<P, true, false> : oz1_issue_probe_kernel<P, false, false>);
  EMU_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  cudaEvent_t e0, e1;
  EMU_CUDA(ctx, cudaEventCreate(&e0));
  EMU_CUDA(ctx, cudaEventCreate(&e1));
  long long *dcyc = static_cast<long long *>(ctx->ws);
  kern<<<ctx->num_sms, 128, smem, ctx->stream>>>(iters / 8 + 1, nullptr);
  EMU_CUDA(ctx, cudaEventRecord(e0, ctx->stream));
  kern<<<ctx->num_sms, 128, smem, ctx->stream>>>(iters, dcyc);
  EMU_CUDA(ctx, cudaEventRecord(e1, ctx->stream));
  EMU_CUDA(ctx, cudaEventSynchronize(e1));
  EMU_CUDA(ctx, cudaEventElapsedTime(ms, e0, e1));
  if (cycles) EMU_CUDA(ctx, cudaMemcpy(cycles, dcyc, sizeof(long long), cudaMemcpyDeviceToHost));
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  ctx->launches += 2;
  return EMUGEMM_OK;
}

int launch_oz1_issue_probe(emugemm_ctx *ctx, int p, int coll, int iters, float *ms, int *ctas, long long *cycles) {
  if (iters < 1 || p < 1 || p > 8) return EMUGEMM_ERR_ARG;
  if (!ctx->ws || ctx->ws_bytes < 8) return EMUGEMM_ERR_WORKSPACE;
  *ctas = ctx->num_sms;
  switch (p) {
    case 1: return issue_probe_p<1>(ctx, coll, iters, ms, cycles);
    case 2: return issue_probe_p<2>(ctx, coll, iters, ms, cycles);
    case 3: return issue_probe_p<3>(ctx, coll, iters, ms, cycles);
    case 4: return issue_probe_p<4>(ctx, coll, iters, ms, cycles);
    case 5: return issue_probe_p<5>(ctx, coll, iters, ms, cycles);
    case 6: return issue_probe_p<6>(ctx, coll, iters, ms, cycles);
    case 7: return issue_probe_p<7>(ctx, coll, iters, ms, cycles);
    default: return issue_probe_p<8>(ctx, coll, iters, ms, cycles);
  }
}

#endif  // EMUGEMM_PROBES

}  // namespace emu
