// gemm_oz2.cu -- Ozaki Scheme II per-modulus INT8 GEMM with the modular
// reduction fused into the epilogue.
//
// What it computes (Eq. 6-7): for every modulus m_l,
//   C'_l = sym( A'_l B'_l , m_l )  written as INT8; the INT32 product never
// reaches global memory (Eq. 15).  3M (PAPER.md:244-262,
// Eq. 16-18): per modulus T1 = re.re, T2 = im.im, T3 = Sigma.Sigma, each reduced
// mod m_l; T1 and T2 stay in registers as INT8 while T3 is computed, then
// c_re = sym(T1 - T2), c_im = sym(T3 - T1 - T2) are the only two tiles written.
//
// B200-first design: ONE persistent launch covers all moduli (work item =
// (modulus, tile, product)); 128 x 256 tiles, 4-stage TMA ring of 128-byte
// k-blocks, TMEM holds two 256-column INT32 accumulators so the mod-epilogue of
// one item overlaps the MMAs of the next (the paper reuses one accumulator and
// overlaps only with TMA prefetch).
#include "common.cuh"
#include "ptx.cuh"
#include "gemm_common.cuh"

namespace emu {

constexpr int kOz2NT = 256;
constexpr int kOz2Stages = 4;
constexpr int kOz2BStage = kOz2NT * kBlockK;  // 32 KB
constexpr int kOz2StageBytes = kAStageBytes + kOz2BStage;
constexpr int kOz2Smem = kOz2Stages * kOz2StageBytes + 1024 + 256;

struct Oz2Dev {
  int64_t m, n;
  int kblocks;
  int mt, nt_tiles, n_moduli;
  int nprod;              // 1 real, 3 for 3M
  int8_t *CR;
  unsigned long long *cycles;
  int mod[kMaxModuli];
  unsigned magic[kMaxModuli];  // ceil(2^39 / m)
};

// symmetric residue of a signed INT32 accumulator (|x| < 2^31) modulo m (odd m, 151 <= m <= 255) or 256.
// u = |x| < 2^31; q = floor(u magic / 2^39) with magic = ceil(2^39/m) < 2^32 is exact because the error
// term u (magic - 2^39/m) / 2^39 < 2^31 / 2^39 = 2^-8 <= 1/m.
__device__ __forceinline__ int sym_mod_i32(int x, int m, unsigned magic) {
  if (m == 256) return static_cast<int>(static_cast<int8_t>(x & 0xFF));  // two's complement low byte
  const unsigned u = static_cast<unsigned>(x < 0 ? -x : x);
  const unsigned q = __umulhi(u, magic) >> 7;
  int r = static_cast<int>(u - q * static_cast<unsigned>(m));  // [0, m)
  if (r >= (m + 1) / 2) r -= m;                                // symmetric, odd m: sym(-u) = -sym(u)
  return x < 0 ? -r : r;
}
__device__ __forceinline__ int sym_small_rt(int t, int m) {  // t in (-2m, 2m) -> symmetric range (R15)
  const int hi = (m + 1) / 2;
  if (t >= hi) t -= m;
  if (t >= hi) t -= m;
  if (t < hi - m) t += m;
  if (t < hi - m) t += m;
  return t;
}
__device__ __forceinline__ unsigned pack4i(int a, int b, int c, int d) {
  return (static_cast<unsigned>(a) & 0xFFu) | ((static_cast<unsigned>(b) & 0xFFu) << 8) |
         ((static_cast<unsigned>(c) & 0xFFu) << 16) | ((static_cast<unsigned>(d) & 0xFFu) << 24);
}
__device__ __forceinline__ int unpack_i8(unsigned w, int i) {
  return static_cast<int>(static_cast<int8_t>((w >> (8 * i)) & 0xFFu));
}

__device__ __forceinline__ void store16(int8_t *dst, const unsigned (&w)[4], int64_t gcol, int64_t n, bool vec_ok) {
  if (vec_ok && gcol + 16 <= n) {
    *reinterpret_cast<uint4 *>(dst) = make_uint4(w[0], w[1], w[2], w[3]);
  } else {
#pragma unroll
    for (int c = 0; c < 16; ++c)
      if (gcol + c < n) dst[c] = static_cast<int8_t>((w[c >> 2] >> (8 * (c & 3))) & 0xFFu);
  }
}

__global__ void __launch_bounds__(kGemmThreads, 1)
oz2_gemm_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const Oz2Dev a) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint64_t *bars = reinterpret_cast<uint64_t *>(smem + kOz2Stages * kOz2StageBytes);
  uint64_t *full = bars, *empty = bars + kOz2Stages, *tfull = bars + 2 * kOz2Stages, *tempty = tfull + 2;
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(tempty + 2);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int tiles_per_mod = a.mt * a.nt_tiles;
  const int num_tiles = tiles_per_mod * a.n_moduli;

  if (threadIdx.x == 0) {
    for (int i = 0; i < kOz2Stages; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&tfull[i], 1); mbar_init(&tempty[i], kEpiWarps); }
    fence_mbar_init();
    tma_prefetch_desc(&tmA);
    tma_prefetch_desc(&tmB);
  }
  if (warp == 1) {
    tmem_alloc(tmem_slot, 512);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const long long t_start = clock64();

  if (warp == 0) {
    if (lane == 0) {
      int st = 0;
      uint32_t ph = 0;
      for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
        const int l = tile / tiles_per_mod;
        int mb, nb;
        tile_coords(tile - l * tiles_per_mod, a.mt, a.nt_tiles, mb, nb);
        for (int q = 0; q < a.nprod; ++q) {
          const int plane = q * a.n_moduli + l;
          for (int kb = 0; kb < a.kblocks; ++kb) {
            mbar_wait(&empty[st], ph ^ 1);
            mbar_arrive_expect_tx(&full[st], kOz2StageBytes);
            uint8_t *dst = smem + st * kOz2StageBytes;
            tma_load_3d(dst, &tmA, &full[st], kb * kBlockK, mb * kTileM, plane);
            tma_load_3d(dst + kAStageBytes, &tmB, &full[st], kb * kBlockK, nb * kOz2NT, plane);
            if (++st == kOz2Stages) { st = 0; ph ^= 1; }
          }
        }
      }
    }
    __syncwarp();
  } else if (warp == 1) {
    if (lane == 0) {
      int st = 0;
      uint32_t ph = 0;
      uint32_t item = 0;
      constexpr uint32_t idesc = make_idesc_i8(kTileM, kOz2NT);
      for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
        for (int q = 0; q < a.nprod; ++q, ++item) {
          const uint32_t slot = item & 1, tph = (item >> 1) & 1;
          mbar_wait(&tempty[slot], tph ^ 1);
          tc_fence_after();
          for (int kb = 0; kb < a.kblocks; ++kb) {
            mbar_wait(&full[st], ph);
            tc_fence_after();
            const uint32_t a_base = smem_u32(smem + st * kOz2StageBytes), b_base = a_base + kAStageBytes;
#pragma unroll
            for (int ks = 0; ks < kBlockK / 32; ++ks)
              umma_i8(tmem_base + slot * kOz2NT, make_sdesc_sw128(a_base + ks * 32), make_sdesc_sw128(b_base + ks * 32),
                      idesc, (kb | ks) ? 1u : 0u);
            umma_commit(&empty[st]);
            if (++st == kOz2Stages) { st = 0; ph ^= 1; }
          }
          umma_commit(&tfull[slot]);
        }
      }
    }
    __syncwarp();
  } else {
    const int ew = warp - 2, quad = warp & 3, half = ew >> 2;
    const int row = quad * 32 + lane;
    const uint32_t trow = tmem_base + (static_cast<uint32_t>(quad * 32) << 16);
    const bool vec_ok = (a.n % 16 == 0) && ((reinterpret_cast<uintptr_t>(a.CR) & 15) == 0);
    const int64_t plane_sz = a.m * a.n;
    uint32_t item = 0;
    unsigned t1[32], t2[32];  // T1, T2 of this thread's 128 columns as packed INT8 (3M only)
    for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
      const int l = tile / tiles_per_mod;
      int mb, nb;
      tile_coords(tile - l * tiles_per_mod, a.mt, a.nt_tiles, mb, nb);
      const int mod = a.mod[l];
      const unsigned magic = a.magic[l];
      const int64_t grow = static_cast<int64_t>(mb) * kTileM + row;
      const bool row_ok = grow < a.m;
      for (int q = 0; q < a.nprod; ++q, ++item) {
        const uint32_t slot = item & 1, tph = (item >> 1) & 1;
        mbar_wait(&tfull[slot], tph);
        tc_fence_after();
#pragma unroll
        for (int ch = 0; ch < 8; ++ch) {
          const int c0 = half * 128 + ch * 16;
          uint32_t v[16];
          tmem_ld16(trow + slot * kOz2NT + c0, v);
          tmem_ld_wait();
          unsigned w[4];
#pragma unroll
          for (int g = 0; g < 4; ++g)
            w[g] = pack4i(sym_mod_i32(static_cast<int>(v[4 * g]), mod, magic), sym_mod_i32(static_cast<int>(v[4 * g + 1]), mod, magic),
                          sym_mod_i32(static_cast<int>(v[4 * g + 2]), mod, magic), sym_mod_i32(static_cast<int>(v[4 * g + 3]), mod, magic));
          const int64_t gcol = static_cast<int64_t>(nb) * kOz2NT + c0;
          if (a.nprod == 1) {
            if (row_ok && gcol < a.n)
              store16(a.CR + (static_cast<int64_t>(l) * a.m + grow) * a.n + gcol, w, gcol, a.n, vec_ok);
          } else if (q == 0) {
#pragma unroll
            for (int g = 0; g < 4; ++g) t1[ch * 4 + g] = w[g];
          } else if (q == 1) {
#pragma unroll
            for (int g = 0; g < 4; ++g) t2[ch * 4 + g] = w[g];
          } else {
            unsigned wr[4], wi[4];
#pragma unroll
            for (int g = 0; g < 4; ++g) {
              int re[4], im[4];
#pragma unroll
              for (int b = 0; b < 4; ++b) {
                const int x1 = unpack_i8(t1[ch * 4 + g], b), x2 = unpack_i8(t2[ch * 4 + g], b), x3 = unpack_i8(w[g], b);
                re[b] = sym_small_rt(x1 - x2, mod);
                im[b] = sym_small_rt(x3 - x1 - x2, mod);
              }
              wr[g] = pack4i(re[0], re[1], re[2], re[3]);
              wi[g] = pack4i(im[0], im[1], im[2], im[3]);
            }
            if (row_ok && gcol < a.n) {
              int8_t *o = a.CR + (static_cast<int64_t>(l) * a.m + grow) * a.n + gcol;
              store16(o, wr, gcol, a.n, vec_ok);
              store16(o + a.n_moduli * plane_sz, wi, gcol, a.n, vec_ok);
            }
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&tempty[slot]);
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem_base, 512);
  if (blockIdx.x == 0 && threadIdx.x == 0 && a.cycles) atomicAdd(a.cycles, static_cast<unsigned long long>(clock64() - t_start));
}

int launch_oz2_gemm(emugemm_ctx *ctx, const Oz2GemmArgs &g) {
  if (g.m == 0 || g.n == 0 || g.kpad == 0) return EMUGEMM_OK;
  const int parts = g.is3m ? 3 : 1;
  CUtensorMap tmA, tmB;
  EMU_TRY(encode_planes_tmap(ctx, &tmA, g.RA, g.kpad, g.m, static_cast<int64_t>(parts) * g.n_moduli, kTileM, 1));
  EMU_TRY(encode_planes_tmap(ctx, &tmB, g.RB, g.kpad, g.n, static_cast<int64_t>(parts) * g.n_moduli, kOz2NT, 1));
  Oz2Dev d;
  d.m = g.m; d.n = g.n;
  d.kblocks = static_cast<int>(g.kpad / kBlockK);
  d.mt = static_cast<int>((g.m + kTileM - 1) / kTileM);
  d.nt_tiles = static_cast<int>((g.n + kOz2NT - 1) / kOz2NT);
  d.n_moduli = g.n_moduli;
  d.nprod = parts;
  d.CR = g.CR;
  d.cycles = g.cycles;
  int mod[24];
  oz2_moduli_host(g.n_moduli, mod);
  for (int l = 0; l < kMaxModuli; ++l) {
    d.mod[l] = l < g.n_moduli ? mod[l] : 256;
    d.magic[l] = static_cast<unsigned>(((1ull << 39) + static_cast<unsigned long long>(d.mod[l]) - 1ull) /
                                       static_cast<unsigned long long>(d.mod[l]));
  }
  const int64_t tiles = static_cast<int64_t>(d.mt) * d.nt_tiles * d.n_moduli;
  const int grid = tiles < ctx->num_sms ? static_cast<int>(tiles) : ctx->num_sms;
  EMU_CUDA(ctx, cudaFuncSetAttribute(oz2_gemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kOz2Smem));
  oz2_gemm_kernel<<<grid, kGemmThreads, kOz2Smem, ctx->stream>>>(tmA, tmB, d);
  ctx->launches++;
  EMU_CUDA(ctx, cudaGetLastError());
  return EMUGEMM_OK;
}

}  // namespace emu
