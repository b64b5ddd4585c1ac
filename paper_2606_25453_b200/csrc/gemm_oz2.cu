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
// (modulus, pair tile, product)).  A CTA PAIR (cluster of 2, tcgen05 cta_group::2)
// owns a 256 x 256 output tile: each CTA loads its own 128 rows of A and its own
// 128 of the 256 B rows per 128-byte k-block (32 KB per stage and CTA instead of
// 48 KB), the leader CTA issues one 256 x 256 x 32 MMA per k32 for both SMs, and
// each CTA's tensor core reads only half of B from its shared memory.  6-stage
// TMA ring; TMEM holds two 256-column INT32 accumulators per CTA so the
// mod-epilogue of one item overlaps the MMAs of the next (the paper reuses one
// accumulator and overlaps only with TMA prefetch).
//
// Fused variant (template parameter FNP > 0, real DGEMM only): a work item is an OUTPUT tile
// and the moduli are the inner loop; the residues of the pair's tile go to a private scratch of 2 x N x 32 KB per CTA
// (two buffers, alternating by tile; the [N][m][n] planes are never written), and the epilogue warps run the exact FP64
// CRT of crt_dev.cuh on their own rows of the PREVIOUS tile, 8 columns after every modulus epilogue of the current one,
// and write C: the reconstruction hides under the tensor-core work of the next tile.  DESIGN.md 5.7 has the measurements.
#include "common.cuh"
#include "ptx.cuh"
#include "gemm_common.cuh"
#include "crt_dev.cuh"

namespace emu {

constexpr int kOz2NT = 256;                   // tile columns
constexpr int kOz2PairM = 2 * kTileM;         // tile rows of a CTA pair
constexpr int kOz2KPerStage = 2;              // 128-byte k-blocks per ring stage: 8 MMAs per barrier wait / commit
constexpr int kOz2Stages = 3;
constexpr int kOz2BStage = (kOz2NT / 2) * kBlockK;  // 16 KB: this CTA's half of the B rows
constexpr int kOz2KbBytes = kAStageBytes + kOz2BStage;         // one k-block: A 16 KB + this CTA's B half 16 KB
constexpr int kOz2StageBytes = kOz2KPerStage * kOz2KbBytes;
constexpr int kOz2Smem = kOz2Stages * kOz2StageBytes + 1024 + 256;

struct Oz2Dev {
  int64_t m, n;
  int kblocks;  // k-blocks of this launch, starting at k-block kb0 of the planes
  int kb0;
  int mt, nt_tiles, n_moduli;
  int nbatch;  // strided batched call: entry b uses plane rows [b m, (b+1) m) / [b n, (b+1) n) and CR[l][b]
  int8_t *CR;
  unsigned long long *cycles;
  int group_m;  // rasterisation group (tile_coords)
  int serp;     // serpentine k (see gemm_oz1.cu)
  unsigned long long *wave_ctr;  // wave barrier (see gemm_oz1.cu), null: none
  int n_waves;
  int dbg;
  int mod[kMaxModuli];
  unsigned cvec[kMaxModuli];    // bytes (256^j mod m), j = 0..3 (byte 0 = 256^0)
  unsigned c0[kMaxModuli];      // (m - 2^31 mod m) mod m
  unsigned magic[kMaxModuli];   // ceil(2^32 / m)
};

// Symmetric residue of a signed INT32 accumulator modulo m <= 256 in 6 integer instructions, no branch:
//   u = x + 2^31 (flip the sign bit), s = sum_j byte_j(u) (256^j mod m) + c0  ==  x (mod m), 0 <= s < 2^18
//   q = floor(s M / 2^32), M = ceil(2^32 / m): exact because s (M m - 2^32) / (m 2^32) < 2^18 / 2^32 < 1/m
//   r = s - q m in [0, m), then r -= m if r >= ceil(m/2)  (R11, R13).  m = 256 reduces to the low byte.
struct ModK {
  unsigned cvec, c0, magic, m, half;
};
__device__ __forceinline__ unsigned dot_mod(uint32_t x, const ModK &k) {  // == x (mod m), in [0, 2^18)
  return __dp4a(x ^ 0x80000000u, k.cvec, k.c0);
}
__device__ __forceinline__ unsigned reduce_mod(unsigned s, const ModK &k) {  // s < 2^24 -> [0, m)
  return s - __umulhi(s, k.magic) * k.m;
}
__device__ __forceinline__ int to_sym(unsigned r, const ModK &k) {  // [0, m) -> [ceil(m/2) - m, ceil(m/2) - 1]
  return static_cast<int>(r) - (r >= k.half ? static_cast<int>(k.m) : 0);
}
__device__ __forceinline__ int sym_mod_i32(uint32_t x, const ModK &k) { return to_sym(reduce_mod(dot_mod(x, k), k), k); }
// low bytes of a, b, c, d -> one word (3 PRMT)
__device__ __forceinline__ unsigned pack4i(unsigned a, unsigned b, unsigned c, unsigned d) {
  return __byte_perm(__byte_perm(a, b, 0x0040), __byte_perm(c, d, 0x0040), 0x5410);
}
__device__ __forceinline__ unsigned byte_u(unsigned w, int i) { return __byte_perm(w, 0u, 0x4440u | static_cast<unsigned>(i)); }

// 32 packed residues (8 words) of one row -> global, two 16-byte stores = one full 32-byte sector
__device__ __forceinline__ void store32(int8_t *dst, const unsigned (&w)[8], int64_t gcol, int64_t n, bool vec_ok) {
  if (vec_ok && gcol + 32 <= n) {
    reinterpret_cast<uint4 *>(dst)[0] = make_uint4(w[0], w[1], w[2], w[3]);
    reinterpret_cast<uint4 *>(dst)[1] = make_uint4(w[4], w[5], w[6], w[7]);
  } else {
#pragma unroll
    for (int c = 0; c < 32; ++c)
      if (gcol + c < n) dst[c] = static_cast<int8_t>((w[c >> 2] >> (8 * (c & 3))) & 0xFFu);
  }
}

// reconstruction arguments of the fused variant (unused when FNP == 0)
struct Oz2Fuse {
  CrtConst k;
  const int32_t *eA, *eB;
  int tsum;            // tA + tB
  double alpha, beta;
  double *C;
  int64_t ldc;
  int64_t batch_stride_c;  // elements between the C matrices of consecutive batch entries
};
constexpr int kOz2ScratchPlane = kTileM * kOz2NT;  // 32 KB: one modulus of one CTA's 128 x 256 half tile

// NPROD: 1 real (Eq. 6-7), 3: 3M (Eq. 16-18).  FNP: 0 = residue planes to global memory (CRT in crt.cu); > 0 = fused
// reconstruction with FNP = ceil(N / 2) modulus pairs (NPROD == 1 only).
template <int NPROD, int FNP>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kGemmThreads, 1)
oz2_gemm_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const Oz2Dev a,
                const __grid_constant__ Oz2Fuse f) {
  constexpr bool FUSED = FNP > 0;
  static_assert(!FUSED || NPROD == 1, "the fused reconstruction covers the real product");
  extern __shared__ uint8_t smem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint64_t *bars = reinterpret_cast<uint64_t *>(smem + kOz2Stages * kOz2StageBytes);
  uint64_t *full = bars, *empty = bars + kOz2Stages, *tfull = bars + 2 * kOz2Stages, *tempty = tfull + 2;
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(tempty + 2);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t cta = cluster_ctarank();  // 0 = leader (issues the MMAs), 1 = peer
  const int cluster_id = blockIdx.x >> 1, num_clusters = gridDim.x >> 1;
  const int tiles_per_mod = a.mt * a.nt_tiles;  // a.mt counts PAIR tiles of 256 rows
  // unfused: tile = (batch entry, modulus, tile of the modulus), NPROD products each; fused: tile = (batch entry, output tile),
  // the N moduli are the inner loop
  const int tiles_per_entry = FUSED ? tiles_per_mod : tiles_per_mod * a.n_moduli;
  const int num_tiles = tiles_per_entry * a.nbatch;
  const int n_inner = FUSED ? a.n_moduli : NPROD;

  if (threadIdx.x == 0) {
    // full[s] (leader's is the one used): 1 arrival (leader's expect_tx) + the bytes of BOTH CTAs' loads;
    // empty[s], tfull[b]: 1 arrival from the leader's multicast commit; tempty[b] (leader's): all epilogue warps of the pair
    for (int i = 0; i < kOz2Stages; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&tfull[i], 1); mbar_init(&tempty[i], 2 * kEpiWarps); }
    fence_mbar_init();
    tma_prefetch_desc(&tmA);
    tma_prefetch_desc(&tmB);
  }
  if (warp == 1) {
    tmem_alloc_cg2(tmem_slot, 512);
    tmem_relinquish_cg2();
  }
  tc_fence_before();
  cluster_sync_all();  // the peer's barriers must be initialised before remote arrivals / remote complete_tx
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const long long t_start = clock64();

  if (warp == 0) {
    // ===================== TMA producer (one per CTA: own A rows, own half of the B rows) =====================
    if (lane == 0) {
      int st = 0;
      uint32_t ph = 0;
      int wave = 0;
      bool wave_off = false;  // a barrier wait ran into its bound: no more waiting in this launch (arrivals continue)
      for (int tile = cluster_id; tile < num_tiles; tile += num_clusters, ++wave) {
        // re-align the producers of all CTAs at every tile (see gemm_oz1.cu): the pairs that share an A or a B panel then ask
        // for the same k-block of the same product at the same time, and it comes from DRAM once
        if (a.wave_ctr && wave > 0 && !wave_off) wave_off = !grid_wait(a.wave_ctr, static_cast<unsigned long long>(wave) * gridDim.x);
        const int bidx = tile / tiles_per_entry, te = tile - bidx * tiles_per_entry;
        const int l = FUSED ? 0 : te / tiles_per_mod;
        int mb, nb;
        tile_coords(te - l * tiles_per_mod, a.mt, a.nt_tiles, mb, nb, a.group_m);
        const int arow = static_cast<int>(bidx * a.m) + mb * kOz2PairM + static_cast<int>(cta) * kTileM;
        const int brow = static_cast<int>(bidx * a.n) + nb * kOz2NT + static_cast<int>(cta) * (kOz2NT / 2);
        // exact integer accumulation: odd tiles of this pair walk k downwards (serpentine), so the k-blocks its L2
        // neighbourhood touched last are the first ones asked for again
        const bool rev = a.serp && (((tile - cluster_id) / num_clusters) & 1);
        const int nstage = (a.kblocks + kOz2KPerStage - 1) / kOz2KPerStage;
        // the arrival on the wave barrier is signalled a few stages before the last load of the tile (see gemm_oz1.cu)
        constexpr int kWaveLead = 6;
        const int arrive_sidx = nstage - 1 - kWaveLead > 0 ? nstage - 1 - kWaveLead : 0;
        for (int q = 0; q < n_inner; ++q) {
          const int plane = FUSED ? q : q * a.n_moduli + l;
          for (int sidx = 0; sidx < nstage; ++sidx) {
            const int kb = (rev ? nstage - 1 - sidx : sidx) * kOz2KPerStage;
            const int nkb = (a.kblocks - kb < kOz2KPerStage) ? a.kblocks - kb : kOz2KPerStage;
            if (a.wave_ctr && q == n_inner - 1 && sidx == arrive_sidx) grid_arrive(a.wave_ctr);
            mbar_wait(&empty[st], ph ^ 1);
            const uint32_t full_leader = mapa_u32(&full[st], 0);
            if (cta == 0) mbar_arrive_expect_tx(&full[st], 2 * nkb * kOz2KbBytes);
            for (int i = 0; i < nkb; ++i) {
              uint8_t *dst = smem + st * kOz2StageBytes + i * kOz2KbBytes;
              tma_load_3d_cg2(dst, &tmA, full_leader, (a.kb0 + kb + i) * kBlockK, arow, plane);
              tma_load_3d_cg2(dst + kAStageBytes, &tmB, full_leader, (a.kb0 + kb + i) * kBlockK, brow, plane);
            }
            if (++st == kOz2Stages) { st = 0; ph ^= 1; }
          }
        }
      }
      if (a.wave_ctr)
        for (; wave < a.n_waves; ++wave) grid_arrive(a.wave_ctr);
    }
    __syncwarp();
  } else if (warp == 1) {
    // ===================== MMA issuer (leader CTA only) =====================
    if (lane == 0 && cta == 0) {
      int st = 0;
      uint32_t ph = 0;
      uint32_t item = 0;
      constexpr uint32_t idesc = make_idesc_i8(kOz2PairM, kOz2NT);
      bool ready = false;  // look-ahead probe of the next stage's barrier (see gemm_oz1.cu)
      const int nstage = (a.kblocks + kOz2KPerStage - 1) / kOz2KPerStage;
      for (int tile = cluster_id; tile < num_tiles; tile += num_clusters) {
        const bool rev = a.serp && (((tile - cluster_id) / num_clusters) & 1);  // the producer's k direction for this tile
        for (int q = 0; q < n_inner; ++q, ++item) {
          const uint32_t slot = item & 1, tph = (item >> 1) & 1;
          mbar_wait(&tempty[slot], tph ^ 1);
          tc_fence_after();
          for (int sidx = 0; sidx < nstage; ++sidx) {
            const int kb = (rev ? nstage - 1 - sidx : sidx) * kOz2KPerStage;  // only the (possibly short) last stage differs
            const int nkb = (a.kblocks - kb < kOz2KPerStage) ? a.kblocks - kb : kOz2KPerStage;
            if (!ready) mbar_wait(&full[st], ph);
            tc_fence_after();
            const uint32_t s_base = smem_u32(smem + st * kOz2StageBytes);
            const int st_cur = st;
            if (++st == kOz2Stages) { st = 0; ph ^= 1; }
            ready = mbar_try_wait(&full[st], ph);
#pragma unroll
            for (int i = 0; i < kOz2KPerStage; ++i) {
              if (i < nkb) {
                const uint32_t a_base = s_base + i * kOz2KbBytes, b_base = a_base + kAStageBytes;
#pragma unroll
                for (int ks = 0; ks < kBlockK / 32; ++ks)
                  umma_i8_cg2(tmem_base + slot * kOz2NT, make_sdesc_sw128(a_base + ks * 32), make_sdesc_sw128(b_base + ks * 32),
                              idesc, (sidx | i | ks) ? 1u : 0u);
              }
            }
            umma_commit_cg2(&empty[st_cur], 3);  // both CTAs' producers may refill the stage
          }
          umma_commit_cg2(&tfull[slot], 3);      // both CTAs' epilogues may drain their 128 rows
        }
      }
    }
    __syncwarp();
  } else {
    const int ew = warp - 2, quad = warp & 3, half = ew >> 2;
    const int row = quad * 32 + lane;
    const uint32_t trow = tmem_base + (static_cast<uint32_t>(quad * 32) << 16);
    const bool vec_ok = (a.n % 16 == 0) && ((reinterpret_cast<uintptr_t>(a.CR) & 15) == 0);
    const int64_t plane_sz = a.m * a.n * a.nbatch;
    uint32_t item = 0;
    unsigned t1[NPROD == 3 ? 32 : 1], t2[NPROD == 3 ? 32 : 1];  // T1, T2 of this thread's 128 columns as packed INT8 (3M)
    const uint32_t tempty_leader[2] = {mapa_u32(&tempty[0], 0), mapa_u32(&tempty[1], 0)};
    // fused: the reconstruction of the PREVIOUS tile (its residues sit in the other scratch buffer) is spread over the N
    // modulus epilogues of the current tile, 8 columns per step, so that it never delays the release of an accumulator
    // by more than one step (a whole-tile burst of ~200k clk after the last modulus stalled the tensor pipe: 5.9 -> 7.9 ms)
    struct PrevTile { int8_t *scratch; int64_t grow, gcol0; int bidx; bool row_ok; } prev = {nullptr, 0, 0, 0, false};
    int crt_done = 16;  // 8-column steps of the previous tile already reconstructed (16 = nothing pending)
    int tile_ord = 0;
    auto crt_step = [&](const int ch) {
      if constexpr (FUSED) {
        constexpr int J = (FNP + 1) / 2;
        const int64_t gcol = prev.gcol0 + ch * 8;
        if (!prev.row_ok || gcol >= a.n || EMU_PROBE_FLAG(a.dbg, 0x80000)) return;
        uint2 w[2 * FNP];
#pragma unroll
        for (int l = 0; l < 2 * FNP; ++l) {
          w[l] = make_uint2(0u, 0u);
          if ((l < 2 * FNP - 1 || l < a.n_moduli) && !EMU_PROBE_FLAG(a.dbg, 0x100000))
            w[l] = *reinterpret_cast<const uint2 *>(prev.scratch + static_cast<int64_t>(l) * kOz2ScratchPlane + ch * 8);
        }
        const int eAi = __ldg(f.eA + prev.bidx * a.m + prev.grow) - f.tsum - kCrtSC;
        const int32_t *eBp = f.eB + prev.bidx * a.n;
        double *crow = f.C + prev.bidx * f.batch_stride_c + prev.grow * f.ldc;
        const bool vec_c = (f.ldc % 4 == 0) && ((reinterpret_cast<uintptr_t>(f.C) & 31) == 0) && ((f.batch_stride_c & 3) == 0);
#pragma unroll
        for (int g = 0; g < 2; ++g) {
          double acc[4][J], v[4];
#pragma unroll
          for (int pq = 0; pq < FNP; ++pq)
            crt_accumulate_pair<J>(f.k, pq, g == 0 ? w[2 * pq].x : w[2 * pq].y, g == 0 ? w[2 * pq + 1].x : w[2 * pq + 1].y, acc, pq == 0);
          const int64_t c0 = gcol + 4 * g;
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const int eb = (c0 + e < a.n) ? __ldg(eBp + c0 + e) : 0;
            v[e] = crt_scale_pow2(crt_finish<J>(f.k, acc[e]), eAi + eb);
          }
          double *o = crow + c0;
          if (f.beta != 0.0) {
#pragma unroll
            for (int e = 0; e < 4; ++e)
              if (c0 + e < a.n) v[e] = fma(f.alpha, v[e], f.beta * o[e]);
          } else if (f.alpha != 1.0) {
#pragma unroll
            for (int e = 0; e < 4; ++e) v[e] *= f.alpha;
          }
          if (vec_c && c0 + 4 <= a.n) {
            asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(o), "d"(v[0]), "d"(v[1]), "d"(v[2]), "d"(v[3]) : "memory");
          } else {
#pragma unroll
            for (int e = 0; e < 4; ++e)
              if (c0 + e < a.n) o[e] = v[e];
          }
        }
      }
    };
    for (int tile = cluster_id; tile < num_tiles; tile += num_clusters, ++tile_ord) {
      const int bidx = tile / tiles_per_entry, te = tile - bidx * tiles_per_entry;
      const int l0 = FUSED ? 0 : te / tiles_per_mod;
      int mb, nb;
      tile_coords(te - l0 * tiles_per_mod, a.mt, a.nt_tiles, mb, nb, a.group_m);
      const int64_t grow = static_cast<int64_t>(mb) * kOz2PairM + cta * kTileM + row;
      const bool row_ok = grow < a.m;
      // fused: this thread's 128 residues of modulus q go to [q][row][half * 128 ...] of the CTA's scratch buffer (tile_ord & 1)
      int8_t *scratch = FUSED ? a.CR + ((static_cast<int64_t>(blockIdx.x) * 2 + (tile_ord & 1)) * a.n_moduli) * kOz2ScratchPlane +
                                    row * kOz2NT + half * 128
                              : nullptr;
      auto drain = [&](const int q) {  // the epilogue of one accumulator: product q (unfused) or modulus q (fused)
        const int l = FUSED ? q : l0;
        ModK mk;
        mk.cvec = a.cvec[l]; mk.c0 = a.c0[l]; mk.magic = a.magic[l]; mk.m = static_cast<unsigned>(a.mod[l]); mk.half = (mk.m + 1) / 2;
        const uint32_t slot = item & 1, tph = (item >> 1) & 1;
        mbar_wait(&tfull[slot], tph);
        tc_fence_after();
        if (!EMU_PROBE_FLAG(a.dbg, 2)) {
          // 4 chunks of 32 columns, TMEM loads of chunk i+1 in flight while chunk i is reduced
          uint32_t va[32], vb[32];
          const uint32_t tcol = trow + slot * kOz2NT + half * 128;
          tmem_ld32(tcol, va);
#pragma unroll
          for (int ch = 0; ch < 4; ++ch) {
            uint32_t(&v)[32] = (ch & 1) ? vb : va;
            uint32_t(&vn)[32] = (ch & 1) ? va : vb;
            tmem_ld_wait();
            if (ch + 1 < 4) tmem_ld32(tcol + (ch + 1) * 32, vn);
            const int64_t gcol = static_cast<int64_t>(nb) * kOz2NT + half * 128 + ch * 32;
            if constexpr (NPROD == 1) {
              unsigned w[8];
#pragma unroll
              for (int g = 0; g < 8; ++g)
                w[g] = pack4i(sym_mod_i32(v[4 * g], mk), sym_mod_i32(v[4 * g + 1], mk), sym_mod_i32(v[4 * g + 2], mk),
                              sym_mod_i32(v[4 * g + 3], mk));
              if constexpr (FUSED) {
                uint4 *dst = reinterpret_cast<uint4 *>(scratch + static_cast<int64_t>(q) * kOz2ScratchPlane + ch * 32);
                dst[0] = make_uint4(w[0], w[1], w[2], w[3]);
                dst[1] = make_uint4(w[4], w[5], w[6], w[7]);
              } else if (row_ok && gcol < a.n && !EMU_PROBE_FLAG(a.dbg, 4)) {
                store32(a.CR + ((static_cast<int64_t>(l) * a.nbatch + bidx) * a.m + grow) * a.n + gcol, w, gcol, a.n, vec_ok);
              }
            } else if (q < 2) {
              // T1 / T2 stay on chip as unsigned residues in [0, m), four per register
#pragma unroll
              for (int g = 0; g < 8; ++g) {
                const unsigned w = pack4i(reduce_mod(dot_mod(v[4 * g], mk), mk), reduce_mod(dot_mod(v[4 * g + 1], mk), mk),
                                          reduce_mod(dot_mod(v[4 * g + 2], mk), mk), reduce_mod(dot_mod(v[4 * g + 3], mk), mk));
                if (q == 0) t1[ch * 8 + g] = w; else t2[ch * 8 + g] = w;
              }
            } else {
              // c_re = sym(T1 - T2), c_im = sym(T3 - T1 - T2) (Eq. 16): all in residues, one reduction for the
              // imaginary part (T3's byte dot product + 2m - r1 - r2 < 2^19), two compares for the real part
              unsigned wr[8], wi[8];
#pragma unroll
              for (int g = 0; g < 8; ++g) {
                unsigned re[4], im[4];
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                  const unsigned r1 = byte_u(t1[ch * 8 + g], b), r2 = byte_u(t2[ch * 8 + g], b);
                  int d = static_cast<int>(r1) - static_cast<int>(r2);            // (-m, m)
                  d -= (d >= static_cast<int>(mk.half)) ? static_cast<int>(mk.m) : 0;
                  d += (d < static_cast<int>(mk.half) - static_cast<int>(mk.m)) ? static_cast<int>(mk.m) : 0;
                  re[b] = static_cast<unsigned>(d);
                  const unsigned vi = dot_mod(v[4 * g + b], mk) + 2u * mk.m - r1 - r2;  // >= 0, == T3 - T1 - T2 (mod m)
                  im[b] = static_cast<unsigned>(to_sym(reduce_mod(vi, mk), mk));
                }
                wr[g] = pack4i(re[0], re[1], re[2], re[3]);
                wi[g] = pack4i(im[0], im[1], im[2], im[3]);
              }
              if (row_ok && gcol < a.n && !EMU_PROBE_FLAG(a.dbg, 4)) {
                int8_t *o = a.CR + ((static_cast<int64_t>(l) * a.nbatch + bidx) * a.m + grow) * a.n + gcol;
                store32(o, wr, gcol, a.n, vec_ok);
                store32(o + a.n_moduli * plane_sz, wi, gcol, a.n, vec_ok);
              }
            }
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_remote(tempty_leader[slot]);  // the leader's MMA thread waits for both CTAs
        ++item;
        if constexpr (FUSED) {  // the previous tile's share of reconstruction steps for this modulus
          while (crt_done < 16 && crt_done * a.n_moduli < 16 * (q + 1)) crt_step(crt_done++);
        }
      };
      if constexpr (FUSED) {
#pragma unroll 1
        for (int q = 0; q < n_inner; ++q) drain(q);
      } else {
#pragma unroll
        for (int q = 0; q < NPROD; ++q) drain(q);
      }
      if constexpr (FUSED) {
        while (crt_done < 16) crt_step(crt_done++);  // (only if N > 16 steps could not be placed: never for N <= 20)
        prev.scratch = scratch; prev.grow = grow; prev.gcol0 = static_cast<int64_t>(nb) * kOz2NT + half * 128; prev.bidx = bidx;
        prev.row_ok = row_ok;
        crt_done = 0;
      }
    }
    if constexpr (FUSED) {
      while (crt_done < 16) crt_step(crt_done++);  // the last tile of this CTA
    }
  }

  tc_fence_before();
  cluster_sync_all();  // neither CTA may free TMEM / exit while the pair's MMAs or remote arrivals are in flight
  if (warp == 1) tmem_dealloc_cg2(tmem_base, 512);
  if (blockIdx.x == 0 && threadIdx.x == 0 && a.cycles) atomicAdd(a.cycles, static_cast<unsigned long long>(clock64() - t_start));
}

int launch_oz2_gemm(emugemm_ctx *ctx, const Oz2GemmArgs &g) {
  if (g.m == 0 || g.n == 0 || g.kpad == 0) return EMUGEMM_OK;
  const int parts = g.is3m ? 3 : 1;
  CUtensorMap tmA, tmB;
  const int batch = g.batch > 0 ? g.batch : 1;
  EMU_TRY(encode_planes_tmap(ctx, &tmA, g.RA, g.kpad, g.m * batch, static_cast<int64_t>(parts) * g.n_moduli, kTileM, 1));
  EMU_TRY(encode_planes_tmap(ctx, &tmB, g.RB, g.kpad, g.n * batch, static_cast<int64_t>(parts) * g.n_moduli, kOz2NT / 2, 1));
  Oz2Dev d;
  d.m = g.m; d.n = g.n;
  const int64_t k0 = g.k1 > 0 ? g.k0 : 0, k1 = g.k1 > 0 ? g.k1 : g.kpad;
  if (k0 < 0 || k1 > g.kpad || k0 >= k1 || (k0 % kBlockK) || (k1 % kBlockK) || k1 - k0 > kOz2MaxChunkK) return EMUGEMM_ERR_ARG;
  d.kb0 = static_cast<int>(k0 / kBlockK);
  d.kblocks = static_cast<int>((k1 - k0) / kBlockK);
  d.mt = static_cast<int>((g.m + kOz2PairM - 1) / kOz2PairM);  // pair tiles
  d.nt_tiles = static_cast<int>((g.n + kOz2NT - 1) / kOz2NT);
  d.n_moduli = g.n_moduli;
  d.nbatch = batch;
  d.CR = g.CR;
  d.cycles = g.cycles;
  d.group_m = pick_group_m(ctx->dbg_flags, kGroupM);
  d.serp = EMU_PROBE_FLAG(ctx->dbg_flags, 128) ? 0 : 1;
  d.dbg = ctx->dbg_flags;
  int mod[24];
  oz2_moduli_host(g.n_moduli, mod);
  for (int l = 0; l < kMaxModuli; ++l) {
    const unsigned m = static_cast<unsigned>(l < g.n_moduli ? mod[l] : 256);
    d.mod[l] = static_cast<int>(m);
    unsigned pw[4], r = 1u % m;
    for (int j = 0; j < 4; ++j) { pw[j] = r; r = (r * 256u) % m; }
    d.cvec[l] = pw[0] | (pw[1] << 8) | (pw[2] << 16) | (pw[3] << 24);
    const unsigned two31 = static_cast<unsigned>((1ull << 31) % m);
    d.c0[l] = (m - two31) % m;
    d.magic[l] = static_cast<unsigned>(((1ull << 32) + m - 1ull) / m);
  }
  const bool fused = g.fused != nullptr;
  if (fused && g.is3m) return EMUGEMM_ERR_ARG;
  // work items of the persistent loop: (entry, modulus, tile) or, fused, (entry, output tile) with the moduli inside
  const int64_t tiles = static_cast<int64_t>(d.mt) * d.nt_tiles * (fused ? 1 : d.n_moduli) * batch;
  if (tiles >= (1LL << 31)) return EMUGEMM_ERR_ARG;
  const int pairs = ctx->num_sms / 2;
  const int grid = 2 * (tiles < pairs ? static_cast<int>(tiles) : pairs);
  Oz2Fuse fz = {};
  void (*kern)(CUtensorMap, CUtensorMap, Oz2Dev, Oz2Fuse) = g.is3m ? oz2_gemm_kernel<3, 0> : oz2_gemm_kernel<1, 0>;
  if (fused) {
    const Oz2CrtArgs &c = *g.fused;
    if (!crt_constants_host(g.n_moduli, fz.k) || fz.k.J != (fz.k.NP + 1) / 2) return EMUGEMM_ERR_ARG;
    fz.eA = c.eA; fz.eB = c.eB; fz.tsum = c.tA + c.tB; fz.alpha = c.alpha[0]; fz.beta = c.beta[0];
    fz.C = c.C; fz.ldc = c.ldc; fz.batch_stride_c = c.batch_stride_c;
    switch (fz.k.NP) {  // the BASELINE range N = 12 ... 20 and the FP32-level N = 8 ... 11
      case 4: kern = oz2_gemm_kernel<1, 4>; break;
      case 5: kern = oz2_gemm_kernel<1, 5>; break;
      case 6: kern = oz2_gemm_kernel<1, 6>; break;
      case 7: kern = oz2_gemm_kernel<1, 7>; break;
      case 8: kern = oz2_gemm_kernel<1, 8>; break;
      case 9: kern = oz2_gemm_kernel<1, 9>; break;
      case 10: kern = oz2_gemm_kernel<1, 10>; break;
      default: return EMUGEMM_ERR_ARG;
    }
    if (static_cast<size_t>(grid) * 2 * g.n_moduli * kOz2ScratchPlane > g.scratch_bytes) return EMUGEMM_ERR_WORKSPACE;  // two buffers per CTA
  }
  EMU_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kOz2Smem));
  // Wave barrier (gemm_oz1.cu): only when all CTAs are co-resident by the occupancy query, there are at least two waves
  // and the k-loop is long enough (>= 64 k-blocks per product, >= 16 for the fused variant whose tile is N products long)
  // for the early arrival (kWaveLead stages before the item's last load) to hide the re-alignment.
  // Measured A/B on two boxes (profiles/r2_wave_barrier.md), barrier on / off:
  //   3M 8192^3 N = 18    19.6 / 20.9 and 19.8 / 21.2 ms (DRAM reads 50.5 -> 31.3 GB)          -> on
  //   3M 8192^3 N = 14    14.8 / 16.3 and 15.7 / 14.9 ms (within the box-to-box spread)         -> on (same rule as N = 18)
  //   real 16384^3 N = 15 43.9 / 49.9 and 45.9 / 50.5 ms (a modulus' planes, 2 x 268 MB, exceed the L2) -> on from k = 16,384
  //   real 8192^3 N = 16  5.76 / 6.12 and 5.86 / 5.74 ms: a modulus' planes (2 x 67 MB) fit the L2, the DRAM reads do not
  //                       change (5.57 / 5.53 GB) and the barrier costs 2.7 % per clock (an item is one modulus, 23 us) -> off
  // Probes build: 0x20000 forces it on for the real product at shorter k, 0x10000 switches it off everywhere.
  d.wave_ctr = nullptr;
  d.n_waves = 0;
  const bool want_sync = !EMU_PROBE_FLAG(ctx->dbg_flags, 0x10000) &&
                         (g.is3m || fused || d.kblocks >= 128 || EMU_PROBE_FLAG(ctx->dbg_flags, 0x20000));
  if (g.wave_ctr && want_sync && tiles > grid / 2 && d.kblocks >= (fused ? 16 : 64)) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(static_cast<unsigned>(grid));
    cfg.blockDim = dim3(kGemmThreads);
    cfg.dynamicSmemBytes = kOz2Smem;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    int max_clusters = 0;
    if (cudaOccupancyMaxActiveClusters(&max_clusters, kern, &cfg) == cudaSuccess && max_clusters >= grid / 2) {
      d.wave_ctr = g.wave_ctr;
      d.n_waves = static_cast<int>((tiles + grid / 2 - 1) / (grid / 2));
    }
  }
  // plain launch: a barrier wait that runs into its bound gives up (ptx.cuh), so co-residency is an optimisation only
  kern<<<grid, kGemmThreads, kOz2Smem, ctx->stream>>>(tmA, tmB, d, fz);
  ctx->launches++;
  EMU_CUDA(ctx, cudaGetLastError());
  return EMUGEMM_OK;
}

// ---- Scheme II k-chunking: output residues of k-chunks add modulo m_l ---------------------------------------
struct Oz2AddMod {
  int mod[kMaxModuli];
};
__global__ void __launch_bounds__(256) oz2_residue_add_kernel(int8_t *__restrict__ CR, const int8_t *__restrict__ T, int n_moduli,
                                                              int64_t plane_elems, const __grid_constant__ Oz2AddMod mk) {
  const int plane = blockIdx.y;
  const int m = mk.mod[plane % n_moduli], half = (m + 1) / 2;
  int8_t *c = CR + static_cast<int64_t>(plane) * plane_elems;
  const int8_t *t = T + static_cast<int64_t>(plane) * plane_elems;
  for (int64_t i = static_cast<int64_t>(blockIdx.x) * 256 + threadIdx.x; i < plane_elems; i += static_cast<int64_t>(gridDim.x) * 256) {
    int s = static_cast<int>(c[i]) + static_cast<int>(t[i]);  // both symmetric residues: |s| <= m
    s += (s < 0) ? m : 0;                                     // [0, m]
    s -= (s >= m) ? m : 0;                                    // [0, m)
    s -= (s >= half) ? m : 0;                                 // [ceil(m/2) - m, ceil(m/2) - 1]  (R11, R13)
    c[i] = static_cast<int8_t>(s);
  }
}

int launch_oz2_residue_add(emugemm_ctx *ctx, int8_t *CR, const int8_t *T, int n_moduli, int planes, int64_t plane_elems) {
  if (planes <= 0 || plane_elems <= 0) return EMUGEMM_OK;
  Oz2AddMod mk;
  int mod[24];
  oz2_moduli_host(n_moduli, mod);
  for (int l = 0; l < kMaxModuli; ++l) mk.mod[l] = l < n_moduli ? mod[l] : 256;
  int64_t gx = (plane_elems + 255) / 256;
  if (gx > 4096) gx = 4096;
  oz2_residue_add_kernel<<<dim3(static_cast<unsigned>(gx), static_cast<unsigned>(planes)), 256, 0, ctx->stream>>>(CR, T, n_moduli, plane_elems, mk);
  ctx->launches++;
  EMU_CUDA(ctx, cudaGetLastError());
  return EMUGEMM_OK;
}

}  // namespace emu
