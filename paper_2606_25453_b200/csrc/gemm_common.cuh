// gemm_common.cuh -- constants and the tile rasterisation shared by the fused GEMM kernels.
#pragma once
#include "common.cuh"

namespace emu {

constexpr int kEpiWarps = 8;                       // epilogue warps (two per TMEM lane quadrant)
constexpr int kGemmThreads = 64 + kEpiWarps * 32;  // warp 0 TMA, warp 1 MMA, warps 2.. epilogue
constexpr int kAStageBytes = kTileM * kBlockK;     // 16 KB: 128 rows x 128 B of k
constexpr int kSmemLimit = 232448;                 // 227 KB per CTA on sm_100
constexpr int kGroupM = 8;                         // default rasterisation: groups of 8 m-blocks, n-blocks fastest across a group

// tile -> (m-block, n-block): consecutive tiles (= concurrently resident CTAs) cover group_m m-blocks x
// ~workers/group_m n-blocks, so each A row-panel and each B panel is shared by several CTAs through L2.
__device__ __forceinline__ void tile_coords(int tile, int mt, int nt, int &mb, int &nb, int group_m = kGroupM) {
  const int per_group = group_m * nt;
  const int g = tile / per_group;
  const int first = g * group_m;
  const int gsz = (mt - first < group_m) ? (mt - first) : group_m;
  const int r = tile - g * per_group;
  mb = first + r % gsz;
  nb = r / gsz;
}

// Host side: rasterisation group for the fused kernels.  Probes build: bits 8-15 of the experiment flags override it.
inline int pick_group_m(int dbg_flags, int dflt) {
  const int o = EMU_PROBE_FLAG(dbg_flags, 0xFF00) >> 8;
  return o > 0 ? o : dflt;
}

}  // namespace emu
