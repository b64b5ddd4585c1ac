// gemm_common.cuh -- constants and the tile rasterisation shared by the fused GEMM kernels.
#pragma once
#include "common.cuh"

namespace emu {

constexpr int kEpiWarps = 8;                       // epilogue warps (two per TMEM lane quadrant)
constexpr int kGemmThreads = 64 + kEpiWarps * 32;  // warp 0 TMA, warp 1 MMA, warps 2.. epilogue
constexpr int kAStageBytes = kTileM * kBlockK;     // 16 KB: 128 rows x 128 B of k
constexpr int kSmemLimit = 232448;                 // 227 KB per CTA on sm_100
constexpr int kGroupM = 8;                         // rasterisation: groups of 8 m-blocks, n-blocks fastest across a group

// tile -> (m-block, n-block): consecutive tiles (= concurrently resident CTAs) cover kGroupM m-blocks x
// ~num_sms/kGroupM n-blocks, so each A row-panel is shared by ~18 CTAs and each B panel by 8 through L2.
__device__ __forceinline__ void tile_coords(int tile, int mt, int nt, int &mb, int &nb) {
  const int per_group = kGroupM * nt;
  const int g = tile / per_group;
  const int first = g * kGroupM;
  const int gsz = (mt - first < kGroupM) ? (mt - first) : kGroupM;
  const int r = tile - g * per_group;
  mb = first + r % gsz;
  nb = r / gsz;
}

}  // namespace emu
