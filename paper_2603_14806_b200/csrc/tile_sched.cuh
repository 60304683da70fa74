// Dynamic, in-order tile scheduling for the persistent kernels (K2 and K1).
//
// With a static assignment (CTA pair g takes tiles g, g + G, g + 2G, ...) nothing keeps the pairs
// in step: small speed differences between SMs accumulate over the ~440 tiles of a pair, the set
// of tiles in flight spreads over many channels / row blocks, and the sharing of operand blocks
// through L2 collapses (measured at N = 4096: 41-58 GB instead of 9 GB of DRAM reads per launch).
// Handing the tiles out in index order from one global counter -- as the hardware block scheduler
// would, but to persistent CTAs -- keeps the window of tiles in flight compact.  Every tile is
// computed the same way whichever pair gets it, so results stay bitwise reproducible.
//
// The counter is launch-private: one 32-bit word in caller-owned device memory (workspace tail /
// stage scratch), zeroed on the caller's stream ahead of the launch (api.cu arm_sched_words).
// K1's tiles share nothing, but its a / b stores are 128-byte rows 32 MB apart: adjacent tiles fill
// the same DRAM pages only if they are written at about the same time, and the in-order scheduler
// (TileRing below) made K1 13-15 % faster.  K3 keeps the static assignment: the same scheduler
// measured no gain there (its stores are contiguous 32 KB blocks).
#pragma once

#include "ptx.cuh"

namespace foldcp {

// Single-CTA flavour: one thread draws tile indices and publishes them in a ring in shared memory;
// every other role waits on the entry's "full" mbarrier, reads it and releases it on "empty".
template <int kDepth>
struct TileRing {
  uint32_t base;   // shared address: kDepth full barriers, kDepth empty barriers, kDepth slots
  static constexpr int kBytes = kDepth * 20;
  __device__ __forceinline__ uint32_t full(int s) const { return base + 8u * s; }
  __device__ __forceinline__ uint32_t empty(int s) const { return base + 8u * (kDepth + s); }
  __device__ __forceinline__ uint32_t slot(int s) const { return base + 16u * kDepth + 4u * s; }
  __device__ __forceinline__ void init(uint32_t consumers) const {
    for (int s = 0; s < kDepth; ++s) {
      ptx::mbar_init(full(s), 1);
      ptx::mbar_init(empty(s), consumers);
    }
  }
  __device__ __forceinline__ int produce(int i, unsigned int* sched, int num_tiles) const {
    const int s = i % kDepth;
    ptx::mbar_wait(empty(s), ((i / kDepth) & 1) ^ 1u);
    const unsigned int drawn = atomicAdd(sched, 1u);
    const int tile = drawn < static_cast<unsigned int>(num_tiles) ? static_cast<int>(drawn) : -1;
    ptx::sts32(slot(s), static_cast<uint32_t>(tile));
    ptx::mbar_arrive(full(s));
    return tile;
  }
  __device__ __forceinline__ int consume(int i) const {
    const int s = i % kDepth;
    ptx::mbar_wait(full(s), (i / kDepth) & 1);
    const int tile = static_cast<int>(ptx::lds32(slot(s)));
    ptx::mbar_arrive(empty(s));
    return tile;
  }
  __device__ __forceinline__ int consume_warp(int i, int lane) const {
    int tile = 0;
    if (lane == 0) tile = consume(i);
    return __shfl_sync(0xffffffffu, tile, 0);
  }
};

}  // namespace foldcp
