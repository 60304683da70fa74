// K2 -- the triangle contraction (Eq. 2-3):
//
//   outgoing  o[c][i][j] = sum_k a[c][i][k] * b[c][j][k]      O_c = A_c  B_c^T   (operands K-major)
//   incoming  o[c][i][j] = sum_k a[c][k][i] * b[c][k][j]      O_c = A_c^T B_c    (operands MN-major)
//
// a, b, o are channel-major 16-bit [c][N][N]; c independent N x N x N GEMMs with fp32 accumulation.
// a and b are fp16 on the forward path and bf16 in the gradient GEMMs (K2Params::ab_fmt, a field of
// the instruction descriptor); o / the gradients are written as bf16.
// "The outgoing and incoming variants differ only in which operand is transposed" (PAPER.md line
// 132): here that is literally one bit per operand in the tcgen05 instruction descriptor plus the
// TMA box coordinates -- the data is never moved.
//
// Kernel shape (persistent, warp-specialised, one CTA per SM, optionally CTA pairs):
//   warp 0      TMA producer   : 64x64 bf16 boxes (128-byte swizzle) -> smem ring of kStages
//   warp 1      MMA issuer     : one elected thread, tcgen05.mma kind::f16, D in tensor memory
//   warp 2      TMEM allocator : 512 columns = two 128 x 256 fp32 accumulators (double buffer)
//   warps 4-7   epilogue       : tcgen05.ld -> bf16 -> swizzled smem -> TMA store, overlapped
//                                with the next tile's main loop through the second accumulator
// kCtaGroup = 2 pairs two SMs on one 256 x 256 tile (cta_group::2): each CTA stages its own 128
// rows of A and 128 of the 256 B rows, halving per-SM shared-memory operand traffic.
// The two operand majors are independent template parameters (kAMn, kBMn): the forward uses
// (K, K) and (MN, MN), the gradients of the contraction also the mixed (K, MN) form.
// Tiles are not assigned statically: the leader's producer thread draws them in index order from
// a global counter (tile_sched.cuh) and publishes them to the other roles through a small ring.
#include <type_traits>

#include "common.h"
#include "ptx.cuh"
#include "tile_sched.cuh"

namespace foldcp {
namespace {

constexpr int kBlockK = 64;        // k elements per pipeline stage (= one 128-byte swizzle row)
constexpr int kBoxBytes = 64 * 64 * 2;  // one TMA box: 64 x 64 bf16
constexpr int kTileN = 256;
constexpr int kUmmaK = 16;
constexpr int kThreads = 256;
constexpr int kEpiBufBytes = 128 * 64 * 2;  // 128 rows x 64 bf16 columns
constexpr int kAccumCols = 256;

template <int kCtaGroup>
struct Cfg {
  static constexpr int kTileM = 128 * kCtaGroup;
  static constexpr int kABytes = 2 * kBoxBytes;                  // 128 x 64 per CTA
  static constexpr int kBBoxes = (kTileN / kCtaGroup) / 64;      // 4 or 2
  static constexpr int kBBytes = kBBoxes * kBoxBytes;
  static constexpr int kStageBytes = kABytes + kBBytes;          // 48 KB or 32 KB
  static constexpr int kStages = kCtaGroup == 1 ? 4 : 6;
  static constexpr int kEpiBytes = 2 * kEpiBufBytes;
  static constexpr int kBarBytes = 1024;
  static constexpr int kSmemBytes = kStages * kStageBytes + kEpiBytes + kBarBytes + 1024;
};

#ifdef FOLDCP_K2_PROBE
// bring-up instrumentation (never in the product build): cycles the MMA issuer / producer spend
// waiting, per CTA pair: [0] issuer total, [1] issuer wait full (operands), [2] issuer wait tempty
// (accumulator hand-back), [3] issuer wait tile ring, [4] producer total, [5] producer wait empty,
// [6] tiles, [7] epilogue wait tfull (warp 4)
__device__ unsigned long long g_k2_probe[128][8];
#define K2_PROBE_T0(var) const long long var = clock64()
#define K2_PROBE_ADD(acc, t0) acc += clock64() - (t0)
#else
#define K2_PROBE_T0(var)
#define K2_PROBE_ADD(acc, t0)
#endif

// Operand blocks of one launch.  A launch contracts nq pairs of operand blocks into ONE output
// block,  D = sum_q op(X_q) op(Y_q)^T,  with the accumulator resident in tensor memory across all of
// them.  nq = 1 is the single-GPU op (whole tensors); nq = sqrt(P) is one rank's share of the
// paper's Cannon-style distributed contraction: the q-th pair are the
// blocks the rank multiplies in ring step q, each behind its own tensor map -- local memory or, on
// an NVLink / NVSwitch node, a peer GPU's memory mapped into this address space (every peer is one
// hop away, so the ring's store-and-forward shifts become direct TMA reads and "partial results
// accumulate into the output block" without ever leaving TMEM).
constexpr int kMaxBlocks = 4;   // a 4 x 4 context-parallel grid
struct K2Maps {
  CUtensorMap a[kMaxBlocks];
  CUtensorMap b[kMaxBlocks];
  CUtensorMap o;
};

struct K2Params {
  int N;
  int nq;          // operand block pairs contracted by this launch (1 .. kMaxBlocks)
  int tiles_m;
  int tiles_n;
  int num_tiles;   // channels * tiles_m * tiles_n
  int num_kb;      // ceil(N / 64)
  int l2_hints;    // 1: evict_last loads / evict_first stores; 2: stores only; 3: B evict_last, o evict_first
  int serpentine;  // 1: odd column panels sweep their m-tiles downwards
  int panel_n;     // tile rasterisation: n-tiles per column panel (>= 1)
  unsigned int* sched;   // next tile index: launch-private, zeroed on the stream before the launch
  uint32_t ab_fmt;       // operand format of both inputs: ptx::kFmtBF16 or ptx::kFmtF16
  int o_f16;             // 1: the result is written as IEEE fp16 after scaling by o_scale (the fused
                         // forward path: K3 normalises o anyway, see contract_o_scale); 0: bf16
  float o_scale;         // a power of two
};

// Tile rasterisation inside one channel: column panels of `panel_n` n-tiles, m fastest-varying
// between panels' rows.  The ~74 tile pairs in flight then share a few A row-blocks and one narrow
// B panel, and consecutive waves re-use that B panel from L2 instead of streaming all of B_c.
__device__ __forceinline__ void decode_tile(const K2Params& prm, int r, int* tm, int* tn) {
  const int w = prm.panel_n;
  const int full = prm.tiles_n / w;
  const int in_full = full * prm.tiles_m * w;
  if (r < in_full) {
    const int p = r / (prm.tiles_m * w);
    const int q = r - p * prm.tiles_m * w;
    const int row = q / w;
    // serpentine: the A row blocks the previous panel touched last are the first ones of this panel
    *tm = (prm.serpentine && (p & 1)) ? prm.tiles_m - 1 - row : row;
    *tn = p * w + (q - row * w);
  } else {
    const int q = r - in_full;
    const int wl = prm.tiles_n - full * w;
    *tm = q / wl;
    *tn = full * w + (q - (q / wl) * wl);
  }
}

template <int kCtaGroup, bool kAMn, bool kBMn>
__global__ void __launch_bounds__(kThreads, 1)
k2_contract_kernel(const __grid_constant__ K2Maps maps, const K2Params prm) {
  using C = Cfg<kCtaGroup>;
  extern __shared__ uint8_t smem_raw[];
  // 128-byte swizzle needs 1024-byte aligned tiles
  const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t stage_base = smem_base;
  const uint32_t epi_base = smem_base + C::kStages * C::kStageBytes;
  const uint32_t bar_base = epi_base + C::kEpiBytes;
  // barrier layout (8 bytes each)
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (C::kStages + s); };
  auto tfull_bar = [&](int s) { return bar_base + 8u * (2 * C::kStages + s); };
  auto tempty_bar = [&](int s) { return bar_base + 8u * (2 * C::kStages + 2 + s); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * C::kStages + 4);
  // dynamic tile scheduler: a 4-deep ring of tile indices per CTA, written by the leader's
  // producer thread into both CTAs of the pair
  constexpr int kRing = 4;
  auto tsfull_bar = [&](int s) { return bar_base + 8u * (2 * C::kStages + 6 + s); };
  auto tsempty_bar = [&](int s) { return bar_base + 8u * (2 * C::kStages + 6 + kRing + s); };  // leader's
  auto tile_slot = [&](int s) { return bar_base + 8u * (2 * C::kStages + 6 + 2 * kRing) + 4u * s; };

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const uint32_t cta_rank = (kCtaGroup == 2) ? ptx::cluster_ctarank() : 0u;
  const bool is_leader = cta_rank == 0;

  const CUtensorMap& tmap_o = maps.o;
  if (warp == 0 && lane == 0) {
    for (int q = 0; q < prm.nq; ++q) {
      ptx::prefetch_tmap(&maps.a[q]);
      ptx::prefetch_tmap(&maps.b[q]);
    }
    ptx::prefetch_tmap(&tmap_o);
  }
  if (warp == 1 && lane == 0) {
    for (int s = 0; s < C::kStages; ++s) {
      ptx::mbar_init(full_bar(s), 1);
      ptx::mbar_init(empty_bar(s), 1);
    }
    for (int s = 0; s < kRing; ++s) {
      ptx::mbar_init(tsfull_bar(s), 1);
      ptx::mbar_init(tsempty_bar(s), 5 * kCtaGroup);   // every consumer of both CTAs, see below
      ptx::sts32(tile_slot(s), 0xfffffffeu);           // sentinel: "nothing published yet"
    }
    for (int s = 0; s < 2; ++s) {
      ptx::mbar_init(tfull_bar(s), 1);
      ptx::mbar_init(tempty_bar(s), 4 * kCtaGroup);   // one arrival per epilogue warp per CTA
    }
    ptx::fence_mbar_init();
  }
  if (warp == 2) {
    ptx::tmem_alloc<kCtaGroup>(tmem_slot, 512);
  }
  ptx::tc_fence_before();
  if constexpr (kCtaGroup == 2) {
    ptx::cluster_sync();
  } else {
    __syncthreads();
  }
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  const int tiles_per_ch = prm.tiles_m * prm.tiles_n;

  // ---- dynamic, in-order tile scheduler ---------------------------------------------------
  // Tiles are handed out in index order from one global counter, like the hardware block
  // scheduler would, but to persistent CTA pairs.  With a static assignment (pair g takes tiles
  // g, g + G, ...) nothing keeps the pairs in step: small speed differences between SMs add up
  // over the ~440 tiles of a pair, the tiles in flight spread over many channels / row blocks,
  // and the sharing of A_c / B_c blocks through L2 collapses (measured at N = 4096: 41-58 GB of
  // DRAM reads per launch on some B200s against 8.6 GB of operands; 9 GB with one tile per CTA
  // pair under the hardware scheduler).  In-order dispatch keeps the window of tiles in flight
  // compact.  Every tile is computed the same way whichever pair gets it: results stay bitwise
  // reproducible.
  // The leader's producer thread draws the index (draw_tile / publish_tile below) and writes it into
  // a 4-deep ring in both CTAs;
  // every other consumer (peer producer, MMA issuer, epilogue warps) waits on its local "full"
  // barrier, reads it and releases the entry on the leader's "empty" barrier.  -1 = no more tiles.
  //
  // No cluster-scope release / acquire anywhere on this path: ptxas turns
  // mbarrier.arrive.release.cluster into MEMBAR.ALL.GPU + ERRBAR + CGAERRBAR (~3000 cycles), and
  // one of those per tile in the MMA issuer (measured: 8.5 % of its time at N = 4096) and in the
  // peer's producer drained the operand pipeline at every tile boundary.  Instead:
  //   leader CTA   slot + "full" barrier in its own shared memory: CTA-scope release / acquire;
  //   peer CTA     the leader stores the index into the peer's slot with a plain st.shared::cluster
  //                and the peer's consumers poll the word itself (volatile load) until it differs
  //                from the value they saw in that slot one ring round earlier -- tile indices only
  //                grow within a launch and -1 ends it, so the value is its own flag;
  //   "empty"      consumers signal with a relaxed arrive (remote for the peer): they publish
  //                nothing, they only report that the slot has been read.
  // last_seen[s]: the value this thread consumed from ring slot s (peer only); starts at the
  // sentinel the slots are initialised with.
  constexpr uint32_t kSlotSentinel = 0xfffffffeu;
  uint32_t last_seen[kRing];
#pragma unroll
  for (int s = 0; s < kRing; ++s) last_seen[s] = kSlotSentinel;
  auto consume_tile = [&](int i) -> int {
    const int s = i % kRing;
    uint32_t v;
    if (is_leader) {
      ptx::mbar_wait(tsfull_bar(s), (i / kRing) & 1);
      asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(tile_slot(s)) : "memory");
      ptx::mbar_arrive(tsempty_bar(s));
    } else {
      uint32_t seen = kSlotSentinel;
#pragma unroll
      for (int k = 0; k < kRing; ++k) seen = (k == s) ? last_seen[k] : seen;
      do {
        asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(v) : "r"(tile_slot(s)) : "memory");
      } while (v == seen);
#pragma unroll
      for (int k = 0; k < kRing; ++k) last_seen[k] = (k == s) ? v : last_seen[k];
      ptx::mbar_arrive_relaxed_cluster(ptx::mapa(tsempty_bar(s), 0));
    }
    return static_cast<int>(v);
  };
  // Drawing and publishing are split: the atomic is issued at the start of a tile's loads and its
  // result is only needed when that tile's loads have all been issued, so its ~1 us round trip to
  // L2 overlaps the producer's own work instead of holding back the first loads of the tile.
  auto draw_tile = [&](int i) -> unsigned int {
    ptx::mbar_wait(tsempty_bar(i % kRing), ((i / kRing) & 1) ^ 1u);
    return atomicAdd(prm.sched, 1u);
  };
  auto publish_tile = [&](int i, unsigned int drawn) -> int {
    const int s = i % kRing;
    const int tile = drawn < static_cast<unsigned int>(prm.num_tiles) ? static_cast<int>(drawn) : -1;
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(tile_slot(s)), "r"(tile) : "memory");
    ptx::mbar_arrive(tsfull_bar(s));
    if constexpr (kCtaGroup == 2)
      ptx::st_shared_cluster_u32(ptx::mapa(tile_slot(s), 1), static_cast<uint32_t>(tile));
    return tile;
  };

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (ptx::elect_one()) {
      // a_c / b_c are re-read by every tile of channel c: keep them in L2, stream o past them
      const uint64_t pol_ld = prm.l2_hints == 1 ? ptx::kL2EvictLast : ptx::kL2EvictNormal;
      const uint64_t pol_ld_b = (prm.l2_hints == 1 || prm.l2_hints == 3) ? ptx::kL2EvictLast : ptx::kL2EvictNormal;
      int stage = 0;
      uint32_t phase = 0;
#ifdef FOLDCP_K2_PROBE
      long long pr_wait = 0;
      const long long pr_t0 = clock64();
#endif
      // the leader draws the next tile while it issues this tile's loads and publishes it afterwards
      int tnext = is_leader ? publish_tile(0, draw_tile(0)) : consume_tile(0);
      for (int it = 0;; ++it) {
        const int t = tnext;
        if (t < 0) break;
        unsigned int drawn = 0;
        if (is_leader) drawn = draw_tile(it + 1);
        const int ch = t / tiles_per_ch;
        const int r = t - ch * tiles_per_ch;
        int tm, tn;
        decode_tile(prm, r, &tm, &tn);
        const int m0 = tm * C::kTileM + static_cast<int>(cta_rank) * 128;
        const int n0 = tn * kTileN + static_cast<int>(cta_rank) * (kTileN / kCtaGroup);
        for (int q = 0; q < prm.nq; ++q) {
        const CUtensorMap& tmap_a = maps.a[q];
        const CUtensorMap& tmap_b = maps.b[q];
        for (int kb = 0; kb < prm.num_kb; ++kb) {
          K2_PROBE_T0(tw);
          ptx::mbar_wait(empty_bar(stage), phase ^ 1u);
          K2_PROBE_ADD(pr_wait, tw);
          const uint32_t sa = stage_base + stage * C::kStageBytes;
          const uint32_t sb = sa + C::kABytes;
          const int k0 = kb * kBlockK;
          uint32_t bar = full_bar(stage);
          if constexpr (kCtaGroup == 2) {
            if (is_leader) ptx::mbar_arrive_expect_tx(bar, 2 * C::kStageBytes);
            bar = ptx::mapa(bar, 0);
          } else {
            ptx::mbar_arrive_expect_tx(bar, C::kStageBytes);
          }
#pragma unroll
          for (int bx = 0; bx < 2; ++bx) {
            const int mn = m0 + 64 * bx;
            const int c0 = kAMn ? mn : k0;   // innermost tensor coordinate (column)
            const int c1 = kAMn ? k0 : mn;   // row
            if constexpr (kCtaGroup == 2) {
              ptx::tma_load_3d_2sm_hint(sa + bx * kBoxBytes, &tmap_a, bar, c0, c1, ch, pol_ld);
            } else {
              ptx::tma_load_3d_hint(sa + bx * kBoxBytes, &tmap_a, bar, c0, c1, ch, pol_ld);
            }
          }
#pragma unroll
          for (int bx = 0; bx < C::kBBoxes; ++bx) {
            const int mn = n0 + 64 * bx;
            const int c0 = kBMn ? mn : k0;
            const int c1 = kBMn ? k0 : mn;
            if constexpr (kCtaGroup == 2) {
              ptx::tma_load_3d_2sm_hint(sb + bx * kBoxBytes, &tmap_b, bar, c0, c1, ch, pol_ld_b);
            } else {
              ptx::tma_load_3d_hint(sb + bx * kBoxBytes, &tmap_b, bar, c0, c1, ch, pol_ld_b);
            }
          }
          if (++stage == C::kStages) {
            stage = 0;
            phase ^= 1u;
          }
        }
        }
        tnext = is_leader ? publish_tile(it + 1, drawn) : consume_tile(it + 1);
      }
#ifdef FOLDCP_K2_PROBE
      if (is_leader) {
        g_k2_probe[blockIdx.x / kCtaGroup][4] = clock64() - pr_t0;
        g_k2_probe[blockIdx.x / kCtaGroup][5] = pr_wait;
      }
#endif
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (leader CTA only) =====================
    if (is_leader && ptx::elect_one()) {
      const uint32_t idesc = ptx::make_idesc_f16kind(C::kTileM, kTileN, prm.ab_fmt, prm.ab_fmt,
                                                     kAMn ? 1 : 0, kBMn ? 1 : 0);
      // K-major : rows of 128 B, 8-row atoms 1024 B apart (SBO); one UMMA_K = 32 B along the row
      // MN-major: 64-element MN groups kBoxBytes apart (LBO), 8-k atoms 1024 B apart (SBO);
      //           one UMMA_K = two 8-k atoms = 2048 B
      constexpr uint32_t lbo_a = kAMn ? kBoxBytes : 16, lbo_b = kBMn ? kBoxBytes : 16;
      constexpr uint32_t sbo = 1024;
      constexpr uint32_t kstep_a = kAMn ? 2048 : 32, kstep_b = kBMn ? 2048 : 32;
      int stage = 0;
      uint32_t phase = 0;
#ifdef FOLDCP_K2_PROBE
      long long w_full = 0, w_tempty = 0, w_ring = 0, ntiles = 0;
      const long long is_t0 = clock64();
#endif
      for (int it = 0;; ++it) {
        K2_PROBE_T0(tr);
        const int tcur = consume_tile(it);
        K2_PROBE_ADD(w_ring, tr);
        if (tcur < 0) break;
        const int as = it & 1;
        const uint32_t aphase = (it >> 1) & 1;
        K2_PROBE_T0(te);
        ptx::mbar_wait(tempty_bar(as), aphase ^ 1u);
        K2_PROBE_ADD(w_tempty, te);
#ifdef FOLDCP_K2_PROBE
        ++ntiles;
#endif
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + as * kAccumCols;
        const int total_kb = prm.num_kb * prm.nq;      // the accumulator lives across all blocks
        for (int kb = 0; kb < total_kb; ++kb) {
          K2_PROBE_T0(tf);
          ptx::mbar_wait(full_bar(stage), phase);
          K2_PROBE_ADD(w_full, tf);
          ptx::tc_fence_after();
          const uint32_t sa = stage_base + stage * C::kStageBytes;
          const uint32_t sb = sa + C::kABytes;
#pragma unroll
          for (int k = 0; k < kBlockK / kUmmaK; ++k) {
            const uint64_t da = ptx::make_smem_desc_sw128(sa + k * kstep_a, lbo_a, sbo);
            const uint64_t db = ptx::make_smem_desc_sw128(sb + k * kstep_b, lbo_b, sbo);
            ptx::umma_bf16<kCtaGroup>(d_tmem, da, db, idesc, (kb | k) != 0 ? 1u : 0u);
          }
          ptx::umma_commit<kCtaGroup>(empty_bar(stage));   // smem slot free once these MMAs retire
          if (++stage == C::kStages) {
            stage = 0;
            phase ^= 1u;
          }
        }
        ptx::umma_commit<kCtaGroup>(tfull_bar(as));        // accumulator ready for the epilogue
      }
#ifdef FOLDCP_K2_PROBE
      g_k2_probe[blockIdx.x / kCtaGroup][0] = clock64() - is_t0;
      g_k2_probe[blockIdx.x / kCtaGroup][1] = w_full;
      g_k2_probe[blockIdx.x / kCtaGroup][2] = w_tempty;
      g_k2_probe[blockIdx.x / kCtaGroup][3] = w_ring;
      g_k2_probe[blockIdx.x / kCtaGroup][6] = ntiles;
#endif
    }
  } else if (warp >= 4) {
    // ===================== epilogue: TMEM -> bf16 -> smem -> TMA store =====================
    const int q = warp - 4;                 // TMEM lane quadrant this warp may read
    const int row = q * 32 + lane;          // row of the CTA's 128-row tile
    const bool store_thread = (warp == 4 && lane == 0);
    const uint64_t pol_st = prm.l2_hints ? ptx::kL2EvictFirst : ptx::kL2EvictNormal;
    int chunk_ctr = 0;
    for (int it = 0;; ++it) {
      int t = 0;
      if (lane == 0) t = consume_tile(it);
      t = __shfl_sync(0xffffffffu, t, 0);
      if (t < 0) break;
      const int ch = t / tiles_per_ch;
      const int r = t - ch * tiles_per_ch;
      int tm, tn;
      decode_tile(prm, r, &tm, &tn);
      const int m0 = tm * C::kTileM + static_cast<int>(cta_rank) * 128;
      const int n0 = tn * kTileN;
      const int as = it & 1;
      const uint32_t aphase = (it >> 1) & 1;
      ptx::mbar_wait(tfull_bar(as), aphase);
      ptx::tc_fence_after();
#pragma unroll 1
      for (int j = 0; j < kAccumCols / 64; ++j, ++chunk_ctr) {
        const uint32_t buf = epi_base + (chunk_ctr & 1) * kEpiBufBytes;
        // the store issued two chunks ago read this buffer: wait until it has been drained
        if (store_thread) ptx::tma_store_wait_read<1>();
        ptx::named_bar_sync(1, 128);
        uint32_t v0[32], v1[32];
        const uint32_t taddr = tmem_base + (static_cast<uint32_t>(q * 32) << 16) +
                               as * kAccumCols + j * 64;
        ptx::tmem_ld_32x32(taddr, v0);
        ptx::tmem_ld_32x32(taddr + 32, v1);
        ptx::tmem_ld_wait();
        if (j == kAccumCols / 64 - 1) {
          // accumulator fully read: hand it back to the MMA issuer (in the leader CTA)
          ptx::tc_fence_before();
          __syncwarp();
          if (lane == 0) {
            // (tcgen05.wait::ld + fence::before_thread_sync above order the TMEM reads; the
            // arrive itself publishes nothing, so it is relaxed when it goes to the leader CTA)
            if (is_leader) {
              ptx::mbar_arrive(tempty_bar(as));
            } else {
              ptx::mbar_arrive_relaxed_cluster(ptx::mapa(tempty_bar(as), 0));
            }
          }
        }
        const uint32_t row_addr = buf + row * 128;
        auto store_chunks = [&](auto f16_tag) {
          constexpr bool kF16 = decltype(f16_tag)::value;
          const float sc = prm.o_scale;
#pragma unroll
          for (int cchunk = 0; cchunk < 8; ++cchunk) {
            const uint32_t* src = (cchunk < 4) ? &v0[cchunk * 8] : &v1[(cchunk - 4) * 8];
            uint32_t pk[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const float lo = __uint_as_float(src[2 * i]), hi = __uint_as_float(src[2 * i + 1]);
              pk[i] = kF16 ? ptx::pack_f16x2(lo * sc, hi * sc) : ptx::pack_bf16x2(lo, hi);
            }
            const uint32_t dst = row_addr + ((cchunk ^ (row & 7)) << 4);
            asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(dst), "r"(pk[0]), "r"(pk[1]),
                         "r"(pk[2]), "r"(pk[3])
                         : "memory");
          }
        };
        if (prm.o_f16) store_chunks(std::true_type{}); else store_chunks(std::false_type{});
        ptx::fence_proxy_async_smem();
        ptx::named_bar_sync(1, 128);
        if (store_thread) {
          ptx::tma_store_3d_hint(&tmap_o, buf, n0 + j * 64, m0, ch, pol_st);
          ptx::tma_store_commit();
        }
      }
    }
    if (store_thread) ptx::tma_store_wait<0>();
  }

  // ===================== teardown =====================
  ptx::tc_fence_before();
  if constexpr (kCtaGroup == 2) {
    ptx::cluster_sync();
  } else {
    __syncthreads();
  }
  if (warp == 2) {
    ptx::tmem_dealloc<kCtaGroup>(tmem_base, 512);
  }
}

template <int kCtaGroup, bool kAMn, bool kBMn>
int launch_variant(const K2Maps& maps, const K2Params& prm, int sm_count, cudaStream_t stream) {
  using C = Cfg<kCtaGroup>;
  auto kern = k2_contract_kernel<kCtaGroup, kAMn, kBMn>;
  if (ensure_dynamic_smem(reinterpret_cast<const void*>(kern), C::kSmemBytes) != FOLDCP_OK)
    return FOLDCP_ERR_CUDA;
  int groups = sm_count / kCtaGroup;
  if (groups > prm.num_tiles) groups = prm.num_tiles;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(groups * kCtaGroup);
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = C::kSmemBytes;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = kCtaGroup;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  if (cudaLaunchKernelEx(&cfg, kern, maps, prm) != cudaSuccess) return FOLDCP_ERR_CUDA;
  return FOLDCP_OK;
}

int g_k2_cta_group = 2;

}  // namespace

// D_c = sum_q op(X_q,c) op(Y_q,c)^T per channel for the four operand layouts:
//   x_mn = 0: X_c is [m][k] (k contiguous, K-major)    x_mn = 1: X_c is [k][m] (m contiguous)
//   y_mn = 0: Y_c is [n][k]                            y_mn = 1: Y_c is [k][n]
// i.e. d[c][m][n] = sum_q sum_k X_q(m, k) Y_q(n, k); every block is a dense [c][N][N] tensor.  The
// forward contraction uses (0,0) / (1,1); its gradients also need the mixed (0,1) form; nq > 1 is
// the blocked (Cannon) form.
int launch_k2_gemm_blocks_bf16(const void* const* x, const void* const* y, int nq, void* d, int N,
                               bool x_mn, bool y_mn, bool xy_f16, unsigned int* sched,
                               cudaStream_t stream, float d_f16_scale = 0.f) {
  if (nq < 1 || nq > kMaxBlocks) return FOLDCP_ERR_UNSUPPORTED;
  DeviceInfo dev;
  if (!get_device_info(&dev)) return FOLDCP_ERR_CUDA;
  static const int cta_group = [] {
    const char* e = debug_env("FOLDCP_K2_CTA_GROUP");
    return (e && e[0] == '1') ? 1 : g_k2_cta_group;
  }();
  const uint64_t n = static_cast<uint64_t>(N);
  const uint64_t dims[3] = {n, n, static_cast<uint64_t>(kChannels)};
  const uint64_t strides[2] = {n * 2, n * n * 2};
  const uint32_t box_ld[3] = {64, 64, 1};
  const uint32_t box_st[3] = {64, 128, 1};
  K2Maps maps;
  int st;
  for (int q = 0; q < kMaxBlocks; ++q) {
    const int src = q < nq ? q : 0;     // unused slots repeat block 0: never read, but well-formed
    if ((st = encode_tensor_map(&maps.a[q], x[src], 2, 3, dims, strides, box_ld, true)) != FOLDCP_OK)
      return st;
    if ((st = encode_tensor_map(&maps.b[q], y[src], 2, 3, dims, strides, box_ld, true)) != FOLDCP_OK)
      return st;
  }
  if ((st = encode_tensor_map(&maps.o, d, 2, 3, dims, strides, box_st, true)) != FOLDCP_OK)
    return st;
  K2Params prm;
  prm.N = N;
  prm.nq = nq;
  const int tile_m = 128 * cta_group;
  prm.tiles_m = (N + tile_m - 1) / tile_m;
  prm.tiles_n = (N + kTileN - 1) / kTileN;
  prm.num_tiles = kChannels * prm.tiles_m * prm.tiles_n;
  prm.num_kb = (N + kBlockK - 1) / kBlockK;
  static const int l2_hints = [] {
    const char* e = debug_env("FOLDCP_K2_L2_HINTS");
    return e ? atoi(e) : 0;   // 1: loads evict_last + stores evict_first; 2: stores only
  }();
  prm.l2_hints = l2_hints;
  static const int panel = [] {
    const char* e = debug_env("FOLDCP_K2_PANEL");
    return e ? atoi(e) : 0;
  }();
  // Default rasterisation (measured with the in-order scheduler): plain row-major while one row
  // of tiles spans at most 16 n-tiles (N <= 4096: 9 GB of DRAM reads for 8.6 GB of operands);
  // beyond that, column panels of 8 n-tiles, so that the ~74 tiles in flight keep sharing one
  // narrow B panel (N = 8192: 104 GB instead of 554 GB, 105 instead of 132 ms).  Wider panels
  // read MORE (12: 127 GB, 16: 162 GB, 24: 232 GB, also with evict_last on the B loads): a 64 MB
  // panel does not stay resident in the 126 MB L2 next to the streaming A blocks and o stores.
  const int auto_panel = prm.tiles_n <= 16 ? prm.tiles_n : 8;
  prm.panel_n = (panel >= 1 && panel < prm.tiles_n) ? panel : auto_panel;
  // odd panels sweep their m-tiles downwards, so the A row blocks still in L2 from the end of the
  // previous sweep are re-used first (N = 8192: 107 instead of 115 GB of DRAM reads, time neutral)
  static const int serp = [] {
    const char* e = debug_env("FOLDCP_K2_SERP");
    return e ? atoi(e) : 1;
  }();
  prm.serpentine = serp;
  prm.sched = sched;
  prm.ab_fmt = xy_f16 ? ptx::kFmtF16 : ptx::kFmtBF16;
  prm.o_f16 = d_f16_scale != 0.f ? 1 : 0;       // 0 = bf16 result, unscaled
  prm.o_scale = d_f16_scale != 0.f ? d_f16_scale : 1.f;
  const int sms = dev.sm_count;
  if (cta_group == 2) {
    if (x_mn) return y_mn ? launch_variant<2, true, true>(maps, prm, sms, stream)
                          : launch_variant<2, true, false>(maps, prm, sms, stream);
    return y_mn ? launch_variant<2, false, true>(maps, prm, sms, stream)
                : launch_variant<2, false, false>(maps, prm, sms, stream);
  }
  if (x_mn) return y_mn ? launch_variant<1, true, true>(maps, prm, sms, stream)
                        : launch_variant<1, true, false>(maps, prm, sms, stream);
  return y_mn ? launch_variant<1, false, true>(maps, prm, sms, stream)
              : launch_variant<1, false, false>(maps, prm, sms, stream);
}

int launch_k2_gemm_bf16(const void* x, const void* y, void* d, int N, bool x_mn, bool y_mn,
                        bool xy_f16, unsigned int* sched, cudaStream_t stream,
                        float d_f16_scale = 0.f) {
  return launch_k2_gemm_blocks_bf16(&x, &y, 1, d, N, x_mn, y_mn, xy_f16, sched, stream, d_f16_scale);
}

// One rank's share of the Cannon-style distributed contraction: o_block = sum_q of Eq. 2 / Eq. 3 on
// the block pairs (a_blocks[q], b_blocks[q]).
int launch_k2_contract_blocks_bf16(const void* const* a_blocks, const void* const* b_blocks, int nq,
                                   void* o_block, int nb, int direction, bool ab_f16,
                                   unsigned int* sched, cudaStream_t stream) {
  const bool inc = direction == FOLDCP_INCOMING;
  return launch_k2_gemm_blocks_bf16(a_blocks, b_blocks, nq, o_block, nb, inc, inc, ab_f16, sched,
                                    stream);
}

int launch_k2_contract_bf16(const void* a, const void* b, void* o, int N, int direction,
                            bool ab_f16, float o_f16_scale, unsigned int* sched,
                            cudaStream_t stream) {
  const bool inc = direction == FOLDCP_INCOMING;
  return launch_k2_gemm_bf16(a, b, o, N, inc, inc, ab_f16, sched, stream, o_f16_scale);
}

// Gradients of the contraction (oracle/trimul_oracle.py contraction_backward):
//   outgoing: d_a = dO B       -> X = dO (K-major), Y = B (MN-major)
//             d_b = dO^T A     -> X = dO (MN-major), Y = A (MN-major)
//   incoming: d_a = B dO^T     -> X = B (K-major),  Y = dO (K-major)
//             d_b = A dO       -> X = A (K-major),  Y = dO (MN-major)
int launch_k2_contract_backward_bf16(const void* d_o, const void* a, const void* b, void* d_a,
                                     void* d_b, int N, int direction, unsigned int* sched0,
                                     unsigned int* sched1, cudaStream_t stream) {
  int st;
  if (direction == FOLDCP_OUTGOING) {
    if ((st = launch_k2_gemm_bf16(d_o, b, d_a, N, false, true, false, sched0, stream)) != FOLDCP_OK)
      return st;
    return launch_k2_gemm_bf16(d_o, a, d_b, N, true, true, false, sched1, stream);
  }
  if ((st = launch_k2_gemm_bf16(b, d_o, d_a, N, false, false, false, sched0, stream)) != FOLDCP_OK)
    return st;
  return launch_k2_gemm_bf16(a, d_o, d_b, N, false, true, false, sched1, stream);
}

}  // namespace foldcp

#ifdef FOLDCP_K2_PROBE
extern "C" int foldcp_debug_k2_probe_read(unsigned long long* host_out) {
  return static_cast<int>(cudaMemcpyFromSymbol(host_out, foldcp::g_k2_probe,
                                               sizeof(unsigned long long) * 128 * 8));
}
#endif
