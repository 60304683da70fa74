// K1 -- input LayerNorm + the four gated projections + pair mask (
// a, b are "projections of the pair representation ... with element-wise
// gating"; north_star / AF3 Alg. 12 lines 1-3):
//
//   z'  = LN(z; gamma_in, beta_in, eps)                     per pair, over the 128 channels
//   a   = M * sigmoid(W_ga z' + b_ga) * (W_a z' + b_a)      b likewise
//
// z is [R = N*N][128] channel-last bf16; a and b are written channel-major [128][R] as fp16 (or
// bf16, see kOutF16), which is the layout K2's TMA boxes want for both directions.
//
// The GEMM is oriented so that the OUTPUT CHANNEL is the MMA M dimension (TMEM lane) and the
// PAIR is the MMA N dimension (TMEM column):   D[ch][pair] = W[ch][k] * z'[pair][k]^T.
// A thread of the epilogue then owns one channel and a run of consecutive pairs -- exactly a
// contiguous run of the channel-major output -- and the projection and its gate for the same
// (channel, pair) sit in the same thread (two accumulators, same lane, same column).
//
// With the weights as the A operand they can live in TENSOR MEMORY for the whole kernel
// (tcgen05.mma with A from TMEM): 4 matrices x 64 columns = half of TMEM, no shared memory and
// no shared-memory operand traffic for them.  The LayerNorm affine is folded into them once per
// CTA:  W z' + b = (W diag(gamma)) n + (W beta + b),  n = (z - mean) * rstd,  so the LayerNorm
// warps only normalise.  W diag(gamma) is rounded to fp16 (2^-12 relative; n is fp16 too -- see
// common.h kNormFp16), the folded bias stays fp32 in registers.
//
// Persistent kernel, one CTA per SM, 28 warps (FOLDCP_K1_TEAMS = 4; 16 warps with 2), tile = 128 pairs:
//   warp 0       TMA producer : z tiles into a kZStages-deep ring
//   warps 1, 2   MMA issuers  : per tile eight "units" (pair quarter pq, tensor u in {a, b}); a unit
//                               = projection + gate MMA (M=128 ch, N=32 pairs, K=128) into one
//                               64-column TMEM slot; four slots, two per tensor.  Warp 1 issues
//                               tensor a's units, warp 2 (after allocating TMEM: 512 columns =
//                               256 weights + 4 x 64 accumulators) tensor b's: 128 small MMAs per
//                               tile were one thread's whole instruction budget
//   LayerNorm    8 warps      : ln_rows.cuh -- z rows -> registers -> two-pass mean/variance in
//                               fp32 -> n written back in place as the K-major B operand; also
//                               stage the pair mask and an "all ones" flag per tile
//   epilogue     16 warps     : four teams of four warps (tensor x pair-quarter parity = one TMEM
//                               slot each): tcgen05.ld both accumulators -> bias, sigmoid, gate,
//                               mask in packed fp32 -> bf16 -> swizzled smem -> TMA store
//                               [128 ch][64 pairs] per tensor (also: once per CTA they fold and
//                               park the weights in TMEM).  Four sigmoid-issuing warps per
//                               scheduler keep the MUFU pipe busier than two (measured -7 %).
#include <cuda_bf16.h>

#include "common.h"
#include "ln_rows.cuh"
#include "ptx.cuh"
#include "tile_sched.cuh"

namespace foldcp {
namespace {

constexpr int kC = kChannels;                   // 128
constexpr int kTilePairs = 128;
// warp roles: 0 TMA, 1 MMA, 2 TMEM allocator, 3 idle, then LayerNorm warps, then epilogue teams
#ifndef FOLDCP_K1_TEAMS
#define FOLDCP_K1_TEAMS 4
#endif
constexpr int kTeams = FOLDCP_K1_TEAMS;         // epilogue teams of 4 warps: 2 or 4
constexpr int kPar = kTeams / 2;                // teams per output tensor (pair-quarter parities)
constexpr int kLnWarps = kTeams == 2 ? 4 : 8;   // 4 teams leave 72 registers/thread: one row in flight
// role order: the issue arbiter favours higher warp ids (FOLDCP_K1_LN_HIGH=1 puts the LayerNorm
// warps, which feed everything else, above the epilogue teams)
#ifndef FOLDCP_K1_LN_HIGH
#define FOLDCP_K1_LN_HIGH 0
#endif
constexpr int kWarpEpi = FOLDCP_K1_LN_HIGH ? 4 : 4 + kLnWarps;   // a multiple of 4 (TMEM lane quadrants)
constexpr int kWarpLn = FOLDCP_K1_LN_HIGH ? 4 + 4 * kTeams : 4;
constexpr int kThreads = (4 + kLnWarps + 4 * kTeams) * 32;
static_assert(kTeams == 2 || kTeams == 4, "two or four epilogue teams");
constexpr int kHalfBox = 128 * 64 * 2;          // 16 KB: one TMA box, 128 rows x 64 bf16
constexpr int kMatBytes = 2 * kHalfBox;         // 32 KB: a 128 x 128 16-bit tile (two k-halves)
#ifndef FOLDCP_K1_ZSTAGES
#define FOLDCP_K1_ZSTAGES 4
#endif
constexpr int kZStages = FOLDCP_K1_ZSTAGES;      // 4 (with 4 staging buffers) or 2 (with 8)
constexpr int kMaskSlots = 8;                   // >= kZStages + 3 (see the epilogue), power of 2
// staging buffers [128 ch][64 pairs]: (tensor, 64-pair group) of a tile, and with a 2-deep z ring a
// second set so that the stores of two tiles are in flight
constexpr int kOutSets = kZStages == 2 ? 2 : 1;
constexpr int kOutBufs = 4 * kOutSets;

constexpr int kOffZ = 0;                                   // z ring
constexpr int kOffOut = kOffZ + kZStages * kMatBytes;      // staging buffers
constexpr int kOffMask = kOffOut + kOutBufs * kHalfBox;    // fp32 pair mask per tile slot
constexpr int kOffFlag = kOffMask + kMaskSlots * kTilePairs * 4;   // 4 "all ones" words per slot
constexpr int kOffBar = kOffFlag + kMaskSlots * 16;
constexpr int kRingDepth = 8;
constexpr int kOffRing = kOffBar + 256;
constexpr int kSmemBytes = kOffRing + TileRing<kRingDepth>::kBytes;
static_assert(kSmemBytes <= 232448, "K1 shared memory exceeds 227 KB");
static_assert((3 * kZStages + 10 + 2 * kOutBufs) * 8 <= 256, "barrier region too small");

constexpr int kTmemW = 0;        // columns 0..255: four weight matrices, 64 columns each
constexpr int kTmemAcc = 256;    // columns 256..511: four slots of (projection 32 | gate 32)

#ifdef FOLDCP_K1_PROBE
// bring-up instrumentation (never in the product build): cycles per CTA.  [0] producer total,
// [1] producer wait zempty, [2] issuer wait zready, [3] issuer wait tempty, [4] LayerNorm wait zfull,
// [5] LayerNorm work, [6] epilogue (team 0, quadrant 0) wait tfull, [7] wait oempty, [8] total,
// [9] store issuer wait ofull, [10] tiles, [11] store issuer wait read
__device__ unsigned long long g_k1_probe[160][16];
#define K1_PROBE_T0(var) const long long var = clock64()
#define K1_PROBE_ADD(acc, t0) acc += clock64() - (t0)
#define K1_PROBE_DECL(var) long long var = 0
#define K1_PROBE_PUT(idx, val) g_k1_probe[blockIdx.x][idx] = static_cast<unsigned long long>(val)
#else
#define K1_PROBE_T0(var)
#define K1_PROBE_ADD(acc, t0)
#define K1_PROBE_DECL(var)
#define K1_PROBE_PUT(idx, val)
#endif

struct K1Params {
  const __nv_bfloat16* mask;   // [R] or nullptr
  const __nv_bfloat16* w[4];   // W_a, W_ga, W_b, W_gb: [128][128] row-major
  const float* bias[4];        // b_a, b_ga, b_b, b_gb (each may be nullptr)
  const float* gamma;
  const float* beta;
  float eps;
  long long R;                 // number of pairs
  int num_tiles;
  unsigned int* sched;
  float2* stats;               // [R] (mean, rstd) of every pair's LayerNorm(z), or nullptr: K3 re-uses them
  int dbg_skip;                // debug builds only: 1 no LayerNorm arithmetic, 2 no epilogue arithmetic, 4 no TMA stores
};

#ifdef FOLDCP_DEBUG_KNOBS
#define K1_DBG_SKIP(bit) ((prm.dbg_skip & (bit)) != 0)
#else
#define K1_DBG_SKIP(bit) false
#endif

// kOutF16: a and b are written as IEEE fp16 (the forward path: 11-bit significand, see the header's
// numerics notes) instead of bf16 (the backward pass's recomputation, whose contraction-gradient
// GEMMs pair a / b with bf16 gradients -- tcgen05 kind::f16 wants both operands in one format)
template <bool kTanhSigmoid, bool kOutF16>
__global__ void __launch_bounds__(kThreads, 1)
k1_project_kernel(const __grid_constant__ CUtensorMap tmap_z,
                  const __grid_constant__ CUtensorMap tmap_a,
                  const __grid_constant__ CUtensorMap tmap_b, const K1Params prm) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t smem = ptx::smem_u32(smem_raw);
  if ((smem & 1023u) != 0) __trap();   // 128-byte swizzle needs 1024-byte aligned tiles

  const uint32_t bar = smem + kOffBar;
  auto zfull = [&](int s) { return bar + 8u * s; };
  auto zempty = [&](int s) { return bar + 8u * (kZStages + s); };
  auto zready = [&](int s) { return bar + 8u * (2 * kZStages + s); };
  auto tfull = [&](int u) { return bar + 8u * (3 * kZStages + u); };
  auto tempty = [&](int u) { return bar + 8u * (3 * kZStages + 4 + u); };
  const uint32_t tmem_slot = bar + 8u * (3 * kZStages + 8);
  const uint32_t wready = bar + 8u * (3 * kZStages + 9);   // weights are in TMEM
  auto ofull = [&](int b) { return bar + 8u * (3 * kZStages + 10 + b); };    // staging buffer b
  auto oempty = [&](int b) { return bar + 8u * (3 * kZStages + 10 + kOutBufs + b); };   // (set, tensor, group)
  const TileRing<kRingDepth> ring{smem + kOffRing};
  constexpr uint32_t kRingConsumers = 2 + 1 + kLnWarps + 4 * kTeams;   // 2 MMA, store, LN, epilogue

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(&tmap_z);
    ptx::prefetch_tmap(&tmap_a);
    ptx::prefetch_tmap(&tmap_b);
  }
  if (warp == 1 && lane == 0) {
    for (int s = 0; s < kZStages; ++s) {
      ptx::mbar_init(zfull(s), 1);
      ptx::mbar_init(zempty(s), 2);        // one commit per MMA issuer
      ptx::mbar_init(zready(s), kLnWarps * 32);
    }
    for (int u = 0; u < 4; ++u) {
      ptx::mbar_init(tfull(u), 1);
      ptx::mbar_init(tempty(u), 4);
    }
    ptx::mbar_init(wready, 4 * kTeams);
    ring.init(kRingConsumers);
    for (int b = 0; b < kOutBufs; ++b) {
      ptx::mbar_init(ofull(b), 4 * kPar);   // one arrival per warp that fills the buffer
      ptx::mbar_init(oempty(b), 1);
    }
    ptx::fence_mbar_init();
  }
  if (warp == 2) ptx::tmem_alloc<1>(tmem_slot, 512);
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));


  if (warp == 0) {
    // ===================== TMA producer =====================
    if (ptx::elect_one()) {
      int it = 0;
      K1_PROBE_DECL(pw);
      K1_PROBE_T0(p0);
      for (;; ++it) {
        const int t = ring.produce(it, prm.sched, prm.num_tiles);
        if (t < 0) break;
        const int s = it % kZStages;
        K1_PROBE_T0(t1);
        ptx::mbar_wait(zempty(s), ((it / kZStages) & 1) ^ 1u);
        K1_PROBE_ADD(pw, t1);
        ptx::mbar_arrive_expect_tx(zfull(s), kMatBytes);
        const uint32_t dst = smem + kOffZ + s * kMatBytes;
        const int row0 = t * kTilePairs;          // < 2^31: R <= 2^30 (N <= 32768)
        ptx::tma_load_2d(dst, &tmap_z, zfull(s), 0, row0);
        ptx::tma_load_2d(dst + kHalfBox, &tmap_z, zfull(s), 64, row0);
      }
      K1_PROBE_PUT(0, clock64() - p0);
      K1_PROBE_PUT(1, pw);
      K1_PROBE_PUT(10, it);
    }
  } else if (warp == 1 || warp == 2) {
    // ===================== MMA issuers: warp 1 tensor a, warp 2 tensor b =====================
    // 128 small MMAs per tile (N = 32) cost the issuing thread ~25 cycles each -- with one issuer that
    // thread's instruction stream was the kernel's critical path at the power-capped clock (probe:
    // busy 3,200 of 4,200 cycles per tile).  Two issuers on two SM partitions, one per output tensor.
    const int u = warp - 1;
    if (ptx::elect_one()) {
      // A = folded weights in TMEM, B = n (K-major, 32 pairs), both fp16 (or both bf16)
      constexpr uint32_t kFmt = kNormFp16 ? ptx::kFmtF16 : ptx::kFmtBF16;
      constexpr uint32_t idesc = ptx::make_idesc_f16kind(128, 32, kFmt, kFmt, 0, 0);
      ptx::mbar_wait(wready, 0);
      ptx::tc_fence_after();
      K1_PROBE_DECL(iw_z);
      K1_PROBE_DECL(iw_t);
      int it = 0;
      for (;; ++it) {
        if (ring.consume(it) < 0) break;
        const int s = it % kZStages;
        K1_PROBE_T0(t1);
        ptx::mbar_wait(zready(s), (it / kZStages) & 1);
        K1_PROBE_ADD(iw_z, t1);
        ptx::tc_fence_after();
        const uint32_t zb = smem + kOffZ + s * kMatBytes;
#pragma unroll
        for (int pq = 0; pq < 4; ++pq) {
          {
            // slot 2u + (pq & 1): each tensor's team alternates between its two slots, so this
            // unit's MMAs overlap the team's epilogue of the previous unit
            const uint32_t slot = static_cast<uint32_t>(2 * u + (pq & 1));
            const uint32_t use = static_cast<uint32_t>(it * 2 + (pq >> 1));   // per-slot use count
            K1_PROBE_T0(t2);
            ptx::mbar_wait(tempty(slot), (use & 1u) ^ 1u);
            K1_PROBE_ADD(iw_t, t2);
            ptx::tc_fence_after();
#pragma unroll
            for (int m2 = 0; m2 < 2; ++m2) {
              const uint32_t a_tmem = tmem_base + kTmemW + (2 * u + m2) * 64;
              const uint32_t d_tmem = tmem_base + kTmemAcc + slot * 64 + m2 * 32;
#pragma unroll
              for (int k = 0; k < 8; ++k) {
                // rows pq*32.. of the tile: 32 rows x 128 B = 4 KB into each k-half box
                const uint32_t off = pq * 4096 + (k >> 2) * kHalfBox + (k & 3) * 32;
                const uint64_t db = ptx::make_smem_desc_sw128(zb + off, 16, 1024);
                ptx::umma_f16_ts(d_tmem, a_tmem + k * 8, db, idesc, k != 0 ? 1u : 0u);
              }
            }
            ptx::umma_commit<1>(tfull(slot));
          }
        }
        ptx::umma_commit<1>(zempty(s));   // stage reusable once all MMAs of the tile (both issuers') retired
      }
      if (u == 0) {
        K1_PROBE_PUT(2, iw_z);
        K1_PROBE_PUT(3, iw_t);
      }
    }
  } else if (warp == 3) {
    // ===================== TMA store issuer =====================
    // The epilogue warps only arrive on ofull(b) when their part of staging buffer b is written
    // and carry on; this thread issues the store and hands the buffer back (oempty) once the
    // previous store has finished reading shared memory.  No block-wide barrier in the epilogue.
    if (ptx::elect_one()) {
      int it = 0, prev = -1;
      K1_PROBE_DECL(sw_f);
      K1_PROBE_DECL(sw_r);
      for (;; ++it) {
        const int t = ring.consume(it);
        if (t < 0) break;
#pragma unroll
        for (int g = 0; g < 2; ++g) {
#pragma unroll
          for (int u = 0; u < 2; ++u) {
            const int b = (it % kOutSets) * 4 + 2 * u + g;
            K1_PROBE_T0(t1);
            ptx::mbar_wait(ofull(b), (it / kOutSets) & 1);
            K1_PROBE_ADD(sw_f, t1);
            if (!K1_DBG_SKIP(4))
              ptx::tma_store_2d(u == 0 ? &tmap_a : &tmap_b, smem + kOffOut + b * kHalfBox,
                                t * kTilePairs + g * 64, 0);
            ptx::tma_store_commit();
            if (prev >= 0) {
              K1_PROBE_T0(t2);
              ptx::tma_store_wait_read<1>();
              K1_PROBE_ADD(sw_r, t2);
              ptx::mbar_arrive(oempty(prev));
            }
            prev = b;
          }
        }
      }
      ptx::tma_store_wait<0>();
      K1_PROBE_PUT(9, sw_f);
      K1_PROBE_PUT(11, sw_r);
    }
  } else if (warp >= kWarpLn && warp < kWarpLn + kLnWarps) {
    // ===================== LayerNorm =====================
    const int r = threadIdx.x - kWarpLn * 32;
    // the pair mask is fetched one tile ahead so that its latency never sits on the critical path
    auto load_mask = [&](int t) -> unsigned short {
      if (prm.mask == nullptr || r >= kTilePairs) return static_cast<unsigned short>(0x3f80);
      if (t < 0) return static_cast<unsigned short>(0);
      const long long p = static_cast<long long>(t) * kTilePairs + r;
      return p < prm.R ? __ldg(reinterpret_cast<const unsigned short*>(prm.mask) + p)
                       : static_cast<unsigned short>(0);
    };
    K1_PROBE_DECL(lw);
    K1_PROBE_DECL(lc);
    int tnext = ring.consume_warp(0, lane);
    unsigned short mnext = load_mask(tnext);
    int it = 0;
    for (;; ++it) {
      const int t = tnext;
      if (t < 0) break;
      const int s = it % kZStages;
      const unsigned short mraw = mnext;
      tnext = ring.consume_warp(it + 1, lane);
      mnext = load_mask(tnext);
      K1_PROBE_T0(t1);
      ptx::mbar_wait(zfull(s), (it / kZStages) & 1);
      K1_PROBE_ADD(lw, t1);
      K1_PROBE_T0(t2);
      if (!K1_DBG_SKIP(1))
      layernorm_rows_inplace<kNormFp16, false, kLnWarps == 4 ? 2 : 1, kLnWarps * 32>(
          smem + kOffZ + s * kMatBytes, kHalfBox, r, 0, 0, prm.eps,
          [&](uint32_t row, float mean, float rstd) {
            const long long p = static_cast<long long>(t) * kTilePairs + row;
            if (prm.stats != nullptr && p < prm.R) prm.stats[p] = make_float2(mean, rstd);
          });
      const int ms = it & (kMaskSlots - 1);
      if (r < kTilePairs) {   // warp-uniform: the first four LayerNorm warps stage mask and flag
        reinterpret_cast<float*>(smem_raw + kOffMask)[ms * kTilePairs + r] =
            __uint_as_float(static_cast<uint32_t>(mraw) << 16);
        const bool ones = __all_sync(0xffffffffu, mraw == 0x3f80);
        if (lane == 0)
          reinterpret_cast<uint32_t*>(smem_raw + kOffFlag)[ms * 4 + (warp - kWarpLn)] =
              ones ? 1u : 0u;
      }
      ptx::fence_proxy_async_smem();
      ptx::mbar_arrive(zready(s));
      K1_PROBE_ADD(lc, t2);
    }
    if (threadIdx.x == kWarpLn * 32) {
      K1_PROBE_PUT(4, lw);
      K1_PROBE_PUT(5, lc);
    }
  } else if (warp >= kWarpEpi && warp < kWarpEpi + 4 * kTeams) {
    // ===================== epilogue =====================
    // warp -> TMEM lane quadrant q (hardware rule: warp % 4) and team = (tensor h, parity par)
    const int q = warp & 3;
    const int team = (warp - kWarpEpi) >> 2;
    const int h = team & 1;          // output tensor: 0 = a, 1 = b
    const int par = team >> 1;       // which pair quarters (pq % kPar == par) this team handles
    const int ch = q * 32 + lane;                       // output channel = TMEM lane
    const uint32_t lane_base = tmem_base + (static_cast<uint32_t>(q * 32) << 16);
    constexpr float kLog2e = 1.4426950408889634f;
    // sigmoid(x) = 0.5 tanh(0.5 x) + 0.5   or   1 / (1 + 2^(-x log2 e))
    constexpr float kGateScale = kTanhSigmoid ? 0.5f : -kLog2e;

    // ---- once per CTA: fold the LayerNorm affine into the weights, park them in TMEM ----
    // every thread computes its channel's four folded biases  W beta + b ; warps 8-11 store
    // W_a, W_ga and warps 12-15 store W_b, W_gb as  W diag(gamma)  (row ch -> TMEM lane ch)
    // tanh form: a = M sigma(g) p = M (tanh(g/2) + 1) (p/2) -- the two factors 1/2 go into the
    // folded weights and biases (exact: a power of two), saving a multiply per element
    constexpr float kWScale = kTanhSigmoid ? 0.5f : 1.0f;
    float fb[4];
#pragma unroll 1
    for (int m = 0; m < 4; ++m) {
      const uint4* wrow = reinterpret_cast<const uint4*>(prm.w[m] + static_cast<size_t>(ch) * kC);
      const bool mine = par == 0 && (m >> 1) == h;
      float acc = 0.f;
#pragma unroll 1
      for (int half = 0; half < 2; ++half) {
        uint32_t packed[32];
#pragma unroll
        for (int kc = 0; kc < 8; ++kc) {
          const int k0 = half * 64 + kc * 8;
          const uint4 wv = __ldg(wrow + half * 8 + kc);
          const float4 g0 = __ldg(reinterpret_cast<const float4*>(prm.gamma + k0));
          const float4 g1 = __ldg(reinterpret_cast<const float4*>(prm.gamma + k0 + 4));
          const float4 b0 = __ldg(reinterpret_cast<const float4*>(prm.beta + k0));
          const float4 b1 = __ldg(reinterpret_cast<const float4*>(prm.beta + k0 + 4));
          const uint32_t ww[4] = {wv.x, wv.y, wv.z, wv.w};
          const float gg[8] = {g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, g1.z, g1.w};
          const float bb[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const float lo = ptx::bf16_lo(ww[e]), hi = ptx::bf16_hi(ww[e]);
            acc = fmaf(lo, bb[2 * e], acc);
            acc = fmaf(hi, bb[2 * e + 1], acc);
            packed[kc * 4 + e] =
                ptx::pack_norm<kNormFp16>(kWScale * lo * gg[2 * e], kWScale * hi * gg[2 * e + 1]);
          }
        }
        if (mine) ptx::tmem_st_32x32(lane_base + kTmemW + m * 64 + half * 32, packed);
      }
      fb[m] = acc + (prm.bias[m] ? prm.bias[m][ch] : 0.f);
    }
    ptx::tmem_st_wait();
    ptx::tc_fence_before();
    __syncwarp();
    if (lane == 0) ptx::mbar_arrive(wready);

    // this thread's team handles tensor h only (a: matrices 0, 1; b: matrices 2, 3)
    const float fbp = kWScale * (h ? fb[2] : fb[0]);
    const float fbg = (kTanhSigmoid ? 0.5f : kGateScale) * (h ? fb[3] : fb[1]);
    const ptx::f32x2 bias_p2 = ptx::pk2(fbp, fbp), bias_g2 = ptx::pk2(fbg, fbg);
    const ptx::f32x2 gscale2 = ptx::pk2(kGateScale, kGateScale);
    const ptx::f32x2 one2 = ptx::pk2(1.0f, 1.0f);
    (void)gscale2;
    (void)one2;

    const uint32_t sw = static_cast<uint32_t>(ch & 7);

    // one 16-column chunk: bias, sigmoid gate, (mask), bf16 pack
    auto compute_chunk = [&](const uint32_t (&vp)[16], const uint32_t (&vg)[16], uint32_t maddr, bool masked, uint32_t (&packed)[8]) {
#pragma unroll
      for (int j4 = 0; j4 < 4; ++j4) {
        ptx::f32x2 m2[2];
        if (masked) ptx::lds128x2(maddr + j4 * 16, m2);
#pragma unroll
        for (int e2 = 0; e2 < 2; ++e2) {
          const int j = j4 * 4 + e2 * 2;
          ptx::f32x2 pj = ptx::add2(ptx::pk2u(vp[j], vp[j + 1]), bias_p2);
          float v0, v1;
          if constexpr (kTanhSigmoid) {
            // pj = p/2, gx = g/2 (scales folded into the weights): a = M (tanh(gx) + 1) pj
            float g0, g1;
            ptx::upk2(ptx::add2(ptx::pk2u(vg[j], vg[j + 1]), bias_g2), g0, g1);
            if (masked) pj = ptx::mul2(pj, m2[e2]);
            ptx::upk2(ptx::fma2(pj, ptx::pk2(ptx::tanh_approx(g0), ptx::tanh_approx(g1)), pj), v0, v1);
          } else {
            float g0, g1, d0, d1;
            ptx::upk2(ptx::fma2(ptx::pk2u(vg[j], vg[j + 1]), gscale2, bias_g2), g0, g1);
            ptx::upk2(ptx::add2(ptx::pk2(ptx::ex2_approx(g0), ptx::ex2_approx(g1)), one2), d0, d1);
            if (masked) pj = ptx::mul2(pj, m2[e2]);
            ptx::upk2(ptx::mul2(pj, ptx::pk2(ptx::rcp_approx(d0), ptx::rcp_approx(d1))), v0, v1);
          }
          packed[j4 * 2 + e2] = ptx::pack_norm<kOutF16>(v0, v1);
        }
      }
    };

    // A team is four warps, one per TMEM lane quadrant.  kTeams = 2: team h owns tensor h (a / b)
    // and both of its TMEM slots, so the MMAs of unit pq+1 run while it post-processes unit pq.
    // kTeams = 4: two teams per tensor, one per slot (pair quarters of one parity each); more
    // warps per scheduler keep the MUFU pipe (the sigmoids) busier.  A unit is 32 pairs; two units
    // fill one [128 ch][64 pairs] staging buffer (128-byte rows: narrower TMA stores are markedly
    // slower), stored once both halves are in.  Tensors a and b are handled independently (own
    // barrier, store thread and staging buffers).
    constexpr bool kPrefetch = kTeams == 2;     // enough registers for a second tcgen05.ld buffer
    K1_PROBE_DECL(ew_t);
    K1_PROBE_DECL(ew_o);
    K1_PROBE_T0(e0);
    int it = 0;
    for (;; ++it) {
      if (ring.consume_warp(it, lane) < 0) break;
      const int ms = it & (kMaskSlots - 1);
      bool masked = true;
#pragma unroll
      for (int i = 0; i < 4 / kPar; ++i) {
        const int pq = par + kPar * i;
        const int g = pq >> 1;                                            // 64-pair group
        const uint32_t slot = static_cast<uint32_t>(2 * h + (pq & 1));
        const uint32_t use = static_cast<uint32_t>(it * 2 + g);          // per-slot use count
        const int b = (it % kOutSets) * 4 + 2 * h + g;                    // staging buffer
        K1_PROBE_T0(t1);
        ptx::mbar_wait(tfull(slot), use & 1u);
        K1_PROBE_ADD(ew_t, t1);
        ptx::tc_fence_after();
        if (i == 0) {
          // written by the LayerNorm warps before zready, hence visible after this tile's tfull
          uint32_t f[4];
          ptx::lds128(smem + kOffFlag + ms * 16, f);
          masked = (f[0] & f[1] & f[2] & f[3]) == 0u;   // warp-uniform
        }
        const uint32_t taddr = lane_base + kTmemAcc + slot * 64;
        const uint32_t maddr = smem + kOffMask + (ms * kTilePairs + pq * 32) * 4;
        const uint32_t row_addr = smem + kOffOut + b * kHalfBox + ch * 128;
        // 32 columns in two chunks of 16
        uint32_t vp[kPrefetch ? 2 : 1][16], vg[kPrefetch ? 2 : 1][16];
        ptx::tmem_ld_32x16(taddr, vp[0]);
        ptx::tmem_ld_32x16(taddr + 32, vg[0]);
        // first write of this team into buffer b for this tile: last tile's store has read it
        K1_PROBE_T0(t2);
        if (kPar == 2 || (pq & 1) == 0) ptx::mbar_wait(oempty(b), ((it / kOutSets) & 1) ^ 1u);
        K1_PROBE_ADD(ew_o, t2);
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          const int cb = kPrefetch ? k : 0;
          ptx::tmem_ld_wait();
          if (k == 0) {
            if constexpr (kPrefetch) {
              // the tcgen05.ld of the second chunk is in flight while the first is computed
              ptx::tmem_ld_32x16(taddr + 16, vp[1]);
              ptx::tmem_ld_32x16(taddr + 32 + 16, vg[1]);
            }
          } else {
            // accumulators are in registers: hand the TMEM slot back to the issuer (the mask
            // slot stays valid: kMaskSlots >= kZStages + 3)
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(tempty(slot));
          }
          uint32_t packed[8];
          if (K1_DBG_SKIP(2)) {
#pragma unroll
            for (int i = 0; i < 8; ++i) packed[i] = vp[cb][2 * i] ^ vg[cb][2 * i + 1];
          } else if (masked) {
            compute_chunk(vp[cb], vg[cb], maddr + k * 64, true, packed);
          } else {
            compute_chunk(vp[cb], vg[cb], maddr + k * 64, false, packed);
          }
          if constexpr (!kPrefetch) {
            if (k == 0) {
              ptx::tmem_ld_32x16(taddr + 16, vp[0]);
              ptx::tmem_ld_32x16(taddr + 32 + 16, vg[0]);
            }
          }
          const uint32_t c16 = static_cast<uint32_t>((pq & 1) * 4 + k * 2);
          ptx::sts128(row_addr + ((c16 ^ sw) << 4), packed[0], packed[1], packed[2], packed[3]);
          ptx::sts128(row_addr + (((c16 + 1) ^ sw) << 4), packed[4], packed[5], packed[6],
                      packed[7]);
        }
        if (kPar == 2 || (pq & 1)) {
          // this warp's share of the 64-pair group is in shared memory: tell the store issuer
          ptx::fence_proxy_async_smem();
          __syncwarp();
          if (lane == 0) ptx::mbar_arrive(ofull(b));
        }
      }
    }
    if (threadIdx.x == kWarpEpi * 32) {
      K1_PROBE_PUT(6, ew_t);
      K1_PROBE_PUT(7, ew_o);
      K1_PROBE_PUT(8, clock64() - e0);
    }
  }

  // ===================== teardown =====================
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 2) ptx::tmem_dealloc<1>(tmem_base, 512);
}

bool k1_tanh_sigmoid() {
  static const bool v = [] {
    const char* e = debug_env("FOLDCP_K1_SIGMOID");   // "exp" = ex2+rcp (2 MUFU), default tanh (1 MUFU)
    return !(e && e[0] == 'e');
  }();
  return v;
}

}  // namespace

int launch_k1_project_bf16(const void* z, const void* mask, const foldcp_trimul_params* p, int N,
                           void* a, void* b, bool ab_f16, void* z_stats, unsigned int* sched,
                           cudaStream_t stream) {
  DeviceInfo dev;
  if (!get_device_info(&dev)) return FOLDCP_ERR_CUDA;
  const uint64_t R = static_cast<uint64_t>(N) * N;
  CUtensorMap tz, ta, tb;
  int st;
  {
    const uint64_t dims[2] = {kC, R};
    const uint64_t strides[1] = {kC * 2};
    const uint32_t box[2] = {64, 128};
    if ((st = encode_tensor_map(&tz, z, 2, 2, dims, strides, box, true)) != FOLDCP_OK) return st;
  }
  {
    const uint64_t dims[2] = {R, kC};
    static const uint64_t dbg_pad = [] {
      const char* e = debug_env("FOLDCP_K1_PAD");     // timing experiment: padded channel stride (bytes)
      return e ? static_cast<uint64_t>(atoll(e)) : 0ull;
    }();
    const uint64_t strides[1] = {R * 2 + dbg_pad};
    const uint32_t box[2] = {64, 128};
    if ((st = encode_tensor_map(&ta, a, 2, 2, dims, strides, box, true)) != FOLDCP_OK) return st;
    if ((st = encode_tensor_map(&tb, b, 2, 2, dims, strides, box, true)) != FOLDCP_OK) return st;
  }
  K1Params prm;
  prm.mask = static_cast<const __nv_bfloat16*>(mask);
  prm.w[0] = static_cast<const __nv_bfloat16*>(p->w_a);
  prm.w[1] = static_cast<const __nv_bfloat16*>(p->w_a_gate);
  prm.w[2] = static_cast<const __nv_bfloat16*>(p->w_b);
  prm.w[3] = static_cast<const __nv_bfloat16*>(p->w_b_gate);
  prm.bias[0] = p->b_a;
  prm.bias[1] = p->b_a_gate;
  prm.bias[2] = p->b_b;
  prm.bias[3] = p->b_b_gate;
  prm.gamma = p->ln_in_gamma;
  prm.beta = p->ln_in_beta;
  prm.eps = p->ln_eps;
  prm.R = static_cast<long long>(R);
  prm.num_tiles = static_cast<int>((R + kTilePairs - 1) / kTilePairs);
  prm.sched = sched;
  prm.stats = static_cast<float2*>(z_stats);
  static const int dbg_skip = [] {
    const char* e = debug_env("FOLDCP_K1_SKIP");
    return e ? atoi(e) : 0;
  }();
  prm.dbg_skip = dbg_skip;
  const int grid = prm.num_tiles < dev.sm_count ? prm.num_tiles : dev.sm_count;
  const bool tanh_sig = k1_tanh_sigmoid();
  auto kern = tanh_sig ? (ab_f16 ? k1_project_kernel<true, true> : k1_project_kernel<true, false>)
                       : (ab_f16 ? k1_project_kernel<false, true> : k1_project_kernel<false, false>);
  if (ensure_dynamic_smem(reinterpret_cast<const void*>(kern), kSmemBytes) != FOLDCP_OK)
    return FOLDCP_ERR_CUDA;
  kern<<<grid, kThreads, kSmemBytes, stream>>>(tz, ta, tb, prm);
  return check_launch();
}

}  // namespace foldcp

#ifdef FOLDCP_K1_PROBE
extern "C" int foldcp_debug_k1_probe_read(unsigned long long* host_out) {
  return static_cast<int>(cudaMemcpyFromSymbol(host_out, foldcp::g_k1_probe,
                                               sizeof(unsigned long long) * 160 * 16));
}
#endif
