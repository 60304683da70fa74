// K3 -- output gate + output LayerNorm + output projection + mask (
// north_star subsystem (3); AF3 Alg. 12 line 4):
//
//   g   = sigmoid(W_g LN(z; gamma_in, beta_in) + b_g)          recomputed from z, never stored
//   out = [M *] g * (W_o LN(o; gamma_out, beta_out) + b_o)     written bf16, channel-last
//
// o is channel-major [128][R] (K2's output: bf16, or fp16 scaled by a power of two on the fused
// path), z and out are [R][128] channel-last bf16.  Recomputing g here instead of materialising it
// in K1 keeps the workspace at a + b + o (N = 8192 fits) and keeps g in fp32.
//
// WHAT BOUNDS THIS KERNEL.  Inside the step the SM clock sits at the power cap (1.1 - 1.3 GHz) and
// K3 is bound by SHARED-MEMORY BANDWIDTH (128 B / clock / SM), not by HBM and not by issue slots:
// ncu on the r1 kernel and its successors showed LSU + tensor-operand + TMA wavefronts adding up to
// ~96 % of the elapsed cycles (profiles/r2_k3_notes.md).  A 128-pair tile unavoidably costs the TMA
// fill (512 wavefronts), the operand fetch of two 128 x 128 x 128 MMAs (~780), staging + TMA store
// of the output (512) and one read of each tile for the statistics (512).  Everything else had to go:
//
//  * The LayerNorms are NOT applied to the tiles (r1 rewrote both in place: 1024 more wavefronts and
//    a proxy fence on the MMA's critical path).  With x a pair's 128 raw channels, mean / rstd its
//    statistics and W' = W diag(gamma) the folded weight,
//        W LN(x) + b  =  rstd * [ W' x  -  mean (W' 1)  +  (1 / rstd) (W beta + b) ]
//    the tensor core multiplies the tiles exactly as TMA delivered them, and the two rank-one terms
//    are ALSO given to the tensor core: one more MMA of K = 16 per GEMM whose A operand holds, per
//    pair, -mean and 1/rstd and whose B operand holds, per channel, s = W' 1 and t = W beta + b,
//    each split into three pieces of the operand format (bf16: 3 x 8 bits, fp16: 3 x 11 bits) so
//    that the products carry fp32 precision (six cross terms per product, twelve of the sixteen
//    K slots).  s is summed from the ROUNDED folded weights, so D - mean s = sum_k w'_k (x_k - mean)
//    holds for the weights the tensor core really uses: a row's common offset cancels.
//  * The epilogue then needs NO per-channel constant at all -- out = rstd-scaled accumulators through
//    the gate -- where the row-per-thread form loaded four constants per output (2048 wavefronts of
//    broadcast loads per tile, as much as everything else together).
//
// GEMM orientation: the PAIR is the MMA M dimension (TMEM lane), the OUTPUT CHANNEL the N
// dimension (TMEM column):
//   D_g[pair][ch] = z[pair][k]    * W_g'[ch][k]^T     A K-major  (bf16 z tile; W_g' rounded to bf16)
//   D_o[pair][ch] = o[k][pair]^T  * W_o'[ch][k]^T     A MN-major (the o tile is [k][pair], pairs
//                                                     contiguous: the transposition K2's
//                                                     channel-major output needs is done by the
//                                                     tensor core's operand fetch, not by us)
//   D_*          += X_*[pair][16] * Y_*[ch][16]^T     the rank-one corrections (K-major, unswizzled)
// tcgen05 kind::f16 wants both operands of an MMA in one format: W_o' is fp16 when o is fp16
// (fused path: no rounding of o beyond K2's own 2^-12) and bf16 when o is bf16 (stage entry point).
//
// Persistent kernel, one CTA per SM, 28 warps, tile = 128 pairs:
//   warp 0       TMA producer : W_g, W_o once (resident), then (z tile, o tile) into a 2-deep ring
//   warp 1       MMA issuer   : 16 MMAs on the raw tiles the moment they land, then the two
//                               correction MMAs once the statistics are in; 256-column TMEM slot,
//                               two slots, so the epilogue overlaps the next tile's MMAs
//   warp 2       TMEM allocator
//   warps 4-11   epilogue     : tcgen05.ld (fragment shape 16x256b) -> rstd, sigmoid gate, mask in
//                               packed fp32 -> bf16 -> swizzled smem -> TMA store [128 pairs][64 ch]
//   warps 12-19  statistics of o : thread = 2 pairs x 32 channels of the [k][pair] tile
//   warps 20-27  statistics of z : ln_rows.cuh layernorm_rows_stats (4 lanes per pair row)
#include <cuda_bf16.h>
#include <cuda_fp16.h>

// 28 warps, most of them waiting on an mbarrier most of the time: their try_wait loops would take
// every fifth issue slot of the SM partition; with a suspend-time hint a waiting warp sleeps
#ifndef FOLDCP_MBAR_HINT_NS
#define FOLDCP_MBAR_HINT_NS 4000
#endif
#include "common.h"
#include "ln_rows.cuh"
#include "ptx.cuh"
#include "rank1.cuh"

namespace foldcp {
namespace {

constexpr int kC = kChannels;
constexpr int kTilePairs = 128;
// warp roles: 0 TMA, 1 MMA, 2 TMEM allocator, 3 idle, then epilogue, statistics(o), statistics(z).
// The order matters: the issue arbiter favours higher warp ids, and the statistics sit on the
// critical path (statistics -> correction MMAs -> accumulator ready -> epilogue) while the epilogue
// only has to keep up.
constexpr int kEpiWarps = 8;
constexpr int kLnoWarps = 8;
constexpr int kLnzWarps = 8;
constexpr int kWarpEpi = 4;                          // a multiple of 4 (TMEM lane quadrants)
constexpr int kWarpLno = kWarpEpi + kEpiWarps;
constexpr int kWarpLnz = kWarpLno + kLnoWarps;
constexpr int kThreads = (kWarpLnz + kLnzWarps) * 32;
static_assert(kWarpEpi % 4 == 0, "epilogue warps must start at a TMEM lane-quadrant boundary");
// 28 warps leave 72 registers per thread at launch; the twenty control / statistics warps give
// some up (setmaxnreg, per aligned group of four warps) for the eight epilogue warps
constexpr int kRegsOther = 64;
constexpr int kRegsEpi = 88;
constexpr int kHalfBox = 128 * 64 * 2;          // 16 KB: one TMA box (128 rows x 128 bytes)
constexpr int kMatBytes = 2 * kHalfBox;         // 32 KB
constexpr int kStages = 2;
constexpr int kStageBytes = 2 * kMatBytes;      // z tile + o tile
constexpr int kXBytes = 128 * 16 * 2;           // 4 KB: a [128][16] correction operand
// an overflowed fp32 variance (|x| beyond ~1e18, outside the documented range) must not turn into
// 0 * inf: the variance is capped, so rstd >= 1e-19 and 1 / rstd stays finite
constexpr float kMaxVar = 1.0e38f;
constexpr float kMinRstd = 1.0e-19f;

constexpr int kOffW = 0;                                   // W_g', W_o'
constexpr int kOffStage = kOffW + 2 * kMatBytes;           // ring: [z | o] per stage
constexpr int kOffOut = kOffStage + kStages * kStageBytes; // ONE staging buffer [128 pairs][64 ch]
constexpr int kOffY = kOffOut + kHalfBox;                  // Y_g, Y_o: per-channel side, resident
constexpr int kOffX = kOffY + 2 * kXBytes;                 // X_z, X_o: per-pair side, one tile
constexpr int kOffRstd = kOffX + 2 * kXBytes;              // per stage: float2[128] (rstd_z, rstd_o)
constexpr int kOffBar = kOffRstd + kStages * kTilePairs * 8;
constexpr int kSmemBytes = kOffBar + 256;
static_assert(kSmemBytes <= 232448, "K3 shared memory exceeds 227 KB");

struct K3Params {
  const __nv_bfloat16* mask;   // [R] or nullptr (also nullptr when mask_output == 0)
  const __nv_bfloat16* z_res;  // z [R][128] when out = z + update (add_residual), else nullptr
  const float2* z_stats;       // [R] (mean, rstd) of LayerNorm(z) from K1, or nullptr: computed here
  const float* g_in;
  const float* b_in;
  const float* g_out;
  const float* b_out;
  const __nv_bfloat16* w_g;    // [128][128] row-major (also read through tmap_wg)
  const __nv_bfloat16* w_o;
  const float* bias_g;         // may be nullptr
  const float* bias_o;         // may be nullptr
  float eps_z;                 // LayerNorm epsilon of z
  float eps_o;                 // of o: eps * o_scale^2 when o arrives scaled (LN(s o; s^2 eps) = LN(o; eps))
  long long R;
  int num_tiles;
  int dbg_skip;                // debug builds only: 1 skip z statistics, 2 skip o statistics, 4 skip epilogue math,
                               // 8 no wait for the previous store's read (timing only), 16 no stores
};

#ifdef FOLDCP_DEBUG_KNOBS
#define K3_DBG_SKIP(bit) ((prm.dbg_skip & (bit)) != 0)
#else
#define K3_DBG_SKIP(bit) false
#endif

#ifdef FOLDCP_K3_PROBE
// bring-up instrumentation (never in the product build): cycles per CTA.  [0] producer total,
// [1] producer wait sempty, [2] issuer wait tempty, [3] issuer wait full, [4] z-stats wait full,
// [5] z-stats work, [6] o-stats wait full, [7] o-stats work, [8] epilogue wait sready,
// [9] epilogue wait tfull, [10] epilogue barrier 1 (+ store-read wait), [11] epilogue barrier 2,
// [12] epilogue total, [13] tiles, [14] epilogue tcgen05.ld + wait, [15] issuer wait sready
__device__ unsigned long long g_k3_probe[160][16];
#define K3_PROBE_T0(var) const long long var = clock64()
#define K3_PROBE_ADD(acc, t0) acc += clock64() - (t0)
#define K3_PROBE_DECL(var) long long var = 0
#define K3_PROBE_PUT(idx, val) g_k3_probe[blockIdx.x][idx] = static_cast<unsigned long long>(val)
#else
#define K3_PROBE_T0(var)
#define K3_PROBE_ADD(acc, t0)
#define K3_PROBE_DECL(var)
#define K3_PROBE_PUT(idx, val)
#endif

// the folded weight  0.5 w gamma  as the tensor core will see it (the factor 1/2 belongs to the tanh
// form of the sigmoid, below): ONE expression, used both to build the resident operand and to sum s
template <bool kF16>
__device__ __forceinline__ uint32_t fold_pack(uint32_t w2, float g_lo, float g_hi) {
  return ptx::pack_norm<kF16>(0.5f * ptx::bf16_lo(w2) * g_lo, 0.5f * ptx::bf16_hi(w2) * g_hi);
}
template <bool kF16>
__device__ __forceinline__ float packed_sum(uint32_t v) {
  if constexpr (kF16) {
    const __half2 h = *reinterpret_cast<const __half2*>(&v);
    return __low2float(h) + __high2float(h);
  } else {
    return ptx::bf16_lo(v) + ptx::bf16_hi(v);
  }
}
// 16-bit pair word of the o tile -> fp32x2 (exact)
template <bool kF16>
__device__ __forceinline__ ptx::f32x2 o2_to_f32x2(uint32_t v) {
  if constexpr (kF16) {
    const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&v));
    return ptx::pk2(f.x, f.y);
  } else {
    return ptx::bf16x2_to_f32x2(v);
  }
}

// One row of a correction operand: the sixteen K slots that pair  (u, v)  on the per-pair side with
// (s, t)  on the per-channel side so that the MMA adds  u s + v t  with all cross terms down to
// 2^-24:   per-pair side     u1 u1 u2 u1 u2 u3 | v1 v1 v2 v1 v2 v3 | 0 0 0 0
//          per-channel side  s1 s2 s1 s3 s2 s1 | t1 t2 t1 t3 t2 t1 | 0 0 0 0
// (split3 and the unswizzled K-major row layout: rank1.cuh)
template <bool kF16>
__device__ __forceinline__ void write_pair_side(uint32_t base, uint32_t r, float u, float v) {
  uint32_t a[3], b[3];
  split3<kF16>(u, a);
  split3<kF16>(v, b);
  const uint32_t addr = rank1_row_addr(base, r);
  ptx::sts128(addr, a[0] | (a[0] << 16), a[1] | (a[0] << 16), a[1] | (a[2] << 16), b[0] | (b[0] << 16));
  ptx::sts128(addr + 128, b[1] | (b[0] << 16), b[1] | (b[2] << 16), 0u, 0u);
}
template <bool kF16>
__device__ __forceinline__ void write_channel_side(uint32_t base, uint32_t r, float s, float t) {
  uint32_t a[3], b[3];
  split3<kF16>(s, a);
  split3<kF16>(t, b);
  const uint32_t addr = rank1_row_addr(base, r);
  ptx::sts128(addr, a[0] | (a[1] << 16), a[0] | (a[2] << 16), a[1] | (a[0] << 16), b[0] | (b[1] << 16));
  ptx::sts128(addr + 128, b[0] | (b[2] << 16), b[1] | (b[0] << 16), 0u, 0u);
}

// kOF16: the o tile (and therefore W_o') is fp16; kResidual: out = z + update
template <bool kOF16, bool kResidual>
__global__ void __launch_bounds__(kThreads, 1)
k3_finalize_kernel(const __grid_constant__ CUtensorMap tmap_z,
                   const __grid_constant__ CUtensorMap tmap_o,
                   const __grid_constant__ CUtensorMap tmap_wg,
                   const __grid_constant__ CUtensorMap tmap_wo,
                   const __grid_constant__ CUtensorMap tmap_out, const K3Params prm) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t smem = ptx::smem_u32(smem_raw);
  if ((smem & 1023u) != 0) __trap();

  const uint32_t bar = smem + kOffBar;
  const uint32_t wfull = bar;
  auto full = [&](int s) { return bar + 8u * (1 + s); };        // tile landed (TMA)
  // stage reusable: the MMAs on the tiles have retired and the statistics warps have read them.
  // (Nothing else holds a stage: HBM latency under load is ~4 us, the two stages are all the bytes
  // this SM keeps in flight, so every cycle a stage waits for arithmetic is bandwidth lost.)
  auto sempty = [&](int s) { return bar + 8u * (3 + s); };
  auto tfull = [&](int u) { return bar + 8u * (5 + u); };       // accumulators complete
  auto tempty = [&](int u) { return bar + 8u * (7 + u); };      // accumulators read
  auto sready = [&](int s) { return bar + 8u * (9 + s); };      // statistics of the tile in stage s written
  const uint32_t xfree = bar + 8u * 11;                          // correction MMAs have read X_z, X_o
  auto rfree = [&](int b) { return bar + 8u * (12 + b); };      // epilogue has taken rstd buffer b
  const uint32_t tmem_slot = bar + 8u * 14;

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(&tmap_z);
    ptx::prefetch_tmap(&tmap_o);
    ptx::prefetch_tmap(&tmap_out);
  }
  if (warp == 1 && lane == 0) {
    ptx::mbar_init(wfull, 1);
    for (int s = 0; s < kStages; ++s) {
      ptx::mbar_init(full(s), 1);
      // (with K1's statistics the z warps never touch the tile)
      ptx::mbar_init(sempty(s), 1 + kLnoWarps + (prm.z_stats != nullptr ? 0 : kLnzWarps));
      ptx::mbar_init(rfree(s), kEpiWarps);
      ptx::mbar_init(sready(s), kLnzWarps + kLnoWarps);
    }
    for (int u = 0; u < 2; ++u) {
      ptx::mbar_init(tfull(u), 1);
      ptx::mbar_init(tempty(u), kEpiWarps);
    }
    ptx::mbar_init(xfree, 1);
    ptx::fence_mbar_init();
  }
  if (warp == 2) ptx::tmem_alloc<1>(tmem_slot, 512);
  if (threadIdx.x >= 128 && threadIdx.x < 384) {
    // Per output channel of each GEMM:  t = 0.5 (W beta + b)  (exact fold of the LayerNorm shift,
    // fp32 from the bf16 weights) and  s = sum_k w'_k  over the ROUNDED folded weights; both go,
    // split, into the channel's row of the resident correction operand Y.
    const int id = threadIdx.x - 128;
    const int m = id >> 7, ch = id & 127;
    const uint4* wrow = reinterpret_cast<const uint4*>((m ? prm.w_o : prm.w_g) + ch * kC);
    const float* beta = m ? prm.b_out : prm.b_in;
    const float* gam = m ? prm.g_out : prm.g_in;
    const float* bias = m ? prm.bias_o : prm.bias_g;
    float acc = 0.f, ssum = 0.f;
#pragma unroll 4
    for (int kc = 0; kc < 16; ++kc) {
      const uint4 wv = __ldg(wrow + kc);
      const float4 b0 = __ldg(reinterpret_cast<const float4*>(beta + kc * 8));
      const float4 b1 = __ldg(reinterpret_cast<const float4*>(beta + kc * 8 + 4));
      const float4 g0 = __ldg(reinterpret_cast<const float4*>(gam + kc * 8));
      const float4 g1 = __ldg(reinterpret_cast<const float4*>(gam + kc * 8 + 4));
      acc = fmaf(ptx::bf16_lo(wv.x), b0.x, acc);
      acc = fmaf(ptx::bf16_hi(wv.x), b0.y, acc);
      acc = fmaf(ptx::bf16_lo(wv.y), b0.z, acc);
      acc = fmaf(ptx::bf16_hi(wv.y), b0.w, acc);
      acc = fmaf(ptx::bf16_lo(wv.z), b1.x, acc);
      acc = fmaf(ptx::bf16_hi(wv.z), b1.y, acc);
      acc = fmaf(ptx::bf16_lo(wv.w), b1.z, acc);
      acc = fmaf(ptx::bf16_hi(wv.w), b1.w, acc);
      if (m == 0 || !kOF16) {
        ssum += packed_sum<false>(fold_pack<false>(wv.x, g0.x, g0.y));
        ssum += packed_sum<false>(fold_pack<false>(wv.y, g0.z, g0.w));
        ssum += packed_sum<false>(fold_pack<false>(wv.z, g1.x, g1.y));
        ssum += packed_sum<false>(fold_pack<false>(wv.w, g1.z, g1.w));
      } else {
        ssum += packed_sum<true>(fold_pack<true>(wv.x, g0.x, g0.y));
        ssum += packed_sum<true>(fold_pack<true>(wv.y, g0.z, g0.w));
        ssum += packed_sum<true>(fold_pack<true>(wv.z, g1.x, g1.y));
        ssum += packed_sum<true>(fold_pack<true>(wv.w, g1.z, g1.w));
      }
    }
    // tanh form: out = M sigma(g) y = M (tanh(g/2) + 1) (y/2): both factors 1/2 are folded into
    // the weights (fold_pack) and t (exact: a power of two)
    const float t = 0.5f * (acc + (bias ? bias[ch] : 0.f));
    if (m == 0 || !kOF16) {
      write_channel_side<false>(smem + kOffY + m * kXBytes, ch, ssum, t);
    } else {
      write_channel_side<true>(smem + kOffY + m * kXBytes, ch, ssum, t);
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  // weights: loaded once per CTA, resident for the whole kernel
  if (warp == 0 && ptx::elect_one()) {
    ptx::mbar_arrive_expect_tx(wfull, 2 * kMatBytes);
    ptx::tma_load_2d(smem + kOffW, &tmap_wg, wfull, 0, 0);
    ptx::tma_load_2d(smem + kOffW + kHalfBox, &tmap_wg, wfull, 64, 0);
    ptx::tma_load_2d(smem + kOffW + kMatBytes, &tmap_wo, wfull, 0, 0);
    ptx::tma_load_2d(smem + kOffW + kMatBytes + kHalfBox, &tmap_wo, wfull, 64, 0);
  }
  {
    // The resident weights become  W' = 0.5 W diag(gamma)  in the format of the tile they multiply
    // (bf16 for the gate; fp16 or bf16 for the output projection), in place: elementwise apart from
    // the gamma index, which follows from the position under the 128-byte swizzle.
    ptx::mbar_wait(wfull, 0);
    for (int off = threadIdx.x * 16; off < 2 * kMatBytes; off += kThreads * 16) {
      const int m = off / kMatBytes, rem = off % kMatBytes;
      const int box = rem / kHalfBox, row = (rem % kHalfBox) / 128, pc = (rem % 128) / 16;
      const int k0 = box * 64 + ((pc ^ (row & 7)) * 8);
      const float* gam = (m ? prm.g_out : prm.g_in) + k0;
      const float4 g0 = __ldg(reinterpret_cast<const float4*>(gam));
      const float4 g1 = __ldg(reinterpret_cast<const float4*>(gam + 4));
      uint32_t v[4];
      ptx::lds128(smem + kOffW + off, v);
      if (m == 0 || !kOF16) {
        v[0] = fold_pack<false>(v[0], g0.x, g0.y);
        v[1] = fold_pack<false>(v[1], g0.z, g0.w);
        v[2] = fold_pack<false>(v[2], g1.x, g1.y);
        v[3] = fold_pack<false>(v[3], g1.z, g1.w);
      } else {
        v[0] = fold_pack<true>(v[0], g0.x, g0.y);
        v[1] = fold_pack<true>(v[1], g0.z, g0.w);
        v[2] = fold_pack<true>(v[2], g1.x, g1.y);
        v[3] = fold_pack<true>(v[3], g1.z, g1.w);
      }
      ptx::sts128(smem + kOffW + off, v[0], v[1], v[2], v[3]);
    }
    ptx::fence_proxy_async_smem();     // also covers the Y rows written above
    __syncthreads();
  }

  const int first = blockIdx.x;
  const int stride = gridDim.x;

  if (warp < kWarpEpi) ptx::setmaxnreg_dec<kRegsOther>();
  if (warp == 0) {
    // ===================== TMA producer =====================
    if (ptx::elect_one()) {
      int it = 0;
      K3_PROBE_DECL(pw);
      K3_PROBE_T0(p0t);
      for (int t = first; t < prm.num_tiles; t += stride, ++it) {
        const int s = it & 1;
        K3_PROBE_T0(tw);
        ptx::mbar_wait(sempty(s), ((it >> 1) & 1) ^ 1u);
        K3_PROBE_ADD(pw, tw);
        ptx::mbar_arrive_expect_tx(full(s), kStageBytes);
        const uint32_t zdst = smem + kOffStage + s * kStageBytes;
        const uint32_t odst = zdst + kMatBytes;
        const int p0 = t * kTilePairs;
        ptx::tma_load_2d(zdst, &tmap_z, full(s), 0, p0);             // [128 pairs][ch 0..63]
        ptx::tma_load_2d(zdst + kHalfBox, &tmap_z, full(s), 64, p0); // [128 pairs][ch 64..127]
        ptx::tma_load_2d(odst, &tmap_o, full(s), p0, 0);             // [128 ch][pairs 0..63]
        ptx::tma_load_2d(odst + kHalfBox, &tmap_o, full(s), p0 + 64, 0);
      }
      K3_PROBE_PUT(0, clock64() - p0t);
      K3_PROBE_PUT(1, pw);
      K3_PROBE_PUT(13, it);
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (ptx::elect_one()) {
      constexpr uint32_t kOFmt = kOF16 ? ptx::kFmtF16 : ptx::kFmtBF16;
      constexpr uint32_t idesc_g = ptx::make_idesc_f16kind(128, kC, ptx::kFmtBF16, ptx::kFmtBF16, 0, 0);
      // A = o, MN-major
      constexpr uint32_t idesc_o = ptx::make_idesc_f16kind(128, kC, kOFmt, kOFmt, 1, 0);
      // the correction MMA of the o GEMM: both operands K-major
      constexpr uint32_t idesc_ox = ptx::make_idesc_f16kind(128, kC, kOFmt, kOFmt, 0, 0);
      const uint64_t dxz = ptx::make_smem_desc_noswizzle(smem + kOffX, 128, 256);
      const uint64_t dxo = ptx::make_smem_desc_noswizzle(smem + kOffX + kXBytes, 128, 256);
      const uint64_t dyg = ptx::make_smem_desc_noswizzle(smem + kOffY, 128, 256);
      const uint64_t dyo = ptx::make_smem_desc_noswizzle(smem + kOffY + kXBytes, 128, 256);
      K3_PROBE_DECL(iw_t);
      K3_PROBE_DECL(iw_f);
      K3_PROBE_DECL(iw_s);
      int it = 0;
      for (int t = first; t < prm.num_tiles; t += stride, ++it) {
        const int s = it & 1;
        const int slot = it & 1;
        const uint32_t zb = smem + kOffStage + s * kStageBytes;
        const uint32_t ob = zb + kMatBytes;
        K3_PROBE_T0(t1);
        ptx::mbar_wait(tempty(slot), ((it >> 1) & 1) ^ 1u);
        K3_PROBE_ADD(iw_t, t1);
        K3_PROBE_T0(t2);
        ptx::mbar_wait(full(s), (it >> 1) & 1);
        K3_PROBE_ADD(iw_f, t2);
        ptx::tc_fence_after();
        const uint32_t d_g = tmem_base + slot * 256;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const uint32_t off = (k >> 2) * kHalfBox + (k & 3) * 32;
          const uint64_t da = ptx::make_smem_desc_sw128(zb + off, 16, 1024);
          const uint64_t db = ptx::make_smem_desc_sw128(smem + kOffW + off, 16, 1024);
          ptx::umma_bf16<1>(d_g, da, db, idesc_g, k != 0 ? 1u : 0u);
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          // A MN-major: 64-pair groups kHalfBox apart (LBO), 8-channel atoms 1024 B apart (SBO),
          // one UMMA_K = 16 channels = 2048 B
          const uint64_t da = ptx::make_smem_desc_sw128(ob + k * 2048, kHalfBox, 1024);
          const uint32_t off = (k >> 2) * kHalfBox + (k & 3) * 32;
          const uint64_t db = ptx::make_smem_desc_sw128(smem + kOffW + kMatBytes + off, 16, 1024);
          ptx::umma_bf16<1>(d_g + 128, da, db, idesc_o, k != 0 ? 1u : 0u);
        }
        ptx::umma_commit<1>(sempty(s));      // the tiles themselves are not needed beyond this point
        // the rank-one corrections, once this tile's statistics are in X_z / X_o
        K3_PROBE_T0(t3);
        ptx::mbar_wait(sready(s), (it >> 1) & 1);
        K3_PROBE_ADD(iw_s, t3);
        ptx::tc_fence_after();
        ptx::umma_bf16<1>(d_g, dxz, dyg, idesc_g, 1u);
        ptx::umma_bf16<1>(d_g + 128, dxo, dyo, idesc_ox, 1u);
        ptx::umma_commit<1>(xfree);
        ptx::umma_commit<1>(tfull(slot));
      }
      K3_PROBE_PUT(2, iw_t);
      K3_PROBE_PUT(3, iw_f);
      K3_PROBE_PUT(15, iw_s);
    }
  } else if (warp >= kWarpLnz) {
    // ===================== statistics of the z tile (4 lanes per pair row) =====================
    ptx::setmaxnreg_dec<kRegsOther>();
    const int r = threadIdx.x - kWarpLnz * 32;
    if (prm.z_stats != nullptr) {
      // K1 normalised the same rows and left (mean, rstd) in the workspace: only turn them into the
      // correction operand X_z (one row per thread of the first four warps)
      auto load_stats = [&](int t) -> float2 {
        const long long p = static_cast<long long>(t) * kTilePairs + r;
        return (r < kTilePairs && t < prm.num_tiles && p < prm.R) ? __ldg(prm.z_stats + p)
                                                                     : make_float2(0.f, 1.f);
      };
      // (three tiles ahead: HBM latency under load exceeds a tile's time)
      float2 sq0 = load_stats(first), sq1 = load_stats(first + stride), sq2 = load_stats(first + 2 * stride);
      int it = 0;
      for (int t = first; t < prm.num_tiles; t += stride, ++it) {
        const int s = it & 1;
        const float2 st = sq0;
        sq0 = sq1;
        sq1 = sq2;
        sq2 = load_stats(t + 3 * stride);
        if (it > 0) ptx::mbar_wait(xfree, (it - 1) & 1);
        if (it > 1) ptx::mbar_wait(rfree(s), ((it >> 1) - 1) & 1);
        if (r < kTilePairs) {
          // (rstd = 0 only when the fp32 variance overflowed, |z| beyond ~1e18: stay finite)
          const float rstd = fmaxf(st.y, kMinRstd);
          write_pair_side<false>(smem + kOffX, static_cast<uint32_t>(r), -st.x, __frcp_rn(rstd));
          ptx::sts32(smem + kOffRstd + s * kTilePairs * 8 + r * 8, __float_as_uint(rstd));
        }
        ptx::fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(sready(s));
      }
    } else {
    K3_PROBE_DECL(zw);
    K3_PROBE_DECL(zc);
    int it = 0;
    for (int t = first; t < prm.num_tiles; t += stride, ++it) {
      const int s = it & 1;
      K3_PROBE_T0(t1);
      ptx::mbar_wait(full(s), (it >> 1) & 1);
      K3_PROBE_ADD(zw, t1);
      K3_PROBE_T0(t2);
      const uint32_t rstd_base = smem + kOffRstd + s * kTilePairs * 8;
      bool released = false;
      if (!K3_DBG_SKIP(1))
        layernorm_rows_stats<2, kLnzWarps * 32>(
            smem + kOffStage + s * kStageBytes, kHalfBox, r,
            [&]() {
              // the rows are in registers: hand the stage back before the arithmetic
              __syncwarp();
              if (lane == 0) ptx::mbar_arrive(sempty(s));
              released = true;
              // X_z still feeds the previous tile's correction MMA until that has retired, and the
              // rstd buffer the epilogue of two tiles ago (both long done by now)
              if (it > 0) ptx::mbar_wait(xfree, (it - 1) & 1);
              if (it > 1) ptx::mbar_wait(rfree(s), ((it >> 1) - 1) & 1);
            },
            [&](uint32_t row, float mean, float var) {
              const float ve = fminf(var + prm.eps_z, kMaxVar);
              const float rstd = rsqrtf(ve);
              write_pair_side<false>(smem + kOffX, row, -mean, ve * rstd);
              ptx::sts32(rstd_base + row * 8u, __float_as_uint(rstd));
            });
      ptx::fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) {
        if (!released) ptx::mbar_arrive(sempty(s));
        ptx::mbar_arrive(sready(s));
      }
      K3_PROBE_ADD(zc, t2);
    }
    if (threadIdx.x == kWarpLnz * 32) {
      K3_PROBE_PUT(4, zw);
      K3_PROBE_PUT(5, zc);
    }
    }
  } else if (warp >= kWarpLno && warp < kWarpLnz) {
    // ===================== statistics of the o tile, [channel][pair] =====================
    ptx::setmaxnreg_dec<kRegsOther>();
    // Warp w8 owns 16 pairs; lane = (channel quarter cq = 32 channels, pair-pair pl).  One
    // ld.shared.b32 = 2 adjacent pairs of one channel.  The four quarters visit their rows in the
    // order i ^ 2cq, which puts their 32-byte segments under four different swizzle phases:
    // conflict-free.  Shifted one-sweep accumulation as in layernorm_rows_stats (the shift is the
    // pair's channel-0 value); the quarters combine with two shuffles.
    const int w8 = warp - kWarpLno;
    const uint32_t cq = static_cast<uint32_t>(lane >> 3);
    const uint32_t pl = static_cast<uint32_t>(lane & 7);
    const uint32_t box = static_cast<uint32_t>(w8 >> 2);
    const uint32_t c16 = static_cast<uint32_t>((w8 & 3) * 2) + (pl >> 2);   // 16-byte chunk in row
    const uint32_t within = (pl & 3u) * 4u;
    // row k = 32 cq + 8 g + (jj ^ 2cq), g = 0..3, jj = 0..7: everything that depends on jj is
    // folded into eight per-thread offsets, 8 g becomes an immediate (1024 B per g)
    uint32_t toff[8];
#pragma unroll
    for (uint32_t jj = 0; jj < 8; ++jj) {
      const uint32_t k7 = jj ^ (2u * cq);
      toff[jj] = box * kHalfBox + (cq * 32u + k7) * 128u + ((c16 ^ k7) << 4) + within;
    }
    const uint32_t pair0 = box * 64u + static_cast<uint32_t>(w8 & 3) * 16u + pl * 2u;
    // The output mask rides on rstd_o (out = (tanh + 1) (M rstd_o D_o) [+ z]: M = 1 leaves the bits
    // untouched, M = 0 gives exact zeros), so the epilogue never sees it.  Two bf16 mask values per
    // thread, fetched three tiles ahead: HBM latency under this kernel's own load is ~4 us, longer
    // than a tile.
    auto load_mask2 = [&](int t) -> uint32_t {
      if (prm.mask == nullptr) return 0x3f803f80u;   // bf16 (1.0, 1.0)
      if (t >= prm.num_tiles) return 0u;
      const long long p = static_cast<long long>(t) * kTilePairs + pair0;
      return p < prm.R ? __ldg(reinterpret_cast<const uint32_t*>(prm.mask + p)) : 0u;   // R is even
    };
    uint32_t mq0 = load_mask2(first), mq1 = load_mask2(first + stride), mq2 = load_mask2(first + 2 * stride);
    K3_PROBE_DECL(ow);
    K3_PROBE_DECL(oc);
    int it = 0;
    for (int t = first; t < prm.num_tiles; t += stride, ++it) {
      const int s = it & 1;
      const uint32_t m2 = mq0;
      mq0 = mq1;
      mq1 = mq2;
      mq2 = load_mask2(t + 3 * stride);
      K3_PROBE_T0(t1);
      ptx::mbar_wait(full(s), (it >> 1) & 1);
      K3_PROBE_ADD(ow, t1);
      K3_PROBE_T0(t2);
      const uint32_t tile = smem + kOffStage + s * kStageBytes + kMatBytes;
      if (!K3_DBG_SKIP(2)) {
        uint32_t w[32];
#pragma unroll
        for (uint32_t g = 0; g < 4; ++g)
#pragma unroll
          for (uint32_t jj = 0; jj < 8; ++jj) w[g * 8 + jj] = ptx::lds32(tile + toff[jj] + g * 1024u);
        // shift: the word the cq = 0 lane loaded first (channel 0 of both pairs)
        const uint32_t cw = __shfl_sync(0xffffffffu, w[0], static_cast<int>(pl));
        float c0, c1;
        ptx::upk2(o2_to_f32x2<kOF16>(cw), c0, c1);
        const ptx::f32x2 nc = ptx::pk2(-c0, -c1);
        ptx::f32x2 a0 = ptx::pk2(0.f, 0.f), a1 = a0, b0 = a0, b1 = a0;
#pragma unroll
        for (int i = 0; i < 32; i += 2) {
          const ptx::f32x2 d0 = ptx::add2(o2_to_f32x2<kOF16>(w[i]), nc);
          const ptx::f32x2 d1 = ptx::add2(o2_to_f32x2<kOF16>(w[i + 1]), nc);
          a0 = ptx::add2(a0, d0);
          a1 = ptx::add2(a1, d1);
          b0 = ptx::fma2(d0, d0, b0);
          b1 = ptx::fma2(d1, d1, b1);
        }
        float s10, s11, s20, s21;
        ptx::upk2(ptx::add2(a0, a1), s10, s11);
        ptx::upk2(ptx::add2(b0, b1), s20, s21);
        // the tile has been consumed: hand the stage back before the reductions
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(sempty(s));
        if (it > 0) ptx::mbar_wait(xfree, (it - 1) & 1);
        if (it > 1) ptx::mbar_wait(rfree(s), ((it >> 1) - 1) & 1);
        s10 += __shfl_xor_sync(0xffffffffu, s10, 8);
        s11 += __shfl_xor_sync(0xffffffffu, s11, 8);
        s20 += __shfl_xor_sync(0xffffffffu, s20, 8);
        s21 += __shfl_xor_sync(0xffffffffu, s21, 8);
        s10 += __shfl_xor_sync(0xffffffffu, s10, 16);
        s11 += __shfl_xor_sync(0xffffffffu, s11, 16);
        s20 += __shfl_xor_sync(0xffffffffu, s20, 16);
        s21 += __shfl_xor_sync(0xffffffffu, s21, 16);
        if (cq == 0) {
          const float md0 = s10 * (1.0f / kC), md1 = s11 * (1.0f / kC);
          const float ve0 = fminf(fmaxf(fmaf(-md0, md0, s20 * (1.0f / kC)), 0.f) + prm.eps_o, kMaxVar);
          const float ve1 = fminf(fmaxf(fmaf(-md1, md1, s21 * (1.0f / kC)), 0.f) + prm.eps_o, kMaxVar);
          const float r0 = rsqrtf(ve0), r1 = rsqrtf(ve1);
          write_pair_side<kOF16>(smem + kOffX + kXBytes, pair0, -(c0 + md0), ve0 * r0);
          write_pair_side<kOF16>(smem + kOffX + kXBytes, pair0 + 1, -(c1 + md1), ve1 * r1);
          const uint32_t ra = smem + kOffRstd + s * kTilePairs * 8 + pair0 * 8u + 4u;
          ptx::sts32(ra, __float_as_uint(r0 * ptx::bf16_lo(m2)));
          ptx::sts32(ra + 8, __float_as_uint(r1 * ptx::bf16_hi(m2)));
        }
      } else {
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(sempty(s));
      }
      ptx::fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(sready(s));
      K3_PROBE_ADD(oc, t2);
    }
    if (threadIdx.x == kWarpLno * 32) {
      K3_PROBE_PUT(6, ow);
      K3_PROBE_PUT(7, oc);
    }
  } else if (warp >= kWarpEpi && warp < kWarpLno) {
    // ===================== epilogue (thread = pair) =====================
    // With the LayerNorm terms inside the accumulators the epilogue needs no per-channel constant:
    //   out = (tanh(rstd_z D_g) + 1) (M rstd_o D_o) [+ z]        (M rides on rstd_o, see there)
    // Warp = (lane quadrant q) x (32-channel part e of the 64 channels in flight); the tile's two
    // channel halves go one after the other through ONE [128 pairs][64 ch] staging buffer, a half's
    // 32 outputs being computed into registers first so that the wait for the previous TMA store to
    // have read the buffer is covered by arithmetic.  Row-per-thread tcgen05.ld (32x32b) keeps the
    // staging stores 16 bytes wide: the MUFU, conversion and shared-memory instructions all go
    // through the same issue queue, so fewer, wider shared-memory instructions matter.
    ptx::setmaxnreg_inc<kRegsEpi>();
    const int q = warp & 3;                       // TMEM lane quadrant (hardware: warp % 4)
    const int e = (warp - kWarpEpi) >> 2;         // which 32 of the 64 channels
    const int r = q * 32 + lane;                  // pair within the tile
    const uint32_t stage_buf = smem + kOffOut;
    const uint32_t row_addr = stage_buf + r * 128;
    const uint32_t sw = static_cast<uint32_t>(r & 7);
    const bool store_thread = (warp == kWarpEpi && lane == 0);
    constexpr uint32_t kEpiBar = 1;
    K3_PROBE_DECL(ew_s);
    K3_PROBE_DECL(ew_t);
    K3_PROBE_DECL(ew_b1);
    K3_PROBE_DECL(ew_b2);
    K3_PROBE_DECL(ew_ld);
    K3_PROBE_T0(e0t);
    int it = 0;
    for (int t = first; t < prm.num_tiles; t += stride, ++it) {
      const int s = it & 1;
      const int slot = it & 1;
      K3_PROBE_T0(t2);
      ptx::mbar_wait(sready(s), (it >> 1) & 1);             // rstd of this tile (long complete:
      ptx::mbar_wait(tfull(slot), (it >> 1) & 1);           // the correction MMAs waited for it)
      K3_PROBE_ADD(ew_t, t2);
      ptx::tc_fence_after();
      float rz, ro;
      ptx::upk2(ptx::lds64x(smem + kOffRstd + s * kTilePairs * 8 + r * 8), rz, ro);
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(rfree(s));            // the rstd buffer may be rewritten
      const uint32_t tbase = tmem_base + (static_cast<uint32_t>(q * 32) << 16) + slot * 256 + e * 32;
      const long long p = static_cast<long long>(t) * kTilePairs + r;
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        uint32_t packed[16];
#pragma unroll
        for (int c = 0; c < 2; ++c) {
          uint32_t vg[16], vo[16];
          const int ch0 = h * 64 + e * 32 + c * 16;          // first of this chunk's 16 channels
          K3_PROBE_T0(t5);
          ptx::tmem_ld_32x16(tbase + h * 64 + c * 16, vg);
          ptx::tmem_ld_32x16(tbase + 128 + h * 64 + c * 16, vo);
          // residual: this pair's 16 raw z channels (the tile was just read by TMA: an L2 hit)
          uint32_t zr[8] = {0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
          if constexpr (kResidual) {
            if (p < prm.R) {
              const uint4* zp = reinterpret_cast<const uint4*>(prm.z_res + p * kC + ch0);
              const uint4 zr0 = __ldg(zp), zr1 = __ldg(zp + 1);
              zr[0] = zr0.x; zr[1] = zr0.y; zr[2] = zr0.z; zr[3] = zr0.w;
              zr[4] = zr1.x; zr[5] = zr1.y; zr[6] = zr1.z; zr[7] = zr1.w;
            }
          }
          ptx::tmem_ld_wait();
          K3_PROBE_ADD(ew_ld, t5);
          if (h == 1 && c == 1) {
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(tempty(slot));
          }
          if (K3_DBG_SKIP(4)) {
#pragma unroll
            for (int i = 0; i < 8; ++i) packed[c * 8 + i] = vo[2 * i] ^ vg[2 * i + 1];
          } else {
#pragma unroll
            for (int j = 0; j < 16; j += 2) {
              // g/2 = rstd_z D_g ,  y/2 = M rstd_o D_o  (everything else is already in D)
              const ptx::f32x2 gx = ptx::mul2(ptx::pk2u(vg[j], vg[j + 1]), ptx::pk2(rz, rz));
              const ptx::f32x2 y = ptx::mul2(ptx::pk2u(vo[j], vo[j + 1]), ptx::pk2(ro, ro));
              float g0, g1, v0, v1;
              ptx::upk2(gx, g0, g1);
              const ptx::f32x2 th = K3_DBG_SKIP(32) ? gx : ptx::pk2(ptx::tanh_approx(g0), ptx::tanh_approx(g1));
              // out = (tanh(g/2) + 1) (y/2) [+ z]
              ptx::f32x2 v = ptx::fma2(y, th, y);
              if constexpr (kResidual) v = ptx::add2(v, ptx::bf16x2_to_f32x2(zr[j >> 1]));
              ptx::upk2(v, v0, v1);
              packed[c * 8 + (j >> 1)] = K3_DBG_SKIP(64) ? (__float_as_uint(v0) ^ __float_as_uint(v1)) : ptx::pack_bf16x2(v0, v1);
            }
          }
        }
        // the previous store out of the staging buffer has read it
        K3_PROBE_T0(t3);
        if (store_thread && !K3_DBG_SKIP(8)) ptx::tma_store_wait_read<0>();
        ptx::named_bar_sync(kEpiBar, kEpiWarps * 32);
        K3_PROBE_ADD(ew_b1, t3);
#pragma unroll
        for (int i = 0; i < 4; ++i)
          ptx::sts128(row_addr + ((static_cast<uint32_t>(e * 4 + i) ^ sw) << 4), packed[4 * i],
                      packed[4 * i + 1], packed[4 * i + 2], packed[4 * i + 3]);
        ptx::fence_proxy_async_smem();
        K3_PROBE_T0(t4);
        ptx::named_bar_sync(kEpiBar, kEpiWarps * 32);
        K3_PROBE_ADD(ew_b2, t4);
        if (store_thread && !K3_DBG_SKIP(16)) {
          ptx::tma_store_2d(&tmap_out, stage_buf, h * 64, t * kTilePairs);
          ptx::tma_store_commit();
        }
      }
    }
    if (store_thread) {
      K3_PROBE_PUT(8, ew_s);
      K3_PROBE_PUT(9, ew_t);
      K3_PROBE_PUT(10, ew_b1);
      K3_PROBE_PUT(11, ew_b2);
      K3_PROBE_PUT(12, clock64() - e0t);
      K3_PROBE_PUT(14, ew_ld);
    }
    if (store_thread) ptx::tma_store_wait<0>();
  }

  // ===================== teardown =====================
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 2) ptx::tmem_dealloc<1>(tmem_base, 512);
}

}  // namespace

// o_f16: o holds IEEE fp16 values scaled by o_scale (a power of two; K2 on the fused path), else
// bf16 unscaled (o_scale = 1)
int launch_k3_finalize_bf16(const void* o, const void* z, const void* mask,
                            const foldcp_trimul_params* p, int N, void* out, bool o_f16,
                            float o_scale, const void* z_stats, cudaStream_t stream) {
  DeviceInfo dev;
  if (!get_device_info(&dev)) return FOLDCP_ERR_CUDA;
  const uint64_t R = static_cast<uint64_t>(N) * N;
  CUtensorMap tz, to, twg, two, tout;
  int st;
  const uint32_t box[2] = {64, 128};
  {
    const uint64_t dims[2] = {kC, R};
    const uint64_t strides[1] = {kC * 2};
    if ((st = encode_tensor_map(&tz, z, 2, 2, dims, strides, box, true)) != FOLDCP_OK) return st;
    if ((st = encode_tensor_map(&tout, out, 2, 2, dims, strides, box, true)) != FOLDCP_OK)
      return st;
  }
  {
    const uint64_t dims[2] = {R, kC};
    const uint64_t strides[1] = {R * 2};
    if ((st = encode_tensor_map(&to, o, 2, 2, dims, strides, box, true)) != FOLDCP_OK) return st;
  }
  {
    const uint64_t dims[2] = {kC, kC};
    const uint64_t strides[1] = {kC * 2};
    if ((st = encode_tensor_map(&twg, p->w_g, 2, 2, dims, strides, box, true)) != FOLDCP_OK)
      return st;
    if ((st = encode_tensor_map(&two, p->w_o, 2, 2, dims, strides, box, true)) != FOLDCP_OK)
      return st;
  }
  K3Params prm;
  prm.mask = p->mask_output ? static_cast<const __nv_bfloat16*>(mask) : nullptr;
  prm.z_res = p->add_residual ? static_cast<const __nv_bfloat16*>(z) : nullptr;
  prm.z_stats = static_cast<const float2*>(z_stats);
  prm.g_in = p->ln_in_gamma;
  prm.b_in = p->ln_in_beta;
  prm.g_out = p->ln_out_gamma;
  prm.b_out = p->ln_out_beta;
  prm.w_g = static_cast<const __nv_bfloat16*>(p->w_g);
  prm.w_o = static_cast<const __nv_bfloat16*>(p->w_o);
  prm.bias_g = p->b_g;
  prm.bias_o = p->b_o;
  prm.eps_z = p->ln_eps;
  prm.eps_o = p->ln_eps * o_scale * o_scale;
  prm.R = static_cast<long long>(R);
  prm.num_tiles = static_cast<int>((R + kTilePairs - 1) / kTilePairs);
  static const int dbg_skip = [] {
    const char* e = debug_env("FOLDCP_K3_SKIP");
    return e ? atoi(e) : 0;
  }();
  prm.dbg_skip = dbg_skip;
  const int grid = prm.num_tiles < dev.sm_count ? prm.num_tiles : dev.sm_count;
  const bool res = p->add_residual != 0;
  auto kern = o_f16 ? (res ? k3_finalize_kernel<true, true> : k3_finalize_kernel<true, false>)
                    : (res ? k3_finalize_kernel<false, true> : k3_finalize_kernel<false, false>);
  if (ensure_dynamic_smem(reinterpret_cast<const void*>(kern), kSmemBytes) != FOLDCP_OK)
    return FOLDCP_ERR_CUDA;
  kern<<<grid, kThreads, kSmemBytes, stream>>>(tz, to, twg, two, tout, prm);
  return check_launch();
}

}  // namespace foldcp

#ifdef FOLDCP_K3_PROBE
extern "C" int foldcp_debug_k3_probe_read(unsigned long long* host_out) {
  return static_cast<int>(cudaMemcpyFromSymbol(host_out, foldcp::g_k3_probe,
                                               sizeof(unsigned long long) * 160 * 16));
}
#endif
