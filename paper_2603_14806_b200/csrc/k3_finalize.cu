// K3 -- output gate + output LayerNorm + output projection + mask (
// north_star subsystem (3); AF3 Alg. 12 line 4):
//
//   g   = sigmoid(W_g LN(z; gamma_in, beta_in) + b_g)          recomputed from z, never stored
//   out = [M *] g * (W_o LN(o; gamma_out, beta_out) + b_o)     written bf16, channel-last
//
// o is channel-major [128][R] bf16 (K2's output), z and out are [R][128] channel-last bf16.
// Recomputing g here instead of materialising it in K1 keeps the workspace at a + b + o
// (N = 8192 fits) and keeps g in fp32 (a bf16 round trip of g costs accuracy -- SURVEY 8(c)).
//
// GEMM orientation: the PAIR is the MMA M dimension (TMEM lane), the OUTPUT CHANNEL the N
// dimension (TMEM column), so an epilogue thread owns a contiguous run of one pair's output row:
//   D_g[pair][ch] = z'[pair][k]      * W_g[ch][k]^T     A K-major  (z tile as TMA delivers it)
//   D_o[pair][ch] = LN(o)[k][pair]^T * W_o[ch][k]^T     A MN-major (o tile is [k][pair], pairs
//                                                       contiguous: the transposition K2's
//                                                       channel-major output needs is done by the
//                                                       tensor core's operand fetch, not by us)
//
// Both LayerNorm affines are folded into the GEMMs once per CTA (W LN(x) + b =
// (W diag(gamma)) n + (W beta + b), n = (x - mean) * rstd): gamma goes into the resident weights
// while they are converted to the operand format of the normalised tiles (fp16, see common.h),
// beta into per-channel fp32 biases in shared memory.  The LayerNorm warps only normalise.
//
// Persistent kernel, one CTA per SM, 24 warps, tile = 128 pairs:
//   warp 0       TMA producer : W_g, W_o once (resident), then (z tile, o tile) into a 2-deep ring
//   warp 1       MMA issuer   : two MMAs (M=128 pairs, N=128 ch, K=128) into a 256-column TMEM
//                               slot; two slots, so the epilogue overlaps the next tile's MMAs
//   warp 2       TMEM allocator
//   warps 4-7    LayerNorm(z) : ln_rows.cuh (rows in registers, two-pass statistics, in place)
//   warps 8-15   LayerNorm(o) : thread = 2 pairs x 32 channels of the [k][pair] tile, held in
//                               registers, exact two-pass statistics combined across the four
//                               channel quarters with shuffles, in place
//   warps 16-23  epilogue     : tcgen05.ld -> bias, sigmoid gate, mask in packed fp32 -> bf16 ->
//                               swizzled smem -> TMA store [128 pairs][64 ch]
#include <cuda_bf16.h>

#include "common.h"
#include "ln_rows.cuh"
#include "ptx.cuh"

namespace foldcp {
namespace {

constexpr int kC = kChannels;
constexpr int kTilePairs = 128;
// warp roles: 0 TMA, 1 MMA, 2 TMEM allocator, 3 idle, then LayerNorm(z), LayerNorm(o), epilogue
#ifndef FOLDCP_K3_LNZ_WARPS
#define FOLDCP_K3_LNZ_WARPS 4
#endif
constexpr int kLnzWarps = FOLDCP_K3_LNZ_WARPS;       // 4 or 8
constexpr int kWarpLnz = 4;
constexpr int kWarpLno = kWarpLnz + kLnzWarps;       // 8 warps
constexpr int kWarpEpi = kWarpLno + 8;               // 8 warps; a multiple of 4 (TMEM lane quadrants)
constexpr int kThreads = (kWarpEpi + 8) * 32;
static_assert(kLnzWarps == 4 || kLnzWarps == 8, "LayerNorm(z) runs on 4 or 8 warps");
constexpr int kHalfBox = 128 * 64 * 2;          // 16 KB: one TMA box (128 rows x 128 bytes)
constexpr int kMatBytes = 2 * kHalfBox;         // 32 KB
constexpr int kStages = 2;
constexpr int kStageBytes = 2 * kMatBytes;      // z tile + o tile

constexpr int kOffW = 0;                                   // W_g, W_o
constexpr int kOffStage = kOffW + 2 * kMatBytes;           // ring: [z | o] per stage
constexpr int kOffOut = kOffStage + kStages * kStageBytes; // 2 staging buffers [128 pairs][64 ch]
constexpr int kOffVec = kOffOut + 2 * kHalfBox;            // folded biases t_g[128], t_o[128] (fp32)
constexpr int kOffBar = kOffVec + 2 * kC * 4;
constexpr int kSmemBytes = kOffBar + 128;
static_assert(kSmemBytes <= 232448, "K3 shared memory exceeds 227 KB");

struct K3Params {
  const __nv_bfloat16* mask;   // [R] or nullptr (also nullptr when mask_output == 0)
  const __nv_bfloat16* z_res;  // z [R][128] when out = z + update (add_residual), else nullptr
  const float* g_in;
  const float* b_in;
  const float* g_out;
  const float* b_out;
  const __nv_bfloat16* w_g;    // [128][128] row-major (also read through tmap_wg)
  const __nv_bfloat16* w_o;
  const float* bias_g;         // may be nullptr
  const float* bias_o;         // may be nullptr
  float eps;
  long long R;
  int num_tiles;
  int dbg_skip;                // debug builds only: 1 skip LN(z) math, 2 skip LN(o) math, 4 skip epilogue math
};

#ifdef FOLDCP_DEBUG_KNOBS
#define K3_DBG_SKIP(bit) ((prm.dbg_skip & (bit)) != 0)
#else
#define K3_DBG_SKIP(bit) false
#endif

template <bool kTanhSigmoid>
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
  auto full = [&](int s) { return bar + 8u * (1 + s); };
  auto sempty = [&](int s) { return bar + 8u * (3 + s); };
  auto zready = [&](int s) { return bar + 8u * (5 + s); };
  auto oready = [&](int s) { return bar + 8u * (7 + s); };
  auto tfull = [&](int u) { return bar + 8u * (9 + u); };
  auto tempty = [&](int u) { return bar + 8u * (11 + u); };
  const uint32_t tmem_slot = bar + 8u * 13;

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
      ptx::mbar_init(sempty(s), 1);
      ptx::mbar_init(zready(s), kLnzWarps * 32);
      ptx::mbar_init(oready(s), 256);
    }
    for (int u = 0; u < 2; ++u) {
      ptx::mbar_init(tfull(u), 1);
      ptx::mbar_init(tempty(u), 8);
    }
    ptx::fence_mbar_init();
  }
  if (warp == 2) ptx::tmem_alloc<1>(tmem_slot, 512);
  if (threadIdx.x >= 128 && threadIdx.x < 384) {
    // Fold the LayerNorm shifts into the biases:  W LN(x) + b = (W diag(gamma)) n + (W beta + b)
    // with n = (x - mean) * rstd.  Thread -> (matrix, output channel); fp32, from the bf16 weights.
    const int id = threadIdx.x - 128;
    const int m = id >> 7, ch = id & 127;
    const uint4* wrow = reinterpret_cast<const uint4*>((m ? prm.w_o : prm.w_g) + ch * kC);
    const float* beta = m ? prm.b_out : prm.b_in;
    const float* bias = m ? prm.bias_o : prm.bias_g;
    float acc = 0.f;
#pragma unroll 4
    for (int kc = 0; kc < 16; ++kc) {
      const uint4 wv = __ldg(wrow + kc);
      const float4 b0 = __ldg(reinterpret_cast<const float4*>(beta + kc * 8));
      const float4 b1 = __ldg(reinterpret_cast<const float4*>(beta + kc * 8 + 4));
      acc = fmaf(ptx::bf16_lo(wv.x), b0.x, acc);
      acc = fmaf(ptx::bf16_hi(wv.x), b0.y, acc);
      acc = fmaf(ptx::bf16_lo(wv.y), b0.z, acc);
      acc = fmaf(ptx::bf16_hi(wv.y), b0.w, acc);
      acc = fmaf(ptx::bf16_lo(wv.z), b1.x, acc);
      acc = fmaf(ptx::bf16_hi(wv.z), b1.y, acc);
      acc = fmaf(ptx::bf16_lo(wv.w), b1.z, acc);
      acc = fmaf(ptx::bf16_hi(wv.w), b1.w, acc);
    }
    // tanh form: out = M sigma(g) y = M (tanh(g/2) + 1) (y/2): both factors 1/2 are folded into
    // the weights and these biases (exact: a power of two)
    reinterpret_cast<float*>(smem_raw + kOffVec)[id] =
        (kTanhSigmoid ? 0.5f : 1.0f) * (acc + (bias ? bias[ch] : 0.f));
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
    // The resident weights become  W diag(gamma)  in the operand format of the normalised tiles
    // (fp16 unless FOLDCP_NORM_FP16=0), in place: elementwise apart from the gamma index, which
    // follows from the position under the 128-byte swizzle.
    ptx::mbar_wait(wfull, 0);
    for (int off = threadIdx.x * 16; off < 2 * kMatBytes; off += kThreads * 16) {
      const int m = off / kMatBytes, rem = off % kMatBytes;
      const int box = rem / kHalfBox, row = (rem % kHalfBox) / 128, pc = (rem % 128) / 16;
      const int k0 = box * 64 + ((pc ^ (row & 7)) * 8);
      const float* gam = (m ? prm.g_out : prm.g_in) + k0;
      const float4 g0 = __ldg(reinterpret_cast<const float4*>(gam));
      const float4 g1 = __ldg(reinterpret_cast<const float4*>(gam + 4));
      constexpr float ws = kTanhSigmoid ? 0.5f : 1.0f;
      uint32_t v[4];
      ptx::lds128(smem + kOffW + off, v);
      v[0] = ptx::pack_norm<kNormFp16>(ws * ptx::bf16_lo(v[0]) * g0.x, ws * ptx::bf16_hi(v[0]) * g0.y);
      v[1] = ptx::pack_norm<kNormFp16>(ws * ptx::bf16_lo(v[1]) * g0.z, ws * ptx::bf16_hi(v[1]) * g0.w);
      v[2] = ptx::pack_norm<kNormFp16>(ws * ptx::bf16_lo(v[2]) * g1.x, ws * ptx::bf16_hi(v[2]) * g1.y);
      v[3] = ptx::pack_norm<kNormFp16>(ws * ptx::bf16_lo(v[3]) * g1.z, ws * ptx::bf16_hi(v[3]) * g1.w);
      ptx::sts128(smem + kOffW + off, v[0], v[1], v[2], v[3]);
    }
    ptx::fence_proxy_async_smem();
    __syncthreads();
  }

  const int first = blockIdx.x;
  const int stride = gridDim.x;


  if (warp == 0) {
    // ===================== TMA producer =====================
    if (ptx::elect_one()) {
      int it = 0;
      for (int t = first; t < prm.num_tiles; t += stride, ++it) {
        const int s = it & 1;
        ptx::mbar_wait(sempty(s), ((it >> 1) & 1) ^ 1u);
        ptx::mbar_arrive_expect_tx(full(s), kStageBytes);
        const uint32_t zdst = smem + kOffStage + s * kStageBytes;
        const uint32_t odst = zdst + kMatBytes;
        const int p0 = t * kTilePairs;
        ptx::tma_load_2d(zdst, &tmap_z, full(s), 0, p0);             // [128 pairs][ch 0..63]
        ptx::tma_load_2d(zdst + kHalfBox, &tmap_z, full(s), 64, p0); // [128 pairs][ch 64..127]
        ptx::tma_load_2d(odst, &tmap_o, full(s), p0, 0);             // [128 ch][pairs 0..63]
        ptx::tma_load_2d(odst + kHalfBox, &tmap_o, full(s), p0 + 64, 0);
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (ptx::elect_one()) {
      constexpr uint32_t kNormFmt = kNormFp16 ? ptx::kFmtF16 : ptx::kFmtBF16;
      constexpr uint32_t idesc_g = ptx::make_idesc_f16kind(128, kC, kNormFmt, kNormFmt, 0, 0);
      // A = LN(o), MN-major
      constexpr uint32_t idesc_o = ptx::make_idesc_f16kind(128, kC, kNormFmt, kNormFmt, 1, 0);
      ptx::mbar_wait(wfull, 0);
      int it = 0;
      for (int t = first; t < prm.num_tiles; t += stride, ++it) {
        const int s = it & 1;
        const int slot = it & 1;
        const uint32_t zb = smem + kOffStage + s * kStageBytes;
        const uint32_t ob = zb + kMatBytes;
        ptx::mbar_wait(tempty(slot), ((it >> 1) & 1) ^ 1u);
        ptx::mbar_wait(zready(s), (it >> 1) & 1);
        ptx::tc_fence_after();
        const uint32_t d_g = tmem_base + slot * 256;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const uint32_t off = (k >> 2) * kHalfBox + (k & 3) * 32;
          const uint64_t da = ptx::make_smem_desc_sw128(zb + off, 16, 1024);
          const uint64_t db = ptx::make_smem_desc_sw128(smem + kOffW + off, 16, 1024);
          ptx::umma_bf16<1>(d_g, da, db, idesc_g, k != 0 ? 1u : 0u);
        }
        ptx::mbar_wait(oready(s), (it >> 1) & 1);
        ptx::tc_fence_after();
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          // A MN-major: 64-pair groups kHalfBox apart (LBO), 8-channel atoms 1024 B apart (SBO),
          // one UMMA_K = 16 channels = 2048 B
          const uint64_t da = ptx::make_smem_desc_sw128(ob + k * 2048, kHalfBox, 1024);
          const uint32_t off = (k >> 2) * kHalfBox + (k & 3) * 32;
          const uint64_t db = ptx::make_smem_desc_sw128(smem + kOffW + kMatBytes + off, 16, 1024);
          ptx::umma_bf16<1>(d_g + 128, da, db, idesc_o, k != 0 ? 1u : 0u);
        }
        ptx::umma_commit<1>(tfull(slot));
        ptx::umma_commit<1>(sempty(s));
      }
    }
  } else if (warp >= kWarpLnz && warp < kWarpLno) {
    // ===================== LayerNorm(z) (4 lanes per pair row) =====================
    const int r = threadIdx.x - 128;
    int it = 0;
    for (int t = first; t < prm.num_tiles; t += stride, ++it) {
      const int s = it & 1;
      ptx::mbar_wait(full(s), (it >> 1) & 1);
      if (!K3_DBG_SKIP(1))
        layernorm_rows_inplace<kNormFp16, false, 1, kLnzWarps * 32>(smem + kOffStage + s * kStageBytes, kHalfBox,
                                                       r, 0, 0, prm.eps);
      ptx::fence_proxy_async_smem();
      ptx::mbar_arrive(zready(s));
    }
  } else if (warp >= kWarpLno && warp < kWarpEpi) {
    // ===================== LayerNorm(o) on the [channel][pair] tile =====================
    // Warp w8 owns 16 pairs; lane = (channel quarter cq = 32 channels, pair-pair pl).  One
    // ld.shared.b32 = 2 adjacent pairs of one channel, and the thread's 32 words stay in registers
    // (one pass over shared memory, exact two-pass statistics).  The four quarters visit their
    // rows in the order i ^ 2cq, which puts their 32-byte segments under four different swizzle
    // phases: conflict-free.  Statistics combine across the quarters with two shuffles.
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
    int it = 0;
    for (int t = first; t < prm.num_tiles; t += stride, ++it) {
      const int s = it & 1;
      ptx::mbar_wait(full(s), (it >> 1) & 1);
      const uint32_t tile = smem + kOffStage + s * kStageBytes + kMatBytes;
      if (K3_DBG_SKIP(2)) {
        ptx::fence_proxy_async_smem();
        ptx::mbar_arrive(oready(s));
        continue;
      }
      uint32_t w[32];
#pragma unroll
      for (uint32_t g = 0; g < 4; ++g)
#pragma unroll
        for (uint32_t jj = 0; jj < 8; ++jj) w[g * 8 + jj] = ptx::lds32(tile + toff[jj] + g * 1024u);
      ptx::f32x2 sa = ptx::bf16x2_to_f32x2(w[0]), sb = ptx::bf16x2_to_f32x2(w[1]);
#pragma unroll
      for (int i = 2; i < 32; i += 2) {
        sa = ptx::add2(sa, ptx::bf16x2_to_f32x2(w[i]));
        sb = ptx::add2(sb, ptx::bf16x2_to_f32x2(w[i + 1]));
      }
      float s0, s1;
      ptx::upk2(ptx::add2(sa, sb), s0, s1);
      s0 += __shfl_xor_sync(0xffffffffu, s0, 8);
      s1 += __shfl_xor_sync(0xffffffffu, s1, 8);
      s0 += __shfl_xor_sync(0xffffffffu, s0, 16);
      s1 += __shfl_xor_sync(0xffffffffu, s1, 16);
      const float m0 = s0 * (1.0f / kC), m1 = s1 * (1.0f / kC);
      const ptx::f32x2 nm = ptx::pk2(-m0, -m1);
      ptx::f32x2 qa = ptx::pk2(0.f, 0.f), qb = qa;
#pragma unroll
      for (int i = 0; i < 32; i += 2) {
        const ptx::f32x2 d0 = ptx::add2(ptx::bf16x2_to_f32x2(w[i]), nm);
        const ptx::f32x2 d1 = ptx::add2(ptx::bf16x2_to_f32x2(w[i + 1]), nm);
        qa = ptx::fma2(d0, d0, qa);
        qb = ptx::fma2(d1, d1, qb);
      }
      float q0, q1;
      ptx::upk2(ptx::add2(qa, qb), q0, q1);
      q0 += __shfl_xor_sync(0xffffffffu, q0, 8);
      q1 += __shfl_xor_sync(0xffffffffu, q1, 8);
      q0 += __shfl_xor_sync(0xffffffffu, q0, 16);
      q1 += __shfl_xor_sync(0xffffffffu, q1, 16);
      const float r0 = rsqrtf(q0 * (1.0f / kC) + prm.eps), r1 = rsqrtf(q1 * (1.0f / kC) + prm.eps);
      const ptx::f32x2 rr = ptx::pk2(r0, r1);
      const ptx::f32x2 nn = ptx::pk2(-m0 * r0, -m1 * r1);
#pragma unroll
      for (uint32_t g = 0; g < 4; ++g)
#pragma unroll
        for (uint32_t jj = 0; jj < 8; ++jj)
          ptx::sts32(tile + toff[jj] + g * 1024u,
                     ptx::pack_norm2<kNormFp16>(
                         ptx::fma2(ptx::bf16x2_to_f32x2(w[g * 8 + jj]), rr, nn)));
      ptx::fence_proxy_async_smem();
      ptx::mbar_arrive(oready(s));
    }
  } else if (warp >= kWarpEpi) {
    // ===================== epilogue (thread = pair, 64 output channels) =====================
    const int q = warp & 3;                       // TMEM lane quadrant (hardware: warp % 4)
    const int h = (warp - kWarpEpi) >> 2;               // channel half
    const int r = q * 32 + lane;                  // pair within the tile
    const uint32_t stage_buf = smem + kOffOut + h * kHalfBox;
    const uint32_t row_addr = stage_buf + r * 128;
    const uint32_t sw = static_cast<uint32_t>(r & 7);
    const bool store_thread = (q == 0 && lane == 0);
    const uint32_t bar_id = 1 + h;
    constexpr float kLog2e = 1.4426950408889634f;
    constexpr float kGateScale = kTanhSigmoid ? 0.5f : -kLog2e;
    const ptx::f32x2 gscale2 = ptx::pk2(kGateScale, kGateScale);
    const ptx::f32x2 one2 = ptx::pk2(1.0f, 1.0f);
    (void)gscale2;
    (void)one2;
    // folded biases (fp32) of this thread's 64 channels
    const uint32_t tg_addr = smem + kOffVec + h * 64 * 4, to_addr = tg_addr + kC * 4;
    // the pair mask is fetched one tile ahead so that its latency never sits on the critical path
    auto load_mask = [&](int t) -> unsigned short {
      if (prm.mask == nullptr) return static_cast<unsigned short>(0x3f80);   // bf16 1.0
      if (t >= prm.num_tiles) return static_cast<unsigned short>(0);
      const long long p = static_cast<long long>(t) * kTilePairs + r;
      return p < prm.R ? __ldg(reinterpret_cast<const unsigned short*>(prm.mask) + p)
                       : static_cast<unsigned short>(0);
    };
    unsigned short mnext = load_mask(first);
    int it = 0;
    for (int t = first; t < prm.num_tiles; t += stride, ++it) {
      const int slot = it & 1;
      const unsigned short mraw = mnext;
      mnext = load_mask(t + stride);
      ptx::mbar_wait(tfull(slot), (it >> 1) & 1);
      ptx::tc_fence_after();
      const float mval = __uint_as_float(static_cast<uint32_t>(mraw) << 16);
      const ptx::f32x2 mval2 = ptx::pk2(mval, mval);
      const uint32_t taddr = tmem_base + (static_cast<uint32_t>(q * 32) << 16) + slot * 256 + h * 64;
      const long long p = static_cast<long long>(t) * kTilePairs + r;
#pragma unroll
      for (int chunk = 0; chunk < 4; ++chunk) {
        // residual: this pair's 16 raw z channels (the tile was just read by TMA: an L2 hit)
        uint4 zr0 = make_uint4(0u, 0u, 0u, 0u), zr1 = zr0;
        if (prm.z_res != nullptr && p < prm.R) {
          const uint4* zp = reinterpret_cast<const uint4*>(prm.z_res + p * kC + h * 64 + chunk * 16);
          zr0 = __ldg(zp);
          zr1 = __ldg(zp + 1);
        }
        const uint32_t zr[8] = {zr0.x, zr0.y, zr0.z, zr0.w, zr1.x, zr1.y, zr1.z, zr1.w};
        uint32_t vg[16], vo[16];
        ptx::tmem_ld_32x16(taddr + chunk * 16, vg);
        ptx::tmem_ld_32x16(taddr + 128 + chunk * 16, vo);
        ptx::tmem_ld_wait();
        if (chunk == 3) {
          ptx::tc_fence_before();
          __syncwarp();
          if (lane == 0) ptx::mbar_arrive(tempty(slot));
        }
        uint32_t packed[8];
        if (K3_DBG_SKIP(4)) {
#pragma unroll
          for (int i = 0; i < 8; ++i) packed[i] = vo[2 * i] ^ vg[2 * i + 1];
        } else {
#pragma unroll
        for (int j4 = 0; j4 < 4; ++j4) {
          ptx::f32x2 bg2[2], bo2[2];
          ptx::lds128x2(tg_addr + (chunk * 16 + j4 * 4) * 4, bg2);
          ptx::lds128x2(to_addr + (chunk * 16 + j4 * 4) * 4, bo2);
#pragma unroll
          for (int e2 = 0; e2 < 2; ++e2) {
            const int j = j4 * 4 + e2 * 2;
            const ptx::f32x2 zres = ptx::bf16x2_to_f32x2(zr[j4 * 2 + e2]);   // 0 without residual
            const ptx::f32x2 y = ptx::mul2(ptx::add2(ptx::pk2u(vo[j], vo[j + 1]), bo2[e2]), mval2);
            float g0, g1, v0, v1;
            if constexpr (kTanhSigmoid) {
              // y and the gate pre-activation arrive halved: out = (tanh(g/2) + 1) (y/2) [+ z]
              ptx::upk2(ptx::add2(ptx::pk2u(vg[j], vg[j + 1]), bg2[e2]), g0, g1);
              ptx::upk2(ptx::fma2(y, ptx::pk2(ptx::tanh_approx(g0), ptx::tanh_approx(g1)),
                                  ptx::add2(y, zres)), v0, v1);
            } else {
              float d0, d1;
              ptx::upk2(ptx::mul2(ptx::add2(ptx::pk2u(vg[j], vg[j + 1]), bg2[e2]), gscale2), g0, g1);
              ptx::upk2(ptx::add2(ptx::pk2(ptx::ex2_approx(g0), ptx::ex2_approx(g1)), one2), d0, d1);
              ptx::upk2(ptx::fma2(y, ptx::pk2(ptx::rcp_approx(d0), ptx::rcp_approx(d1)), zres), v0, v1);
            }
            packed[j4 * 2 + e2] = ptx::pack_bf16x2(v0, v1);
          }
        }
        }
        if (chunk == 0) {
          if (store_thread) ptx::tma_store_wait_read<0>();
          ptx::named_bar_sync(bar_id, 128);
        }
        ptx::sts128(row_addr + ((static_cast<uint32_t>(chunk * 2) ^ sw) << 4), packed[0], packed[1],
                    packed[2], packed[3]);
        ptx::sts128(row_addr + ((static_cast<uint32_t>(chunk * 2 + 1) ^ sw) << 4), packed[4],
                    packed[5], packed[6], packed[7]);
      }
      ptx::fence_proxy_async_smem();
      ptx::named_bar_sync(bar_id, 128);
      if (store_thread) {
        ptx::tma_store_2d(&tmap_out, stage_buf, h * 64, t * kTilePairs);
        ptx::tma_store_commit();
      }
    }
    if (store_thread) ptx::tma_store_wait<0>();
  }

  // ===================== teardown =====================
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 2) ptx::tmem_dealloc<1>(tmem_base, 512);
}

bool k3_tanh_sigmoid() {
  static const bool v = [] {
    const char* e = debug_env("FOLDCP_K3_SIGMOID");   // "exp" = ex2+rcp (2 MUFU), default tanh (1 MUFU)
    return !(e && e[0] == 'e');
  }();
  return v;
}

}  // namespace

int launch_k3_finalize_bf16(const void* o, const void* z, const void* mask,
                            const foldcp_trimul_params* p, int N, void* out, cudaStream_t stream) {
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
  prm.g_in = p->ln_in_gamma;
  prm.b_in = p->ln_in_beta;
  prm.g_out = p->ln_out_gamma;
  prm.b_out = p->ln_out_beta;
  prm.w_g = static_cast<const __nv_bfloat16*>(p->w_g);
  prm.w_o = static_cast<const __nv_bfloat16*>(p->w_o);
  prm.bias_g = p->b_g;
  prm.bias_o = p->b_o;
  prm.eps = p->ln_eps;
  prm.R = static_cast<long long>(R);
  prm.num_tiles = static_cast<int>((R + kTilePairs - 1) / kTilePairs);
  static const int dbg_skip = [] {
    const char* e = debug_env("FOLDCP_K3_SKIP");
    return e ? atoi(e) : 0;
  }();
  prm.dbg_skip = dbg_skip;
  const int grid = prm.num_tiles < dev.sm_count ? prm.num_tiles : dev.sm_count;
  const bool tanh_sig = k3_tanh_sigmoid();
  auto kern = tanh_sig ? k3_finalize_kernel<true> : k3_finalize_kernel<false>;
  if (ensure_dynamic_smem(reinterpret_cast<const void*>(kern), kSmemBytes) != FOLDCP_OK)
    return FOLDCP_ERR_CUDA;
  kern<<<grid, kThreads, kSmemBytes, stream>>>(tz, to, twg, two, tout, prm);
  return check_launch();
}

}  // namespace foldcp
