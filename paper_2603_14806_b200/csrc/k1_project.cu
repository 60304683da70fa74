// K1 -- input LayerNorm + the four gated projections + pair mask (
// a, b are "projections of the pair representation ... with element-wise
// gating"; north_star / AF3 Alg. 12 lines 1-3):
//
//   z'  = LN(z; gamma_in, beta_in, eps)                     per pair, over the 128 channels
//   a   = M * sigmoid(W_ga z' + b_ga) * (W_a z' + b_a)      b likewise
//
// z is [R = N*N][128] channel-last bf16; a and b are written channel-major [128][R] bf16, which
// is the layout K2's TMA boxes want for both directions.
//
// The GEMM is oriented so that the OUTPUT CHANNEL is the MMA M dimension (TMEM lane) and the
// PAIR is the MMA N dimension (TMEM column):   D[ch][pair] = W[ch][k] * z'[pair][k]^T.
// A thread of the epilogue then owns one channel and a run of consecutive pairs -- exactly a
// contiguous run of the channel-major output -- and the projection and its gate for the same
// (channel, pair) sit in the same thread (two accumulators, same lane, same column).
//
// Persistent kernel, one CTA per SM, 16 warps, tile = 128 pairs:
//   warp 0       TMA producer : weights once (4 x 32 KB, resident), then z tiles into a 2-deep ring
//   warp 1       MMA issuer   : per tile two "units" (a, b), each = projection + gate MMA
//                               (M=128 ch, N=128 pairs, K=128) into one 256-column TMEM slot
//   warp 2       TMEM allocator (512 columns = 2 slots; the epilogue of unit a overlaps the
//                               MMAs of unit b and vice versa)
//   warps 4-7    LayerNorm    : ln_rows.cuh -- z rows (bf16, 128-byte-swizzled TMA tile) ->
//                               registers -> two-pass mean/variance in fp32 -> z' written back in
//                               place as the K-major B operand; also stages the pair mask
//   warps 8-15   epilogue     : tcgen05.ld both accumulators -> bias, sigmoid, gate, mask in
//                               fp32 -> bf16 -> swizzled smem -> TMA store [128 ch][64 pairs]
#include <cuda_bf16.h>

#include "common.h"
#include "ln_rows.cuh"
#include "ptx.cuh"

namespace foldcp {
namespace {

constexpr int kC = kChannels;                   // 128
constexpr int kTilePairs = 128;
constexpr int kThreads = 512;
constexpr int kHalfBox = 128 * 64 * 2;          // 16 KB: one TMA box, 128 rows x 64 bf16
constexpr int kMatBytes = 2 * kHalfBox;         // 32 KB: a 128 x 128 bf16 operand (two k-halves)
constexpr int kZStages = 2;
constexpr int kMaskSlots = 3;

constexpr int kOffW = 0;                                  // 4 weight matrices
constexpr int kOffZ = kOffW + 4 * kMatBytes;              // z ring
constexpr int kOffOut = kOffZ + kZStages * kMatBytes;     // 2 staging buffers [128 ch][64 pairs]
constexpr int kOffGamma = kOffOut + 2 * kHalfBox;
constexpr int kOffBeta = kOffGamma + kC * 4;
constexpr int kOffMask = kOffBeta + kC * 4;
constexpr int kOffBar = kOffMask + kMaskSlots * kTilePairs * 4;
constexpr int kSmemBytes = kOffBar + 128;
static_assert(kSmemBytes <= 232448, "K1 shared memory exceeds 227 KB");

struct K1Params {
  const __nv_bfloat16* mask;   // [R] or nullptr
  const float* gamma;
  const float* beta;
  const float* bias[4];        // b_a, b_ga, b_b, b_gb (each may be nullptr)
  float eps;
  long long R;                 // number of pairs
  int num_tiles;
};

template <bool kTanhSigmoid>
__global__ void __launch_bounds__(kThreads, 1)
k1_project_kernel(const __grid_constant__ CUtensorMap tmap_z,
                  const __grid_constant__ CUtensorMap tmap_w0,
                  const __grid_constant__ CUtensorMap tmap_w1,
                  const __grid_constant__ CUtensorMap tmap_w2,
                  const __grid_constant__ CUtensorMap tmap_w3,
                  const __grid_constant__ CUtensorMap tmap_a,
                  const __grid_constant__ CUtensorMap tmap_b, const K1Params prm) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t smem = ptx::smem_u32(smem_raw);
  if ((smem & 1023u) != 0) __trap();   // 128-byte swizzle needs 1024-byte aligned tiles

  const uint32_t bar = smem + kOffBar;
  const uint32_t wfull = bar;
  auto zfull = [&](int s) { return bar + 8u * (1 + s); };
  auto zempty = [&](int s) { return bar + 8u * (3 + s); };
  auto zready = [&](int s) { return bar + 8u * (5 + s); };
  auto tfull = [&](int u) { return bar + 8u * (7 + u); };
  auto tempty = [&](int u) { return bar + 8u * (9 + u); };
  const uint32_t tmem_slot = bar + 8u * 11;

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(&tmap_z);
    ptx::prefetch_tmap(&tmap_a);
    ptx::prefetch_tmap(&tmap_b);
  }
  if (warp == 1 && lane == 0) {
    ptx::mbar_init(wfull, 1);
    for (int s = 0; s < kZStages; ++s) {
      ptx::mbar_init(zfull(s), 1);
      ptx::mbar_init(zempty(s), 1);
      ptx::mbar_init(zready(s), 128);
    }
    for (int u = 0; u < 2; ++u) {
      ptx::mbar_init(tfull(u), 1);
      ptx::mbar_init(tempty(u), 8);
    }
    ptx::fence_mbar_init();
  }
  if (warp == 2) ptx::tmem_alloc<1>(tmem_slot, 512);
  if (warp == 3) {
    float* g = reinterpret_cast<float*>(smem_raw + kOffGamma);
    float* b = reinterpret_cast<float*>(smem_raw + kOffBeta);
    for (int c = lane; c < kC; c += 32) {
      g[c] = prm.gamma[c];
      b[c] = prm.beta[c];
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  // weights: loaded once per CTA, resident for the whole kernel
  if (warp == 0 && ptx::elect_one()) {
    ptx::mbar_arrive_expect_tx(wfull, 4 * kMatBytes);
    const CUtensorMap* wm[4] = {&tmap_w0, &tmap_w1, &tmap_w2, &tmap_w3};
#pragma unroll
    for (int m = 0; m < 4; ++m) {
      ptx::tma_load_2d(smem + kOffW + m * kMatBytes, wm[m], wfull, 0, 0);
      ptx::tma_load_2d(smem + kOffW + m * kMatBytes + kHalfBox, wm[m], wfull, 64, 0);
    }
  }
  if constexpr (kNormFp16) {
    // kind::f16 needs A and B in the same 16-bit format: the bf16 weights become fp16 in place
    ptx::mbar_wait(wfull, 0);
    ptx::smem_bf16_to_f16_inplace(smem + kOffW, 4 * kMatBytes, threadIdx.x, kThreads);
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
        ptx::mbar_wait(zempty(s), ((it >> 1) & 1) ^ 1u);
        ptx::mbar_arrive_expect_tx(zfull(s), kMatBytes);
        const uint32_t dst = smem + kOffZ + s * kMatBytes;
        const int row0 = t * kTilePairs;          // < 2^31: R <= 2^30 (N <= 32768)
        ptx::tma_load_2d(dst, &tmap_z, zfull(s), 0, row0);
        ptx::tma_load_2d(dst + kHalfBox, &tmap_z, zfull(s), 64, row0);
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (ptx::elect_one()) {
      // A = weights, B = z', both K-major, both fp16 (or both bf16)
      constexpr uint32_t kFmt = kNormFp16 ? ptx::kFmtF16 : ptx::kFmtBF16;
      constexpr uint32_t idesc = ptx::make_idesc_f16kind(128, kTilePairs, kFmt, kFmt, 0, 0);
      ptx::mbar_wait(wfull, 0);
      int it = 0;
      for (int t = first; t < prm.num_tiles; t += stride, ++it) {
        const int s = it & 1;
        ptx::mbar_wait(zready(s), (it >> 1) & 1);
        ptx::tc_fence_after();
        const uint32_t zb = smem + kOffZ + s * kMatBytes;
#pragma unroll
        for (int u = 0; u < 2; ++u) {
          ptx::mbar_wait(tempty(u), (it & 1) ^ 1u);
          ptx::tc_fence_after();
#pragma unroll
          for (int m2 = 0; m2 < 2; ++m2) {
            const uint32_t wa = smem + kOffW + (2 * u + m2) * kMatBytes;
            const uint32_t d_tmem = tmem_base + u * 256 + m2 * 128;
#pragma unroll
            for (int k = 0; k < 8; ++k) {
              const uint32_t off = (k >> 2) * kHalfBox + (k & 3) * 32;
              const uint64_t da = ptx::make_smem_desc_sw128(wa + off, 16, 1024);
              const uint64_t db = ptx::make_smem_desc_sw128(zb + off, 16, 1024);
              ptx::umma_bf16<1>(d_tmem, da, db, idesc, k != 0 ? 1u : 0u);
            }
          }
          ptx::umma_commit<1>(tfull(u));
        }
        ptx::umma_commit<1>(zempty(s));   // z' stage reusable once all four MMAs retired
      }
    }
  } else if (warp >= 4 && warp < 8) {
    // ===================== LayerNorm (thread = pair) =====================
    const int r = threadIdx.x - 128;
    const uint32_t gaddr = smem + kOffGamma, baddr = smem + kOffBeta;
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
      const int s = it & 1;
      const unsigned short mraw = mnext;
      mnext = load_mask(t + stride);
      ptx::mbar_wait(zfull(s), (it >> 1) & 1);
      layernorm_rows_inplace<kNormFp16>(smem + kOffZ + s * kMatBytes, kHalfBox, r, gaddr, baddr, prm.eps);
      reinterpret_cast<float*>(smem_raw + kOffMask)[(it % kMaskSlots) * kTilePairs + r] =
          __uint_as_float(static_cast<uint32_t>(mraw) << 16);
      ptx::fence_proxy_async_smem();
      ptx::mbar_arrive(zready(s));
    }
  } else if (warp >= 8) {
    // ===================== epilogue =====================
    // warp -> TMEM lane quadrant q (hardware rule: warp % 4) and column half h (64 pairs)
    const int q = warp & 3;
    const int h = (warp - 8) >> 2;
    const int ch = q * 32 + lane;                       // output channel = TMEM lane
    const uint32_t stage_buf = smem + kOffOut + h * kHalfBox;
    const uint32_t row_addr = stage_buf + ch * 128;
    const uint32_t sw = static_cast<uint32_t>(ch & 7);
    const bool store_thread = (q == 0 && lane == 0);
    const uint32_t bar_id = 1 + h;
    constexpr float kLog2e = 1.4426950408889634f;
    // packed fp32x2 constants: sigmoid(x) = 0.5 tanh(0.5 x) + 0.5  or  1 / (1 + 2^(-x log2 e))
    constexpr float kGateScale = kTanhSigmoid ? 0.5f : -kLog2e;
    const ptx::f32x2 gscale2 = ptx::pk2(kGateScale, kGateScale);
    const ptx::f32x2 half2 = ptx::pk2(0.5f, 0.5f), one2 = ptx::pk2(1.0f, 1.0f);
    (void)half2;
    (void)one2;
    ptx::f32x2 bias_p2[2], bias_g2[2];
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      const float bp = prm.bias[2 * u] ? prm.bias[2 * u][ch] : 0.f;
      const float bg = kGateScale * (prm.bias[2 * u + 1] ? prm.bias[2 * u + 1][ch] : 0.f);
      bias_p2[u] = ptx::pk2(bp, bp);
      bias_g2[u] = ptx::pk2(bg, bg);
    }
    int it = 0;
    for (int t = first; t < prm.num_tiles; t += stride, ++it) {
      const uint32_t mask_addr =
          smem + kOffMask + ((it % kMaskSlots) * kTilePairs + h * 64) * 4;
      const int p0 = t * kTilePairs + h * 64;
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        ptx::mbar_wait(tfull(u), it & 1);
        ptx::tc_fence_after();
        const uint32_t taddr =
            tmem_base + (static_cast<uint32_t>(q * 32) << 16) + u * 256 + h * 64;
        // 64 columns per warp and unit, in four chunks of 16; the tcgen05.ld of chunk c+1 is in
        // flight while chunk c is being computed (two register buffers)
        uint32_t vp[2][16], vg[2][16];
        ptx::tmem_ld_32x16(taddr, vp[0]);
        ptx::tmem_ld_32x16(taddr + 128, vg[0]);
#pragma unroll
        for (int chunk = 0; chunk < 4; ++chunk) {
          const int cb = chunk & 1;
          ptx::tmem_ld_wait();
          if (chunk < 3) {
            ptx::tmem_ld_32x16(taddr + (chunk + 1) * 16, vp[cb ^ 1]);
            ptx::tmem_ld_32x16(taddr + 128 + (chunk + 1) * 16, vg[cb ^ 1]);
          }
          uint32_t packed[8];
#pragma unroll
          for (int j4 = 0; j4 < 4; ++j4) {
            ptx::f32x2 m2[2];
            ptx::lds128x2(mask_addr + (chunk * 16 + j4 * 4) * 4, m2);
#pragma unroll
            for (int e2 = 0; e2 < 2; ++e2) {
              const int j = j4 * 4 + e2 * 2;
              const ptx::f32x2 pj = ptx::add2(ptx::pk2u(vp[cb][j], vp[cb][j + 1]), bias_p2[u]);
              const ptx::f32x2 gx =
                  ptx::fma2(ptx::pk2u(vg[cb][j], vg[cb][j + 1]), gscale2, bias_g2[u]);
              float g0, g1;
              ptx::upk2(gx, g0, g1);
              ptx::f32x2 sg;
              if constexpr (kTanhSigmoid) {
                sg = ptx::fma2(ptx::pk2(ptx::tanh_approx(g0), ptx::tanh_approx(g1)), half2, half2);
              } else {
                float d0, d1;
                ptx::upk2(ptx::add2(ptx::pk2(ptx::ex2_approx(g0), ptx::ex2_approx(g1)), one2), d0, d1);
                sg = ptx::pk2(ptx::rcp_approx(d0), ptx::rcp_approx(d1));
              }
              float v0, v1;
              ptx::upk2(ptx::mul2(ptx::mul2(pj, m2[e2]), sg), v0, v1);
              packed[j4 * 2 + e2] = ptx::pack_bf16x2(v0, v1);
            }
          }
          if (chunk == 3) {
            // accumulators and mask slot fully consumed: hand the TMEM slot back to the issuer
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(tempty(u));
          }
          if (chunk == 0) {
            // the previous unit's TMA store must have finished reading the staging buffer
            if (store_thread) ptx::tma_store_wait_read<0>();
            ptx::named_bar_sync(bar_id, 128);
          }
          ptx::sts128(row_addr + ((static_cast<uint32_t>(chunk * 2) ^ sw) << 4), packed[0],
                      packed[1], packed[2], packed[3]);
          ptx::sts128(row_addr + ((static_cast<uint32_t>(chunk * 2 + 1) ^ sw) << 4), packed[4],
                      packed[5], packed[6], packed[7]);
        }
        ptx::fence_proxy_async_smem();
        ptx::named_bar_sync(bar_id, 128);
        if (store_thread) {
          ptx::tma_store_2d(u == 0 ? &tmap_a : &tmap_b, stage_buf, p0, 0);
          ptx::tma_store_commit();
        }
      }
    }
    if (store_thread) ptx::tma_store_wait<0>();
  }

  // ===================== teardown =====================
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 2) ptx::tmem_dealloc<1>(tmem_base, 512);
}

bool k1_tanh_sigmoid() {
  static const bool v = [] {
    const char* e = getenv("FOLDCP_K1_SIGMOID");   // "exp" = ex2+rcp (2 MUFU), default tanh (1 MUFU)
    return !(e && e[0] == 'e');
  }();
  return v;
}

}  // namespace

int launch_k1_project_bf16(const void* z, const void* mask, const foldcp_trimul_params* p, int N,
                           void* a, void* b, cudaStream_t stream) {
  DeviceInfo dev;
  if (!get_device_info(&dev)) return FOLDCP_ERR_CUDA;
  const uint64_t R = static_cast<uint64_t>(N) * N;
  CUtensorMap tz, tw[4], ta, tb;
  int st;
  {
    const uint64_t dims[2] = {kC, R};
    const uint64_t strides[1] = {kC * 2};
    const uint32_t box[2] = {64, 128};
    if ((st = encode_tensor_map(&tz, z, 2, 2, dims, strides, box, true)) != FOLDCP_OK) return st;
  }
  {
    const uint64_t dims[2] = {kC, kC};
    const uint64_t strides[1] = {kC * 2};
    const uint32_t box[2] = {64, 128};
    const void* w[4] = {p->w_a, p->w_a_gate, p->w_b, p->w_b_gate};
    for (int m = 0; m < 4; ++m)
      if ((st = encode_tensor_map(&tw[m], w[m], 2, 2, dims, strides, box, true)) != FOLDCP_OK)
        return st;
  }
  {
    const uint64_t dims[2] = {R, kC};
    const uint64_t strides[1] = {R * 2};
    const uint32_t box[2] = {64, 128};
    if ((st = encode_tensor_map(&ta, a, 2, 2, dims, strides, box, true)) != FOLDCP_OK) return st;
    if ((st = encode_tensor_map(&tb, b, 2, 2, dims, strides, box, true)) != FOLDCP_OK) return st;
  }
  K1Params prm;
  prm.mask = static_cast<const __nv_bfloat16*>(mask);
  prm.gamma = p->ln_in_gamma;
  prm.beta = p->ln_in_beta;
  prm.bias[0] = p->b_a;
  prm.bias[1] = p->b_a_gate;
  prm.bias[2] = p->b_b;
  prm.bias[3] = p->b_b_gate;
  prm.eps = p->ln_eps;
  prm.R = static_cast<long long>(R);
  prm.num_tiles = static_cast<int>((R + kTilePairs - 1) / kTilePairs);
  const int grid = prm.num_tiles < dev.sm_count ? prm.num_tiles : dev.sm_count;
  const bool tanh_sig = k1_tanh_sigmoid();
  auto kern = tanh_sig ? k1_project_kernel<true> : k1_project_kernel<false>;
  static bool attr_set[2] = {false, false};
  if (!attr_set[tanh_sig]) {
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes) !=
        cudaSuccess)
      return FOLDCP_ERR_CUDA;
    attr_set[tanh_sig] = true;
  }
  kern<<<grid, kThreads, kSmemBytes, stream>>>(tz, tw[0], tw[1], tw[2], tw[3], ta, tb, prm);
  return check_launch();
}

}  // namespace foldcp
