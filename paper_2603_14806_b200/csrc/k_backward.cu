// Backward pass around the contraction on tcgen05 (bf16 mode; PAPER.md lines
// 92-96: every Fold-CP module hand-writes its backward with the forward's algorithm).  The fp32
// exact mode uses the CUDA-core kernels of simt_backward.cu; the gradients of Eq. 2-3 themselves run
// on the contraction kernel (k2_contract.cu).
//
//   K3-backward  (kPass = 0)   d_out, z, o  ->  d_o (in place over o), the gate's share of d_zhat,
//                              Acc_g = sum d_gg^T zhat, Acc_o = sum d_y^T ohat, db_g, db_o
//   K1-backward  (kPass = 1/2) d_a (pass 1) or d_b (pass 2), z  ->  d_zhat += ..., Acc / db of the
//                              projection and its gate; pass 2 closes with the LayerNorm(z)
//                              backward and writes d_z
//
// The LayerNorm affines are folded exactly as in the forward kernels: with xhat = (x - mean) rstd,
//     W LN(x) + b = (W diag(gamma)) xhat + (W beta + b)
// so one resident matrix W' = W diag(gamma) (bf16, [t][k]) serves
//     the forward product      pre[p][t]  = sum_k xhat[p][k] W'[t][k]     (B operand, K-major)
//     the data gradient        d_xhat[p][k] = sum_t d_pre[p][t] W'[t][k]  (B operand, MN-major)
// and the parameter gradients follow from ONE accumulated matrix per projection,
//     Acc[t][k] = sum_pairs d_pre[p][t] xhat[p][k]   (A = d_pre tile MN-major, B = xhat tile):
//     dW[t][k]   = Acc[t][k] gamma[k] + db[t] beta[k]          db[t] = sum_pairs d_pre[p][t]
//     dgamma[k]  = sum_t W[t][k] Acc[t][k]                     dbeta[k] = sum_t W[t][k] db[t]
// (assemble_param_grads_kernel, fixed summation order => bitwise reproducible).  Acc lives in
// tensor memory for the whole kernel; tiles are assigned statically so that every CTA's partial
// sums do not depend on scheduling.
//
// Kernel shape: persistent, 256 threads, tile = 128 pairs, bulk-synchronous phases per tile
// (TMA loads -> LayerNorm -> MMA 1 -> gate / chain-rule epilogue -> MMA 2 + 3 -> LayerNorm-backward
// epilogue -> stores).  No warp specialisation: this path trades overlap for simplicity; it is
// ~40x faster than the CUDA-core tail and within ~2x of its HBM traffic floor.
// All operand tiles are bf16 (gradients need bf16's range; tcgen05 kind::f16 wants one format).
#include <cuda_bf16.h>

#include "common.h"
#include "ptx.cuh"

namespace foldcp {
namespace {

constexpr int kC = kChannels;            // 128
constexpr int kTilePairs = 128;
constexpr int kThreads = 256;
constexpr int kHalfBox = 128 * 64 * 2;   // 16 KB: one TMA box, 128 rows x 128 bytes
constexpr int kMat = 2 * kHalfBox;       // 32 KB: a 128 x 128 16-bit tile

constexpr int kOffW0 = 0;                // W0' [t][k]
constexpr int kOffW1 = kMat;             // W1' [t][k]
constexpr int kOffZT = 2 * kMat;         // z tile -> zhat            [p][k]
constexpr int kOffXT = 3 * kMat;         // K3: o tile -> ohat -> d_o [k][p];  K1: d_a / d_b tile [t][p]
constexpr int kOffGT = 4 * kMat;         // K3: d_out -> d_y          [p][t];  K1: d_p     [p][t]
constexpr int kOffHT = 5 * kMat;         // K3: d_gg                  [p][t];  K1: d_gate  [p][t]
constexpr int kOffVec = 6 * kMat;        // fp32: t0[128] t1[128] rstd0[128] rstd1[128] mask[128]
constexpr int kOffBar = kOffVec + 5 * kC * 4;
constexpr int kSmemBytes = kOffBar + 64;
static_assert(kSmemBytes <= 232448, "backward tail shared memory exceeds 227 KB");

constexpr int kTmemD0 = 0, kTmemD1 = 128, kTmemAcc0 = 256, kTmemAcc1 = 384;

// per-CTA record written at the end of a launch: Acc0 [t][k], Acc1 [t][k], db0 [t], db1 [t]
constexpr int kRecFloats = 2 * kC * kC + 2 * kC;

struct TailParams {
  const __nv_bfloat16* mask;    // [R] or nullptr (K3: nullptr when mask_output == 0)
  const __nv_bfloat16* w0;      // raw weights [t][k] (K3: W_g, W_o; K1: W, W_gate)
  const __nv_bfloat16* w1;
  const float* bias0;           // may be nullptr
  const float* bias1;
  const float* gamma0;          // LayerNorm affine folded into w0 (always ln_in)
  const float* beta0;
  const float* gamma1;          // folded into w1 (K3: ln_out; K1: ln_in)
  const float* beta1;
  float eps;
  long long R;
  int num_tiles;
  int add_residual;             // K1 final pass: d_z += d_out
  float* dzp;                   // [R][128] fp32 accumulator of d_zhat
  const __nv_bfloat16* d_out;   // [R][128] (K1 final pass, residual only)
  __nv_bfloat16* d_z;           // [R][128] (K1 final pass)
  float* rec;                   // [grid][kRecFloats]
};

__device__ __forceinline__ float sigmoid_fast(float x) {
  return ptx::rcp_approx(1.0f + ptx::ex2_approx(-1.4426950408889634f * x));
}

// address of element (row, col) of a [128 rows][128 cols] 16-bit tile stored as two 128-byte-
// swizzled TMA boxes (cols 0..63 | 64..127)
__device__ __forceinline__ uint32_t tile_addr(uint32_t tile, uint32_t row, uint32_t col) {
  const uint32_t box = col >> 6, c = col & 63u;
  return tile + box * kHalfBox + row * 128u + ((((c >> 3) ^ (row & 7u))) << 4) + (c & 7u) * 2u;
}

// All elements (row = 0..127) of ONE column of such a tile: the eight swizzle phases are folded into
// eight per-thread offsets once, so that an access costs one add (row = 8 g + j -> g * 1024 + off[j]).
struct ColAccess {
  uint32_t base;
  uint32_t off[8];
  __device__ __forceinline__ ColAccess(uint32_t tile, uint32_t col) {
    const uint32_t c = col & 63u;
    base = tile + (col >> 6) * kHalfBox + (c & 7u) * 2u;
#pragma unroll
    for (uint32_t j = 0; j < 8; ++j) off[j] = j * 128u + (((c >> 3) ^ j) << 4);
  }
  // row must be a compile-time expression modulo 8 for the offset to stay in a register
  __device__ __forceinline__ uint32_t addr(uint32_t row) const {
    return base + (row >> 3) * 1024u + off[row & 7u];
  }
};

__device__ __forceinline__ float lds_bf16(uint32_t addr) {
  unsigned short v;
  asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(addr));
  return __uint_as_float(static_cast<uint32_t>(v) << 16);
}
__device__ __forceinline__ void sts_bf16(uint32_t addr, float x) {
  const unsigned short v = __bfloat16_as_ushort(__float2bfloat16_rn(x));
  asm volatile("st.shared.u16 [%0], %1;" ::"r"(addr), "h"(v) : "memory");
}

// LayerNorm statistics + normalisation of a pair-major tile [128 pairs][128 ch] in place (bf16):
// two threads per row (64 channels each), exact two-pass statistics in fp32, xhat written back.
// rstd of every row goes to rstd_out[row] (shared memory).
__device__ __forceinline__ void normalise_rows(uint32_t tile, int tid, float eps, float* rstd_out) {
  const uint32_t row = static_cast<uint32_t>(tid >> 1), h = static_cast<uint32_t>(tid & 1);
  const uint32_t base = tile + h * kHalfBox + row * 128u;
  float x[64];
#pragma unroll
  for (uint32_t i = 0; i < 8; ++i) {
    uint32_t w[4];
    ptx::lds128(base + (((i ^ (4u * h)) ^ (row & 7u)) << 4), w);   // logical chunk i ^ 4h
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      x[i * 8 + 2 * e] = ptx::bf16_lo(w[e]);
      x[i * 8 + 2 * e + 1] = ptx::bf16_hi(w[e]);
    }
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < 64; ++i) s += x[i];
  s += __shfl_xor_sync(0xffffffffu, s, 1);
  const float mu = s * (1.0f / kC);
  float v = 0.f;
#pragma unroll
  for (int i = 0; i < 64; ++i) v = fmaf(x[i] - mu, x[i] - mu, v);
  v += __shfl_xor_sync(0xffffffffu, v, 1);
  const float rstd = rsqrtf(v * (1.0f / kC) + eps);
  if (h == 0) rstd_out[row] = rstd;
#pragma unroll
  for (uint32_t i = 0; i < 8; ++i) {
    uint32_t w[4];
#pragma unroll
    for (int e = 0; e < 4; ++e)
      w[e] = ptx::pack_bf16x2((x[i * 8 + 2 * e] - mu) * rstd, (x[i * 8 + 2 * e + 1] - mu) * rstd);
    ptx::sts128(base + (((i ^ (4u * h)) ^ (row & 7u)) << 4), w[0], w[1], w[2], w[3]);
  }
}

// The same for a channel-major tile [128 ch][128 pairs] (K2's output layout): statistics over the
// ROWS for every column.  Thread = 1 pair x 64 channels (two threads per pair).
__device__ __forceinline__ void normalise_cols(uint32_t tile, int tid, float eps, float* rstd_out) {
  const uint32_t p = static_cast<uint32_t>(tid & 127), h = static_cast<uint32_t>(tid >> 7);
  const ColAccess col(tile, p);
  const uint32_t hb = h * 64u * 128u;                 // rows 64 h ..: 64 rows of 128 bytes
  float x[64];
#pragma unroll
  for (uint32_t i = 0; i < 64; ++i) x[i] = lds_bf16(col.addr(i) + hb);
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < 64; ++i) s += x[i];
  // the partner thread (other channel half of the same pair) sits 128 threads away: via smem
  __shared__ float xch[2][2][128];
  xch[0][h][p] = s;
  __syncthreads();
  const float mu = (xch[0][0][p] + xch[0][1][p]) * (1.0f / kC);
  float v = 0.f;
#pragma unroll
  for (int i = 0; i < 64; ++i) v = fmaf(x[i] - mu, x[i] - mu, v);
  xch[1][h][p] = v;
  __syncthreads();
  const float rstd = rsqrtf((xch[1][0][p] + xch[1][1][p]) * (1.0f / kC) + eps);
  if (h == 0) rstd_out[p] = rstd;
  const float nm = -mu * rstd;
#pragma unroll
  for (uint32_t i = 0; i < 64; ++i) sts_bf16(col.addr(i) + hb, fmaf(x[i], rstd, nm));
}

// D[tmem] (+)= A * B for 128 x 128 x 128 operand tiles of the four layouts used here.
//   a_kmajor: A tile is [m rows][K contiguous]; else [K rows][m contiguous] (MN-major)
//   b_kmajor: B tile is [n rows][K contiguous]; else [K rows][n contiguous] (MN-major)
__device__ __forceinline__ void mma_128(uint32_t d_tmem, uint32_t a_tile, bool a_kmajor,
                                        uint32_t b_tile, bool b_kmajor, bool accumulate_first) {
  const uint32_t idesc = ptx::make_idesc_f16kind(128, 128, ptx::kFmtBF16, ptx::kFmtBF16,
                                                 a_kmajor ? 0 : 1, b_kmajor ? 0 : 1);
#pragma unroll
  for (uint32_t k = 0; k < 8; ++k) {
    const uint32_t koff = (k >> 2) * kHalfBox + (k & 3u) * 32u;   // K-major: 16 K elements = 32 B
    const uint64_t da = a_kmajor ? ptx::make_smem_desc_sw128(a_tile + koff, 16, 1024)
                                 : ptx::make_smem_desc_sw128(a_tile + k * 2048u, kHalfBox, 1024);
    const uint64_t db = b_kmajor ? ptx::make_smem_desc_sw128(b_tile + koff, 16, 1024)
                                 : ptx::make_smem_desc_sw128(b_tile + k * 2048u, kHalfBox, 1024);
    ptx::umma_bf16<1>(d_tmem, da, db, idesc, (accumulate_first || k != 0) ? 1u : 0u);
  }
}

// kPass: 0 = K3-backward, 1 = K1-backward for a (accumulates into dzp), 2 = K1-backward for b
// (final: LayerNorm(z) backward, writes d_z)
template <int kPass>
__global__ void __launch_bounds__(kThreads, 1)
tail_backward_kernel(const __grid_constant__ CUtensorMap tmap_z,     // z   [R][128]
                     const __grid_constant__ CUtensorMap tmap_x,     // K3: o / d_o [128][R]; K1: d_a / d_b
                     const __grid_constant__ CUtensorMap tmap_g,     // K3: d_out [R][128]; K1: unused
                     const __grid_constant__ CUtensorMap tmap_w0,
                     const __grid_constant__ CUtensorMap tmap_w1, const TailParams prm) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t smem = ptx::smem_u32(smem_raw);
  if ((smem & 1023u) != 0) __trap();
  float* vec = reinterpret_cast<float*>(smem_raw + kOffVec);
  float* t0 = vec;                 // folded bias of matrix 0
  float* t1 = vec + kC;
  float* rstd_z = vec + 2 * kC;
  float* rstd_o = vec + 3 * kC;
  float* msk = vec + 4 * kC;
  const uint32_t load_bar = smem + kOffBar, mma_bar = load_bar + 8, w_bar = load_bar + 16;
  const uint32_t tmem_slot = load_bar + 24;

  const int tid = threadIdx.x;
  const int warp = tid >> 5, lane = tid & 31;

  if (tid == 0) {
    ptx::prefetch_tmap(&tmap_z);
    ptx::prefetch_tmap(&tmap_x);
    if (kPass == 0) ptx::prefetch_tmap(&tmap_g);
    ptx::mbar_init(load_bar, 1);
    ptx::mbar_init(mma_bar, 1);
    ptx::mbar_init(w_bar, 1);
    ptx::fence_mbar_init();
  }
  if (warp == 1) ptx::tmem_alloc<1>(tmem_slot, 512);
  {
    // folded biases  W beta + b  (fp32, from the raw bf16 weights)
    const int m = tid >> 7, ch = tid & 127;
    const uint4* wrow = reinterpret_cast<const uint4*>((m ? prm.w1 : prm.w0) + ch * kC);
    const float* beta = m ? prm.beta1 : prm.beta0;
    const float* bias = m ? prm.bias1 : prm.bias0;
    float acc = 0.f;
#pragma unroll 4
    for (int kc = 0; kc < 16; ++kc) {
      const uint4 wv = __ldg(wrow + kc);
      const uint32_t ww[4] = {wv.x, wv.y, wv.z, wv.w};
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        acc = fmaf(ptx::bf16_lo(ww[e]), __ldg(beta + kc * 8 + 2 * e), acc);
        acc = fmaf(ptx::bf16_hi(ww[e]), __ldg(beta + kc * 8 + 2 * e + 1), acc);
      }
    }
    (m ? t1 : t0)[ch] = acc + (bias ? bias[ch] : 0.f);
  }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  // resident weights: W' = W diag(gamma), bf16, in place under the swizzle
  if (tid == 0) {
    ptx::mbar_arrive_expect_tx(w_bar, 2 * kMat);
    ptx::tma_load_2d(smem + kOffW0, &tmap_w0, w_bar, 0, 0);
    ptx::tma_load_2d(smem + kOffW0 + kHalfBox, &tmap_w0, w_bar, 64, 0);
    ptx::tma_load_2d(smem + kOffW1, &tmap_w1, w_bar, 0, 0);
    ptx::tma_load_2d(smem + kOffW1 + kHalfBox, &tmap_w1, w_bar, 64, 0);
  }
  ptx::mbar_wait(w_bar, 0);
  for (int off = tid * 16; off < 2 * kMat; off += kThreads * 16) {
    const int m = off / kMat, rem = off % kMat;
    const int box = rem / kHalfBox, row = (rem % kHalfBox) / 128, pc = (rem % 128) / 16;
    const int k0 = box * 64 + ((pc ^ (row & 7)) * 8);
    const float* gam = (m ? prm.gamma1 : prm.gamma0) + k0;
    uint32_t v[4];
    ptx::lds128(smem + kOffW0 + off, v);
#pragma unroll
    for (int e = 0; e < 4; ++e)
      v[e] = ptx::pack_bf16x2(ptx::bf16_lo(v[e]) * __ldg(gam + 2 * e),
                              ptx::bf16_hi(v[e]) * __ldg(gam + 2 * e + 1));
    ptx::sts128(smem + kOffW0 + off, v[0], v[1], v[2], v[3]);
  }
  ptx::fence_proxy_async_smem();
  __syncthreads();

  const uint32_t ZT = smem + kOffZT, XT = smem + kOffXT, GT = smem + kOffGT, HT = smem + kOffHT;
  const uint32_t W0 = smem + kOffW0, W1 = smem + kOffW1;
  const int q = warp & 3;                       // TMEM lane quadrant of this warp
  const int h = warp >> 2;                      // column half handled in the first epilogue
  const int r = q * 32 + lane;                  // pair (row of the tile) = TMEM lane
  const uint32_t lane_base = tmem_base + (static_cast<uint32_t>(q * 32) << 16);
  float db_acc = 0.f;                           // thread tid: column tid & 127 of GT (tid < 128) / HT
  uint32_t mma_phase = 0;

  int it = 0;
  for (int t = blockIdx.x; t < prm.num_tiles; t += gridDim.x, ++it) {
    const int p0 = t * kTilePairs;
    // ---------------- loads
    if (tid == 0) {
      if (kPass == 0) ptx::tma_store_wait_read<0>();        // last tile's d_o store has read XT
      ptx::mbar_arrive_expect_tx(load_bar, (kPass == 0 ? 3 : 2) * kMat);
      ptx::tma_load_2d(ZT, &tmap_z, load_bar, 0, p0);
      ptx::tma_load_2d(ZT + kHalfBox, &tmap_z, load_bar, 64, p0);
      ptx::tma_load_2d(XT, &tmap_x, load_bar, p0, 0);
      ptx::tma_load_2d(XT + kHalfBox, &tmap_x, load_bar, p0 + 64, 0);
      if (kPass == 0) {
        ptx::tma_load_2d(GT, &tmap_g, load_bar, 0, p0);
        ptx::tma_load_2d(GT + kHalfBox, &tmap_g, load_bar, 64, p0);
      }
    }
    if (tid < kTilePairs) {
      const long long p = static_cast<long long>(p0) + tid;
      float mv = 0.f;
      if (p < prm.R)
        mv = prm.mask ? __bfloat162float(prm.mask[p]) : 1.0f;
      msk[tid] = mv;
    }
    ptx::mbar_wait(load_bar, it & 1);
    // ---------------- LayerNorm statistics, normalised tiles in place
    normalise_rows(ZT, tid, prm.eps, rstd_z);
    if (kPass == 0) normalise_cols(XT, tid, prm.eps, rstd_o);
    ptx::fence_proxy_async_smem();
    ptx::tc_fence_before();
    __syncthreads();
    // ---------------- MMA 1: forward products (recomputation)
    if (tid == 0) {
      ptx::tc_fence_after();
      mma_128(tmem_base + kTmemD0, ZT, true, W0, true, false);            // zhat W0'^T
      if (kPass == 0)
        mma_128(tmem_base + kTmemD1, XT, false, W1, true, false);         // ohat (MN-major A) W_o'^T
      else
        mma_128(tmem_base + kTmemD1, ZT, true, W1, true, false);          // zhat W_gate'^T
      ptx::umma_commit<1>(mma_bar);
    }
    ptx::mbar_wait(mma_bar, mma_phase);
    mma_phase ^= 1u;
    ptx::tc_fence_after();
    // ---------------- epilogue 1: chain rule through gate / projection; thread = (pair r, half h)
    {
      const float mv = msk[r];
      const ColAccess xcol(XT, static_cast<uint32_t>(r));
      (void)xcol;
#pragma unroll 1
      for (int chunk = 0; chunk < 4; ++chunk) {
        const int c0 = h * 64 + chunk * 16;
        uint32_t v0[16], v1[16];
        ptx::tmem_ld_32x16(lane_base + kTmemD0 + c0, v0);
        ptx::tmem_ld_32x16(lane_base + kTmemD1 + c0, v1);
        ptx::tmem_ld_wait();
        float up[16];                                   // upstream gradient of this (pair, channel)
        if (kPass == 0) {
          uint32_t w[4];
#pragma unroll
          for (int half8 = 0; half8 < 2; ++half8) {
            ptx::lds128(tile_addr(GT, r, c0 + half8 * 8), w);
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              up[half8 * 8 + 2 * e] = ptx::bf16_lo(w[e]) * mv;
              up[half8 * 8 + 2 * e + 1] = ptx::bf16_hi(w[e]) * mv;
            }
          }
        } else {
#pragma unroll
          for (int j = 0; j < 16; ++j)
            up[j] = lds_bf16(xcol.addr(j) + static_cast<uint32_t>(c0) * 128u) * mv;   // c0 % 16 == 0
        }
        uint32_t pg[8], ph[8];
#pragma unroll
        for (int j = 0; j < 16; j += 2) {
          float g_out[2], h_out[2];
#pragma unroll
          for (int e = 0; e < 2; ++e) {
            const float pre0 = __uint_as_float(v0[j + e]) + t0[c0 + j + e];
            const float pre1 = __uint_as_float(v1[j + e]) + t1[c0 + j + e];
            if (kPass == 0) {
              // out = M g y, g = sigmoid(pre0), y = pre1:  d_y = up g,  d_gg = up y g (1 - g)
              const float g = sigmoid_fast(pre0);
              g_out[e] = up[j + e] * g;                          // d_y   -> GT
              h_out[e] = up[j + e] * pre1 * g * (1.0f - g);      // d_gg  -> HT
            } else {
              // t = M s p, p = pre0, s = sigmoid(pre1):  d_p = up s,  d_gate = up p s (1 - s)
              const float s = sigmoid_fast(pre1);
              g_out[e] = up[j + e] * s;                          // d_p    -> GT
              h_out[e] = up[j + e] * pre0 * s * (1.0f - s);      // d_gate -> HT
            }
          }
          pg[j >> 1] = ptx::pack_bf16x2(g_out[0], g_out[1]);
          ph[j >> 1] = ptx::pack_bf16x2(h_out[0], h_out[1]);
        }
        ptx::sts128(tile_addr(GT, r, c0), pg[0], pg[1], pg[2], pg[3]);
        ptx::sts128(tile_addr(GT, r, c0 + 8), pg[4], pg[5], pg[6], pg[7]);
        ptx::sts128(tile_addr(HT, r, c0), ph[0], ph[1], ph[2], ph[3]);
        ptx::sts128(tile_addr(HT, r, c0 + 8), ph[4], ph[5], ph[6], ph[7]);
      }
    }
    ptx::tc_fence_before();
    ptx::fence_proxy_async_smem();
    __syncthreads();
    // ---------------- MMA 2 (data gradients) and MMA 3 (parameter-gradient accumulators)
    if (tid == 0) {
      ptx::tc_fence_after();
      const bool acc = it != 0;
      if (kPass == 0) {
        mma_128(tmem_base + kTmemD0, GT, true, W1, false, false);        // d_ohat  = d_y  W_o'
        mma_128(tmem_base + kTmemD1, HT, true, W0, false, false);        // d_zhat  = d_gg W_g'
        mma_128(tmem_base + kTmemAcc0, HT, false, ZT, false, acc);       // Acc_g  += d_gg^T zhat
        mma_128(tmem_base + kTmemAcc1, GT, false, XT, true, acc);        // Acc_o  += d_y^T  ohat
      } else {
        mma_128(tmem_base + kTmemD0, GT, true, W0, false, false);        // d_zhat  = d_p W'
        mma_128(tmem_base + kTmemD0, HT, true, W1, false, true);         //         + d_gate W_gate'
        mma_128(tmem_base + kTmemAcc0, GT, false, ZT, false, acc);       // Acc    += d_p^T zhat
        mma_128(tmem_base + kTmemAcc1, HT, false, ZT, false, acc);       // Acc_gt += d_gate^T zhat
      }
      ptx::umma_commit<1>(mma_bar);
    }
    // bias gradients: column sums of GT (threads 0..127) and HT (128..255) over the tile's pairs
    {
      const ColAccess col(tid < 128 ? GT : HT, static_cast<uint32_t>(tid & 127));
      float s0 = 0.f, s1 = 0.f;
#pragma unroll
      for (uint32_t p = 0; p < 128; p += 2) {
        s0 += lds_bf16(col.addr(p));
        s1 += lds_bf16(col.addr(p + 1));
      }
      db_acc += s0 + s1;
    }
    ptx::mbar_wait(mma_bar, mma_phase);
    mma_phase ^= 1u;
    ptx::tc_fence_after();
    // ---------------- epilogue 2
    if (kPass == 0) {
      if (warp < 4) {
        // d_o = rstd (d_ohat - mean(d_ohat) - ohat mean(d_ohat ohat)), written over ohat [k][p]
        float m1 = 0.f, m2 = 0.f;
        const ColAccess ocol(XT, static_cast<uint32_t>(r));
#pragma unroll 1
        for (int chunk = 0; chunk < 4; ++chunk) {
          uint32_t v[32];
          ptx::tmem_ld_32x32(lane_base + kTmemD0 + chunk * 32, v);
          ptx::tmem_ld_wait();
          const uint32_t cb = static_cast<uint32_t>(chunk) * 4096u;     // 32 rows of 128 bytes
#pragma unroll
          for (int j = 0; j < 32; ++j) {
            const float d = __uint_as_float(v[j]);
            m1 += d;
            m2 = fmaf(d, lds_bf16(ocol.addr(j) + cb), m2);
          }
        }
        m1 *= (1.0f / kC);
        m2 *= (1.0f / kC);
        const float rs = rstd_o[r];
#pragma unroll 1
        for (int chunk = 0; chunk < 4; ++chunk) {
          uint32_t v[32];
          ptx::tmem_ld_32x32(lane_base + kTmemD0 + chunk * 32, v);
          ptx::tmem_ld_wait();
          const uint32_t cb = static_cast<uint32_t>(chunk) * 4096u;
#pragma unroll
          for (int j = 0; j < 32; ++j) {
            const uint32_t a = ocol.addr(j) + cb;
            sts_bf16(a, rs * (__uint_as_float(v[j]) - m1 - lds_bf16(a) * m2));
          }
        }
      } else {
        // the gate's share of d_zhat: first writer of dzp
        const long long p = static_cast<long long>(p0) + r;
#pragma unroll 1
        for (int chunk = 0; chunk < 4; ++chunk) {
          uint32_t v[32];
          ptx::tmem_ld_32x32(lane_base + kTmemD1 + chunk * 32, v);
          ptx::tmem_ld_wait();
          if (p < prm.R) {
            float4* dst = reinterpret_cast<float4*>(prm.dzp + p * kC + chunk * 32);
#pragma unroll
            for (int j = 0; j < 8; ++j)
              dst[j] = make_float4(__uint_as_float(v[4 * j]), __uint_as_float(v[4 * j + 1]),
                                   __uint_as_float(v[4 * j + 2]), __uint_as_float(v[4 * j + 3]));
          }
        }
      }
      ptx::tc_fence_before();
      ptx::fence_proxy_async_smem();
      __syncthreads();
      if (tid == 0) {
        ptx::tma_store_2d(&tmap_x, XT, p0, 0);
        ptx::tma_store_2d(&tmap_x, XT + kHalfBox, p0 + 64, 0);
        ptx::tma_store_commit();
      }
    } else {
      if (warp < 4) {
        const long long p = static_cast<long long>(p0) + r;
        const bool live = p < prm.R;
        if (kPass == 1) {
#pragma unroll 1
          for (int chunk = 0; chunk < 4; ++chunk) {
            uint32_t v[32];
            ptx::tmem_ld_32x32(lane_base + kTmemD0 + chunk * 32, v);
            ptx::tmem_ld_wait();
            if (live) {
              float4* dst = reinterpret_cast<float4*>(prm.dzp + p * kC + chunk * 32);
#pragma unroll
              for (int j = 0; j < 8; ++j) {
                float4 cur = dst[j];
                cur.x += __uint_as_float(v[4 * j]);
                cur.y += __uint_as_float(v[4 * j + 1]);
                cur.z += __uint_as_float(v[4 * j + 2]);
                cur.w += __uint_as_float(v[4 * j + 3]);
                dst[j] = cur;
              }
            }
          }
        } else {
          // total d_zhat, then d_z = rstd (d_zhat - mean(d_zhat) - zhat mean(d_zhat zhat)) [+ d_out]
          float m1 = 0.f, m2 = 0.f;
          auto load_xhat = [&](int chunk, float (&xh)[32]) {
#pragma unroll
            for (int c8 = 0; c8 < 4; ++c8) {
              uint32_t w[4];
              ptx::lds128(tile_addr(ZT, r, chunk * 32 + c8 * 8), w);
#pragma unroll
              for (int e = 0; e < 4; ++e) {
                xh[c8 * 8 + 2 * e] = ptx::bf16_lo(w[e]);
                xh[c8 * 8 + 2 * e + 1] = ptx::bf16_hi(w[e]);
              }
            }
          };
#pragma unroll 1
          for (int chunk = 0; chunk < 4; ++chunk) {
            uint32_t v[32];
            ptx::tmem_ld_32x32(lane_base + kTmemD0 + chunk * 32, v);
            ptx::tmem_ld_wait();
            float xh[32];
            load_xhat(chunk, xh);
            const float4* src = reinterpret_cast<const float4*>(prm.dzp + p * kC + chunk * 32);
#pragma unroll
            for (int j = 0; j < 8; ++j) {
              const float4 cur = live ? src[j] : make_float4(0.f, 0.f, 0.f, 0.f);
              const float d[4] = {cur.x + __uint_as_float(v[4 * j]), cur.y + __uint_as_float(v[4 * j + 1]),
                                  cur.z + __uint_as_float(v[4 * j + 2]), cur.w + __uint_as_float(v[4 * j + 3])};
#pragma unroll
              for (int e = 0; e < 4; ++e) {
                m1 += d[e];
                m2 = fmaf(d[e], xh[4 * j + e], m2);
              }
            }
          }
          m1 *= (1.0f / kC);
          m2 *= (1.0f / kC);
          const float rs = rstd_z[r];
#pragma unroll 1
          for (int chunk = 0; chunk < 4; ++chunk) {
            uint32_t v[32];
            ptx::tmem_ld_32x32(lane_base + kTmemD0 + chunk * 32, v);
            ptx::tmem_ld_wait();
            if (live) {
              float xh[32];
              load_xhat(chunk, xh);
              const float4* src = reinterpret_cast<const float4*>(prm.dzp + p * kC + chunk * 32);
              uint4* dst = reinterpret_cast<uint4*>(prm.d_z + p * kC + chunk * 32);
              const uint4* res = reinterpret_cast<const uint4*>(prm.d_out + p * kC + chunk * 32);
#pragma unroll
              for (int j8 = 0; j8 < 4; ++j8) {
                const float4 c0 = src[2 * j8], c1 = src[2 * j8 + 1];
                const float cur[8] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w};
                float o[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                  const int k = j8 * 8 + e;
                  o[e] = rs * (cur[e] + __uint_as_float(v[k]) - m1 - xh[k] * m2);
                }
                if (prm.add_residual) {
                  const uint4 rv = __ldg(res + j8);
                  const uint32_t rw[4] = {rv.x, rv.y, rv.z, rv.w};
#pragma unroll
                  for (int e = 0; e < 4; ++e) {
                    o[2 * e] += ptx::bf16_lo(rw[e]);
                    o[2 * e + 1] += ptx::bf16_hi(rw[e]);
                  }
                }
                uint4 pk;
                pk.x = ptx::pack_bf16x2(o[0], o[1]);
                pk.y = ptx::pack_bf16x2(o[2], o[3]);
                pk.z = ptx::pack_bf16x2(o[4], o[5]);
                pk.w = ptx::pack_bf16x2(o[6], o[7]);
                dst[j8] = pk;
              }
            }
          }
        }
      }
      ptx::tc_fence_before();
      __syncthreads();
    }
  }

  // ---------------- the CTA's record: Acc0, Acc1 (tensor memory -> global), db0, db1
  if (kPass == 0 && tid == 0) ptx::tma_store_wait<0>();
  ptx::tc_fence_after();
  {
    float* rec = prm.rec + static_cast<size_t>(blockIdx.x) * kRecFloats;
    const int tt = q * 32 + lane;              // row t of Acc = TMEM lane
#pragma unroll 1
    for (int m = 0; m < 2; ++m) {
#pragma unroll 1
      for (int chunk = 0; chunk < 2; ++chunk) {
        uint32_t v[32];
        ptx::tmem_ld_32x32(lane_base + (m ? kTmemAcc1 : kTmemAcc0) + h * 64 + chunk * 32, v);
        ptx::tmem_ld_wait();
        float4* dst = reinterpret_cast<float4*>(rec + m * kC * kC + tt * kC + h * 64 + chunk * 32);
#pragma unroll
        for (int j = 0; j < 8; ++j)
          dst[j] = make_float4(__uint_as_float(v[4 * j]), __uint_as_float(v[4 * j + 1]),
                               __uint_as_float(v[4 * j + 2]), __uint_as_float(v[4 * j + 3]));
      }
    }
    // GT's column sums belong to matrix: K3 -> d_y (matrix 1 = W_o); K1 -> d_p (matrix 0)
    // HT's:                              K3 -> d_gg (matrix 0 = W_g); K1 -> d_gate (matrix 1)
    const int which = (tid < 128) ? (kPass == 0 ? 1 : 0) : (kPass == 0 ? 0 : 1);
    rec[2 * kC * kC + which * kC + (tid & 127)] = db_acc;
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 1) ptx::tmem_dealloc<1>(tmem_base, 512);
}

// ---- parameter gradients from the per-CTA records ------------------------------------------------
// One (Acc, db) pair per projection matrix m; records of the three launches sit one after another:
//   launch 0 (K3): matrix 0 = W_g, 1 = W_o;  launch 1: 0 = W_a, 1 = W_a_gate;  launch 2: W_b, W_b_gate
struct AssembleParams {
  const float* rec;           // [3][blocks][kRecFloats]
  int blocks;
  float* sums;                // scratch [6][kC*kC + kC]: reduced Acc and db per matrix
  const __nv_bfloat16* w[6];  // raw weights in the order g, o, a, a_gate, b, b_gate
  const float* gamma_in;
  const float* beta_in;
  const float* gamma_out;
  const float* beta_out;
  float* dW[6];
  float* db[6];
  float* dgamma_in;
  float* dbeta_in;
  float* dgamma_out;
  float* dbeta_out;
};

// phase 1: fixed-order sum over the CTAs' records
__global__ void reduce_records_kernel(const AssembleParams prm) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;    // element of one matrix record
  const int m = blockIdx.y;                               // 0..5
  if (e >= kC * kC + kC) return;
  const int launch = m >> 1, slot = m & 1;
  const size_t off = e < kC * kC ? static_cast<size_t>(slot) * kC * kC + e
                                 : static_cast<size_t>(2) * kC * kC + slot * kC + (e - kC * kC);
  const float* base = prm.rec + static_cast<size_t>(launch) * prm.blocks * kRecFloats + off;
  float s = 0.f;
  for (int b = 0; b < prm.blocks; ++b) s += base[static_cast<size_t>(b) * kRecFloats];
  prm.sums[static_cast<size_t>(m) * (kC * kC + kC) + e] = s;
}

// phase 2: dW, db per matrix; dgamma / dbeta of both LayerNorms
__global__ void assemble_param_grads_kernel(const AssembleParams prm) {
  const int m = blockIdx.x;              // 0..5: per-matrix outputs;  6: LayerNorm-in; 7: LayerNorm-out
  const int tid = threadIdx.x;           // 128 threads
  const size_t stride = kC * kC + kC;
  if (m < 6) {
    const float* acc = prm.sums + m * stride;
    const float* db = acc + kC * kC;
    const float* gamma = m == 1 ? prm.gamma_out : prm.gamma_in;
    const float* beta = m == 1 ? prm.beta_out : prm.beta_in;
    if (prm.dW[m])
      for (int e = tid; e < kC * kC; e += 128) {
        const int t = e / kC, k = e % kC;
        prm.dW[m][e] = fmaf(acc[e], gamma[k], db[t] * beta[k]);
      }
    if (prm.db[m]) prm.db[m][tid] = db[tid];
    return;
  }
  // thread = channel k:  dgamma[k] = sum_m sum_t W_m[t][k] Acc_m[t][k],  dbeta[k] = sum_m sum_t W_m[t][k] db_m[t]
  const bool out_ln = m == 7;
  float dg = 0.f, dbt = 0.f;
  for (int mm = 0; mm < 6; ++mm) {
    if ((mm == 1) != out_ln) continue;
    const float* acc = prm.sums + mm * stride;
    const float* db = acc + kC * kC;
    for (int t = 0; t < kC; ++t) {
      const float w = __bfloat162float(prm.w[mm][t * kC + tid]);
      dg = fmaf(w, acc[t * kC + tid], dg);
      dbt = fmaf(w, db[t], dbt);
    }
  }
  float* dgo = out_ln ? prm.dgamma_out : prm.dgamma_in;
  float* dbo = out_ln ? prm.dbeta_out : prm.dbeta_in;
  if (dgo) dgo[tid] = dg;
  if (dbo) dbo[tid] = dbt;
}

int tail_grid(const DeviceInfo& dev, int num_tiles) {
  int g = dev.sm_count < kMaxBackwardBlocks ? dev.sm_count : kMaxBackwardBlocks;
  return num_tiles < g ? num_tiles : g;
}

}  // namespace

size_t backward_tc_scratch_floats() {
  return static_cast<size_t>(3) * kMaxBackwardBlocks * kRecFloats + 6 * (kC * kC + kC);
}

// phase 0: K3-backward; 1: K1-backward for a; 2: K1-backward for b (final) + parameter gradients.
// o_io: o on entry of phase 0, d_o afterwards; scratch: backward_tc_scratch_floats() floats.
int launch_tc_tail_backward(int phase, const void* d_out, const void* z, const void* mask,
                            const foldcp_trimul_params* p, int N, void* o_io, const void* d_a,
                            const void* d_b, float* dzp, float* scratch,
                            const foldcp_trimul_grads* g, void* d_z, cudaStream_t s) {
  DeviceInfo dev;
  if (!get_device_info(&dev)) return FOLDCP_ERR_CUDA;
  const uint64_t R = static_cast<uint64_t>(N) * N;
  const int num_tiles = static_cast<int>((R + kTilePairs - 1) / kTilePairs);
  const int grid = tail_grid(dev, num_tiles);
  float* rec = scratch;
  float* sums = scratch + static_cast<size_t>(3) * kMaxBackwardBlocks * kRecFloats;
  CUtensorMap tz, tx, tg, tw0, tw1;
  int st;
  const uint32_t box[2] = {64, 128};
  const uint64_t dims_pm[2] = {kC, R};          // pair-major [R][128]
  const uint64_t str_pm[1] = {kC * 2};
  const uint64_t dims_cm[2] = {R, kC};          // channel-major [128][R]
  const uint64_t str_cm[1] = {R * 2};
  const uint64_t dims_w[2] = {kC, kC};
  if ((st = encode_tensor_map(&tz, z, 2, 2, dims_pm, str_pm, box, true)) != FOLDCP_OK) return st;
  const void* xptr = phase == 0 ? o_io : (phase == 1 ? d_a : d_b);
  if ((st = encode_tensor_map(&tx, xptr, 2, 2, dims_cm, str_cm, box, true)) != FOLDCP_OK) return st;
  if ((st = encode_tensor_map(&tg, d_out, 2, 2, dims_pm, str_pm, box, true)) != FOLDCP_OK) return st;
  TailParams prm;
  prm.eps = p->ln_eps;
  prm.R = static_cast<long long>(R);
  prm.num_tiles = num_tiles;
  prm.add_residual = p->add_residual;
  prm.dzp = dzp;
  prm.d_out = static_cast<const __nv_bfloat16*>(d_out);
  prm.d_z = static_cast<__nv_bfloat16*>(d_z);
  prm.rec = rec + static_cast<size_t>(phase) * grid * kRecFloats;
  prm.gamma0 = p->ln_in_gamma;
  prm.beta0 = p->ln_in_beta;
  if (phase == 0) {
    prm.mask = p->mask_output ? static_cast<const __nv_bfloat16*>(mask) : nullptr;
    prm.w0 = static_cast<const __nv_bfloat16*>(p->w_g);
    prm.w1 = static_cast<const __nv_bfloat16*>(p->w_o);
    prm.bias0 = p->b_g;
    prm.bias1 = p->b_o;
    prm.gamma1 = p->ln_out_gamma;
    prm.beta1 = p->ln_out_beta;
  } else {
    prm.mask = static_cast<const __nv_bfloat16*>(mask);
    prm.w0 = static_cast<const __nv_bfloat16*>(phase == 1 ? p->w_a : p->w_b);
    prm.w1 = static_cast<const __nv_bfloat16*>(phase == 1 ? p->w_a_gate : p->w_b_gate);
    prm.bias0 = phase == 1 ? p->b_a : p->b_b;
    prm.bias1 = phase == 1 ? p->b_a_gate : p->b_b_gate;
    prm.gamma1 = p->ln_in_gamma;
    prm.beta1 = p->ln_in_beta;
  }
  if ((st = encode_tensor_map(&tw0, prm.w0, 2, 2, dims_w, str_pm, box, true)) != FOLDCP_OK) return st;
  if ((st = encode_tensor_map(&tw1, prm.w1, 2, 2, dims_w, str_pm, box, true)) != FOLDCP_OK) return st;
  const void* kern = phase == 0 ? reinterpret_cast<const void*>(tail_backward_kernel<0>)
                   : phase == 1 ? reinterpret_cast<const void*>(tail_backward_kernel<1>)
                                : reinterpret_cast<const void*>(tail_backward_kernel<2>);
  if (ensure_dynamic_smem(kern, kSmemBytes) != FOLDCP_OK) return FOLDCP_ERR_CUDA;
  if (phase == 0) tail_backward_kernel<0><<<grid, kThreads, kSmemBytes, s>>>(tz, tx, tg, tw0, tw1, prm);
  else if (phase == 1) tail_backward_kernel<1><<<grid, kThreads, kSmemBytes, s>>>(tz, tx, tg, tw0, tw1, prm);
  else tail_backward_kernel<2><<<grid, kThreads, kSmemBytes, s>>>(tz, tx, tg, tw0, tw1, prm);
  if ((st = check_launch()) != FOLDCP_OK || phase != 2) return st;

  AssembleParams ap;
  ap.rec = rec;
  ap.blocks = grid;
  ap.sums = sums;
  const void* ws[6] = {p->w_g, p->w_o, p->w_a, p->w_a_gate, p->w_b, p->w_b_gate};
  float* dWs[6] = {g->w_g, g->w_o, g->w_a, g->w_a_gate, g->w_b, g->w_b_gate};
  float* dbs[6] = {g->b_g, g->b_o, g->b_a, g->b_a_gate, g->b_b, g->b_b_gate};
  for (int m = 0; m < 6; ++m) {
    ap.w[m] = static_cast<const __nv_bfloat16*>(ws[m]);
    ap.dW[m] = dWs[m];
    ap.db[m] = dbs[m];
  }
  ap.gamma_in = p->ln_in_gamma;
  ap.beta_in = p->ln_in_beta;
  ap.gamma_out = p->ln_out_gamma;
  ap.beta_out = p->ln_out_beta;
  ap.dgamma_in = g->ln_in_gamma;
  ap.dbeta_in = g->ln_in_beta;
  ap.dgamma_out = g->ln_out_gamma;
  ap.dbeta_out = g->ln_out_beta;
  reduce_records_kernel<<<dim3((kC * kC + kC + 255) / 256, 6), 256, 0, s>>>(ap);
  assemble_param_grads_kernel<<<8, 128, 0, s>>>(ap);
  return check_launch();
}

}  // namespace foldcp
