// Input LayerNorm of one [128 pairs][128 channels] bf16 tile held in shared memory exactly as TMA
// delivers it: two boxes (channels 0..63 | 64..127) of 128 rows x 128 bytes with the 128-byte
// swizzle (16-byte chunk index ^= row & 7).  The normalised, affine-transformed tile is written
// back in place (as fp16 when kF16, else bf16), which is the canonical K-major SWIZZLE_128B operand layout tcgen05.mma reads.
//
// 128 threads, two passes of 64 rows; two adjacent lanes share a row (one 64-channel box each)
// and combine their statistics with one shuffle.  Statistics are two-pass (mean, then centred
// sum of squares) in fp32 on the register-resident row, so they are exact for bf16 inputs up to
// fp32 summation error.  Used by K1 (z' feeds the four projections) and K3 (z' feeds the gate).
#pragma once

#include "ptx.cuh"

namespace foldcp {

// tile  : shared address of box 0 (box 1 is box_stride bytes further)
// tid   : 0..127 within the LayerNorm warp group
// gaddr / baddr : shared addresses of gamma[128] / beta[128] (fp32)
template <bool kF16>
__device__ __forceinline__ void layernorm_rows_inplace(uint32_t tile, uint32_t box_stride, int tid,
                                                       uint32_t gaddr, uint32_t baddr, float eps) {
  const uint32_t half = static_cast<uint32_t>(tid & 1);
  // chunk visiting order differs between the two lanes of a row (xor 5) so that a quarter-warp's
  // eight 16-byte loads fall in eight different bank groups and the gamma/beta broadcasts of the
  // two halves do not collide either
  const uint32_t cx = half * 5u;
#pragma unroll 1
  for (int pass = 0; pass < 2; ++pass) {
    const uint32_t r = static_cast<uint32_t>(pass * 64 + (tid >> 1));
    const uint32_t sw = r & 7u;
    const uint32_t row = tile + half * box_stride + r * 128u;
    uint32_t x[8][4];
#pragma unroll
    for (uint32_t c = 0; c < 8; ++c) ptx::lds128(row + (((c ^ cx) ^ sw) << 4), x[c]);
    float sum = 0.f;
#pragma unroll
    for (int c = 0; c < 8; ++c)
#pragma unroll
      for (int e = 0; e < 4; ++e) sum += ptx::bf16_lo(x[c][e]) + ptx::bf16_hi(x[c][e]);
    sum += __shfl_xor_sync(0xffffffffu, sum, 1);
    const float mu = sum * (1.0f / 128.0f);
    float var = 0.f;
#pragma unroll
    for (int c = 0; c < 8; ++c)
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const float d0 = ptx::bf16_lo(x[c][e]) - mu, d1 = ptx::bf16_hi(x[c][e]) - mu;
        var = fmaf(d0, d0, var);
        var = fmaf(d1, d1, var);
      }
    var += __shfl_xor_sync(0xffffffffu, var, 1);
    const float rstd = rsqrtf(var * (1.0f / 128.0f) + eps);
    const float nmr = -mu * rstd;
#pragma unroll
    for (uint32_t c = 0; c < 8; ++c) {
      const uint32_t cl = c ^ cx;                         // logical chunk = 8 channels
      const uint32_t voff = (half * 64u + cl * 8u) * 4u;  // byte offset of its gamma / beta
      float g[8], b[8];
      ptx::lds128f(gaddr + voff, *reinterpret_cast<float(*)[4]>(&g[0]));
      ptx::lds128f(gaddr + voff + 16, *reinterpret_cast<float(*)[4]>(&g[4]));
      ptx::lds128f(baddr + voff, *reinterpret_cast<float(*)[4]>(&b[0]));
      ptx::lds128f(baddr + voff + 16, *reinterpret_cast<float(*)[4]>(&b[4]));
      uint32_t y[4];
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const float n0 = fmaf(ptx::bf16_lo(x[c][e]), rstd, nmr);
        const float n1 = fmaf(ptx::bf16_hi(x[c][e]), rstd, nmr);
        y[e] = ptx::pack_norm<kF16>(fmaf(n0, g[2 * e], b[2 * e]), fmaf(n1, g[2 * e + 1], b[2 * e + 1]));
      }
      ptx::sts128(row + ((cl ^ sw) << 4), y[0], y[1], y[2], y[3]);
    }
  }
}

}  // namespace foldcp
