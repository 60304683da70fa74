// Input LayerNorm of one [128 pairs][128 channels] bf16 tile held in shared memory exactly as TMA
// delivers it: two boxes (channels 0..63 | 64..127) of 128 rows x 128 bytes with the 128-byte
// swizzle (16-byte chunk index ^= row & 7).  The normalised, affine-transformed tile is written
// back in place (as fp16 when kF16, else bf16), which is the canonical K-major SWIZZLE_128B
// operand layout tcgen05.mma reads.
//
// 128 threads, two passes of 2 x 32 rows; four adjacent lanes share a row (32 channels each, held
// unpacked in registers) and combine their statistics with two shuffles.  Statistics are
// two-pass (mean, then centred sum of squares) in fp32, so they are exact for bf16 inputs up to
// fp32 summation error.  All arithmetic is packed fp32x2 (FADD2 / FFMA2): the kernels that call
// this are issue-bound, not FLOP-bound.  Used by K1 (z' feeds the four projections) and K3
// (z' feeds the output gate).
#pragma once

#include "ptx.cuh"

namespace foldcp {

// tile  : shared address of box 0 (box 1 is box_stride bytes further)
// tid   : 0..127 within the LayerNorm warp group
// gaddr / baddr : shared addresses of gamma[128] / beta[128] (fp32)
// kAffine = false: plain normalisation (x - mean) * rstd; gamma / beta are then folded into the
// weights and biases of the GEMM that consumes the tile (gaddr / baddr unused).
// kRows = rows per thread in flight (2 = more latency hiding, ~100 registers; 1 = ~60 registers).
// kLnThreads = threads of the LayerNorm group (128 or 256; 256 only with kRows = 1).
// `emit(row, mean, rstd)` is called by one lane per row with the row's statistics (K1 hands them
// to K3 through the workspace, which then does not recompute them).
struct NoRowStats {
  __device__ __forceinline__ void operator()(uint32_t, float, float) const {}
};
template <bool kF16, bool kAffine = true, int kRows = 2, int kLnThreads = 128,
          typename Emit = NoRowStats>
__device__ __forceinline__ void layernorm_rows_inplace(uint32_t tile, uint32_t box_stride, int tid,
                                                       uint32_t gaddr, uint32_t baddr, float eps,
                                                       Emit&& emit = Emit()) {
  const uint32_t j = static_cast<uint32_t>(tid & 3);        // quarter of the row: channels 32j..
  const uint32_t box = j >> 1;
  const uint32_t cbase = (j & 1u) * 4u;                      // first 16-byte chunk inside the box
  // Lane j visits its four chunks in the order t ^ j: a quarter-warp (2 rows x 4 lanes) then hits
  // eight distinct bank groups with its data and four distinct ones with gamma / beta.
  // Each thread works on two rows (r, r + 32) at once: the two dependency chains (loads, sums,
  // shuffles, rsqrt) interleave, which matters because one LayerNorm warp per scheduler is
  // latency-bound, not throughput-bound.
  static_assert(kLnThreads == 128 || (kLnThreads == 256 && kRows == 1), "unsupported LayerNorm shape");
  constexpr int kRowsPerPass = (kLnThreads / 4) * kRows;
#pragma unroll 1
  for (int pass = 0; pass < 128 / kRowsPerPass; ++pass) {
    const uint32_t r0 = static_cast<uint32_t>(pass * kRowsPerPass + (tid >> 2));
    const uint32_t sw = r0 & 7u;                              // (r0 + 32) & 7 is the same
    const uint32_t row0 = tile + box * box_stride + r0 * 128u;
    ptx::f32x2 x[kRows][4][4];
#pragma unroll
    for (uint32_t q = 0; q < kRows; ++q)
#pragma unroll
      for (uint32_t t = 0; t < 4; ++t) {
        uint32_t w[4];
        ptx::lds128(row0 + q * 4096u + (((cbase + (t ^ j)) ^ sw) << 4), w);
#pragma unroll
        for (int e = 0; e < 4; ++e) x[q][t][e] = ptx::bf16x2_to_f32x2(w[e]);
      }
    float mu[kRows], rstd[kRows];
    float sum[kRows];
#pragma unroll
    for (int q = 0; q < kRows; ++q) {
      ptx::f32x2 s2 = ptx::add2(x[q][0][0], x[q][0][1]), s3 = ptx::add2(x[q][0][2], x[q][0][3]);
#pragma unroll
      for (int t = 1; t < 4; ++t) {
        s2 = ptx::add2(s2, ptx::add2(x[q][t][0], x[q][t][1]));
        s3 = ptx::add2(s3, ptx::add2(x[q][t][2], x[q][t][3]));
      }
      float slo, shi;
      ptx::upk2(ptx::add2(s2, s3), slo, shi);
      sum[q] = slo + shi;
    }
#pragma unroll
    for (int q = 0; q < kRows; ++q) sum[q] += __shfl_xor_sync(0xffffffffu, sum[q], 1);
#pragma unroll
    for (int q = 0; q < kRows; ++q) sum[q] += __shfl_xor_sync(0xffffffffu, sum[q], 2);
    float var[kRows];
#pragma unroll
    for (int q = 0; q < kRows; ++q) {
      mu[q] = sum[q] * (1.0f / 128.0f);
      const ptx::f32x2 nmu = ptx::pk2(-mu[q], -mu[q]);
      ptx::f32x2 v2 = ptx::pk2(0.f, 0.f), v3 = v2;
#pragma unroll
      for (int t = 0; t < 4; ++t)
#pragma unroll
        for (int e = 0; e < 4; e += 2) {
          const ptx::f32x2 d0 = ptx::add2(x[q][t][e], nmu), d1 = ptx::add2(x[q][t][e + 1], nmu);
          v2 = ptx::fma2(d0, d0, v2);
          v3 = ptx::fma2(d1, d1, v3);
        }
      float slo, shi;
      ptx::upk2(ptx::add2(v2, v3), slo, shi);
      var[q] = slo + shi;
    }
#pragma unroll
    for (int q = 0; q < kRows; ++q) var[q] += __shfl_xor_sync(0xffffffffu, var[q], 1);
#pragma unroll
    for (int q = 0; q < kRows; ++q) var[q] += __shfl_xor_sync(0xffffffffu, var[q], 2);
    ptx::f32x2 rs2[kRows], nmr2[kRows];
#pragma unroll
    for (int q = 0; q < kRows; ++q) {
      rstd[q] = rsqrtf(var[q] * (1.0f / 128.0f) + eps);
      rs2[q] = ptx::pk2(rstd[q], rstd[q]);
      const float nmr = -mu[q] * rstd[q];
      nmr2[q] = ptx::pk2(nmr, nmr);
      if (j == 0) emit(r0 + static_cast<uint32_t>(q) * 32u, mu[q], rstd[q]);
    }
#pragma unroll
    for (uint32_t t = 0; t < 4; ++t) {
      const uint32_t tt = t ^ j;
      const uint32_t voff = (32u * j + 8u * tt) * 4u;       // byte offset of this chunk's gamma/beta
      ptx::f32x2 g[4], b[4];
      if constexpr (kAffine) {
        ptx::lds128x2(gaddr + voff, *reinterpret_cast<ptx::f32x2(*)[2]>(&g[0]));
        ptx::lds128x2(gaddr + voff + 16, *reinterpret_cast<ptx::f32x2(*)[2]>(&g[2]));
        ptx::lds128x2(baddr + voff, *reinterpret_cast<ptx::f32x2(*)[2]>(&b[0]));
        ptx::lds128x2(baddr + voff + 16, *reinterpret_cast<ptx::f32x2(*)[2]>(&b[2]));
      }
#pragma unroll
      for (uint32_t q = 0; q < kRows; ++q) {
        uint32_t y[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          ptx::f32x2 n = ptx::fma2(x[q][t][e], rs2[q], nmr2[q]);
          if constexpr (kAffine) n = ptx::fma2(n, g[e], b[e]);
          y[e] = ptx::pack_norm2<kF16>(n);
        }
        ptx::sts128(row0 + q * 4096u + (((cbase + tt) ^ sw) << 4), y[0], y[1], y[2], y[3]);
      }
    }
  }
}

// LayerNorm STATISTICS of the same tile, nothing written back to it: per pair row r, mean and
// biased variance over the 128 channels, handed to `emit(row, mean, var)` by ONE lane per row (a
// consumer then applies the normalisation after the GEMM, see k3_finalize.cu).  One sweep over the
// row with a shifted accumulation: d = x - c with c the row's own first channel, S1 = sum d,
// S2 = sum d^2, mean = c + S1 / 128, var = S2 / 128 - (S1 / 128)^2.  The shift is a sample of the
// row, so |mean - c| is of the order of the row's spread and the subtraction cancels nothing that
// matters, whatever the row's common offset (|mean| >> sigma is as safe as with two passes).
// kLnThreads (128 or 256) threads, four adjacent lanes per row, kRows rows per thread in flight.
// `tile_read()` is called once the thread has consumed everything it loads from the tile (the tile
// may be handed back to its producer then), before the shuffles and the emits.
template <int kRows, int kLnThreads, typename TileRead, typename Emit>
__device__ __forceinline__ void layernorm_rows_stats(uint32_t tile, uint32_t box_stride, int tid,
                                                     TileRead&& tile_read, Emit&& emit) {
  const uint32_t j = static_cast<uint32_t>(tid & 3);
  const uint32_t box = j >> 1;
  const uint32_t cbase = (j & 1u) * 4u;
  constexpr int kRowStep = kLnThreads / 4;                    // rows between a thread's rows in flight
  constexpr int kRowsPerPass = kRowStep * kRows;
  static_assert(128 % kRowsPerPass == 0 && kRowStep % 8 == 0, "unsupported LayerNorm shape");
#pragma unroll 1
  for (int pass = 0; pass < 128 / kRowsPerPass; ++pass) {
    const uint32_t r0 = static_cast<uint32_t>(pass * kRowsPerPass + (tid >> 2));
    const uint32_t sw = r0 & 7u;                              // (r0 + kRowStep) & 7 is the same
    const uint32_t row0 = tile + box * box_stride + r0 * 128u;
    uint32_t w[kRows][4][4];
#pragma unroll
    for (uint32_t q = 0; q < kRows; ++q)
#pragma unroll
      for (uint32_t t = 0; t < 4; ++t)
        ptx::lds128(row0 + q * (kRowStep * 128u) + (((cbase + (t ^ j)) ^ sw) << 4), w[q][t]);
    float s1[kRows], s2[kRows], c[kRows];
#pragma unroll
    for (int q = 0; q < kRows; ++q) {
      // the shift: the first channel lane 0 of the row's quad loaded -- any channel would do
      c[q] = __shfl_sync(0xffffffffu, ptx::bf16_lo(w[q][0][0]), tid & 28);
      const ptx::f32x2 nc = ptx::pk2(-c[q], -c[q]);
      ptx::f32x2 a0 = ptx::pk2(0.f, 0.f), a1 = a0, b0 = a0, b1 = a0;
#pragma unroll
      for (int t = 0; t < 4; ++t)
#pragma unroll
        for (int e = 0; e < 4; e += 2) {
          const ptx::f32x2 d0 = ptx::add2(ptx::bf16x2_to_f32x2(w[q][t][e]), nc);
          const ptx::f32x2 d1 = ptx::add2(ptx::bf16x2_to_f32x2(w[q][t][e + 1]), nc);
          a0 = ptx::add2(a0, d0);
          a1 = ptx::add2(a1, d1);
          b0 = ptx::fma2(d0, d0, b0);
          b1 = ptx::fma2(d1, d1, b1);
        }
      float lo, hi;
      ptx::upk2(ptx::add2(a0, a1), lo, hi);
      s1[q] = lo + hi;
      ptx::upk2(ptx::add2(b0, b1), lo, hi);
      s2[q] = lo + hi;
    }
    if (pass == 128 / kRowsPerPass - 1) tile_read();
#pragma unroll
    for (int q = 0; q < kRows; ++q) {
      s1[q] += __shfl_xor_sync(0xffffffffu, s1[q], 1);
      s2[q] += __shfl_xor_sync(0xffffffffu, s2[q], 1);
    }
#pragma unroll
    for (int q = 0; q < kRows; ++q) {
      s1[q] += __shfl_xor_sync(0xffffffffu, s1[q], 2);
      s2[q] += __shfl_xor_sync(0xffffffffu, s2[q], 2);
    }
    if (j == 0) {
#pragma unroll
      for (uint32_t q = 0; q < kRows; ++q) {
        const float md = s1[q] * (1.0f / 128.0f);
        const float var = fmaxf(fmaf(-md, md, s2[q] * (1.0f / 128.0f)), 0.f);
        emit(r0 + q * kRowStep, c[q] + md, var);
      }
    }
  }
}

}  // namespace foldcp
