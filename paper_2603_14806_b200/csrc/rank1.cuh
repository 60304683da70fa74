// Rank-one terms given to the tensor core (used by K1 for its biases and by K3 for the LayerNorm
// terms): a per-row constant x is split into three pieces of the MMA's operand format,
// x = x1 + x2 + x3 (round to nearest each time; the remainders are exact in fp32: 24 bits of x from
// bf16 pieces, more from fp16 ones), and laid out as one row of an unswizzled K-major operand of
// K = 16 (ptx::make_smem_desc_noswizzle with lbo 128, sbo 256): slots 0..7 of row r at
// (r / 8) * 256 + (r % 8) * 16, slots 8..15 another 128 bytes on.
#pragma once

#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include "ptx.cuh"

namespace foldcp {

template <bool kF16>
__device__ __forceinline__ void split3(float x, uint32_t (&p)[3]) {
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    if constexpr (kF16) {
      // saturating: a value beyond fp16's range (outside the documented preconditions) stays finite
      const uint32_t h2 = ptx::pack_f16x2(x, 0.f);
      p[i] = h2 & 0xffffu;
      x -= __half2float(__ushort_as_half(static_cast<unsigned short>(h2 & 0xffffu)));
    } else {
      const __nv_bfloat16 h = __float2bfloat16_rn(x);
      p[i] = static_cast<uint32_t>(__bfloat16_as_ushort(h));
      x -= __bfloat162float(h);
    }
  }
}

__device__ __forceinline__ uint32_t rank1_row_addr(uint32_t base, uint32_t r) {
  return base + (r >> 3) * 256u + (r & 7u) * 16u;
}

// 1.0 in the operand format
template <bool kF16>
__device__ __forceinline__ uint32_t one16() {
  return kF16 ? 0x3c00u : 0x3f80u;
}

// row r = ( x1 x2 x3 0 ... 0 ): against a row of ones ( 1 1 1 0 ... 0 ) the MMA adds x
template <bool kF16>
__device__ __forceinline__ void write_rank1_value_row(uint32_t base, uint32_t r, float x) {
  uint32_t a[3];
  split3<kF16>(x, a);
  const uint32_t addr = rank1_row_addr(base, r);
  ptx::sts128(addr, a[0] | (a[1] << 16), a[2], 0u, 0u);
  ptx::sts128(addr + 128, 0u, 0u, 0u, 0u);
}
template <bool kF16>
__device__ __forceinline__ void write_rank1_ones_row(uint32_t base, uint32_t r) {
  const uint32_t o = one16<kF16>();
  const uint32_t addr = rank1_row_addr(base, r);
  ptx::sts128(addr, o | (o << 16), o, 0u, 0u);
  ptx::sts128(addr + 128, 0u, 0u, 0u, 0u);
}

}  // namespace foldcp
