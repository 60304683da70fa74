// Host-side helpers shared by the translation units of libfoldcp_trimul: status plumbing,
// tensor-map (TMA descriptor) encoding through the driver entry point, launch-config helpers.
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>

#include "../../include/foldcp_trimul.h"

namespace foldcp {

// The LayerNorm outputs z' and LN(o) only ever exist as on-chip MMA operand tiles.  They are bounded
// (|LN(x)| <= sqrt(c-1) |gamma| + |beta|), so they are held in fp16 (11-bit significand) rather
// than bf16 (8-bit).  tcgen05 kind::f16 wants A and B in the same format (a mixed f16 x bf16
// descriptor is an illegal instruction on sm_100a), so each CTA converts its resident bf16 weights
// to fp16 in shared memory once (exact for 2^-14 <= |w| <= 65504).  Two of the four bf16 rounding
// points of the pipeline disappear at no cost
// (error budget).  Set to 0 to fall back to bf16 operand tiles.
#ifndef FOLDCP_NORM_FP16
#define FOLDCP_NORM_FP16 1
#endif
constexpr bool kNormFp16 = FOLDCP_NORM_FP16 != 0;

constexpr int kChannels = 128;  // c_z = c_hidden = 128 is the only supported channel count (A13)

// Tile-scheduler counters of one call: 256 bytes of caller-owned device memory (tail of the
// workspace / `scratch` of the stage entry points), zeroed on the caller's stream by
// arm_sched_words() ahead of the launches.  Word 0 serves K1 (or the first K2 launch of a stage
// call), word 16 (byte 64) K2 (or the second launch of contract_backward).
constexpr size_t kSchedScratchBytes = FOLDCP_SCHED_SCRATCH_BYTES;
int arm_sched_words(void* scratch, cudaStream_t stream);
inline unsigned int* sched_word(void* scratch, int which) {
  return reinterpret_cast<unsigned int*>(static_cast<uint8_t*>(scratch) + 64 * which);
}

// A/B knobs read from the environment exist only in -DFOLDCP_DEBUG_KNOBS builds (bring-up and
// measurement); the shipped library reads no environment variable and has one path per dtype.
inline const char* debug_env(const char* name) {
#ifdef FOLDCP_DEBUG_KNOBS
  return getenv(name);
#else
  (void)name;
  return nullptr;
#endif
}

struct DeviceInfo {
  int sm_count;
  int cc_major;
  int cc_minor;
};

// cached per device ordinal; returns false on CUDA error
bool get_device_info(DeviceInfo* info);

// Encode a tiled tensor map over a row-major tensor whose innermost dimension is dims[0].
//   elem_bytes: 2 (bf16) or 4 (f32); rank 2..4; strides_bytes[i] = byte stride of dims[i+1]
//   swizzle: 0 = none, 64 = SWIZZLE_64B (inner box 64 bytes), anything else (1 / true / 128) =
//            SWIZZLE_128B (inner box 128 bytes)
// Returns FOLDCP_OK or FOLDCP_ERR_CUDA.
int encode_tensor_map(CUtensorMap* map, const void* base, int elem_bytes, int rank,
                      const uint64_t* dims, const uint64_t* strides_bytes, const uint32_t* box,
                      int swizzle);

// ----- stage launchers (device pointers; return foldcp_status_t) -----
// `sched`: zeroed tile-scheduler counter(s) of this launch (see kSchedScratchBytes)
// ab_f16: a and b hold IEEE fp16 (forward path) instead of bf16.
// o_f16_scale: 0 = o is written as bf16; otherwise o is written as IEEE fp16 after multiplication
// by this power of two (the fused forward path: K3's LayerNorm(o) absorbs the scale exactly through
// eps * scale^2, and fp16 carries 11 significant bits where bf16 carries 8)
int launch_k2_contract_bf16(const void* a, const void* b, void* o, int N, int direction,
                            bool ab_f16, float o_f16_scale, unsigned int* sched,
                            cudaStream_t stream);
// the scale of the fused path: 2^-ceil(log2(N) / 2), i.e. about 1 / sqrt(N) -- o is a sum of N
// products a b, typically sqrt(N) sigma_a sigma_b, at worst N max|a b|; fp16 holds up to 65504
inline float contract_o_scale(int N) {
  int lg = 0;
  while ((1 << lg) < N) ++lg;
  return 1.0f / static_cast<float>(1 << ((lg + 1) / 2));
}

// blocked (Cannon) form: o_block[c][nb][nb] = sum_q contraction(a_blocks[q], b_blocks[q]), each
// block a dense [c][nb][nb] tensor, nq <= kMaxContractBlocks; accumulator resident in TMEM
constexpr int kMaxContractBlocks = 4;
int launch_k2_contract_blocks_bf16(const void* const* a_blocks, const void* const* b_blocks, int nq,
                                   void* o_block, int nb, int direction, bool ab_f16,
                                   unsigned int* sched, cudaStream_t stream);
int launch_simt_contract_blocks(const void* const* a_blocks, const void* const* b_blocks, int nq,
                                void* o_block, int nb, int dtype, int direction, cudaStream_t s);

int launch_k2_contract_backward_bf16(const void* d_o, const void* a, const void* b, void* d_a,
                                     void* d_b, int N, int direction, unsigned int* sched0,
                                     unsigned int* sched1, cudaStream_t stream);

int launch_simt_project(const void* z, const void* mask, const foldcp_trimul_params* p, int N,
                        void* a, void* b, cudaStream_t stream);
int launch_simt_contract(const void* a, const void* b, void* o, int N, int dtype, int direction,
                         cudaStream_t stream);
int launch_simt_contract_backward(const void* d_o, const void* a, const void* b, void* d_a,
                                  void* d_b, int N, int dtype, int direction, cudaStream_t stream);
int launch_simt_finalize(const void* o, const void* z, const void* mask,
                         const foldcp_trimul_params* p, int N, void* out, cudaStream_t stream);

// z_stats: [N*N] float2 (mean, rstd) of LayerNorm(z) written for K3 (fused path), or nullptr
int launch_k1_project_bf16(const void* z, const void* mask, const foldcp_trimul_params* p, int N,
                           void* a, void* b, bool ab_f16, void* z_stats, unsigned int* sched,
                           cudaStream_t stream);
// o_f16: o holds fp16 values scaled by the power of two o_scale (the fused path, see
// contract_o_scale); otherwise bf16 with o_scale = 1 (stage entry point, backward recomputation)
// z_stats: what K1 wrote (see above), or nullptr: K3 then computes the statistics of z itself
int launch_k3_finalize_bf16(const void* o, const void* z, const void* mask,
                            const foldcp_trimul_params* p, int N, void* out, bool o_f16,
                            float o_scale, const void* z_stats, cudaStream_t stream);

// Backward pass around the contraction (simt_backward.cu): phase 0 = K3-backward (o -> d_o in
// place, dzp written), 1 = K1-backward for a, 2 = K1-backward for b + LayerNorm(z) backward.
// `scratch`: backward_scratch_floats(blocks) floats; at most kMaxBackwardBlocks persistent blocks.
constexpr int kMaxBackwardBlocks = 160;
size_t backward_scratch_floats(int blocks);
int launch_simt_tail_backward(int phase, const void* d_out, const void* z, const void* mask,
                              const foldcp_trimul_params* p, int N, void* o_io, const void* d_a,
                              const void* d_b, float* dzp, float* scratch,
                              const foldcp_trimul_grads* g, void* d_z, cudaStream_t s);

// The same three phases on tcgen05 (k_backward.cu, bf16 mode); phase 2 also assembles all
// parameter gradients.  `scratch`: backward_tc_scratch_floats() floats.
size_t backward_tc_scratch_floats();
int launch_tc_tail_backward(int phase, const void* d_out, const void* z, const void* mask,
                            const foldcp_trimul_params* p, int N, void* o_io, const void* d_a,
                            const void* d_b, float* dzp, float* scratch,
                            const foldcp_trimul_grads* g, void* d_z, cudaStream_t s);

// Opt a kernel in to `bytes` of dynamic shared memory, once per (kernel, device); thread-safe.
// Returns FOLDCP_OK or FOLDCP_ERR_CUDA.
int ensure_dynamic_smem(const void* kernel, int bytes);

inline int check_launch() {
  return cudaPeekAtLastError() == cudaSuccess ? FOLDCP_OK : FOLDCP_ERR_CUDA;
}

}  // namespace foldcp
