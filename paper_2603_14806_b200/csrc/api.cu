// C-ABI boundary of libfoldcp_trimul (include/foldcp_trimul.h): argument validation, workspace
// carving, stage dispatch.  Never allocates, frees or synchronises; enqueues on the caller's
// stream and returns a status code.
#include <cstdlib>
#include <cstring>
#include <mutex>

#include "common.h"

namespace foldcp {

// ----------------------------------------------------------------------------- device info
bool get_device_info(DeviceInfo* info) {
  constexpr int kMaxDev = 64;
  static DeviceInfo cache[kMaxDev];
  static bool valid[kMaxDev] = {};
  static std::mutex mu;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDev) return false;
  std::lock_guard<std::mutex> lock(mu);
  if (!valid[dev]) {
    DeviceInfo d;
    if (cudaDeviceGetAttribute(&d.sm_count, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&d.cc_major, cudaDevAttrComputeCapabilityMajor, dev) !=
            cudaSuccess ||
        cudaDeviceGetAttribute(&d.cc_minor, cudaDevAttrComputeCapabilityMinor, dev) != cudaSuccess)
      return false;
    cache[dev] = d;
    valid[dev] = true;
  }
  *info = cache[dev];
  return true;
}

// ----------------------------------------------------------------------------- tile scheduler
// K1 and K2 draw their tiles in index order from an atomic counter (tile_sched.cuh).  The counter
// is launch-private and stream-ordered: it lives in caller-owned device memory (the tail of the
// workspace for foldcp_trimul, the `scratch` argument of the stage entry points) and is zeroed
// with a memset node on the caller's stream ahead of the launches that use it.  No process-global
// device state: any number of calls may be in flight on any number of streams (each with its own
// workspace / scratch), and a captured graph carries its own memset.
int arm_sched_words(void* scratch, cudaStream_t stream) {
  return cudaMemsetAsync(scratch, 0, kSchedScratchBytes, stream) == cudaSuccess ? FOLDCP_OK
                                                                               : FOLDCP_ERR_CUDA;
}

// ----------------------------------------------------------------------------- launch attributes
int ensure_dynamic_smem(const void* kernel, int bytes) {
  constexpr int kMaxDev = 64, kMaxKernels = 32;
  static const void* seen[kMaxDev][kMaxKernels] = {};
  static std::mutex mu;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDev) return FOLDCP_ERR_CUDA;
  std::lock_guard<std::mutex> lock(mu);
  int free_slot = -1;
  for (int i = 0; i < kMaxKernels; ++i) {
    if (seen[dev][i] == kernel) return FOLDCP_OK;
    if (seen[dev][i] == nullptr && free_slot < 0) free_slot = i;
  }
  if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes) !=
      cudaSuccess)
    return FOLDCP_ERR_CUDA;
  if (free_slot >= 0) seen[dev][free_slot] = kernel;
  return FOLDCP_OK;
}

// ----------------------------------------------------------------------------- tensor maps
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode_fn() {
  static EncodeTiledFn fn = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) !=
            cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      p = nullptr;
    return reinterpret_cast<EncodeTiledFn>(p);
  }();
  return fn;
}

// L2 promotion size of every tensor map: 256 B (debug knob FOLDCP_TMAP_L2PROMO = 0 / 64 / 128 / 256)
static CUtensorMapL2promotion l2_promotion() {
  static const CUtensorMapL2promotion v = [] {
    const char* e = debug_env("FOLDCP_TMAP_L2PROMO");
    const int n = e ? atoi(e) : 256;
    return n == 0     ? CU_TENSOR_MAP_L2_PROMOTION_NONE
           : n == 64  ? CU_TENSOR_MAP_L2_PROMOTION_L2_64B
           : n == 128 ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B
                      : CU_TENSOR_MAP_L2_PROMOTION_L2_256B;
  }();
  return v;
}

int encode_tensor_map(CUtensorMap* map, const void* base, int elem_bytes, int rank,
                      const uint64_t* dims, const uint64_t* strides_bytes, const uint32_t* box,
                      int swizzle) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) return FOLDCP_ERR_CUDA;
  cuuint64_t d[5], s[4];
  cuuint32_t b[5], e[5];
  for (int i = 0; i < rank; ++i) {
    d[i] = dims[i];
    b[i] = box[i];
    e[i] = 1;
    if (i + 1 < rank) s[i] = strides_bytes[i];
  }
  const CUtensorMapDataType dt =
      elem_bytes == 2 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
  const CUresult r =
      fn(map, dt, static_cast<cuuint32_t>(rank), const_cast<void*>(base), d, s, b, e,
         CU_TENSOR_MAP_INTERLEAVE_NONE,
         swizzle == 64 ? CU_TENSOR_MAP_SWIZZLE_64B
         : swizzle != 0 ? CU_TENSOR_MAP_SWIZZLE_128B
                        : CU_TENSOR_MAP_SWIZZLE_NONE,
         l2_promotion(), CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? FOLDCP_OK : FOLDCP_ERR_CUDA;
}

// ----------------------------------------------------------------------------- validation
namespace {

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

inline size_t elem_bytes(int dtype) { return dtype == FOLDCP_F32 ? 4 : 2; }

inline bool overlaps(const void* p, size_t pn, const void* q, size_t qn) {
  const uintptr_t a = reinterpret_cast<uintptr_t>(p), b = reinterpret_cast<uintptr_t>(q);
  return a < b + qn && b < a + pn;
}

int check_shape(int N, int c_z, int c_hidden, int dtype) {
  if (dtype != FOLDCP_F32 && dtype != FOLDCP_BF16) return FOLDCP_ERR_INVALID_ARG;
  if (N <= 0 || c_z <= 0 || c_hidden <= 0) return FOLDCP_ERR_INVALID_ARG;
  if (c_z != kChannels || c_hidden != kChannels) return FOLDCP_ERR_UNSUPPORTED;
  if (dtype == FOLDCP_BF16 && (N % 8) != 0) return FOLDCP_ERR_UNSUPPORTED;
  if (N > 32768) return FOLDCP_ERR_UNSUPPORTED;   // a/b/o alone would exceed 180 GB
  return FOLDCP_OK;
}

int check_params(const foldcp_trimul_params* p) {
  if (!p) return FOLDCP_ERR_INVALID_ARG;
  if (p->struct_size != sizeof(foldcp_trimul_params)) return FOLDCP_ERR_INVALID_ARG;
  if (p->dtype != FOLDCP_F32 && p->dtype != FOLDCP_BF16) return FOLDCP_ERR_INVALID_ARG;
  if (!(p->ln_eps >= 0.0f)) return FOLDCP_ERR_INVALID_ARG;
  if (p->reserved0 != 0 || (p->add_residual != 0 && p->add_residual != 1) ||
      (p->mask_output != 0 && p->mask_output != 1))
    return FOLDCP_ERR_INVALID_ARG;
  const void* required[] = {p->ln_in_gamma, p->ln_in_beta, p->w_a, p->w_a_gate, p->w_b,
                            p->w_b_gate, p->w_g, p->ln_out_gamma, p->ln_out_beta, p->w_o};
  for (const void* q : required)
    if (!q) return FOLDCP_ERR_INVALID_ARG;
  const void* all[] = {p->ln_in_gamma, p->ln_in_beta, p->w_a, p->w_a_gate, p->w_b, p->w_b_gate,
                       p->b_a, p->b_a_gate, p->b_b, p->b_b_gate, p->w_g, p->b_g,
                       p->ln_out_gamma, p->ln_out_beta, p->w_o, p->b_o};
  for (const void* q : all)
    if (q && !aligned16(q)) return FOLDCP_ERR_ALIGNMENT;
  return FOLDCP_OK;
}

int check_arch() {
  DeviceInfo d;
  if (!get_device_info(&d)) return FOLDCP_ERR_CUDA;
  return (d.cc_major == 10 && d.cc_minor == 0) ? FOLDCP_OK : FOLDCP_ERR_ARCH;   // sm_100a cubin only
}

// The shipped library has ONE path per dtype: bf16 -> the tcgen05 kernels, fp32 -> the FFMA
// kernels.  Only a -DFOLDCP_DEBUG_KNOBS build can send the bf16 mode through the FFMA kernels
// (FOLDCP_FORCE_SIMT=1, all three stages; a and b are then bf16) for bring-up cross-checks.
bool bf16_on_tensor_cores() {
  static const bool v = [] {
    const char* f = debug_env("FOLDCP_FORCE_SIMT");
    return !(f && f[0] == '1');
  }();
  return v;
}

}  // namespace
}  // namespace foldcp

using namespace foldcp;

namespace {
// (mean, rstd) of LayerNorm(z) per pair, handed from K1 to K3 in bf16 mode; a multiple of 256 bytes
size_t z_stats_bytes(int N, int dtype) {
  if (dtype != FOLDCP_BF16) return 0;
  return (static_cast<size_t>(N) * N * sizeof(float2) + 255) & ~static_cast<size_t>(255);
}
}  // namespace

extern "C" {

size_t foldcp_trimul_workspace_bytes(int N, int c_z, int c_hidden, int dtype) {
  if (check_shape(N, c_z, c_hidden, dtype) != FOLDCP_OK) return 0;
  return 3 * static_cast<size_t>(kChannels) * N * N * elem_bytes(dtype) + z_stats_bytes(N, dtype) +
         kSchedScratchBytes;
}

namespace {
// scratch of a stage entry point: required in bf16 mode (checked on the host, before anything is
// enqueued), then zeroed on the stream
int check_scratch(const void* scratch, int dtype) {
  if (dtype != FOLDCP_BF16) return FOLDCP_OK;
  if (!scratch) return FOLDCP_ERR_WORKSPACE;
  return aligned16(scratch) ? FOLDCP_OK : FOLDCP_ERR_ALIGNMENT;
}
int prepare_scratch(void* scratch, int dtype, cudaStream_t s) {
  return dtype == FOLDCP_BF16 ? arm_sched_words(scratch, s) : FOLDCP_OK;
}
}  // namespace

namespace {
// the stage bodies: arguments already validated, scheduler words already zeroed on the stream.
// ab_f16: in bf16 mode the intermediates a, b are IEEE fp16 (forward path) rather than bf16.
int project_stage(const void* z, const void* mask, const foldcp_trimul_params* params, int N,
                  void* a, void* b, bool ab_f16, void* z_stats, void* sched_area, cudaStream_t s) {
  if (params->dtype == FOLDCP_BF16 && bf16_on_tensor_cores())
    return launch_k1_project_bf16(z, mask, params, N, a, b, ab_f16, z_stats,
                                  sched_word(sched_area, 0), s);
  return launch_simt_project(z, mask, params, N, a, b, s);
}
int contract_stage(const void* a, const void* b, int N, int dtype, int direction, void* o,
                   bool ab_f16, float o_f16_scale, void* sched_area, int word, cudaStream_t s) {
  if (dtype == FOLDCP_BF16 && bf16_on_tensor_cores())
    return launch_k2_contract_bf16(a, b, o, N, direction, ab_f16, o_f16_scale,
                                   sched_word(sched_area, word), s);
  return launch_simt_contract(a, b, o, N, dtype, direction, s);
}
int finalize_stage(const void* o, const void* z, const void* mask,
                   const foldcp_trimul_params* params, int N, void* out, bool o_f16, float o_scale,
                   const void* z_stats, cudaStream_t s) {
  if (params->dtype == FOLDCP_BF16 && bf16_on_tensor_cores())
    return launch_k3_finalize_bf16(o, z, mask, params, N, out, o_f16, o_scale, z_stats, s);
  return launch_simt_finalize(o, z, mask, params, N, out, s);
}
}  // namespace

int foldcp_trimul_project(const void* z, const void* mask, const foldcp_trimul_params* params,
                          int N, int c_z, int c_hidden, void* a, void* b, void* scratch,
                          void* stream) {
  int st = check_params(params);
  if (st != FOLDCP_OK) return st;
  if ((st = check_shape(N, c_z, c_hidden, params->dtype)) != FOLDCP_OK) return st;
  if (!z || !a || !b) return FOLDCP_ERR_INVALID_ARG;
  if (!aligned16(z) || !aligned16(a) || !aligned16(b) || (mask && !aligned16(mask)))
    return FOLDCP_ERR_ALIGNMENT;
  const size_t bytes = static_cast<size_t>(N) * N * kChannels * elem_bytes(params->dtype);
  if (overlaps(a, bytes, z, bytes) || overlaps(b, bytes, z, bytes) || overlaps(a, bytes, b, bytes))
    return FOLDCP_ERR_ALIAS;
  if ((st = check_scratch(scratch, params->dtype)) != FOLDCP_OK) return st;
  if ((st = check_arch()) != FOLDCP_OK) return st;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if ((st = prepare_scratch(scratch, params->dtype, s)) != FOLDCP_OK) return st;
  return project_stage(z, mask, params, N, a, b, /*ab_f16=*/true, nullptr, scratch, s);
}

int foldcp_trimul_contract(const void* a, const void* b, int N, int c_hidden, int dtype,
                           int direction, void* o, void* scratch, void* stream) {
  const bool o_f16 = dtype == FOLDCP_BF16_F16ALL;     // ... and o fp16, scaled (the fused form)
  const bool ab_f16 = dtype == FOLDCP_BF16_F16AB || o_f16;   // a, b fp16 (what K1 writes)
  if (ab_f16) {
    if (!bf16_on_tensor_cores()) return FOLDCP_ERR_UNSUPPORTED;
    dtype = FOLDCP_BF16;
  }
  int st = check_shape(N, kChannels, c_hidden, dtype);
  if (st != FOLDCP_OK) return st;
  if (direction != FOLDCP_OUTGOING && direction != FOLDCP_INCOMING) return FOLDCP_ERR_INVALID_ARG;
  if (!a || !b || !o) return FOLDCP_ERR_INVALID_ARG;
  if (!aligned16(a) || !aligned16(b) || !aligned16(o)) return FOLDCP_ERR_ALIGNMENT;
  const size_t bytes = static_cast<size_t>(N) * N * kChannels * elem_bytes(dtype);
  if (overlaps(o, bytes, a, bytes) || overlaps(o, bytes, b, bytes)) return FOLDCP_ERR_ALIAS;
  if ((st = check_scratch(scratch, dtype)) != FOLDCP_OK) return st;
  if ((st = check_arch()) != FOLDCP_OK) return st;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if ((st = prepare_scratch(scratch, dtype, s)) != FOLDCP_OK) return st;
  return contract_stage(a, b, N, dtype, direction, o, ab_f16, o_f16 ? contract_o_scale(N) : 0.f,
                        scratch, 0, s);
}

int foldcp_trimul_contract_blocks(const void* const* a_blocks, const void* const* b_blocks,
                                  int nblocks, int nb, int c_hidden, int dtype, int direction,
                                  void* o_block, void* scratch, void* stream) {
  const bool ab_f16 = dtype == FOLDCP_BF16_F16AB;
  if (ab_f16) {
    if (!bf16_on_tensor_cores()) return FOLDCP_ERR_UNSUPPORTED;
    dtype = FOLDCP_BF16;
  }
  int st = check_shape(nb, kChannels, c_hidden, dtype);
  if (st != FOLDCP_OK) return st;
  if (direction != FOLDCP_OUTGOING && direction != FOLDCP_INCOMING) return FOLDCP_ERR_INVALID_ARG;
  if (!a_blocks || !b_blocks || !o_block || nblocks < 1) return FOLDCP_ERR_INVALID_ARG;
  if (nblocks > kMaxContractBlocks) return FOLDCP_ERR_UNSUPPORTED;
  if (!aligned16(o_block)) return FOLDCP_ERR_ALIGNMENT;
  const size_t bytes = static_cast<size_t>(nb) * nb * kChannels * elem_bytes(dtype);
  for (int q = 0; q < nblocks; ++q) {
    if (!a_blocks[q] || !b_blocks[q]) return FOLDCP_ERR_INVALID_ARG;
    if (!aligned16(a_blocks[q]) || !aligned16(b_blocks[q])) return FOLDCP_ERR_ALIGNMENT;
    if (overlaps(o_block, bytes, a_blocks[q], bytes) || overlaps(o_block, bytes, b_blocks[q], bytes))
      return FOLDCP_ERR_ALIAS;
  }
  if ((st = check_scratch(scratch, dtype)) != FOLDCP_OK) return st;
  if ((st = check_arch()) != FOLDCP_OK) return st;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if ((st = prepare_scratch(scratch, dtype, s)) != FOLDCP_OK) return st;
  if (dtype == FOLDCP_BF16 && bf16_on_tensor_cores())
    return launch_k2_contract_blocks_bf16(a_blocks, b_blocks, nblocks, o_block, nb, direction,
                                          ab_f16, sched_word(scratch, 0), s);
  return launch_simt_contract_blocks(a_blocks, b_blocks, nblocks, o_block, nb, dtype, direction, s);
}

int foldcp_trimul_contract_backward(const void* d_o, const void* a, const void* b, int N,
                                    int c_hidden, int dtype, int direction, void* d_a, void* d_b,
                                    void* scratch, void* stream) {
  int st = check_shape(N, kChannels, c_hidden, dtype);
  if (st != FOLDCP_OK) return st;
  if (direction != FOLDCP_OUTGOING && direction != FOLDCP_INCOMING) return FOLDCP_ERR_INVALID_ARG;
  if (!d_o || !a || !b || !d_a || !d_b) return FOLDCP_ERR_INVALID_ARG;
  if (!aligned16(d_o) || !aligned16(a) || !aligned16(b) || !aligned16(d_a) || !aligned16(d_b))
    return FOLDCP_ERR_ALIGNMENT;
  const size_t bytes = static_cast<size_t>(N) * N * kChannels * elem_bytes(dtype);
  const void* ins[3] = {d_o, a, b};
  for (const void* in : ins)
    if (overlaps(d_a, bytes, in, bytes) || overlaps(d_b, bytes, in, bytes)) return FOLDCP_ERR_ALIAS;
  if (overlaps(d_a, bytes, d_b, bytes)) return FOLDCP_ERR_ALIAS;
  if ((st = check_scratch(scratch, dtype)) != FOLDCP_OK) return st;
  if ((st = check_arch()) != FOLDCP_OK) return st;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if ((st = prepare_scratch(scratch, dtype, s)) != FOLDCP_OK) return st;
  if (dtype == FOLDCP_BF16 && bf16_on_tensor_cores())
    return launch_k2_contract_backward_bf16(d_o, a, b, d_a, d_b, N, direction,
                                            sched_word(scratch, 0), sched_word(scratch, 1), s);
  return launch_simt_contract_backward(d_o, a, b, d_a, d_b, N, dtype, direction, s);
}

int foldcp_trimul_finalize(const void* o, const void* z, const void* mask,
                           const foldcp_trimul_params* params, int N, int c_z, int c_hidden,
                           void* out, void* stream) {
  int st = check_params(params);
  if (st != FOLDCP_OK) return st;
  if ((st = check_shape(N, c_z, c_hidden, params->dtype)) != FOLDCP_OK) return st;
  if (!o || !z || !out) return FOLDCP_ERR_INVALID_ARG;
  if (!aligned16(o) || !aligned16(z) || !aligned16(out) || (mask && !aligned16(mask)))
    return FOLDCP_ERR_ALIGNMENT;
  const size_t bytes = static_cast<size_t>(N) * N * kChannels * elem_bytes(params->dtype);
  if (overlaps(out, bytes, z, bytes) || overlaps(out, bytes, o, bytes)) return FOLDCP_ERR_ALIAS;
  if ((st = check_arch()) != FOLDCP_OK) return st;
  return finalize_stage(o, z, mask, params, N, out, false, 1.0f, nullptr,
                        static_cast<cudaStream_t>(stream));
}

int foldcp_trimul_project_stats(const void* z, const void* mask, const foldcp_trimul_params* params,
                                int N, int c_z, int c_hidden, void* a, void* b, void* z_stats,
                                void* scratch, void* stream) {
  int st = check_params(params);
  if (st != FOLDCP_OK) return st;
  if ((st = check_shape(N, c_z, c_hidden, params->dtype)) != FOLDCP_OK) return st;
  if (params->dtype != FOLDCP_BF16 || !bf16_on_tensor_cores()) return FOLDCP_ERR_UNSUPPORTED;
  if (!z || !a || !b || !z_stats) return FOLDCP_ERR_INVALID_ARG;
  if (!aligned16(z) || !aligned16(a) || !aligned16(b) || !aligned16(z_stats) ||
      (mask && !aligned16(mask)))
    return FOLDCP_ERR_ALIGNMENT;
  const size_t bytes = static_cast<size_t>(N) * N * kChannels * elem_bytes(params->dtype);
  const size_t sbytes = static_cast<size_t>(N) * N * sizeof(float2);
  if (overlaps(a, bytes, z, bytes) || overlaps(b, bytes, z, bytes) || overlaps(a, bytes, b, bytes) ||
      overlaps(z_stats, sbytes, z, bytes) || overlaps(z_stats, sbytes, a, bytes) ||
      overlaps(z_stats, sbytes, b, bytes))
    return FOLDCP_ERR_ALIAS;
  if ((st = check_scratch(scratch, params->dtype)) != FOLDCP_OK) return st;
  if ((st = check_arch()) != FOLDCP_OK) return st;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if ((st = prepare_scratch(scratch, params->dtype, s)) != FOLDCP_OK) return st;
  return project_stage(z, mask, params, N, a, b, /*ab_f16=*/true, z_stats, scratch, s);
}

int foldcp_trimul_finalize_fused(const void* o, const void* z, const void* z_stats, const void* mask,
                                 const foldcp_trimul_params* params, int N, int c_z, int c_hidden,
                                 void* out, void* stream) {
  int st = check_params(params);
  if (st != FOLDCP_OK) return st;
  if ((st = check_shape(N, c_z, c_hidden, params->dtype)) != FOLDCP_OK) return st;
  if (params->dtype != FOLDCP_BF16 || !bf16_on_tensor_cores()) return FOLDCP_ERR_UNSUPPORTED;
  if (!o || !z || !out) return FOLDCP_ERR_INVALID_ARG;
  if (!aligned16(o) || !aligned16(z) || !aligned16(out) || (mask && !aligned16(mask)) ||
      (z_stats && !aligned16(z_stats)))
    return FOLDCP_ERR_ALIGNMENT;
  const size_t bytes = static_cast<size_t>(N) * N * kChannels * elem_bytes(params->dtype);
  if (overlaps(out, bytes, z, bytes) || overlaps(out, bytes, o, bytes) ||
      (z_stats && overlaps(out, bytes, z_stats, static_cast<size_t>(N) * N * sizeof(float2))))
    return FOLDCP_ERR_ALIAS;
  if ((st = check_arch()) != FOLDCP_OK) return st;
  return finalize_stage(o, z, mask, params, N, out, true, contract_o_scale(N), z_stats,
                        static_cast<cudaStream_t>(stream));
}

float foldcp_trimul_o_scale(int N) { return N > 0 ? contract_o_scale(N) : 0.f; }

int foldcp_trimul(const void* z, const void* mask, const foldcp_trimul_params* params, int N,
                  int c_z, int c_hidden, int direction, void* out, void* stream) {
  int st = check_params(params);
  if (st != FOLDCP_OK) return st;
  if (direction != FOLDCP_OUTGOING && direction != FOLDCP_INCOMING) return FOLDCP_ERR_INVALID_ARG;
  if (!z || !out) return FOLDCP_ERR_INVALID_ARG;
  if ((st = check_shape(N, c_z, c_hidden, params->dtype)) != FOLDCP_OK) return st;
  if (!aligned16(z) || !aligned16(out) || (mask && !aligned16(mask))) return FOLDCP_ERR_ALIGNMENT;
  const size_t need = foldcp_trimul_workspace_bytes(N, c_z, c_hidden, params->dtype);
  if (!params->workspace || params->workspace_bytes < need) return FOLDCP_ERR_WORKSPACE;
  if ((reinterpret_cast<uintptr_t>(params->workspace) & 255u) != 0) return FOLDCP_ERR_ALIGNMENT;
  const size_t tensor_bytes = static_cast<size_t>(N) * N * kChannels * elem_bytes(params->dtype);
  if (overlaps(out, tensor_bytes, z, tensor_bytes) ||
      overlaps(out, tensor_bytes, params->workspace, need) ||
      overlaps(z, tensor_bytes, params->workspace, need))
    return FOLDCP_ERR_ALIAS;
  if ((st = check_arch()) != FOLDCP_OK) return st;

  // workspace: a | b | o (channel-major) | LayerNorm(z) statistics (bf16 mode) | tile counters
  uint8_t* ws = static_cast<uint8_t*>(params->workspace);
  void* a = ws;
  void* b = ws + tensor_bytes;
  void* o = ws + 2 * tensor_bytes;
  const bool tc = params->dtype == FOLDCP_BF16 && bf16_on_tensor_cores();
  void* z_stats = tc ? ws + 3 * tensor_bytes : nullptr;
  void* sched_area = ws + 3 * tensor_bytes + z_stats_bytes(N, params->dtype);
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (params->dtype == FOLDCP_BF16 && (st = arm_sched_words(sched_area, s)) != FOLDCP_OK) return st;
  if ((st = project_stage(z, mask, params, N, a, b, true, z_stats, sched_area, s)) != FOLDCP_OK)
    return st;
  // bf16 mode: o travels from K2 to K3 as fp16 scaled by ~1/sqrt(N) (see contract_o_scale)
  const float o_scale = tc ? contract_o_scale(N) : 0.f;
  if ((st = contract_stage(a, b, N, params->dtype, direction, o, true, o_scale, sched_area, 1, s)) !=
      FOLDCP_OK)
    return st;
  return finalize_stage(o, z, mask, params, N, out, tc, tc ? o_scale : 1.0f, z_stats, s);
}

namespace {
// staged weights + per-block partial sums: the larger of the CUDA-core and the tcgen05 tail's needs
size_t backward_scratch_bytes() {
  const size_t a = backward_scratch_floats(kMaxBackwardBlocks), b = backward_tc_scratch_floats();
  return ((a > b ? a : b) * sizeof(float) + 255) & ~static_cast<size_t>(255);
}
}  // namespace

size_t foldcp_trimul_backward_workspace_bytes(int N, int c_z, int c_hidden, int dtype) {
  if (check_shape(N, c_z, c_hidden, dtype) != FOLDCP_OK) return 0;
  const size_t pairs = static_cast<size_t>(N) * N;
  return 5 * pairs * kChannels * elem_bytes(dtype)            // a, b, o / d_o, d_a, d_b
         + pairs * kChannels * sizeof(float)                  // d_z' accumulator
         + backward_scratch_bytes() + kSchedScratchBytes;
}

int foldcp_trimul_backward(const void* d_out, const void* z, const void* mask,
                           const foldcp_trimul_params* params, int N, int c_z, int c_hidden,
                           int direction, void* d_z, const foldcp_trimul_grads* grads,
                           void* stream) {
  int st = check_params(params);
  if (st != FOLDCP_OK) return st;
  if (!grads || grads->struct_size != sizeof(foldcp_trimul_grads) || grads->reserved0 != 0)
    return FOLDCP_ERR_INVALID_ARG;
  if (direction != FOLDCP_OUTGOING && direction != FOLDCP_INCOMING) return FOLDCP_ERR_INVALID_ARG;
  if (!d_out || !z || !d_z) return FOLDCP_ERR_INVALID_ARG;
  if ((st = check_shape(N, c_z, c_hidden, params->dtype)) != FOLDCP_OK) return st;
  if (!aligned16(d_out) || !aligned16(z) || !aligned16(d_z) || (mask && !aligned16(mask)))
    return FOLDCP_ERR_ALIGNMENT;
  float* const gp[] = {grads->ln_in_gamma, grads->ln_in_beta, grads->w_a, grads->w_a_gate,
                       grads->w_b, grads->w_b_gate, grads->b_a, grads->b_a_gate, grads->b_b,
                       grads->b_b_gate, grads->w_g, grads->b_g, grads->ln_out_gamma,
                       grads->ln_out_beta, grads->w_o, grads->b_o};
  for (const float* q : gp)
    if (q && (reinterpret_cast<uintptr_t>(q) & 3u) != 0) return FOLDCP_ERR_ALIGNMENT;
  const size_t need = foldcp_trimul_backward_workspace_bytes(N, c_z, c_hidden, params->dtype);
  if (!params->workspace || params->workspace_bytes < need) return FOLDCP_ERR_WORKSPACE;
  if ((reinterpret_cast<uintptr_t>(params->workspace) & 255u) != 0) return FOLDCP_ERR_ALIGNMENT;
  const size_t tb = static_cast<size_t>(N) * N * kChannels * elem_bytes(params->dtype);
  if (overlaps(d_z, tb, z, tb) || overlaps(d_z, tb, d_out, tb) ||
      overlaps(d_z, tb, params->workspace, need) || overlaps(z, tb, params->workspace, need) ||
      overlaps(d_out, tb, params->workspace, need))
    return FOLDCP_ERR_ALIAS;
  if ((st = check_arch()) != FOLDCP_OK) return st;

  // workspace: a | b | o -> d_o | d_a | d_b | d_z' (fp32) | staged weights + partials | counters
  uint8_t* ws = static_cast<uint8_t*>(params->workspace);
  void* a = ws;
  void* b = ws + tb;
  void* o = ws + 2 * tb;
  void* d_a = ws + 3 * tb;
  void* d_b = ws + 4 * tb;
  float* dzp = reinterpret_cast<float*>(ws + 5 * tb);
  float* scratch = dzp + static_cast<size_t>(N) * N * kChannels;
  void* sched_area = reinterpret_cast<uint8_t*>(scratch) + backward_scratch_bytes();
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const int dt = params->dtype;
  if (dt == FOLDCP_BF16 && (st = arm_sched_words(sched_area, s)) != FOLDCP_OK) return st;
  // recompute the forward intermediates with the forward kernels; a and b as bf16 here, because
  // the gradient GEMMs below pair them with the bf16 d_o (one operand format per tcgen05.mma)
  if ((st = project_stage(z, mask, params, N, a, b, false, nullptr, sched_area, s)) != FOLDCP_OK)
    return st;
  if ((st = contract_stage(a, b, N, dt, direction, o, false, 0.f, sched_area, 1, s)) != FOLDCP_OK)
    return st;
  // the tail around the contraction: tcgen05 kernels in bf16 mode, CUDA-core kernels in fp32 mode
  const bool tc = dt == FOLDCP_BF16 && bf16_on_tensor_cores();
  auto tail = [&](int phase) {
    return tc ? launch_tc_tail_backward(phase, d_out, z, mask, params, N, o, d_a, d_b, dzp, scratch,
                                        grads, d_z, s)
              : launch_simt_tail_backward(phase, d_out, z, mask, params, N, o, d_a, d_b, dzp,
                                          scratch, grads, d_z, s);
  };
  // K3-backward: o -> d_o in place
  if ((st = tail(0)) != FOLDCP_OK) return st;
  // gradients of Eq. 2-3
  if (tc)
    st = launch_k2_contract_backward_bf16(o, a, b, d_a, d_b, N, direction,
                                          sched_word(sched_area, 2), sched_word(sched_area, 3), s);
  else
    st = launch_simt_contract_backward(o, a, b, d_a, d_b, N, dt, direction, s);
  if (st != FOLDCP_OK) return st;
  // K1-backward for a, then for b (closing with the LayerNorm(z) backward)
  if ((st = tail(1)) != FOLDCP_OK) return st;
  return tail(2);
}

int foldcp_trimul_batched(const void* z, const void* mask, const foldcp_trimul_params* params,
                          int batch, int N, int c_z, int c_hidden, int direction, void* out,
                          void* stream) {
  if (batch <= 0) return FOLDCP_ERR_INVALID_ARG;
  int st = check_params(params);
  if (st != FOLDCP_OK) return st;
  if ((st = check_shape(N, c_z, c_hidden, params->dtype)) != FOLDCP_OK) return st;
  if (!z || !out) return FOLDCP_ERR_INVALID_ARG;
  const size_t eb = elem_bytes(params->dtype);
  const size_t tensor_bytes = static_cast<size_t>(N) * N * kChannels * eb;
  const size_t mask_bytes = static_cast<size_t>(N) * N * eb;
  // every batch element must itself satisfy the 16-byte alignment rule
  if (batch > 1 && ((tensor_bytes | mask_bytes) & 15u) != 0) return FOLDCP_ERR_ALIGNMENT;
  if (overlaps(out, tensor_bytes * batch, z, tensor_bytes * batch)) return FOLDCP_ERR_ALIAS;
  for (int b = 0; b < batch; ++b) {
    const uint8_t* zb = static_cast<const uint8_t*>(z) + b * tensor_bytes;
    const uint8_t* mb = mask ? static_cast<const uint8_t*>(mask) + b * mask_bytes : nullptr;
    uint8_t* ob = static_cast<uint8_t*>(out) + b * tensor_bytes;
    if ((st = foldcp_trimul(zb, mb, params, N, c_z, c_hidden, direction, ob, stream)) != FOLDCP_OK)
      return st;
  }
  return FOLDCP_OK;
}

int foldcp_trimul_launches_per_call(int dtype) {
  (void)dtype;
  return 3;
}

const char* foldcp_status_string(int status) {
  switch (status) {
    case FOLDCP_OK: return "ok";
    case FOLDCP_ERR_INVALID_ARG: return "invalid argument";
    case FOLDCP_ERR_UNSUPPORTED: return "unsupported shape";
    case FOLDCP_ERR_ALIGNMENT: return "misaligned pointer";
    case FOLDCP_ERR_WORKSPACE: return "workspace missing or too small";
    case FOLDCP_ERR_ALIAS: return "an output overlaps an input, another output or the workspace";
    case FOLDCP_ERR_ARCH: return "device is not sm_100 (compute capability 10.0)";
    case FOLDCP_ERR_CUDA: return "CUDA error";
    case FOLDCP_ERR_STATIC_LIMIT:
      return "problem exceeds the static workspace (FOLDCP_STATIC_WORKSPACE_BYTES): use foldcp_trimul";
    default: return "unknown status";
  }
}

int foldcp_version(void) { return 140; }   // 1.4: foldcp_trimul_static (1.3: z statistics in the workspace)

}  // extern "C"
