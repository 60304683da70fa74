// Triangle attention (section 3.2 lines 98-115, Eq. 1; AF3 Alg. 14/15):
// a first correct CUDA path on the CUDA cores, fp32 arithmetic, for both storage types.
//
//   ta_project_kernel    z' = LN(z);  q, k, v = W z';  g = sigmoid(W_g z');  t = W_t z'  (t also transposed)
//   ta_attention_kernel  per (line, head): out[pos] = g * softmax_k(q[pos] . k[k] / sqrt(c) + t[pos][k] + mb[k]) v
//                        -- online softmax over key chunks staged in shared memory; "line" is the row i
//                        (starting node) or the column j (ending node), "pos" the other pair index, so
//                        the ending node is the same kernel with swapped strides and the transposed bias
//   ta_output_kernel     out = W_o (g * o)
// Layouts: z / out [N][N][128]; workspace q, k, v, g fp32 [N][N][128] (head-major inside: h * 32 + d);
// t, tT fp32 [H][N][N].
#include <cuda_bf16.h>

#include "../../include/foldcp_triattn.h"
#include "common.h"

namespace foldcp {
namespace {

constexpr int C = kChannels;      // c_z = H * c_head = 128
constexpr int kHead = 32;
constexpr int kHeads = 4;
constexpr int kPairsPerBlock = 16;
constexpr int kKeyChunk = 64;
constexpr int kQueries = 128;     // threads of an attention block = query positions

template <typename T> __device__ __forceinline__ float ldf(const T* p);
template <> __device__ __forceinline__ float ldf<float>(const float* p) { return *p; }
template <> __device__ __forceinline__ float ldf<__nv_bfloat16>(const __nv_bfloat16* p) {
  return __bfloat162float(*p);
}
template <typename T> __device__ __forceinline__ void stf(T* p, float v);
template <> __device__ __forceinline__ void stf<float>(float* p, float v) { *p = v; }
template <> __device__ __forceinline__ void stf<__nv_bfloat16>(__nv_bfloat16* p, float v) {
  *p = __float2bfloat16_rn(v);
}

// block = 128 threads (thread = output channel), 16 consecutive pairs
template <typename T>
__global__ void __launch_bounds__(128)
ta_project_kernel(const T* __restrict__ z, const T* __restrict__ w_q, const T* __restrict__ w_k,
                  const T* __restrict__ w_v, const T* __restrict__ w_g, const T* __restrict__ w_t,
                  const float* __restrict__ gamma, const float* __restrict__ beta, float eps, int N,
                  float* __restrict__ q, float* __restrict__ k, float* __restrict__ v,
                  float* __restrict__ g, float* __restrict__ t, float* __restrict__ tT) {
  __shared__ float zs[kPairsPerBlock][C];
  const long long npairs = static_cast<long long>(N) * N;
  const long long p0 = static_cast<long long>(blockIdx.x) * kPairsPerBlock;
  const int np = static_cast<int>(min(static_cast<long long>(kPairsPerBlock), npairs - p0));
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  for (int p = 0; p < np; ++p) zs[p][tid] = ldf(z + (p0 + p) * C + tid);
  __syncthreads();
  for (int p = warp; p < np; p += 4) {     // LayerNorm: one warp per row, two-pass statistics
    float x[4], s = 0.f;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      x[i] = zs[p][lane + 32 * i];
      s += x[i];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    const float mu = s * (1.0f / C);
    float var = 0.f;
#pragma unroll
    for (int i = 0; i < 4; ++i) var += (x[i] - mu) * (x[i] - mu);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) var += __shfl_xor_sync(0xffffffffu, var, o);
    const float rstd = 1.0f / sqrtf(var * (1.0f / C) + eps);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int c = lane + 32 * i;
      zs[p][c] = (x[i] - mu) * rstd * gamma[c] + beta[c];
    }
  }
  __syncthreads();
  float aq[kPairsPerBlock], ak[kPairsPerBlock], av[kPairsPerBlock], ag[kPairsPerBlock];
#pragma unroll
  for (int p = 0; p < kPairsPerBlock; ++p) aq[p] = ak[p] = av[p] = ag[p] = 0.f;
  for (int c = 0; c < C; ++c) {
    const float wq = ldf(w_q + tid * C + c), wk = ldf(w_k + tid * C + c), wv = ldf(w_v + tid * C + c),
                wg = ldf(w_g + tid * C + c);
#pragma unroll
    for (int p = 0; p < kPairsPerBlock; ++p) {
      const float x = zs[p][c];
      aq[p] = fmaf(wq, x, aq[p]);
      ak[p] = fmaf(wk, x, ak[p]);
      av[p] = fmaf(wv, x, av[p]);
      ag[p] = fmaf(wg, x, ag[p]);
    }
  }
  for (int p = 0; p < np; ++p) {
    const long long o = (p0 + p) * C + tid;
    q[o] = aq[p];
    k[o] = ak[p];
    v[o] = av[p];
    g[o] = 1.0f / (1.0f + expf(-ag[p]));
  }
  // the triangular bias: thread (p, h) for the first 16 * H threads
  if (tid < kPairsPerBlock * kHeads) {
    const int p = tid / kHeads, h = tid % kHeads;
    if (p < np) {
      float acc = 0.f;
      for (int c = 0; c < C; ++c) acc = fmaf(ldf(w_t + h * C + c), zs[p][c], acc);
      const long long pair = p0 + p;
      const long long i = pair / N, j = pair % N;
      t[(static_cast<long long>(h) * N + i) * N + j] = acc;
      tT[(static_cast<long long>(h) * N + j) * N + i] = acc;
    }
  }
}

// grid (ceil(N / 128), N lines, H); thread = query position `pos`; keys in chunks of 64 through smem.
// address of pair (line, x): line * ls + x * xs  (starting node: ls = N, xs = 1; ending: ls = 1, xs = N)
template <typename T>
__global__ void __launch_bounds__(kQueries)
ta_attention_kernel(const float* __restrict__ q, const float* __restrict__ k,
                    const float* __restrict__ v, const float* __restrict__ g,
                    const float* __restrict__ tb,    // [H][N][N]: bias of (query pos, key pos)
                    const T* __restrict__ mask, int N, long long ls, long long xs,
                    float* __restrict__ og) {         // g * o, written over q's slot
  __shared__ float ks[kKeyChunk][kHead];
  __shared__ float vs[kKeyChunk][kHead];
  __shared__ float ms[kKeyChunk];
  const int line = blockIdx.y, h = blockIdx.z;
  const int pos = blockIdx.x * kQueries + threadIdx.x;
  const bool active = pos < N;
  const float scale = rsqrtf(static_cast<float>(kHead));
  float qr[kHead], acc[kHead];
  const long long qaddr = (static_cast<long long>(line) * ls + static_cast<long long>(active ? pos : 0) * xs) * C + h * kHead;
#pragma unroll
  for (int d = 0; d < kHead; ++d) {
    qr[d] = active ? q[qaddr + d] * scale : 0.f;
    acc[d] = 0.f;
  }
  float m = -INFINITY, l = 0.f;
  const float* trow = tb + (static_cast<long long>(h) * N + (active ? pos : 0)) * N;
  for (int k0 = 0; k0 < N; k0 += kKeyChunk) {
    const int nk = min(kKeyChunk, N - k0);
    __syncthreads();
    for (int e = threadIdx.x; e < nk * kHead; e += kQueries) {
      const int kk = e / kHead, d = e % kHead;
      const long long a = (static_cast<long long>(line) * ls + static_cast<long long>(k0 + kk) * xs) * C + h * kHead + d;
      ks[kk][d] = k[a];
      vs[kk][d] = v[a];
    }
    for (int kk = threadIdx.x; kk < nk; kk += kQueries)
      ms[kk] = mask ? -1.0e9f * (1.0f - ldf(mask + static_cast<long long>(line) * ls + static_cast<long long>(k0 + kk) * xs)) : 0.f;
    __syncthreads();
    if (active) {
      for (int kk = 0; kk < nk; ++kk) {
        float s = trow[k0 + kk] + ms[kk];
#pragma unroll
        for (int d = 0; d < kHead; ++d) s = fmaf(qr[d], ks[kk][d], s);
        if (s > m) {                       // online softmax: rescale what has been accumulated
          const float r = expf(m - s);
          l *= r;
#pragma unroll
          for (int d = 0; d < kHead; ++d) acc[d] *= r;
          m = s;
        }
        const float pexp = expf(s - m);
        l += pexp;
#pragma unroll
        for (int d = 0; d < kHead; ++d) acc[d] = fmaf(pexp, vs[kk][d], acc[d]);
      }
    }
  }
  if (active) {
    const float inv = 1.0f / l;
#pragma unroll
    for (int d = 0; d < kHead; ++d) og[qaddr + d] = g[qaddr + d] * acc[d] * inv;
  }
}

// block = 128 threads (thread = output channel), 16 consecutive pairs
template <typename T>
__global__ void __launch_bounds__(128)
ta_output_kernel(const float* __restrict__ og, const T* __restrict__ w_o, long long npairs,
                 T* __restrict__ out) {
  __shared__ float os[kPairsPerBlock][C];
  const long long p0 = static_cast<long long>(blockIdx.x) * kPairsPerBlock;
  const int np = static_cast<int>(min(static_cast<long long>(kPairsPerBlock), npairs - p0));
  const int tid = threadIdx.x;
  for (int p = 0; p < np; ++p) os[p][tid] = og[(p0 + p) * C + tid];
  __syncthreads();
  float acc[kPairsPerBlock];
#pragma unroll
  for (int p = 0; p < kPairsPerBlock; ++p) acc[p] = 0.f;
  for (int c = 0; c < C; ++c) {
    const float w = ldf(w_o + tid * C + c);
#pragma unroll
    for (int p = 0; p < kPairsPerBlock; ++p) acc[p] = fmaf(w, os[p][c], acc[p]);
  }
  for (int p = 0; p < np; ++p) stf(out + (p0 + p) * C + tid, acc[p]);
}

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
inline bool overlaps(const void* p, size_t pn, const void* q, size_t qn) {
  const uintptr_t a = reinterpret_cast<uintptr_t>(p), b = reinterpret_cast<uintptr_t>(q);
  return a < b + qn && b < a + pn;
}

template <typename T>
int launch_all(const void* z, const void* mask, const foldcp_triattn_params* p, int N, int node,
               void* out, cudaStream_t s) {
  const long long npairs = static_cast<long long>(N) * N;
  float* ws = static_cast<float*>(p->workspace);
  float* q = ws;
  float* k = q + npairs * C;
  float* v = k + npairs * C;
  float* g = v + npairs * C;
  float* t = g + npairs * C;
  float* tT = t + npairs * kHeads;
  const int pblocks = static_cast<int>((npairs + kPairsPerBlock - 1) / kPairsPerBlock);
  ta_project_kernel<T><<<pblocks, 128, 0, s>>>(
      static_cast<const T*>(z), static_cast<const T*>(p->w_q), static_cast<const T*>(p->w_k),
      static_cast<const T*>(p->w_v), static_cast<const T*>(p->w_g), static_cast<const T*>(p->w_t),
      p->ln_gamma, p->ln_beta, p->ln_eps, N, q, k, v, g, t, tT);
  const bool starting = node == FOLDCP_TRIATTN_STARTING;
  const dim3 grid((N + kQueries - 1) / kQueries, N, kHeads);
  ta_attention_kernel<T><<<grid, kQueries, 0, s>>>(q, k, v, g, starting ? t : tT,
                                                   static_cast<const T*>(mask), N,
                                                   starting ? N : 1, starting ? 1 : N, q);
  ta_output_kernel<T><<<pblocks, 128, 0, s>>>(q, static_cast<const T*>(p->w_o), npairs,
                                              static_cast<T*>(out));
  return check_launch();
}

}  // namespace
}  // namespace foldcp

using namespace foldcp;

extern "C" {

size_t foldcp_triattn_workspace_bytes(int N, int c_z, int n_heads, int dtype) {
  if ((dtype != FOLDCP_F32 && dtype != FOLDCP_BF16) || N <= 0 || c_z != C || n_heads != kHeads)
    return 0;
  const size_t np = static_cast<size_t>(N) * N;
  return (np * (4 * C + 2 * kHeads) * sizeof(float) + 255) & ~static_cast<size_t>(255);
}

int foldcp_triattn(const void* z, const void* mask, const foldcp_triattn_params* p, int N, int c_z,
                   int node, void* out, void* stream) {
  if (!p || p->struct_size != sizeof(foldcp_triattn_params)) return FOLDCP_ERR_INVALID_ARG;
  if (p->dtype != FOLDCP_F32 && p->dtype != FOLDCP_BF16) return FOLDCP_ERR_INVALID_ARG;
  if (N <= 0 || c_z <= 0 || p->n_heads <= 0) return FOLDCP_ERR_INVALID_ARG;
  if (node != FOLDCP_TRIATTN_STARTING && node != FOLDCP_TRIATTN_ENDING) return FOLDCP_ERR_INVALID_ARG;
  if (c_z != C || p->n_heads != kHeads) return FOLDCP_ERR_UNSUPPORTED;
  if (N > 32768) return FOLDCP_ERR_UNSUPPORTED;
  const void* req[] = {z, out, p->ln_gamma, p->ln_beta, p->w_q, p->w_k, p->w_v, p->w_g, p->w_t, p->w_o};
  for (const void* r : req)
    if (!r) return FOLDCP_ERR_INVALID_ARG;
  for (const void* r : req)
    if (!aligned16(r)) return FOLDCP_ERR_ALIGNMENT;
  if (mask && !aligned16(mask)) return FOLDCP_ERR_ALIGNMENT;
  const size_t need = foldcp_triattn_workspace_bytes(N, c_z, p->n_heads, p->dtype);
  if (!p->workspace || p->workspace_bytes < need) return FOLDCP_ERR_WORKSPACE;
  if ((reinterpret_cast<uintptr_t>(p->workspace) & 255u) != 0) return FOLDCP_ERR_ALIGNMENT;
  const size_t tbytes = static_cast<size_t>(N) * N * C * (p->dtype == FOLDCP_F32 ? 4 : 2);
  if (overlaps(out, tbytes, z, tbytes) || overlaps(out, tbytes, p->workspace, need) ||
      overlaps(z, tbytes, p->workspace, need))
    return FOLDCP_ERR_ALIAS;
  DeviceInfo d;
  if (!get_device_info(&d)) return FOLDCP_ERR_CUDA;
  if (!(d.cc_major == 10 && d.cc_minor == 0)) return FOLDCP_ERR_ARCH;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  return p->dtype == FOLDCP_F32 ? launch_all<float>(z, mask, p, N, node, out, s)
                                : launch_all<__nv_bfloat16>(z, mask, p, N, node, out, s);
}

}  // extern "C"
