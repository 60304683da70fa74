// Plain CUDA-core (FFMA) implementation of the three stages, fp32 arithmetic throughout.
//
// This is the FOLDCP_F32 "exact" mode (BASELINE.json config 0: relative error <= 1e-5, which TF32
// tensor cores cannot reach -- DESIGN.md reading A11).  The kernels are templated on the storage
// type so the same code can also run on bf16 tensors; that instantiation is the on-device
// cross-check used while bringing up the tcgen05 kernels (FOLDCP_FORCE_SIMT=1), never the default
// bf16 path.
//
// Layouts: z/out [N][N][128] channel-last; a/b/o [128][N][N] channel-major; mask [N][N].
#include <cuda_bf16.h>

#include "common.h"

namespace foldcp {
namespace {

constexpr int C = kChannels;      // 128
constexpr int kPairsPerBlock = 16;

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

__device__ __forceinline__ float sigmoidf_acc(float x) { return 1.0f / (1.0f + expf(-x)); }

// LayerNorm of kPairsPerBlock rows of 128 channels held in smem (one warp per 4 rows).
// rows[p][c] is overwritten with the normalised, affine-transformed value.
__device__ __forceinline__ void block_layernorm(float (*rows)[C], int nrows, const float* gamma,
                                                const float* beta, float eps) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int p = warp; p < nrows; p += 4) {
    float x[4], s = 0.f;
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      x[t] = rows[p][lane + 32 * t];
      s += x[t];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    const float mu = s * (1.0f / C);
    float v = 0.f;
#pragma unroll
    for (int t = 0; t < 4; ++t) v += (x[t] - mu) * (x[t] - mu);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const float rstd = 1.0f / sqrtf(v * (1.0f / C) + eps);
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      const int c = lane + 32 * t;
      rows[p][c] = (x[t] - mu) * rstd * gamma[c] + beta[c];
    }
  }
}

// ---------------------------------------------------------------------------------------------
// stage 1: z' = LN(z);  a = M * sigmoid(W_ga z' + b_ga) * (W_a z' + b_a);  b likewise
// block = 128 threads (thread = output channel), 16 consecutive pairs (flat index over N*N)
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(128)
simt_project_kernel(const T* __restrict__ z, const T* __restrict__ mask, const T* __restrict__ w_a,
                    const T* __restrict__ w_ga, const T* __restrict__ w_b,
                    const T* __restrict__ w_gb, const float* __restrict__ b_a,
                    const float* __restrict__ b_ga, const float* __restrict__ b_b,
                    const float* __restrict__ b_gb, const float* __restrict__ gamma,
                    const float* __restrict__ beta, float eps, long long npairs,
                    T* __restrict__ a_out, T* __restrict__ b_out) {
  __shared__ float zs[kPairsPerBlock][C];
  __shared__ float ms[kPairsPerBlock];
  const long long p0 = static_cast<long long>(blockIdx.x) * kPairsPerBlock;
  const int np = static_cast<int>(min(static_cast<long long>(kPairsPerBlock), npairs - p0));
  const int tid = threadIdx.x;
  for (int p = 0; p < np; ++p) zs[p][tid] = ldf(z + (p0 + p) * C + tid);
  if (tid < np) ms[tid] = mask ? ldf(mask + p0 + tid) : 1.0f;
  __syncthreads();
  block_layernorm(zs, np, gamma, beta, eps);
  __syncthreads();

  float acc[4][kPairsPerBlock];
#pragma unroll
  for (int m = 0; m < 4; ++m)
#pragma unroll
    for (int p = 0; p < kPairsPerBlock; ++p) acc[m][p] = 0.f;
  const T* wr[4] = {w_a + tid * C, w_ga + tid * C, w_b + tid * C, w_gb + tid * C};
  for (int k = 0; k < C; ++k) {
    float w[4];
#pragma unroll
    for (int m = 0; m < 4; ++m) w[m] = ldf(wr[m] + k);
#pragma unroll
    for (int p = 0; p < kPairsPerBlock; ++p) {
      const float x = zs[p][k];
#pragma unroll
      for (int m = 0; m < 4; ++m) acc[m][p] = fmaf(w[m], x, acc[m][p]);
    }
  }
  const float ba = b_a ? b_a[tid] : 0.f, bga = b_ga ? b_ga[tid] : 0.f;
  const float bb = b_b ? b_b[tid] : 0.f, bgb = b_gb ? b_gb[tid] : 0.f;
  for (int p = 0; p < np; ++p) {
    const float av = ms[p] * sigmoidf_acc(acc[1][p] + bga) * (acc[0][p] + ba);
    const float bv = ms[p] * sigmoidf_acc(acc[3][p] + bgb) * (acc[2][p] + bb);
    stf(a_out + static_cast<long long>(tid) * npairs + p0 + p, av);
    stf(b_out + static_cast<long long>(tid) * npairs + p0 + p, bv);
  }
}

// ---------------------------------------------------------------------------------------------
// stage 2: per-channel contraction, 64 x 64 output tile per block, 16 x 16 threads, 4 x 4 each
//   outgoing: o[i][j] = sum_k A[i][k] B[j][k]      incoming: o[i][j] = sum_k A[k][i] B[k][j]
// ---------------------------------------------------------------------------------------------
// nq operand block pairs are contracted into one output block (nq = 1: whole tensors; nq > 1: one
// rank's share of the Cannon-style distributed contraction)
struct BlockPtrs {
  const void* a[kMaxContractBlocks];
  const void* b[kMaxContractBlocks];
  int nq;
};

template <typename T, bool kXMn, bool kYMn>
__global__ void __launch_bounds__(256)
simt_contract_kernel(const BlockPtrs blocks, T* __restrict__ o, int N) {
  constexpr int TS = 64, KS = 16;
  __shared__ float As[KS][TS + 1];
  __shared__ float Bs[KS][TS + 1];
  const long long chan = static_cast<long long>(blockIdx.z) * N * N;
  const int i0 = blockIdx.y * TS, j0 = blockIdx.x * TS;
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  float acc[4][4] = {};
  for (int q = 0; q < blocks.nq; ++q) {
  const T* A = static_cast<const T*>(blocks.a[q]) + chan;
  const T* B = static_cast<const T*>(blocks.b[q]) + chan;
  for (int k0 = 0; k0 < N; k0 += KS) {
    for (int e = threadIdx.x; e < TS * KS; e += 256) {
      // each operand is read along its contiguous index: [k][mn] when MN-major, [mn][k] otherwise
      {
        int mn, kk;
        if (kXMn) { mn = e % TS; kk = e / TS; } else { kk = e % KS; mn = e / KS; }
        const int k = k0 + kk, gi = i0 + mn;
        float av = 0.f;
        if (k < N && gi < N)
          av = ldf(kXMn ? A + static_cast<long long>(k) * N + gi
                        : A + static_cast<long long>(gi) * N + k);
        As[kk][mn] = av;
      }
      {
        int mn, kk;
        if (kYMn) { mn = e % TS; kk = e / TS; } else { kk = e % KS; mn = e / KS; }
        const int k = k0 + kk, gj = j0 + mn;
        float bv = 0.f;
        if (k < N && gj < N)
          bv = ldf(kYMn ? B + static_cast<long long>(k) * N + gj
                        : B + static_cast<long long>(gj) * N + k);
        Bs[kk][mn] = bv;
      }
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < KS; ++kk) {
      float ar[4], br[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        ar[u] = As[kk][ty + 16 * u];
        br[u] = Bs[kk][tx + 16 * u];
      }
#pragma unroll
      for (int u = 0; u < 4; ++u)
#pragma unroll
        for (int v = 0; v < 4; ++v) acc[u][v] = fmaf(ar[u], br[v], acc[u][v]);
    }
    __syncthreads();
  }
  }
#pragma unroll
  for (int u = 0; u < 4; ++u)
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      const int gi = i0 + ty + 16 * u, gj = j0 + tx + 16 * v;
      if (gi < N && gj < N) stf(o + chan + static_cast<long long>(gi) * N + gj, acc[u][v]);
    }
}

// ---------------------------------------------------------------------------------------------
// stage 3: out = [M] * sigmoid(W_g LN(z) + b_g) * (W_o LN(o) + b_o)
// block = 128 threads (thread = output channel), 16 consecutive pairs
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(128)
simt_finalize_kernel(const T* __restrict__ o, const T* __restrict__ z, const T* __restrict__ mask,
                     const T* __restrict__ w_g, const T* __restrict__ w_o,
                     const float* __restrict__ b_g, const float* __restrict__ b_o,
                     const float* __restrict__ g_in, const float* __restrict__ be_in,
                     const float* __restrict__ g_out, const float* __restrict__ be_out, float eps,
                     int mask_output, int add_residual, long long npairs, T* __restrict__ out) {
  __shared__ float zs[kPairsPerBlock][C];
  __shared__ float os[kPairsPerBlock][C];
  __shared__ float ms[kPairsPerBlock];
  const long long p0 = static_cast<long long>(blockIdx.x) * kPairsPerBlock;
  const int np = static_cast<int>(min(static_cast<long long>(kPairsPerBlock), npairs - p0));
  const int tid = threadIdx.x;
  float zres[kPairsPerBlock];
#pragma unroll
  for (int p = 0; p < kPairsPerBlock; ++p) zres[p] = 0.f;
#pragma unroll
  for (int p = 0; p < kPairsPerBlock; ++p) {
    if (p >= np) break;
    zs[p][tid] = ldf(z + (p0 + p) * C + tid);
    if (add_residual) zres[p] = zs[p][tid];
    os[p][tid] = ldf(o + static_cast<long long>(tid) * npairs + p0 + p);
  }
  if (tid < np) ms[tid] = (mask && mask_output) ? ldf(mask + p0 + tid) : 1.0f;
  __syncthreads();
  block_layernorm(zs, np, g_in, be_in, eps);
  block_layernorm(os, np, g_out, be_out, eps);
  __syncthreads();
  float accg[kPairsPerBlock], acco[kPairsPerBlock];
#pragma unroll
  for (int p = 0; p < kPairsPerBlock; ++p) accg[p] = acco[p] = 0.f;
  const T* wg = w_g + tid * C;
  const T* wo = w_o + tid * C;
  for (int k = 0; k < C; ++k) {
    const float g = ldf(wg + k), w = ldf(wo + k);
#pragma unroll
    for (int p = 0; p < kPairsPerBlock; ++p) {
      accg[p] = fmaf(g, zs[p][k], accg[p]);
      acco[p] = fmaf(w, os[p][k], acco[p]);
    }
  }
  const float bg = b_g ? b_g[tid] : 0.f, bo = b_o ? b_o[tid] : 0.f;
#pragma unroll
  for (int p = 0; p < kPairsPerBlock; ++p) {
    if (p >= np) break;
    const float v = ms[p] * sigmoidf_acc(accg[p] + bg) * (acco[p] + bo);
    stf(out + (p0 + p) * C + tid, zres[p] + v);
  }
}

template <typename T>
int project_t(const void* z, const void* mask, const foldcp_trimul_params* p, int N, void* a,
              void* b, cudaStream_t s) {
  const long long npairs = static_cast<long long>(N) * N;
  const unsigned blocks = static_cast<unsigned>((npairs + kPairsPerBlock - 1) / kPairsPerBlock);
  simt_project_kernel<T><<<blocks, 128, 0, s>>>(
      static_cast<const T*>(z), static_cast<const T*>(mask), static_cast<const T*>(p->w_a),
      static_cast<const T*>(p->w_a_gate), static_cast<const T*>(p->w_b),
      static_cast<const T*>(p->w_b_gate), p->b_a, p->b_a_gate, p->b_b, p->b_b_gate,
      p->ln_in_gamma, p->ln_in_beta, p->ln_eps, npairs, static_cast<T*>(a), static_cast<T*>(b));
  return check_launch();
}

// d[c][m][n] = sum_k X(m, k) Y(n, k); x_mn / y_mn: the operand is stored [k][m] / [k][n]
template <typename T>
int gemm_blocks_t(const void* const* x, const void* const* y, int nq, void* d, int N, bool x_mn,
                  bool y_mn, cudaStream_t s) {
  if (nq < 1 || nq > kMaxContractBlocks) return FOLDCP_ERR_UNSUPPORTED;
  const unsigned t = (N + 63) / 64;
  dim3 grid(t, t, C);
  BlockPtrs bp;
  bp.nq = nq;
  for (int q = 0; q < kMaxContractBlocks; ++q) {
    bp.a[q] = x[q < nq ? q : 0];
    bp.b[q] = y[q < nq ? q : 0];
  }
  T* D = static_cast<T*>(d);
  if (x_mn && y_mn) simt_contract_kernel<T, true, true><<<grid, 256, 0, s>>>(bp, D, N);
  else if (x_mn) simt_contract_kernel<T, true, false><<<grid, 256, 0, s>>>(bp, D, N);
  else if (y_mn) simt_contract_kernel<T, false, true><<<grid, 256, 0, s>>>(bp, D, N);
  else simt_contract_kernel<T, false, false><<<grid, 256, 0, s>>>(bp, D, N);
  return check_launch();
}

template <typename T>
int gemm_t(const void* x, const void* y, void* d, int N, bool x_mn, bool y_mn, cudaStream_t s) {
  return gemm_blocks_t<T>(&x, &y, 1, d, N, x_mn, y_mn, s);
}

template <typename T>
int contract_t(const void* a, const void* b, void* o, int N, int direction, cudaStream_t s) {
  const bool inc = direction == FOLDCP_INCOMING;
  return gemm_t<T>(a, b, o, N, inc, inc, s);
}

// same operand assignments as launch_k2_contract_backward_bf16 (k2_contract.cu)
template <typename T>
int contract_backward_t(const void* d_o, const void* a, const void* b, void* d_a, void* d_b, int N,
                        int direction, cudaStream_t s) {
  int st;
  if (direction == FOLDCP_OUTGOING) {
    if ((st = gemm_t<T>(d_o, b, d_a, N, false, true, s)) != FOLDCP_OK) return st;
    return gemm_t<T>(d_o, a, d_b, N, true, true, s);
  }
  if ((st = gemm_t<T>(b, d_o, d_a, N, false, false, s)) != FOLDCP_OK) return st;
  return gemm_t<T>(a, d_o, d_b, N, false, true, s);
}

template <typename T>
int finalize_t(const void* o, const void* z, const void* mask, const foldcp_trimul_params* p,
               int N, void* out, cudaStream_t s) {
  const long long npairs = static_cast<long long>(N) * N;
  const unsigned blocks = static_cast<unsigned>((npairs + kPairsPerBlock - 1) / kPairsPerBlock);
  simt_finalize_kernel<T><<<blocks, 128, 0, s>>>(
      static_cast<const T*>(o), static_cast<const T*>(z), static_cast<const T*>(mask),
      static_cast<const T*>(p->w_g), static_cast<const T*>(p->w_o), p->b_g, p->b_o,
      p->ln_in_gamma, p->ln_in_beta, p->ln_out_gamma, p->ln_out_beta, p->ln_eps, p->mask_output,
      p->add_residual, npairs, static_cast<T*>(out));
  return check_launch();
}

}  // namespace

int launch_simt_project(const void* z, const void* mask, const foldcp_trimul_params* p, int N,
                        void* a, void* b, cudaStream_t s) {
  return p->dtype == FOLDCP_F32 ? project_t<float>(z, mask, p, N, a, b, s)
                                : project_t<__nv_bfloat16>(z, mask, p, N, a, b, s);
}
int launch_simt_contract(const void* a, const void* b, void* o, int N, int dtype, int direction,
                         cudaStream_t s) {
  return dtype == FOLDCP_F32 ? contract_t<float>(a, b, o, N, direction, s)
                             : contract_t<__nv_bfloat16>(a, b, o, N, direction, s);
}
int launch_simt_contract_blocks(const void* const* a_blocks, const void* const* b_blocks, int nq,
                                void* o_block, int nb, int dtype, int direction, cudaStream_t s) {
  const bool inc = direction == FOLDCP_INCOMING;
  return dtype == FOLDCP_F32
             ? gemm_blocks_t<float>(a_blocks, b_blocks, nq, o_block, nb, inc, inc, s)
             : gemm_blocks_t<__nv_bfloat16>(a_blocks, b_blocks, nq, o_block, nb, inc, inc, s);
}
int launch_simt_contract_backward(const void* d_o, const void* a, const void* b, void* d_a,
                                  void* d_b, int N, int dtype, int direction, cudaStream_t s) {
  return dtype == FOLDCP_F32 ? contract_backward_t<float>(d_o, a, b, d_a, d_b, N, direction, s)
                             : contract_backward_t<__nv_bfloat16>(d_o, a, b, d_a, d_b, N, direction, s);
}
int launch_simt_finalize(const void* o, const void* z, const void* mask,
                         const foldcp_trimul_params* p, int N, void* out, cudaStream_t s) {
  return p->dtype == FOLDCP_F32 ? finalize_t<float>(o, z, mask, p, N, out, s)
                                : finalize_t<__nv_bfloat16>(o, z, mask, p, N, out, s);
}

}  // namespace foldcp
