// Backward pass of the triangle multiplicative update around the contraction (
// every Fold-CP module hand-writes its backward with the forward's
// algorithm).  The O(N^3) part -- the gradients of Eq. 2-3 -- runs on the tcgen05 contraction
// kernel (k2_contract.cu); this file holds the O(N^2 c^2) rest as plain CUDA-core kernels with fp32
// arithmetic, templated on the storage type (fp32 exact mode / bf16 tensors):
//
//   K3-backward  d_out -> d_o (through gate, output projection and LayerNorm(o)), the gate's
//                contribution to d_z' and the gradients of W_o, b_o, gamma_out, beta_out, W_g, b_g
//   K1-backward  d_a (then d_b) -> contribution to d_z' through the gated projection; the second
//                pass closes with the LayerNorm(z) backward, writes d_z and the gradients of
//                gamma_in, beta_in; each pass yields the gradients of its W, b, W_gate, b_gate
//
// Forward intermediates are recomputed from z, o (activation recomputation: nothing but a, b, o is
// kept between forward and backward, and those are recomputed by the forward kernels themselves).
//
// Structure of both kernels: persistent blocks of 128 threads, kP = 16 pairs per iteration, chunks
// assigned statically (block b takes chunks b, b + grid, ...), so every block's partial sums -- and
// after the fixed-order reduction every parameter gradient -- are bitwise reproducible.  Weight
// gradients dW = sum_pairs d_y^T x accumulate in shared memory ([k][t], 64 KB per matrix) over the
// block's whole life and are written once; the reduce kernel adds the per-block partials in block
// order.  The weights are staged once per call as fp32 W[t][k] and W^T[k][t] so that both the
// forward product (thread = output channel) and the data gradient (thread = input channel) read
// them coalesced.
#include <cuda_bf16.h>

#include "common.h"

namespace foldcp {
namespace {

constexpr int C = kChannels;   // 128
constexpr int kP = 16;         // pairs per block iteration

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

// ---- staged weights: six matrices, each as W[t][k] and W^T[k][t], fp32 -----------------------
// order: 0 W_a, 1 W_a_gate, 2 W_b, 3 W_b_gate, 4 W_g, 5 W_o
constexpr size_t kMat = static_cast<size_t>(C) * C;
constexpr size_t kStagedWeightsFloats = 12 * kMat;
__device__ __forceinline__ const float* staged_w(const float* base, int m) { return base + 2 * m * kMat; }
__device__ __forceinline__ const float* staged_wt(const float* base, int m) {
  return base + (2 * m + 1) * kMat;
}

struct WeightPtrs {
  const void* w[6];
};

template <typename T>
__global__ void stage_weights_kernel(WeightPtrs wp, float* staged) {
  const int m = blockIdx.y;
  const T* w = static_cast<const T*>(wp.w[m]);
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < C * C; e += gridDim.x * blockDim.x) {
    const int t = e / C, k = e % C;
    const float v = ldf(w + e);
    staged[2 * m * kMat + e] = v;
    staged[(2 * m + 1) * kMat + static_cast<size_t>(k) * C + t] = v;
  }
}

// ---- per-block partial sums ---------------------------------------------------------------------
// One record per block and launch; the reduce kernel sums records in block order.
//   [0, 16384)       dW of matrix A of the launch, stored [k][t]
//   [16384, 32768)   dW of matrix B
//   [32768, +128)    bias gradient A      [32896, +128)  bias gradient B
//   [33024, +128)    LayerNorm gamma grad [33152, +128)  LayerNorm beta grad
constexpr int kPartFloats = 2 * C * C + 4 * C;

// LayerNorm statistics of kP rows held as rows[p][c] (p-major): one warp per 4 rows.  Leaves
// xhat = (x - mean) * rstd in place and returns rstd per row through rstd_out.
__device__ __forceinline__ void block_normalise(float (*rows)[C], int nrows, float eps,
                                                float* rstd_out) {
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
    for (int t = 0; t < 4; ++t) rows[p][lane + 32 * t] = (x[t] - mu) * rstd;
    if (lane == 0) rstd_out[p] = rstd;
  }
}

// sum over the 128 threads (channels) of v[p] for p < kP; result broadcast through `red`
// (red: [4][kP] floats of shared memory).  All 128 threads must call.
__device__ __forceinline__ void block_sum_rows(float (&v)[kP], float (*red)[kP]) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll
  for (int p = 0; p < kP; ++p) {
    float s = v[p];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) red[warp][p] = s;
  }
  __syncthreads();
#pragma unroll
  for (int p = 0; p < kP; ++p) v[p] = (red[0][p] + red[1][p]) + (red[2][p] + red[3][p]);
  __syncthreads();
}

// y[p] = sum_k Wt[k][tid] * x[k][p]   (thread = output channel; x is [k][kP] in shared memory)
__device__ __forceinline__ void gemv_rows(const float* __restrict__ wt, const float (*x)[kP],
                                          float (&acc)[kP]) {
#pragma unroll
  for (int p = 0; p < kP; ++p) acc[p] = 0.f;
  const int tid = threadIdx.x;
#pragma unroll 4
  for (int k = 0; k < C; ++k) {
    const float w = __ldg(wt + k * C + tid);
    const float4* xr = reinterpret_cast<const float4*>(x[k]);
#pragma unroll
    for (int q = 0; q < kP / 4; ++q) {
      const float4 xv = xr[q];
      acc[4 * q + 0] = fmaf(w, xv.x, acc[4 * q + 0]);
      acc[4 * q + 1] = fmaf(w, xv.y, acc[4 * q + 1]);
      acc[4 * q + 2] = fmaf(w, xv.z, acc[4 * q + 2]);
      acc[4 * q + 3] = fmaf(w, xv.w, acc[4 * q + 3]);
    }
  }
}

// acc[p] += sum_t d[t][p] * W[t][tid]   (thread = input channel k; d is [t][kP] in shared memory)
__device__ __forceinline__ void gemv_rows_t(const float* __restrict__ w, const float (*d)[kP],
                                            float (&acc)[kP]) {
  const int tid = threadIdx.x;
#pragma unroll 4
  for (int t = 0; t < C; ++t) {
    const float wv = __ldg(w + t * C + tid);
    const float4* dr = reinterpret_cast<const float4*>(d[t]);
#pragma unroll
    for (int q = 0; q < kP / 4; ++q) {
      const float4 dv = dr[q];
      acc[4 * q + 0] = fmaf(wv, dv.x, acc[4 * q + 0]);
      acc[4 * q + 1] = fmaf(wv, dv.y, acc[4 * q + 1]);
      acc[4 * q + 2] = fmaf(wv, dv.z, acc[4 * q + 2]);
      acc[4 * q + 3] = fmaf(wv, dv.w, acc[4 * q + 3]);
    }
  }
}

// dW[k][tid] += sum_p dy[p] * x[k][p]   (thread = output channel t; dW [k][t] in shared memory)
__device__ __forceinline__ void wgrad_accumulate(float* dW, const float (&dy)[kP],
                                                 const float (*x)[kP]) {
  const int tid = threadIdx.x;
#pragma unroll 4
  for (int k = 0; k < C; ++k) {
    const float4* xr = reinterpret_cast<const float4*>(x[k]);
    float s0 = 0.f, s1 = 0.f;
#pragma unroll
    for (int q = 0; q < kP / 4; ++q) {
      const float4 xv = xr[q];
      s0 = fmaf(dy[4 * q + 0], xv.x, s0);
      s1 = fmaf(dy[4 * q + 1], xv.y, s1);
      s0 = fmaf(dy[4 * q + 2], xv.z, s0);
      s1 = fmaf(dy[4 * q + 3], xv.w, s1);
    }
    dW[k * C + tid] += s0 + s1;
  }
}

struct BwdShared {
  float dWA[C * C];        // [k][t]
  float dWB[C * C];
  float x[C][kP];          // operand of the first product, [k][p]
  float y[C][kP];          // second operand / second product's input
  float xhat[C][kP];       // normalised rows kept for the LayerNorm backward, [k][p]
  float dA[C][kP];         // gradient rows, [t][p]
  float dB[C][kP];
  float rows[kP][C];       // staging for the row-wise LayerNorm statistics, [p][c]
  float rstd[kP];
  float msk[kP];
  float red[4][kP];
};

struct K3BwdParams {
  const void* d_out;       // [R][128]
  const void* z;           // [R][128]
  void* o;                 // [128][R] in: o, out: d_o (in place, per pair)
  const void* mask;        // [R] or nullptr
  const float* staged;     // staged weights
  const float* b_g;        // may be nullptr
  const float* b_o;
  const float* g_in;
  const float* be_in;
  const float* g_out;
  const float* be_out;
  float eps;
  int mask_output;
  long long R;
  float* dzp;              // [R][128] fp32: receives the gate's contribution to d_z'
  float* part;             // [grid][kPartFloats]
};

// ---------------------------------------------------------------------------------------------
// K3-backward
//   forward (recomputed):  z' = LN(z), g = sigmoid(W_g z' + b_g), on = LN(o), y = W_o on + b_o
//   out = Mo g y  =>  d_y = d_out Mo g,  d_gg = d_out Mo y g (1 - g)
//   dW_o = sum d_y^T on, db_o = sum d_y, dW_g = sum d_gg^T z', db_g = sum d_gg
//   d_on = d_y W_o, dgamma_out = sum d_on ohat, dbeta_out = sum d_on, d_o = LN-backward(d_on)
//   dzp  = d_gg W_g   (the gate's share of d_z'; the projections' shares are added by K1-backward)
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(128, 1) simt_finalize_backward_kernel(const K3BwdParams prm) {
  extern __shared__ __align__(16) uint8_t smem_raw[];
  BwdShared& sh = *reinterpret_cast<BwdShared*>(smem_raw);
  const int tid = threadIdx.x;
  const T* d_out = static_cast<const T*>(prm.d_out);
  const T* z = static_cast<const T*>(prm.z);
  T* o = static_cast<T*>(prm.o);
  const T* mask = static_cast<const T*>(prm.mask);
  const float* wt_g = staged_wt(prm.staged, 4);
  const float* wt_o = staged_wt(prm.staged, 5);
  const float* w_g = staged_w(prm.staged, 4);
  const float* w_o = staged_w(prm.staged, 5);
  for (int e = tid; e < C * C; e += 128) {
    sh.dWA[e] = 0.f;
    sh.dWB[e] = 0.f;
  }
  const float bg = prm.b_g ? prm.b_g[tid] : 0.f, bo = prm.b_o ? prm.b_o[tid] : 0.f;
  const float gin = prm.g_in[tid], bin = prm.be_in[tid];
  const float gout = prm.g_out[tid], bout = prm.be_out[tid];
  float db_o = 0.f, db_g = 0.f, dgam = 0.f, dbet = 0.f;
  const long long chunks = (prm.R + kP - 1) / kP;
  for (long long ch = blockIdx.x; ch < chunks; ch += gridDim.x) {
    const long long p0 = ch * kP;
    const int np = static_cast<int>(min(static_cast<long long>(kP), prm.R - p0));
    __syncthreads();
    // ---- z' = LN(z) -> sh.x [k][p]
    for (int p = 0; p < kP; ++p) sh.rows[p][tid] = p < np ? ldf(z + (p0 + p) * C + tid) : 0.f;
    if (tid < kP)
      sh.msk[tid] = (tid < np) ? ((mask && prm.mask_output) ? ldf(mask + p0 + tid) : 1.0f) : 0.f;
    __syncthreads();
    block_normalise(sh.rows, kP, prm.eps, sh.rstd);
    __syncthreads();
#pragma unroll
    for (int p = 0; p < kP; ++p) sh.x[tid][p] = sh.rows[p][tid] * gin + bin;
    __syncthreads();
    // ---- on = LN(o) -> sh.y [k][p], ohat -> sh.xhat
    for (int p = 0; p < kP; ++p)
      sh.rows[p][tid] = p < np ? ldf(o + static_cast<long long>(tid) * prm.R + p0 + p) : 0.f;
    __syncthreads();
    block_normalise(sh.rows, kP, prm.eps, sh.rstd);
    __syncthreads();
#pragma unroll
    for (int p = 0; p < kP; ++p) {
      const float xh = sh.rows[p][tid];
      sh.xhat[tid][p] = xh;
      sh.y[tid][p] = xh * gout + bout;
    }
    __syncthreads();
    // ---- forward products (thread = output channel)
    float accg[kP], acco[kP];
    gemv_rows(wt_g, sh.x, accg);
    gemv_rows(wt_o, sh.y, acco);
    float dy[kP], dgg[kP];
#pragma unroll
    for (int p = 0; p < kP; ++p) {
      const float g = sigmoidf_acc(accg[p] + bg);
      const float y = acco[p] + bo;
      const float dout = (p < np ? ldf(d_out + (p0 + p) * C + tid) : 0.f) * sh.msk[p];
      dy[p] = dout * g;
      dgg[p] = dout * y * g * (1.0f - g);
      db_o += dy[p];
      db_g += dgg[p];
      sh.dA[tid][p] = dy[p];
      sh.dB[tid][p] = dgg[p];
    }
    // ---- weight gradients (thread = output channel t, accumulators [k][t] in shared memory)
    wgrad_accumulate(sh.dWA, dy, sh.y);      // dW_o += d_y^T on
    wgrad_accumulate(sh.dWB, dgg, sh.x);     // dW_g += d_gg^T z'
    __syncthreads();
    // ---- data gradients (thread = input channel k)
    float don[kP], dzg[kP];
#pragma unroll
    for (int p = 0; p < kP; ++p) don[p] = dzg[p] = 0.f;
    gemv_rows_t(w_o, sh.dA, don);
    gemv_rows_t(w_g, sh.dB, dzg);
    float m1[kP], m2[kP];
#pragma unroll
    for (int p = 0; p < kP; ++p) {
      const float xh = sh.xhat[tid][p];
      dgam += don[p] * xh;
      dbet += don[p];
      don[p] *= gout;                         // d_ohat
      m1[p] = don[p];
      m2[p] = don[p] * xh;
    }
    block_sum_rows(m1, sh.red);
    block_sum_rows(m2, sh.red);
    for (int p = 0; p < np; ++p) {
      const float xh = sh.xhat[tid][p];
      const float v = sh.rstd[p] * (don[p] - m1[p] * (1.0f / C) - xh * m2[p] * (1.0f / C));
      stf(o + static_cast<long long>(tid) * prm.R + p0 + p, v);
      prm.dzp[(p0 + p) * C + tid] = dzg[p];
    }
  }
  __syncthreads();
  float* part = prm.part + static_cast<size_t>(blockIdx.x) * kPartFloats;
  for (int e = tid; e < C * C; e += 128) {
    part[e] = sh.dWA[e];
    part[C * C + e] = sh.dWB[e];
  }
  part[2 * C * C + tid] = db_o;
  part[2 * C * C + C + tid] = db_g;
  part[2 * C * C + 2 * C + tid] = dgam;
  part[2 * C * C + 3 * C + tid] = dbet;
}

struct K1BwdParams {
  const void* z;           // [R][128]
  const void* mask;        // [R] or nullptr
  const void* d_t;         // [128][R] gradient of the projected tensor of this pass (d_a or d_b)
  const void* d_out;       // [R][128], only read when add_residual
  const float* staged;
  int m_proj;              // staged matrix index of the projection (0: W_a, 2: W_b); gate = +1
  const float* b_proj;     // may be nullptr
  const float* b_gate;
  const float* g_in;
  const float* be_in;
  float eps;
  int add_residual;
  long long R;
  float* dzp;              // [R][128] fp32, read-modify-write
  void* d_z;               // [R][128], written by the final pass
  float* part;
};

// ---------------------------------------------------------------------------------------------
// K1-backward, one pass per projected tensor t in {a, b}:
//   forward (recomputed): z' = LN(z), p = W z' + b, gate = W_gate z' + b_gate, s = sigmoid(gate)
//   t = M s p  =>  d_p = d_t M s,  d_gate = d_t M p s (1 - s)
//   dW = sum d_p^T z', db = sum d_p, dW_gate = sum d_gate^T z', db_gate = sum d_gate
//   dzp += d_p W + d_gate W_gate
// kFinal (second pass): d_z = LN-backward(dzp) [+ d_out], dgamma_in = sum dzp zhat, dbeta_in = sum dzp
// ---------------------------------------------------------------------------------------------
template <typename T, bool kFinal>
__global__ void __launch_bounds__(128, 1) simt_project_backward_kernel(const K1BwdParams prm) {
  extern __shared__ __align__(16) uint8_t smem_raw[];
  BwdShared& sh = *reinterpret_cast<BwdShared*>(smem_raw);
  const int tid = threadIdx.x;
  const T* z = static_cast<const T*>(prm.z);
  const T* mask = static_cast<const T*>(prm.mask);
  const T* d_t = static_cast<const T*>(prm.d_t);
  const float* wt_p = staged_wt(prm.staged, prm.m_proj);
  const float* wt_s = staged_wt(prm.staged, prm.m_proj + 1);
  const float* w_p = staged_w(prm.staged, prm.m_proj);
  const float* w_s = staged_w(prm.staged, prm.m_proj + 1);
  for (int e = tid; e < C * C; e += 128) {
    sh.dWA[e] = 0.f;
    sh.dWB[e] = 0.f;
  }
  const float bp = prm.b_proj ? prm.b_proj[tid] : 0.f, bs = prm.b_gate ? prm.b_gate[tid] : 0.f;
  const float gin = prm.g_in[tid], bin = prm.be_in[tid];
  float db_p = 0.f, db_s = 0.f, dgam = 0.f, dbet = 0.f;
  const long long chunks = (prm.R + kP - 1) / kP;
  for (long long ch = blockIdx.x; ch < chunks; ch += gridDim.x) {
    const long long p0 = ch * kP;
    const int np = static_cast<int>(min(static_cast<long long>(kP), prm.R - p0));
    __syncthreads();
    for (int p = 0; p < kP; ++p) sh.rows[p][tid] = p < np ? ldf(z + (p0 + p) * C + tid) : 0.f;
    if (tid < kP) sh.msk[tid] = (tid < np) ? (mask ? ldf(mask + p0 + tid) : 1.0f) : 0.f;
    __syncthreads();
    block_normalise(sh.rows, kP, prm.eps, sh.rstd);
    __syncthreads();
#pragma unroll
    for (int p = 0; p < kP; ++p) {
      const float xh = sh.rows[p][tid];
      sh.xhat[tid][p] = xh;
      sh.x[tid][p] = xh * gin + bin;
    }
    __syncthreads();
    float accp[kP], accs[kP];
    gemv_rows(wt_p, sh.x, accp);
    gemv_rows(wt_s, sh.x, accs);
    float dp[kP], ds[kP];
#pragma unroll
    for (int p = 0; p < kP; ++p) {
      const float pv = accp[p] + bp;
      const float s = sigmoidf_acc(accs[p] + bs);
      const float dt =
          (p < np ? ldf(d_t + static_cast<long long>(tid) * prm.R + p0 + p) : 0.f) * sh.msk[p];
      dp[p] = dt * s;
      ds[p] = dt * pv * s * (1.0f - s);
      db_p += dp[p];
      db_s += ds[p];
      sh.dA[tid][p] = dp[p];
      sh.dB[tid][p] = ds[p];
    }
    wgrad_accumulate(sh.dWA, dp, sh.x);
    wgrad_accumulate(sh.dWB, ds, sh.x);
    __syncthreads();
    float dz[kP];
#pragma unroll
    for (int p = 0; p < kP; ++p) dz[p] = p < np ? prm.dzp[(p0 + p) * C + tid] : 0.f;
    gemv_rows_t(w_p, sh.dA, dz);
    gemv_rows_t(w_s, sh.dB, dz);
    if constexpr (!kFinal) {
      for (int p = 0; p < np; ++p) prm.dzp[(p0 + p) * C + tid] = dz[p];
    } else {
      float m1[kP], m2[kP];
#pragma unroll
      for (int p = 0; p < kP; ++p) {
        const float xh = sh.xhat[tid][p];
        dgam += dz[p] * xh;
        dbet += dz[p];
        dz[p] *= gin;                           // d_zhat
        m1[p] = dz[p];
        m2[p] = dz[p] * xh;
      }
      block_sum_rows(m1, sh.red);
      block_sum_rows(m2, sh.red);
      T* d_z = static_cast<T*>(prm.d_z);
      const T* d_out = static_cast<const T*>(prm.d_out);
      for (int p = 0; p < np; ++p) {
        const float xh = sh.xhat[tid][p];
        float v = sh.rstd[p] * (dz[p] - m1[p] * (1.0f / C) - xh * m2[p] * (1.0f / C));
        if (prm.add_residual) v += ldf(d_out + (p0 + p) * C + tid);
        stf(d_z + (p0 + p) * C + tid, v);
      }
    }
  }
  __syncthreads();
  float* part = prm.part + static_cast<size_t>(blockIdx.x) * kPartFloats;
  for (int e = tid; e < C * C; e += 128) {
    part[e] = sh.dWA[e];
    part[C * C + e] = sh.dWB[e];
  }
  part[2 * C * C + tid] = db_p;
  part[2 * C * C + C + tid] = db_s;
  part[2 * C * C + 2 * C + tid] = dgam;
  part[2 * C * C + 3 * C + tid] = dbet;
}

// ---- fixed-order reduction of the per-block partials into the caller's gradient buffers --------
struct ReduceParams {
  const float* part;   // [nblocks][kPartFloats]
  int nblocks;
  float* dWA;          // [t][k] row-major (torch Linear.weight layout) or nullptr
  float* dWB;
  float* v0;           // four [128] vectors, each may be nullptr
  float* v1;
  float* v2;
  float* v3;
};

__global__ void reduce_partials_kernel(const ReduceParams prm) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= kPartFloats) return;
  float s = 0.f;
  for (int b = 0; b < prm.nblocks; ++b) s += prm.part[static_cast<size_t>(b) * kPartFloats + e];
  if (e < 2 * C * C) {
    float* dst = e < C * C ? prm.dWA : prm.dWB;
    const int r = e % (C * C), k = r / C, t = r % C;     // partials are [k][t]
    if (dst) dst[t * C + k] = s;
  } else {
    const int r = e - 2 * C * C, which = r / C, i = r % C;
    float* dst = which == 0 ? prm.v0 : which == 1 ? prm.v1 : which == 2 ? prm.v2 : prm.v3;
    if (dst) dst[i] = s;
  }
}

int backward_grid(const DeviceInfo& dev, long long R) {
  const long long chunks = (R + kP - 1) / kP;
  const long long blocks = dev.sm_count < kMaxBackwardBlocks ? dev.sm_count : kMaxBackwardBlocks;
  return static_cast<int>(chunks < blocks ? chunks : blocks);
}

template <typename T>
int tail_backward_t(const void* d_out, const void* z, const void* mask,
                    const foldcp_trimul_params* p, int N, void* o_io, const void* d_a,
                    const void* d_b, int phase, float* dzp, float* staged, float* part,
                    const foldcp_trimul_grads* g, void* d_z, cudaStream_t s) {
  DeviceInfo dev;
  if (!get_device_info(&dev)) return FOLDCP_ERR_CUDA;
  const long long R = static_cast<long long>(N) * N;
  const int grid = backward_grid(dev, R);
  const int smem = static_cast<int>(sizeof(BwdShared));
  ReduceParams rp;
  rp.part = part;
  rp.nblocks = grid;
  const int rgrid = (kPartFloats + 255) / 256;
  if (phase == 0) {
    // weights staged once per call, then K3-backward
    WeightPtrs wp;
    wp.w[0] = p->w_a; wp.w[1] = p->w_a_gate; wp.w[2] = p->w_b; wp.w[3] = p->w_b_gate;
    wp.w[4] = p->w_g; wp.w[5] = p->w_o;
    stage_weights_kernel<T><<<dim3(16, 6), 256, 0, s>>>(wp, staged);
    auto kern = simt_finalize_backward_kernel<T>;
    if (ensure_dynamic_smem(reinterpret_cast<const void*>(kern), smem) != FOLDCP_OK)
      return FOLDCP_ERR_CUDA;
    K3BwdParams k;
    k.d_out = d_out; k.z = z; k.o = o_io; k.mask = mask; k.staged = staged;
    k.b_g = p->b_g; k.b_o = p->b_o; k.g_in = p->ln_in_gamma; k.be_in = p->ln_in_beta;
    k.g_out = p->ln_out_gamma; k.be_out = p->ln_out_beta; k.eps = p->ln_eps;
    k.mask_output = p->mask_output; k.R = R; k.dzp = dzp; k.part = part;
    kern<<<grid, 128, smem, s>>>(k);
    rp.dWA = g->w_o; rp.dWB = g->w_g; rp.v0 = g->b_o; rp.v1 = g->b_g;
    rp.v2 = g->ln_out_gamma; rp.v3 = g->ln_out_beta;
    reduce_partials_kernel<<<rgrid, 256, 0, s>>>(rp);
    return check_launch();
  }
  const bool final_pass = phase == 2;
  K1BwdParams k;
  k.z = z; k.mask = mask; k.d_t = final_pass ? d_b : d_a; k.d_out = d_out; k.staged = staged;
  k.m_proj = final_pass ? 2 : 0;
  k.b_proj = final_pass ? p->b_b : p->b_a;
  k.b_gate = final_pass ? p->b_b_gate : p->b_a_gate;
  k.g_in = p->ln_in_gamma; k.be_in = p->ln_in_beta; k.eps = p->ln_eps;
  k.add_residual = p->add_residual; k.R = R; k.dzp = dzp; k.d_z = d_z; k.part = part;
  if (final_pass) {
    auto kern = simt_project_backward_kernel<T, true>;
    if (ensure_dynamic_smem(reinterpret_cast<const void*>(kern), smem) != FOLDCP_OK)
      return FOLDCP_ERR_CUDA;
    kern<<<grid, 128, smem, s>>>(k);
    rp.dWA = g->w_b; rp.dWB = g->w_b_gate; rp.v0 = g->b_b; rp.v1 = g->b_b_gate;
    rp.v2 = g->ln_in_gamma; rp.v3 = g->ln_in_beta;
  } else {
    auto kern = simt_project_backward_kernel<T, false>;
    if (ensure_dynamic_smem(reinterpret_cast<const void*>(kern), smem) != FOLDCP_OK)
      return FOLDCP_ERR_CUDA;
    kern<<<grid, 128, smem, s>>>(k);
    rp.dWA = g->w_a; rp.dWB = g->w_a_gate; rp.v0 = g->b_a; rp.v1 = g->b_a_gate;
    rp.v2 = nullptr; rp.v3 = nullptr;
  }
  reduce_partials_kernel<<<rgrid, 256, 0, s>>>(rp);
  return check_launch();
}

}  // namespace

size_t backward_scratch_floats(int blocks) {
  return kStagedWeightsFloats + static_cast<size_t>(blocks) * kPartFloats;
}

// phase 0: K3-backward (o -> d_o in place, dzp written); phase 1: K1-backward for a (d_a);
// phase 2: K1-backward for b (d_b), closing with the LayerNorm(z) backward -> d_z.
// `scratch` = backward_scratch_floats() floats: staged weights followed by the per-block partials.
int launch_simt_tail_backward(int phase, const void* d_out, const void* z, const void* mask,
                              const foldcp_trimul_params* p, int N, void* o_io, const void* d_a,
                              const void* d_b, float* dzp, float* scratch,
                              const foldcp_trimul_grads* g, void* d_z, cudaStream_t s) {
  float* staged = scratch;
  float* part = scratch + kStagedWeightsFloats;
  return p->dtype == FOLDCP_F32
             ? tail_backward_t<float>(d_out, z, mask, p, N, o_io, d_a, d_b, phase, dzp, staged,
                                      part, g, d_z, s)
             : tail_backward_t<__nv_bfloat16>(d_out, z, mask, p, N, o_io, d_a, d_b, phase, dzp,
                                              staged, part, g, d_z, s);
}

}  // namespace foldcp
