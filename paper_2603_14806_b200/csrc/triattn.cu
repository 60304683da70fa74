// Triangle attention (section 3.2 lines 98-115, Eq. 1; AF3 Alg. 14/15).
//
// bf16 mode -- everything on tcgen05, three launches:
//   ta_rows_gemm_kernel<true>   z tile -> LayerNorm (with its affine, in place, fp16) -> q, k, v, gate and
//                               the triangular bias as tensor-core GEMMs; fp16 outputs [pair][128]
//   ta_attention_tc_kernel      per (128 queries, line, head): S = Q K^T into TMEM, softmax warps (thread =
//                               query row) add the bias tile and the key mask and write P = exp2(s - m) as
//                               fp16, O_blk = P V, running output in registers; "line" is the row i
//                               (starting node) or the column j (ending node) -- the ending node is the
//                               same kernel on tensor maps with swapped strides and the transposed bias
//   ta_rows_gemm_kernel<false>  out = W_o (g * o)
// fp32 mode -- the exact mode (1e-5 relative), plain CUDA-core kernels with the same three stages:
//   ta_project_kernel, ta_attention_kernel (online softmax over key chunks in shared memory),
//   ta_output_kernel.
// Layouts: z / out [N][N][128]; intermediates [N][N][128] (head-major inside: h * 32 + d), fp16 in bf16
// mode, fp32 in fp32 mode; triangular bias [H][N][N] in both orientations.
#include <cuda_bf16.h>
#include <cuda_fp16.h>

// The attention kernel's issuing warp waits for the softmax warps most of the time, and it shares an
// SM partition with one softmax warp of every co-resident CTA: without a suspend-time hint its
// try_wait loop was a third of all executed instructions (ncu source page) and slowed exactly the
// warps it was waiting for.
#ifndef FOLDCP_MBAR_HINT_NS
#define FOLDCP_MBAR_HINT_NS 2000
#endif
#include "../../include/foldcp_triattn.h"
#include "common.h"
#include "ln_rows.cuh"
#include "ptx.cuh"

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

constexpr float kLog2e = 1.4426950408889634f;
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
    g[o] = 1.0f / (1.0f + expf(-ag[p]));
    q[o] = aq[p];
    k[o] = ak[p];
    v[o] = av[p];
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


// ---------------------------------------------------------------------------------------------
// Tensor-core attention (bf16 mode): one CTA per (128 queries, line, head), key blocks of 128.
//   S = Q K^T                 tcgen05.mma M=128 (queries) N=128 (keys) K=32, fp16 operands, into TMEM
//   softmax (4 warps, thread = query row = TMEM lane): S + triangular bias tile + key mask, running
//                             maximum, p = exp2(s - m) written as fp16 into the P tile
//   O_blk = P V               tcgen05.mma M=128 N=32 K=128, V tile as an MN-major B operand
//   acc = acc * 2^(m_old - m_new) + O_blk   in registers; out = g * acc / l at the end
// Operand layouts: Q and K tiles [128 rows][32 d] arrive through a 5-D tensor map as unswizzled core
// matrices ([row / 8][d / 8][row % 8][8 halves]: lbo 128, sbo 512 -- the same descriptor form K3's
// rank-one operands use), and the V tile [128 keys][32 d] through the same map: for the product P V it
// is an MN-major operand (d contiguous), the same core matrices read with the roles of lbo / sbo
// swapped (for an MN-major unswizzled operand lbo is the stride between K-adjacent core matrices and
// sbo between MN-adjacent ones -- measured: the other assignment fails parity); the bias tile and P are 128-byte-swizzled K-major tiles of two
// 64-key boxes (K3's z tile).  The ending node is the same kernel on tensor maps with swapped
// strides and the transposed bias -- no data is moved.
// ---------------------------------------------------------------------------------------------
constexpr int kTcThreads = 160;                   // warp 0: TMA + MMA issue; warps 1-4: softmax
// Shared memory, tensor memory and registers are sized for FOUR CTAs per SM (the chain load -> S ->
// softmax -> P V -> running output is serial inside a CTA, and the kernel's speed follows the number
// of resident softmax warps): the P tile overwrites the bias tile in place (a thread turns its own
// row's 16-byte chunks of t into p, same swizzle), the P V result lands in the first 32 of S's 128 TMEM
// columns (S is dead once P is written), and the V tile is loaded into the K tile's buffer once
// S = Q K^T has retired (under the softmax, which takes far longer) -- 49 KB and 128 columns per CTA.
constexpr int kTcOffT = 0;                        // bias tile [128 q][128 k] fp16, two SW128 boxes; then P
constexpr int kTcOffP = kTcOffT;
constexpr int kTcOffK = 32768;                    // K tile, then V tile: unswizzled core matrices, 8 KB
constexpr int kTcOffV = kTcOffK;
constexpr int kTcOffQ = 40960;                    // Q tile     unswizzled core matrices, 8 KB
constexpr int kTcOffM = 49152;                    // key mask bias, 128 floats
constexpr int kTcOffMh = 49664;                   // the same as 128 halves (pass 1 works on half pairs)
constexpr int kTcOffBar = 49920;
constexpr int kTcSmem = kTcOffBar + 64;
constexpr int kTcCtasPerSm = 4;
constexpr int kTcTmemCols = 128;

struct TcAttnParams {
  const __half* g;       // [N*N][128]  sigmoid gate
  const void* mask;      // bf16 [N][N] or nullptr
  __half* og;            // [N*N][128]  g * o: the A operand of the output projection
  int N;
  long long ls, xs;      // pair (line, x) = line * ls + x * xs
};

__global__ void __launch_bounds__(kTcThreads, kTcCtasPerSm)
ta_attention_tc_kernel(const __grid_constant__ CUtensorMap tmap_q,
                       const __grid_constant__ CUtensorMap tmap_k,
                       const __grid_constant__ CUtensorMap tmap_v,
                       const __grid_constant__ CUtensorMap tmap_t, const TcAttnParams prm) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t smem = ptx::smem_u32(smem_raw);
  const uint32_t bar = smem + kTcOffBar;
  const uint32_t bar_q = bar, bar_kv = bar + 8, bar_s = bar + 16, bar_p = bar + 24, bar_o = bar + 32,
                 bar_free = bar + 40, bar_v = bar + 48, tmem_slot = bar + 56;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int N = prm.N;
  const int pos0 = blockIdx.x * 128, line = blockIdx.y, h = blockIdx.z;
  const int nblocks = (N + 127) / 128;

  if (warp == 0) {
    if (lane == 0) {
      ptx::mbar_init(bar_q, 1);
      ptx::mbar_init(bar_kv, 1);
      ptx::mbar_init(bar_s, 1);
      ptx::mbar_init(bar_p, 4);
      ptx::mbar_init(bar_o, 1);
      ptx::mbar_init(bar_free, 4);
      ptx::mbar_init(bar_v, 1);
      ptx::fence_mbar_init();
    }
    __syncwarp();
    ptx::tmem_alloc<1>(tmem_slot, kTcTmemCols);
  }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));
  const uint32_t tm_s = tmem_base, tm_o = tmem_base;   // O block over S's first 32 columns

  if (warp == 0) {
    if (ptx::elect_one()) {
      constexpr uint32_t idesc_s = ptx::make_idesc_f16kind(128, 128, ptx::kFmtF16, ptx::kFmtF16, 0, 0);
      // B = V tile [key][d], d contiguous: an MN-major operand
      constexpr uint32_t idesc_o = ptx::make_idesc_f16kind(128, 32, ptx::kFmtF16, ptx::kFmtF16, 0, 1);
      ptx::mbar_arrive_expect_tx(bar_q, 8192);
      ptx::tma_load_5d(smem + kTcOffQ, &tmap_q, bar_q, 0, 0, h * 4, pos0 / 8, line);
      ptx::mbar_wait(bar_q, 0);
      for (int b = 0; b < nblocks; ++b) {
        const int k0 = b * 128;
        if (b > 0) ptx::mbar_wait(bar_free, (b - 1) & 1);
        ptx::mbar_arrive_expect_tx(bar_kv, 8192 + 32768);
        ptx::tma_load_5d(smem + kTcOffK, &tmap_k, bar_kv, 0, 0, h * 4, k0 / 8, line);
        ptx::tma_load_2d(smem + kTcOffT, &tmap_t, bar_kv, k0, h * N + pos0);
        ptx::tma_load_2d(smem + kTcOffT + 16384, &tmap_t, bar_kv, k0 + 64, h * N + pos0);
        ptx::mbar_wait(bar_kv, b & 1);
        ptx::tc_fence_after();
#pragma unroll
        for (int ks = 0; ks < 2; ++ks)       // K = 32 = two MMAs of K = 16 (two core matrices each)
          ptx::umma_bf16<1>(tm_s, ptx::make_smem_desc_noswizzle(smem + kTcOffQ + ks * 256, 128, 512),
                            ptx::make_smem_desc_noswizzle(smem + kTcOffK + ks * 256, 128, 512), idesc_s,
                            ks ? 1u : 0u);
        ptx::umma_commit<1>(bar_s);
        // S has retired: the K tile is dead, its buffer takes the V tile while the softmax runs
        ptx::mbar_wait(bar_s, b & 1);
        ptx::mbar_arrive_expect_tx(bar_v, 8192);
        ptx::tma_load_5d(smem + kTcOffV, &tmap_v, bar_v, 0, 0, h * 4, k0 / 8, line);
        ptx::mbar_wait(bar_p, b & 1);
        ptx::mbar_wait(bar_v, b & 1);
        ptx::tc_fence_after();
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {     // K = 128 keys
          const uint32_t offp = (ks >> 2) * 16384 + (ks & 3) * 32;
          // V core matrices [key / 8][d / 8][key % 8][8 halves]: key-adjacent 512 B apart (lbo of an
          // MN-major operand), d-adjacent 128 B apart (sbo); one MMA of K = 16 keys = two key groups
          ptx::umma_bf16<1>(tm_o, ptx::make_smem_desc_sw128(smem + kTcOffP + offp, 16, 1024),
                            ptx::make_smem_desc_noswizzle(smem + kTcOffV + ks * 1024, 512, 128), idesc_o,
                            ks ? 1u : 0u);
        }
        ptx::umma_commit<1>(bar_o);
      }
    }
  } else {
    // ===================== softmax: thread = query row =====================
    const int quad = warp & 3;
    const int r = quad * 32 + lane;            // query row of the tile = TMEM lane
    const int st = threadIdx.x - 32;           // 0..127: the key this thread fetches the mask of
    const int pos = pos0 + r;
    const bool active = pos < N;
    const uint32_t lane_addr = static_cast<uint32_t>(quad * 32) << 16;
    const uint32_t sw = static_cast<uint32_t>(r & 7);
    float acc[kHead];
#pragma unroll
    for (int d = 0; d < kHead; ++d) acc[d] = 0.f;
    float m = -INFINITY, l = 0.f;
    for (int b = 0; b < nblocks; ++b) {
      const int k0 = b * 128;
      {
        // mask bias of key k0 + st (in log2 units); keys beyond N do not exist
        float mb = 0.f;
        const int kp = k0 + st;
        if (kp >= N) {
          mb = -INFINITY;
        } else if (prm.mask != nullptr) {
          const float mv = __bfloat162float(static_cast<const __nv_bfloat16*>(prm.mask)[line * prm.ls + kp * prm.xs]);
          mb = -1.0e9f * kLog2e * (1.0f - mv);
        }
        reinterpret_cast<float*>(smem_raw + kTcOffM)[st] = mb;
        reinterpret_cast<__half*>(smem_raw + kTcOffMh)[st] = __float2half_rn(fmaxf(mb, -60000.0f));
      }
      ptx::named_bar_sync(1, 128);
      ptx::mbar_wait(bar_s, b & 1);
      ptx::tc_fence_after();
      // no mask tensor and all 128 keys of the block exist: the per-key term is zero (uniform branch)
      const bool has_mb = prm.mask != nullptr || k0 + 128 > N;
      // this row's 16-byte chunk of the bias / P tile that holds keys kk0 .. kk0 + 7
      auto tchunk = [&](int kk0) -> uint32_t {
        return smem + kTcOffT + (kk0 >> 6) * 16384 + r * 128 + ((static_cast<uint32_t>((kk0 >> 3) & 7) ^ sw) << 4);
      };
      // Both passes read S in eight pieces of 16 columns, the next piece's tcgen05.ld in flight while
      // the current one is worked on (three warps per SM partition cannot hide that latency otherwise).
      // pass 1: the block's row maximum, on half pairs.  The maximum is only the reference point of
      // the exponentials (p and the row sum use the same one), so fp16 accuracy -- a few hundredths
      // at |x| < 100 -- is plenty: p <= 2^0.1.  A masked key is -60000 here (finite: a block with
      // masked keys only still yields a finite reference).
      __half2 hm = __half2half2(__ushort_as_half(static_cast<unsigned short>(0xFC00)));   // -inf
      uint32_t sv[2][16];
      ptx::tmem_ld_32x16(tm_s + lane_addr, sv[0]);
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        ptx::tmem_ld_wait();
        // the last piece's prefetch is pass 2's first piece
        ptx::tmem_ld_32x16(tm_s + lane_addr + ((c + 1) & 7) * 16, sv[(c + 1) & 1]);
#pragma unroll
        for (int i = 0; i < 2; ++i) {
          const int kk0 = c * 16 + i * 8;
          uint32_t tw[4], mw[4];
          ptx::lds128(tchunk(kk0), tw);
          if (has_mb) ptx::lds128(smem + kTcOffMh + kk0 * 2, mw);
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            __half2 xh = __floats2half2_rn(__uint_as_float(sv[c & 1][i * 8 + e * 2]),
                                           __uint_as_float(sv[c & 1][i * 8 + e * 2 + 1]));
            xh = __hadd2(xh, *reinterpret_cast<const __half2*>(&tw[e]));
            if (has_mb) xh = __hadd2(xh, *reinterpret_cast<const __half2*>(&mw[e]));
            hm = __hmax2(hm, xh);
          }
        }
      }
      const float bmax = fmaxf(__low2float(hm), __high2float(hm));
      const float m_new = fmaxf(m, bmax);
      const float m_use = m_new == -INFINITY ? 0.f : m_new;     // a row with no key yet: p = 0 everywhere
      const float resc = ptx::ex2_approx(m - m_use);              // 0 on the first block
      // pass 2: p = exp2(x - m_new), row sum; p replaces t in place (this thread's own chunks)
      float lsum0 = 0.f, lsum1 = 0.f;
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        ptx::tmem_ld_wait();
        if (c + 1 < 8) ptx::tmem_ld_32x16(tm_s + lane_addr + (c + 1) * 16, sv[(c + 1) & 1]);
#pragma unroll
        for (int i = 0; i < 2; ++i) {
          const int kk0 = c * 16 + i * 8;
          uint32_t tw[4], pw[4];
          const uint32_t addr = tchunk(kk0);
          ptx::lds128(addr, tw);
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const float2 tf = __half22float2(*reinterpret_cast<const __half2*>(&tw[e]));
            float x0 = __uint_as_float(sv[c & 1][i * 8 + e * 2]) + tf.x;
            float x1 = __uint_as_float(sv[c & 1][i * 8 + e * 2 + 1]) + tf.y;
            if (has_mb) {
              const float2 mb = *reinterpret_cast<const float2*>(smem_raw + kTcOffM + (kk0 + e * 2) * 4);
              x0 += mb.x;
              x1 += mb.y;
            }
            const float p0 = ptx::ex2_approx(x0 - m_use);
            const float p1 = ptx::ex2_approx(x1 - m_use);
            lsum0 += p0;
            lsum1 += p1;
            pw[e] = ptx::pack_f16x2(p0, p1);
          }
          ptx::sts128(addr, pw[0], pw[1], pw[2], pw[3]);
        }
      }
      const float lsum = lsum0 + lsum1;
      l = l * resc + lsum;
      m = m_new;
      ptx::tc_fence_before();
      ptx::fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(bar_p);
      // O_blk = P V, then the running output
      ptx::mbar_wait(bar_o, b & 1);
      ptx::tc_fence_after();
      uint32_t ov[32];
      ptx::tmem_ld_32x32(tm_o + lane_addr, ov);
      ptx::tmem_ld_wait();
#pragma unroll
      for (int d = 0; d < kHead; ++d) acc[d] = fmaf(acc[d], resc, __uint_as_float(ov[d]));
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(bar_free);
    }
    if (active) {
      // l = 0: a row without any unmasked key (outside the documented precondition) gives zeros
      const float inv = l > 0.f ? 1.0f / l : 0.f;
      const long long a = (static_cast<long long>(line) * prm.ls + static_cast<long long>(pos) * prm.xs) * C + h * kHead;
#pragma unroll
      for (int d = 0; d < kHead; d += 8) {
        const uint4 gv = *reinterpret_cast<const uint4*>(prm.g + a + d);
        const uint32_t gw[4] = {gv.x, gv.y, gv.z, gv.w};
        uint32_t ow[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const float2 gf = __half22float2(*reinterpret_cast<const __half2*>(&gw[e]));
          ow[e] = ptx::pack_f16x2(gf.x * acc[d + 2 * e] * inv, gf.y * acc[d + 2 * e + 1] * inv);
        }
        *reinterpret_cast<uint4*>(prm.og + a + d) = make_uint4(ow[0], ow[1], ow[2], ow[3]);
      }
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 0) ptx::tmem_dealloc<1>(tmem_base, kTcTmemCols);
}


// ---------------------------------------------------------------------------------------------
// Tensor-core projections (bf16 mode).  One persistent kernel, tile = 128 pairs, bulk-synchronous per
// tile (TMA -> LayerNorm -> MMA -> epilogue -> TMA store): these GEMMs move ~1.3 KB per pair against
// the attention's O(N) work per pair, so simplicity wins over overlap here.
//   kProj = true : z tile (bf16) -> LayerNorm with its affine, in place, fp16 -> round A: q, k and the
//                  triangular bias t (N = 16, four rows used); round B: v, gate.  Outputs q16 (times
//                  log2(e) / sqrt(c)), k16, v16, g16 = sigmoid as fp16 [pair][128]; t * log2(e) as fp16 in
//                  both orientations.
//   kProj = false: og tile (fp16, the attention's gated output) -> out = W_o og as bf16.
// Operands exactly as in K3 (pairs = MMA M, output channel = MMA N, K-major 128-byte-swizzled tiles);
// the bf16 weights become fp16 in shared memory once per CTA (exact).
// ---------------------------------------------------------------------------------------------
constexpr int kRgThreads = 256;
constexpr int kRgHalfBox = 128 * 64 * 2;       // 16 KB
constexpr int kRgMat = 2 * kRgHalfBox;         // 32 KB

template <bool kProj>
struct RgSmem {
  static constexpr int kMats = kProj ? 4 : 1;
  static constexpr int kOffW = 0;
  static constexpr int kOffWt = kMats * kRgMat;                 // W_t padded to 16 rows: two boxes of 2 KB
  static constexpr int kOffIn = kOffWt + (kProj ? 4096 : 0);    // input tile
  static constexpr int kOffStage = kOffIn + kRgMat;             // staging [128 pairs][128 ch] 16-bit
  static constexpr int kOffVec = kOffStage + kRgMat;            // gamma[128], beta[128] fp32
  static constexpr int kOffBar = kOffVec + 1024;
  static constexpr int kBytes = kOffBar + 64;
};

struct RgParams {
  const float* gamma;
  const float* beta;
  float eps;
  int N;
  long long R;
  int num_tiles;
  __half* t16s;      // [H][N][N]
  __half* t16e;
};

template <bool kProj>
__global__ void __launch_bounds__(kRgThreads, 1)
ta_rows_gemm_kernel(const __grid_constant__ CUtensorMap tmap_in,
                    const __grid_constant__ CUtensorMap tmap_w0,
                    const __grid_constant__ CUtensorMap tmap_w1,
                    const __grid_constant__ CUtensorMap tmap_w2,
                    const __grid_constant__ CUtensorMap tmap_w3,
                    const __grid_constant__ CUtensorMap tmap_wt,
                    const __grid_constant__ CUtensorMap tmap_o0,
                    const __grid_constant__ CUtensorMap tmap_o1,
                    const __grid_constant__ CUtensorMap tmap_o2,
                    const __grid_constant__ CUtensorMap tmap_o3, const RgParams prm) {
  using L = RgSmem<kProj>;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t smem = ptx::smem_u32(smem_raw);
  const uint32_t bar = smem + L::kOffBar;
  const uint32_t bar_w = bar, bar_in = bar + 8, bar_mma = bar + 16, tmem_slot = bar + 24;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, tid = threadIdx.x;
  const CUtensorMap* wmaps[4] = {&tmap_w0, &tmap_w1, &tmap_w2, &tmap_w3};
  const CUtensorMap* omaps[4] = {&tmap_o0, &tmap_o1, &tmap_o2, &tmap_o3};

  if (tid == 0) {
    ptx::mbar_init(bar_w, 1);
    ptx::mbar_init(bar_in, 1);
    ptx::mbar_init(bar_mma, 1);
    ptx::fence_mbar_init();
  }
  if (warp == 1) ptx::tmem_alloc<1>(tmem_slot, 512);
  if (kProj && tid < 128) {
    reinterpret_cast<float*>(smem_raw + L::kOffVec)[tid] = prm.gamma[tid];
    reinterpret_cast<float*>(smem_raw + L::kOffVec)[128 + tid] = prm.beta[tid];
  }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  // weights: once per CTA, bf16 -> fp16 in place (exact for |w| in [2^-14, 65504])
  if (tid == 0) {
    ptx::mbar_arrive_expect_tx(bar_w, L::kMats * kRgMat + (kProj ? 4096 : 0));
    for (int m = 0; m < L::kMats; ++m) {
      ptx::tma_load_2d(smem + L::kOffW + m * kRgMat, wmaps[m], bar_w, 0, 0);
      ptx::tma_load_2d(smem + L::kOffW + m * kRgMat + kRgHalfBox, wmaps[m], bar_w, 64, 0);
    }
    if (kProj) {
      ptx::tma_load_2d(smem + L::kOffWt, &tmap_wt, bar_w, 0, 0);        // rows 4..15: out of bounds = 0
      ptx::tma_load_2d(smem + L::kOffWt + 2048, &tmap_wt, bar_w, 64, 0);
    }
  }
  ptx::mbar_wait(bar_w, 0);
  ptx::smem_bf16_to_f16_inplace(smem + L::kOffW, L::kMats * kRgMat + (kProj ? 4096 : 0), tid, kRgThreads);
  ptx::fence_proxy_async_smem();
  __syncthreads();

  constexpr uint32_t idesc128 = ptx::make_idesc_f16kind(128, 128, ptx::kFmtF16, ptx::kFmtF16, 0, 0);
  constexpr uint32_t idesc16 = ptx::make_idesc_f16kind(128, 16, ptx::kFmtF16, ptx::kFmtF16, 0, 0);
  const int q4 = warp & 3;                   // TMEM lane quadrant
  const int half = warp >> 2;                // which 64 output channels
  const int r = q4 * 32 + lane;              // pair row of the tile
  const uint32_t lane_addr = static_cast<uint32_t>(q4 * 32) << 16;
  const uint32_t sw = static_cast<uint32_t>(r & 7);
  uint32_t mma_phase = 0;

  auto issue_gemm = [&](int m, uint32_t dcol) {       // D[dcol ..] = in_tile * W_m^T
#pragma unroll
    for (int ks = 0; ks < 8; ++ks) {
      const uint32_t off = (ks >> 2) * kRgHalfBox + (ks & 3) * 32;
      ptx::umma_bf16<1>(tmem_base + dcol, ptx::make_smem_desc_sw128(smem + L::kOffIn + off, 16, 1024),
                        ptx::make_smem_desc_sw128(smem + L::kOffW + m * kRgMat + off, 16, 1024), idesc128,
                        ks ? 1u : 0u);
    }
  };
  // epilogue of one matrix: this thread's 64 channels of its pair -> staging -> one TMA store
  auto epilogue = [&](int m, uint32_t dcol, const CUtensorMap* omap, int tile) {
    if (tid == 0) ptx::tma_store_wait_read<0>();         // the previous store has read the staging tile
    __syncthreads();
#pragma unroll
    for (int c = 0; c < 2; ++c) {
      uint32_t v[32];
      ptx::tmem_ld_32x32(tmem_base + lane_addr + dcol + half * 64 + c * 32, v);
      ptx::tmem_ld_wait();
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        uint32_t pw[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          float x0 = __uint_as_float(v[i * 8 + e * 2]), x1 = __uint_as_float(v[i * 8 + e * 2 + 1]);
          if (kProj) {
            if (m == 0) {                                // q carries 1/sqrt(c) and log2(e)
              x0 *= kLog2e * 0.17677669529663687f;
              x1 *= kLog2e * 0.17677669529663687f;
            } else if (m == 3) {                         // gate
              x0 = 1.0f / (1.0f + __expf(-x0));
              x1 = 1.0f / (1.0f + __expf(-x1));
            }
            pw[e] = ptx::pack_f16x2(x0, x1);
          } else {
            pw[e] = ptx::pack_bf16x2(x0, x1);
          }
        }
        ptx::sts128(smem + L::kOffStage + half * kRgHalfBox + r * 128 +
                        ((static_cast<uint32_t>(c * 4 + i) ^ sw) << 4),
                    pw[0], pw[1], pw[2], pw[3]);
      }
    }
    ptx::tc_fence_before();
    ptx::fence_proxy_async_smem();
    __syncthreads();
    if (tid == 0) {
      ptx::tma_store_2d(omap, smem + L::kOffStage, 0, tile * 128);
      ptx::tma_store_2d(omap, smem + L::kOffStage + kRgHalfBox, 64, tile * 128);
      ptx::tma_store_commit();
    }
  };

  int it = 0;
  if (tid == 0 && static_cast<int>(blockIdx.x) < prm.num_tiles) {
    ptx::mbar_arrive_expect_tx(bar_in, kRgMat);
    ptx::tma_load_2d(smem + L::kOffIn, &tmap_in, bar_in, 0, blockIdx.x * 128);
    ptx::tma_load_2d(smem + L::kOffIn + kRgHalfBox, &tmap_in, bar_in, 64, blockIdx.x * 128);
  }
  for (int t = blockIdx.x; t < prm.num_tiles; t += gridDim.x, ++it) {
    ptx::mbar_wait(bar_in, it & 1);
    if (kProj) {
      layernorm_rows_inplace<true, true, 1, kRgThreads>(smem + L::kOffIn, kRgHalfBox, tid, smem + L::kOffVec,
                                                        smem + L::kOffVec + 512, prm.eps);
      ptx::fence_proxy_async_smem();
    }
    __syncthreads();
    // ---- round A: q, k, t  (or the only matrix)
    if (tid == 0) {
      ptx::tc_fence_after();
      issue_gemm(0, 0);
      if (kProj) {
        issue_gemm(1, 128);
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {
          const uint32_t off = (ks >> 2) * kRgHalfBox + (ks & 3) * 32;
          const uint32_t offt = (ks >> 2) * 2048 + (ks & 3) * 32;
          ptx::umma_bf16<1>(tmem_base + 256, ptx::make_smem_desc_sw128(smem + L::kOffIn + off, 16, 1024),
                            ptx::make_smem_desc_sw128(smem + L::kOffWt + offt, 16, 1024), idesc16,
                            ks ? 1u : 0u);
        }
      }
      ptx::umma_commit<1>(bar_mma);
    }
    ptx::mbar_wait(bar_mma, mma_phase);
    mma_phase ^= 1u;
    ptx::tc_fence_after();
    epilogue(0, 0, omaps[0], t);
    if (kProj) {
      epilogue(1, 128, omaps[1], t);
      if (half == 0) {
        // the triangular bias of this thread's pair: four heads, both orientations
        uint32_t tv[8];
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                     : "=r"(tv[0]), "=r"(tv[1]), "=r"(tv[2]), "=r"(tv[3]), "=r"(tv[4]), "=r"(tv[5]),
                       "=r"(tv[6]), "=r"(tv[7])
                     : "r"(tmem_base + lane_addr + 256)
                     : "memory");
        ptx::tmem_ld_wait();
        const long long pair = static_cast<long long>(t) * 128 + r;
        if (pair < prm.R) {
          const long long i = pair / prm.N, j = pair % prm.N;
#pragma unroll
          for (int h = 0; h < kHeads; ++h) {
            const __half th = __float2half_rn(__uint_as_float(tv[h]) * kLog2e);
            prm.t16s[(static_cast<long long>(h) * prm.N + i) * prm.N + j] = th;
            prm.t16e[(static_cast<long long>(h) * prm.N + j) * prm.N + i] = th;
          }
        }
      }
      // ---- round B: v, gate (the accumulators of round A have been read by everybody)
      ptx::tc_fence_before();
      __syncthreads();
      if (tid == 0) {
        ptx::tc_fence_after();
        issue_gemm(2, 0);
        issue_gemm(3, 128);
        ptx::umma_commit<1>(bar_mma);
      }
      ptx::mbar_wait(bar_mma, mma_phase);
      mma_phase ^= 1u;
      ptx::tc_fence_after();
    }
    // the input tile is free: fetch the next one while the last epilogues run
    if (tid == 0 && t + static_cast<int>(gridDim.x) < prm.num_tiles) {
      ptx::mbar_arrive_expect_tx(bar_in, kRgMat);
      ptx::tma_load_2d(smem + L::kOffIn, &tmap_in, bar_in, 0, (t + gridDim.x) * 128);
      ptx::tma_load_2d(smem + L::kOffIn + kRgHalfBox, &tmap_in, bar_in, 64, (t + gridDim.x) * 128);
    }
    if (kProj) {
      epilogue(2, 0, omaps[2], t);
      epilogue(3, 128, omaps[3], t);
    }
    ptx::tc_fence_before();
    __syncthreads();     // accumulators read before the next tile's MMAs overwrite them
  }
  if (tid == 0) ptx::tma_store_wait<0>();
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 1) ptx::tmem_dealloc<1>(tmem_base, 512);
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

// workspace layout: fp32 mode  q | k | v | g | t | tT  (floats);  bf16 mode  q16 | k16 | v16 | g16 | og16 |
// t16s | t16e  (halves)
size_t workspace_bytes_for(int N, int dtype) {
  const size_t np = static_cast<size_t>(N) * N;
  const size_t b = dtype == FOLDCP_F32 ? np * (4 * C + 2 * kHeads) * sizeof(float)
                                       : np * (5 * C + 2 * kHeads) * sizeof(__half);
  return (b + 255) & ~static_cast<size_t>(255);
}

int launch_f32(const void* z, const void* mask, const foldcp_triattn_params* p, int N, int node,
               void* out, cudaStream_t s) {
  using T = float;
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

int launch_bf16(const void* z, const void* mask, const foldcp_triattn_params* p, int N, int node,
                void* out, cudaStream_t s) {
  DeviceInfo dev;
  if (!get_device_info(&dev)) return FOLDCP_ERR_CUDA;
  const long long npairs = static_cast<long long>(N) * N;
  __half* q16 = static_cast<__half*>(p->workspace);
  __half* k16 = q16 + npairs * C;
  __half* v16 = k16 + npairs * C;
  __half* g16 = v16 + npairs * C;
  __half* og16 = g16 + npairs * C;
  __half* t16s = og16 + npairs * C;
  __half* t16e = t16s + npairs * kHeads;
  const bool starting = node == FOLDCP_TRIATTN_STARTING;
  const uint64_t n = static_cast<uint64_t>(N), R = n * n;
  int st;
  auto rows_map = [&](CUtensorMap* m, const void* base) {   // [R][128] 16-bit, box 64 x 128, SW128
    const uint64_t dims[2] = {C, R};
    const uint64_t strides[1] = {C * 2};
    const uint32_t box[2] = {64, 128};
    return encode_tensor_map(m, base, 2, 2, dims, strides, box, 1);
  };
  auto weight_map = [&](CUtensorMap* m, const void* base, uint64_t rows, uint32_t box_rows) {
    const uint64_t dims[2] = {C, rows};
    const uint64_t strides[1] = {C * 2};
    const uint32_t box[2] = {64, box_rows};
    return encode_tensor_map(m, base, 2, 2, dims, strides, box, 1);
  };
  RgParams rp;
  rp.gamma = p->ln_gamma;
  rp.beta = p->ln_beta;
  rp.eps = p->ln_eps;
  rp.N = N;
  rp.R = npairs;
  rp.num_tiles = static_cast<int>((npairs + 127) / 128);
  rp.t16s = t16s;
  rp.t16e = t16e;
  const int grid_rg = rp.num_tiles < dev.sm_count ? rp.num_tiles : dev.sm_count;
  {
    // LayerNorm + q / k / v / gate / triangular-bias projections on the tensor cores
    CUtensorMap tin, w[4], wt, o[4];
    if ((st = rows_map(&tin, z)) != FOLDCP_OK) return st;
    const void* ws[4] = {p->w_q, p->w_k, p->w_v, p->w_g};
    const void* os[4] = {q16, k16, v16, g16};
    for (int m = 0; m < 4; ++m) {
      if ((st = weight_map(&w[m], ws[m], C, 128)) != FOLDCP_OK) return st;
      if ((st = rows_map(&o[m], os[m])) != FOLDCP_OK) return st;
    }
    if ((st = weight_map(&wt, p->w_t, kHeads, 16)) != FOLDCP_OK) return st;
    auto kern = ta_rows_gemm_kernel<true>;
    if (ensure_dynamic_smem(reinterpret_cast<const void*>(kern), RgSmem<true>::kBytes) != FOLDCP_OK)
      return FOLDCP_ERR_CUDA;
    kern<<<grid_rg, kRgThreads, RgSmem<true>::kBytes, s>>>(tin, w[0], w[1], w[2], w[3], wt, o[0], o[1],
                                                           o[2], o[3], rp);
  }
  {
    CUtensorMap tq, tk, tv, tt;
    // q16 / k16 / v16 [N*N][128] as (8 halves, row % 8, d / 8, row / 8 within the line, line): a box of
    // (8, 8, 4, 16, 1) lands in shared memory as unswizzled 8 x 16-byte core matrices
    const uint64_t row = C * 2;                                    // bytes of one pair's 128 halves
    const uint64_t xs = starting ? row : n * row, ls = starting ? n * row : row;
    const uint64_t dims[5] = {8, 8, C / 8, n / 8, n};
    const uint64_t strides[4] = {xs, 16, 8 * xs, ls};
    const uint32_t box[5] = {8, 8, 4, 16, 1};
    if ((st = encode_tensor_map(&tq, q16, 2, 5, dims, strides, box, 0)) != FOLDCP_OK) return st;
    if ((st = encode_tensor_map(&tk, k16, 2, 5, dims, strides, box, 0)) != FOLDCP_OK) return st;
    if ((st = encode_tensor_map(&tv, v16, 2, 5, dims, strides, box, 0)) != FOLDCP_OK) return st;
    const uint64_t tdims[2] = {n, n * kHeads};
    const uint64_t tstrides[1] = {n * 2};
    const uint32_t tbox[2] = {64, 128};
    if ((st = encode_tensor_map(&tt, starting ? t16s : t16e, 2, 2, tdims, tstrides, tbox, 1)) != FOLDCP_OK)
      return st;
    TcAttnParams prm;
    prm.g = g16;
    prm.mask = mask;
    prm.og = og16;
    prm.N = N;
    prm.ls = starting ? N : 1;
    prm.xs = starting ? 1 : N;
    if (ensure_dynamic_smem(reinterpret_cast<const void*>(ta_attention_tc_kernel), kTcSmem) != FOLDCP_OK)
      return FOLDCP_ERR_CUDA;
    const dim3 grid((N + 127) / 128, N, kHeads);
    ta_attention_tc_kernel<<<grid, kTcThreads, kTcSmem, s>>>(tq, tk, tv, tt, prm);
  }
  {
    // out = W_o (g * o)
    CUtensorMap tin, w, o;
    if ((st = rows_map(&tin, og16)) != FOLDCP_OK) return st;
    if ((st = weight_map(&w, p->w_o, C, 128)) != FOLDCP_OK) return st;
    if ((st = rows_map(&o, out)) != FOLDCP_OK) return st;
    auto kern = ta_rows_gemm_kernel<false>;
    if (ensure_dynamic_smem(reinterpret_cast<const void*>(kern), RgSmem<false>::kBytes) != FOLDCP_OK)
      return FOLDCP_ERR_CUDA;
    kern<<<grid_rg, kRgThreads, RgSmem<false>::kBytes, s>>>(tin, w, w, w, w, w, o, o, o, o, rp);
  }
  return check_launch();
}

}  // namespace
}  // namespace foldcp

using namespace foldcp;

extern "C" {

size_t foldcp_triattn_workspace_bytes(int N, int c_z, int n_heads, int dtype) {
  if ((dtype != FOLDCP_F32 && dtype != FOLDCP_BF16) || N <= 0 || c_z != C || n_heads != kHeads)
    return 0;
  if (dtype == FOLDCP_BF16 && N % 8 != 0) return 0;     // 16-byte TMA row strides, like foldcp_trimul
  return workspace_bytes_for(N, dtype);
}

int foldcp_triattn(const void* z, const void* mask, const foldcp_triattn_params* p, int N, int c_z,
                   int node, void* out, void* stream) {
  if (!p || p->struct_size != sizeof(foldcp_triattn_params)) return FOLDCP_ERR_INVALID_ARG;
  if (p->dtype != FOLDCP_F32 && p->dtype != FOLDCP_BF16) return FOLDCP_ERR_INVALID_ARG;
  if (N <= 0 || c_z <= 0 || p->n_heads <= 0) return FOLDCP_ERR_INVALID_ARG;
  if (node != FOLDCP_TRIATTN_STARTING && node != FOLDCP_TRIATTN_ENDING) return FOLDCP_ERR_INVALID_ARG;
  if (c_z != C || p->n_heads != kHeads) return FOLDCP_ERR_UNSUPPORTED;
  if (N > 32768 || (p->dtype == FOLDCP_BF16 && N % 8 != 0)) return FOLDCP_ERR_UNSUPPORTED;
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
  return p->dtype == FOLDCP_F32 ? launch_f32(z, mask, p, N, node, out, s)
                                : launch_bf16(z, mask, p, N, node, out, s);
}

}  // extern "C"
