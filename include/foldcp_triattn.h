/*
 * foldcp_triattn.h -- C ABI of triangle attention.
 *
 * The operation (section 3.2, lines 98-115, Eq. 1):
 *       Q, K, V = proj(z),   output = softmax(Q K^T / sqrt(d) + tri_bias(z) + mask_bias) V
 *   "multi-head attention over the rows (or columns) of the pair tensor, with an additive triangular
 *   bias derived from the same representation"; the LayerNorm, the gate and the output projection
 *   around it are those of AF3 supplementary Alg. 14 (starting node, rows) / 15 (ending node,
 *   columns):
 *       z'      = LayerNorm(z; ln_gamma, ln_beta, ln_eps)            over c_z, biased variance
 *       q, k, v = W_q z', W_k z', W_v z'        [N,N,H,c]            no biases
 *       t       = W_t z'                        [N,N,H]              the triangular bias
 *       g       = sigmoid(W_g z')               [N,N,H,c]
 *     starting:  s_ijk = q_ij . k_ik / sqrt(c) + t_jk + mb_ik ,  o_ij = g_ij * sum_k softmax_k(s_ijk) v_ik
 *     ending:    s_ijk = q_ij . k_kj / sqrt(c) + t_ki + mb_kj ,  o_ij = g_ij * sum_k softmax_k(s_ijk) v_kj
 *       out_ij  = W_o concat_h(o_ij)            [N,N,c_z]
 *   with mb = -1e9 * (1 - M) for the pair mask M (values 0 or 1; NULL = all ones).
 *
 * FOLDCP_BF16: three tcgen05 launches -- LayerNorm + q / k / v / gate / bias projections as tensor-core
 * GEMMs, attention with S = Q K^T and O = P V on the tensor cores (softmax on exp2 with a running
 * maximum; q, k, v, the gate, P and the gated output are held as IEEE fp16, the triangular bias as
 * fp16), output projection.  Needs N % 8 == 0 (16-byte TMA strides), like foldcp_trimul.
 * FOLDCP_F32: the exact mode, plain CUDA-core kernels with fp32 arithmetic, any N.
 * Both are checked element by element against the fp64 oracle (oracle/triattn_oracle.py).
 *
 * Conventions as in foldcp_trimul.h: device pointers owned by the caller, params struct in host
 * memory, asynchronous on `stream`, no allocation, status codes of foldcp_status_t.
 */
#ifndef FOLDCP_TRIATTN_H_
#define FOLDCP_TRIATTN_H_

#include "foldcp_trimul.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef enum { FOLDCP_TRIATTN_STARTING = 0, FOLDCP_TRIATTN_ENDING = 1 } foldcp_triattn_node_t;

typedef struct {
  uint32_t struct_size;     /* = sizeof(foldcp_triattn_params) */
  int32_t dtype;            /* FOLDCP_F32 or FOLDCP_BF16: dtype of z, mask, out and the six matrices */
  float ln_eps;
  int32_t n_heads;          /* H; H * c_head = 128, c_head = 32: H = 4 is the supported shape */
  const float* ln_gamma;    /* [c_z] fp32 */
  const float* ln_beta;     /* [c_z] */
  const void* w_q;          /* [H*c_head][c_z] row-major */
  const void* w_k;
  const void* w_v;
  const void* w_g;
  const void* w_t;          /* [H][c_z] */
  const void* w_o;          /* [c_z][H*c_head] */
  void* workspace;          /* >= foldcp_triattn_workspace_bytes(), 256-byte aligned */
  size_t workspace_bytes;
} foldcp_triattn_params;

/*
 *   z, out  [N][N][c_z] device, dtype = params->dtype; c_z = 128; N >= 1 (bf16 mode: N % 8 == 0)
 *   mask    [N][N] device, same dtype, values 0 / 1 (the KEY position's mask enters the softmax as
 *           -1e9; every query row is expected to keep at least one unmasked key)
 *   node    foldcp_triattn_node_t
 * out must not overlap z or the workspace.
 */
int foldcp_triattn(const void* z, const void* mask, const foldcp_triattn_params* params, int N,
                   int c_z, int node, void* out, void* stream);

/* q, k, v, gate (and, in bf16 mode, the gated output) as [N][N][128] in fp32 / fp16 plus the triangular
 * bias in both orientations; 0 if the shape / dtype is unsupported. */
size_t foldcp_triattn_workspace_bytes(int N, int c_z, int n_heads, int dtype);

#ifdef __cplusplus
}
#endif
#endif /* FOLDCP_TRIATTN_H_ */
