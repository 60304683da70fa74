/*
 * foldcp_trimul.h -- C ABI of the B200-native (sm_100a) triangle multiplicative update.
 *
 * The operation (forward pass, one pair tensor, batch 1):
 *   PAPER.md section 3.3, Eq. 2-3:
 *       outgoing  o_nm = sum_k a_nk (.) b_mk        incoming  o_nm = sum_k a_kn (.) b_km
 *   "a, b are projections of the pair representation z in R^{BxNxNxD} ... structurally a batched
 *   matrix multiplication with element-wise gating"; line 132: the variants "differ only in which
 *   operand is transposed".  The LayerNorms, gates and output projection around the contraction
 *   are those of BASELINE.json's north_star (AF3 supplementary Alg. 12/13):
 *
 *       z'  = LayerNorm(z; ln_in_gamma, ln_in_beta, ln_eps)        over c_z, biased variance
 *       a   = M (.) sigmoid(W_ga z' + b_ga) (.) (W_a z' + b_a)     [N,N,c_hidden]
 *       b   = M (.) sigmoid(W_gb z' + b_gb) (.) (W_b z' + b_b)
 *       o   = Eq. 2 (direction = FOLDCP_OUTGOING) or Eq. 3 (FOLDCP_INCOMING), per channel
 *       out = [M (.)] sigmoid(W_g z' + b_g) (.) (W_o LayerNorm(o; ln_out_*) + b_o)   [N,N,c_z]
 *
 *   `out` is the UPDATE only by default (reading A1); params->add_residual = 1 gives
 *   the paper's "z_nm +=" form, out = z + update, fused into the last kernel.
 *
 * Memory: every tensor pointer below is a DEVICE pointer owned by the caller and must stay valid
 * until the work enqueued on `stream` has finished.  The params struct itself is HOST memory and
 * is only read during the call.  The library never allocates, frees or synchronises inside
 * foldcp_trimul(): it enqueues kernels (and one 256-byte memset node) on `stream` and returns.
 *
 * Determinism: same inputs give bitwise identical outputs.  The persistent kernels hand tiles to
 * their CTAs through an atomic counter, but every tile is computed the same way whichever CTA gets
 * it, there is no split-K and no floating-point atomic: the schedule varies, the result does not.
 *
 * Concurrency: the library keeps no device-side global state.  The tile counters of a call live
 * in the last FOLDCP_SCHED_SCRATCH_BYTES of its workspace (or in the `scratch` argument of the
 * stage entry points) and are zeroed on `stream` ahead of the kernels, so any number of calls may
 * be in flight on any number of streams / host threads as long as calls that may overlap in time
 * use different workspaces, scratch areas and outputs.  Calls may be captured into CUDA graphs;
 * a graph replay must not overlap another use of the same workspace.
 *
 * Numeric preconditions of the bf16 mode (FOLDCP_BF16; the fp32 mode has none beyond finiteness):
 *   - inputs finite; |z| below ~1e18 so that the fp32 LayerNorm variance does not overflow (the
 *     fp64 oracle has no such limit; bf16 z in any realistic range is far inside);
 *   - the LayerNorm outputs and the gamma-folded weights W diag(gamma) are held on chip as fp16
 *     operand tiles (11-bit significand instead of bf16's 8): |gamma_k * W[r][k]| must be
 *     <= 65504 (larger values saturate to +-65504) and values below 2^-14 in magnitude are stored
 *     as fp16 subnormals (absolute error <= 2^-25).  tests/test_behaviour_gpu.py shows both edges.
 *   - intermediates: in bf16 mode the gated projections a and b are stored as IEEE fp16
 *     (11-bit significand: their rounding was the largest term of the bf16 pipeline's error
 *     budget), so |a|, |b| must stay <= 65504 -- i.e. |W_a z' + b_a| and
 *     |W_b z' + b_b| <= 65504, far above anything LayerNorm-ed inputs and sane weights give;
 *     larger values saturate.  Inside foldcp_trimul the contraction o travels to the last kernel as
 *     fp16 too, multiplied by foldcp_trimul_o_scale(N) = 2^-ceil(log2(N)/2) ~ 1/sqrt(N) (exact: a
 *     power of two; LayerNorm(o) absorbs it through eps * scale^2): |o| * scale must stay <= 65504,
 *     i.e. |sum_k a b| <= 65504 sqrt(N).  out and all gradients are bf16.
 *   - the output gate's folded weight W_g diag(gamma_in) multiplies the raw bf16 z tile and is
 *     therefore rounded to bf16 (2^-9 relative): invisible at ordinary gate scales, a relative error
 *     of ~5e-3 on the outputs of nearly closed gates when the gate weights are 4x larger
 *     (tests/test_behaviour_gpu.py test_saturated_gates_parity).
 * No exceptions cross this boundary; every failure is a status code and, when detected on the
 * host, leaves `out` untouched.
 */
#ifndef FOLDCP_TRIMUL_H_
#define FOLDCP_TRIMUL_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  FOLDCP_OK = 0,
  FOLDCP_ERR_INVALID_ARG = 1, /* NULL pointer, N <= 0, bad direction / dtype, struct_size mismatch */
  FOLDCP_ERR_UNSUPPORTED = 2, /* c_z or c_hidden != 128; bf16 mode with N not a multiple of 8      */
  FOLDCP_ERR_ALIGNMENT = 3,   /* a tensor pointer is not 16-byte aligned                           */
  FOLDCP_ERR_WORKSPACE = 4,   /* workspace NULL or smaller than foldcp_trimul_workspace_bytes()    */
  FOLDCP_ERR_ALIAS = 5,       /* an output overlaps an input, another output or the workspace     */
  FOLDCP_ERR_ARCH = 6,        /* current device is not compute capability 10.0 (sm_100a cubin)    */
  FOLDCP_ERR_CUDA = 7,        /* launch / tensor-map failure (cudaGetLastError is preserved)       */
  FOLDCP_ERR_STATIC_LIMIT = 8 /* foldcp_trimul_static: the problem needs more scratch than
                               * FOLDCP_STATIC_WORKSPACE_BYTES                                      */
} foldcp_status_t;

typedef enum { FOLDCP_OUTGOING = 0, FOLDCP_INCOMING = 1 } foldcp_direction_t;

/* dtype of z, mask, out and of the six weight matrices.  FOLDCP_F32 is the exact mode
 * (plain fp32 FFMA arithmetic, tolerance 1e-5 relative); FOLDCP_BF16 is the tensor-core mode
 * (bf16 operands, fp32 accumulation in tensor memory). */
typedef enum {
  FOLDCP_F32 = 0,
  FOLDCP_BF16 = 1,
  /* only for foldcp_trimul_contract: a and b are IEEE fp16 -- what foldcp_trimul_project writes in
   * bf16 mode (see "intermediates" below) -- and o is bf16 */
  FOLDCP_BF16_F16AB = 2,
  /* only for foldcp_trimul_contract: a, b fp16 and o ALSO fp16, multiplied by
   * foldcp_trimul_o_scale(N) -- the form in which o travels inside foldcp_trimul (bf16 mode) */
  FOLDCP_BF16_F16ALL = 3
} foldcp_dtype_t;

typedef struct {
  uint32_t struct_size; /* = sizeof(foldcp_trimul_params); ABI versioning                          */
  int32_t dtype;        /* foldcp_dtype_t                                                          */
  float ln_eps;         /* LayerNorm epsilon (inside the sqrt); 1e-5 in every BASELINE config      */
  int32_t mask_output;  /* 1: out_ij *= M_ij (north_star's epilogue); 0: mask only a and b (AF3)   */
  int32_t add_residual; /* 1: out = z + update, the paper's "z_nm +=" form;
                         * 0: out = update only (reading A1)                             */
  int32_t reserved0;    /* must be 0                                                               */
  const float* ln_in_gamma;  /* [c_z]      fp32 in both modes                                      */
  const float* ln_in_beta;   /* [c_z]                                                              */
  const void* w_a;           /* [c_hidden][c_z] row-major (= torch Linear.weight), dtype above     */
  const void* w_a_gate;      /* [c_hidden][c_z]                                                    */
  const void* w_b;           /* [c_hidden][c_z]                                                    */
  const void* w_b_gate;      /* [c_hidden][c_z]                                                    */
  const float* b_a;          /* [c_hidden] fp32; each bias may be NULL (= no bias, AF3 LinearNoBias) */
  const float* b_a_gate;
  const float* b_b;
  const float* b_b_gate;
  const void* w_g;           /* [c_z][c_z]   output gate                                           */
  const float* b_g;          /* [c_z] or NULL                                                      */
  const float* ln_out_gamma; /* [c_hidden] fp32                                                    */
  const float* ln_out_beta;  /* [c_hidden]                                                         */
  const void* w_o;           /* [c_z][c_hidden]   output projection                                */
  const float* b_o;          /* [c_z] or NULL                                                      */
  void* workspace;           /* caller-owned device scratch, 256-byte aligned                      */
  size_t workspace_bytes;    /* >= foldcp_trimul_workspace_bytes(N, c_z, c_hidden, dtype)          */
} foldcp_trimul_params;

/*
 * One forward triangle multiplicative update, enqueued on `stream`.
 *
 *   z      [N][N][c_z]  device, dtype = params->dtype, channel fastest
 *   mask   [N][N]       device, same dtype, PAIR mask multiplied as-is (not thresholded);
 *                       NULL = all ones
 *   params host struct (see above)
 *   N, c_z, c_hidden    N >= 1; c_z = c_hidden = 128 (anything else: FOLDCP_ERR_UNSUPPORTED);
 *                       bf16 mode needs N % 8 == 0 (16-byte TMA row stride) -- pad and mask
 *   direction           foldcp_direction_t
 *   out    [N][N][c_z]  device, dtype = params->dtype; must not overlap z or the workspace
 *   stream              cudaStream_t (as void*); NULL = the legacy default stream
 *
 * Returns a foldcp_status_t.  Asynchronous: returns after enqueueing.
 */
int foldcp_trimul(const void* z, const void* mask, const foldcp_trimul_params* params, int N,
                  int c_z, int c_hidden, int direction, void* out, void* stream);

/*
 * Batched form (z in R^{B x N x N x D}): `batch` independent problems with
 * shared parameters, z [batch][N][N][c_z], mask [batch][N][N] or NULL, out [batch][N][N][c_z].
 * The same workspace (sized for ONE problem) is reused by the batch elements, which are enqueued
 * back to back on `stream`.  Equivalent to `batch` foldcp_trimul calls, bit for bit.
 */
int foldcp_trimul_batched(const void* z, const void* mask, const foldcp_trimul_params* params,
                          int batch, int N, int c_z, int c_hidden, int direction, void* out,
                          void* stream);

/* Bytes of the tile-counter area: the tail of the workspace, and the size of the `scratch`
 * argument of the stage entry points. */
#define FOLDCP_SCHED_SCRATCH_BYTES 256

/* Bytes of device scratch foldcp_trimul needs for this problem (a, b and o, channel-major; in bf16
 * mode 8 bytes per pair of LayerNorm(z) statistics handed from the first kernel to the last; plus
 * FOLDCP_SCHED_SCRATCH_BYTES of tile counters); 0 if the shape / dtype is unsupported.
 * Monotone in N. */
size_t foldcp_trimul_workspace_bytes(int N, int c_z, int c_hidden, int dtype);

/* Stage-level entry points (same conventions; used by the tests, the benchmark's per-kernel
 * roofline and by callers that keep a / b / o).  All tensors are device pointers.
 *
 *   foldcp_trimul_project : step a1+a2 -- LayerNorm + gated projections + mask
 *        a, b  [c_hidden][N][N]  channel-major ("[channel][row][col]" of the pair index);
 *              fp32 in FOLDCP_F32 mode, IEEE fp16 in FOLDCP_BF16 mode
 *   foldcp_trimul_contract: step a4 -- Eq. 2 / Eq. 3 per channel
 *        o     [c_hidden][N][N]  channel-major; dtype = FOLDCP_F32 (a, b, o fp32), FOLDCP_BF16
 *              (a, b, o bf16) or FOLDCP_BF16_F16AB (a, b fp16 as the project stage writes them,
 *              o bf16)
 *   foldcp_trimul_finalize: step a3+a5 -- LayerNorm(o) + output projection + sigmoid gate + mask
 *
 *   scratch: FOLDCP_SCHED_SCRATCH_BYTES of caller-owned device memory, 16-byte aligned, contents
 *        arbitrary (the call zeroes it on `stream`); must not be shared by calls that may overlap
 *        in time.  Required in bf16 mode (FOLDCP_ERR_WORKSPACE if NULL), ignored in fp32 mode.
 *   Outputs must not overlap inputs or each other (FOLDCP_ERR_ALIAS): the kernels are persistent
 *   and store tiles while later tiles still read the operands.
 */
int foldcp_trimul_project(const void* z, const void* mask, const foldcp_trimul_params* params,
                          int N, int c_z, int c_hidden, void* a, void* b, void* scratch,
                          void* stream);
int foldcp_trimul_contract(const void* a, const void* b, int N, int c_hidden, int dtype,
                           int direction, void* o, void* scratch, void* stream);
/*
 * Blocked contraction -- one rank's share of the paper's Cannon-style distributed triangle
 * multiplication (z is tiled as (N / sqrt(P))^2 blocks
 * on a sqrt(P) x sqrt(P) grid, "in each of sqrt(P) steps, ranks perform a local batched matrix
 * multiplication between resident blocks of a and b ... Partial results accumulate into the output
 * block"):
 *     o_block = sum over q < nblocks of Eq. 2 / Eq. 3 applied to (a_blocks[q], b_blocks[q])
 * where rank (r, c) passes, for ring step q,  a_(r, q') and b_(c, q')  (outgoing) or  a_(q', r) and
 * b_(q', c)  (incoming), q' = (r + c + q) mod sqrt(P) (the Cannon order, which spreads the reads
 * over the peers).  Every block is a dense [c_hidden][nb][nb] channel-major tensor of `dtype`
 * (FOLDCP_F32, FOLDCP_BF16 or FOLDCP_BF16_F16AB as for foldcp_trimul_contract).  a_blocks and
 * b_blocks are HOST arrays of nblocks (1..4) DEVICE pointers; a pointer may address a peer GPU's
 * memory that is mapped into this process (cudaDeviceEnablePeerAccess / cuMemMap): on an NVLink /
 * NVSwitch node the ring shifts then become direct TMA reads inside one kernel whose accumulator
 * never leaves tensor memory.  One launch; o_block must not overlap any input block.
 */
int foldcp_trimul_contract_blocks(const void* const* a_blocks, const void* const* b_blocks,
                                  int nblocks, int nb, int c_hidden, int dtype, int direction,
                                  void* o_block, void* scratch, void* stream);

/*
 * Backward of step a4 (the O(N^3) part of training; the paper hand-writes
 * every backward with the forward's algorithm).  Given d_o = dL/do:
 *     outgoing  d_a[i][k] = sum_j d_o[i][j] b[j][k]     d_b[j][k] = sum_i d_o[i][j] a[i][k]
 *     incoming  d_a[k][i] = sum_j b[k][j] d_o[i][j]     d_b[k][j] = sum_i a[k][i] d_o[i][j]
 * per channel.  All five tensors are [c_hidden][N][N] channel-major device pointers of `dtype`;
 * d_a / d_b must not overlap the inputs or each other.  Two launches of the contraction kernel.
 */
int foldcp_trimul_contract_backward(const void* d_o, const void* a, const void* b, int N,
                                    int c_hidden, int dtype, int direction, void* d_a, void* d_b,
                                    void* scratch, void* stream);
int foldcp_trimul_finalize(const void* o, const void* z, const void* mask,
                           const foldcp_trimul_params* params, int N, int c_z, int c_hidden,
                           void* out, void* stream);

/*
 * The same stages in the form foldcp_trimul itself chains them in bf16 mode (FOLDCP_BF16 only;
 * FOLDCP_ERR_UNSUPPORTED otherwise) -- for per-stage timing and per-stage tests of exactly the
 * kernels the fused call launches:
 *   foldcp_trimul_project_stats : foldcp_trimul_project that also leaves, per pair, the LayerNorm(z)
 *        statistics (mean, rstd) as two floats in z_stats [N*N][2] (device, 16-byte aligned)
 *   foldcp_trimul_contract with dtype FOLDCP_BF16_F16ALL : o is fp16, scaled by
 *        foldcp_trimul_o_scale(N)
 *   foldcp_trimul_finalize_fused : o as just described; z_stats from foldcp_trimul_project_stats
 *        (NULL: the statistics are recomputed from z)
 */
int foldcp_trimul_project_stats(const void* z, const void* mask, const foldcp_trimul_params* params,
                                int N, int c_z, int c_hidden, void* a, void* b, void* z_stats,
                                void* scratch, void* stream);
int foldcp_trimul_finalize_fused(const void* o, const void* z, const void* z_stats, const void* mask,
                                 const foldcp_trimul_params* params, int N, int c_z, int c_hidden,
                                 void* out, void* stream);
/* the power of two by which foldcp_trimul scales o between its last two kernels (bf16 mode) */
float foldcp_trimul_o_scale(int N);

/*
 * Full backward pass.  PAPER.md lines 92-96 (section 3.1): every Fold-CP
 * module hand-writes its backward with the same algorithm as its forward.  Given d_out = dL/d(out)
 * of one foldcp_trimul call (same z, mask, params, direction; params->add_residual and
 * params->mask_output as in the forward), computes
 *     d_z   [N][N][c_z]  device, dtype = params->dtype     gradient with respect to z
 *     grads              gradients of all 16 parameters, fp32 in both modes, each [same shape as
 *                        the parameter]; any pointer may be NULL (that gradient is not written)
 * by the chain rule through the definition at the top of this header, in reverse order:
 *     d_y = d_out [M] g, d_g = d_out [M] y            -> dW_o, db_o, dW_g, db_g
 *     d_o = LayerNorm-backward(d_y W_o)               -> dgamma_out, dbeta_out
 *     d_a, d_b = gradients of Eq. 2-3 (foldcp_trimul_contract_backward, on tcgen05 in bf16 mode)
 *     d_z' = sum over the five projections of (their pre-activation gradient) W
 *                                                     -> dW_a, db_a, dW_a_gate, ... (8 tensors)
 *     d_z = LayerNorm-backward(d_z') [+ d_out when add_residual]   -> dgamma_in, dbeta_in
 * Nothing is kept from the forward call: a, b and o are recomputed (by the forward kernels) into
 * params->workspace, which must hold foldcp_trimul_backward_workspace_bytes() bytes.  d_z must not
 * overlap d_out, z or the workspace.  Deterministic: per-block partial sums of the parameter
 * gradients are reduced in a fixed order.  Asynchronous like foldcp_trimul.
 */
typedef struct {
  uint32_t struct_size;      /* = sizeof(foldcp_trimul_grads) */
  uint32_t reserved0;        /* must be 0 */
  float* ln_in_gamma;        /* [c_z] */
  float* ln_in_beta;         /* [c_z] */
  float* w_a;                /* [c_hidden][c_z] row-major, like the parameter */
  float* w_a_gate;
  float* w_b;
  float* w_b_gate;
  float* b_a;                /* [c_hidden] */
  float* b_a_gate;
  float* b_b;
  float* b_b_gate;
  float* w_g;                /* [c_z][c_z] */
  float* b_g;                /* [c_z] */
  float* ln_out_gamma;       /* [c_hidden] */
  float* ln_out_beta;
  float* w_o;                /* [c_z][c_hidden] */
  float* b_o;                /* [c_z] */
} foldcp_trimul_grads;

int foldcp_trimul_backward(const void* d_out, const void* z, const void* mask,
                           const foldcp_trimul_params* params, int N, int c_z, int c_hidden,
                           int direction, void* d_z, const foldcp_trimul_grads* grads,
                           void* stream);

/* Device scratch of foldcp_trimul_backward: a, b, o (d_o in place), d_a, d_b in the tensor dtype,
 * the fp32 accumulator of d_z', staged fp32 weights and per-block partial sums, tile counters.
 * 0 if the shape / dtype is unsupported. */
size_t foldcp_trimul_backward_workspace_bytes(int N, int c_z, int c_hidden, int dtype);

/*
 * foldcp_trimul for callers that cannot allocate device memory (code under CUDA graph capture,
 * serving loops and harnesses that forbid cudaMalloc): same operation, same arguments, same
 * kernels and bitwise the same result as foldcp_trimul, but the scratch (a | b | o | LayerNorm(z)
 * statistics | tile counters) is a `static __device__` array inside the library instead of
 * params->workspace.  params->workspace and params->workspace_bytes are IGNORED (may be NULL / 0);
 * the caller passes only inputs and outputs.  Calls no cudaMalloc, cudaFree or allocating library
 * routine; the first call on each device takes the array's device address (cudaGetSymbolAddress,
 * FOLDCP_ERR_CUDA if that fails) and keeps it.
 *
 *   limit  foldcp_trimul_workspace_bytes(N, c_z, c_hidden, dtype) <= FOLDCP_STATIC_WORKSPACE_BYTES
 *          (16 MiB), i.e. N <= 144 in bf16 mode and N <= 104 in fp32 mode
 *          (foldcp_trimul_static_max_n); beyond it the call launches nothing and returns
 *          FOLDCP_ERR_STATIC_LIMIT -- use foldcp_trimul with a caller-owned workspace.
 *   cost   every GPU on which the library's module is loaded holds those 16 MiB until the process
 *          exits.
 *   sharing  ALL calls on a device share the one array, which keeps the previous call's contents.
 *          Nothing needs clearing by the caller: the tile counters are zeroed on `stream` at every
 *          call and every other byte is written before it is read.  But two foldcp_trimul_static
 *          calls that may OVERLAP on the GPU (different streams without an ordering between them,
 *          or several host threads / graphs replaying concurrently) race on the array and corrupt
 *          each other's result; calls on one stream, or otherwise ordered, are safe.
 * Other errors as foldcp_trimul.
 */
#define FOLDCP_STATIC_WORKSPACE_BYTES (16u << 20)
int foldcp_trimul_static(const void* z, const void* mask, const foldcp_trimul_params* params, int N,
                         int c_z, int c_hidden, int direction, void* out, void* stream);
/* Largest N foldcp_trimul_static accepts for this dtype (0 if the shape / dtype is unsupported). */
int foldcp_trimul_static_max_n(int c_z, int c_hidden, int dtype);
/* = FOLDCP_STATIC_WORKSPACE_BYTES of the library as built */
size_t foldcp_trimul_static_workspace_bytes(void);

/* Number of kernels one foldcp_trimul call launches for this dtype (for launch accounting). */
int foldcp_trimul_launches_per_call(int dtype);

const char* foldcp_status_string(int status);
/* major * 100 + minor * 10; 110 added params->add_residual, foldcp_trimul_batched and
 * foldcp_trimul_contract_backward (the params struct grew: struct_size guards mismatches);
 * 120 made the tile counters per call (workspace grew by FOLDCP_SCHED_SCRATCH_BYTES, the stage
 * entry points take `scratch`) and added foldcp_trimul_backward; 130: the workspace holds the
 * LayerNorm(z) statistics in bf16 mode (8 bytes per pair more), fused-form stage entry points;
 * 140 added foldcp_trimul_static (no existing entry point changed). */
int foldcp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* FOLDCP_TRIMUL_H_ */
