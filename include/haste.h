/* include/haste.h -- C ABI of the HASTE hot path on one B200 (sm_100a).
 *
 * What it is: the group-shared fixed fan-in sparse output layer of HASTE
 * (arxiv/paper_2606_01117) and its small dense head, forward fused with the
 * BCE-with-logits objective, plus the full backward.  Citations are lines of the
 * paper's text (PAPER.md:<line>):
 *
 *   labels are partitioned into groups of G; group g shares one support
 *   I_g = idx[g, 0..K) of K input features, label l keeps its own K weights
 *   W[l, 0..K):
 *     z[i,l]  = bias[l] + sum_j W[l,j] * X[i, idx[l/G, j]]
 *     loss    = s * sum_i sum_l ( softplus(z[i,l]) - y[i,l] z[i,l] ) PAPER.md:111 (Eq. 3), s = 1/B
 *     dY[i,l] = s * ( sigmoid(z[i,l]) - y[i,l] )
 *     dW[l,j] = sum_i dY[i,l] * X[i, idx[l/G, j]]
 *     dX[i,f] = sum_l sum_{j: idx[l/G,j]=f} dY[i,l] * W[l,j]
 *   dense head over the frequent labels: z = b + X_h W_h^T, same objective,
 *     dW_h = dY^T X_h, dX_h = dY W_h
 *
 * (Paper symbols: H -> d, F -> K, number of groups K_paper -> NG = ceil(L/G).)
 *
 * Conventions
 *  - Every tensor pointer is DEVICE memory owned by the caller (unless a
 *    parameter says "host"); the library never frees or keeps it past the call.
 *    A handle owns only its workspace (X^T copy, dX^T accumulator, loss partials,
 *    TMA descriptors), sized from B_max at create and freed at destroy.
 *  - Calls enqueue work on `stream` (a cudaStream_t passed as void*; NULL is the
 *    legacy default stream) and return without synchronising.  `loss` is a device
 *    scalar.  A handle is not thread-safe: one stream at a time per handle.
 *  - Every function returns a haste_status_t; 0 is success.  Nothing throws, aborts
 *    or prints.  Argument errors are detected on the host before any launch.
 *    Index CONTENTS are not checked by the hot calls; haste_validate_index does it.
 *  - Pointers to X, W, idx, dY, dW (and Z, momentum) must be 16-byte aligned.
 *  - idx rows may hold any values in [0,d): duplicates add, order is free
 *    (reading R4).  HASTE_IDX_SORTED_DISTINCT is a caller's promise that
 *    haste_validate_index checks; no kernel relies on it (the dX kernel tests every
 *    row itself and sends a row that is not strictly ascending down its atomic path).
 *  - Targets: one CSR over GLOBAL label ids, ascending and distinct within a row;
 *    a layer looks only at ids in [label_offset, label_offset + L).
 *  - dY of the sparse tail lives in a library-defined layout (group-blocked:
 *    element (i,l) at ((l/G)*B + i)*G + l%G, type `dtype`); use haste_dy_bytes,
 *    haste_dy_unpack and haste_dy_pack to size and convert it.  dY of the head is
 *    plain [B, L_h] row-major.
 */
#ifndef HASTE_H_
#define HASTE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct haste_layer haste_layer_t; /* opaque; sparse tail */
typedef struct haste_head haste_head_t;   /* opaque; dense head  */

typedef enum {
  HASTE_OK = 0,
  HASTE_ERR_INVALID_ARG = -1, /* NULL required pointer, B > B_max, misaligned pointer, bad sizes */
  HASTE_ERR_BAD_INDEX = -2,   /* haste_validate_index: value outside [0,d) or broken sorted-distinct promise */
  HASTE_ERR_UNSUPPORTED = -3, /* shape/dtype the kernels do not cover */
  HASTE_ERR_CUDA = -4,        /* CUDA runtime/driver error; text in haste_last_error() */
  HASTE_ERR_NOMEM = -5
} haste_status_t;

typedef enum { HASTE_F32 = 0, HASTE_BF16 = 1 } haste_dtype_t;

typedef enum {
  HASTE_IDX_SORTED_DISTINCT = 1u, /* promise: every idx row strictly ascending */
  HASTE_DETERMINISTIC = 2u,       /* no float atomics on dX: bit-identical results from run to run (slower path; the sparse tail
                                     needs a shape of the tcgen05 family for it, else haste_create returns HASTE_ERR_UNSUPPORTED;
                                     costs a workspace of num_SMs * d * 512 bytes) */
  HASTE_FORCE_SIMT = 4u,          /* use the generic CUDA-core kernels even where tcgen05 kernels exist */
  HASTE_XT_FROM_FORWARD = 8u      /* promise: every haste_backward on this handle follows a haste_forward_loss (or
                                     haste_forward_logits) on the SAME handle with the SAME X and B, nothing in between on that
                                     handle: the backward then reuses the forward's transposed copy of X instead of rebuilding
                                     it (one launch and ~9 us less per step at config 3).  Without the flag the backward
                                     never depends on an earlier call. */
} haste_flags_t;

typedef struct {
  int32_t d;              /* input features (paper H)                                       */
  int64_t L;              /* labels in THIS layer; need not be a multiple of G (R3)         */
  int32_t G, K;           /* labels per group; fan-in per group (paper F)                   */
  int32_t B_max;          /* largest batch any call will pass                               */
  haste_dtype_t dtype;    /* type of X, W, dY; accumulation is always fp32                  */
  haste_dtype_t dw_dtype; /* type of dW                                                     */
  int64_t label_offset;   /* global id of this layer's label 0 in the targets' CSR          */
  float loss_scale;       /* 0 -> 1/B per call (Eq. 3); otherwise used as given             */
  uint32_t flags;         /* haste_flags_t bits                                             */
} haste_config_t;

/* ---- sparse tail ------------------------------------------- */

/* Allocates the handle and its workspace on `cuda_device`.  *out is NULL on failure. */
int haste_create(haste_layer_t** out, const haste_config_t* cfg, int cuda_device);
int haste_destroy(haste_layer_t* h);

/* Bytes of the dY buffer for a call with batch B (NG * B * G elements of `dtype`). */
size_t haste_dy_bytes(const haste_layer_t* h, int B);

/* Checks idx [NG,K] (device): every value in [0,d) and, if the handle promised
 * HASTE_IDX_SORTED_DISTINCT, every row strictly ascending.  Synchronises `stream`.
 * Returns HASTE_OK or HASTE_ERR_BAD_INDEX. */
int haste_validate_index(haste_layer_t* h, const int32_t* idx, void* stream);

/* Forward + fused BCE-with-logits.  The B x L logits are not
 * written unless logits_out is given. */
int haste_forward_loss(haste_layer_t* h, int B,
                       const void* X,             /* [B,d] row-major, dtype                                   */
                       const int32_t* idx,        /* [NG,K] int32, NG = ceil(L/G); values in [0,d)            */
                       const void* W,             /* [L,K] row-major, dtype                                   */
                       const float* bias,         /* [L] fp32 or NULL                                         */
                       const int32_t* tgt_rowptr, /* [B+1]                                                    */
                       const int32_t* tgt_col,    /* [nnz] global label ids, ascending within a row           */
                       float* loss,               /* device scalar, overwritten; NULL -> not computed         */
                       void* dY,                  /* haste_dy_bytes(h,B), overwritten; NULL -> inference only */
                       float* logits_out,         /* optional [B,L] row-major fp32, or NULL                   */
                       void* stream);

/* Forward + fused BCE AND the weight gradient in one call (the first slice of the single-pass step):
 * exactly haste_forward_loss(..., logits_out = NULL) followed by haste_backward(..., dW, dbias, dX = NULL) -- the same
 * loss, dY, dW (in the handle's dw_dtype) and dbias, with the same argument meanings, layouts and ownership.  dY is
 * required (the input-gradient step, haste_backward with dX only, still reads it).  For bf16 handles with G = 64,
 * K in {64, 128} and B <= 512 this is ONE kernel in which the gathered tile X[:, idx_g] and the dY tile just produced are
 * still on chip when the weight-gradient contraction runs: dY is written once and never read back, X^T is gathered
 * once.  Every other shape runs the two calls one after the other.  X, idx, W, dY, dW 16-byte aligned. */
int haste_forward_loss_dw(haste_layer_t* h, int B, const void* X, const int32_t* idx, const void* W, const float* bias,
                          const int32_t* tgt_rowptr, const int32_t* tgt_col, float* loss, void* dY,
                          void* dW /* [L,K] dw_dtype or NULL */, float* dbias /* [L] fp32 or NULL */, void* stream);

/* Logits-only forward (z = <w_l, h_I> per label; the inference pass behind Eq. 4):
 * Z receives z[i,l] = bias[l] + sum_j W[l,j] X[i, idx[l/G, j]] rounded to `dtype`, in the library's dY layout
 * ([NG][B][G], haste_dy_bytes(h,B) bytes, padding labels >= L written as zero; haste_dy_unpack converts it to
 * [B,L] fp32).  No targets, no loss, nothing else written.  tcgen05 kernel family only (HASTE_ERR_UNSUPPORTED
 * otherwise: use haste_forward_loss with logits_out there).  X, idx, W, Z 16-byte aligned. */
int haste_forward_logits(haste_layer_t* h, int B, const void* X, const int32_t* idx, const void* W,
                         const float* bias /* [L] fp32 or NULL */, void* Z, void* stream);

/* Fused top-k inference (Eq. 4: P@k needs only the k highest-scoring labels of a row): the forward
 * contraction with an epilogue that keeps, per batch row, the k largest logits z[i,l] = bias[l] + <w_l, x_I> and their
 * labels; the B x L logits are never written.  1 <= k <= 8.
 *   out_val [B,k] fp32: the logits (fp32 accumulation of the bf16 products, not rounded), descending;
 *   out_idx [B,k] int64: GLOBAL label ids (label_offset + l); ties go to the smaller label; -1 (value -inf) where the
 *                        layer has fewer than k labels.
 * tcgen05 kernel family only (HASTE_ERR_UNSUPPORTED otherwise).  The first call allocates a workspace of
 * num_SMs * 32 KiB in the handle. */
int haste_forward_topk(haste_layer_t* h, int B, const void* X, const int32_t* idx, const void* W,
                       const float* bias /* [L] fp32 or NULL */, int k, float* out_val, int64_t* out_idx, void* stream);

/* haste_forward_topk without any allocation in the call (for callers that cannot call cudaMalloc: code under CUDA graph
 * capture, tight serving loops, harnesses that forbid it).  Same arguments, same results.  The candidate lists of the
 * forward kernel live in a file-scope device array of the library image instead of a workspace the first call
 * allocates: 4.625 MiB (the lists of at most 148 CTAs x 4 epilogue sets x 128 rows x 8 candidates, logits + labels), held
 * by every GPU that loads the library until the process exits.  Its device address is looked up once per device inside
 * haste_create; this call does no cudaMalloc / cudaFree and calls no allocating library routine.
 *   - A device with more than 148 SMs needs longer lists than the array holds: HASTE_ERR_UNSUPPORTED, nothing launched
 *     (use haste_forward_topk there).
 *   - ONE array per device, shared by every handle and every call: two calls that overlap on the GPU (different streams,
 *     or different handles on one device) race on it.  Calls on one stream are ordered and safe.
 *   - The array keeps the last call's contents; nothing in it needs clearing between calls (the forward kernel writes
 *     every list the merge kernel of the same call reads). */
int haste_forward_topk_static(haste_layer_t* h, int B, const void* X, const int32_t* idx, const void* W,
                              const float* bias /* [L] fp32 or NULL */, int k, float* out_val, int64_t* out_idx, void* stream);

/* Backward from a dY in the library layout. */
int haste_backward(haste_layer_t* h, int B,
                   const void* X, const int32_t* idx, const void* W, const void* dY,
                   void* dW,          /* [L,K] row-major, dw_dtype; overwritten.  NULL -> skipped */
                   float* dbias,      /* [L] fp32, overwritten, or NULL                           */
                   float* dX,         /* [B,d] row-major fp32.  NULL -> skipped                   */
                   int accumulate_dX, /* 0: overwrite dX; 1: add to its contents                  */
                   void* stream);

/* Backward with the optimizer step of the output layer fused into the weight-gradient kernel: "SGD with
 * momentum for the final layer" (the heavy-ball form, optional L2 decay -- DESIGN.md reading R13):
 *     g = dW[l,j] (never written to memory)      v[l,j] <- mu v[l,j] + g + weight_decay W[l,j]
 *     W[l,j] <- W[l,j] - lr v[l,j]   (fp32 arithmetic, W rounded once to bf16)
 * and for the bias, if given: vb[l] <- mu vb[l] + db[l];  b[l] <- b[l] - lr vb[l]  (no decay).
 * dX, if wanted, is computed FIRST, from W as the forward used it.  W [L,K] bf16 and momentum [L,K] fp32 are read and
 * written in place (16-byte aligned); bias / bias_momentum [L] fp32 both given or both NULL.  A call with B = 0 is a
 * no-op.  tcgen05 kernel family without HASTE_DETERMINISTIC, (G, K) other than (32, 128): otherwise HASTE_ERR_UNSUPPORTED
 * and nothing is modified. */
int haste_backward_sgd(haste_layer_t* h, int B, const void* X, const int32_t* idx, void* W, const void* dY,
                       float* momentum, float* bias, float* bias_momentum, float lr, float mu, float weight_decay,
                       float* dX, int accumulate_dX, void* stream);

/* Group-shared rewiring, Algorithm 3 of the paper; readings in DESIGN.md R15.
 *   scores S[k,j] = mean over the labels l of group k of |W[l,j]|   (fp32, labels in ascending order)
 *   the m = floor(NG K rho) smallest entries of S are pruned        (ties: smaller k K + j first)
 *   pruned slot: idx[k,j] <- Unif{0..d-1}; W[l,j] <- 0 (init_random = 0) or Unif(-1/sqrt(K), 1/sqrt(K)) (init_random = 1)
 *   for every label l of group k; momentum[l,j] <- 0 if a momentum buffer is given.
 * Random numbers come from a counter-based generator keyed by `seed` (SplitMix64; the result does not depend on the launch).
 * resort != 0: every touched idx row is re-sorted ascending (stable) and the W (and momentum) columns of its labels are
 * permuted with it -- the layer's function does not change, and sorted rows keep the fast path of the dX kernel.
 * Regrowth may duplicate a feature inside a row (the paper does not de-duplicate either): every kernel here handles that.
 * idx [NG,K] int32, W [L,K] dtype, momentum [L,K] fp32 or NULL: device memory, updated in place.  *n_pruned (host, may be
 * NULL) receives m.  Any G, K <= 3000, both dtypes.  Asynchronous on `stream`. */
int haste_rewire(haste_layer_t* h, int32_t* idx, void* W, float* momentum, float rho, int init_random, uint64_t seed,
                 int resort, int64_t* n_pruned, void* stream);

/* dY layout helpers: library layout <-> plain [B,L] row-major fp32. */
int haste_dy_unpack(const haste_layer_t* h, int B, const void* dY, float* out_BL, void* stream);
int haste_dy_pack(const haste_layer_t* h, int B, const float* in_BL, void* dY, void* stream);

/* ---- dense head ---------------------------------------------------- */

int haste_head_create(haste_head_t** out, int32_t d, int64_t L_h, int32_t B_max, haste_dtype_t dtype,
                      int64_t label_offset, float loss_scale, uint32_t flags, int cuda_device);
int haste_head_destroy(haste_head_t* h);

int haste_head_forward_loss(haste_head_t* h, int B,
                            const void* X,    /* [B,d] row-major, dtype (the head's own input) */
                            const void* Wh,   /* [L_h,d] row-major, dtype                                     */
                            const float* bias,/* [L_h] fp32 or NULL                                           */
                            const int32_t* tgt_rowptr, const int32_t* tgt_col,
                            float* loss,      /* device scalar or NULL                                        */
                            void* dY,         /* [B,L_h] row-major, dtype; NULL -> inference only             */
                            float* logits_out,/* optional [B,L_h] fp32                                        */
                            void* stream);

int haste_head_backward(haste_head_t* h, int B, const void* X, const void* Wh, const void* dY,
                        void* dWh,    /* [L_h,d] row-major, dtype; NULL -> skipped */
                        float* dbias, /* [L_h] fp32 or NULL                        */
                        float* dX,    /* [B,d] fp32; NULL -> skipped               */
                        int accumulate_dX, void* stream);

/* ---- diagnostics ---------------------------------------------------------------------- */

const char* haste_status_string(int status);
const char* haste_last_error(void); /* thread-local detail of the last failure */

/* Which kernel family a handle runs: 0 = generic CUDA-core (SIMT), 1 = tcgen05/TMEM/TMA. */
int haste_kernel_family(const haste_layer_t* h);
int haste_head_kernel_family(const haste_head_t* h);

/* Kernels the last forward / backward call on this handle launched (for bench.py's gpu_launches). */
int haste_last_launch_count(const haste_layer_t* h);
int haste_head_last_launch_count(const haste_head_t* h);

/* Per-kernel device timing (measurement support).  haste_set_profiling(h, depth)
 * with depth > 0 makes every forward / backward call record CUDA events on the caller's stream
 * around its kernels and keeps the last `depth` calls (depth = 0 turns it off; the default).
 * haste_kernel_ms waits for the events of one recorded run of `kernel` -- age 0 is the most recent
 * run, age 1 the one before ... -- and returns its duration in milliseconds
 * (HASTE_ERR_INVALID_ARG if no such run is held). */
typedef enum {
  HASTE_KERNEL_FORWARD = 0, /* forward contraction + fused BCE epilogue */
  HASTE_KERNEL_DW = 1,      /* weight gradient                            */
  HASTE_KERNEL_DX = 2,      /* input gradient scatter-add                    */
  HASTE_KERNEL_PREP_FWD = 3,/* X -> X^T before the forward                                  */
  HASTE_KERNEL_PREP_BWD = 4,/* X -> X^T and dX^T clear before the backward                  */
  HASTE_KERNEL_POST_BWD = 5 /* dX^T -> dX                                                   */
} haste_kernel_t;
int haste_set_profiling(haste_layer_t* h, int depth);
int haste_kernel_ms(haste_layer_t* h, int kernel /* haste_kernel_t */, int age, float* ms);
int haste_head_set_profiling(haste_head_t* h, int depth);
/* head kernels: HASTE_KERNEL_FORWARD, and HASTE_KERNEL_DW = the whole backward (dW_h, db, dX_h) */
int haste_head_kernel_ms(haste_head_t* h, int kernel, int age, float* ms);

#ifdef __cplusplus
}
#endif
#endif /* HASTE_H_ */
