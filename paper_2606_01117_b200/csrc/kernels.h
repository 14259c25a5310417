// kernels.h -- launcher declarations shared by the C-ABI layer (haste_api.cu) and the
// kernel translation units.  Every launcher enqueues on `st` and returns a haste_status_t.
#pragma once
#include "common.cuh"

namespace haste {

// ---- prep / utility kernels (util_kernels.cu) ----
// Xt[f][b] = X[b][f] for b < B, 0 for B <= b < Bzero (Bzero <= Bpad, the row pitch).
int launch_transpose_pad(haste_dtype_t dt, const void* X, void* Xt, int B, int d, int Bpad, int Bzero, cudaStream_t st);
// dX[b][f] (=|+=) dXt[f][b]
int launch_untranspose_f32(float* dXt, float* dX, int B, int d, int Bpad, int accumulate, cudaStream_t st);
// fused top-k: merge the forward kernel's per-thread candidates into the k best (value, global label id) per batch row
int launch_topk_merge(const float* cand_val, const int* cand_idx, int NP, int S, int NSET, int NT, int B, int k,
                      int64_t label_offset, float* out_val, int64_t* out_idx, cudaStream_t st);
int launch_reduce_dx_parts(const float* part, float* dXt, int d, int Bpad, int NT, int S, cudaStream_t st);
int launch_finalize_loss(const double* acc, const float* partials, int n_partials, float scale, float* loss, cudaStream_t st);
int launch_dy_unpack(haste_dtype_t dt, const void* dY, float* out_BL, int B, int64_t L, int G, cudaStream_t st);
int launch_dy_pack(haste_dtype_t dt, const float* in_BL, void* dY, int B, int64_t L, int G, cudaStream_t st);
int launch_validate_index(const int32_t* idx, int64_t NG, int K, int d, int check_sorted, int* flag, cudaStream_t st);

// ---- Algorithm 3, group-shared rewiring (rewire.cu): any G, K, dtype; ws = rewire_workspace_bytes(NG, K) bytes of device memory
size_t rewire_workspace_bytes(int64_t NG, int K);
int launch_rewire(haste_dtype_t dt, int32_t* idx, void* W, float* mom, int64_t L, int G, int K, int d, int64_t m, int init_random,
                  uint64_t seed, int resort, void* ws, cudaStream_t st);

// ---- generic CUDA-core family (simt_kernels.cu): any G, K, d; fp32 or bf16 storage ----
int launch_simt_forward(haste_dtype_t dt, const TailShape& sh, const void* Xt, const int32_t* idx, const void* W,
                        const float* bias, const int32_t* rowptr, const int32_t* col, double* loss_acc, void* dY,
                        float* logits_out, cudaStream_t st);
int launch_simt_dw(haste_dtype_t dt, haste_dtype_t dw_dt, const TailShape& sh, const void* Xt, const int32_t* idx,
                   const void* dY, void* dW, float* dbias, cudaStream_t st);
int launch_simt_dx(haste_dtype_t dt, const TailShape& sh, const int32_t* idx, const void* W, const void* dY,
                   float* dXt, cudaStream_t st);

// Dense head, CUDA-core family.
struct HeadShape {
  int d, B;
  int64_t L;
  int64_t label_offset;
  float s;
};
int launch_simt_head_forward(haste_dtype_t dt, const HeadShape& sh, const void* X, const void* Wh, const float* bias,
                             const int32_t* rowptr, const int32_t* col, double* loss_acc, void* dY, float* logits_out,
                             cudaStream_t st);
int launch_simt_head_backward(haste_dtype_t dt, const HeadShape& sh, const void* X, const void* Wh, const void* dY,
                              void* dWh, float* dbias, float* dX, int accumulate_dX, cudaStream_t st);

}  // namespace haste
