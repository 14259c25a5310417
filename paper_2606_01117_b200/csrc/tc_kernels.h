// tc_kernels.h -- interface of the tcgen05 / TMEM / TMA kernel family (sm_100a) to the
// C-ABI layer.  bf16 storage, fp32 accumulate.  See tc_tail.cu / tc_head.cu.
#pragma once
#include "common.cuh"
#include "kernels.h"

namespace haste {

struct TcTailState;
struct TcHeadState;

// Shapes the tcgen05 sparse-tail kernels cover (everything else runs the SIMT family).
bool tc_tail_supported(const haste_config_t& cfg, int device);
int tc_tail_create(TcTailState** out, const haste_config_t& cfg, int Bpad, int device);
void tc_tail_destroy(TcTailState* s);
int tc_tail_num_partials(const TcTailState* s);
// geometry of the forward launch, for the merge of the fused top-k candidates (launch_topk_merge)
struct TopkGeom { int k; int NP, S, NSET; };     // k: in (the caller's k, picks the list length); the rest: out
// loss_partials: workspace of 1024 floats (per-CTA unscaled partials + the arrival ticket, zeroed at create) or NULL;
// loss: device scalar that the last CTA of the forward kernel writes (s * sum of the partials; no second launch).
// z_mode = 1: logits-only forward, the dY buffer receives the logits (same layout and dtype); no targets, no loss.
int tc_tail_forward(TcTailState* s, const TailShape& sh, const void* Xt, const int32_t* idx, const void* W,
                    const float* bias, const int32_t* rowptr, const int32_t* col, float* loss_partials, float* loss, void* dY,
                    float* logits_out, int z_mode, float* topk_val, int* topk_idx, TopkGeom* geom, cudaStream_t st, int* n_launches);
// z_mode = 2: fused top-k; topk_val / topk_idx: [grid][sets][128][8] candidate workspace (grid <= num SMs, sets <= 4)
int tc_tail_dw(TcTailState* s, const TailShape& sh, const void* Xt, const int32_t* idx, const void* dY, void* dW,
               float* dbias, cudaStream_t st, int* n_launches);
// forward + loss + dY AND the weight gradient in one kernel (tc_fused.cu): G = 64, K in {64, 128}, B <= 512; otherwise
// HASTE_ERR_UNSUPPORTED with nothing launched
int tc_tail_forward_dw(TcTailState* s, const TailShape& sh, const void* Xt, const int32_t* idx, const void* W, const float* bias,
                       const int32_t* rowptr, const int32_t* col, float* loss_partials, float* loss, void* dY, void* dW,
                       float* dbias, cudaStream_t st, int* n_launches);
// dW with the SGD-momentum step of the output layer as its epilogue (tc_dw.cu): W, mom (and bias, bmom) updated in place
int tc_tail_dw_sgd(TcTailState* s, const TailShape& sh, const void* Xt, const int32_t* idx, const void* dY, void* W, float* mom,
                   float* bias, float* bmom, float lr, float mu, float wd, cudaStream_t st, int* n_launches);
// dx_part: null, or (HASTE_DETERMINISTIC) private partial tiles [tc_tail_dx_parts()][d][128] fp32, zeroed by the caller: the kernel
// then uses no float atomics and the caller sums the tiles of a batch tile in stripe order (launch_reduce_dx_parts)
int tc_tail_dx(TcTailState* s, const TailShape& sh, const int32_t* idx, const void* W, const void* dY, float* dXt,
               float* dx_part, cudaStream_t st, int* n_launches);
// grid of the dX kernel for this batch size: NT batch tiles x S stripes (CTA = stripe * NT + batch tile)
void tc_tail_dx_grid(const TcTailState* s, const TailShape& sh, int* NT, int* S);
int tc_tail_num_sms(const TcTailState* s);
// on-chip accumulating version (tc_dx_acc.cu)
int tc_tail_dx_acc(TcTailState* s, const TailShape& sh, const int32_t* idx, const void* W, const void* dY, float* dXt,
                   float* part, cudaStream_t st);

bool tc_head_supported(int d, int64_t L_h, int B_max, haste_dtype_t dtype, int device);
int tc_head_create(TcHeadState** out, int d, int64_t L_h, int B_max, int device);
void tc_head_destroy(TcHeadState* s);
int tc_head_num_partials(const TcHeadState* s);
int tc_head_forward(TcHeadState* s, const HeadShape& sh, const void* X, const void* Wh, const float* bias,
                    const int32_t* rowptr, const int32_t* col, float* loss_partials, float* loss, void* dY, float* logits_out,
                    cudaStream_t st, int* n_launches);
int tc_head_backward(TcHeadState* s, const HeadShape& sh, const void* X, const void* Wh, const void* dY, void* dWh,
                     float* dbias, float* dX, int accumulate_dX, int deterministic, cudaStream_t st, int* n_launches);

}  // namespace haste
