// tc_dx.cu -- dispatch of the input-gradient step of the HASTE sparse tail (sm_100a; bf16 in, fp32 accumulate).
//
//   dX[:, idx_g] += dY_g [B x G] * W_g [G x K]   over all groups g
//
// One kernel implements it (tc_dx_acc.cu: one CTA per (128-row batch tile, stripe of groups), the reduction over the
// CTA's groups kept on chip; also the HASTE_DETERMINISTIC variant).  The choice depends on the shape only, never on
// the environment.  DESIGN.md section 5 records the round-2 two-CTA-cluster kernel that was built, measured and dropped.
#include <algorithm>

#include "tc_common.cuh"
#include "tc_kernels.h"

namespace haste {

void tc_tail_dx_grid(const TcTailState* s, const TailShape& sh, int* NT, int* S) {
  *NT = ceil_div(sh.B, 128);
  *S = (int)std::min<int64_t>(sh.NG, std::max(1, s->num_sms / *NT));
}
int tc_tail_num_sms(const TcTailState* s) { return s->num_sms; }

int tc_tail_dx(TcTailState* s, const TailShape& sh, const int32_t* idx, const void* W, const void* dY, float* dXt,
               float* dx_part, cudaStream_t st, int* n_launches) {
  *n_launches = 1;
  if (!((sh.G == 8 || sh.G == 16 || sh.G == 32 || sh.G == 64 || sh.G == 128) && (sh.K == 64 || sh.K == 128))) return HASTE_ERR_UNSUPPORTED;
  return tc_tail_dx_acc(s, sh, idx, W, dY, dXt, dx_part, st);
}

}  // namespace haste
