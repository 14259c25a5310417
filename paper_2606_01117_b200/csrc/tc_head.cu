// tc_head.cu -- tcgen05 dense-head kernels (placeholder while the family is brought up).
#include "tc_kernels.h"
namespace haste {
struct TcHeadState { int dummy; };
bool tc_head_supported(int, int64_t, int, haste_dtype_t, int) { return false; }
int tc_head_create(TcHeadState**, int, int64_t, int, int) { return HASTE_ERR_UNSUPPORTED; }
void tc_head_destroy(TcHeadState*) {}
int tc_head_num_partials(const TcHeadState*) { return 0; }
int tc_head_forward(TcHeadState*, const HeadShape&, const void*, const void*, const float*, const int32_t*, const int32_t*,
                    float*, void*, float*, cudaStream_t, int*) { return HASTE_ERR_UNSUPPORTED; }
int tc_head_backward(TcHeadState*, const HeadShape&, const void*, const void*, const void*, void*, float*, float*, int,
                     cudaStream_t, int*) { return HASTE_ERR_UNSUPPORTED; }
}
