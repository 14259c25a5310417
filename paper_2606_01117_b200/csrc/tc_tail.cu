// tc_tail.cu -- tcgen05 sparse-tail kernels (placeholder while the family is brought up).
#include "tc_kernels.h"
namespace haste {
struct TcTailState { int dummy; };
bool tc_tail_supported(const haste_config_t&, int) { return false; }
int tc_tail_create(TcTailState**, const haste_config_t&, int, int) { return HASTE_ERR_UNSUPPORTED; }
void tc_tail_destroy(TcTailState*) {}
int tc_tail_num_partials(const TcTailState*) { return 0; }
int tc_tail_forward(TcTailState*, const TailShape&, const void*, const int32_t*, const void*, const float*, const int32_t*,
                    const int32_t*, float*, void*, float*, cudaStream_t, int*) { return HASTE_ERR_UNSUPPORTED; }
int tc_tail_dw(TcTailState*, const TailShape&, const void*, const int32_t*, const void*, void*, float*, cudaStream_t, int*) { return HASTE_ERR_UNSUPPORTED; }
int tc_tail_dx(TcTailState*, const TailShape&, const int32_t*, const void*, const void*, float*, cudaStream_t, int*) { return HASTE_ERR_UNSUPPORTED; }
}
