// common.cuh -- shared device/host helpers of the HASTE CUDA path (product code; the
// fp64 oracle under oracle/ shares nothing with this directory).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/haste.h"

namespace haste {

typedef __nv_bfloat16 bf16;

// ---- error plumbing (thread-local detail string, no exceptions across the ABI) ----
void set_error(const char* fmt, ...);
#define HASTE_CUDA_TRY(expr)                                                                  \
  do {                                                                                        \
    cudaError_t _e = (expr);                                                                  \
    if (_e != cudaSuccess) {                                                                  \
      haste::set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e), __FILE__, __LINE__); \
      return HASTE_ERR_CUDA;                                                                  \
    }                                                                                         \
  } while (0)
#define HASTE_LAUNCH_CHECK()                                                                  \
  do {                                                                                        \
    cudaError_t _e = cudaGetLastError();                                                      \
    if (_e != cudaSuccess) {                                                                  \
      haste::set_error("kernel launch failed: %s (%s:%d)", cudaGetErrorString(_e), __FILE__, __LINE__); \
      return HASTE_ERR_CUDA;                                                                  \
    }                                                                                         \
  } while (0)

// ---- programmatic dependent launch (PDL) ----
// Every kernel of a training step is launched with the programmatic-stream-serialization attribute and runs
//     <prologue that touches no global memory>;  pdl_wait();  pdl_trigger();  <the kernel>
// pdl_wait returns once the preceding kernel of the stream has completed and its writes are visible; pdl_trigger then lets
// the NEXT kernel's CTAs be placed on SMs as this kernel's CTAs leave them, where they run their own prologue (barrier
// init, TMEM allocation, descriptor prefetch) and block in their pdl_wait.  Launch latency and prologue thus overlap the
// tail of the kernel before; the data dependence is unchanged (nothing is read or written before pdl_wait, and every kernel
// launched this way waits, so completion is transitive along the stream).  After anything that is not a kernel launched
// this way (a memset, an event) the attribute has no effect.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
template <typename... KArgs, typename... Args>
static inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

static inline int ceil_div(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }
static inline int round_up(int a, int b) { return (a + b - 1) / b * b; }

// ---- dtype helpers ----
__device__ __forceinline__ float to_f32(float v) { return v; }
__device__ __forceinline__ float to_f32(bf16 v) { return __bfloat162float(v); }
template <typename T> __device__ __forceinline__ T from_f32(float v);
template <> __device__ __forceinline__ float from_f32<float>(float v) { return v; }
template <> __device__ __forceinline__ bf16 from_f32<bf16>(float v) { return __float2bfloat16_rn(v); }

// ---- BCE-with-logits pieces in fp32 (reading R5: with-logits form) ----
// softplus(z) = max(z,0) + log1p(exp(-|z|)); sigmoid(z) evaluated without overflow.
// Precise variant (fp32 configs): libm-grade expf/log1pf.
__device__ __forceinline__ void bce_terms_precise(float z, float& softplus, float& sigma) {
  const float e = expf(-fabsf(z));
  softplus = fmaxf(z, 0.f) + log1pf(e);
  const float r = 1.f / (1.f + e);
  sigma = z >= 0.f ? r : e * r;
}

// ---- workspace shared by all kernel families of one sparse-tail handle ----
struct TailShape {
  int d, G, K, B, Bpad;   // Bpad: row pitch (elements) of the X^T / dX^T workspaces
  int64_t L, NG;
  int64_t label_offset;
  float s;                // loss scale of this call
};

}  // namespace haste
