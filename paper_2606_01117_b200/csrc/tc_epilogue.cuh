// tc_epilogue.cuh -- the fused BCE-with-logits epilogue shared by the sparse-tail forward (tc_tail.cu)
// and the dense-head forward (tc_head.cu): PAPER.md:111 (Eq. 3), with-logits form (reading R5).
#pragma once
#include "tc_common.cuh"

namespace haste {
namespace tc {

__device__ __forceinline__ float tanh_approx(float x) {
  float y;
  asm("tanh.approx.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&v);
}

// 32 logits of one batch row: z -> dY (bf16x2 packed) and the row's loss terms.
//   sigma(z) = 1/2 + 1/2 tanh(z/2)  (one MUFU op);  softplus(z) = max(z,0) - ln( sigma(|z|) ), and the
//   logs of a tile are taken once on the PRODUCT of the factors sigma(|z|) in [1/2,1)  (<= 16 per chain).
// SLOW: some label of this chunk is a positive of this row, or the chunk holds padding labels (>= L).
template <bool SLOW, bool BIAS>
__device__ __forceinline__ void epi32(const uint32_t (&v)[32], uint32_t sbias, uint32_t ymask, int nvalid, float s,
                                      float hs, float (&R)[4], float (&P)[4], uint32_t (&out)[16], float* zout) {
  float bv[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
  for (int j = 0; j < 32; j += 2) {
    float dy[2];
    if (BIAS && (j & 3) == 0) {
      const float4 t4 = lds128f(sbias + j * 4);
      bv[0] = t4.x; bv[1] = t4.y; bv[2] = t4.z; bv[3] = t4.w;
    }
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      const int jj = j + u;
      float z = __uint_as_float(v[jj]);
      if (BIAS) z += bv[jj & 3];
      const float t = tanh_approx(0.5f * z);
      float d = fmaf(t, hs, hs);
      float f = fmaf(fabsf(t), 0.5f, 0.5f);
      float r = fmaxf(z, 0.f);
      if (SLOW) {
        const bool valid = jj < nvalid;
        const bool y = (ymask >> jj) & 1u;
        if (y) { d -= s; r -= z; }
        if (!valid) { d = 0.f; f = 1.f; r = 0.f; }
        if (zout && valid) zout[jj] = z;
      }
      dy[u] = d;
      P[jj & 3] *= f;
      R[jj & 3] += r;
    }
    out[j >> 1] = pack_bf16x2(dy[0], dy[1]);
  }
}

}  // namespace tc
}  // namespace haste
