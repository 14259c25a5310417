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

// Packed fp32 pairs (sm_100: one instruction, two lanes of fp32 math).  The epilogue is issue-bound, so the ops that
// exist in packed form (mul, fma, add) are done two logits at a time; tanh, |.| and max stay scalar.
__device__ __forceinline__ uint64_t pk2(float lo, float hi) {
  uint64_t r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void upk2(uint64_t v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ uint64_t mul2(uint64_t a, uint64_t b) {
  uint64_t r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ uint64_t add2(uint64_t a, uint64_t b) {
  uint64_t r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t c) {
  uint64_t r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}

__device__ __forceinline__ float max3(float a, float b, float c) {
  float r;
  asm("max.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
  return r;
}
__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float rcp_approx(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// 8 logits (J0 .. J0+7) of one batch row.  SL: one of them may be a positive of the row or a padding label (>= L).
// The fast evaluation (the caller has checked |z| <= 2.5, see epi32): t = tanh.approx(z/2), ONE MUFU op per logit, and then
//   dY = s sigma(z) = s/2 + (s/2) t                                   (minus s at a positive)
//   loss term of a negative: softplus(z)  = -ln sigma(-z) = -ln(1/2 - t/2)
//   loss term of a positive: softplus(-z) = -ln sigma(z)  = -ln(1/2 + t/2)
// so the term is the log of ONE factor per logit, multiplied into the running product P (no max(z,0), no |t|, no sum): 3.5
// instructions per logit in packed f32x2 form.  With |z| <= 2.5 a factor is >= 0.076: 16 of them cannot underflow, and the
// 2.4e-4 absolute error of tanh.approx is at most 0.3 % of it.
template <bool SL, bool BIAS, int J0>
__device__ __forceinline__ void epi8(const uint32_t (&v)[32], uint32_t sbias, uint32_t ymask, int nvalid, float s, uint64_t half2,
                                     uint64_t hs2, uint64_t (&P2)[2], uint32_t (&out)[16], float* zout) {
  uint64_t bv2[2] = {0ull, 0ull};
  const uint64_t nhalf2 = pk2(-0.5f, -0.5f);
#pragma unroll
  for (int j = J0; j < J0 + 8; j += 2) {
    if (BIAS && (j & 3) == 0) {
      const float4 t4 = lds128f(sbias + j * 4);
      bv2[0] = pk2(t4.x, t4.y); bv2[1] = pk2(t4.z, t4.w);
    }
    uint64_t z2 = pk2(__uint_as_float(v[j]), __uint_as_float(v[j + 1]));
    if (BIAS) z2 = add2(z2, bv2[(j >> 1) & 1]);
    float zh0, zh1;
    upk2(mul2(z2, half2), zh0, zh1);
    const uint64_t t2 = pk2(tanh_approx(zh0), tanh_approx(zh1));
    uint64_t d2 = fma2(t2, hs2, hs2);              // s sigma(z)
    uint64_t f2 = fma2(t2, nhalf2, half2);         // sigma(-z)
    if (SL) {
      float d0, d1, f0, f1;
      upk2(d2, d0, d1);
      upk2(f2, f0, f1);
      const bool valid0 = j < nvalid, valid1 = j + 1 < nvalid;
      if ((ymask >> j) & 1u) { d0 -= s; f0 = 1.f - f0; }
      if ((ymask >> (j + 1)) & 1u) { d1 -= s; f1 = 1.f - f1; }
      if (!valid0) { d0 = 0.f; f0 = 1.f; }
      if (!valid1) { d1 = 0.f; f1 = 1.f; }
      if (zout) {
        float z0, z1;
        upk2(z2, z0, z1);
        if (valid0) zout[j] = z0;
        if (valid1) zout[j + 1] = z1;
      }
      d2 = pk2(d0, d1);
      f2 = pk2(f0, f1);
    }
    P2[(j >> 1) & 1] = mul2(P2[(j >> 1) & 1], f2);
    float d0, d1;
    upk2(d2, d0, d1);
    out[j >> 1] = pack_bf16x2(d0, d1);
  }
}

// The exact-enough evaluation of 32 logits (see epi32), ONE copy of the code for every caller: it is rare on a freshly
// initialised layer, and four inlined copies per call site pushed the forward kernels out of the instruction cache
// (0.184 -> 0.262 ms).  io: v[32] accumulators in, then R[4], P[4] in/out at 32..39 and out[16] at 40..55 (a call through
// memory; only this path pays for it).  nj: how many of the 32 are there (narrow groups: 8 or 16).
static __device__ __noinline__ void epi32_wide(uint32_t* io, uint32_t sbias, int has_bias, uint32_t ymask, int nvalid, float s, float* zout, int nj) {
  float R[4], P[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) { R[k] = __uint_as_float(io[32 + k]); P[k] = __uint_as_float(io[36 + k]); }
#pragma unroll 4
  for (int j = 0; j < nj; j += 2) {
    float z0 = __uint_as_float(io[j]), z1 = __uint_as_float(io[j + 1]);
    if (has_bias) {
      float b0, b1;
      asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(b0), "=f"(b1) : "r"(sbias + j * 4));
      z0 += b0; z1 += b1;
    }
    const float e0 = ex2_approx(fabsf(z0) * -1.4426950408889634f), e1 = ex2_approx(fabsf(z1) * -1.4426950408889634f);
    float f0 = rcp_approx(1.f + e0), f1 = rcp_approx(1.f + e1);            // sigma(|z|)
    float d0 = s * (z0 >= 0.f ? f0 : e0 * f0), d1 = s * (z1 >= 0.f ? f1 : e1 * f1);
    float r0 = fmaxf(z0, 0.f), r1 = fmaxf(z1, 0.f);
    if ((ymask >> j) & 1u) { d0 -= s; r0 -= z0; }
    if ((ymask >> (j + 1)) & 1u) { d1 -= s; r1 -= z1; }
    if (j >= nvalid) { d0 = 0.f; f0 = 1.f; r0 = 0.f; }
    if (j + 1 >= nvalid) { d1 = 0.f; f1 = 1.f; r1 = 0.f; }
    if (zout && j < nvalid) zout[j] = z0;
    if (zout && j + 1 < nvalid) zout[j + 1] = z1;
    // same chains as the packed code: logit jj feeds R[jj & 3] and P[jj & 3]
    P[j & 3] *= f0; P[(j + 1) & 3] *= f1;
    R[j & 3] += r0; R[(j + 1) & 3] += r1;
    io[40 + (j >> 1)] = pack_bf16x2(d0, d1);
  }
#pragma unroll
  for (int k = 0; k < 4; ++k) { io[32 + k] = __float_as_uint(R[k]); io[36 + k] = __float_as_uint(P[k]); }
}

// 32 logits of one batch row: z -> dY (bf16x2 packed) and the row's loss terms.
//   Every loss term is minus the log of a factor in (0, 1], and the logs of a tile are taken once on the PRODUCT of the
//   factors (<= 16 per chain P[k]); the wide evaluation also adds max(z,0) - y z into the sums R[k]:
//   loss += (R[0]+R[1]+R[2]+R[3]) - ln 2 * log2(P[0] P[1] P[2] P[3]) at the caller.
// sigma has two evaluations:
//   fast: sigma(z) = 1/2 + 1/2 tanh.approx(z/2), ONE MUFU op per logit.  tanh.approx is good to 2^-11 RELATIVE to tanh,
//         i.e. up to 2.4e-4 absolute on sigma: 0.3 % of sigma(-2.5) = 0.076, the size of the bf16 rounding of dY, and
//         worse below.  So it is accepted only if every |z| of the warp's 32 x 32 logits is <= 2.5 (bounded by
//         max |accumulator| + max |bias|; true of a freshly initialised layer: |z| has std 0.23 in config 3's tail and
//         0.55 in its dense head);
//   wide: otherwise (the trained regime: confident negatives, sigma ~ 1e-4) the 32 logits are evaluated with
//         e = 2^(-|z| log2 e), sigma(|z|) = 1/(1+e), sigma(-|z|) = e/(1+e): two MUFU ops, relative error ~1e-6 for any z.
// SLOW: some label of this chunk may be a positive of some row of the warp, or the chunk holds padding labels (>= L), or
// logits are wanted; the decision is then refined per 8 logits (warp-uniform), because the special-case code costs more
// than the math itself and positives are rare (in the dense head ~70 % of the (warp, 128-label tile) pairs hold one).
// Chains: logit jj feeds P[jj & 3] (and, wide evaluation, R[jj & 3]); pair (j, j+1) = the two lanes of packed chain (j >> 1) & 1.
// NV: the chunk holds NV = 8, 16 or 32 logits (v[0 .. NV), out[0 .. NV/2)); groups of fewer than 32 labels have NV = G.
template <bool SLOW, bool BIAS, int NV = 32>
__device__ __forceinline__ void epi32(const uint32_t (&v)[32], uint32_t sbias, uint32_t ymask, int nvalid, float s,
                                      float hs, float (&R)[4], float (&P)[4], uint32_t (&out)[16], float* zout) {
  // which evaluation: max |accumulator| over the warp's 32 x 32 logits (+ max |bias| of the 32 labels) against 2.5
  float a4[4] = {0.f, 0.f, 0.f, 0.f};          // four independent chains: one chain of 16 would be ~70 cycles of latency per chunk
#pragma unroll
  for (int j = 0; j < NV; j += 2) a4[(j >> 1) & 3] = max3(a4[(j >> 1) & 3], fabsf(__uint_as_float(v[j])), fabsf(__uint_as_float(v[j + 1])));
  float am = max3(fmaxf(a4[0], a4[1]), a4[2], a4[3]);
  if (BIAS) {
    float b = 0.f;
    if (NV == 32 || (threadIdx.x & 31) < NV) asm volatile("ld.shared.f32 %0, [%1];" : "=f"(b) : "r"(sbias + (threadIdx.x & 31) * 4));
    am += __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(fabsf(b))));
  }
  if (__any_sync(0xffffffffu, am > 2.5f)) {
    uint32_t io[56];
#pragma unroll
    for (int j = 0; j < 32; ++j) io[j] = j < NV ? v[j] : 0u;
#pragma unroll
    for (int k = 0; k < 4; ++k) { io[32 + k] = __float_as_uint(R[k]); io[36 + k] = __float_as_uint(P[k]); }
    epi32_wide(io, sbias, BIAS ? 1 : 0, SLOW ? ymask : 0u, SLOW ? nvalid : NV, s, SLOW ? zout : nullptr, NV);
#pragma unroll
    for (int k = 0; k < 4; ++k) { R[k] = __uint_as_float(io[32 + k]); P[k] = __uint_as_float(io[36 + k]); }
#pragma unroll
    for (int k = 0; k < NV / 2; ++k) out[k] = io[40 + k];
    return;
  }
  uint64_t P2[2] = {pk2(P[0], P[1]), pk2(P[2], P[3])};      // (the fast path adds nothing to R: its loss terms are all in P)
  const uint64_t half2 = pk2(0.5f, 0.5f), hs2 = pk2(hs, hs);
#define HASTE_EPI8(J0_)                                                                                             \
  if (SLOW) {                                                                                                        \
    const bool sl = __any_sync(0xffffffffu, ((ymask >> J0_) & 0xffu) != 0u) || nvalid < J0_ + 8 || zout != nullptr; \
    if (sl) epi8<true, BIAS, J0_>(v, sbias, ymask, nvalid, s, half2, hs2, P2, out, zout);                  \
    else epi8<false, BIAS, J0_>(v, sbias, 0u, 32, s, half2, hs2, P2, out, nullptr);                        \
  } else {                                                                                                           \
    epi8<false, BIAS, J0_>(v, sbias, 0u, 32, s, half2, hs2, P2, out, nullptr);                             \
  }
  HASTE_EPI8(0)
  if constexpr (NV > 8) { HASTE_EPI8(8) }
  if constexpr (NV > 16) { HASTE_EPI8(16) HASTE_EPI8(24) }
#undef HASTE_EPI8
  upk2(P2[0], P[0], P[1]); upk2(P2[1], P[2], P[3]);
}

}  // namespace tc
}  // namespace haste
