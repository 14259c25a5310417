// simt_kernels.cu -- generic CUDA-core kernel family of the HASTE sparse tail.
//
// Correct for ANY G, K, d, partial last group, unsorted / duplicated idx (reading R4),
// fp32 or bf16 storage, fp32 accumulate.  It is the path of the fp32 config, of the
// small-G points of the kernel sweep (G = 1 is the per-label fixed fan-in comparison
// kernel) and of any shape the tcgen05 family does not cover.
//
// Data layout: X^T [d][Bpad] (batch contiguous, so a gathered feature is one coalesced
// row), W [L][K], dY group-blocked [NG][B][G], dX^T [d][Bpad] fp32.
#include "kernels.h"

namespace haste {

// Position of the first entry >= key in the ascending array col[lo..hi).
__device__ __forceinline__ int lower_bound_i32(const int32_t* __restrict__ col, int lo, int hi, int64_t key) {
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if ((int64_t)col[mid] < key) lo = mid + 1; else hi = mid;
  }
  return lo;
}
__device__ __forceinline__ float csr_contains(const int32_t* __restrict__ col, int p0, int p1, int64_t gid) {
  float y = 0.f;
  for (int p = p0; p < p1; ++p) if ((int64_t)col[p] == gid) y = 1.f;
  return y;
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

template <typename T, int VEC> struct WVec;
template <> struct WVec<float, 4> {
  static __device__ __forceinline__ void load(const float* p, float (&w)[4]) {
    const float4 v = *reinterpret_cast<const float4*>(p); w[0] = v.x; w[1] = v.y; w[2] = v.z; w[3] = v.w;
  }
};
template <> struct WVec<bf16, 4> {
  static __device__ __forceinline__ void load(const bf16* p, float (&w)[4]) {
    const uint2 v = *reinterpret_cast<const uint2*>(p);
    w[0] = __uint_as_float(v.x << 16); w[1] = __uint_as_float(v.x & 0xffff0000u);
    w[2] = __uint_as_float(v.y << 16); w[3] = __uint_as_float(v.y & 0xffff0000u);
  }
};
template <typename T> struct WVec<T, 1> {
  static __device__ __forceinline__ void load(const T* p, float (&w)[1]) { w[0] = to_f32(p[0]); }
};

// ---------------------------------------------------------------------------------
// Forward + fused BCE.  Block = (group g, 32 batch rows); the K
// gathered rows of X^T are staged once in shared memory and reused by all labels of
// the group ("gather-once").  lane = batch row, warps stride over quads of labels.
// ---------------------------------------------------------------------------------
template <typename T, int VEC>
__global__ void __launch_bounds__(128)
simt_forward_kernel(TailShape sh, const T* __restrict__ Xt, const int32_t* __restrict__ idx, const T* __restrict__ W,
                    const float* __restrict__ bias, const int32_t* __restrict__ rowptr,
                    const int32_t* __restrict__ col, double* loss_acc, T* __restrict__ dY,
                    float* __restrict__ logits) {
  extern __shared__ float smem[];
  float* Hs = smem;                                // [K][32]
  int* sidx = reinterpret_cast<int*>(smem + (size_t)sh.K * 32);
  const int64_t g = blockIdx.x;
  const int b0 = blockIdx.y * 32;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const int K = sh.K, G = sh.G, B = sh.B;
  const int nl = (int)min((int64_t)G, sh.L - g * G);
  const int b = b0 + lane;
  const bool vb = b < B;

  for (int k = threadIdx.x; k < K; k += blockDim.x) sidx[k] = idx[g * K + k];
  __syncthreads();
  for (int k = warp; k < K; k += nw)
    Hs[k * 32 + lane] = vb ? to_f32(Xt[(int64_t)sidx[k] * sh.Bpad + b]) : 0.f;
  __syncthreads();

  const int64_t glo = sh.label_offset + g * G;
  int p0 = 0, p1 = 0;
  if (vb && rowptr) {
    const int r0 = rowptr[b], r1 = rowptr[b + 1];
    p0 = lower_bound_i32(col, r0, r1, glo);
    p1 = lower_bound_i32(col, p0, r1, glo + nl);
  }
  float loss_local = 0.f;
  for (int q = warp; 4 * q < G; q += nw) {
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    const int l0 = 4 * q;
    for (int k = 0; k < K; k += VEC) {
      float h[VEC];
#pragma unroll
      for (int v = 0; v < VEC; ++v) h[v] = Hs[(k + v) * 32 + lane];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        if (l0 + j < nl) {
          float w[VEC];
          WVec<T, VEC>::load(W + (g * G + l0 + j) * K + k, w);
#pragma unroll
          for (int v = 0; v < VEC; ++v) acc[j] = fmaf(w[v], h[v], acc[j]);
        }
      }
    }
    if (vb) {
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int lp = l0 + j;
        if (lp >= G) break;
        float dy = 0.f;
        if (lp < nl) {
          const int64_t l = g * G + lp;
          const float z = acc[j] + (bias ? bias[l] : 0.f);
          const float y = csr_contains(col, p0, p1, glo + lp);
          float sp, sg;
          bce_terms_precise(z, sp, sg);
          loss_local += sp - y * z;
          dy = sh.s * (sg - y);
          if (logits) logits[(int64_t)b * sh.L + l] = z;
        }
        if (dY) dY[(g * B + b) * G + lp] = from_f32<T>(dy);   // padding labels of the last group: 0
      }
    }
  }
  if (loss_acc) {
    loss_local = warp_sum(loss_local);
    if (lane == 0) atomicAdd(loss_acc, (double)loss_local);
  }
}

template <typename T>
static int forward_T(const TailShape& sh, const void* Xt, const int32_t* idx, const void* W, const float* bias,
                     const int32_t* rowptr, const int32_t* col, double* loss_acc, void* dY, float* logits,
                     cudaStream_t st) {
  const int nw = sh.G >= 16 ? 4 : (sh.G >= 8 ? 2 : 1);
  dim3 grid((unsigned)sh.NG, ceil_div(sh.B, 32));
  const size_t smem = (size_t)sh.K * 32 * 4 + (size_t)sh.K * 4;
  if (grid.y > 65535) { set_error("B too large for the SIMT forward grid"); return HASTE_ERR_UNSUPPORTED; }
  if (sh.K % 4 == 0) {
    if (smem > 48 * 1024)
      HASTE_CUDA_TRY(cudaFuncSetAttribute(simt_forward_kernel<T, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    simt_forward_kernel<T, 4><<<grid, 32 * nw, smem, st>>>(sh, (const T*)Xt, idx, (const T*)W, bias, rowptr, col,
                                                         loss_acc, (T*)dY, logits);
  } else {
    if (smem > 48 * 1024)
      HASTE_CUDA_TRY(cudaFuncSetAttribute(simt_forward_kernel<T, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    simt_forward_kernel<T, 1><<<grid, 32 * nw, smem, st>>>(sh, (const T*)Xt, idx, (const T*)W, bias, rowptr, col,
                                                         loss_acc, (T*)dY, logits);
  }
  HASTE_LAUNCH_CHECK();
  return HASTE_OK;
}

int launch_simt_forward(haste_dtype_t dt, const TailShape& sh, const void* Xt, const int32_t* idx, const void* W,
                        const float* bias, const int32_t* rowptr, const int32_t* col, double* loss_acc, void* dY,
                        float* logits_out, cudaStream_t st) {
  if (sh.NG == 0 || sh.B == 0) return HASTE_OK;
  return dt == HASTE_F32 ? forward_T<float>(sh, Xt, idx, W, bias, rowptr, col, loss_acc, dY, logits_out, st)
                         : forward_T<bf16>(sh, Xt, idx, W, bias, rowptr, col, loss_acc, dY, logits_out, st);
}

// ---------------------------------------------------------------------------------
// Weight gradient dW_g = dY_g^T H_g.  Block = (group, 16 labels,
// 128 fan-in slots); thread = one slot k, 16 accumulators (one per label); the batch
// is streamed through shared memory 32 rows at a time.
// ---------------------------------------------------------------------------------
template <typename T, typename TW>
__global__ void __launch_bounds__(128)
simt_dw_kernel(TailShape sh, const T* __restrict__ Xt, const int32_t* __restrict__ idx, const T* __restrict__ dY,
               TW* __restrict__ dW, float* __restrict__ dbias) {
  __shared__ float Hs[128][33];
  __shared__ __align__(16) float Ds[32][16];
  __shared__ int sidx[128];
  const int64_t g = blockIdx.x;
  const int lb = blockIdx.y * 16, kbase = blockIdx.z * 128;
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
  const int K = sh.K, G = sh.G, B = sh.B;
  const int nl = (int)min((int64_t)G, sh.L - g * G);
  if (lb >= nl) return;
  sidx[t] = (kbase + t < K) ? idx[g * K + kbase + t] : -1;
  float acc[16];
#pragma unroll
  for (int r = 0; r < 16; ++r) acc[r] = 0.f;
  float dbsum = 0.f;
  for (int b0 = 0; b0 < B; b0 += 32) {
    __syncthreads();
    for (int r = warp; r < 128; r += 4) {
      const int f = sidx[r];
      Hs[r][lane] = (f >= 0 && b0 + lane < B) ? to_f32(Xt[(int64_t)f * sh.Bpad + b0 + lane]) : 0.f;
    }
#pragma unroll
    for (int e = t; e < 512; e += 128) {
      const int bb = e >> 4, ll = e & 15;
      Ds[bb][ll] = (b0 + bb < B && lb + ll < nl) ? to_f32(dY[(g * B + b0 + bb) * G + lb + ll]) : 0.f;
    }
    __syncthreads();
#pragma unroll 4
    for (int bb = 0; bb < 32; ++bb) {
      const float h = Hs[t][bb];
      const float4* dr = reinterpret_cast<const float4*>(&Ds[bb][0]);
#pragma unroll
      for (int v = 0; v < 4; ++v) {
        const float4 dv = dr[v];
        acc[4 * v + 0] = fmaf(dv.x, h, acc[4 * v + 0]);
        acc[4 * v + 1] = fmaf(dv.y, h, acc[4 * v + 1]);
        acc[4 * v + 2] = fmaf(dv.z, h, acc[4 * v + 2]);
        acc[4 * v + 3] = fmaf(dv.w, h, acc[4 * v + 3]);
      }
    }
    if (dbias && blockIdx.z == 0 && t < 16)
      for (int bb = 0; bb < 32; ++bb) dbsum += Ds[bb][t];
  }
  if (dW && kbase + t < K) {
#pragma unroll
    for (int r = 0; r < 16; ++r)
      if (lb + r < nl) dW[(g * G + lb + r) * K + kbase + t] = from_f32<TW>(acc[r]);
  }
  if (dbias && blockIdx.z == 0 && t < 16 && lb + t < nl) dbias[g * G + lb + t] = dbsum;
}

int launch_simt_dw(haste_dtype_t dt, haste_dtype_t dw_dt, const TailShape& sh, const void* Xt, const int32_t* idx,
                   const void* dY, void* dW, float* dbias, cudaStream_t st) {
  if (sh.NG == 0) return HASTE_OK;
  dim3 grid((unsigned)sh.NG, ceil_div(sh.G, 16), ceil_div(sh.K, 128));
#define HASTE_DW(T, TW) simt_dw_kernel<T, TW><<<grid, 128, 0, st>>>(sh, (const T*)Xt, idx, (const T*)dY, (TW*)dW, dbias)
  if (dt == HASTE_F32 && dw_dt == HASTE_F32) HASTE_DW(float, float);
  else if (dt == HASTE_F32) HASTE_DW(float, bf16);
  else if (dw_dt == HASTE_F32) HASTE_DW(bf16, float);
  else HASTE_DW(bf16, bf16);
#undef HASTE_DW
  HASTE_LAUNCH_CHECK();
  return HASTE_OK;
}

// ---------------------------------------------------------------------------------
// Input gradient dX[:, I_g] += dY_g W_g as a scatter-add into dX^T.
// Block = (group, 32 batch rows); lane = batch row, warps stride over quads of slots;
// the reduction over groups is a coalesced fp32 red.global.add (atomics also make
// duplicated indices inside a group additive, reading R4).
// ---------------------------------------------------------------------------------
template <typename T, int VEC>
__global__ void __launch_bounds__(128)
simt_dx_kernel(TailShape sh, const int32_t* __restrict__ idx, const T* __restrict__ W, const T* __restrict__ dY,
               float* __restrict__ dXt) {
  extern __shared__ float Ds[];   // [32][G+1]
  const int64_t g = blockIdx.x;
  const int b0 = blockIdx.y * 32;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const int K = sh.K, G = sh.G, B = sh.B, GP = G + 1;
  const int nl = (int)min((int64_t)G, sh.L - g * G);
  const int nb = min(32, B - b0);
  for (int e = threadIdx.x; e < 32 * G; e += blockDim.x) {
    const int bb = e / G, ll = e % G;
    Ds[bb * GP + ll] = (bb < nb && ll < nl) ? to_f32(dY[(g * B + b0 + bb) * G + ll]) : 0.f;
  }
  __syncthreads();
  const int b = b0 + lane;
  for (int q = warp; VEC * q < K; q += nw) {
    float acc[VEC];
#pragma unroll
    for (int v = 0; v < VEC; ++v) acc[v] = 0.f;
    for (int lp = 0; lp < nl; ++lp) {
      const float dy = Ds[lane * GP + lp];
      float w[VEC];
      WVec<T, VEC>::load(W + (g * G + lp) * K + VEC * q, w);
#pragma unroll
      for (int v = 0; v < VEC; ++v) acc[v] = fmaf(dy, w[v], acc[v]);
    }
    if (b < B) {
#pragma unroll
      for (int v = 0; v < VEC; ++v) {
        const int f = idx[g * K + VEC * q + v];
        atomicAdd(dXt + (int64_t)f * sh.Bpad + b, acc[v]);
      }
    }
  }
}

template <typename T>
static int dx_T(const TailShape& sh, const int32_t* idx, const void* W, const void* dY, float* dXt, cudaStream_t st) {
  dim3 grid((unsigned)sh.NG, ceil_div(sh.B, 32));
  const size_t smem = (size_t)32 * (sh.G + 1) * 4;
  if (sh.K % 4 == 0) {
    if (smem > 48 * 1024)
      HASTE_CUDA_TRY(cudaFuncSetAttribute(simt_dx_kernel<T, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    simt_dx_kernel<T, 4><<<grid, 128, smem, st>>>(sh, idx, (const T*)W, (const T*)dY, dXt);
  } else {
    if (smem > 48 * 1024)
      HASTE_CUDA_TRY(cudaFuncSetAttribute(simt_dx_kernel<T, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    simt_dx_kernel<T, 1><<<grid, 128, smem, st>>>(sh, idx, (const T*)W, (const T*)dY, dXt);
  }
  HASTE_LAUNCH_CHECK();
  return HASTE_OK;
}

int launch_simt_dx(haste_dtype_t dt, const TailShape& sh, const int32_t* idx, const void* W, const void* dY,
                   float* dXt, cudaStream_t st) {
  if (sh.NG == 0 || sh.B == 0) return HASTE_OK;
  return dt == HASTE_F32 ? dx_T<float>(sh, idx, W, dY, dXt, st) : dx_T<bf16>(sh, idx, W, dY, dXt, st);
}

}  // namespace haste
