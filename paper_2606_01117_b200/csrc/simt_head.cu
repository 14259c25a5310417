// simt_head.cu -- dense head over the frequent labels, generic
// CUDA-core family: one strided 64x64x16 register-tiled GEMM with three epilogues
// (fused BCE loss, typed store, fp32 store/accumulate).  Used for fp32 handles and as
// the fallback of the tcgen05 head kernels.
#include "kernels.h"

namespace haste {

enum { EPI_LOSS = 0, EPI_STORE_T = 1, EPI_STORE_F32 = 2 };

struct GemmEpi {
  // EPI_LOSS
  const float* bias; const int32_t* rowptr; const int32_t* col; int64_t label_offset; float s;
  double* loss_acc; void* dY; float* logits;
  // EPI_STORE_*
  void* out; int accumulate;
};

__device__ __forceinline__ int lb_i32(const int32_t* __restrict__ col, int lo, int hi, int64_t key) {
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if ((int64_t)col[mid] < key) lo = mid + 1; else hi = mid;
  }
  return lo;
}

// C[m][n] = sum_k A(m,k) * B(n,k);  A(m,k) = A[m*sAm + k*sAk],  B(n,k) = Bm[n*sBn + k*sBk].
template <typename T, int EPI>
__global__ void __launch_bounds__(256)
simt_gemm_kernel(int M, int N, int Kd, const T* __restrict__ A, int64_t sAm, int64_t sAk, const T* __restrict__ Bm,
                 int64_t sBn, int64_t sBk, GemmEpi ep) {
  __shared__ __align__(16) float As[16][68];
  __shared__ __align__(16) float Bs[16][68];
  const int m0 = blockIdx.y * 64, n0 = blockIdx.x * 64;
  const int t = threadIdx.x, tx = t & 15, ty = t >> 4;
  float acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;

  for (int k0 = 0; k0 < Kd; k0 += 16) {
#pragma unroll
    for (int e = t; e < 1024; e += 256) {
      int mm, kk;
      if (sAk == 1) { mm = e >> 4; kk = e & 15; } else { kk = e >> 6; mm = e & 63; }
      const int m = m0 + mm, k = k0 + kk;
      As[kk][mm] = (m < M && k < Kd) ? to_f32(A[m * sAm + k * sAk]) : 0.f;
    }
#pragma unroll
    for (int e = t; e < 1024; e += 256) {
      int nn, kk;
      if (sBk == 1) { nn = e >> 4; kk = e & 15; } else { kk = e >> 6; nn = e & 63; }
      const int n = n0 + nn, k = k0 + kk;
      Bs[kk][nn] = (n < N && k < Kd) ? to_f32(Bm[n * sBn + k * sBk]) : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < 16; ++kk) {
      const float4 a = *reinterpret_cast<const float4*>(&As[kk][ty * 4]);
      const float4 b = *reinterpret_cast<const float4*>(&Bs[kk][tx * 4]);
      const float av[4] = {a.x, a.y, a.z, a.w}, bv[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(av[i], bv[j], acc[i][j]);
    }
    __syncthreads();
  }

  if (EPI == EPI_LOSS) {
    float loss_local = 0.f;
    T* dY = reinterpret_cast<T*>(ep.dY);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int b = m0 + ty * 4 + i;
      if (b >= M) continue;
      const int64_t glo = ep.label_offset + n0 + tx * 4;
      int p0 = 0, p1 = 0;
      if (ep.rowptr) {
        const int r0 = ep.rowptr[b], r1 = ep.rowptr[b + 1];
        p0 = lb_i32(ep.col, r0, r1, glo);
        p1 = lb_i32(ep.col, p0, r1, glo + 4);
      }
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int n = n0 + tx * 4 + j;
        if (n >= N) continue;
        const float z = acc[i][j] + (ep.bias ? ep.bias[n] : 0.f);
        float y = 0.f;
        for (int p = p0; p < p1; ++p) if ((int64_t)ep.col[p] == glo + j) y = 1.f;
        float sp, sg;
        bce_terms_precise(z, sp, sg);
        loss_local += sp - y * z;
        if (dY) dY[(int64_t)b * N + n] = from_f32<T>(ep.s * (sg - y));
        if (ep.logits) ep.logits[(int64_t)b * N + n] = z;
      }
    }
    if (ep.loss_acc) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) loss_local += __shfl_xor_sync(0xffffffffu, loss_local, o);
      if ((t & 31) == 0) atomicAdd(ep.loss_acc, (double)loss_local);
    }
  } else {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int m = m0 + ty * 4 + i;
      if (m >= M) continue;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int n = n0 + tx * 4 + j;
        if (n >= N) continue;
        if (EPI == EPI_STORE_T) {
          reinterpret_cast<T*>(ep.out)[(int64_t)m * N + n] = from_f32<T>(acc[i][j]);
        } else {
          float* p = reinterpret_cast<float*>(ep.out) + (int64_t)m * N + n;
          *p = ep.accumulate ? *p + acc[i][j] : acc[i][j];
        }
      }
    }
  }
}

// db[l] = sum_b dY[b][l]
template <typename T>
__global__ void head_dbias_kernel(const T* __restrict__ dY, float* __restrict__ db, int B, int64_t L) {
  const int64_t l = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (l >= L) return;
  float acc = 0.f;
  for (int b = 0; b < B; ++b) acc += to_f32(dY[(int64_t)b * L + l]);
  db[l] = acc;
}

template <typename T>
static int head_forward_T(const HeadShape& sh, const void* X, const void* Wh, const float* bias, const int32_t* rowptr,
                          const int32_t* col, double* loss_acc, void* dY, float* logits, cudaStream_t st) {
  GemmEpi ep{};
  ep.bias = bias; ep.rowptr = rowptr; ep.col = col; ep.label_offset = sh.label_offset; ep.s = sh.s;
  ep.loss_acc = loss_acc; ep.dY = dY; ep.logits = logits;
  dim3 grid(ceil_div(sh.L, 64), ceil_div(sh.B, 64));
  // z[b][l] = sum_f X[b][f] Wh[l][f]
  simt_gemm_kernel<T, EPI_LOSS><<<grid, 256, 0, st>>>(sh.B, (int)sh.L, sh.d, (const T*)X, (int64_t)sh.d, 1,
                                                      (const T*)Wh, (int64_t)sh.d, 1, ep);
  HASTE_LAUNCH_CHECK();
  return HASTE_OK;
}

int launch_simt_head_forward(haste_dtype_t dt, const HeadShape& sh, const void* X, const void* Wh, const float* bias,
                             const int32_t* rowptr, const int32_t* col, double* loss_acc, void* dY, float* logits_out,
                             cudaStream_t st) {
  if (sh.L == 0 || sh.B == 0) return HASTE_OK;
  return dt == HASTE_F32 ? head_forward_T<float>(sh, X, Wh, bias, rowptr, col, loss_acc, dY, logits_out, st)
                         : head_forward_T<bf16>(sh, X, Wh, bias, rowptr, col, loss_acc, dY, logits_out, st);
}

template <typename T>
static int head_backward_T(const HeadShape& sh, const void* X, const void* Wh, const void* dY, void* dWh, float* dbias,
                           float* dX, int accumulate_dX, cudaStream_t st) {
  const int L = (int)sh.L;
  if (dWh) {   // dWh[l][f] = sum_b dY[b][l] X[b][f]
    GemmEpi ep{}; ep.out = dWh;
    dim3 grid(ceil_div(sh.d, 64), ceil_div(L, 64));
    simt_gemm_kernel<T, EPI_STORE_T><<<grid, 256, 0, st>>>(L, sh.d, sh.B, (const T*)dY, 1, (int64_t)L, (const T*)X, 1,
                                                         (int64_t)sh.d, ep);
    HASTE_LAUNCH_CHECK();
  }
  if (dX) {    // dX[b][f] = sum_l dY[b][l] Wh[l][f]
    GemmEpi ep{}; ep.out = dX; ep.accumulate = accumulate_dX;
    dim3 grid(ceil_div(sh.d, 64), ceil_div(sh.B, 64));
    simt_gemm_kernel<T, EPI_STORE_F32><<<grid, 256, 0, st>>>(sh.B, sh.d, L, (const T*)dY, (int64_t)L, 1, (const T*)Wh, 1,
                                                           (int64_t)sh.d, ep);
    HASTE_LAUNCH_CHECK();
  }
  if (dbias) {
    head_dbias_kernel<T><<<ceil_div(L, 256), 256, 0, st>>>((const T*)dY, dbias, sh.B, sh.L);
    HASTE_LAUNCH_CHECK();
  }
  return HASTE_OK;
}

int launch_simt_head_backward(haste_dtype_t dt, const HeadShape& sh, const void* X, const void* Wh, const void* dY,
                              void* dWh, float* dbias, float* dX, int accumulate_dX, cudaStream_t st) {
  if (sh.L == 0 || sh.B == 0) return HASTE_OK;
  return dt == HASTE_F32 ? head_backward_T<float>(sh, X, Wh, dY, dWh, dbias, dX, accumulate_dX, st)
                         : head_backward_T<bf16>(sh, X, Wh, dY, dWh, dbias, dX, accumulate_dX, st);
}

}  // namespace haste
