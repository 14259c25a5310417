// util_kernels.cu -- prep and utility kernels of the HASTE path:
//   X -> X^T (zero-padded batch columns) so that "gather K features" is a gather of K
//   contiguous rows (gather-once); dX^T -> dX; loss finalisation; dY
//   layout pack/unpack; index validation.
#include "kernels.h"
#include <cmath>

namespace haste {

// ---------------------------------------------------------------------------------
// Xt[f][b] = X[b][f]; columns B..Bzero-1 are written as zeros.  32x32 smem tile.
// ---------------------------------------------------------------------------------
template <typename T>
__global__ void transpose_pad_kernel(const T* __restrict__ X, T* __restrict__ Xt, int B, int d, int Bpad, int Bzero) {
  __shared__ T tile[32][33];
  const int f0 = blockIdx.x * 32, b0 = blockIdx.y * 32;
  const int tx = threadIdx.x, ty = threadIdx.y;  // 32 x 8
  pdl_wait();
  pdl_trigger();
#pragma unroll
  for (int r = ty; r < 32; r += 8) {
    const int b = b0 + r, f = f0 + tx;
    T v = from_f32<T>(0.f);
    if (b < B && f < d) v = X[(int64_t)b * d + f];
    tile[r][tx] = v;
  }
  __syncthreads();
#pragma unroll
  for (int r = ty; r < 32; r += 8) {
    const int f = f0 + r, b = b0 + tx;
    if (f < d && b < Bzero) Xt[(int64_t)f * Bpad + b] = tile[tx][r];
  }
}

int launch_transpose_pad(haste_dtype_t dt, const void* X, void* Xt, int B, int d, int Bpad, int Bzero, cudaStream_t st) {
  dim3 grid(ceil_div(d, 32), ceil_div(Bzero, 32)), block(32, 8);
  if (dt == HASTE_F32)
    HASTE_CUDA_TRY(launch_pdl(transpose_pad_kernel<float>, grid, block, 0, st, (const float*)X, (float*)Xt, B, d, Bpad, Bzero));
  else
    HASTE_CUDA_TRY(launch_pdl(transpose_pad_kernel<bf16>, grid, block, 0, st, (const bf16*)X, (bf16*)Xt, B, d, Bpad, Bzero));
  return HASTE_OK;
}

// dX[b][f] (=|+=) dXt[f][b]; what is read from dXt is zeroed behind it, so the workspace is clean for the next backward
// pass without a memset between that pass's kernels (haste_api.cu keeps a host flag for the passes that end early)
__global__ void untranspose_f32_kernel(float* __restrict__ dXt, float* __restrict__ dX, int B, int d, int Bpad,
                                       int accumulate) {
  __shared__ float tile[32][33];
  const int b0 = blockIdx.x * 32, f0 = blockIdx.y * 32;
  const int tx = threadIdx.x, ty = threadIdx.y;
  pdl_wait();
  pdl_trigger();
  float v[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {       // all four loads first: the stores behind them may alias as far as the compiler knows
    const int f = f0 + ty + 8 * i, b = b0 + tx;
    v[i] = (f < d && b < B) ? __ldcg(dXt + (int64_t)f * Bpad + b) : 0.f;
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int f = f0 + ty + 8 * i, b = b0 + tx;
    if (f < d && b < B) dXt[(int64_t)f * Bpad + b] = 0.f;
    tile[ty + 8 * i][tx] = v[i];
  }
  __syncthreads();
#pragma unroll
  for (int r = ty; r < 32; r += 8) {
    const int b = b0 + r, f = f0 + tx;
    if (b < B && f < d) {
      float v = tile[tx][r];
      float* p = dX + (int64_t)b * d + f;
      if (accumulate) v += *p;
      *p = v;
    }
  }
}

int launch_untranspose_f32(float* dXt, float* dX, int B, int d, int Bpad, int accumulate, cudaStream_t st) {
  dim3 grid(ceil_div(B, 32), ceil_div(d, 32)), block(32, 8);
  HASTE_CUDA_TRY(launch_pdl(untranspose_f32_kernel, grid, block, 0, st, dXt, dX, B, d, Bpad, accumulate));
  return HASTE_OK;
}

// HASTE_DETERMINISTIC: dXt[f][bt*128 + r] = sum over stripes s (in order) of part[s*NT + bt][f][r]   (tc_dx_acc.cu private tiles)
__global__ void reduce_dx_parts_kernel(const float* __restrict__ part, float* __restrict__ dXt, int d, int Bpad, int NT, int S) {
  const int r = threadIdx.x, f = blockIdx.x, bt = blockIdx.y;
  float v = 0.f;
  for (int s = 0; s < S; ++s) v += part[((size_t)(s * NT + bt) * d + f) * 128 + r];
  dXt[(size_t)f * Bpad + bt * 128 + r] = v;
}
int launch_reduce_dx_parts(const float* part, float* dXt, int d, int Bpad, int NT, int S, cudaStream_t st) {
  reduce_dx_parts_kernel<<<dim3(d, NT), 128, 0, st>>>(part, dXt, d, Bpad, NT, S);
  HASTE_LAUNCH_CHECK();
  return HASTE_OK;
}

// loss = scale * (acc + sum(partials[0..n)))  -- one thread, fixed order: deterministic.
__global__ void finalize_loss_kernel(const double* acc, const float* partials, int n, float scale, float* loss) {
  __shared__ double red[256];
  double v = 0.0;
  for (int i = threadIdx.x; i < n; i += blockDim.x) v += (double)partials[i];
  red[threadIdx.x] = v;
  __syncthreads();
  for (int o = blockDim.x / 2; o > 0; o >>= 1) {
    if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) *loss = (float)((double)scale * ((acc ? *acc : 0.0) + red[0]));
}

int launch_finalize_loss(const double* acc, const float* partials, int n_partials, float scale, float* loss,
                         cudaStream_t st) {
  finalize_loss_kernel<<<1, 256, 0, st>>>(acc, partials, n_partials, scale, loss);
  HASTE_LAUNCH_CHECK();
  return HASTE_OK;
}

// ---------------------------------------------------------------------------------
// Fused top-k inference (Eq. 4): merge of the candidates the forward kernel's epilogue threads kept
// (8 per thread; tc_tail.cu, z_mode 2).  Batch row b sits in batch tile bt = b / 128 of tile pair pr = bt / 2; its
// candidates are those of CTAs (stripe s, pair pr), s < S, and of the epilogue sets that worked on that tile (all sets if
// the pair has one tile, the sets of matching parity if it has two).  One warp per row: every lane keeps the best 8 of
// its share, then k rounds of a warp-wide arg-max (ties: larger value first, then smaller label index) pop the winners.
// ---------------------------------------------------------------------------------
__global__ void topk_merge_kernel(const float* __restrict__ cv, const int* __restrict__ ci, int NP, int S, int NSET, int NT,
                                  int B, int k, int64_t label_offset, float* __restrict__ out_val, int64_t* __restrict__ out_idx) {
  const int b = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (b >= B) return;
  const int bt = b >> 7, r = b & 127, pr = bt >> 1;
  const int ntp = min(2, NT - 2 * pr);
  const int nsets = ntp == 2 ? NSET / 2 : NSET;           // sets that saw this tile
  const int per_cta = nsets * 8, total = S * per_cta;
  float tv[8];
  int ti[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) { tv[i] = -INFINITY; ti[i] = 0x7fffffff; }
  // 8 candidates per lane at a time: their loads are in flight together (one by one the scan is a chain of L2 round trips:
  // 42 us for 512 rows), then they are inserted in order
  for (int e0 = lane; e0 < total; e0 += 32 * 8) {
    float zc[8];
    int lc[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int e = e0 + 32 * u;
      zc[u] = -INFINITY; lc[u] = -1;
      if (e < total) {
        const int s = e / per_cta, w = e - s * per_cta;
        const int set = ntp == 2 ? 2 * (w >> 3) + (bt & 1) : (w >> 3);
        const size_t o = ((((size_t)s * NP + pr) * NSET + set) * 128 + r) * 8 + (w & 7);
        zc[u] = __ldcg(cv + o);
        lc[u] = __ldcg(ci + o);
      }
    }
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const float z = zc[u];
      const int l = lc[u];
      if (l >= 0 && (z > tv[7] || (z == tv[7] && l < ti[7]))) {
        tv[7] = z; ti[7] = l;
#pragma unroll
        for (int i = 7; i > 0; --i)
          if (tv[i] > tv[i - 1] || (tv[i] == tv[i - 1] && ti[i] < ti[i - 1])) {
            const float a = tv[i]; tv[i] = tv[i - 1]; tv[i - 1] = a;
            const int c = ti[i]; ti[i] = ti[i - 1]; ti[i - 1] = c;
          }
      }
    }
  }
  for (int round = 0; round < k; ++round) {
    float bv = tv[0];
    int bi = ti[0], bl = lane;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const float ov = __shfl_xor_sync(0xffffffffu, bv, o);
      const int oi = __shfl_xor_sync(0xffffffffu, bi, o), ol = __shfl_xor_sync(0xffffffffu, bl, o);
      if (ov > bv || (ov == bv && (oi < bi || (oi == bi && ol < bl)))) { bv = ov; bi = oi; bl = ol; }
    }
    if (lane == 0) {
      out_val[(size_t)b * k + round] = bv;
      out_idx[(size_t)b * k + round] = bi == 0x7fffffff ? -1 : label_offset + bi;
    }
    if (lane == bl) {       // the winner pops its head
#pragma unroll
      for (int i = 0; i < 7; ++i) { tv[i] = tv[i + 1]; ti[i] = ti[i + 1]; }
      tv[7] = -INFINITY; ti[7] = 0x7fffffff;
    }
  }
}
int launch_topk_merge(const float* cv, const int* ci, int NP, int S, int NSET, int NT, int B, int k, int64_t label_offset,
                      float* out_val, int64_t* out_idx, cudaStream_t st) {
  topk_merge_kernel<<<ceil_div(B, 4), 128, 0, st>>>(cv, ci, NP, S, NSET, NT, B, k, label_offset, out_val, out_idx);
  HASTE_LAUNCH_CHECK();
  return HASTE_OK;
}

// dY library layout: element (i,l) at ((l/G)*B + i)*G + l%G.
template <typename T>
__global__ void dy_unpack_kernel(const T* __restrict__ dY, float* __restrict__ out, int B, int64_t L, int G) {
  const int64_t n = (int64_t)B * L;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
    const int64_t i = e / L, l = e % L;
    out[e] = to_f32(dY[((l / G) * B + i) * G + (l % G)]);
  }
}
template <typename T>
__global__ void dy_pack_kernel(const float* __restrict__ in, T* __restrict__ dY, int B, int64_t L, int G, int64_t NG) {
  const int64_t n = NG * B * G;  // padding labels (>= L) of the last group are written as zero
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
    const int64_t g = e / ((int64_t)B * G), r = e % ((int64_t)B * G);
    const int64_t i = r / G, l = g * G + r % G;
    dY[e] = from_f32<T>(l < L ? in[i * L + l] : 0.f);
  }
}

int launch_dy_unpack(haste_dtype_t dt, const void* dY, float* out_BL, int B, int64_t L, int G, cudaStream_t st) {
  const int64_t n = (int64_t)B * L;
  const int blocks = (int)((n + 255) / 256 < 148 * 16 ? (n + 255) / 256 : 148 * 16);
  if (n == 0) return HASTE_OK;
  if (dt == HASTE_F32)
    dy_unpack_kernel<float><<<blocks, 256, 0, st>>>((const float*)dY, out_BL, B, L, G);
  else
    dy_unpack_kernel<bf16><<<blocks, 256, 0, st>>>((const bf16*)dY, out_BL, B, L, G);
  HASTE_LAUNCH_CHECK();
  return HASTE_OK;
}

int launch_dy_pack(haste_dtype_t dt, const float* in_BL, void* dY, int B, int64_t L, int G, cudaStream_t st) {
  const int64_t NG = (L + G - 1) / G, n = NG * B * G;
  if (n == 0) return HASTE_OK;
  const int blocks = (int)((n + 255) / 256 < 148 * 16 ? (n + 255) / 256 : 148 * 16);
  if (dt == HASTE_F32)
    dy_pack_kernel<float><<<blocks, 256, 0, st>>>(in_BL, (float*)dY, B, L, G, NG);
  else
    dy_pack_kernel<bf16><<<blocks, 256, 0, st>>>(in_BL, (bf16*)dY, B, L, G, NG);
  HASTE_LAUNCH_CHECK();
  return HASTE_OK;
}

// flag |= 1 if any value is outside [0,d); flag |= 2 if check_sorted and a row is not strictly ascending.
__global__ void validate_index_kernel(const int32_t* __restrict__ idx, int64_t n, int K, int d, int check_sorted,
                                      int* flag) {
  int bad = 0;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
    const int v = idx[e];
    if (v < 0 || v >= d) bad |= 1;
    if (check_sorted && (e % K) != 0 && idx[e - 1] >= v) bad |= 2;
  }
  if (bad) atomicOr(flag, bad);
}

int launch_validate_index(const int32_t* idx, int64_t NG, int K, int d, int check_sorted, int* flag, cudaStream_t st) {
  const int64_t n = NG * K;
  if (n == 0) return HASTE_OK;
  const int blocks = (int)((n + 255) / 256 < 148 * 8 ? (n + 255) / 256 : 148 * 8);
  validate_index_kernel<<<blocks, 256, 0, st>>>(idx, n, K, d, check_sorted, flag);
  HASTE_LAUNCH_CHECK();
  return HASTE_OK;
}

}  // namespace haste
