// rewire.cu -- Algorithm 3 of the paper, group-shared rewiring of the fixed fan-in supports, on the GPU.
//
//   1. scores   S[k,j] = mean over the labels l of group k of |w_l[j]|            one streaming pass over W
//   2. select   the m = floor(NG K rho) smallest entries of S                     radix select on the fp32 bit patterns
//   3. regrow   I_k[j] <- Unif{0..d-1} for every selected (k,j)                   counter-based generator
//   4. reinit   w_l[j] <- 0 or Unif(-1/sqrt(K), 1/sqrt(K)) for the group's labels
//   (+ momentum of reinitialised weights <- 0; optional stable re-sort of the touched idx rows with their columns)
// Readings: DESIGN.md R15.  A score decides an integer (which slots go), so it is computed in a fixed way -- fp32, labels
// added in ascending order, one division by the label count -- and ties go to the smaller flat index k K + j: the result
// does not depend on the launch configuration.  Random numbers: SplitMix64 finaliser of seed + golden ratio * (counter + 1).
// Everything here is HBM- or L2-bound bookkeeping (W is read once, the 4-byte scores are L2-resident); any (G, K, dtype).
#include <cmath>

#include "kernels.h"

namespace haste {

__device__ __forceinline__ uint64_t rw_mix(uint64_t seed, uint64_t counter) {
  uint64_t z = seed + 0x9e3779b97f4a7c15ULL * (counter + 1);
  z = (z ^ (z >> 30)) * 0xbf58476d1ce4e5b9ULL;
  z = (z ^ (z >> 27)) * 0x94d049bb133111ebULL;
  return z ^ (z >> 31);
}

// ---- 1. scores: block = one group, thread j walks its column of the group's rows (coalesced across j)
template <typename T>
__global__ void rw_scores_kernel(const T* __restrict__ W, float* __restrict__ S, int64_t L, int G, int K) {
  const int64_t k = blockIdx.x;
  const int64_t l0 = k * G, l1 = min(L, l0 + (int64_t)G);
  for (int j = threadIdx.x; j < K; j += blockDim.x) {
    float acc = 0.f;
    for (int64_t l = l0; l < l1; ++l) acc = acc + fabsf(to_f32(W[l * K + j]));
    S[k * K + j] = acc / (float)(l1 - l0);
  }
}

// ---- 2a. the m-th smallest key (scores are >= 0, so their bit patterns order like the values): 4 passes of 8 bits, one block
// out[0] = the key t; out[1] = how many of the entries EQUAL to t are taken (all entries below t are)
__global__ void rw_select_kernel(const uint32_t* __restrict__ keys, int64_t n, int64_t m, uint32_t* __restrict__ out) {
  __shared__ unsigned int hist[256];
  __shared__ uint32_t s_prefix;
  __shared__ long long s_rem;
  if (threadIdx.x == 0) { s_prefix = 0u; s_rem = m; }
  for (int pass = 0; pass < 4; ++pass) {
    const int shift = 24 - 8 * pass;
    const uint32_t himask = pass == 0 ? 0u : 0xffffffffu << (shift + 8);
    for (int i = threadIdx.x; i < 256; i += blockDim.x) hist[i] = 0u;
    __syncthreads();
    const uint32_t prefix = s_prefix;
    // scores crowd into a few digits: lanes with the same digit elect one of them to add for all (one atomic per warp and
    // digit instead of 32 on one word)
    for (int64_t base = 0; base < n; base += blockDim.x) {
      const int64_t e = base + threadIdx.x;
      const uint32_t key = e < n ? keys[e] : 0u;
      const bool in = e < n && (key & himask) == prefix;
      const uint32_t dg = in ? (key >> shift) & 255u : 0xffffffffu;
      const unsigned peers = __match_any_sync(0xffffffffu, dg);
      if (in && (threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(&hist[dg], (unsigned)__popc(peers));
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      long long rem = s_rem, cum = 0;
      int dg = 0;
      for (; dg < 256; ++dg) {
        if (cum + hist[dg] >= rem) break;
        cum += hist[dg];
      }
      s_rem = rem - cum;
      s_prefix = prefix | ((uint32_t)dg << shift);
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) { out[0] = s_prefix; out[1] = (uint32_t)s_rem; }
}

// ---- 2b. entries equal to t per chunk of RW_CHUNK entries (for the rank of an equal entry in flat-index order)
constexpr int RW_CHUNK = 4096;
__global__ void rw_count_kernel(const uint32_t* __restrict__ keys, int64_t n, const uint32_t* __restrict__ sel, int* __restrict__ counts) {
  __shared__ int s_cnt;
  if (threadIdx.x == 0) s_cnt = 0;
  __syncthreads();
  const uint32_t t = sel[0];
  const int64_t e0 = (int64_t)blockIdx.x * RW_CHUNK;
  int c = 0;
  for (int i = threadIdx.x; i < RW_CHUNK; i += blockDim.x)
    if (e0 + i < n && keys[e0 + i] == t) ++c;
  if (c) atomicAdd(&s_cnt, c);
  __syncthreads();
  if (threadIdx.x == 0) counts[blockIdx.x] = s_cnt;
}

// ---- 2c. the mask: key < t, or key == t and fewer than need_eq equal entries precede it in flat-index order
__global__ void rw_mark_kernel(const uint32_t* __restrict__ keys, int64_t n, const uint32_t* __restrict__ sel, const int* __restrict__ counts,
                               unsigned char* __restrict__ mask) {
  __shared__ int s_base;
  __shared__ int s_scan[256];
  const uint32_t t = sel[0];
  const long long need_eq = sel[1];
  if (threadIdx.x == 0) {
    long long b = 0;
    for (int i = 0; i < (int)blockIdx.x; ++i) b += counts[i];
    s_base = (int)min(b, (long long)0x7fffffff);
  }
  __syncthreads();
  const int64_t e0 = (int64_t)blockIdx.x * RW_CHUNK;
  // thread i owns the contiguous run [i * PER, (i + 1) * PER) of the chunk, so that ranks follow the flat index
  constexpr int PER = RW_CHUNK / 256;
  int c = 0;
  for (int r = 0; r < PER; ++r) {
    const int64_t e = e0 + threadIdx.x * PER + r;
    if (e < n && keys[e] == t) ++c;
  }
  s_scan[threadIdx.x] = c;
  __syncthreads();
  for (int o = 1; o < 256; o <<= 1) {       // inclusive scan (Hillis-Steele)
    const int v = threadIdx.x >= o ? s_scan[threadIdx.x - o] : 0;
    __syncthreads();
    s_scan[threadIdx.x] += v;
    __syncthreads();
  }
  long long rank = (long long)s_base + s_scan[threadIdx.x] - c;
  for (int r = 0; r < PER; ++r) {
    const int64_t e = e0 + threadIdx.x * PER + r;
    if (e >= n) break;
    const uint32_t key = keys[e];
    unsigned char mk = key < t ? 1 : 0;
    if (key == t) { mk = rank < need_eq ? 1 : 0; ++rank; }
    mask[e] = mk;
  }
}

// ---- 3 + 4 (+ momentum reset, + re-sort): block = one group
template <typename T>
__global__ void rw_apply_kernel(int32_t* __restrict__ idx, T* __restrict__ W, float* __restrict__ mom, const unsigned char* __restrict__ mask,
                                int64_t L, int G, int K, int d, int init_random, uint64_t seed, float r32, int resort) {
  extern __shared__ int sm[];
  int* s_idx = sm;                // [K] the row after regrowth
  int* s_perm = sm + K;           // [K] slot that moves to position j
  int* s_mask = sm + 2 * K;       // [K]
  float* s_row = reinterpret_cast<float*>(sm + 3 * K);   // [K]
  __shared__ int s_touched;
  const int64_t k = blockIdx.x;
  const int64_t l0 = k * G, l1 = min(L, l0 + (int64_t)G);
  if (threadIdx.x == 0) s_touched = 0;
  __syncthreads();
  for (int j = threadIdx.x; j < K; j += blockDim.x) {
    const int mk = mask[k * K + j];
    int f = idx[k * K + j];
    if (mk) {
      f = (int)__umul64hi(rw_mix(seed, (uint64_t)(k * K + j)), (uint64_t)d);     // floor(d h / 2^64): Unif{0..d-1}
      idx[k * K + j] = f;
      s_touched = 1;
    }
    s_idx[j] = f;
    s_mask[j] = mk;
  }
  __syncthreads();
  if (!s_touched) return;
  const int nl = (int)(l1 - l0);
  for (int e = threadIdx.x; e < nl * K; e += blockDim.x) {
    const int j = e % K;
    if (!s_mask[j]) continue;
    const int64_t l = l0 + e / K;
    float w = 0.f;
    if (init_random) {
      const uint64_t hw = rw_mix(seed ^ 0x5851f42d4c957f2dULL, (uint64_t)(l * K + j));
      const float a = (float)(2.0 * ((double)(hw >> 41) * (1.0 / 8388608.0)) - 1.0);     // exact: 23 random bits
      w = __fmul_rn(a, r32);
    }
    W[l * K + j] = from_f32<T>(w);
    if (mom) mom[l * K + j] = 0.f;
  }
  if (!resort) return;
  __syncthreads();
  // stable rank of every slot: slots with a smaller feature, or the same feature and a smaller position, come first
  for (int j = threadIdx.x; j < K; j += blockDim.x) {
    const int f = s_idx[j];
    int r = 0;
    for (int i = 0; i < K; ++i) r += (s_idx[i] < f) || (s_idx[i] == f && i < j);
    s_perm[r] = j;
  }
  __syncthreads();
  for (int j = threadIdx.x; j < K; j += blockDim.x) idx[k * K + j] = s_idx[s_perm[j]];
  for (int64_t l = l0; l < l1; ++l) {
    __syncthreads();
    for (int j = threadIdx.x; j < K; j += blockDim.x) s_row[j] = to_f32(W[l * K + j]);
    __syncthreads();
    for (int j = threadIdx.x; j < K; j += blockDim.x) W[l * K + j] = from_f32<T>(s_row[s_perm[j]]);
    if (mom) {
      __syncthreads();
      for (int j = threadIdx.x; j < K; j += blockDim.x) s_row[j] = mom[l * K + j];
      __syncthreads();
      for (int j = threadIdx.x; j < K; j += blockDim.x) mom[l * K + j] = s_row[s_perm[j]];
    }
  }
}

size_t rewire_workspace_bytes(int64_t NG, int K) {
  const int64_t n = NG * K;
  const int64_t nb = (n + RW_CHUNK - 1) / RW_CHUNK;
  return (size_t)(n * 4 + n + 16 + nb * 4 + 64);
}

// ws: rewire_workspace_bytes() bytes.  m = floor(NG K rho) is computed by the caller (host, double).
int launch_rewire(haste_dtype_t dt, int32_t* idx, void* W, float* mom, int64_t L, int G, int K, int d, int64_t m, int init_random,
                  uint64_t seed, int resort, void* ws, cudaStream_t st) {
  const int64_t NG = (L + G - 1) / G, n = NG * K;
  if (n == 0 || m <= 0) return HASTE_OK;
  if (m > n) m = n;
  const int64_t nb = (n + RW_CHUNK - 1) / RW_CHUNK;
  if (NG > 0x7fffffffLL || nb > 0x7fffffffLL || K > 3000) return HASTE_ERR_UNSUPPORTED;    // (apply kernel: 16 K bytes of shared memory)
  float* S = reinterpret_cast<float*>(ws);
  unsigned char* mask = reinterpret_cast<unsigned char*>(ws) + n * 4;
  uint32_t* sel = reinterpret_cast<uint32_t*>(reinterpret_cast<unsigned char*>(ws) + ((n * 5 + 15) / 16) * 16);
  int* counts = reinterpret_cast<int*>(sel + 4);
  const int tb = K >= 256 ? 256 : (K >= 128 ? 128 : 64);
  if (dt == HASTE_F32) rw_scores_kernel<float><<<(unsigned)NG, tb, 0, st>>>((const float*)W, S, L, G, K);
  else rw_scores_kernel<bf16><<<(unsigned)NG, tb, 0, st>>>((const bf16*)W, S, L, G, K);
  HASTE_LAUNCH_CHECK();
  rw_select_kernel<<<1, 1024, 0, st>>>(reinterpret_cast<const uint32_t*>(S), n, m, sel);
  HASTE_LAUNCH_CHECK();
  rw_count_kernel<<<(unsigned)nb, 256, 0, st>>>(reinterpret_cast<const uint32_t*>(S), n, sel, counts);
  HASTE_LAUNCH_CHECK();
  rw_mark_kernel<<<(unsigned)nb, 256, 0, st>>>(reinterpret_cast<const uint32_t*>(S), n, sel, counts, mask);
  HASTE_LAUNCH_CHECK();
  const float r32 = (float)(1.0 / std::sqrt((double)K));
  const size_t smem = (size_t)K * 16;
  if (dt == HASTE_F32)
    rw_apply_kernel<float><<<(unsigned)NG, 128, smem, st>>>(idx, (float*)W, mom, mask, L, G, K, d, init_random, seed, r32, resort);
  else
    rw_apply_kernel<bf16><<<(unsigned)NG, 128, smem, st>>>(idx, (bf16*)W, mom, mask, L, G, K, d, init_random, seed, r32, resort);
  HASTE_LAUNCH_CHECK();
  return HASTE_OK;
}

}  // namespace haste
