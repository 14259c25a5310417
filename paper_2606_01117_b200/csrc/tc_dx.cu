// tc_dx.cu -- tcgen05 input-gradient kernels of the HASTE sparse tail (sm_100a; bf16 in, fp32 accumulate).
//
//   dX[:, idx_g] += dY_g [B x G] * W_g [G x K]   over all groups g
//
// Kernel "red" (this file, first version): per (group, 128-row batch tile)
//   P^T [128 batch lanes x K slot columns] = dY tile (A, K-major, one TMA box) * W_g (B, MN-major: the
//   [G x K] block of W as it sits in HBM), fp32 in TMEM; the epilogue thread that owns batch row b adds
//   column k into dX^T[idx_g[k]][b] with red.global.add.f32 (a warp writes 32 consecutive floats of one
//   feature row).  The reduction over groups happens in L2: 1.47 T adds/s measured
//   (profiles/r01_probe_microbench.txt), which bounds this version.
#include <algorithm>
#include <cstdlib>
#include <cstring>

#include "tc_common.cuh"
#include "tc_kernels.h"

namespace haste {
using namespace tc;

struct DxParams {
  float* dXt;           // [d][Bpad] fp32, zeroed by the caller
  const int32_t* idx;   // [NG][K]
  int B, Bpad, NT, S;   // NT batch tiles of 128; S group stripes (grid = NT * S)
  int64_t NG;
};

template <int G, int K> struct DxCfg {
  static constexpr int Y_BYTES = G * 256;                 // [G/64 k-blocks][128 batch rows][128 B]
  static constexpr int W_BYTES = G * K * 2;               // [K/64 slot atoms][G label rows][128 B]
  static constexpr int I_BYTES = 1024;                    // K int32 (<= 512 B), padded
  static constexpr int STAGE = Y_BYTES + W_BYTES + I_BYTES;
  static constexpr int NST = STAGE <= 40960 ? 4 : 3;
  static constexpr int OFF_BAR = NST * STAGE;
  static constexpr int OFF_MISC = OFF_BAR + (2 * NST + 4) * 8;
  static constexpr int SMEM = OFF_MISC + 64 + 1024;
};

__device__ __forceinline__ void red_add_f32(float* addr, float v) {
  asm volatile("red.global.add.f32 [%0], %1;" ::"l"(addr), "f"(v) : "memory");
}
__device__ __forceinline__ void bulk_load_1d(uint32_t dst_smem, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst_smem), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ int lds32i(uint32_t addr) {
  int v;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}

template <int G, int K>
__global__ void __launch_bounds__(192, 1)
tc_dx_red_kernel(const __grid_constant__ CUtensorMap tmY, const __grid_constant__ CUtensorMap tmW, const DxParams p) {
  using C = DxCfg<G, K>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const uint32_t sbase = smem_u32(smem);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::OFF_BAR);
  uint64_t* full = bars;                    // [NST] count 1 + tx
  uint64_t* empty = bars + C::NST;          // [NST] count 5: umma commit + 4 epilogue warps (they read idx from the stage)
  uint64_t* t_full = bars + 2 * C::NST;     // [2]
  uint64_t* t_empty = t_full + 2;           // [2] count 4
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + C::OFF_MISC);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int bt = blockIdx.x % p.NT, stripe = blockIdx.x / p.NT;
  const int n_my = p.NG > stripe ? (int)((p.NG - stripe + p.S - 1) / p.S) : 0;

  if (threadIdx.x == 0) {
    for (int i = 0; i < C::NST; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], 5); }
    for (int i = 0; i < 2; ++i) { mbar_init(&t_full[i], 1); mbar_init(&t_empty[i], 4); }
    fence_barrier_init();
  }
  if (warp == 5 && lane == 0) { tma_prefetch_desc(&tmY); tma_prefetch_desc(&tmW); }
  if (warp == 4) tmem_alloc<2 * K>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 5) {
    if (lane == 0) {
      for (int i = 0; i < n_my; ++i) {
        const int64_t g = stripe + (int64_t)i * p.S;
        const int st = i % C::NST;
        mbar_wait(&empty[st], ((i / C::NST) & 1) ^ 1);
        mbar_arrive_expect_tx(&full[st], C::Y_BYTES + C::W_BYTES + K * 4);
        uint8_t* s0 = smem + st * C::STAGE;
#pragma unroll
        for (int kb = 0; kb < G / 64; ++kb) tma_load_3d(s0 + kb * 16384, &tmY, &full[st], kb * 64, bt * 128, (int)g);
#pragma unroll
        for (int a = 0; a < K / 64; ++a) tma_load_2d(s0 + C::Y_BYTES + a * (G * 128), &tmW, &full[st], a * 64, (int)(g * G));
        bulk_load_1d(sbase + st * C::STAGE + C::Y_BYTES + C::W_BYTES, p.idx + g * K, K * 4, &full[st]);
      }
    }
  } else if (warp == 4) {
    if (lane == 0) {
      constexpr uint32_t idesc = make_idesc_bf16(128, K, /*A (dY) K-major*/ 0, /*B (W) MN-major*/ 1);
      for (int i = 0; i < n_my; ++i) {
        const int st = i % C::NST, slot = i & 1;
        mbar_wait(&full[st], (i / C::NST) & 1);
        mbar_wait(&t_empty[slot], ((i >> 1) & 1) ^ 1);
        tc_fence_after();
        const uint32_t y0 = sbase + st * C::STAGE, w0 = y0 + C::Y_BYTES;
        const uint32_t d = tmem_base + slot * K;
#pragma unroll
        for (int j = 0; j < G / 16; ++j) {
          const uint64_t ad = make_sdesc_sw128(y0 + (j >> 2) * 16384 + (j & 3) * 32, 16, 1024);
          const uint64_t bd = make_sdesc_sw128(w0 + j * 2048, G * 128, 1024);
          umma_f16(d, ad, bd, idesc, j ? 1u : 0u);
        }
        umma_commit(&empty[st]);
        umma_commit(&t_full[slot]);
      }
    }
  } else {
    const int q = warp;
    const int b = bt * 128 + q * 32 + lane;
    const bool vb = b < p.B;
    for (int i = 0; i < n_my; ++i) {
      const int st = i % C::NST, slot = i & 1;
      mbar_wait(&full[st], (i / C::NST) & 1);       // idx of this group is in the stage
      mbar_wait(&t_full[slot], (i >> 1) & 1);
      tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + slot * K;
      const uint32_t sidx = sbase + st * C::STAGE + C::Y_BYTES + C::W_BYTES;
#pragma unroll 1
      for (int c = 0; c < K / 32; ++c) {
        uint32_t v[32];
        tmem_ld32(taddr + c * 32, v);
        tmem_ld_wait();
        if (vb) {
#pragma unroll
          for (int j = 0; j < 32; ++j) {
            const int f = lds32i(sidx + (c * 32 + j) * 4);
            red_add_f32(p.dXt + (size_t)f * p.Bpad + b, __uint_as_float(v[j]));
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) { mbar_arrive(&t_empty[slot]); mbar_arrive(&empty[st]); }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 4) { tc_fence_after(); tmem_dealloc<2 * K>(tmem_base); }
}


template <int G, int K>
static int launch_dx_red(TcTailState* s, const TailShape& sh, const int32_t* idx, const void* W, const void* dY, float* dXt,
                         cudaStream_t st) {
  using C = DxCfg<G, K>;
  static_assert(C::SMEM <= 232448, "shared memory budget");
  CUtensorMap tmY, tmW;
  {
    const uint64_t dims[3] = {(uint64_t)G, (uint64_t)sh.B, (uint64_t)sh.NG};
    const uint64_t str[2] = {(uint64_t)G * 2, (uint64_t)sh.B * G * 2};
    const uint32_t box[3] = {64, 128, 1};
    int rc = encode_tmap(&tmY, 2, dY, 3, dims, str, box, 128);
    if (rc) return rc;
  }
  {
    const uint64_t dims[2] = {(uint64_t)K, (uint64_t)sh.L};
    const uint64_t str[1] = {(uint64_t)K * 2};
    const uint32_t box[2] = {64, (uint32_t)G};
    int rc = encode_tmap(&tmW, 2, W, 2, dims, str, box, 128);
    if (rc) return rc;
  }
  DxParams p;
  p.dXt = dXt; p.idx = idx; p.B = sh.B; p.Bpad = sh.Bpad; p.NT = ceil_div(sh.B, 128); p.NG = sh.NG;
  if (p.NT > s->num_sms) return HASTE_ERR_UNSUPPORTED;
  p.S = (int)std::min<int64_t>(sh.NG, std::max(1, s->num_sms / p.NT));
  HASTE_CUDA_TRY(cudaFuncSetAttribute(tc_dx_red_kernel<G, K>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM));
  tc_dx_red_kernel<G, K><<<p.NT * p.S, 192, C::SMEM, st>>>(tmY, tmW, p);
  HASTE_LAUNCH_CHECK();
  return HASTE_OK;
}

void tc_tail_dx_grid(const TcTailState* s, const TailShape& sh, int* NT, int* S) {
  *NT = ceil_div(sh.B, 128);
  *S = (int)std::min<int64_t>(sh.NG, std::max(1, s->num_sms / *NT));
}
int tc_tail_num_sms(const TcTailState* s) { return s->num_sms; }

int tc_tail_dx(TcTailState* s, const TailShape& sh, const int32_t* idx, const void* W, const void* dY, float* dXt,
               float* dx_part, cudaStream_t st, int* n_launches) {
  *n_launches = 1;
  if (dx_part) {   // deterministic mode: only the accumulating kernel has an atomic-free variant
    if ((sh.G == 32 || sh.G == 64 || sh.G == 128) && (sh.K == 64 || sh.K == 128)) return tc_tail_dx_acc(s, sh, idx, W, dY, dXt, dx_part, st);
    return HASTE_ERR_UNSUPPORTED;
  }
  static const bool use_red = getenv("HASTE_DX_KERNEL") && !strcmp(getenv("HASTE_DX_KERNEL"), "red");   // first version, for comparison
  static const bool use_mma = getenv("HASTE_DX_KERNEL") && !strcmp(getenv("HASTE_DX_KERNEL"), "mma");
  static const bool use_hyb = getenv("HASTE_DX_KERNEL") && !strcmp(getenv("HASTE_DX_KERNEL"), "hyb");
  if (use_hyb) {
    const int rc = tc_tail_dx_hyb(s, sh, idx, W, dY, dXt, st);
    if (rc != HASTE_ERR_UNSUPPORTED) return rc;
  }
  if (use_mma) {
    const int rc = tc_tail_dx_mma(s, sh, idx, W, dY, dXt, st);
    if (rc != HASTE_ERR_UNSUPPORTED) return rc;
  }
#define HASTE_DX(G_, K_)                                                                   \
  if (sh.G == G_ && sh.K == K_)                                                            \
    return use_red ? launch_dx_red<G_, K_>(s, sh, idx, W, dY, dXt, st) : tc_tail_dx_acc(s, sh, idx, W, dY, dXt, nullptr, st)
  HASTE_DX(64, 128); HASTE_DX(64, 64); HASTE_DX(128, 64); HASTE_DX(128, 128);
#undef HASTE_DX
  if (sh.G == 32 && (sh.K == 64 || sh.K == 128)) return tc_tail_dx_acc(s, sh, idx, W, dY, dXt, nullptr, st);   // 64-byte-swizzle operand: acc kernel only
  return HASTE_ERR_UNSUPPORTED;
}

}  // namespace haste
