// tc_dw.cu -- tcgen05 weight-gradient kernel of the HASTE sparse tail (sm_100a; bf16 in, fp32 accumulate).
//
//   dW_g [G x K] = dY_g^T [G x B] * H_g [B x K],  H_g = X[:, idx_g]
//   db_g [G]     = dY_g^T * 1
//
// Persistent CTAs, one per SM, groups strided over the grid.  The batch (the contraction) is streamed in
// k-blocks of 64 rows through a shared-memory ring:
//   A operand (M = labels): the dY k-block [64 batch rows][G labels] exactly as it sits in HBM (one TMA box per
//     64 labels, 128-byte swizzle) read as an MN-major operand -- no transposition anywhere;
//   B operand (N = fan-in slots): H^T k-block [K rows][64 batch] gathered from X^T with 16-byte cp.async
//     (a row of X^T is one feature, batch contiguous), K-major; the image carries a few extra rows of
//     ones, so accumulator column K is sum_b dY[b][l] = db[l] at no extra operand traffic.
//   D [G lanes x (K + extra) columns] fp32 in TMEM, double buffered across groups.
// warp roles (320 threads): warps 0-3 epilogue (TMEM -> registers -> swizzled smem rows -> TMA store of dW
// rows; a thread owns one label, so a dW row is written as it is stored), warps 4-7 gather producers,
// warp 8 MMA issuer, warp 9 TMA loader of dY.
#include <algorithm>
#include <cstring>

#include "tc_common.cuh"
#include "tc_kernels.h"

namespace haste {
using namespace tc;

struct DwParams {
  const bf16* Xt;       // [d][Bpad], zero for b >= B up to the next multiple of 128
  const int32_t* idx;   // [NG][K]
  float* dbias;         // [L] or null
  int write_dw;
  // SGD instance (haste_backward_sgd): the gradient never leaves the chip; W and the momentum are updated in place
  bf16* W;              // [L][K] in/out
  float* mom;           // [L][K] fp32 momentum buffer, in/out
  float* bias;          // [L] in/out or null
  float* bmom;          // [L] in/out or null (required with bias)
  float lr, mu, wd;
  int B, Bpad, NKB;     // NKB = ceil(B / 128) k-blocks
  int64_t L, NG;
};

template <int G, int K, bool F32, bool SGD = false> struct DwCfg {
  // G = 32: two consecutive groups form one virtual group of GV = 64 labels and KV = 2K slots (their idx rows are
  // adjacent in memory, so are their labels).  D [64 x 2K] then holds dW_g in rows 0-31 x columns [0,K) and dW_{g+1}
  // in rows 32-63 x columns [K,2K); the off-diagonal blocks are computed and ignored (the tensor pipe has the room).
  // G < 64 otherwise (G = 32 with K = 128, whose pair would need N = 264; G = 16; G = 8): the MMA is still M = 64, but only
  // its first G label rows are real -- the A descriptor walks on into whatever follows the dY image, and accumulator
  // rows G .. 63 are never read (rows of D are independent).  The tensor pipe has the room: what bounds a narrow group
  // is the gather of its K feature rows, which G labels share instead of 64.  G = 8: the TMA box is 16 labels wide over
  // a tensor that has 8, so labels 8-15 of every row arrive as zeros and the image is the G = 16 one.
  static constexpr bool PAIR = G == 32 && K == 64;
  static constexpr bool PADM = G < 64 && !PAIR;
  static constexpr int GL = PAIR ? 64 : G;                  // labels per (virtual) group
  static constexpr int GV = G < 64 ? 64 : G;                // MMA M
  static constexpr int YROW = PADM ? (G >= 32 ? 64 : 32) : (PAIR ? 64 : 128);   // bytes per batch row of the dY image
  static constexpr int KV = PAIR ? 2 * K : K;               // gathered slots per (virtual) group
  static constexpr int NE = GV == 128 ? 16 : 8;             // rows of ones appended to the H image
  static constexpr int N = KV + NE;                         // MMA N
  static_assert(N <= 256, "MMA N");
  // a k-block is 128 batch rows = two 64-row halves (one 128-byte swizzle row holds 64 bf16): the issuing thread
  // pays one barrier wait and one commit per 8 MMAs (with 64-row k-blocks its ~0.3 us loop overhead per k-block
  // was the kernel's bottleneck)
  static constexpr int HH_BYTES = (KV + 16) * 128;          // one half of the H image, multiple of 1024
  static constexpr int YH_BYTES = PADM ? 64 * YROW : GV * 128;   // one half of the dY image: [G/64 atoms][64 rows][128 B]; PAIR: [2 groups][64 rows][64 B]; PADM: [64 rows][YROW]
  static constexpr int H_BYTES = 2 * HH_BYTES;
  static constexpr int Y_BYTES = 2 * YH_BYTES;
  static constexpr int STAGE = H_BYTES + Y_BYTES;
  static constexpr int EPI_BYTES = 4 * 4096;                // 4 warps x [32 rows][128 B]
  static constexpr int NST_RAW = (232448 - 1024 - EPI_BYTES - 1024) / STAGE;
  static constexpr int NST = NST_RAW > 8 ? 8 : NST_RAW;
  // producer completion lag: LAG + 1 k-blocks of cp.async in flight per producer warp.  A narrow group's k-block is the same
  // gather for a fraction of the labels, so there the gather's latency is what bounds the kernel: more in flight
  static constexpr int LAG = 2;
  // narrow groups: each producer warp gathers every fourth k-block whole (all K rows), as in the forward (tc_tail.cu,
  // FwdCfg::NARROW): its wait / issue / wait-for-copies / fence / arrive chain is then on the critical path a quarter as often
  static constexpr bool ROT = G <= 16;
  static constexpr int TS = N <= 128 ? 128 : 256;           // TMEM columns per accumulator slot
  static constexpr int OFF_EPI = NST * STAGE;
  static constexpr int OFF_BAR = OFF_EPI + EPI_BYTES;
  static constexpr int NBAR = 2 * NST + 4;
  static constexpr int OFF_MISC = OFF_BAR + NBAR * 8;
  static constexpr int SMEM = OFF_MISC + 64 + 1024;
  static constexpr int RW = GV == 128 ? 32 : 16;            // label rows per epilogue warp (M = 64 fills lanes 0-15 of a quadrant)
  static constexpr int NBOX = F32 ? K / 32 : K / 64;        // 128-byte output boxes per dW row
  static_assert(NST > LAG, "ring too short");
};

__device__ __forceinline__ uint32_t dw_pack_bf16x2(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&v);
}
__device__ __forceinline__ uint32_t tmem_ld1(uint32_t taddr) {
  uint32_t v;
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(v) : "r"(taddr) : "memory");
  return v;
}

template <int G, int K, bool F32, bool SGD>
__global__ void __launch_bounds__(320, 1)
tc_dw_kernel(const __grid_constant__ CUtensorMap tmY, const __grid_constant__ CUtensorMap tmO, const DwParams p) {
  using C = DwCfg<G, K, F32, SGD>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const uint32_t sbase = smem_u32(smem);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::OFF_BAR);
  uint64_t* full = bars;                    // [NST] count 5: 4 producer warps + the TMA thread (expect_tx)
  uint64_t* empty = bars + C::NST;          // [NST] count 1: umma commit
  uint64_t* t_full = bars + 2 * C::NST;     // [2]   count 1: umma commit
  uint64_t* t_empty = t_full + 2;           // [2]   count 4: epilogue warps
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + C::OFF_MISC);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t NGV = C::PAIR ? (p.NG + 1) / 2 : p.NG;                                               // (virtual) groups
  const int n_my = NGV > blockIdx.x ? (int)((NGV - blockIdx.x + gridDim.x - 1) / gridDim.x) : 0;     // groups of this CTA
  // ... taken from the LAST group down: the forward kernel before this one wrote dY in ascending group order, so the
  // groups written last are the ones still in the 126 MB L2 (and the dX kernel after this one, ascending again, finds
  // the groups this kernel read last)
  auto group_of = [&](int i) -> int64_t { return NGV - 1 - (blockIdx.x + (int64_t)i * gridDim.x); };

  if (threadIdx.x == 0) {
    for (int i = 0; i < C::NST; ++i) { mbar_init(&full[i], C::ROT ? 2 : 5); mbar_init(&empty[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&t_full[i], 1); mbar_init(&t_empty[i], 4); }
    fence_barrier_init();
  }
  // rows K .. K+15 of every stage's H image: bf16 1.0 (swizzling permutes equal chunks: write linearly)
  for (int e = threadIdx.x; e < C::NST * 2 * 16 * 8; e += blockDim.x) {
    const int st = e / 256, hf = (e >> 7) & 1, r = e % 128;
    sts128(sbase + st * C::STAGE + hf * C::HH_BYTES + C::KV * 128 + r * 16, 0x3F803F80u, 0x3F803F80u, 0x3F803F80u, 0x3F803F80u);
  }
  fence_proxy_async_smem();
  if (warp == 9 && lane == 0) { tma_prefetch_desc(&tmY); tma_prefetch_desc(&tmO); }
  if (warp == 8) tmem_alloc<2 * C::TS>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  pdl_wait();       // nothing above touches global memory (common.cuh, PDL)
  pdl_trigger();
  const uint32_t tmem_base = *tmem_slot;

  if (warp >= 4 && warp < 8) {
    // ===================== gather producers =====================
    const int pw = warp - 4;
    const int sub = lane >> 3, c = lane & 7;         // 4 rows per instruction, 8 chunks of 16 B per row
    if constexpr (C::ROT) {
      // k-blocks it = pw, pw + 4, ... of this CTA's sequence (group i = it / NKB, k-block kb = it % NKB); lane holds slots
      // lane + 32 t of the current group's idx row; two k-blocks of copies in flight per warp
      constexpr int NI = K / 32;
      int idx_cur[NI];
#pragma unroll
      for (int t = 0; t < NI; ++t) idx_cur[t] = 0;
      int i_cur = -1, prev_st = -1;
      const int n_it = n_my * p.NKB;
      for (int it = pw; it < n_it; it += 4) {
        const int i = it / p.NKB, kb = it - i * p.NKB;
        if (i != i_cur) {
          i_cur = i;
          const int64_t g = group_of(i);
#pragma unroll
          for (int t = 0; t < NI; ++t) idx_cur[t] = __ldg(p.idx + g * K + lane + 32 * t);
        }
        const int st = it % C::NST;
        mbar_wait(&empty[st], ((it / C::NST) & 1) ^ 1);
        const uint32_t dst0 = sbase + st * C::STAGE;
        const bf16* src0 = p.Xt + kb * 128 + c * 8;
#pragma unroll
        for (int r4 = 0; r4 < K / 4; ++r4) {
          const int row = 4 * r4 + sub;
          const int f = __shfl_sync(0xffffffffu, idx_cur[(4 * r4) >> 5], row & 31);
          const uint32_t dst = dst0 + row * 128 + (((uint32_t)(c ^ (row & 7))) << 4);
          const bf16* src = src0 + (size_t)f * p.Bpad;
          cp_async16(dst, src);
          cp_async16(dst + C::HH_BYTES, src + 64);
        }
        cp_async_commit();
        if (prev_st >= 0) {
          cp_async_wait<1>();
          fence_proxy_async_smem();
          __syncwarp();
          if (lane == 0) mbar_arrive(&full[prev_st]);
        }
        prev_st = st;
      }
      if (prev_st >= 0) {
        cp_async_wait<0>();
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) mbar_arrive(&full[prev_st]);
      }
    } else {
    constexpr int RPW = C::KV / 4;                   // slots per producer warp
    // slot (pw*RPW + lane) of virtual group v is idx[v*KV + slot]; the second half of an unpaired last virtual group
    // (no group 2v+1) re-reads the first half's indices: its dY is zero-filled, its output rows are clipped
    auto idx_of = [&](int64_t v) -> int {
      int64_t off = v * C::KV + pw * RPW + lane;
      if (C::PAIR && pw * RPW + lane >= K && 2 * v + 1 >= p.NG) off -= K;
      return __ldg(p.idx + off);
    };
    int idx_cur = 0, idx_nxt = 0;
    if (lane < RPW && n_my > 0) idx_nxt = idx_of(group_of(0));
    int it = 0;
    for (int i = 0; i < n_my; ++i) {
      idx_cur = idx_nxt;
      if (lane < RPW && i + 1 < n_my) idx_nxt = idx_of(group_of(i + 1));
      for (int kb = 0; kb < p.NKB; ++kb, ++it) {
        const int st = it % C::NST;
        mbar_wait(&empty[st], ((it / C::NST) & 1) ^ 1);
        const uint32_t dst0 = sbase + st * C::STAGE;
        const bf16* src0 = p.Xt + kb * 128 + c * 8;
#pragma unroll
        for (int r4 = 0; r4 < RPW / 4; ++r4) {
          const int rr = 4 * r4 + sub;
          const int f = __shfl_sync(0xffffffffu, idx_cur, rr);
          const int row = pw * RPW + rr;
          const uint32_t dst = dst0 + row * 128 + (((uint32_t)(c ^ (row & 7))) << 4);
          const bf16* src = src0 + (size_t)f * p.Bpad;
          cp_async16(dst, src);
          cp_async16(dst + C::HH_BYTES, src + 64);
        }
        cp_async_commit();
        if (it >= C::LAG) {
          cp_async_wait<C::LAG>();
          fence_proxy_async_smem();
          __syncwarp();
          if (lane == 0) mbar_arrive(&full[(it - C::LAG) % C::NST]);
        }
      }
    }
#pragma unroll
    for (int r = C::LAG - 1; r >= 0; --r) {
      const int T = it - 1 - r;
      if (T >= 0) {
        if (r == 3) cp_async_wait<3>(); else if (r == 2) cp_async_wait<2>(); else if (r == 1) cp_async_wait<1>(); else cp_async_wait<0>();
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) mbar_arrive(&full[T % C::NST]);
      }
    }
    }
  } else if (warp == 8) {
    // ===================== MMA issuer =====================
    // whole warp waits, one elected lane issues; descriptors are a per-stage base + compile-time offsets (see tc_tail.cu)
    constexpr uint32_t idesc = make_idesc_bf16(C::GV, C::N, /*A (dY) MN-major*/ 1, /*B (H^T) K-major*/ 0);
    const uint64_t bdesc0 = make_sdesc_sw128(sbase, 16, 1024);
    // A = the dY k-block as stored, MN-major: atoms of 64 labels x 128 B rows, or (PAIR) two groups of 32 labels x 64 B rows
    // PADM: one real atom of 32 (16) labels; the atoms after it are read from the bytes that follow (leading offset 2048 / 512)
    const uint64_t adesc0 = C::PAIR ? make_sdesc_sw64(sbase + C::H_BYTES, 4096, 512)
                          : !C::PADM ? make_sdesc_sw128(sbase + C::H_BYTES, 8192, 1024)
                          : C::YROW == 64 ? make_sdesc_sw64(sbase + C::H_BYTES, 2048, 512)
                                          : make_sdesc_sw32(sbase + C::H_BYTES, 512, 256);
    int it = 0;
    for (int i = 0; i < n_my; ++i) {
      const int slot = i & 1;
      mbar_wait(&t_empty[slot], ((i >> 1) & 1) ^ 1);
      tc_fence_after();
      const uint32_t d = tmem_base + slot * C::TS;
      for (int kb = 0; kb < p.NKB; ++kb, ++it) {
        const int st = it % C::NST;
        mbar_wait(&full[st], (it / C::NST) & 1);
        tc_fence_after();
        if (elect_one()) {
          const uint64_t so = (uint64_t)((st * C::STAGE) >> 4);
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const uint64_t ad = adesc0 + so + (uint64_t)(((j >> 2) * C::YH_BYTES + (j & 3) * (16 * C::YROW)) >> 4);
            const uint64_t bd = bdesc0 + so + (uint64_t)(((j >> 2) * C::HH_BYTES + (j & 3) * 32) >> 4);
            umma_f16(d, ad, bd, idesc, (kb | j) ? 1u : 0u);
          }
          umma_commit(&empty[st]);
          if (kb == p.NKB - 1) umma_commit(&t_full[slot]);
        }
        __syncwarp();
      }
    }
  } else if (warp == 9) {
    // ===================== TMA loader of dY k-blocks =====================
    if (lane == 0) {
      int it = 0;
      for (int i = 0; i < n_my; ++i) {
        const int64_t g = group_of(i);
        for (int kb = 0; kb < p.NKB; ++kb, ++it) {
          const int st = it % C::NST;
          mbar_wait(&empty[st], ((it / C::NST) & 1) ^ 1);
          mbar_arrive_expect_tx(&full[st], C::Y_BYTES);
#pragma unroll
          for (int hf = 0; hf < 2; ++hf)
#pragma unroll
            for (int a = 0; a < (C::PADM ? 1 : C::GV / 64 + (C::PAIR ? 1 : 0)); ++a) {
              uint8_t* dst = smem + st * C::STAGE + C::H_BYTES + hf * C::YH_BYTES + a * (C::PAIR ? 4096 : 8192);
              if (C::PAIR) tma_load_3d(dst, &tmY, &full[st], 0, kb * 128 + hf * 64, (int)(2 * g + a));   // group 2v+a (zero-filled past NG)
              else tma_load_3d(dst, &tmY, &full[st], a * 64, kb * 128 + hf * 64, (int)g);
            }
        }
      }
    }
  } else {
    // ===================== epilogue =====================
    const int q = warp;                                         // TMEM lane quadrant
    const uint32_t sbuf0 = sbase + C::OFF_EPI + q * 4096;
    const uint32_t swz = (uint32_t)(lane & 7);
    int nstore = 0;
    // label rows of this warp that are real: M = 64 puts rows 16 q .. 16 q + 15 into lanes 0-15 of quadrant q
    constexpr int RWC = C::RW;
    const int rwv = C::PADM ? max(0, min(RWC, G - RWC * q)) : RWC;
    for (int i = 0; i < n_my; ++i) {
      const int64_t g = group_of(i);
      const int slot = i & 1;
      mbar_wait(&t_full[slot], (i >> 1) & 1);
      tc_fence_after();
      if (rwv == 0) {                     // (PADM) a quadrant past the group's labels: keep step with the others, nothing to do
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&t_empty[slot]);
        continue;
      }
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + slot * C::TS;
      const uint32_t tcol = taddr + (C::PAIR && q >= 2 ? K : 0);   // PAIR: quadrants 2, 3 hold group 2v+1, whose dW sits in columns [K, 2K)
      if constexpr (SGD) {
        // v <- mu v + (g + wd w);  w <- w - lr v   (reading R13).  The accumulator rows ARE the
        // gradient rows, so dW is never written: 32 columns at a time they go through the warp's staging rows (as for a
        // dW store), and the warp then walks them in memory order -- 8 lanes per label row, 16 bytes of momentum and 8 of
        // W each -- so that every global access is a run of whole 128-byte lines and all of a pass's loads are in flight
        // together.  The next group's rows are pulled into L2 meanwhile.
        const int64_t l0 = g * C::GL + q * C::RW;                    // first label row of this warp
        const int64_t l = l0 + lane;
        const bool own = lane < rwv && l < p.L;
        if (i + 1 < n_my) {
          const int64_t ln0 = l0 - (int64_t)gridDim.x * C::GL;      // the next group of this CTA
          constexpr int WL = K * 2 / 128, ML = K * 4 / 128;          // 128-byte lines per row of W / of the momentum
          for (int e = lane; e < rwv * (WL + ML); e += 32) {
            const int r = e / (WL + ML), b = e - r * (WL + ML);
            if (ln0 + r < p.L) {
              const char* a = b < WL ? reinterpret_cast<const char*>(p.W + (ln0 + r) * K) + b * 128
                                     : reinterpret_cast<const char*>(p.mom + (ln0 + r) * K) + (b - WL) * 128;
              asm volatile("prefetch.global.L2 [%0];" ::"l"(a));
            }
          }
        }
#pragma unroll 1
        for (int c = 0; c < K / 32; ++c) {
          uint32_t gq[32];
          tmem_ld32(tcol + c * 32, gq);
          tmem_ld_wait();
          __syncwarp();                                              // the previous pass has read the staging rows
#pragma unroll
          for (int ch = 0; ch < 8; ++ch)
            sts128(sbuf0 + lane * 128 + ((ch ^ swz) << 4), gq[4 * ch], gq[4 * ch + 1], gq[4 * ch + 2], gq[4 * ch + 3]);
          __syncwarp();
          constexpr int NIT = C::RW / 4;                             // (RW rows x 8 chunks of 4 columns) / 32 lanes
#pragma unroll
          for (int h0 = 0; h0 < NIT; h0 += 4) {
            float4 g4[4], m4[4];
            uint2 w2[4];
            bool ok[4];
#pragma unroll
            for (int t = 0; t < 4; ++t) {
              const int e = lane + 32 * (h0 + t), r = e >> 3, c16 = e & 7;
              ok[t] = r < rwv && l0 + r < p.L;
              g4[t] = lds128f(sbuf0 + r * 128 + ((c16 ^ (r & 7)) << 4));
              if (ok[t]) {
                const size_t o = (size_t)(l0 + r) * K + c * 32 + c16 * 4;
                m4[t] = __ldcg(reinterpret_cast<const float4*>(p.mom + o));
                w2[t] = __ldcg(reinterpret_cast<const uint2*>(p.W + o));
              }
            }
#pragma unroll
            for (int t = 0; t < 4; ++t) {
              if (!ok[t]) continue;
              const int e = lane + 32 * (h0 + t), r = e >> 3, c16 = e & 7;
              const size_t o = (size_t)(l0 + r) * K + c * 32 + c16 * 4;
              const float w0 = __uint_as_float(w2[t].x << 16), w1 = __uint_as_float(w2[t].x & 0xffff0000u);
              const float w2f = __uint_as_float(w2[t].y << 16), w3 = __uint_as_float(w2[t].y & 0xffff0000u);
              float4 v;
              v.x = fmaf(p.mu, m4[t].x, fmaf(p.wd, w0, g4[t].x));
              v.y = fmaf(p.mu, m4[t].y, fmaf(p.wd, w1, g4[t].y));
              v.z = fmaf(p.mu, m4[t].z, fmaf(p.wd, w2f, g4[t].z));
              v.w = fmaf(p.mu, m4[t].w, fmaf(p.wd, w3, g4[t].w));
              *reinterpret_cast<float4*>(p.mom + o) = v;
              *reinterpret_cast<uint2*>(p.W + o) = make_uint2(dw_pack_bf16x2(fmaf(-p.lr, v.x, w0), fmaf(-p.lr, v.y, w1)),
                                                              dw_pack_bf16x2(fmaf(-p.lr, v.z, w2f), fmaf(-p.lr, v.w, w3)));
            }
          }
        }
        if (p.bias) {       // bias: the same step without weight decay; db is accumulator column KV
          const uint32_t v = tmem_ld1(taddr + C::KV);
          tmem_ld_wait();
          if (own) {
            const float vb = fmaf(p.mu, p.bmom[l], __uint_as_float(v));
            p.bmom[l] = vb;
            p.bias[l] = fmaf(-p.lr, vb, p.bias[l]);
          }
        }
      } else if (p.write_dw) {
#pragma unroll 1
        for (int c = 0; c < C::NBOX; ++c, ++nstore) {
          uint32_t out[32];
          if (F32) {
            tmem_ld32(tcol + c * 32, out);
            tmem_ld_wait();
          } else {
            uint32_t v0[32], v1[32];
            tmem_ld32(tcol + c * 64, v0);
            tmem_ld32(tcol + c * 64 + 32, v1);
            tmem_ld_wait();
#pragma unroll
            for (int j = 0; j < 16; ++j) {
              out[j] = dw_pack_bf16x2(__uint_as_float(v0[2 * j]), __uint_as_float(v0[2 * j + 1]));
              out[16 + j] = dw_pack_bf16x2(__uint_as_float(v1[2 * j]), __uint_as_float(v1[2 * j + 1]));
            }
          }
          const uint32_t sbuf = sbuf0;
          if (lane == 0) bulk_wait_read<0>();                   // the previous store has read the staging rows
          __syncwarp();
#pragma unroll
          for (int ch = 0; ch < 8; ++ch)
            sts128(sbuf + lane * 128 + ((ch ^ swz) << 4), out[4 * ch], out[4 * ch + 1], out[4 * ch + 2], out[4 * ch + 3]);
          fence_proxy_async_smem();
          __syncwarp();
          if (lane == 0) {
            tma_store_2d(&tmO, smem + C::OFF_EPI + q * 4096, c * (F32 ? 32 : 64), (int)(g * C::GL + q * C::RW));
            bulk_commit();
          }
        }
      }
      if (!SGD && p.dbias) {
        const uint32_t v = tmem_ld1(taddr + C::KV);
        tmem_ld_wait();
        const int64_t l = g * C::GL + q * C::RW + lane;
        if (lane < rwv && l < p.L) p.dbias[l] = __uint_as_float(v);
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&t_empty[slot]);
    }
    if (lane == 0) bulk_wait<0>();
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 8) { tc_fence_after(); tmem_dealloc<2 * C::TS>(tmem_base); }
}

struct DwSgd { void* W; float* mom; float* bias; float* bmom; float lr, mu, wd; };

template <int G, int K, bool F32, bool SGD = false>
static int launch_dw(TcTailState* s, const TailShape& sh, const void* Xt, const int32_t* idx, const void* dY, void* dW,
                     float* dbias, cudaStream_t st, const DwSgd* sgd = nullptr) {
  using C = DwCfg<G, K, F32, SGD>;
  static_assert(C::SMEM <= 232448, "shared memory budget");
  CUtensorMap tmY, tmO;
  {
    const uint64_t dims[3] = {(uint64_t)G, (uint64_t)sh.B, (uint64_t)sh.NG};
    const uint64_t str[2] = {(uint64_t)G * 2, (uint64_t)sh.B * G * 2};
    // G = 8: a box of 16 labels over a row of 8 -- the TMA fills labels 8-15 with zeros
    const uint32_t box[3] = {(uint32_t)std::min(std::max(G, 16), 64), 64, 1};
    int rc = encode_tmap(&tmY, 2, dY, 3, dims, str, box, C::PADM ? C::YROW : (G >= 64 ? 128 : 64));
    if (rc) return rc;
  }
  if (dW) {
    const int es = F32 ? 4 : 2;
    const uint64_t dims[2] = {(uint64_t)K, (uint64_t)sh.L};
    const uint64_t str[1] = {(uint64_t)K * es};
    const uint32_t box[2] = {(uint32_t)(128 / es), (uint32_t)std::min(C::RW, G)};
    int rc = encode_tmap(&tmO, es, dW, 2, dims, str, box, 128);
    if (rc) return rc;
  } else {
    tmO = tmY;
  }
  DwParams p;
  memset(&p, 0, sizeof(p));
  p.Xt = (const bf16*)Xt; p.idx = idx; p.dbias = dbias; p.write_dw = dW ? 1 : 0;
  if (SGD) { p.W = (bf16*)sgd->W; p.mom = sgd->mom; p.bias = sgd->bias; p.bmom = sgd->bmom; p.lr = sgd->lr; p.mu = sgd->mu; p.wd = sgd->wd; }
  p.B = sh.B; p.Bpad = sh.Bpad; p.NKB = ceil_div(sh.B, 128); p.L = sh.L; p.NG = sh.NG;
  const int grid = (int)std::min<int64_t>(C::PAIR ? (sh.NG + 1) / 2 : sh.NG, s->num_sms);
  HASTE_CUDA_TRY(cudaFuncSetAttribute(tc_dw_kernel<G, K, F32, SGD>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM));
  HASTE_CUDA_TRY(launch_pdl(tc_dw_kernel<G, K, F32, SGD>, dim3(grid), dim3(320), C::SMEM, st, tmY, tmO, p));
  return HASTE_OK;
}

int tc_tail_dw(TcTailState* s, const TailShape& sh, const void* Xt, const int32_t* idx, const void* dY, void* dW,
               float* dbias, cudaStream_t st, int* n_launches) {
  *n_launches = 1;
  const bool f32 = s->cfg.dw_dtype == HASTE_F32;
#define HASTE_DW(G_, K_)                                                                     \
  if (sh.G == G_ && sh.K == K_)                                                              \
    return f32 ? launch_dw<G_, K_, true>(s, sh, Xt, idx, dY, dW, dbias, st)                  \
               : launch_dw<G_, K_, false>(s, sh, Xt, idx, dY, dW, dbias, st)
  HASTE_DW(64, 128); HASTE_DW(64, 64); HASTE_DW(128, 64); HASTE_DW(128, 128); HASTE_DW(32, 64); HASTE_DW(32, 128);
  HASTE_DW(16, 64); HASTE_DW(16, 128); HASTE_DW(8, 64); HASTE_DW(8, 128);
#undef HASTE_DW
  return HASTE_ERR_UNSUPPORTED;
}

// the same contraction with the SGD-momentum step of the output layer as its epilogue: W [L,K] (bf16) and
// mom [L,K] (fp32) updated in place, bias / bmom [L] too if given; the gradient is never written
int tc_tail_dw_sgd(TcTailState* s, const TailShape& sh, const void* Xt, const int32_t* idx, const void* dY, void* W, float* mom,
                   float* bias, float* bmom, float lr, float mu, float wd, cudaStream_t st, int* n_launches) {
  *n_launches = 1;
  const DwSgd sgd = {W, mom, bias, bmom, lr, mu, wd};
#define HASTE_DWS(G_, K_) \
  if (sh.G == G_ && sh.K == K_) return launch_dw<G_, K_, true, true>(s, sh, Xt, idx, dY, nullptr, nullptr, st, &sgd)
  HASTE_DWS(64, 128); HASTE_DWS(64, 64); HASTE_DWS(128, 64); HASTE_DWS(128, 128); HASTE_DWS(32, 64); HASTE_DWS(32, 128);
  HASTE_DWS(16, 64); HASTE_DWS(16, 128); HASTE_DWS(8, 64); HASTE_DWS(8, 128);
#undef HASTE_DWS
  return HASTE_ERR_UNSUPPORTED;
}

}  // namespace haste
