// tc_fused.cu -- forward + fused BCE + weight gradient of the HASTE sparse tail in ONE kernel (sm_100a; bf16 in, fp32
// accumulate): the first slice of the single-pass step ("gather-once").
//
//   per group g, batch tile t:   Z = H_t W_g^T,  dY_t = s (sigma(Z + b) - Y),  loss += BCE      (as tc_tail.cu)
//                                dW_g += dY_t^T H_t,   db_g += dY_t^T 1                        (as tc_dw.cu)
//
// Why: run one after the other, the forward writes dY (the [B, L] gradient of the logits, 80 % of the step's bytes) and
// the dW kernel reads all of it back and gathers H = X[:, idx_g] a second time.  Here the gathered tile H_t and the dY
// tile the epilogue has just produced are BOTH still in shared memory when the weight-gradient MMA runs:
//   * the H image [2 m-blocks][K + 16 rows][128 B] is the forward's MN-major A operand (M = batch) and, read through a
//     second descriptor, the weight gradient's K-major B operand (N = slots, contraction over the batch); its last rows
//     are ones, so accumulator column K is db (as in tc_dw.cu);
//   * the dY staging tile [128 batch rows][128 B = 64 labels] that the epilogue fills for its TMA store is, as it lies,
//     the weight gradient's MN-major A operand (M = labels).
// dY is still written (the dX kernel needs it) but never read back by this kernel, and X^T is gathered once: 1.0 GB of
// DRAM traffic for the two steps instead of 1.69 GB at config 3.
//
// CTA = stripe of groups x ALL batch tiles (B <= 512: up to four tiles of 128 rows), so a group's dW has one owner and
// needs no reduction across CTAs.  Epilogue set t (4 warps) owns batch tile t for the whole kernel (a thread owns one
// batch row, as in tc_tail.cu).  The issuing warp interleaves: forward MMAs of tile T, then the weight-gradient MMAs of
// tile T - 1 (whose dY the epilogue has staged meanwhile) into a TMEM accumulator D_w [64 labels x K + 8] that lives
// across the group's tiles, double buffered across groups; the set whose turn it is writes dW_g / db_g a group later.
#include <algorithm>
#include <cstring>

#include "tc_common.cuh"
#include "tc_epilogue.cuh"
#include "tc_kernels.h"

namespace haste {
using namespace tc;

struct FusedParams {
  const bf16* Xt;          // [d][Bpad]
  const int32_t* idx;      // [NG][K]
  const float* bias;       // [L] or null
  const int32_t* rowptr;   // [B+1] or null
  const int32_t* col;      // [nnz]
  float* partials;         // [1024] unscaled loss partials + ticket (finalize_loss_last_cta), or null
  float* loss;             // device scalar
  void* dW;                // [L][K] bf16 or fp32, or null
  float* dbias;            // [L] or null
  int B, Bpad, NT;         // NT batch tiles of 128 (<= 4)
  int64_t L, NG, label_offset;
  float s;
};

template <int G, int K> struct FusedCfg {
  static_assert(G == 64, "the weight-gradient accumulator is one M = 64 MMA tile");
  static constexpr int NSET = 4;                                // epilogue sets = batch tiles
  static constexpr int HS = 3;                                  // H stages
  static constexpr int LAG = 1;                                 // producer completion lag
  static constexpr int HROWS = K + 16;                          // rows of one m-block of the H image: K slots + ones
  static constexpr int HH_BYTES = HROWS * 128;                  // one m-block (64 batch columns)
  static constexpr int H_BYTES = 2 * HH_BYTES;
  static constexpr int W_BYTES = G * K * 2;                     // [K/64 k-blocks][G rows][128 B]
  static constexpr int WS = 2;
  static constexpr int ST_BYTES = 128 * 64 * 2;                 // one dY staging tile per set: [128 rows][128 B]
  static constexpr int NW = K + 8;                              // weight-gradient MMA N: slots + the ones columns
  static constexpr int DW_COLS = (NW + 15) / 16 * 16;           // TMEM columns per D_w buffer
  static constexpr int T_FWD0 = 2 * DW_COLS;                    // first column of the forward's accumulator ring
  static constexpr int NSLOT = (512 - T_FWD0) / G >= 8 ? 8 : (512 - T_FWD0) / G;   // K = 64: 5, K = 128: 3
  static_assert(NSLOT >= 3, "forward accumulator ring too short");
  // "accumulator ready" barriers.  A parity wait only tells the two most recent phases of a barrier apart, and a set waits
  // for tile T after tile T - NSET: with one barrier per slot and fewer slots than sets (K = 128: 3 < 4) the slot's
  // previous tile T - NSLOT belongs to another set and may not have completed yet -- the wait for T's phase would then
  // succeed at once on the phase before it.  A barrier ring twice as long (tile T: slot T mod NSLOT, barrier T mod NTF)
  // puts the barrier's previous tile T - NTF behind T - NSET, which this set has already seen complete.
  static constexpr int NTF = NSLOT < NSET ? 2 * NSLOT : NSLOT;
  static constexpr int OFF_H = 0;
  static constexpr int OFF_W = OFF_H + HS * H_BYTES;
  static constexpr int OFF_ST = OFF_W + WS * W_BYTES;
  static constexpr int OFF_BIAS = OFF_ST + NSET * ST_BYTES;     // [16 warps][G] fp32
  static constexpr int OFF_BAR = OFF_BIAS + 4 * NSET * G * 4;
  static constexpr int NBAR = 2 * HS + 2 * WS + NTF + NSLOT + 2 * NSET + 4;
  static constexpr int OFF_MISC = OFF_BAR + NBAR * 8;
  static constexpr int SMEM = OFF_MISC + 128 + 1024;
  static constexpr int THREADS = (4 * NSET + 6) * 32;
};

__device__ __forceinline__ uint32_t fz_tmem_ld1(uint32_t taddr) {
  uint32_t v;
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(v) : "r"(taddr) : "memory");
  return v;
}

template <int G, int K, bool F32>
__global__ void __launch_bounds__(FusedCfg<G, K>::THREADS, 1)
tc_fused_kernel(const __grid_constant__ CUtensorMap tmW, const __grid_constant__ CUtensorMap tmY, const FusedParams p) {
  using C = FusedCfg<G, K>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const uint32_t sbase = smem_u32(smem);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::OFF_BAR);
  uint64_t* h_full = bars;                       // [HS]    count 4 (producer warps)
  uint64_t* h_empty = bars + C::HS;              // [HS]    count 1 (commit after the tile's weight-gradient MMAs)
  uint64_t* w_full = bars + 2 * C::HS;           // [WS]    count 1 + tx
  uint64_t* w_empty = w_full + C::WS;            // [WS]    count 1 (commit)
  uint64_t* t_full = w_empty + C::WS;            // [NTF]   count 1 (commit after the tile's forward MMAs)
  uint64_t* t_empty = t_full + C::NTF;           // [NSLOT] count 4 (epilogue warps of the tile's set)
  uint64_t* s_full = t_empty + C::NSLOT;         // [NSET]  count 4: the set's dY tile is staged (A operand of the weight gradient)
  uint64_t* s_empty = s_full + C::NSET;          // [NSET]  count 1 (commit: the weight-gradient MMAs have read it)
  uint64_t* dw_full = s_empty + C::NSET;         // [2]     count 1 (commit after the group's last weight-gradient MMA)
  uint64_t* dw_empty = dw_full + 2;              // [2]     count 4 (the set that wrote dW_g out)
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + C::OFF_MISC);
  float* loss_red = reinterpret_cast<float*>(smem + C::OFF_MISC + 16);   // [4 * NSET]

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int stripe = blockIdx.x, S = gridDim.x, NT = p.NT;
  const int ngl = p.NG > stripe ? (int)((p.NG - stripe + S - 1) / S) : 0;   // groups of this CTA
  const int total = ngl * NT;                                               // tiles: T = gl * NT + t

  if (threadIdx.x == 0) {
    for (int i = 0; i < C::HS; ++i) { mbar_init(&h_full[i], 4); mbar_init(&h_empty[i], 1); }
    for (int i = 0; i < C::WS; ++i) { mbar_init(&w_full[i], 1); mbar_init(&w_empty[i], 1); }
    for (int i = 0; i < C::NTF; ++i) mbar_init(&t_full[i], 1);
    for (int i = 0; i < C::NSLOT; ++i) mbar_init(&t_empty[i], 4);
    for (int i = 0; i < C::NSET; ++i) { mbar_init(&s_full[i], 4); mbar_init(&s_empty[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&dw_full[i], 1); mbar_init(&dw_empty[i], 4); }
    fence_barrier_init();
  }
  // rows K .. K+15 of both m-blocks of every H stage: bf16 1.0 (swizzling permutes equal chunks: write linearly)
  for (int e = threadIdx.x; e < C::HS * 2 * 16 * 8; e += blockDim.x) {
    const int st = e / 256, hf = (e >> 7) & 1, r = e % 128;
    sts128(sbase + C::OFF_H + st * C::H_BYTES + hf * C::HH_BYTES + K * 128 + r * 16, 0x3F803F80u, 0x3F803F80u, 0x3F803F80u, 0x3F803F80u);
  }
  fence_proxy_async_smem();
  constexpr int EW = 4 * C::NSET;                                          // epilogue warps
  if (warp == EW + 5 && lane == 0) { tma_prefetch_desc(&tmW); tma_prefetch_desc(&tmY); }
  if (warp == EW + 4) tmem_alloc<512>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  pdl_wait();       // nothing above touches global memory (common.cuh, PDL)
  pdl_trigger();
  const uint32_t tmem_base = *tmem_slot;

  if (warp >= EW && warp < EW + 4) {
    // ===================== gather producers (as tc_tail.cu; the image has K + 16 rows per m-block) =====================
    const int pw = warp - EW;
    constexpr int RPW = K / 4;
    const int sub = lane >> 4, c = lane & 15;
    const uint32_t dst_lane = (uint32_t)((c >> 3) * C::HH_BYTES + (((c & 7)) << 4));
    const int32_t* idx_ptr = p.idx + (int64_t)stripe * K + pw * RPW + lane;
    const int64_t idx_step = (int64_t)S * K;
    int idx_cur = 0, idx_n1 = 0, idx_n2 = 0;
    if (lane < RPW && ngl > 0) {
      idx_n1 = __ldg(idx_ptr);
      if (ngl > 1) idx_n2 = __ldg(idx_ptr + idx_step);
    }
    int gl = 0, t = 0;
    for (int T = 0; T < total; ++T) {
      if (t == 0) {
        idx_cur = idx_n1; idx_n1 = idx_n2;
        if (lane < RPW && gl + 2 < ngl) idx_n2 = __ldg(idx_ptr + (gl + 2) * idx_step);
      }
      const int hs = T % C::HS;
      mbar_wait(&h_empty[hs], ((T / C::HS) & 1) ^ 1);
      const uint32_t dst0 = sbase + C::OFF_H + hs * C::H_BYTES + dst_lane;
      const bf16* src0 = p.Xt + t * 128 + c * 8;
#pragma unroll
      for (int i = 0; i < RPW / 2; ++i) {
        const int kk = 2 * i + sub;
        const int f = __shfl_sync(0xffffffffu, idx_cur, kk);
        const int k = pw * RPW + kk;
        const uint32_t dst = (dst0 + k * 128) ^ ((uint32_t)(k & 7) << 4);
        cp_async16(dst, src0 + (size_t)f * p.Bpad);
      }
      cp_async_commit();
      if (T >= C::LAG) {
        cp_async_wait<C::LAG>();
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) mbar_arrive(&h_full[(T - C::LAG) % C::HS]);
      }
      if (++t == NT) { t = 0; ++gl; }
    }
    if (total > 0) {
      cp_async_wait<0>();
      fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) mbar_arrive(&h_full[(total - 1) % C::HS]);
    }
  } else if (warp == EW + 4) {
    // ===================== MMA issuer: forward of tile T, then the weight gradient of tile T - 1 =====================
    constexpr uint32_t idesc_f = make_idesc_bf16(128, G, /*A (H) MN-major*/ 1, /*B (W) K-major*/ 0);
    constexpr uint32_t idesc_w = make_idesc_bf16(64, C::NW, /*A (dY tile) MN-major*/ 1, /*B (H) K-major*/ 0);
    const uint64_t fa0 = make_sdesc_sw128(sbase + C::OFF_H, C::HH_BYTES, 1024);   // leading offset: the second 64 batch columns
    const uint64_t fb0 = make_sdesc_sw128(sbase + C::OFF_W, 16, 1024);
    const uint64_t wa0 = make_sdesc_sw128(sbase + C::OFF_ST, 8192, 1024);         // [128 batch rows][64 labels], as stored
    const uint64_t wb0 = make_sdesc_sw128(sbase + C::OFF_H, 16, 1024);            // rows = slots (+ ones), 64 batch columns per m-block
    int gl = 0, t = 0, gld = 0, td = 0;
    for (int T = 0; T <= total; ++T) {
      if (T < total) {
        const int ws = gl % C::WS, hs = T % C::HS, slot = T % C::NSLOT;
        if (t == 0) mbar_wait(&w_full[ws], (gl / C::WS) & 1);
        mbar_wait(&h_full[hs], (T / C::HS) & 1);
        mbar_wait(&t_empty[slot], ((T / C::NSLOT) & 1) ^ 1);
        tc_fence_after();
        if (elect_one()) {
          const uint64_t ad0 = fa0 + (uint64_t)((hs * C::H_BYTES) >> 4);
          const uint64_t bd0 = fb0 + (uint64_t)((ws * C::W_BYTES) >> 4);
          const uint32_t d = tmem_base + C::T_FWD0 + slot * G;
#pragma unroll
          for (int j = 0; j < K / 16; ++j)
            umma_f16(d, ad0 + (uint64_t)((j * 2048) >> 4), bd0 + (uint64_t)(((j >> 2) * (G * 128) + (j & 3) * 32) >> 4), idesc_f,
                     j > 0 ? 1u : 0u);
          umma_commit(&t_full[T % C::NTF]);
        }
        __syncwarp();
        if (++t == NT) { t = 0; ++gl; }
      }
      if (T >= 1) {
        const int Td = T - 1;
        const int hs = Td % C::HS, buf = gld & 1;
        if (td == 0) mbar_wait(&dw_empty[buf], ((gld >> 1) & 1) ^ 1);      // D_w buffer written out (two groups ago)
        mbar_wait(&s_full[td], gld & 1);                                    // the epilogue has staged this tile's dY
        tc_fence_after();
        if (elect_one()) {
          const uint64_t ad0 = wa0 + (uint64_t)((td * C::ST_BYTES) >> 4);
          const uint64_t bd0 = wb0 + (uint64_t)((hs * C::H_BYTES) >> 4);
          const uint32_t d = tmem_base + buf * C::DW_COLS;
#pragma unroll
          for (int j = 0; j < 8; ++j)
            umma_f16(d, ad0 + (uint64_t)((j * 2048) >> 4), bd0 + (uint64_t)(((j >> 2) * C::HH_BYTES + (j & 3) * 32) >> 4), idesc_w,
                     (td | j) ? 1u : 0u);
          umma_commit(&h_empty[hs]);                    // (also covers the tile's forward MMAs)
          umma_commit(&s_empty[td]);
          if (td == NT - 1) { umma_commit(&dw_full[buf]); umma_commit(&w_empty[gld % C::WS]); }
        }
        __syncwarp();
        if (++td == NT) { td = 0; ++gld; }
      }
    }
  } else if (warp == EW + 5) {
    // ===================== W loader =====================
    if (lane == 0) {
      for (int gl = 0; gl < ngl; ++gl) {
        const int ws = gl % C::WS;
        const int64_t g = stripe + (int64_t)gl * S;
        mbar_wait(&w_empty[ws], ((gl / C::WS) & 1) ^ 1);
        mbar_arrive_expect_tx(&w_full[ws], C::W_BYTES);
#pragma unroll
        for (int kb = 0; kb < K / 64; ++kb)
          tma_load_2d(smem + C::OFF_W + ws * C::W_BYTES + kb * (G * 128), &tmW, &w_full[ws], kb * 64, (int)(g * G));
      }
    }
  } else if ((warp >> 2) < NT) {
    // ===================== epilogue: set = batch tile, q = TMEM lane quadrant, lane = batch row =====================
    const int set = warp >> 2, q = warp & 3;
    const int row = q * 32 + lane;
    const int b = set * 128 + row;
    const bool valid_row = b < p.B;
    int pc = 0, pe = 0;
    int nxt = 0x7fffffff;
    if (valid_row && p.rowptr) {
      pc = __ldg(p.rowptr + b); pe = __ldg(p.rowptr + b + 1);
      if (pc < pe) nxt = __ldg(p.col + pc);
    }
    float loss_local = 0.f;
    const float hs = 0.5f * p.s;
    constexpr int NCH = G / 32;
    const uint32_t stage_w = sbase + C::OFF_ST + set * C::ST_BYTES + q * 32 * 128;
    const uint32_t stage_row = stage_w + lane * 128;
    const uint32_t swz = (uint32_t)(lane & 7);
    const uint32_t sbias_w = sbase + C::OFF_BIAS + warp * G * 4;

    // D_w of group gd (this CTA's gd-th) -> dW rows and db: M = 64 puts label rows 16 q .. 16 q + 15 into lanes 0-15
    auto dw_out = [&](int gd) {
      const int buf = gd & 1;
      const int64_t g = stripe + (int64_t)gd * S;
      mbar_wait(&dw_full[buf], (gd >> 1) & 1);
      tc_fence_after();
      const uint32_t tw = tmem_base + ((uint32_t)(q * 32) << 16) + buf * C::DW_COLS;
      const int64_t l = g * G + q * 16 + lane;
      const bool own = lane < 16 && l < p.L;
      if (p.dW) {
#pragma unroll 1
        for (int c = 0; c < K / 32; ++c) {
          uint32_t v[32];
          tmem_ld32(tw + c * 32, v);
          tmem_ld_wait();
          if (own) {
            if (F32) {
              float4* o = reinterpret_cast<float4*>(reinterpret_cast<float*>(p.dW) + l * K + c * 32);
#pragma unroll
              for (int i = 0; i < 8; ++i)
                o[i] = make_float4(__uint_as_float(v[4 * i]), __uint_as_float(v[4 * i + 1]), __uint_as_float(v[4 * i + 2]), __uint_as_float(v[4 * i + 3]));
            } else {
              uint4* o = reinterpret_cast<uint4*>(reinterpret_cast<bf16*>(p.dW) + l * K + c * 32);
#pragma unroll
              for (int i = 0; i < 4; ++i)
                o[i] = make_uint4(pack_bf16x2(__uint_as_float(v[8 * i]), __uint_as_float(v[8 * i + 1])),
                                  pack_bf16x2(__uint_as_float(v[8 * i + 2]), __uint_as_float(v[8 * i + 3])),
                                  pack_bf16x2(__uint_as_float(v[8 * i + 4]), __uint_as_float(v[8 * i + 5])),
                                  pack_bf16x2(__uint_as_float(v[8 * i + 6]), __uint_as_float(v[8 * i + 7])));
            }
          }
        }
      }
      if (p.dbias) {
        const uint32_t v = fz_tmem_ld1(tw + K);
        tmem_ld_wait();
        if (own) p.dbias[l] = __uint_as_float(v);
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&dw_empty[buf]);
    };

    int gl = 0;
    for (int T = set; T < total; T += NT, ++gl) {
      const int64_t g = stripe + (int64_t)gl * S;
      const int nl = (int)min((int64_t)G, p.L - g * G);
      const int slot = T % C::NSLOT;
      if (p.bias) {
#pragma unroll
        for (int i = 0; i < NCH; ++i) {
          const int l = i * 32 + lane;
          sts32(sbias_w + l * 4, __float_as_uint(l < nl ? __ldg(p.bias + g * G + l) : 0.f));
        }
      }
      __syncwarp();
      const int64_t glo64 = p.label_offset + g * G;
      const int glo = (int)min(glo64, (int64_t)0x7fffffff), ghi = (int)min(glo64 + nl, (int64_t)0x7fffffff);
      uint32_t ym[NCH];
#pragma unroll
      for (int i = 0; i < NCH; ++i) ym[i] = 0;
      while (nxt < ghi) {
        if (nxt >= glo) {
          const int o = nxt - glo;
#pragma unroll
          for (int i = 0; i < NCH; ++i) if ((o >> 5) == i) ym[i] |= 1u << (o & 31);
        }
        ++pc;
        nxt = pc < pe ? __ldg(p.col + pc) : 0x7fffffff;
      }
      uint32_t anyy = 0;
#pragma unroll
      for (int i = 0; i < NCH; ++i) anyy |= ym[i];
      const bool slow = __any_sync(0xffffffffu, anyy != 0) || nl < G;

      mbar_wait(&t_full[T % C::NTF], (T / C::NTF) & 1);
      tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + C::T_FWD0 + slot * G;
      float R[4] = {0.f, 0.f, 0.f, 0.f}, P[4] = {1.f, 1.f, 1.f, 1.f};
      uint32_t v[32];
#pragma unroll
      for (int sc = 0; sc < NCH; ++sc) {
        uint32_t ymsc = ym[0];
#pragma unroll
        for (int i = 1; i < NCH; ++i) if (sc == i) ymsc = ym[i];
        tmem_ld32(taddr + sc * 32, v);
        tmem_ld_wait();
        if (sc + 1 == NCH) {
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(&t_empty[slot]);
        }
        uint32_t out[16];
        const int nvalid = nl - sc * 32;
        const uint32_t sb = sbias_w + sc * 128;
        if (slow) {
          if (p.bias) epi32<true, true>(v, sb, ymsc, nvalid, p.s, hs, R, P, out, nullptr);
          else epi32<true, false>(v, sb, ymsc, nvalid, p.s, hs, R, P, out, nullptr);
        } else {
          if (p.bias) epi32<false, true>(v, sb, 0u, 32, p.s, hs, R, P, out, nullptr);
          else epi32<false, false>(v, sb, 0u, 32, p.s, hs, R, P, out, nullptr);
        }
        if (sc & 1) {
          loss_local += (R[0] + R[1]) + (R[2] + R[3]) - 0.69314718056f * __log2f((P[0] * P[1]) * (P[2] * P[3]));
#pragma unroll
          for (int i = 0; i < 4; ++i) { R[i] = 0.f; P[i] = 1.f; }
        }
        if (!valid_row) {        // rows past the batch: the TMA store clips them, the weight gradient must see zeros (db)
#pragma unroll
          for (int i = 0; i < 16; ++i) out[i] = 0u;
        }
        if (sc == 0) {
          // the staging rows are free again: the TMA store of the set's previous tile has read them, and so have the
          // weight-gradient MMAs of that tile
          if (lane == 0) bulk_wait_read<0>();
          mbar_wait(&s_empty[set], (gl & 1) ^ 1);
          __syncwarp();
        }
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const uint32_t ch = (uint32_t)((sc & 1) * 4 + i) ^ swz;
          sts128(stage_row + ch * 16, out[4 * i], out[4 * i + 1], out[4 * i + 2], out[4 * i + 3]);
        }
        if (sc == NCH - 1) {
          fence_proxy_async_smem();
          __syncwarp();
          if (lane == 0) {
            tma_store_3d(&tmY, smem + C::OFF_ST + set * C::ST_BYTES + q * 32 * 128, 0, set * 128 + q * 32, (int)g);
            bulk_commit();
            mbar_arrive(&s_full[set]);
          }
        }
      }
      // the weight gradient of the group before, if it is this set's turn: its MMAs finished a tile ago
      if (gl >= 1 && (gl - 1) % NT == set) dw_out(gl - 1);
    }
    if (ngl >= 1 && (ngl - 1) % NT == set) dw_out(ngl - 1);
    if (lane == 0) bulk_wait<0>();
    if (!valid_row) loss_local = 0.f;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) loss_local += __shfl_xor_sync(0xffffffffu, loss_local, o);
    if (lane == 0) loss_red[warp] = loss_local;
  } else {
    if (lane == 0) loss_red[warp] = 0.f;      // sets without a batch tile
  }

  tc_fence_before();
  __syncthreads();
  if (warp == EW + 4) { tc_fence_after(); tmem_dealloc<512>(tmem_base); }
  if (p.partials) {
    float t = 0.f;
    if (threadIdx.x == 0) {
#pragma unroll
      for (int i = 0; i < EW; ++i) t += loss_red[i];
    }
    finalize_loss_last_cta(p.partials, t, p.s, p.loss);
  }
}

template <int G, int K, bool F32>
static int launch_fused(TcTailState* s, const TailShape& sh, const void* Xt, const int32_t* idx, const void* W, const float* bias,
                        const int32_t* rowptr, const int32_t* col, float* partials, float* loss, void* dY, void* dW, float* dbias,
                        cudaStream_t st) {
  using C = FusedCfg<G, K>;
  static_assert(C::SMEM <= 232448, "shared memory budget");
  CUtensorMap tmW, tmY;
  {
    const uint64_t dims[2] = {(uint64_t)K, (uint64_t)sh.L};
    const uint64_t str[1] = {(uint64_t)K * 2};
    const uint32_t box[2] = {64, (uint32_t)G};
    int rc = encode_tmap(&tmW, 2, W, 2, dims, str, box, 128);
    if (rc) return rc;
  }
  {
    const uint64_t dims[3] = {(uint64_t)G, (uint64_t)sh.B, (uint64_t)sh.NG};
    const uint64_t str[2] = {(uint64_t)G * 2, (uint64_t)sh.B * G * 2};
    const uint32_t box[3] = {64, 32, 1};
    int rc = encode_tmap(&tmY, 2, dY, 3, dims, str, box, 128);
    if (rc) return rc;
  }
  FusedParams p;
  memset(&p, 0, sizeof(p));
  p.Xt = (const bf16*)Xt; p.idx = idx; p.bias = bias; p.rowptr = rowptr; p.col = col; p.partials = partials; p.loss = loss;
  p.dW = dW; p.dbias = dbias;
  p.B = sh.B; p.Bpad = sh.Bpad; p.NT = ceil_div(sh.B, 128);
  p.L = sh.L; p.NG = sh.NG; p.label_offset = sh.label_offset; p.s = sh.s;
  const int grid = (int)std::min<int64_t>(sh.NG, s->num_sms);
  HASTE_CUDA_TRY(cudaFuncSetAttribute(tc_fused_kernel<G, K, F32>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM));
  HASTE_CUDA_TRY(launch_pdl(tc_fused_kernel<G, K, F32>, dim3(grid), dim3(C::THREADS), C::SMEM, st, tmW, tmY, p));
  return HASTE_OK;
}

// forward + loss + dY + dW + db in one launch (see the head of this file).  HASTE_ERR_UNSUPPORTED (nothing launched) unless
// G = 64, K in {64, 128} and B <= 512; the caller then runs the two kernels one after the other.
int tc_tail_forward_dw(TcTailState* s, const TailShape& sh, const void* Xt, const int32_t* idx, const void* W, const float* bias,
                       const int32_t* rowptr, const int32_t* col, float* loss_partials, float* loss, void* dY, void* dW,
                       float* dbias, cudaStream_t st, int* n_launches) {
  *n_launches = 1;
  if (sh.G != 64 || sh.B > 512 || !dY) return HASTE_ERR_UNSUPPORTED;
  const bool f32 = s->cfg.dw_dtype == HASTE_F32;
#define HASTE_FZ(K_)                                                                                                     \
  if (sh.K == K_)                                                                                                        \
    return f32 ? launch_fused<64, K_, true>(s, sh, Xt, idx, W, bias, rowptr, col, loss_partials, loss, dY, dW, dbias, st) \
               : launch_fused<64, K_, false>(s, sh, Xt, idx, W, bias, rowptr, col, loss_partials, loss, dY, dW, dbias, st)
  HASTE_FZ(128); HASTE_FZ(64);
#undef HASTE_FZ
  return HASTE_ERR_UNSUPPORTED;
}

}  // namespace haste
