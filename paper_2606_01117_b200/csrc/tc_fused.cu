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
//   * the dY tile [128 batch rows][128 B = 64 labels] that the epilogue writes to shared memory is, as it lies, the
//     weight gradient's MN-major A operand (M = labels).
// dY is still written to HBM (by TMA from that same shared-memory tile; the dX kernel needs it) but never read back by this kernel, and X^T is gathered once: 1.0 GB
// of DRAM traffic for the two steps instead of 1.69 GB at config 3.
//
// CTA = stripe of groups x ALL batch tiles (B <= 512: up to four tiles of 128 rows), so a group's dW has one owner and
// needs no reduction across CTAs.  Tiles are numbered T = group * NT + batch tile.
// What bounds this kernel is how long an H stage lives: from its gather through the forward MMAs and the WHOLE epilogue of
// the tile to the weight-gradient MMAs that read it last.  So a tile's epilogue is made short: EIGHT warps per tile (TMEM
// lane quadrant x 32-label half; a thread does one batch row x 32 labels), two tiles in flight (tile T belongs to the
// warps of parity T & 1), and TWO issuing warps, one per queue: forward MMAs of the next gathered tile; weight-gradient
// MMAs (and the dY store) of the next tile whose dY is in shared memory.  The weight-gradient accumulator
// D_w [64 labels x K + 8] lives in TMEM across a group's tiles, one buffer per group parity, and is written out (dW_g,
// db_g) by the warps of that parity a few tiles later.
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
  bf16* dY;                // [NG][B][64]
  void* dW;                // [L][K] bf16 or fp32, or null
  float* dbias;            // [L] or null
  int B, Bpad, NT;         // NT batch tiles of 128 (<= 4)
  int64_t L, NG, label_offset;
  float s;
};

template <int G, int K> struct FusedCfg {
  static_assert(G == 64, "the weight-gradient accumulator is one M = 64 MMA tile");
  static constexpr int NTS = 2;                                 // tiles in flight in the epilogue (8 warps each)
  static constexpr int HROWS = K + 16;                          // rows of one m-block of the H image: K slots + ones
  static constexpr int HH_BYTES = HROWS * 128;                  // one m-block (64 batch columns)
  static constexpr int H_BYTES = 2 * HH_BYTES;
  static constexpr int HS = K <= 64 ? 6 : 4;                    // H stages: what shared memory holds
  // producer completion lag 0: a producer warp waits for its own copies and signals the tile before it asks for the next
  // stage -- with a lag the signal for tile T would wait for the stage of tile T + 1, i.e. for the weight gradient of
  // tile T + 1 - HS, and only HS - 1 tiles would ever be in flight
  static constexpr int LAG = 0;
  static constexpr int W_BYTES = G * K * 2;                     // [K/64 k-blocks][G rows][128 B]
  static constexpr int WS = 2;
  static constexpr int ST_BYTES = 128 * 64 * 2;                 // one dY tile per tile parity: [128 rows][128 B]
  static constexpr int NW = K + 8;                              // weight-gradient MMA N: slots + the ones columns
  static constexpr int DW_COLS = (NW + 15) / 16 * 16;           // TMEM columns per D_w buffer
  static constexpr int T_FWD0 = 2 * DW_COLS;                    // first column of the forward's accumulator ring
  static constexpr int NSLOT = (512 - T_FWD0) / G >= 4 ? 4 : (512 - T_FWD0) / G;   // K = 64: 4, K = 128: 3
  static_assert(NSLOT >= 3, "forward accumulator ring too short");   // (>= NTS: a set waits for tile T after T - 2, see t_full)
  static constexpr int OFF_H = 0;
  static constexpr int OFF_W = OFF_H + HS * H_BYTES;
  static constexpr int OFF_ST = OFF_W + WS * W_BYTES;
  static constexpr int OFF_BIAS = OFF_ST + NTS * ST_BYTES;      // [16 warps][32] fp32
  static constexpr int OFF_BAR = OFF_BIAS + 16 * 32 * 4;
  static constexpr int NBAR = 2 * HS + 2 * WS + 2 * NSLOT + 2 * NTS + 4;
  static constexpr int OFF_MISC = OFF_BAR + NBAR * 8;
  static constexpr int SMEM = OFF_MISC + 128 + 1024;
  static constexpr int THREADS = (16 + 7) * 32;              // 16 epilogue, 4 producers, 2 MMA issuers, 1 W loader
};

__device__ __forceinline__ uint32_t fz_tmem_ld1(uint32_t taddr) {
  uint32_t v;
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(v) : "r"(taddr) : "memory");
  return v;
}
__device__ __forceinline__ void fz_stg128(void* p, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("st.global.v4.b32 [%0], {%1, %2, %3, %4};" ::"l"(p), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
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
  uint64_t* w_empty = w_full + C::WS;            // [WS]    count 1 (commit after the group's last weight-gradient MMA)
  uint64_t* t_full = w_empty + C::WS;            // [NSLOT] count 1 (commit after the tile's forward MMAs)
  uint64_t* t_empty = t_full + C::NSLOT;         // [NSLOT] count 8 (the tile's epilogue warps have read the accumulator)
  uint64_t* s_full = t_empty + C::NSLOT;         // [NTS]   count 8: the tile's dY is in shared memory (A operand of the weight gradient)
  uint64_t* s_empty = s_full + C::NTS;           // [NTS]   count 2 (commit: the weight-gradient MMAs have read it; the issuing thread: so has its TMA store)
  uint64_t* dw_full = s_empty + C::NTS;          // [2]     count 1 (commit after the group's last weight-gradient MMA)
  uint64_t* dw_empty = dw_full + 2;              // [2]     count 4 (the warps that wrote dW_g out)
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + C::OFF_MISC);
  float* loss_red = reinterpret_cast<float*>(smem + C::OFF_MISC + 16);   // [16]

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int stripe = blockIdx.x, S = gridDim.x, NT = p.NT;
  const int ngl = p.NG > stripe ? (int)((p.NG - stripe + S - 1) / S) : 0;   // groups of this CTA
  const int total = ngl * NT;                                               // tiles: T = gl * NT + t

  if (threadIdx.x == 0) {
    for (int i = 0; i < C::HS; ++i) { mbar_init(&h_full[i], 4); mbar_init(&h_empty[i], 1); }
    for (int i = 0; i < C::WS; ++i) { mbar_init(&w_full[i], 1); mbar_init(&w_empty[i], 1); }
    for (int i = 0; i < C::NSLOT; ++i) { mbar_init(&t_full[i], 1); mbar_init(&t_empty[i], 8); }
    for (int i = 0; i < C::NTS; ++i) { mbar_init(&s_full[i], 8); mbar_init(&s_empty[i], 2); }
    for (int i = 0; i < 2; ++i) { mbar_init(&dw_full[i], 1); mbar_init(&dw_empty[i], 4); }
    fence_barrier_init();
  }
  // rows K .. K+15 of both m-blocks of every H stage: bf16 1.0 (swizzling permutes equal chunks: write linearly)
  for (int e = threadIdx.x; e < C::HS * 2 * 16 * 8; e += blockDim.x) {
    const int st = e / 256, hf = (e >> 7) & 1, r = e % 128;
    sts128(sbase + C::OFF_H + st * C::H_BYTES + hf * C::HH_BYTES + K * 128 + r * 16, 0x3F803F80u, 0x3F803F80u, 0x3F803F80u, 0x3F803F80u);
  }
  fence_proxy_async_smem();
  if (warp == 21 && lane == 0) { tma_prefetch_desc(&tmW); tma_prefetch_desc(&tmY); }
  if (warp == 20) tmem_alloc<512>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  pdl_wait();       // nothing above touches global memory (common.cuh, PDL)
  pdl_trigger();
  const uint32_t tmem_base = *tmem_slot;

  if (warp >= 16 && warp < 20) {
    // ===================== gather producers (as tc_tail.cu; the image has K + 16 rows per m-block) =====================
    const int pw = warp - 16;
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
    if (C::LAG == 1 && total > 0) {
      cp_async_wait<0>();
      fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) mbar_arrive(&h_full[(total - 1) % C::HS]);
    }
  } else if (warp == 20) {
    // ===================== MMA issuer 1 of 2: the forward of every tile =====================
    // (One issuing warp for both queues was measured to be this kernel's bottleneck: it never idled -- 18 idle polls in 280
    // tiles -- while producers and epilogue warps waited 40-55 % of the time.  The two queues touch different accumulators
    // and every hand-over goes through a commit, so they can be issued by two threads.)
    constexpr uint32_t idesc_f = make_idesc_bf16(128, G, /*A (H) MN-major*/ 1, /*B (W) K-major*/ 0);
    const uint64_t fa0 = make_sdesc_sw128(sbase + C::OFF_H, C::HH_BYTES, 1024);   // leading offset: the second 64 batch columns
    const uint64_t fb0 = make_sdesc_sw128(sbase + C::OFF_W, 16, 1024);
    int gl = 0, t = 0;
    for (int T = 0; T < total; ++T) {
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
        umma_commit(&t_full[slot]);
      }
      __syncwarp();
      if (++t == NT) { t = 0; ++gl; }
    }
  } else if (warp == 22) {
    // ===================== MMA issuer 2 of 2: the weight gradient of every tile, and its dY store =====================
    // The tile's forward MMAs have completed before this queue sees the tile (its dY exists), so the commits below, which
    // track this thread's MMAs only, release the H stage and the W stage safely.
    constexpr uint32_t idesc_w = make_idesc_bf16(64, C::NW, /*A (dY tile) MN-major*/ 1, /*B (H) K-major*/ 0);
    const uint64_t wa0 = make_sdesc_sw128(sbase + C::OFF_ST, 8192, 1024);         // [128 batch rows][64 labels], as stored
    const uint64_t wb0 = make_sdesc_sw128(sbase + C::OFF_H, 16, 1024);            // rows = slots (+ ones), 64 batch columns per m-block
    int glw = 0, tw = 0;
    for (int Tw = 0; Tw < total; ++Tw) {
      const int hs = Tw % C::HS, buf = glw & 1;
      if (tw == 0) mbar_wait(&dw_empty[buf], ((glw >> 1) & 1) ^ 1);        // D_w buffer written out (two groups ago)
      mbar_wait(&s_full[Tw & 1], (Tw >> 1) & 1);                             // the epilogue has staged this tile's dY
      tc_fence_after();
      if (elect_one()) {
        const uint64_t ad0 = wa0 + (uint64_t)(((Tw & 1) * C::ST_BYTES) >> 4);
        const uint64_t bd0 = wb0 + (uint64_t)((hs * C::H_BYTES) >> 4);
        const uint32_t d = tmem_base + buf * C::DW_COLS;
#pragma unroll
        for (int j = 0; j < 8; ++j)
          umma_f16(d, ad0 + (uint64_t)((j * 2048) >> 4), bd0 + (uint64_t)(((j >> 2) * C::HH_BYTES + (j & 3) * 32) >> 4), idesc_w,
                   (tw | j) ? 1u : 0u);
        umma_commit(&h_empty[hs]);
        umma_commit(&s_empty[Tw & 1]);
        if (tw == NT - 1) { umma_commit(&dw_full[buf]); umma_commit(&w_empty[glw % C::WS]); }
        // the same tile goes to HBM as dY (rows past the batch are clipped by the tensor map).  elect.sync names the same
        // thread every time, so the bulk groups are this thread's: all but the newest store have been read -> the tile
        // before this one may be overwritten as far as its store is concerned (second arrival on its s_empty)
        tma_store_3d(&tmY, smem + C::OFF_ST + (Tw & 1) * C::ST_BYTES, 0, tw * 128, (int)(stripe + (int64_t)glw * S));
        bulk_commit();
        if (Tw >= 1) { bulk_wait_read<1>(); mbar_arrive(&s_empty[(Tw - 1) & 1]); }
      }
      __syncwarp();
      if (++tw == NT) { tw = 0; ++glw; }
    }
    if (elect_one()) bulk_wait<0>();
    __syncwarp();
  } else if (warp == 21) {
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
  } else if (warp < 16) {
    // ===================== epilogue: warp = (tile parity, 32-label half, TMEM lane quadrant); lane = batch row ===========
    const int q = warp & 3, half = (warp >> 2) & 1, tsel = warp >> 3;
    const int row = q * 32 + lane;
    float loss_local = 0.f;
    const float hs = 0.5f * p.s;
    const uint32_t stage_row = sbase + C::OFF_ST + tsel * C::ST_BYTES + row * 128;
    const uint32_t swz = (uint32_t)(lane & 7);
    const uint32_t sb = sbase + C::OFF_BIAS + warp * 128;

    // D_w of group gd (this CTA's gd-th; buffer gd & 1 = tsel) -> dW rows and db, by the half-0 warps of the parity:
    // M = 64 puts label rows 16 q .. 16 q + 15 into lanes 0-15 of quadrant q
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
              float* o = reinterpret_cast<float*>(p.dW) + l * K + c * 32;
#pragma unroll
              for (int i = 0; i < 8; ++i) fz_stg128(o + 4 * i, v[4 * i], v[4 * i + 1], v[4 * i + 2], v[4 * i + 3]);
            } else {
              bf16* o = reinterpret_cast<bf16*>(p.dW) + l * K + c * 32;
#pragma unroll
              for (int i = 0; i < 4; ++i)
                fz_stg128(o + 8 * i, pack_bf16x2(__uint_as_float(v[8 * i]), __uint_as_float(v[8 * i + 1])),
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
    int my_gd = tsel;                     // next group whose D_w this parity writes out (half-0 warps)
    // one cursor per batch tile into this thread's target rows (b = t * 128 + row): groups ascend for a fixed t, so each
    // row is walked once; in the common case (no positive of the row in the tile) a tile costs no load at all
    int cnxt[4], cpc[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      cnxt[i] = 0x7fffffff; cpc[i] = 0;
      const int bi = i * 128 + row;
      if (i < NT && bi < p.B && p.rowptr) {
        cpc[i] = __ldg(p.rowptr + bi);
        if (cpc[i] < __ldg(p.rowptr + bi + 1)) cnxt[i] = __ldg(p.col + cpc[i]);
      }
    }

    for (int T = tsel; T < total; T += C::NTS) {
      const int gl = T / NT, t = T - gl * NT;
      const int64_t g = stripe + (int64_t)gl * S;
      const int nl = (int)min((int64_t)G, p.L - g * G);
      const int nvalid = nl - half * 32;                       // labels of this warp's half that exist (may be <= 0)
      const int slot = T % C::NSLOT;
      const int b = t * 128 + row;
      const bool valid_row = b < p.B;
      if (p.bias) {
        const int l = half * 32 + lane;
        sts32(sb + lane * 4, __float_as_uint(l < nl ? __ldg(p.bias + g * G + l) : 0.f));
      }
      // positives of this row among the warp's 32 labels
      uint32_t ym = 0;
      {
        const int64_t lo64 = p.label_offset + g * G + half * 32;
        const int lo = (int)min(lo64, (int64_t)0x7fffffff), hi = (int)min(lo64 + max(min(nvalid, 32), 0), (int64_t)0x7fffffff);
        int nxt = cnxt[0];
#pragma unroll
        for (int i = 1; i < 4; ++i) if (t == i) nxt = cnxt[i];
        if (nxt < hi) {                    // (rare) walk the row up to the end of this label range
          int pc = cpc[0];
#pragma unroll
          for (int i = 1; i < 4; ++i) if (t == i) pc = cpc[i];
          const int pe = __ldg(p.rowptr + b + 1);
          while (nxt < hi) {
            if (nxt >= lo) ym |= 1u << (nxt - lo);
            ++pc;
            nxt = pc < pe ? __ldg(p.col + pc) : 0x7fffffff;
          }
#pragma unroll
          for (int i = 0; i < 4; ++i) if (t == i) { cnxt[i] = nxt; cpc[i] = pc; }
        }
      }
      __syncwarp();
      const bool slow = __any_sync(0xffffffffu, ym != 0) || nvalid < 32;

      mbar_wait(&t_full[slot], (T / C::NSLOT) & 1);
      tc_fence_after();
      uint32_t v[32];
      tmem_ld32(tmem_base + ((uint32_t)(q * 32) << 16) + C::T_FWD0 + slot * G + half * 32, v);
      tmem_ld_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&t_empty[slot]);
      float R[4] = {0.f, 0.f, 0.f, 0.f}, P[4] = {1.f, 1.f, 1.f, 1.f};
      uint32_t out[16];
      const int nv = max(nvalid, 0);
      if (slow) {
        if (p.bias) epi32<true, true>(v, sb, ym, nv, p.s, hs, R, P, out, nullptr);
        else epi32<true, false>(v, sb, ym, nv, p.s, hs, R, P, out, nullptr);
      } else {
        if (p.bias) epi32<false, true>(v, sb, 0u, 32, p.s, hs, R, P, out, nullptr);
        else epi32<false, false>(v, sb, 0u, 32, p.s, hs, R, P, out, nullptr);
      }
      if (valid_row) {
        loss_local += (R[0] + R[1]) + (R[2] + R[3]) - 0.69314718056f * __log2f((P[0] * P[1]) * (P[2] * P[3]));
      } else {                   // rows past the batch: the dY store clips them, the weight gradient must see zeros (db)
#pragma unroll
        for (int i = 0; i < 16; ++i) out[i] = 0u;
      }
      // the dY tile of this parity is free again once the weight-gradient MMAs of its previous tile AND that tile's TMA
      // store have read it
      mbar_wait(&s_empty[tsel], ((T >> 1) & 1) ^ 1);
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const uint32_t ch = (uint32_t)(half * 4 + i) ^ swz;
        sts128(stage_row + ch * 16, out[4 * i], out[4 * i + 1], out[4 * i + 2], out[4 * i + 3]);
      }
      fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) mbar_arrive(&s_full[tsel]);
      // D_w of an earlier group of this parity: its last MMAs were issued when tile (my_gd + 1) NT - 1 was staged
      if (half == 0 && my_gd < ngl && T >= (my_gd + 1) * NT + 1) { dw_out(my_gd); my_gd += 2; }
    }
    if (half == 0)
      for (; my_gd < ngl; my_gd += 2) dw_out(my_gd);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) loss_local += __shfl_xor_sync(0xffffffffu, loss_local, o);
    if (lane == 0) loss_red[warp] = loss_local;
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 20) { tc_fence_after(); tmem_dealloc<512>(tmem_base); }
  if (p.partials) {
    float t = 0.f;
    if (threadIdx.x == 0) {
#pragma unroll
      for (int i = 0; i < 16; ++i) t += loss_red[i];
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
  CUtensorMap tmW;
  {
    const uint64_t dims[2] = {(uint64_t)K, (uint64_t)sh.L};
    const uint64_t str[1] = {(uint64_t)K * 2};
    const uint32_t box[2] = {64, (uint32_t)G};
    int rc = encode_tmap(&tmW, 2, W, 2, dims, str, box, 128);
    if (rc) return rc;
  }
  CUtensorMap tmY;
  {
    const uint64_t dims[3] = {(uint64_t)G, (uint64_t)sh.B, (uint64_t)sh.NG};
    const uint64_t str[2] = {(uint64_t)G * 2, (uint64_t)sh.B * G * 2};
    const uint32_t box[3] = {64, 128, 1};          // a whole batch tile
    int rc = encode_tmap(&tmY, 2, dY, 3, dims, str, box, 128);
    if (rc) return rc;
  }
  FusedParams p;
  memset(&p, 0, sizeof(p));
  p.Xt = (const bf16*)Xt; p.idx = idx; p.bias = bias; p.rowptr = rowptr; p.col = col; p.partials = partials; p.loss = loss;
  p.dY = (bf16*)dY; p.dW = dW; p.dbias = dbias;
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
