// tc_tail.cu -- tcgen05 / TMEM / TMA kernels of the HASTE sparse tail (sm_100a; bf16 in, fp32 accumulate).
//
// Forward + fused BCE (PAPER.md:97 "gather-once, dense GEMM per group", :111 Eq. 3):
//   persistent CTAs, one per SM.  A CTA owns a pair of 128-row batch tiles and a stripe of groups.
//   per (group g, batch tile): Z[128 x G] = H_g[128 x K] * W_g^T, H_g = X[:, idx_g] gathered from X^T.
//   warp roles (704 threads):
//     warps 0-15  epilogue: TMEM -> registers -> sigmoid/softplus (1 MUFU per logit) -> bf16 dY
//                 -> swizzled smem tile -> TMA store; loss partial per thread.  Four sets of 4 warps
//                 work on tiles T = set mod 4 (the epilogue is a latency chain per warp: with two sets the
//                 schedulers sat idle 42 % of the time); a thread owns ONE batch row for the whole kernel,
//                 so its CSR target row is walked once with a running cursor.
//     warps 16-19 gather producers: cp.async 16-B chunks of X^T rows idx_g into the swizzled H image.
//     warp 20     MMA issuer (one thread): tcgen05.mma M=128, N=G, K=16 x (K/16) into a TMEM slot ring.
//     warp 21     TMA loader of W_g (the [G x K] block is contiguous in W).
#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <new>

#include "tc_common.cuh"
#include "tc_epilogue.cuh"
#include "tc_kernels.h"
#include <cmath>

namespace haste {

// ---------------------------------------------------------------------------------------------
// host: tensor-map encoding through the driver entry point (no link-time libcuda dependency)
// ---------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn get_encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  return fn;
}

int encode_tmap(CUtensorMap* out, int dtype_bytes, const void* base, int rank, const uint64_t* dims,
                const uint64_t* strides_bytes, const uint32_t* box, int swizzle_bytes) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) { set_error("cuTensorMapEncodeTiled is not available from the driver"); return HASTE_ERR_CUDA; }
  cuuint64_t gd[5]; cuuint64_t gs[4]; cuuint32_t bx[5]; cuuint32_t es[5];
  for (int i = 0; i < rank; ++i) { gd[i] = dims[i]; bx[i] = box[i]; es[i] = 1; }
  for (int i = 0; i + 1 < rank; ++i) gs[i] = strides_bytes[i];
  const CUtensorMapSwizzle sw = swizzle_bytes == 128 ? CU_TENSOR_MAP_SWIZZLE_128B
                              : swizzle_bytes == 64  ? CU_TENSOR_MAP_SWIZZLE_64B
                              : swizzle_bytes == 32  ? CU_TENSOR_MAP_SWIZZLE_32B : CU_TENSOR_MAP_SWIZZLE_NONE;
  const CUtensorMapDataType dt = dtype_bytes == 2 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
  CUresult r = fn(out, dt, (cuuint32_t)rank, const_cast<void*>(base), gd, gs, bx, es, CU_TENSOR_MAP_INTERLEAVE_NONE, sw,
                  CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { set_error("cuTensorMapEncodeTiled failed with CUresult %d", (int)r); return HASTE_ERR_CUDA; }
  return HASTE_OK;
}

using namespace tc;

// ---------------------------------------------------------------------------------------------
// forward
// ---------------------------------------------------------------------------------------------
struct FwdParams {
  const bf16* Xt;          // [d][Bpad]
  const int32_t* idx;      // [NG][K]
  const float* bias;       // [L] or null
  const int32_t* rowptr;   // [B+1] or null
  const int32_t* col;      // [nnz]
  float* partials;         // [1024] unscaled loss partials + ticket (finalize_loss_last_cta), or null
  float* loss;             // device scalar: s * sum of the partials, written by the last CTA
  float* logits;           // [B][L] fp32 or null
  int write_dy;
  int z_mode;              // 1: the dY buffer receives the logits themselves (bf16, same layout); no targets, no loss
                           // 2: nothing is written but the per-thread top-8 logits of each batch row (topk_val / topk_idx)
  float* topk_val;         // [gridDim.x][epilogue sets][128 rows][8] candidate logits (fp32), descending; -inf = none
  int* topk_idx;           // same shape: label index inside this layer
  int B, Bpad, NT, NP, S;  // NT batch tiles of 128; NP tile pairs; S group stripes (grid = NP*S)
  int64_t L, NG, label_offset;
  float s;
};

template <int G, int K> struct FwdCfg {
  static constexpr int NSET = (G == 128 && K == 128) ? 2 : 4;   // epilogue sets (4 warps each); what shared memory allows
  // Narrow groups (G <= 16): a tile is as many gathered bytes as a wide group's but a quarter (an eighth) of the work
  // after it, and what bounds it is the hand-shaking itself: with the wide groups' six barriers per tile and no work at
  // all in any role the kernel took as long as with all of it (config 5, B = 1024, G = 16: 0.79 vs 0.80 ms; a barrier
  // wait costs the waiting warp 100-300 cycles even when it succeeds at once).  So NARROW runs ONE ring of R entries
  // -- H stage, W stage and TMEM slot e = T mod R belong together -- with two barriers per entry:
  //   ready[e]: the producer warp's gather has landed + the W box has landed + the four epilogue warps have drained
  //             the slot (its previous use);   done[e]: the tile's MMAs have completed (one commit).
  // The issuer waits once and commits once per tile; each producer warp takes every fourth tile whole, so its own chain
  // (wait, issue, wait for the copies, fence, arrive) is a quarter as often on the critical path.
  static constexpr bool NARROW = G <= 16;
  static constexpr int HS = NARROW ? (K <= 64 ? 8 : 5) : 3;     // H stages (NARROW: the ring length R)
  static constexpr int LAG = 1;                                 // producer completion lag (< HS-1, or the MMAs serialise)
  // narrow groups (G = 16, 8): the MMA is N = GP = 16 wide (the smallest N of an M = 128 MMA); for G = 8 the upper 8 rows
  // of the W image are never written and the 8 accumulator columns they produce are never read
  static constexpr int GP = G < 16 ? 16 : G;                    // MMA N = accumulator columns per slot = rows of the W image
  static constexpr int CW = G < 32 ? G : 32;                    // logits per epilogue chunk
  static constexpr int NCH = G / CW;                            // chunks per group
  static constexpr int H_BYTES = K * 256;                       // [2 m-blocks][K rows][128 B]
  static constexpr int W_BYTES = GP * K * 2;                    // [K/64 k-blocks][GP rows][128 B]
  static constexpr int W_TX = G * K * 2;                        // bytes the TMA box of a group brings
  static constexpr int WS = NARROW ? HS : W_BYTES <= 16384 ? 3 : 2;   // W stages
  static constexpr int ST_BYTES = 128 * (G < 64 ? G : 64) * 2;  // one dY staging tile (<= 64 labels wide) per epilogue set
  static constexpr int NSLOT = NARROW ? HS : (512 / GP) >= 8 ? 8 : (512 / GP);  // TMEM accumulator ring (GP columns each)
  static constexpr int OFF_H = 0;
  static constexpr int OFF_W = OFF_H + HS * H_BYTES;
  static constexpr int OFF_ST = OFF_W + WS * W_BYTES;
  static constexpr int OFF_BIAS = OFF_ST + NSET * ST_BYTES;     // [16 warps][G] fp32
  static constexpr int OFF_BAR = OFF_BIAS + 4 * NSET * G * 4;
  static constexpr int NBAR = 2 * HS + 2 * WS + 2 * NSLOT;
  static constexpr int OFF_MISC = OFF_BAR + NBAR * 8;           // tmem base, loss scratch
  static constexpr int SMEM = OFF_MISC + 128 + 1024;            // + alignment slack
  static constexpr int THREADS = (4 * NSET + 6) * 32;
};

// TOPK > 0: the fused top-k instances (z_mode 2; candidate lists of TOPK = 5 or 8 entries per thread) and TOPK = -1: the
// logits-only instance (z_mode 1) are kernels of their own, so that they cost the training kernel (TOPK = 0) no registers
template <int G, int K, int TOPK>
__global__ void __launch_bounds__(FwdCfg<G, K>::THREADS, 1)
tc_fwd_kernel(const __grid_constant__ CUtensorMap tmW, const __grid_constant__ CUtensorMap tmY, const FwdParams p) {
  using C = FwdCfg<G, K>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const uint32_t sbase = smem_u32(smem);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::OFF_BAR);
  uint64_t* h_full = bars;                       // [HS]  count 4 (producer warps)
  uint64_t* h_empty = bars + C::HS;              // [HS]  count 1 (umma commit)
  // NARROW: h_full = w_full = t_empty = ready[R] (count 6 + tx), h_empty = w_empty = t_full = done[R] (count 1)
  uint64_t* w_full = C::NARROW ? h_full : bars + 2 * C::HS;           // [WS]  count 1 + tx
  uint64_t* w_empty = C::NARROW ? h_empty : w_full + C::WS;           // [WS]  count 1 (umma commit)
  uint64_t* t_full = C::NARROW ? h_empty : w_empty + C::WS;           // [NSLOT] count 1 (umma commit)
  uint64_t* t_empty = C::NARROW ? h_full : t_full + C::NSLOT;         // [NSLOT] count 4 (epilogue warps of one set)
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + C::OFF_MISC);
  float* loss_red = reinterpret_cast<float*>(smem + C::OFF_MISC + 16);   // [4 * NSET]

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int pr = blockIdx.x % p.NP, stripe = blockIdx.x / p.NP;
  const int ntp = min(2, p.NT - 2 * pr);                                  // batch tiles of this CTA's pair (1 or 2)
  const int tsh = ntp - 1;                                                // T >> tsh = group, T & tsh = tile of the pair
  const int ngl = (int)((p.NG - stripe + p.S - 1) / p.S);                 // groups of this CTA's stripe
  const int total = ngl << tsh;

  if (threadIdx.x == 0) {
    if constexpr (C::NARROW) {
      for (int i = 0; i < C::HS; ++i) {
        mbar_init(&h_full[i], 6); mbar_init(&h_empty[i], 1);
        for (int a = 0; a < 4; ++a) mbar_arrive(&h_full[i]);       // first round: no earlier use of the slot to drain
      }
    } else {
      for (int i = 0; i < C::HS; ++i) { mbar_init(&h_full[i], 4); mbar_init(&h_empty[i], 1); }
      for (int i = 0; i < C::WS; ++i) { mbar_init(&w_full[i], 1); mbar_init(&w_empty[i], 1); }
      for (int i = 0; i < C::NSLOT; ++i) { mbar_init(&t_full[i], 1); mbar_init(&t_empty[i], 4); }
    }
    fence_barrier_init();
  }
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
    // ===================== gather producers =====================
    const int pw = warp - EW;
    if constexpr (C::NARROW) {
      // warp pw gathers tiles T = pw, pw + 4, ... whole: all K rows, two rows per instruction, two tiles in flight
      const int sub = lane >> 4, c = lane & 15;
      const uint32_t dst_lane = (uint32_t)((c >> 3) * (K * 128) + (((c & 7)) << 4));
      constexpr int NI = K / 32;                     // lane holds slots lane + 32 t of the tile's idx row
      int idx_cur[NI], idx_nxt[NI];
      auto load_idx = [&](int T, int (&o)[NI]) {
        const int64_t g = stripe + (int64_t)(T >> tsh) * p.S;
#pragma unroll
        for (int t = 0; t < NI; ++t) o[t] = T < total ? __ldg(p.idx + g * K + lane + 32 * t) : 0;
      };
      load_idx(pw, idx_nxt);
      int prev_hs = -1;
      for (int T = pw; T < total; T += 4) {
        const int which = T & tsh;
#pragma unroll
        for (int t = 0; t < NI; ++t) idx_cur[t] = idx_nxt[t];
        load_idx(T + 4, idx_nxt);
        const int hs = T % C::HS;
        mbar_wait(&h_empty[hs], ((T / C::HS) & 1) ^ 1);
        const int b0 = (2 * pr + which) * 128;
        const uint32_t dst0 = sbase + C::OFF_H + hs * C::H_BYTES + dst_lane;
        const bf16* src0 = p.Xt + b0 + c * 8;
#pragma unroll
        for (int i = 0; i < K / 2; ++i) {
          const int k = 2 * i + sub;
          const int f = __shfl_sync(0xffffffffu, idx_cur[(2 * i) >> 5], k & 31);
          const uint32_t dst = (dst0 + k * 128) ^ ((uint32_t)(k & 7) << 4);
          cp_async16(dst, src0 + (size_t)f * p.Bpad);
        }
        cp_async_commit();
        if (prev_hs >= 0) {
          cp_async_wait<1>();
          fence_proxy_async_smem();
          __syncwarp();
          if (lane == 0) mbar_arrive(&h_full[prev_hs]);
        }
        prev_hs = hs;
      }
      if (prev_hs >= 0) {
        cp_async_wait<0>();
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) mbar_arrive(&h_full[prev_hs]);
      }
    } else {
    constexpr int RPW = K / 4;                       // rows (slots) per producer warp
    const int sub = lane >> 4, c = lane & 15;        // two rows per instruction, 16 chunks of 16 B per row
    const uint32_t dst_lane = (uint32_t)((c >> 3) * (K * 128) + (((c & 7)) << 4));
    const int32_t* idx_ptr = p.idx + (int64_t)stripe * K + pw * RPW + lane;   // this lane's slot of group gl: + gl*S*K
    const int64_t idx_step = (int64_t)p.S * K;
    // slot indices are prefetched two groups ahead so that the gather never waits on an HBM read of idx
    int idx_cur = 0, idx_n1 = 0, idx_n2 = 0;
    if (lane < RPW) {
      idx_n1 = __ldg(idx_ptr);
      if (ngl > 1) idx_n2 = __ldg(idx_ptr + idx_step);
    }
    for (int T = 0; T < total; ++T) {
      const int gl = T >> tsh, which = T & tsh;
      if (which == 0) {
        idx_cur = idx_n1; idx_n1 = idx_n2;
        if (lane < RPW && gl + 2 < ngl) idx_n2 = __ldg(idx_ptr + (gl + 2) * idx_step);
      }
      const int hs = T % C::HS;
      mbar_wait(&h_empty[hs], ((T / C::HS) & 1) ^ 1);
      const int b0 = (2 * pr + which) * 128;
      const uint32_t dst0 = sbase + C::OFF_H + hs * C::H_BYTES + dst_lane;
      const bf16* src0 = p.Xt + b0 + c * 8;
#pragma unroll
      for (int i = 0; i < RPW / 2; ++i) {
        const int kk = 2 * i + sub;
        const int f = __shfl_sync(0xffffffffu, idx_cur, kk);
        const int k = pw * RPW + kk;
        // row k of the image, chunk (c&7) XOR (k&7): the 128-byte swizzle of the UMMA / TMA layouts
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
    }
    // drain the last LAG tiles
#pragma unroll
    for (int r = C::LAG - 1; r >= 0; --r) {
      const int T = total - 1 - r;
      if (T >= 0) {
        if (r == 2) cp_async_wait<2>(); else if (r == 1) cp_async_wait<1>(); else cp_async_wait<0>();
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) mbar_arrive(&h_full[T % C::HS]);
      }
    }
    }
  } else if (warp == EW + 4) {
    // ===================== MMA issuer =====================
    // The whole warp walks the loop and waits; one elected lane issues.  (Issuing from inside `if (lane == 0)` makes
    // ptxas wrap every tcgen05 instruction in an elect/branch loop, and rebuilding both descriptors per MMA is a
    // chain of uniform-datapath ops: together ~1100 cycles per tile, which was this kernel's critical path.)
    constexpr uint32_t idesc = make_idesc_bf16(128, C::GP, /*A MN-major*/ 1, /*B K-major*/ 0);
    const uint64_t adesc0 = make_sdesc_sw128(sbase + C::OFF_H, K * 128, 1024);
    const uint64_t bdesc0 = make_sdesc_sw128(sbase + C::OFF_W, 16, 1024);
    for (int T = 0; T < total; ++T) {
      const int gl = T >> tsh, which = T & tsh;
      const int ws = C::NARROW ? T % C::HS : gl % C::WS, hs = T % C::HS, slot = T % C::NSLOT;
      if constexpr (C::NARROW) {
        mbar_wait(&h_full[hs], (T / C::HS) & 1);                // ready: gather + W landed, slot drained
      } else {
        if (which == 0) mbar_wait(&w_full[ws], (gl / C::WS) & 1);
        mbar_wait(&h_full[hs], (T / C::HS) & 1);
        mbar_wait(&t_empty[slot], ((T / C::NSLOT) & 1) ^ 1);
      }
      tc_fence_after();
      if (elect_one()) {
        const uint64_t ad0 = adesc0 + (uint64_t)((hs * C::H_BYTES) >> 4);       // the address field never carries out
        const uint64_t bd0 = bdesc0 + (uint64_t)((ws * C::W_BYTES) >> 4);
        const uint32_t d = tmem_base + slot * C::GP;
#pragma unroll
        for (int j = 0; j < K / 16; ++j)
          umma_f16(d, ad0 + (uint64_t)((j * 2048) >> 4), bd0 + (uint64_t)(((j >> 2) * (C::GP * 128) + (j & 3) * 32) >> 4), idesc,
                   j > 0 ? 1u : 0u);
        umma_commit(&h_empty[hs]);                              // NARROW: done[e], the only commit
        if constexpr (!C::NARROW) {
          umma_commit(&t_full[slot]);
          if (which == tsh) umma_commit(&w_empty[ws]);
        }
      }
      __syncwarp();
    }
  } else if (warp == EW + 5) {
    // ===================== W loader =====================
    if (C::NARROW && lane == 0) {                               // one (small) W box per tile, into the tile's ring entry
      for (int T = 0; T < total; ++T) {
        const int e = T % C::HS;
        const int64_t g = stripe + (int64_t)(T >> tsh) * p.S;
        mbar_wait(&h_empty[e], ((T / C::HS) & 1) ^ 1);
        mbar_arrive_expect_tx(&h_full[e], C::W_TX);
#pragma unroll
        for (int kb = 0; kb < K / 64; ++kb)
          tma_load_2d(smem + C::OFF_W + e * C::W_BYTES + kb * (C::GP * 128), &tmW, &h_full[e], kb * 64, (int)(g * G));
      }
    } else if (lane == 0) {
      for (int gl = 0; gl < ngl; ++gl) {
        const int ws = gl % C::WS;
        const int64_t g = stripe + (int64_t)gl * p.S;
        mbar_wait(&w_empty[ws], ((gl / C::WS) & 1) ^ 1);
        mbar_arrive_expect_tx(&w_full[ws], C::W_TX);
#pragma unroll
        for (int kb = 0; kb < K / 64; ++kb)
          tma_load_2d(smem + C::OFF_W + ws * C::W_BYTES + kb * (C::GP * 128), &tmW, &w_full[ws], kb * 64, (int)(g * G));
      }
    }
  } else {
    // ===================== epilogue: every warp is self-contained (own rows, own staging, own TMA stores) =====
    const int set = warp >> 2, q = warp & 3;                   // set s works on tiles T = s (mod NSET)
    const int row = q * 32 + lane;                             // row of the batch tile == TMEM lane
    const int my_bt = 2 * pr + (ntp == 2 ? (set & 1) : 0);
    const int b = my_bt * 128 + row;
    const bool valid_row = b < p.B;
    int pc = 0, pe = 0;
    int nxt = 0x7fffffff;
    if (valid_row && p.rowptr) {
      pc = __ldg(p.rowptr + b); pe = __ldg(p.rowptr + b + 1);
      if (pc < pe) nxt = __ldg(p.col + pc);
    }
    float loss_local = 0.f;
    const float hs = 0.5f * p.s;
    // z_mode 2 (fused top-k): the 8 largest logits this thread has seen for its batch row, descending
    constexpr int KL = TOPK > 0 ? TOPK : 1;
    float tv[KL];
    int ti[KL];
#pragma unroll
    for (int i = 0; i < KL; ++i) { tv[i] = -INFINITY; ti[i] = -1; }
    // this warp's 32 rows of the half's staging tile(s); rows are 128 B (G >= 64) or 2 G bytes (64, 32, 16), swizzled as
    // the TMA store of that row length expects (none for 16-byte rows)
    constexpr int CW = C::CW, NCH = C::NCH;
    constexpr int ROWB = G >= 64 ? 128 : G * 2;
    const uint32_t stage_w = sbase + C::OFF_ST + set * C::ST_BYTES + q * 32 * ROWB;
    const uint32_t stage_row = stage_w + lane * ROWB;
    const uint32_t swz = G >= 64 ? (uint32_t)(lane & 7) : G == 32 ? (uint32_t)((lane >> 1) & 3) : G == 16 ? (uint32_t)((lane >> 2) & 1) : 0u;
    const uint32_t sbias_w = sbase + C::OFF_BIAS + warp * G * 4;
    // the group's bias values, fetched one of this warp's tiles ahead (a global load at the head of a tile's chain would
    // be ~700 cycles nothing else in the warp hides)
    auto bias_of = [&](int T, int i) -> float {
      const int64_t gg = stripe + (int64_t)(T >> tsh) * p.S;
      const int l = i * 32 + lane;
      return (T < total && (G >= 32 || l < G) && gg * G + l < p.L) ? __ldg(p.bias + gg * G + l) : 0.f;
    };
    float bnext[NCH];
#pragma unroll
    for (int i = 0; i < NCH; ++i) bnext[i] = p.bias ? bias_of(set, i) : 0.f;
    for (int T = set; T < total; T += C::NSET) {
      const int gl = T >> tsh;
      const int64_t g = stripe + (int64_t)gl * p.S;
      const int nl = (int)min((int64_t)G, p.L - g * G);
      const int slot = T % C::NSLOT;
      if (lane == 0) bulk_wait_read<0>();                      // this warp's previous TMA store has read the staging rows
      if (p.bias) {
#pragma unroll
        for (int i = 0; i < NCH; ++i) {
          const int l = i * 32 + lane;
          if (G >= 32 || l < G) sts32(sbias_w + l * 4, __float_as_uint(bnext[i]));
          bnext[i] = bias_of(T + C::NSET, i);
        }
      }
      __syncwarp();
      // positives of this row inside the group: walk the CSR cursor (ascending groups, fixed row)
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
      const bool slow = __any_sync(0xffffffffu, anyy != 0) || nl < G || p.logits != nullptr;

      mbar_wait(&t_full[slot], (T / C::NSLOT) & 1);
      tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + slot * C::GP;
      float R[4] = {0.f, 0.f, 0.f, 0.f}, P[4] = {1.f, 1.f, 1.f, 1.f};
      uint32_t v[32];                 // one chunk at a time: 16 epilogue warps hide the TMEM latency, registers are short
      // two chunks are unrolled; four copies of the epilogue code (G = 128) overflow the instruction cache (see tc_head.cu)
#pragma unroll(G >= 128 ? 1 : 2)
      for (int sc = 0; sc < NCH; ++sc) {
        uint32_t ymsc = ym[0];
#pragma unroll
        for (int i = 1; i < NCH; ++i) if (sc == i) ymsc = ym[i];
        tmem_ld_first<CW>(taddr + sc * 32, v);
        tmem_ld_wait();
        if (sc + 1 == NCH) {
          // all of this warp's TMEM reads are done: hand the accumulator slot back to the MMA issuer
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(&t_empty[slot]);
        }
        uint32_t out[16];
        float* zout = (p.logits && valid_row) ? p.logits + (size_t)b * p.L + g * G + sc * 32 : nullptr;
        const int nvalid = nl - sc * 32;
        const uint32_t sb = sbias_w + sc * 128;
        if constexpr (TOPK > 0) { // fused top-k: nothing leaves the chip but the row's candidates
          // A thread inserts ~KL ln(n / KL) times over the n labels it sees, so most runs of 8 logits hold nothing above its
          // KL-th best: four 3-input maxima per run find that out, and only the runs that do are looked at one by one.
#pragma unroll
          for (int r8 = 0; r8 < CW / 8; ++r8) {
            float z[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
              const int jj = r8 * 8 + j;
              z[j] = __uint_as_float(v[jj]);
              if (p.bias) {
                float b0;
                asm volatile("ld.shared.f32 %0, [%1];" : "=f"(b0) : "r"(sb + jj * 4));
                z[j] += b0;
              }
              if (jj >= nvalid) z[j] = -INFINITY;
            }
            float m = max3(max3(z[0], z[1], z[2]), max3(z[3], z[4], z[5]), fmaxf(z[6], z[7]));
            // A run that holds a candidate for SOME lane is entered by the whole warp (early in a stripe: most runs), so
            // what happens inside must be short: pull out the run's maximum, insert it, knock it out, look again -- one
            // pass per candidate of the lane that has most (usually one), not one branch per logit.
            const int l0 = (int)(g * G) + sc * 32 + r8 * 8;
            while (m > tv[KL - 1]) {
              int js = 7;
#pragma unroll
              for (int j = 6; j >= 0; --j) js = z[j] == m ? j : js;      // first position of the maximum: earlier labels win ties
              tv[KL - 1] = m; ti[KL - 1] = l0 + js;
#pragma unroll
              for (int i = KL - 1; i > 0; --i)
                if (tv[i] > tv[i - 1]) {
                  const float a = tv[i]; tv[i] = tv[i - 1]; tv[i - 1] = a;
                  const int b_ = ti[i]; ti[i] = ti[i - 1]; ti[i - 1] = b_;
                }
#pragma unroll
              for (int j = 0; j < 8; ++j) z[j] = j == js ? -INFINITY : z[j];
              m = max3(max3(z[0], z[1], z[2]), max3(z[3], z[4], z[5]), fmaxf(z[6], z[7]));
            }
          }
        } else if constexpr (TOPK < 0) {    // logits-only forward: z (+ bias) rounded to bf16, padding labels (>= L) written as zero
#pragma unroll
          for (int j = 0; j < CW; j += 2) {
            float z0 = __uint_as_float(v[j]), z1 = __uint_as_float(v[j + 1]);
            if (p.bias) {
              float b0, b1;
              asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(b0), "=f"(b1) : "r"(sb + j * 4));
              z0 += b0; z1 += b1;
            }
            out[j >> 1] = pack_bf16x2(j < nvalid ? z0 : 0.f, j + 1 < nvalid ? z1 : 0.f);
          }
        } else if (slow) {
          if (p.bias) epi32<true, true, CW>(v, sb, ymsc, nvalid, p.s, hs, R, P, out, zout);
          else epi32<true, false, CW>(v, sb, ymsc, nvalid, p.s, hs, R, P, out, zout);
        } else {
          if (p.bias) epi32<false, true, CW>(v, sb, 0u, CW, p.s, hs, R, P, out, nullptr);
          else epi32<false, false, CW>(v, sb, 0u, CW, p.s, hs, R, P, out, nullptr);
        }
        if (sc & 1) {   // 64 factors in [1/2,1) at most per product: fold into the loss, restart the chains
          loss_local += (R[0] + R[1]) + (R[2] + R[3]) - 0.69314718056f * __log2f((P[0] * P[1]) * (P[2] * P[3]));
#pragma unroll
          for (int i = 0; i < 4; ++i) { R[i] = 0.f; P[i] = 1.f; }
        }
        if (p.write_dy) {
          if (G > 64 && sc == 2) {        // second 64-label half of a wide group reuses the staging rows
            if (lane == 0) bulk_wait_read<0>();
            __syncwarp();
          }
#pragma unroll
          for (int i = 0; i < CW / 8; ++i) {
            const uint32_t ch = (uint32_t)((G >= 64 ? (sc & 1) * 4 : 0) + i) ^ swz;
            sts128(stage_row + ch * 16, out[4 * i], out[4 * i + 1], out[4 * i + 2], out[4 * i + 3]);
          }
          if (sc == NCH - 1 || (G > 64 && sc == 1)) {
            fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) {
              tma_store_3d(&tmY, smem + C::OFF_ST + set * C::ST_BYTES + q * 32 * ROWB, (sc >> 1) * 64, my_bt * 128 + q * 32, (int)g);
              bulk_commit();
            }
          }
        }
      }
      if (NCH & 1)
        loss_local += (R[0] + R[1]) + (R[2] + R[3]) - 0.69314718056f * __log2f((P[0] * P[1]) * (P[2] * P[3]));
    }
    if (lane == 0) bulk_wait<0>();
    if constexpr (TOPK > 0) {
      const size_t o = (((size_t)blockIdx.x * C::NSET + set) * 128 + row) * 8;
#pragma unroll
      for (int i = 0; i < 8; ++i) { p.topk_val[o + i] = (valid_row && i < KL) ? tv[i < KL ? i : 0] : -INFINITY; p.topk_idx[o + i] = i < KL ? ti[i < KL ? i : 0] : -1; }
    }
    if (!valid_row) loss_local = 0.f;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) loss_local += __shfl_xor_sync(0xffffffffu, loss_local, o);
    if (lane == 0) loss_red[warp] = loss_local;
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

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
bool tc_tail_supported(const haste_config_t& cfg, int) {
  if (cfg.dtype != HASTE_BF16) return false;
  if (!(cfg.G == 8 || cfg.G == 16 || cfg.G == 32 || cfg.G == 64 || cfg.G == 128)) return false;
  if (!(cfg.K == 64 || cfg.K == 128)) return false;
  if (cfg.L < 1 || cfg.B_max > 128 * 2 * 128) return false;
  return true;
}

int tc_tail_create(TcTailState** out, const haste_config_t& cfg, int Bpad, int device) {
  TcTailState* s = new (std::nothrow) TcTailState();
  if (!s) return HASTE_ERR_NOMEM;
  s->cfg = cfg; s->device = device; s->Bpad = Bpad;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { delete s; set_error("cudaGetDeviceProperties failed"); return HASTE_ERR_CUDA; }
  if (prop.major != 10) { delete s; set_error("the tcgen05 kernel family needs an sm_100 device (found sm_%d%d)", prop.major, prop.minor); return HASTE_ERR_UNSUPPORTED; }
  s->num_sms = prop.multiProcessorCount;
  s->n_partials = s->num_sms;
  if (!get_encode_fn()) { delete s; set_error("cuTensorMapEncodeTiled is not available from the driver"); return HASTE_ERR_CUDA; }
  *out = s;
  return HASTE_OK;
}
void tc_tail_destroy(TcTailState* s) { delete s; }
int tc_tail_num_partials(const TcTailState* s) { return s->n_partials; }

template <int G, int K>
static int launch_fwd(TcTailState* s, const TailShape& sh, const void* Xt, const int32_t* idx, const void* W, const float* bias,
                      const int32_t* rowptr, const int32_t* col, float* partials, float* loss, void* dY, float* logits, int z_mode,
                      float* topk_val, int* topk_idx, TopkGeom* geom, cudaStream_t st) {
  using C = FwdCfg<G, K>;
  static_assert(C::SMEM <= 232448, "shared memory budget");
  CUtensorMap tmW, tmY;
  {
    const uint64_t dims[2] = {(uint64_t)K, (uint64_t)sh.L};
    const uint64_t str[1] = {(uint64_t)K * 2};
    const uint32_t box[2] = {64, (uint32_t)G};
    int rc = encode_tmap(&tmW, 2, W, 2, dims, str, box, 128);
    if (rc) return rc;
  }
  if (dY) {
    const uint64_t dims[3] = {(uint64_t)G, (uint64_t)sh.B, (uint64_t)sh.NG};
    const uint64_t str[2] = {(uint64_t)G * 2, (uint64_t)sh.B * G * 2};
    const uint32_t box[3] = {(uint32_t)std::min(G, 64), 32, 1};   // one epilogue warp's 32 rows
    int rc = encode_tmap(&tmY, 2, dY, 3, dims, str, box, G >= 64 ? 128 : G * 2);   // 16-byte rows (G = 8): no swizzle
    if (rc) return rc;
  } else {
    tmY = tmW;
  }
  FwdParams p;
  p.Xt = (const bf16*)Xt; p.idx = idx; p.bias = bias; p.rowptr = rowptr; p.col = col; p.partials = partials; p.loss = loss; p.logits = logits;
  p.write_dy = dY ? 1 : 0;
  p.z_mode = z_mode; p.topk_val = topk_val; p.topk_idx = topk_idx;
  p.B = sh.B; p.Bpad = sh.Bpad; p.NT = ceil_div(sh.B, 128); p.NP = (p.NT + 1) / 2;
  p.S = (int)std::min<int64_t>(sh.NG, std::max(1, s->num_sms / p.NP));
  p.L = sh.L; p.NG = sh.NG; p.label_offset = sh.label_offset; p.s = sh.s;
  if (p.NP > s->num_sms) { set_error("batch too large for the tcgen05 forward"); return HASTE_ERR_UNSUPPORTED; }
  const int grid = p.NP * p.S;
  const int topk_k = geom ? geom->k : 0;
  if (geom) { geom->NP = p.NP; geom->S = p.S; geom->NSET = C::NSET; }
  if (z_mode == 2 && topk_k <= 5) {
    HASTE_CUDA_TRY(cudaFuncSetAttribute(tc_fwd_kernel<G, K, 5>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM));
    HASTE_CUDA_TRY(launch_pdl(tc_fwd_kernel<G, K, 5>, dim3(grid), dim3(C::THREADS), C::SMEM, st, tmW, tmY, p));
  } else if (z_mode == 2) {
    HASTE_CUDA_TRY(cudaFuncSetAttribute(tc_fwd_kernel<G, K, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM));
    HASTE_CUDA_TRY(launch_pdl(tc_fwd_kernel<G, K, 8>, dim3(grid), dim3(C::THREADS), C::SMEM, st, tmW, tmY, p));
  } else if (z_mode == 1) {
    HASTE_CUDA_TRY(cudaFuncSetAttribute(tc_fwd_kernel<G, K, -1>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM));
    HASTE_CUDA_TRY(launch_pdl(tc_fwd_kernel<G, K, -1>, dim3(grid), dim3(C::THREADS), C::SMEM, st, tmW, tmY, p));
  } else {
    HASTE_CUDA_TRY(cudaFuncSetAttribute(tc_fwd_kernel<G, K, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM));
    HASTE_CUDA_TRY(launch_pdl(tc_fwd_kernel<G, K, 0>, dim3(grid), dim3(C::THREADS), C::SMEM, st, tmW, tmY, p));
  }
  HASTE_LAUNCH_CHECK();
  return HASTE_OK;
}

int tc_tail_forward(TcTailState* s, const TailShape& sh, const void* Xt, const int32_t* idx, const void* W, const float* bias,
                    const int32_t* rowptr, const int32_t* col, float* loss_partials, float* loss, void* dY, float* logits_out,
                    int z_mode, float* topk_val, int* topk_idx, TopkGeom* geom, cudaStream_t st, int* n_launches) {
  *n_launches = 1;
#define HASTE_FWD(G_, K_) \
  if (sh.G == G_ && sh.K == K_) return launch_fwd<G_, K_>(s, sh, Xt, idx, W, bias, rowptr, col, loss_partials, loss, dY, logits_out, z_mode, topk_val, topk_idx, geom, st)
  HASTE_FWD(64, 128); HASTE_FWD(64, 64); HASTE_FWD(32, 64); HASTE_FWD(32, 128); HASTE_FWD(128, 64); HASTE_FWD(128, 128);
  HASTE_FWD(16, 64); HASTE_FWD(16, 128); HASTE_FWD(8, 64); HASTE_FWD(8, 128);
#undef HASTE_FWD
  set_error("tcgen05 forward: unsupported (G, K)");
  return HASTE_ERR_UNSUPPORTED;
}

}  // namespace haste
