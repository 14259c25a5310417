// tc_head.cu -- tcgen05 / TMEM / TMA kernels of the dense head over the frequent labels.
//
// One warp-specialised persistent GEMM kernel, three instantiations (bf16 operands, fp32 accumulate in TMEM):
//   FWD  Z   [B x L_h] = X_h   [B x d]   * W_h^T            A K-major,  B K-major,  fused BCE epilogue (Eq. 3)
//   DW   dW_h[L_h x d] = dY_h^T[L_h x B] * X_h  [B x d]     A MN-major, B MN-major, bf16 rows out; db_h from one
//                                                           extra N=16 MMA per K-step against a tile of ones
//   DX   dX_h[B x d]   = dY_h  [B x L_h] * W_h  [L_h x d]   A K-major,  B MN-major, split over label slabs, partial
//                                                           tiles added with TMA reduce-add (fp32)
// Every operand is read in the layout it has in HBM: a transposed operand is an MN-major UMMA descriptor, not a copy.
// warp roles (192 threads): warps 0-3 epilogue (thread = accumulator row), warp 4 MMA issuer, warp 5 TMA loader.
#include <algorithm>
#include <cstdint>
#include <cstring>
#include <new>

#include "tc_common.cuh"
#include "tc_epilogue.cuh"
#include "tc_kernels.h"

namespace haste {
using namespace tc;

enum { HEAD_FWD = 0, HEAD_DW = 1, HEAD_DX = 2 };

struct HeadParams {
  int MT, NTL, NSLAB, KB;     // work items: MT x NTL output tiles x NSLAB contraction slabs; KB k-blocks of 64 in all
  int B, d;
  int64_t L, label_offset;
  const float* bias;
  const int32_t* rowptr;
  const int32_t* col;
  float* partials;            // FWD: [1024] per-CTA unscaled loss partials + ticket (finalize_loss_last_cta), or null
  float* loss;                // FWD: device scalar, written by the last CTA
  float* logits;              // FWD: [B][L] fp32 or null
  float* dbias;               // DW: [L] or null
  float4* zero;               // DW: a buffer this kernel zeroes on the side (the dX the next kernel reduces into), or null
  int64_t zero_n;             //     its length in float4
  int write_out;              // FWD: dY; DW: dW_h
  float s;
};

template <int MODE> struct HeadCfg {
  static constexpr bool A_MN = MODE == HEAD_DW;
  static constexpr bool B_MN = MODE != HEAD_FWD;
  static constexpr int BN = MODE == HEAD_FWD ? 128 : (MODE == HEAD_DW ? 192 : 256);
  static constexpr int A_BYTES = 16384;
  static constexpr int B_BYTES = BN * 128;
  static constexpr int STAGE = A_BYTES + B_BYTES;
  static constexpr int EPI_BUFS = MODE == HEAD_DX ? 1 : 2;
  static constexpr int EPI_BYTES = 4 * EPI_BUFS * 4096;
  static constexpr int NST = MODE == HEAD_FWD ? 5 : 4;
  static constexpr int TS = 256;                           // TMEM columns per accumulator slot (2 slots)
  static constexpr int OFF_EPI = NST * STAGE;
  static constexpr int OFF_ONES = OFF_EPI + EPI_BYTES;     // [16 rows][128 B] of bf16 1.0 (DW: db)
  static constexpr int OFF_BIAS = OFF_ONES + 2048;         // [4 warps][128] fp32 (FWD)
  static constexpr int OFF_BAR = OFF_BIAS + 2048;
  static constexpr int OFF_MISC = OFF_BAR + (2 * NST + 4) * 8;
  static constexpr int SMEM = OFF_MISC + 64 + 1024;
};

__device__ __forceinline__ void tma_reduce_add_2d(const CUtensorMap* m, const void* src, int c0, int c1) {
  asm volatile("cp.reduce.async.bulk.tensor.2d.global.shared::cta.add.tile.bulk_group [%0, {%2, %3}], [%1];"
               ::"l"(reinterpret_cast<uint64_t>(m)), "r"(smem_u32(src)), "r"(c0), "r"(c1)
               : "memory");
}
__device__ __forceinline__ uint32_t head_tmem_ld1(uint32_t taddr) {
  uint32_t v;
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(v) : "r"(taddr) : "memory");
  return v;
}

// work item w -> (m tile, n tile, k-block range)
struct HeadItem { int mt, nt, kb0, kb1; };
__device__ __forceinline__ HeadItem head_item(const HeadParams& p, int w) {
  HeadItem it;
  it.mt = w % p.MT;
  const int r = w / p.MT;
  it.nt = r % p.NTL;
  const int slab = r / p.NTL;
  it.kb0 = (int)((int64_t)p.KB * slab / p.NSLAB);
  it.kb1 = (int)((int64_t)p.KB * (slab + 1) / p.NSLAB);
  return it;
}

template <int MODE>
__global__ void __launch_bounds__(192, 1)
tc_head_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
               const __grid_constant__ CUtensorMap tmO, const HeadParams p) {
  using C = HeadCfg<MODE>;
  constexpr int BN = C::BN;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const uint32_t sbase = smem_u32(smem);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::OFF_BAR);
  uint64_t* full = bars;                    // [NST] count 1 + tx
  uint64_t* empty = bars + C::NST;          // [NST] count 1 (umma commit)
  uint64_t* t_full = bars + 2 * C::NST;     // [2]
  uint64_t* t_empty = t_full + 2;           // [2] count 4
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + C::OFF_MISC);
  float* loss_red = reinterpret_cast<float*>(smem + C::OFF_MISC + 16);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_items = p.MT * p.NTL * p.NSLAB;

  if (threadIdx.x == 0) {
    for (int i = 0; i < C::NST; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&t_full[i], 1); mbar_init(&t_empty[i], 4); }
    fence_barrier_init();
  }
  if (MODE == HEAD_DW) {
    for (int e = threadIdx.x; e < 128; e += blockDim.x)
      sts128(sbase + C::OFF_ONES + e * 16, 0x3F803F80u, 0x3F803F80u, 0x3F803F80u, 0x3F803F80u);
    fence_proxy_async_smem();
  }
  if (warp == 5 && lane == 0) { tma_prefetch_desc(&tmA); tma_prefetch_desc(&tmB); tma_prefetch_desc(&tmO); }
  if (warp == 4) tmem_alloc<512>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  pdl_wait();       // nothing above touches global memory (common.cuh, PDL)
  pdl_trigger();
  if (MODE == HEAD_DW && p.zero) {      // no memset between this kernel and the dX kernel that follows it (PDL chain)
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < p.zero_n; e += (int64_t)gridDim.x * blockDim.x)
      p.zero[e] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 5) {
    // ===================== TMA loader =====================
    if (lane == 0) {
      int it = 0;
      for (int w = blockIdx.x; w < n_items; w += gridDim.x) {
        const HeadItem wi = head_item(p, w);
        for (int kb = wi.kb0; kb < wi.kb1; ++kb, ++it) {
          const int st = it % C::NST;
          mbar_wait(&empty[st], ((it / C::NST) & 1) ^ 1);
          mbar_arrive_expect_tx(&full[st], C::STAGE);
          uint8_t* a = smem + st * C::STAGE;
          uint8_t* b = a + C::A_BYTES;
          if (C::A_MN) {
            tma_load_2d(a, &tmA, &full[st], wi.mt * 128, kb * 64);
            tma_load_2d(a + 8192, &tmA, &full[st], wi.mt * 128 + 64, kb * 64);
          } else {
            tma_load_2d(a, &tmA, &full[st], kb * 64, wi.mt * 128);
          }
          if (C::B_MN) {
#pragma unroll
            for (int c = 0; c < BN / 64; ++c) tma_load_2d(b + c * 8192, &tmB, &full[st], wi.nt * BN + c * 64, kb * 64);
          } else {
            tma_load_2d(b, &tmB, &full[st], kb * 64, wi.nt * BN);
          }
        }
      }
    }
  } else if (warp == 4) {
    // ===================== MMA issuer =====================
    // whole warp waits, one elected lane issues; descriptors are a per-stage base + compile-time offsets (see tc_tail.cu)
    constexpr uint32_t idesc = make_idesc_bf16(128, BN, C::A_MN ? 1 : 0, C::B_MN ? 1 : 0);
    constexpr uint32_t idesc_ones = make_idesc_bf16(128, 16, 1, 0);
    const uint64_t adesc0 = C::A_MN ? make_sdesc_sw128(sbase, 8192, 1024) : make_sdesc_sw128(sbase, 16, 1024);
    const uint64_t bdesc0 = C::B_MN ? make_sdesc_sw128(sbase + C::A_BYTES, 8192, 1024) : make_sdesc_sw128(sbase + C::A_BYTES, 16, 1024);
    const uint64_t odesc = make_sdesc_sw128(sbase + C::OFF_ONES, 16, 1024);
    int it = 0, n = 0;
    for (int w = blockIdx.x; w < n_items; w += gridDim.x) {
      const HeadItem wi = head_item(p, w);
      if (wi.kb1 <= wi.kb0) continue;
      const int slot = n & 1;
      mbar_wait(&t_empty[slot], ((n >> 1) & 1) ^ 1);
      tc_fence_after();
      const uint32_t dcol = tmem_base + slot * C::TS;
      const bool with_db = MODE == HEAD_DW && p.dbias != nullptr && wi.nt == 0;
      for (int kb = wi.kb0; kb < wi.kb1; ++kb, ++it) {
        const int st = it % C::NST;
        mbar_wait(&full[st], (it / C::NST) & 1);
        tc_fence_after();
        if (elect_one()) {
          const uint64_t so = (uint64_t)((st * C::STAGE) >> 4);
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const uint64_t ad = adesc0 + so + (uint64_t)((C::A_MN ? j * 2048 : j * 32) >> 4);
            const uint64_t bd = bdesc0 + so + (uint64_t)((C::B_MN ? j * 2048 : j * 32) >> 4);
            const uint32_t acc = (kb > wi.kb0 || j > 0) ? 1u : 0u;
            umma_f16(dcol, ad, bd, idesc, acc);
            if (with_db) umma_f16(dcol + BN, ad, odesc, idesc_ones, acc);
          }
          umma_commit(&empty[st]);
          if (kb == wi.kb1 - 1) umma_commit(&t_full[slot]);
        }
        __syncwarp();
      }
      ++n;
    }
  } else {
    // ===================== epilogue (thread = accumulator row) =====================
    const int q = warp;
    const uint32_t swz = (uint32_t)(lane & 7);
    const uint32_t sbuf0 = sbase + C::OFF_EPI + q * (C::EPI_BUFS * 4096);
    uint8_t* sbuf0_ptr = smem + C::OFF_EPI + q * (C::EPI_BUFS * 4096);
    const uint32_t sbias_w = sbase + C::OFF_BIAS + q * 512;
    float loss_local = 0.f;
    int n = 0, nstore = 0;
    int cur_row = -1, cur_n0 = 0, pc = 0, pe = 0;             // CSR cursor of the forward epilogue
    int64_t nxt = INT64_MAX;
    for (int w = blockIdx.x; w < n_items; w += gridDim.x) {
      const HeadItem wi = head_item(p, w);
      if (wi.kb1 <= wi.kb0) continue;
      const int slot = n & 1;
      const int row = wi.mt * 128 + q * 32 + lane;             // global accumulator row
      const int n0 = wi.nt * BN;
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + slot * C::TS;

      if (MODE == HEAD_FWD) {
        const bool valid_row = row < p.B;
        // positives of this row inside the tile.  A CTA's tiles keep their m tile (grid % MT == 0) and move up in n, so the
        // thread keeps a cursor into its CSR row (sorted columns) instead of re-scanning the row for every tile (that
        // scan, one dependent load per positive, was 15 of the kernel's 42 us); any other tile order resets the cursor.
        uint32_t ym[4] = {0u, 0u, 0u, 0u};
        if (valid_row && p.rowptr) {
          if (row != cur_row || n0 < cur_n0) {
            cur_row = row;
            pc = __ldg(p.rowptr + row); pe = __ldg(p.rowptr + row + 1);
            nxt = pc < pe ? (int64_t)__ldg(p.col + pc) - p.label_offset : INT64_MAX;
          }
          cur_n0 = n0;
          const int64_t hi = min((int64_t)n0 + BN, p.L);
          while (nxt < hi) {
            const int64_t o = nxt - n0;
            if (o >= 0) {
#pragma unroll
              for (int i = 0; i < 4; ++i) if ((int)(o >> 5) == i) ym[i] |= 1u << (o & 31);
            }
            ++pc;
            nxt = pc < pe ? (int64_t)__ldg(p.col + pc) - p.label_offset : INT64_MAX;
          }
        }
        const int nl = (int)min((int64_t)BN, p.L - n0);
        const bool slow = __any_sync(0xffffffffu, (ym[0] | ym[1] | ym[2] | ym[3]) != 0) || nl < BN || p.logits != nullptr;
        if (p.bias) {
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int l = i * 32 + lane;
            sts32(sbias_w + l * 4, __float_as_uint(l < nl ? __ldg(p.bias + n0 + l) : 0.f));
          }
        }
        __syncwarp();
        mbar_wait(&t_full[slot], (n >> 1) & 1);
        tc_fence_after();
        const float hs = 0.5f * p.s;
        float R[4] = {0.f, 0.f, 0.f, 0.f}, P[4] = {1.f, 1.f, 1.f, 1.f};
        float lt = 0.f;
#pragma unroll 1                 // one copy of the epilogue code: unrolled four times it overflows the instruction cache
        for (int sc = 0; sc < 4; ++sc) {
          uint32_t v[32];
          const uint32_t ymsc = sc == 0 ? ym[0] : sc == 1 ? ym[1] : sc == 2 ? ym[2] : ym[3];
          tmem_ld32(taddr + sc * 32, v);
          tmem_ld_wait();
          uint32_t out[16];
          float* zout = (p.logits && valid_row) ? p.logits + (size_t)row * p.L + n0 + sc * 32 : nullptr;
          const uint32_t sb = sbias_w + sc * 128;
          if (slow) {
            if (p.bias) epi32<true, true>(v, sb, ymsc, nl - sc * 32, p.s, hs, R, P, out, zout);
            else epi32<true, false>(v, sb, ymsc, nl - sc * 32, p.s, hs, R, P, out, zout);
          } else {
            if (p.bias) epi32<false, true>(v, sb, 0u, 32, p.s, hs, R, P, out, nullptr);
            else epi32<false, false>(v, sb, 0u, 32, p.s, hs, R, P, out, nullptr);
          }
          if (sc & 1) {
            lt += (R[0] + R[1]) + (R[2] + R[3]) - 0.69314718056f * __log2f((P[0] * P[1]) * (P[2] * P[3]));
#pragma unroll
            for (int i = 0; i < 4; ++i) { R[i] = 0.f; P[i] = 1.f; }
          }
          if (p.write_out) {
            const uint32_t sbuf = sbuf0 + (nstore & 1) * 4096;
            if ((sc & 1) == 0) {
              if (lane == 0) bulk_wait_read<1>();
              __syncwarp();
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const uint32_t ch = (uint32_t)((sc & 1) * 4 + i) ^ swz;
              sts128(sbuf + lane * 128 + ch * 16, out[4 * i], out[4 * i + 1], out[4 * i + 2], out[4 * i + 3]);
            }
            if (sc & 1) {
              fence_proxy_async_smem();
              __syncwarp();
              if (lane == 0) {
                tma_store_2d(&tmO, sbuf0_ptr + (nstore & 1) * 4096, n0 + (sc >> 1) * 64, wi.mt * 128 + q * 32);
                bulk_commit();
              }
              ++nstore;
            }
          }
        }
        if (valid_row) loss_local += lt;
      } else {
        mbar_wait(&t_full[slot], (n >> 1) & 1);
        tc_fence_after();
        constexpr int NBOX = MODE == HEAD_DW ? BN / 64 : BN / 32;
#pragma unroll 1
        for (int c = 0; c < NBOX; ++c) {
          uint32_t out[32];
          if (MODE == HEAD_DX) {
            tmem_ld32(taddr + c * 32, out);
            tmem_ld_wait();
          } else {
            uint32_t v0[32], v1[32];
            tmem_ld32(taddr + c * 64, v0);
            tmem_ld32(taddr + c * 64 + 32, v1);
            tmem_ld_wait();
#pragma unroll
            for (int j = 0; j < 16; ++j) {
              out[j] = pack_bf16x2(__uint_as_float(v0[2 * j]), __uint_as_float(v0[2 * j + 1]));
              out[16 + j] = pack_bf16x2(__uint_as_float(v1[2 * j]), __uint_as_float(v1[2 * j + 1]));
            }
          }
          const int c0 = n0 + c * (MODE == HEAD_DW ? 64 : 32);
          if (c0 >= p.d || (MODE == HEAD_DW && !p.write_out)) continue;     // warp-uniform
          const int bi = C::EPI_BUFS == 2 ? (nstore & 1) : 0;
          if (lane == 0) { if (C::EPI_BUFS == 2) bulk_wait_read<1>(); else bulk_wait_read<0>(); }
          __syncwarp();
#pragma unroll
          for (int ch = 0; ch < 8; ++ch)
            sts128(sbuf0 + bi * 4096 + lane * 128 + ((ch ^ swz) << 4), out[4 * ch], out[4 * ch + 1], out[4 * ch + 2], out[4 * ch + 3]);
          fence_proxy_async_smem();
          __syncwarp();
          if (lane == 0) {
            if (MODE == HEAD_DW) tma_store_2d(&tmO, sbuf0_ptr + bi * 4096, c0, wi.mt * 128 + q * 32);
            else tma_reduce_add_2d(&tmO, sbuf0_ptr + bi * 4096, c0, wi.mt * 128 + q * 32);
            bulk_commit();
          }
          ++nstore;
        }
        if (MODE == HEAD_DW && p.dbias && wi.nt == 0) {
          const uint32_t v = head_tmem_ld1(taddr + BN);
          tmem_ld_wait();
          if (row < p.L) p.dbias[row] = __uint_as_float(v);
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&t_empty[slot]);
      ++n;
    }
    if (lane == 0) bulk_wait<0>();
    if (MODE == HEAD_FWD) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) loss_local += __shfl_xor_sync(0xffffffffu, loss_local, o);
      if (lane == 0) loss_red[warp] = loss_local;
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 4) { tc_fence_after(); tmem_dealloc<512>(tmem_base); }
  if (MODE == HEAD_FWD && p.partials)
    finalize_loss_last_cta(p.partials, threadIdx.x == 0 ? (loss_red[0] + loss_red[1]) + (loss_red[2] + loss_red[3]) : 0.f, p.s, p.loss);
}

// ---------------------------------------------------------------------------------------------
// Forward with 256 x 256 output tiles (two M = 128 accumulators of N = 256: all 512 TMEM columns), for batches of more
// than 128 rows.  Why: with 128 x 128 tiles the kernel is bound by its operand traffic through L2 (201 MB at config 3,
// 23 of its 27 us) and by 3.46 waves of tiles on 148 SMs.  A 256 x 256 tile moves 64 KB per k-block for four times the
// MMA work (98 MB in all), config 3 becomes ONE wave of 128 tiles, and the MMA phase of a tile (96 MMAs of 128 cycles)
// is as long as its loads.  There is one accumulator set, so a CTA's epilogue does not overlap its next tile's MMAs: with
// one tile per CTA nothing is lost.  The CSR scan of the thread's two rows runs before the accumulators are waited for.
// warp roles (576 threads): warps 0-15 epilogue (warp w: TMEM lane quadrant w & 3, M tile (w >> 2) & 1, 128-label half
// w >> 3; four per scheduler, because one warp's chunk is a latency chain: 8 warps took 14.8 k cycles, the MMA phase 16 k),
// warp 16 MMA, warp 17 TMA.
// ---------------------------------------------------------------------------------------------
struct Fwd256Cfg {
  static constexpr int BN = 256, NST = 3;
  static constexpr int A_BYTES = 32768, B_BYTES = 32768, STAGE = A_BYTES + B_BYTES;
  static constexpr int NEW = 16;                            // epilogue warps
  static constexpr int OFF_EPI = 0;                         // [16 warps][2 buffers][32 rows][128 B] OVER the operand stages: a
                                                            // tile's epilogue starts when its last MMA has read them, and the
                                                            // loader waits for the epilogue before it loads the next tile
  static constexpr int OFF_BIAS = NST * STAGE;              // [256] fp32, one copy per CTA
  static constexpr int OFF_BAR = OFF_BIAS + 1024;
  static constexpr int OFF_MISC = OFF_BAR + (2 * NST + 2) * 8;
  static constexpr int SMEM = OFF_MISC + 128 + 1024;
  static constexpr int THREADS = (NEW + 2) * 32;
};

__global__ void __launch_bounds__(Fwd256Cfg::THREADS, 1)
tc_head_fwd256_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                      const __grid_constant__ CUtensorMap tmO, const HeadParams p) {
  using C = Fwd256Cfg;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const uint32_t sbase = smem_u32(smem);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::OFF_BAR);
  uint64_t* full = bars;                    // [NST] count 1 + tx
  uint64_t* empty = bars + C::NST;          // [NST] count 1 (umma commit)
  uint64_t* t_full = bars + 2 * C::NST;     // count 1
  uint64_t* t_empty = t_full + 1;           // count 16: accumulators AND staging (= operand stages) free again
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + C::OFF_MISC);
  float* loss_red = reinterpret_cast<float*>(smem + C::OFF_MISC + 16);   // [16]

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_items = p.MT * p.NTL;         // MT = tiles of 256 rows, NTL = tiles of 256 labels

  if (threadIdx.x == 0) {
    for (int i = 0; i < C::NST; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], 1); }
    mbar_init(t_full, 1); mbar_init(t_empty, C::NEW);
    fence_barrier_init();
  }
  if (warp == C::NEW + 1 && lane == 0) { tma_prefetch_desc(&tmA); tma_prefetch_desc(&tmB); tma_prefetch_desc(&tmO); }
  if (warp == C::NEW) tmem_alloc<512>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  pdl_wait();       // nothing above touches global memory (common.cuh, PDL)
  pdl_trigger();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == C::NEW + 1) {
    if (lane == 0) {
      int it = 0, n = 0;
      for (int w = blockIdx.x; w < n_items; w += gridDim.x, ++n) {
        const int mt = w % p.MT, nt = w / p.MT;
        mbar_wait(t_empty, (n & 1) ^ 1);       // the previous tile's epilogue has left the staging rows (they overlay the stages)
        for (int kb = 0; kb < p.KB; ++kb, ++it) {
          const int st = it % C::NST;
          mbar_wait(&empty[st], ((it / C::NST) & 1) ^ 1);
          mbar_arrive_expect_tx(&full[st], C::STAGE);
          uint8_t* a = smem + st * C::STAGE;
          tma_load_2d(a, &tmA, &full[st], kb * 64, mt * 256);                    // box {64, 256}: both M tiles
          tma_load_2d(a + C::A_BYTES, &tmB, &full[st], kb * 64, nt * 256);       // box {64, 256}
        }
      }
    }
  } else if (warp == C::NEW) {
    constexpr uint32_t idesc = make_idesc_bf16(128, 256, 0, 0);
    const uint64_t adesc0 = make_sdesc_sw128(sbase, 16, 1024);
    const uint64_t bdesc0 = make_sdesc_sw128(sbase + C::A_BYTES, 16, 1024);
    int it = 0, n = 0;
    for (int w = blockIdx.x; w < n_items; w += gridDim.x, ++n) {
      mbar_wait(t_empty, (n & 1) ^ 1);
      tc_fence_after();
      for (int kb = 0; kb < p.KB; ++kb, ++it) {
        const int st = it % C::NST;
        mbar_wait(&full[st], (it / C::NST) & 1);
        tc_fence_after();
        if (elect_one()) {
          const uint64_t so = (uint64_t)((st * C::STAGE) >> 4);
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const uint32_t acc = (kb > 0 || j > 0) ? 1u : 0u;
            const uint64_t bd = bdesc0 + so + (uint64_t)((j * 32) >> 4);
            umma_f16(tmem_base, adesc0 + so + (uint64_t)((j * 32) >> 4), bd, idesc, acc);
            umma_f16(tmem_base + 256, adesc0 + so + (uint64_t)((16384 + j * 32) >> 4), bd, idesc, acc);
          }
          umma_commit(&empty[st]);
          if (kb == p.KB - 1) umma_commit(t_full);
        }
        __syncwarp();
      }
    }
  } else {
    const int q = warp & 3, tile = (warp >> 2) & 1, half = warp >> 3;
    const uint32_t swz = (uint32_t)(lane & 7);
    const uint32_t sbuf0 = sbase + C::OFF_EPI + warp * 8192;
    uint8_t* sbuf0_ptr = smem + C::OFF_EPI + warp * 8192;
    int nstore = 0;
    const uint32_t sbias = sbase + C::OFF_BIAS;
    const float hs = 0.5f * p.s;
    float loss_local = 0.f;
    int n = 0;
    for (int w = blockIdx.x; w < n_items; w += gridDim.x, ++n) {
      const int mt = w % p.MT, nt = w / p.MT;
      const int row = mt * 256 + tile * 128 + q * 32 + lane;
      const int n0 = nt * 256;
      const bool valid_row = row < p.B;
      const int nl = (int)min((int64_t)256, p.L - n0);
      // positives of this row inside the tile's 256 labels: binary search for the first column >= n0, then walk
      uint32_t ym[4] = {0u, 0u, 0u, 0u};          // this warp's four 32-label chunks: labels n0 + half * 128 ...
      if (valid_row && p.rowptr) {
        int lo = __ldg(p.rowptr + row);
        const int pe = __ldg(p.rowptr + row + 1);
        int hi = pe;
        const int64_t want = (int64_t)n0 + half * 128 + p.label_offset;
        while (lo < hi) {
          const int mid = (lo + hi) >> 1;
          if ((int64_t)__ldg(p.col + mid) < want) lo = mid + 1; else hi = mid;
        }
        for (int pc = lo; pc < pe; ++pc) {
          const int64_t o = (int64_t)__ldg(p.col + pc) - want;
          if (o >= min(128, nl - half * 128)) break;
#pragma unroll
          for (int i = 0; i < 4; ++i) if ((int)(o >> 5) == i) ym[i] |= 1u << (o & 31);
        }
      }
      uint32_t anyy = ym[0] | ym[1] | ym[2] | ym[3];
      const bool slow = __any_sync(0xffffffffu, anyy != 0) || nl < 256 || p.logits != nullptr;
      if (p.bias) {           // one copy per CTA: epilogue warps 0-7 fill 32 labels each, then all meet at a named barrier
        const int l = warp * 32 + lane;
        if (warp < 8) sts32(sbias + l * 4, __float_as_uint(l < nl ? __ldg(p.bias + n0 + l) : 0.f));
        named_bar_sync(1, C::NEW * 32);
      }
      mbar_wait(t_full, n & 1);
      tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + tile * 256 + half * 128;
      const int nlh = nl - half * 128;                  // valid labels of this warp's half (may be <= 0)
      float R[4] = {0.f, 0.f, 0.f, 0.f}, P[4] = {1.f, 1.f, 1.f, 1.f};
      float lt = 0.f;
#pragma unroll 1                 // one copy of the epilogue code (instruction cache)
      for (int sc = 0; sc < 4; ++sc) {
        uint32_t v[32];
        const uint32_t ymsc = sc == 0 ? ym[0] : sc == 1 ? ym[1] : sc == 2 ? ym[2] : ym[3];
        tmem_ld32(taddr + sc * 32, v);
        tmem_ld_wait();
        uint32_t out[16];
        float* zout = (p.logits && valid_row) ? p.logits + (size_t)row * p.L + n0 + half * 128 + sc * 32 : nullptr;
        const uint32_t sb = sbias + half * 512 + sc * 128;
        if (slow) {
          if (p.bias) epi32<true, true>(v, sb, ymsc, nlh - sc * 32, p.s, hs, R, P, out, zout);
          else epi32<true, false>(v, sb, ymsc, nlh - sc * 32, p.s, hs, R, P, out, zout);
        } else {
          if (p.bias) epi32<false, true>(v, sb, 0u, 32, p.s, hs, R, P, out, nullptr);
          else epi32<false, false>(v, sb, 0u, 32, p.s, hs, R, P, out, nullptr);
        }
        if (sc & 1) {
          lt += (R[0] + R[1]) + (R[2] + R[3]) - 0.69314718056f * __log2f((P[0] * P[1]) * (P[2] * P[3]));
#pragma unroll
          for (int i = 0; i < 4; ++i) { R[i] = 0.f; P[i] = 1.f; }
        }
        if (p.write_out) {
          const uint32_t sbuf = sbuf0 + (nstore & 1) * 4096;     // two staging buffers: one TMA store may still be reading
          if ((sc & 1) == 0) {
            if (lane == 0) bulk_wait_read<1>();
            __syncwarp();
          }
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const uint32_t ch = (uint32_t)((sc & 1) * 4 + i) ^ swz;
            sts128(sbuf + lane * 128 + ch * 16, out[4 * i], out[4 * i + 1], out[4 * i + 2], out[4 * i + 3]);
          }
          if (sc & 1) {
            fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) {
              tma_store_2d(&tmO, sbuf0_ptr + (nstore & 1) * 4096, n0 + half * 128 + (sc >> 1) * 64, mt * 256 + tile * 128 + q * 32);
              bulk_commit();
            }
            ++nstore;
          }
        }
      }
      if (valid_row) loss_local += lt;
      if (lane == 0) bulk_wait_read<0>();      // this warp's TMA stores have read the staging rows: the loader may overwrite them
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(t_empty);
      if (p.bias) named_bar_sync(1, C::NEW * 32);      // the bias copy is not refilled before every warp has used it
    }
    if (lane == 0) bulk_wait<0>();
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) loss_local += __shfl_xor_sync(0xffffffffu, loss_local, o);
    if (lane == 0) loss_red[warp] = loss_local;
  }

  tc_fence_before();
  __syncthreads();
  if (warp == C::NEW) { tc_fence_after(); tmem_dealloc<512>(tmem_base); }
  if (p.partials) {
    float t = 0.f;
    if (threadIdx.x == 0) {
#pragma unroll
      for (int i = 0; i < C::NEW; ++i) t += loss_red[i];
    }
    finalize_loss_last_cta(p.partials, t, p.s, p.loss);
  }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
struct TcHeadState {
  int d, B_max, device, num_sms, n_partials;
  int64_t L;
};

bool tc_head_supported(int d, int64_t L_h, int, haste_dtype_t dtype, int) {
  return dtype == HASTE_BF16 && d >= 8 && d % 8 == 0 && L_h >= 8 && L_h % 8 == 0 && L_h <= 0x7fffff00LL;
}

int tc_head_create(TcHeadState** out, int d, int64_t L_h, int B_max, int device) {
  TcHeadState* s = new (std::nothrow) TcHeadState();
  if (!s) return HASTE_ERR_NOMEM;
  s->d = d; s->L = L_h; s->B_max = B_max; s->device = device;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { delete s; set_error("cudaGetDeviceProperties failed"); return HASTE_ERR_CUDA; }
  if (prop.major != 10) { delete s; set_error("the tcgen05 kernel family needs an sm_100 device (found sm_%d%d)", prop.major, prop.minor); return HASTE_ERR_UNSUPPORTED; }
  s->num_sms = prop.multiProcessorCount;
  s->n_partials = s->num_sms;
  *out = s;
  return HASTE_OK;
}
void tc_head_destroy(TcHeadState* s) { delete s; }
int tc_head_num_partials(const TcHeadState* s) { return s->n_partials; }

static int map2d(CUtensorMap* m, int es, const void* base, uint64_t inner, uint64_t outer, uint32_t box0, uint32_t box1) {
  const uint64_t dims[2] = {inner, outer};
  const uint64_t str[1] = {inner * (uint64_t)es};
  const uint32_t box[2] = {box0, box1};
  return encode_tmap(m, es, base, 2, dims, str, box, 128);
}

template <int MODE>
static int launch_head(TcHeadState* s, const CUtensorMap& tmA, const CUtensorMap& tmB, const CUtensorMap& tmO, const HeadParams& p,
                       cudaStream_t st) {
  using C = HeadCfg<MODE>;
  static_assert(C::SMEM <= 232448, "shared memory budget");
  const int n_items = p.MT * p.NTL * p.NSLAB;
  const int grid = std::min(n_items, s->num_sms);
  HASTE_CUDA_TRY(cudaFuncSetAttribute(tc_head_kernel<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM));
  HASTE_CUDA_TRY(launch_pdl(tc_head_kernel<MODE>, dim3(grid), dim3(192), C::SMEM, st, tmA, tmB, tmO, p));
  HASTE_LAUNCH_CHECK();
  return HASTE_OK;
}

static HeadParams base_params(const HeadShape& sh) {
  HeadParams p;
  memset(&p, 0, sizeof(p));
  p.B = sh.B; p.d = sh.d; p.L = sh.L; p.label_offset = sh.label_offset; p.s = sh.s;
  p.NSLAB = 1;
  return p;
}

int tc_head_forward(TcHeadState* s, const HeadShape& sh, const void* X, const void* Wh, const float* bias,
                    const int32_t* rowptr, const int32_t* col, float* loss_partials, float* loss, void* dY, float* logits_out,
                    cudaStream_t st, int* n_launches) {
  *n_launches = 1;
  CUtensorMap tmA, tmB, tmO;
  if (sh.B > 128) {     // 256 x 256 tiles (tc_head_fwd256_kernel)
    int rc = map2d(&tmA, 2, X, sh.d, sh.B, 64, 256);
    if (!rc) rc = map2d(&tmB, 2, Wh, sh.d, sh.L, 64, 256);
    if (!rc) { if (dY) rc = map2d(&tmO, 2, dY, sh.L, sh.B, 64, 32); else tmO = tmA; }
    if (rc) return rc;
    HeadParams p = base_params(sh);
    p.MT = ceil_div(sh.B, 256); p.NTL = ceil_div(sh.L, 256); p.KB = ceil_div(sh.d, 64);
    p.bias = bias; p.rowptr = rowptr; p.col = col; p.partials = loss_partials; p.loss = loss; p.logits = logits_out; p.write_out = dY ? 1 : 0;
    const int grid = std::min(p.MT * p.NTL, s->num_sms);
    static_assert(Fwd256Cfg::SMEM <= 232448, "shared memory budget");
    HASTE_CUDA_TRY(cudaFuncSetAttribute(tc_head_fwd256_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, Fwd256Cfg::SMEM));
    HASTE_CUDA_TRY(launch_pdl(tc_head_fwd256_kernel, dim3(grid), dim3(Fwd256Cfg::THREADS), Fwd256Cfg::SMEM, st, tmA, tmB, tmO, p));
    HASTE_LAUNCH_CHECK();
    return HASTE_OK;
  }
  int rc = map2d(&tmA, 2, X, sh.d, sh.B, 64, 128);
  if (!rc) rc = map2d(&tmB, 2, Wh, sh.d, sh.L, 64, 128);
  if (!rc) { if (dY) rc = map2d(&tmO, 2, dY, sh.L, sh.B, 64, 32); else tmO = tmA; }
  if (rc) return rc;
  HeadParams p = base_params(sh);
  p.MT = ceil_div(sh.B, 128); p.NTL = ceil_div(sh.L, HeadCfg<HEAD_FWD>::BN); p.KB = ceil_div(sh.d, 64);
  p.bias = bias; p.rowptr = rowptr; p.col = col; p.partials = loss_partials; p.loss = loss; p.logits = logits_out; p.write_out = dY ? 1 : 0;
  return launch_head<HEAD_FWD>(s, tmA, tmB, tmO, p, st);
}

int tc_head_backward(TcHeadState* s, const HeadShape& sh, const void* X, const void* Wh, const void* dY, void* dWh,
                     float* dbias, float* dX, int accumulate_dX, int deterministic, cudaStream_t st, int* n_launches) {
  *n_launches = 0;
  bool dx_zeroed = false;
  if (dWh || dbias) {
    CUtensorMap tmA, tmB, tmO;
    int rc = map2d(&tmA, 2, dY, sh.L, sh.B, 64, 64);
    if (!rc) rc = map2d(&tmB, 2, X, sh.d, sh.B, 64, 64);
    if (!rc) { if (dWh) rc = map2d(&tmO, 2, dWh, sh.d, sh.L, 64, 32); else tmO = tmA; }
    if (rc) return rc;
    HeadParams p = base_params(sh);
    p.MT = ceil_div(sh.L, 128); p.NTL = dWh ? ceil_div(sh.d, HeadCfg<HEAD_DW>::BN) : 1; p.KB = ceil_div(sh.B, 64);
    p.dbias = dbias; p.write_out = dWh ? 1 : 0;
    if (dX && !accumulate_dX && ((size_t)sh.B * sh.d) % 4 == 0 && (reinterpret_cast<uintptr_t>(dX) & 15u) == 0) {      // the dW kernel zeroes dX for the dX kernel
      p.zero = reinterpret_cast<float4*>(dX); p.zero_n = (int64_t)sh.B * sh.d / 4;
      dx_zeroed = true;
    }
    rc = launch_head<HEAD_DW>(s, tmA, tmB, tmO, p, st);
    if (rc) return rc;
    ++*n_launches;
  }
  if (dX) {
    if (!accumulate_dX && !dx_zeroed) HASTE_CUDA_TRY(cudaMemsetAsync(dX, 0, (size_t)sh.B * sh.d * sizeof(float), st));
    CUtensorMap tmA, tmB, tmO;
    int rc = map2d(&tmA, 2, dY, sh.L, sh.B, 64, 128);
    if (!rc) rc = map2d(&tmB, 2, Wh, sh.d, sh.L, 64, 64);
    if (!rc) rc = map2d(&tmO, 4, dX, sh.d, sh.B, 32, 32);
    if (rc) return rc;
    HeadParams p = base_params(sh);
    p.MT = ceil_div(sh.B, 128); p.NTL = ceil_div(sh.d, HeadCfg<HEAD_DX>::BN); p.KB = ceil_div(sh.L, 64);
    // split over label slabs, partial tiles added with cp.reduce (float atomics): one slab when determinism is asked for
    p.NSLAB = deterministic ? 1 : std::max(1, std::min(p.KB, s->num_sms / (p.MT * p.NTL)));
    rc = launch_head<HEAD_DX>(s, tmA, tmB, tmO, p, st);
    if (rc) return rc;
    ++*n_launches;
  }
  return HASTE_OK;
}

}  // namespace haste
