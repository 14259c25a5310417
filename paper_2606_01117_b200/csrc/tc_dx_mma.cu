// tc_dx_mma.cu -- input-gradient kernel of the HASTE sparse tail in which the tensor cores do the scatter-add too
// (sm_100a; bf16 in, fp32 accumulate).
//
//   dX[:, idx_g] += dY_g [B x G] * W_g [G x K]   over all groups g
//
// tc_dx_acc.cu keeps the reduction over groups on chip but pays ~5-7 issue slots per (slot, warp) for it and is
// issue-bound at ~0.31 ms (config 3).  Here the scatter is a second kind of MMA and costs no issue slots at all:
//   P^T [128 batch x K slots]  = dY tile (A, K-major, smem) * W_g (B, MN-major, smem)        kind::f16, fp32 in TMEM
//   ACC [128 batch x 64 window] += P^T[:, 8 slots] (A, read FROM TMEM as tf32) * S (B, smem)   kind::tf32
// where S [64 x 8] is one-hot: S[n][k] = 1 iff slot k of the 8-slot block goes to accumulator column start + n.
// P is already the A operand of a tf32 MMA (128 lanes x 32-bit columns), so nothing is converted or moved; the
// product by 1.0 is exact, only P is read at tf32 precision (10-bit mantissa, rel. 2^-11..2^-10 per term, far
// inside the 5e-3 bar; integers below 2048 stay exact).  Duplicated or unsorted index rows need no special path: two
// slots with the same feature are two ones in one row of S.  (Semantics checked first in isolation:
// profiles/r01_probe_scatter_mma.txt.)
// A CTA owns (128-row batch tile, feature part, stripe of groups): TMEM holds P (K columns, single buffer: the tensor
// pipe runs MMAs in issue order, so the next group's P cannot overtake this group's scatter MMAs) and the fp32
// accumulator of the part (up to 512 - K features: two parts for d = 768, K = 128).  Roles: warp 0 TMA loader,
// warp 1 MMA issuer, warps 2-5 plan builders (idx_g -> list of {D column, P column, S descriptor} + the S matrices),
// warps 6-9 zero the accumulator at the start and flush it into dX^T at the end.  There is no epilogue.
#include <algorithm>
#include <cstdlib>

#include "tc_common.cuh"
#include "tc_kernels.h"

namespace haste {
using namespace tc;

struct DxMmaParams {
  float* dXt;           // [d][Bpad] fp32, zeroed by the caller
  const int32_t* idx;   // [NG][K]
  int B, Bpad, NT, NP, S, d;
  int FP;               // features per part (multiple of 4); part fp owns [fp*FP, min(d, (fp+1)*FP))
  int FPW;              // accumulator columns of a part: max(64, FP)
  int64_t NG;
};

template <int G, int K> struct DxMmaCfg {
  static constexpr int Y_BYTES = G * 256;                     // [G/64 k-blocks][128 batch rows][128 B]; G = 32: [128 rows][64 B]
  static constexpr int W_BYTES = G * K * 2;                   // [K/64 slot atoms][G label rows][128 B]
  static constexpr int STAGE = Y_BYTES + W_BYTES;
  static constexpr int NST = STAGE <= 32768 ? 3 : 2;
  static constexpr int NA = (STAGE > 32768 && K == 128) ? 2 : 4;   // plan-building warps; warp a builds groups i = a (mod NA) into ring slot a
  static constexpr int S_BYTES = 2048;                        // one S matrix: [64 n][8 k] tf32, K-major, no swizzle
  static constexpr int ACC_MAX = 512 - K;                     // accumulator columns available next to P
  static constexpr int OFF_S = NST * STAGE;
  static constexpr int BUDGET = 232448 - 1024 - 2048;         // - alignment slack - (entries, barriers, misc)
  static constexpr int MAXE_RAW = (BUDGET - OFF_S) / (NA * S_BYTES);
  static constexpr int MAXE = MAXE_RAW > 24 ? 24 : MAXE_RAW;  // scatter MMAs per plan item
  static_assert(MAXE >= 16, "no room for the S matrices");
  static constexpr int HALF = (MAXE / 2) / 4 * 4;             // scatter MMAs per plan item and P half (slots [0,64) / [64,128))
  static_assert(HALF >= 8, "one round of a half must fit one plan item");
  static constexpr int NH = K > 64 ? 2 : 1;                   // P halves
  static constexpr int OFF_ENT = OFF_S + NA * MAXE * S_BYTES; // [NA][MAXE] x 4 B: {8-slot block << 9 | first accumulator column}
  static constexpr int OFF_META = OFF_ENT + NA * MAXE * 4;    // [NA] x 16 B: {n0, n1, flags}
  static constexpr int OFF_BAR = OFF_META + NA * 16;
  static constexpr int NBAR = 2 * NST + 2 * NA + 3;
  static constexpr int OFF_MISC = OFF_BAR + NBAR * 8;
  static constexpr int SMEM = OFF_MISC + 64 + 1024;
  static_assert(SMEM <= 232448, "shared memory budget");
  static constexpr int THREADS = (2 + NA + 4) * 32;
};

__device__ __forceinline__ void dxm_red_add_f32(float* addr, float v) {
  asm volatile("red.global.add.f32 [%0], %1;" ::"l"(addr), "f"(v) : "memory");
}
__device__ __forceinline__ void dxm_tst16z(uint32_t taddr) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1};" ::"r"(taddr),
      "r"(0u)
      : "memory");
}
__device__ __forceinline__ void dxm_tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
// shared-memory matrix descriptor without swizzle (layout type 0): core matrices of 8 rows x 16 B
__device__ __forceinline__ uint64_t dxm_sdesc_none(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr >> 4) & 0x3FFF);
  d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16;
  d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32;
  d |= (uint64_t)1 << 46;
  return d;
}
// ACC[tmem d] += P[tmem a] (tf32, 128 x 8) * S[smem desc] (tf32, 8 x 64)
__device__ __forceinline__ void dxm_umma_scatter(uint32_t d_tmem, uint32_t a_tmem, uint64_t bdesc, uint32_t idesc) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, 1, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}"
      ::"r"(d_tmem), "r"(a_tmem), "l"(bdesc), "r"(idesc)
      : "memory");
}
__device__ __forceinline__ uint4 dxm_lds128u(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
  return v;
}

template <int G, int K>
__global__ void __launch_bounds__(DxMmaCfg<G, K>::THREADS, 1)
tc_dx_mma_kernel(const __grid_constant__ CUtensorMap tmY, const __grid_constant__ CUtensorMap tmW, const DxMmaParams p) {
  using C = DxMmaCfg<G, K>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const uint32_t sbase = smem_u32(smem);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::OFF_BAR);
  uint64_t* full = bars;                        // [NST] TMA (tx) -> issuer
  uint64_t* empty = bars + C::NST;              // [NST] P MMA commit -> TMA
  uint64_t* item_full = bars + 2 * C::NST;      // [NA]  plan builder -> issuer
  uint64_t* item_empty = item_full + C::NA;     // [NA]  scatter MMA commit -> plan builder
  uint64_t* done = item_empty + C::NA;          // [1]   last MMA commit -> flush warps
  uint64_t* p_done = done + 1;                  // [2]   P MMA commit (per half of P) -> issuer: a scatter MMA reads P from TMEM, no hardware interlock
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + C::OFF_MISC);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // blockIdx = (stripe * NP + part) * NT + batch tile: the CTAs that share a dY tile / W_g run side by side (L2 reuse)
  const int bt = blockIdx.x % p.NT, part = (blockIdx.x / p.NT) % p.NP, stripe = blockIdx.x / (p.NT * p.NP);
  const int n_my = p.NG > stripe ? (int)((p.NG - stripe + p.S - 1) / p.S) : 0;
  const int f_lo = part * p.FP, f_hi = min(p.d, f_lo + p.FP);

  if (threadIdx.x == 0) {
    for (int i = 0; i < C::NST; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], 1); }
    for (int i = 0; i < C::NA; ++i) { mbar_init(&item_full[i], 1); mbar_init(&item_empty[i], 1); }
    mbar_init(done, 1);
    mbar_init(&p_done[0], 1); mbar_init(&p_done[1], 1);
    fence_barrier_init();
  }
  if (warp == 0 && lane == 0) { tma_prefetch_desc(&tmY); tma_prefetch_desc(&tmW); }
  if (warp == 1) tmem_alloc<512>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  if (warp >= 2 + C::NA) {                       // zero the accumulator columns [K, K + FPW)
    const uint32_t tl = tmem_base + ((uint32_t)((warp & 3) * 32) << 16) + K;
    for (int c = 0; c < p.FPW; c += 16) dxm_tst16z(tl + min(c, 512 - K - 16));
    dxm_tmem_st_wait();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();

  if (warp == 0) {
    // ===================== TMA loader: dY tile + W_g =====================
    if (lane == 0) {
      for (int i = 0; i < n_my; ++i) {
        const int64_t g = stripe + (int64_t)i * p.S;
        const int st = i % C::NST;
        mbar_wait(&empty[st], ((i / C::NST) & 1) ^ 1);
        mbar_arrive_expect_tx(&full[st], C::STAGE);
        uint8_t* s0 = smem + st * C::STAGE;
#pragma unroll
        for (int kb = 0; kb < (G >= 64 ? G / 64 : 1); ++kb) tma_load_3d(s0 + kb * 16384, &tmY, &full[st], kb * 64, bt * 128, (int)g);
#pragma unroll
        for (int a = 0; a < K / 64; ++a) tma_load_2d(s0 + C::Y_BYTES + a * (G * 128), &tmW, &full[st], a * 64, (int)(g * G));
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (whole warp waits, one elected lane issues) =====================
    // A scatter MMA reads P from TMEM as its A operand and NOTHING orders that read behind the P MMA's writes (measured:
    // the first scatter MMA of a group saw partial sums), so the issuer waits for the P MMA's commit before it issues
    // them.  To keep the tensor pipe fed across that round trip, P is computed in two halves (slots [0,64) and [64,128))
    // and the queue is interleaved:   ... S0(i-1)  P0(i)  S1(i-1)  P1(i)  S0(i)  P0(i+1)  S1(i) ...
    // (Sh = scatter MMAs reading half h, Ph = the MMAs writing it): every wait has two blocks of work queued behind it.
    constexpr uint32_t idesc_p = make_idesc_bf16(128, 64, /*A (dY) K-major*/ 0, /*B (W) MN-major*/ 1);
    constexpr uint32_t idesc_s = (1u << 4) | (2u << 7) | (2u << 10) | ((64u >> 3) << 17) | ((128u >> 4) << 24);   // tf32 x tf32 -> f32, M 128, N 64
    const uint64_t adesc0 = G >= 64 ? make_sdesc_sw128(sbase, 16, 1024) : make_sdesc_sw64(sbase, 16, 512);
    const uint64_t bdesc0 = make_sdesc_sw128(sbase + C::Y_BYTES, G * 128, 1024);
    auto issue_p = [&](int st, int h) {          // P[:, 64h .. 64h+63] = dY tile * W_g[:, 64h .. 64h+63]
      const uint64_t so = (uint64_t)((st * C::STAGE) >> 4);
#pragma unroll
      for (int j = 0; j < G / 16; ++j)
        umma_f16(tmem_base + h * 64, adesc0 + so + (uint64_t)(((j >> 2) * 16384 + (j & 3) * 32) >> 4),
                 bdesc0 + so + (uint64_t)((h * (G * 128) + j * 2048) >> 4), idesc_p, j ? 1u : 0u);
    };
    // A plan entry is ONE word, everything else follows from the entry's position: every operand of tcgen05.mma lives
    // in a uniform register, and each value that comes out of shared memory costs an R2UR on the issuing thread
    // (four of them per MMA made the issue loop the bottleneck: ~60 cycles per scatter MMA).
    static_assert(C::HALF % 4 == 0, "entries are loaded four at a time");
    uint32_t en[C::HALF];
    const uint64_t sdesc0 = dxm_sdesc_none(sbase + C::OFF_S, 128, 256);
    auto load_entries = [&](int a, int h, uint32_t n) {
      const uint32_t ent = sbase + C::OFF_ENT + (a * C::MAXE + h * C::HALF) * 4;
#pragma unroll
      for (int e = 0; e < C::HALF; e += 4)
        if ((uint32_t)e < n) { const uint4 v = dxm_lds128u(ent + e * 4); en[e] = v.x; en[e + 1] = v.y; en[e + 2] = v.z; en[e + 3] = v.w; }
    };
    auto issue_entries = [&](int a, int h, uint32_t n) {       // elected lane only
      const uint64_t sd = sdesc0 + (uint64_t)(((a * C::MAXE + h * C::HALF) * C::S_BYTES) >> 4);
#pragma unroll
      for (int e = 0; e < C::HALF; ++e)
        if ((uint32_t)e < n)
          dxm_umma_scatter(tmem_base + K + (en[e] & 511u), tmem_base + (en[e] >> 9) * 8, sd + (uint64_t)((e * C::S_BYTES) >> 4), idesc_s);
    };
    uint32_t phase = 0;                          // bit a: parity of the next item of ring slot a
    bool pend = false;                           // S1 of the previous group is not issued yet (its item is still held)
    int pend_a = 0;
    uint32_t pend_n1 = 0;
    for (int i = 0; i < n_my; ++i) {
      const int a = i % C::NA, st = i % C::NST;
      mbar_wait(&item_full[a], (phase >> a) & 1);
      phase ^= 1u << a;
      uint4 meta = dxm_lds128u(sbase + C::OFF_META + a * 16);      // {n0, n1, flags (1 = first item of the group, 2 = last)}
      mbar_wait(&full[st], (i / C::NST) & 1);
      tc_fence_after();
      if (elect_one()) {
        issue_p(st, 0);
        umma_commit(&p_done[0]);
        if (C::NH == 1) umma_commit(&empty[st]);
      }
      __syncwarp();
      if (pend) {                                // S1(i-1), behind P0(i)
        load_entries(pend_a, 1, pend_n1);
        mbar_wait(&p_done[1], (i - 1) & 1);
        tc_fence_after();
        if (elect_one()) { issue_entries(pend_a, 1, pend_n1); umma_commit(&item_empty[pend_a]); }
        __syncwarp();
        pend = false;
      }
      if (C::NH == 2) {
        if (elect_one()) { issue_p(st, 1); umma_commit(&p_done[1]); umma_commit(&empty[st]); }
        __syncwarp();
      }
      load_entries(a, 0, meta.x);
      mbar_wait(&p_done[0], i & 1);
      tc_fence_after();
      if (elect_one()) issue_entries(a, 0, meta.x);    // S0(i)
      __syncwarp();
      if (meta.z & 2u) {
        if (C::NH == 2) { pend = true; pend_a = a; pend_n1 = meta.y; }
        else { if (elect_one()) umma_commit(&item_empty[a]); __syncwarp(); }
      } else {
        // rare (an unsorted index row): the group's plan did not fit one item.  Finish it in order, no interleaving.
        if (C::NH == 2) {
          load_entries(a, 1, meta.y);
          mbar_wait(&p_done[1], i & 1);
          tc_fence_after();
          if (elect_one()) issue_entries(a, 1, meta.y);
          __syncwarp();
        }
        for (;;) {
          if (elect_one()) umma_commit(&item_empty[a]);
          __syncwarp();
          mbar_wait(&item_full[a], (phase >> a) & 1);
          phase ^= 1u << a;
          meta = dxm_lds128u(sbase + C::OFF_META + a * 16);
          load_entries(a, 0, meta.x);
          if (elect_one()) issue_entries(a, 0, meta.x);
          __syncwarp();
          load_entries(a, 1, meta.y);
          if (elect_one()) issue_entries(a, 1, meta.y);
          __syncwarp();
          if (meta.z & 2u) break;
        }
        if (elect_one()) umma_commit(&item_empty[a]);
        __syncwarp();
      }
    }
    if (pend) {
      load_entries(pend_a, 1, pend_n1);
      mbar_wait(&p_done[1], (n_my - 1) & 1);
      tc_fence_after();
      if (elect_one()) { issue_entries(pend_a, 1, pend_n1); umma_commit(&item_empty[pend_a]); }
      __syncwarp();
    }
    if (elect_one()) umma_commit(done);
    __syncwarp();
  } else if (warp < 2 + C::NA) {
    // ===================== plan builders: idx_g -> scatter MMAs of this part =====================
    // Lane l < K/8 owns the 8-slot block l of the group.  A round gives every block that still has uncovered slots of
    // this part one scatter MMA: window start = its smallest uncovered feature (4-aligned), 64 columns wide.
    const int aw = warp - 2;
    const uint32_t s_ring = sbase + C::OFF_S + aw * C::MAXE * C::S_BYTES;
    const uint32_t e_ring = sbase + C::OFF_ENT + aw * C::MAXE * 4;
    const uint32_t m_ring = sbase + C::OFF_META + aw * 16;
    const bool own = lane < K / 8;
    const int half = lane >> 3;           // P half of this lane's block (K = 64: always 0)
    int nitems = 0;                       // items published into this ring slot so far
    int nd0 = C::HALF, nd1 = C::HALF;     // S matrices of each half that may hold ones (all of them before first use)
    auto zero_s = [&](int n0, int n1) {
      for (int e = 0; e < n0 + n1; ++e) {
        const uint32_t a = s_ring + (e < n0 ? e : C::HALF + e - n0) * C::S_BYTES + lane * 64;
        sts128(a, 0u, 0u, 0u, 0u); sts128(a + 16, 0u, 0u, 0u, 0u); sts128(a + 32, 0u, 0u, 0u, 0u); sts128(a + 48, 0u, 0u, 0u, 0u);
      }
    };
    int4 nx0 = make_int4(0, 0, 0, 0), nx1 = nx0;
    if (own && aw < n_my) {
      const int4* src = reinterpret_cast<const int4*>(p.idx + (stripe + (int64_t)aw * p.S) * K + lane * 8);
      nx0 = __ldg(src); nx1 = __ldg(src + 1);
    }
    for (int i = aw; i < n_my; i += C::NA) {
      const int64_t g = stripe + (int64_t)i * p.S;
      const int f[8] = {nx0.x - f_lo, nx0.y - f_lo, nx0.z - f_lo, nx0.w - f_lo, nx1.x - f_lo, nx1.y - f_lo, nx1.z - f_lo, nx1.w - f_lo};
      if (own && i + C::NA < n_my) {
        const int4* src = reinterpret_cast<const int4*>(p.idx + (g + (int64_t)C::NA * p.S) * K + lane * 8);
        nx0 = __ldg(src); nx1 = __ldg(src + 1);
      }
      uint32_t rem = 0;                   // uncovered slots of this block that belong to this part
      if (own) {
#pragma unroll
        for (int k = 0; k < 8; ++k) rem |= (uint32_t)(f[k] >= 0 && f[k] < f_hi - f_lo) << k;
      }
      bool first = true;
      int base0 = 0, base1 = 0;
      // the ring slot is free once the scatter MMAs of its previous item have completed
      mbar_wait(&item_empty[aw], ((nitems & 1) ^ 1));
      zero_s(nd0, nd1);
      __syncwarp();
      for (;;) {
        const uint32_t bal = __ballot_sync(0xffffffffu, rem != 0);
        if (bal == 0) break;
        const int c0 = __popc(bal & 0xffu), c1 = __popc(bal >> 8);
        if (base0 + c0 > C::HALF || base1 + c1 > C::HALF) {   // the item is full: publish it, continue the group in a new one
          fence_proxy_async_smem();
          __syncwarp();
          if (lane == 0) {
            sts128(m_ring, (uint32_t)base0, (uint32_t)base1, first ? 1u : 0u, 0u);
            mbar_arrive(&item_full[aw]);
          }
          ++nitems;
          first = false;
          mbar_wait(&item_empty[aw], ((nitems & 1) ^ 1));
          zero_s(base0, base1);
          base0 = 0; base1 = 0;
          __syncwarp();
        }
        if (rem != 0) {
          const int e = half * C::HALF + (half ? base1 + __popc((bal >> 8) & ((1u << (lane - 8)) - 1u)) : base0 + __popc(bal & ((1u << lane) - 1u)));
          int fmin = 0x7fffffff;
#pragma unroll
          for (int k = 0; k < 8; ++k) if ((rem >> k) & 1u) fmin = min(fmin, f[k]);
          const int start = min(fmin & ~3, p.FPW - 64);
          const uint32_t s_e = s_ring + e * C::S_BYTES;
#pragma unroll
          for (int k = 0; k < 8; ++k) {
            const int n = f[k] - start;
            if (((rem >> k) & 1u) && n < 64) {          // n >= 0 because start <= fmin
              sts32(s_e + (n >> 3) * 256 + (k >> 2) * 128 + (n & 7) * 16 + (k & 3) * 4, 0x3f800000u);
              rem &= ~(1u << k);
            }
          }
          sts32(e_ring + e * 4, (uint32_t)((lane << 9) | start));   // {8-slot block, first accumulator column}; S matrix = entry index
        }
        base0 += c0; base1 += c1;
      }
      nd0 = base0; nd1 = base1;
      fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) {
        sts128(m_ring, (uint32_t)base0, (uint32_t)base1, (first ? 1u : 0u) | 2u, 0u);
        mbar_arrive(&item_full[aw]);
      }
      ++nitems;
    }
  } else {
    // ===================== flush: accumulator columns of this part -> dX^T (one reduction per CTA and word) =====================
    const int q = warp & 3;
    const int b = bt * 128 + q * 32 + lane;
    mbar_wait(done, 0);
    tc_fence_after();
    const uint32_t tl = tmem_base + ((uint32_t)(q * 32) << 16) + K;
    float* const gcol = p.dXt + b;
    const int nf = f_hi - f_lo;
    for (int c0 = 0; c0 < nf; c0 += 16) {
      uint32_t v[16];
      const int cc = min(c0, 512 - K - 16);              // never read past the allocation; cc <= c0, index shifted below
      tmem_ld16(tl + cc, v);
      tmem_ld_wait();
      if (b < p.B) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
          const int c = cc + u;
          if (c >= c0 && c < nf) dxm_red_add_f32(gcol + (size_t)(f_lo + c) * p.Bpad, __uint_as_float(v[u]));
        }
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) { tc_fence_after(); tmem_dealloc<512>(tmem_base); }
}

template <int G, int K>
static int launch_dx_mma(TcTailState* s, const TailShape& sh, const int32_t* idx, const void* W, const void* dY, float* dXt,
                         cudaStream_t st) {
  using C = DxMmaCfg<G, K>;
  static_assert(K / 8 <= C::MAXE, "one round of a group must fit one plan item");
  CUtensorMap tmY, tmW;
  {
    const uint64_t dims[3] = {(uint64_t)G, (uint64_t)sh.B, (uint64_t)sh.NG};
    const uint64_t str[2] = {(uint64_t)G * 2, (uint64_t)sh.B * G * 2};
    const uint32_t box[3] = {(uint32_t)std::min(G, 64), 128, 1};
    int rc = encode_tmap(&tmY, 2, dY, 3, dims, str, box, G >= 64 ? 128 : 64);
    if (rc) return rc;
  }
  {
    const uint64_t dims[2] = {(uint64_t)K, (uint64_t)sh.L};
    const uint64_t str[1] = {(uint64_t)K * 2};
    const uint32_t box[2] = {64, (uint32_t)G};
    int rc = encode_tmap(&tmW, 2, W, 2, dims, str, box, 128);
    if (rc) return rc;
  }
  DxMmaParams p;
  p.dXt = dXt; p.idx = idx; p.B = sh.B; p.Bpad = sh.Bpad; p.NT = ceil_div(sh.B, 128); p.NG = sh.NG; p.d = sh.d;
  p.NP = ceil_div(sh.d, C::ACC_MAX);
  p.FP = round_up(ceil_div(sh.d, p.NP), 4);
  p.FPW = std::max(64, p.FP);
  if (p.FPW > C::ACC_MAX || p.NT * p.NP > s->num_sms) return HASTE_ERR_UNSUPPORTED;
  p.S = (int)std::min<int64_t>(sh.NG, std::max(1, s->num_sms / (p.NT * p.NP)));
  HASTE_CUDA_TRY(cudaFuncSetAttribute(tc_dx_mma_kernel<G, K>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM));
  tc_dx_mma_kernel<G, K><<<p.NT * p.NP * p.S, C::THREADS, C::SMEM, st>>>(tmY, tmW, p);
  HASTE_LAUNCH_CHECK();
  return HASTE_OK;
}

int tc_tail_dx_mma(TcTailState* s, const TailShape& sh, const int32_t* idx, const void* W, const void* dY, float* dXt,
                   cudaStream_t st) {
#define HASTE_DXM(G_, K_) if (sh.G == G_ && sh.K == K_) return launch_dx_mma<G_, K_>(s, sh, idx, W, dY, dXt, st)
  HASTE_DXM(64, 128); HASTE_DXM(64, 64); HASTE_DXM(128, 64); HASTE_DXM(128, 128); HASTE_DXM(32, 64); HASTE_DXM(32, 128);
#undef HASTE_DXM
  return HASTE_ERR_UNSUPPORTED;
}

}  // namespace haste
