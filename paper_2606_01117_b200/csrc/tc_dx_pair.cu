// tc_dx_pair.cu -- input-gradient kernel of the HASTE sparse tail, round-2 design (sm_100a; bf16 in, fp32 accumulate).
//
//   dX[:, idx_g] += dY_g [B x G] * W_g [G x K]   over all groups g
//
// What bounds this step is not HBM but the B*NG*K scalar read-modify-writes of the scatter-add (669 M at config 3):
// tc_dx_acc.cu pays ~9 warp instructions per 32 adds and is issue-bound at 0.43 of the HBM roofline.  This kernel
// halves the instruction count per add and removes most of the L2 reductions:
//   * a CTA works on 256 batch rows (two M = 128 MMA tiles), and a thread owns the SAME lane of both tiles, so every
//     accumulator access (tcgen05.ld/st .x2, ld/st.shared.v2, red.global.v2) carries two adds;
//   * two CTAs of a cluster share one stream of (256-row tile, group) units -- the dY tile is loaded once and TMA-
//     multicast into both -- and each owns HALF of the feature range.  Because an idx row is sorted, a CTA's slots
//     are one contiguous slot range [j_lo, j_hi) of the group: it loads only those columns of W_g and computes only
//     those columns of P (jobs of NW slots).  Its half of the features fits mostly on chip:
//       T class: fp32 accumulator column PAIRS in TMEM next to the ring of P buffers
//       S class: fp32 accumulator rows in shared memory ([feature][128 lanes][2 tiles])
//       L class: what fits in neither goes to the workspace with red.global.add.v2.f32
//   * three epilogue sets of four warps (one per TMEM lane quadrant) own one class each, so nothing on chip is
//     atomic and no two warps ever touch the same accumulator word.
// A group whose idx row is not strictly increasing (duplicates / unsorted, legal by DESIGN.md reading R4) is split
// by slot POSITION between the two CTAs and takes the L class for every slot (atomic, correct for any row).
// Output: the workspace dXw [NT2][d][128 lanes][2 tiles] fp32 (zeroed by the caller), NT2 = ceil(B / 256); a small
// kernel (launch_dxw_to_dx) turns it into dX [B, d].
#include <algorithm>
#include <cstdio>
#include <cstring>

#include "tc_common.cuh"
#include "tc_kernels.h"

namespace haste {
using namespace tc;
#ifndef DXP_CS
#define DXP_CS 2
#endif
#ifndef DXP_MC_TMA
#define DXP_MC_TMA 1
#endif
#ifndef DXP_MC_COMMIT
#define DXP_MC_COMMIT 1
#endif

struct DxPairParams {
  float* dXw;           // [NT2][d][128][2] fp32, zeroed by the caller
  const int32_t* idx;   // [NG][K]
  int B, d, NT2;
  int64_t NG, U;        // U = NT2 * NG units, unit u = (tile u / NG, group u % NG)
  int NP;               // clusters (pairs); grid = CS * NP
  int Fc;               // features per CTA of a cluster: CTA r owns [r * Fc, min(d, (r + 1) * Fc))
  int nT, nS;           // features of a CTA's range held in TMEM / in shared memory (the rest: L class)
#ifdef DXP_DEBUG
  volatile int* dbg;
#endif
};

template <int G, int K, int CS_, int NW_, int R_> struct DxPairCfg {
  static constexpr int CS = CS_;                              // CTAs per cluster (1 or 2)
  static constexpr int NW = NW_;                              // slots per job = N of the MMA
  static constexpr int R = R_;                                // ring of P buffers in TMEM, one job each
  static constexpr int NSTY = 2, NSTW = 3, RD = 4, NAUX = 2;
  static constexpr int YB = G * 512;                          // dY tile: [G/64 k-blocks][256 rows][128 B]; G = 32: [256 rows][64 B]
  static constexpr int WB = G * 128;                          // W_g columns [j0, j0 + 64): [G label rows][128 B]
  static constexpr int JMAX = (K + NW - 1) / NW;              // jobs per unit at most
  static constexpr int LIST_LEN = NW + 16;                    // entries per (job, set) list, padded for the last chunk
  static constexpr int PLAN_HDR = 16 + JMAX * 8;              // ints: njobs, j0 (first slot of job 0), tile, -, then per job {lo, n} x 3 sets (+2 pad)
  static constexpr int PLAN_BYTES = (PLAN_HDR * 4 + JMAX * 3 * LIST_LEN * 4 + 127) / 128 * 128;
  static constexpr int PB = R * 2 * NW;                       // first TMEM column of the T accumulators
  static constexpr int T_MAX = (512 - PB - 2) / 2;            // T features (column pairs); the last pair is the dummy
  static constexpr int TDUMMY = 510;
  static constexpr int OFF_W = NSTY * YB;
  static constexpr int OFF_PLAN = OFF_W + NSTW * WB;
  static constexpr int OFF_BAR = OFF_PLAN + RD * PLAN_BYTES;
  static constexpr int NBAR = 2 * NSTY + 2 * NSTW + 2 * R + 2 * RD;
  static constexpr int OFF_MISC = OFF_BAR + NBAR * 8;
  static constexpr int OFF_ACC = (OFF_MISC + 64 + 1023) / 1024 * 1024;
  static constexpr int S_MAX = (232448 - 1024 - OFF_ACC) / 1024 - 1;    // S features (rows of 1 KB) + 1 dummy row
  static constexpr int NSET = 3;                              // epilogue sets: 0 = T, 1 = S, 2 = L
  static constexpr int W_MMA = 4 * NSET, W_LOAD = W_MMA + 1, W_AUX = W_MMA + 2;
  static constexpr int THREADS = (4 * NSET + 2 + NAUX) * 32;
  static constexpr int N_REL = 4 * NSET + 2;                  // consumers of a plan slot: epilogue warps, MMA warp, loader
};

// ---------------------------------------------------------------- PTX helpers of this kernel
__device__ __forceinline__ uint32_t dxp_cluster_rank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void dxp_cluster_sync() {
  // not .aligned: the loader warp comes here with lane 0 apart from the others
  asm volatile("barrier.cluster.arrive.release;\n\tbarrier.cluster.wait.acquire;" ::: "memory");
}
__device__ __forceinline__ void dxp_tma_load_3d_mc(uint32_t dst, const CUtensorMap* m, uint64_t* bar, int c0, int c1, int c2, uint16_t mask) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.multicast::cluster [%0], [%1, {%3, %4, %5}], [%2], %6;"
      ::"r"(dst), "l"(reinterpret_cast<uint64_t>(m)), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "h"(mask)
      : "memory");
}
__device__ __forceinline__ void dxp_commit_mc(uint64_t* bar, uint16_t mask) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
               ::"r"(smem_u32(bar)), "h"(mask) : "memory");
}
__device__ __forceinline__ void dxp_tld2(uint32_t taddr, uint32_t& a, uint32_t& b) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(a), "=r"(b) : "r"(taddr) : "memory");
}
__device__ __forceinline__ void dxp_tst2(uint32_t taddr, uint32_t a, uint32_t b) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(taddr), "r"(a), "r"(b) : "memory");
}
__device__ __forceinline__ void dxp_tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void dxp_tmem_ld8(uint32_t taddr, uint32_t (&v)[8]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
               : "r"(taddr)
               : "memory");
}
template <int N> __device__ __forceinline__ void dxp_tmem_ldn(uint32_t taddr, uint32_t (&v)[N]);
template <> __device__ __forceinline__ void dxp_tmem_ldn<8>(uint32_t taddr, uint32_t (&v)[8]) { dxp_tmem_ld8(taddr, v); }
template <> __device__ __forceinline__ void dxp_tmem_ldn<16>(uint32_t taddr, uint32_t (&v)[16]) { tmem_ld16(taddr, v); }
__device__ __forceinline__ int dxp_lds32i(uint32_t addr) {
  int v;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ int4 dxp_lds128i(uint32_t addr) {
  int4 v;
  asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ float2 dxp_lds64f(uint32_t addr) {
  float2 v;
  asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ void dxp_sts64f(uint32_t addr, float a, float b) {
  asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(addr), "f"(a), "f"(b) : "memory");
}
__device__ __forceinline__ void dxp_red2(const char* addr, float a, float b) {
  asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(addr), "f"(a), "f"(b) : "memory");
}
template <int N> __device__ __forceinline__ void dxp_load_dest(uint32_t addr, int (&dst)[N]) {
#pragma unroll
  for (int i = 0; i < N / 4; ++i) {
    const int4 a = dxp_lds128i(addr + i * 16);
    dst[4 * i] = a.x; dst[4 * i + 1] = a.y; dst[4 * i + 2] = a.z; dst[4 * i + 3] = a.w;
  }
}
template <int NS_SLEEP> __device__ __forceinline__ void dxp_wait(uint64_t* bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) __nanosleep(NS_SLEEP);
}

// one chunk of N slots of the T class: accumulator column pair dst[u] += (P tile 0, P tile 1) column u
template <int N> __device__ __forceinline__ void dxp_chunk_t(uint32_t tp0, uint32_t tp1, uint32_t lst, uint32_t tlane) {
  uint32_t p0[N], p1[N], a0[N], a1[N];
  int dst[N];
  dxp_tmem_ldn<N>(tp0, p0);
  dxp_tmem_ldn<N>(tp1, p1);
  dxp_load_dest<N>(lst, dst);
#pragma unroll
  for (int u = 0; u < N; ++u) dxp_tld2(tlane + dst[u], a0[u], a1[u]);
  tmem_ld_wait();
#pragma unroll
  for (int u = 0; u < N; ++u)
    dxp_tst2(tlane + dst[u], __float_as_uint(__uint_as_float(a0[u]) + __uint_as_float(p0[u])),
             __float_as_uint(__uint_as_float(a1[u]) + __uint_as_float(p1[u])));
}
// one chunk of N slots of the S class: accumulator row (byte offset dst[u]), this thread's two words += P column u
template <int N> __device__ __forceinline__ void dxp_chunk_s(uint32_t tp0, uint32_t tp1, uint32_t lst, uint32_t sown) {
  uint32_t p0[N], p1[N];
  float2 a[N];
  int dst[N];
  dxp_tmem_ldn<N>(tp0, p0);
  dxp_tmem_ldn<N>(tp1, p1);
  dxp_load_dest<N>(lst, dst);
#pragma unroll
  for (int u = 0; u < N; ++u) a[u] = dxp_lds64f(sown + dst[u]);
  tmem_ld_wait();
#pragma unroll
  for (int u = 0; u < N; ++u) dxp_sts64f(sown + dst[u], a[u].x + __uint_as_float(p0[u]), a[u].y + __uint_as_float(p1[u]));
}

#ifdef DXP_DEBUG
#define MARK(v) do { if (lane == 0) { p.dbg[blockIdx.x * 32 + warp] = (v); __threadfence_system(); } } while (0)
#else
#define MARK(v)
#endif
template <int G, int K, int CS, int NW, int R>
__global__ void __launch_bounds__(DxPairCfg<G, K, CS, NW, R>::THREADS, 1)
tc_dx_pair_kernel(const __grid_constant__ CUtensorMap tmY, const __grid_constant__ CUtensorMap tmW, const DxPairParams p) {
  using C = DxPairCfg<G, K, CS, NW, R>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const uint32_t sbase = smem_u32(smem);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::OFF_BAR);
  uint64_t* yfull = bars;                      // [NSTY] TMA (tx, from every CTA of the cluster) -> MMA
  uint64_t* yempty = yfull + C::NSTY;          // [NSTY] MMA commits of ALL CTAs of the cluster -> loader
  uint64_t* wfull = yempty + C::NSTY;          // [NSTW] TMA -> MMA
  uint64_t* wempty = wfull + C::NSTW;          // [NSTW] MMA commit -> loader
  uint64_t* t_full = wempty + C::NSTW;         // [R]    MMA commit -> epilogue
  uint64_t* t_empty = t_full + C::R;           // [R]    12 epilogue warps -> MMA
  uint64_t* d_full = t_empty + C::R;           // [RD]   aux warp -> everyone (plan of the unit ready)
  uint64_t* d_empty = d_full + C::RD;          // [RD]   everyone -> aux warp
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + C::OFF_MISC);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = CS > 1 ? dxp_cluster_rank() : 0u;
  const int pair = blockIdx.x / CS;
  const int64_t u0 = p.U * pair / p.NP, u1 = p.U * (pair + 1) / p.NP;
#ifdef DXP_SKIP
  const int n_my = 0;
#elif defined(DXP_LIMIT)
  const int n_my = min(DXP_LIMIT, (int)(u1 - u0));
#else
  const int n_my = (int)(u1 - u0);
#endif
  const int F_lo = (int)rank * p.Fc, F_hi = min(p.d, F_lo + p.Fc);

  if (threadIdx.x == 0) {
    for (int i = 0; i < C::NSTY; ++i) { mbar_init(&yfull[i], 1); mbar_init(&yempty[i], DXP_MC_COMMIT ? CS : 1); }
    for (int i = 0; i < C::NSTW; ++i) { mbar_init(&wfull[i], 1); mbar_init(&wempty[i], 1); }
    for (int i = 0; i < C::R; ++i) { mbar_init(&t_full[i], 1); mbar_init(&t_empty[i], 4 * C::NSET); }
    for (int i = 0; i < C::RD; ++i) { mbar_init(&d_full[i], 1); mbar_init(&d_empty[i], C::N_REL); }
    fence_barrier_init();
  }
  if (warp == C::W_LOAD && lane == 0) { tma_prefetch_desc(&tmY); tma_prefetch_desc(&tmW); }
  if (warp == C::W_MMA) tmem_alloc<512>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  if (CS > 1) dxp_cluster_sync();              // the peer's barriers exist before anything remote is sent to them
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  MARK(1);

  if (warp == C::W_LOAD) {
    // ===================== loader: this CTA's share of the dY tile (multicast) + its own columns of W_g =====================
    if (lane == 0) {
      constexpr int ROWS = 256 / CS;                               // rows of the tile this CTA fetches for the whole cluster
      constexpr int ROWB = G >= 64 ? 128 : 64;                     // bytes of one row of a k-block image
      int jc = 0;
      for (int i = 0; i < n_my; ++i) {
        const int64_t u = u0 + i;
        const int t = (int)(u / p.NG);
        const int g = (int)(u - (int64_t)t * p.NG);
        const int ys = i % C::NSTY;
        mbar_wait(&yempty[ys], ((i / C::NSTY) & 1) ^ 1);
        MARK(10);
        mbar_arrive_expect_tx(&yfull[ys], C::YB);
        MARK(11);
        const uint32_t y0 = sbase + ys * C::YB + rank * ROWS * ROWB;
#pragma unroll
        for (int kb = 0; kb < (G >= 64 ? G / 64 : 1); ++kb) {
          if (CS > 1 && DXP_MC_TMA)
            dxp_tma_load_3d_mc(y0 + kb * 256 * 128, &tmY, &yfull[ys], kb * 64, t * 256 + (int)rank * ROWS, g, (uint16_t)((1u << CS) - 1));
          else if (CS == 1)
            tma_load_3d(smem + ys * C::YB + kb * 256 * 128, &tmY, &yfull[ys], kb * 64, t * 256, g);
          else
            for (int rr = 0; rr < CS; ++rr)
              tma_load_3d(smem + ys * C::YB + kb * 256 * 128 + rr * ROWS * ROWB, &tmY, &yfull[ys], kb * 64, t * 256 + rr * ROWS, g);
        }
        MARK(12);
        const int ps = i % C::RD;
        mbar_wait(&d_full[ps], (i / C::RD) & 1);
        MARK(13);
        const uint32_t plan = sbase + C::OFF_PLAN + ps * C::PLAN_BYTES;
        const int njobs = dxp_lds32i(plan), j_lo = dxp_lds32i(plan + 4);
        for (int w = 0; w < njobs; ++w, ++jc) {
          const int ws = jc % C::NSTW;
          mbar_wait(&wempty[ws], ((jc / C::NSTW) & 1) ^ 1);
          mbar_arrive_expect_tx(&wfull[ws], C::WB);
          tma_load_2d(smem + C::OFF_W + ws * C::WB, &tmW, &wfull[ws], j_lo + w * NW, g * G);
        }
        MARK(14);
        mbar_arrive(&d_empty[ps]);
      }
      MARK(15);
    }
  } else if (warp == C::W_MMA) {
    // ===================== MMA issuer: P[256 rows x NW slots] of one job into a ring slot =====================
    constexpr uint32_t idesc = make_idesc_bf16(128, NW, /*A (dY) K-major*/ 0, /*B (W) MN-major*/ 1);
    const uint64_t adesc0 = G >= 64 ? make_sdesc_sw128(sbase, 16, 1024) : make_sdesc_sw64(sbase, 16, 512);
    const uint64_t bdesc0 = make_sdesc_sw128(sbase + C::OFF_W, G * 128, 1024);
    int jc = 0;
    for (int i = 0; i < n_my; ++i) {
      const int ys = i % C::NSTY, ps = i % C::RD;
      mbar_wait(&d_full[ps], (i / C::RD) & 1);
      const int njobs = dxp_lds32i(sbase + C::OFF_PLAN + ps * C::PLAN_BYTES);
      MARK(20);
      mbar_wait(&yfull[ys], (i / C::NSTY) & 1);
      MARK(21);
      for (int w = 0; w < njobs; ++w, ++jc) {
        const int ws = jc % C::NSTW, rs = jc % C::R;
        mbar_wait(&wfull[ws], (jc / C::NSTW) & 1);
        mbar_wait(&t_empty[rs], ((jc / C::R) & 1) ^ 1);
        tc_fence_after();
        MARK(22);
        if (elect_one()) {
          const uint64_t ya = adesc0 + (uint64_t)((ys * C::YB) >> 4);
          const uint64_t wb = bdesc0 + (uint64_t)((ws * C::WB) >> 4);
#pragma unroll
          for (int tile = 0; tile < 2; ++tile) {
            const uint32_t dcol = tmem_base + rs * 2 * NW + tile * NW;
#pragma unroll
            for (int j = 0; j < G / 16; ++j) {
              const uint32_t aoff = G >= 64 ? (j >> 2) * (256 * 128) + tile * (128 * 128) + (j & 3) * 32 : tile * (128 * 64) + j * 32;
#ifndef DXP_NO_MMA
              umma_f16(dcol, ya + (uint64_t)(aoff >> 4), wb + (uint64_t)((j * 2048) >> 4), idesc, j ? 1u : 0u);
#endif
            }
          }
          umma_commit(&wempty[ws]);
          umma_commit(&t_full[rs]);
        }
        __syncwarp();
        MARK(23);
      }
      if (elect_one()) {
        if (CS > 1 && DXP_MC_COMMIT) dxp_commit_mc(&yempty[ys], (uint16_t)((1u << CS) - 1));
        else umma_commit(&yempty[ys]);
      }
      __syncwarp();
      MARK(24);
      if (lane == 0) mbar_arrive(&d_empty[ps]);
    }
    MARK(25);
  } else if (warp >= C::W_AUX) {
    // ===================== auxiliary warps: idx_g -> this CTA's slot range, its jobs, one destination list per (job, class) =====================
    constexpr int PER = K / 32;
    const int aw = warp - C::W_AUX;
    const int fT = F_lo + p.nT, fS = fT + p.nS;
    int e[PER], en[PER];
#pragma unroll
    for (int t = 0; t < PER; ++t) { e[t] = 0; en[t] = 0; }
    if (aw < n_my) {
      const int64_t g = (u0 + aw) % p.NG;
#pragma unroll
      for (int t = 0; t < PER; ++t) en[t] = __ldg(p.idx + g * K + lane + 32 * t);
    }
    for (int i = aw; i < n_my; i += C::NAUX) {
      const int64_t u = u0 + i;
      const int tl = (int)(u / p.NG);
      const int ps = i % C::RD;
#pragma unroll
      for (int t = 0; t < PER; ++t) e[t] = en[t];
      if (i + C::NAUX < n_my) {
        const int64_t gn = (u + C::NAUX) % p.NG;
#pragma unroll
        for (int t = 0; t < PER; ++t) en[t] = __ldg(p.idx + gn * K + lane + 32 * t);
      }
      bool inc = true;
#pragma unroll
      for (int t = 0; t < PER; ++t) {
        int nxt = __shfl_down_sync(0xffffffffu, e[t], 1);
        const int wrap = __shfl_sync(0xffffffffu, t + 1 < PER ? e[(t + 1) % PER] : 0x7fffffff, 0);
        if (lane == 31) nxt = wrap;
        inc &= e[t] < nxt;
      }
      const bool strict = __all_sync(0xffffffffu, inc);
      int c_lo = 0, cT = 0, cS = 0, c_hi = 0;
#pragma unroll
      for (int t = 0; t < PER; ++t) { c_lo += e[t] < F_lo; cT += e[t] < fT; cS += e[t] < fS; c_hi += e[t] < F_hi; }
      c_lo = __reduce_add_sync(0xffffffffu, c_lo); cT = __reduce_add_sync(0xffffffffu, cT);
      cS = __reduce_add_sync(0xffffffffu, cS); c_hi = __reduce_add_sync(0xffffffffu, c_hi);
      if (!strict) { c_lo = (int)rank * (K / CS); c_hi = c_lo + K / CS; cT = c_lo; cS = c_lo; }   // by position, everything L
      // jobs are windows of NW slots from j0 on; j0 is c_lo rounded down to 8 slots: a TMA box must start on a 16-byte boundary
      const int j0 = c_lo & ~7;
      const int njobs = c_hi > c_lo ? (c_hi - j0 + NW - 1) / NW : 0;
      dxp_wait<64>(&d_empty[ps], ((i / C::RD) & 1) ^ 1);
      const uint32_t plan = sbase + C::OFF_PLAN + ps * C::PLAN_BYTES;
      const uint32_t lists = plan + C::PLAN_HDR * 4;
      if (lane == 0) { sts32(plan, (uint32_t)njobs); sts32(plan + 4, (uint32_t)j0); sts32(plan + 8, (uint32_t)tl); }
      // per (job, class): first column in the job's window and number of slots
      auto seg = [&](int w, int s, int& start, int& n) {
        const int ws = j0 + w * NW, we = min(ws + NW, c_hi);
        const int a = s == 0 ? c_lo : s == 1 ? cT : cS, b = s == 0 ? cT : s == 1 ? cS : c_hi;
        start = max(a, ws);
        n = max(0, min(b, we) - start);
        if (n == 0) start = ws;
      };
      if (lane < 3 * C::JMAX) {
        const int w = lane / 3, s = lane - 3 * w;
        int start, n;
        seg(w, s, start, n);
        sts32(plan + (16 + w * 8 + 2 * s) * 4, (uint32_t)(start - (j0 + w * NW)));
        sts32(plan + (16 + w * 8 + 2 * s + 1) * 4, (uint32_t)n);
      }
#pragma unroll
      for (int t = 0; t < PER; ++t) {
        const int j = lane + 32 * t, f = e[t];
        if (j >= c_lo && j < c_hi) {
          const int w = (j - j0) / NW;
          const int s = j < cT ? 0 : j < cS ? 1 : 2;
          int start, n;
          seg(w, s, start, n);
          const uint32_t code = s == 0 ? (uint32_t)(C::PB + 2 * (f - F_lo)) : s == 1 ? (uint32_t)((f - fT) * 1024)
                                                                            : (uint32_t)(tl * p.d + f) * 1024u;
          sts32(lists + ((w * 3 + s) * C::LIST_LEN + (j - start)) * 4, code);
        }
      }
      // pad the on-chip lists to whole chunks with the class's dummy destination
#pragma unroll
      for (int w = 0; w < C::JMAX; ++w) {
        const int s = lane >> 4;
        int start, n;
        seg(w, s, start, n);
        sts32(lists + ((w * 3 + s) * C::LIST_LEN + n + (lane & 15)) * 4, s == 0 ? (uint32_t)C::TDUMMY : (uint32_t)(p.nS * 1024));
      }
      __syncwarp();
      MARK(31);
      if (lane == 0) mbar_arrive(&d_full[ps]);
    }
    MARK(32);
  } else {
    // ===================== epilogue: set = class owner, q = TMEM lane quadrant, lane = batch rows (row, row + 128) of the tile =====================
    const int set = warp >> 2, q = warp & 3;
    const int row = q * 32 + lane;
    const uint32_t tlane = tmem_base + ((uint32_t)(q * 32) << 16);
    const uint32_t sown = sbase + C::OFF_ACC + row * 8;                      // + accumulator row * 1024
    char* const gown = reinterpret_cast<char*>(p.dXw) + row * 8;             // + (tile * d + f) * 1024
    const int n_own = set == 0 ? p.nT : set == 1 ? p.nS : 0;                 // accumulators this set owns
    const int f_own = set == 0 ? F_lo : F_lo + p.nT;                         // feature of its accumulator 0
    // add this thread's words of every accumulator the set owns into the workspace rows of tile `t`, then clear them
    auto flush = [&](int t) {
      const bool vb = t * 256 + row < p.B;
      char* const g0 = gown + ((size_t)t * p.d + f_own) * 1024;
      if (set == 0) {
        dxp_tmem_st_wait();
        for (int c0 = 0; c0 < n_own; c0 += 8) {
          uint32_t a[8], b[8];
#pragma unroll
          for (int u = 0; u < 8; ++u) dxp_tld2(tlane + C::PB + 2 * min(c0 + u, C::T_MAX), a[u], b[u]);
          tmem_ld_wait();
#pragma unroll
          for (int u = 0; u < 8; ++u)
            if (vb && c0 + u < n_own) dxp_red2(g0 + (size_t)(c0 + u) * 1024, __uint_as_float(a[u]), __uint_as_float(b[u]));
        }
      } else if (set == 1 && vb) {
        for (int r = 0; r < n_own; ++r) {
          const float2 v = dxp_lds64f(sown + r * 1024);
          dxp_red2(g0 + (size_t)r * 1024, v.x, v.y);
        }
      }
    };
    auto clear = [&]() {
      if (set == 0) {
        for (int c = 0; c <= n_own; ++c) dxp_tst2(tlane + C::PB + 2 * min(c, C::T_MAX), 0u, 0u);
        dxp_tst2(tlane + C::TDUMMY, 0u, 0u);
        dxp_tmem_st_wait();
      } else if (set == 1) {
        for (int r = 0; r <= n_own; ++r) dxp_sts64f(sown + r * 1024, 0.f, 0.f);
      }
    };
    MARK(40);
    clear();
    MARK(41);
    int jc = 0, t_cur = n_my > 0 ? (int)(u0 / p.NG) : 0;
    for (int i = 0; i < n_my; ++i) {
      const int ps = i % C::RD;
      dxp_wait<64>(&d_full[ps], (i / C::RD) & 1);
      const uint32_t plan = sbase + C::OFF_PLAN + ps * C::PLAN_BYTES;
      const uint32_t lists = plan + C::PLAN_HDR * 4;
      const int njobs = dxp_lds32i(plan), t = dxp_lds32i(plan + 8);
      if (t != t_cur) { flush(t_cur); clear(); t_cur = t; }
      const bool vb = t * 256 + row < p.B;
      for (int w = 0; w < njobs; ++w, ++jc) {
        const int rs = jc % C::R;
        const int lo = dxp_lds32i(plan + (16 + w * 8 + 2 * set) * 4), n = dxp_lds32i(plan + (16 + w * 8 + 2 * set + 1) * 4);
        MARK(42);
        dxp_wait<64>(&t_full[rs], (jc / C::R) & 1);
        tc_fence_after();
        MARK(43);
        const uint32_t tp0 = tlane + rs * 2 * NW + lo, tp1 = tp0 + NW;
        const uint32_t lst = lists + (w * 3 + set) * C::LIST_LEN * 4;
#ifdef DXP_NO_EPI
        if (false) {
#else
        if (set == 0) {
#endif
          dxp_tmem_st_wait();                                   // earlier stores to these accumulator columns have landed
          int m = 0;
#pragma unroll 1
          for (; n - m > 8; m += 16) dxp_chunk_t<16>(tp0 + m, tp1 + m, lst + m * 4, tlane);
          if (n - m > 0) dxp_chunk_t<8>(tp0 + m, tp1 + m, lst + m * 4, tlane);
        } else if (set == 1
#ifdef DXP_NO_EPI
         && false
#endif
        ) {
          int m = 0;
#pragma unroll 1
          for (; n - m > 8; m += 16) dxp_chunk_s<16>(tp0 + m, tp1 + m, lst + m * 4, sown);
          if (n - m > 0) dxp_chunk_s<8>(tp0 + m, tp1 + m, lst + m * 4, sown);
        } else {
#ifdef DXP_NO_EPI
          if (false)
#endif
#pragma unroll 1
          for (int m = 0; m < n; m += 8) {
            uint32_t p0[8], p1[8];
            int dst[8];
            dxp_tmem_ld8(tp0 + m, p0);
            dxp_tmem_ld8(tp1 + m, p1);
            dxp_load_dest<8>(lst + m * 4, dst);
            tmem_ld_wait();
            if (vb) {
              if (m + 8 <= n) {
#pragma unroll
                for (int u = 0; u < 8; ++u) dxp_red2(gown + (uint32_t)dst[u], __uint_as_float(p0[u]), __uint_as_float(p1[u]));
              } else {
#pragma unroll
                for (int u = 0; u < 8; ++u)
                  if (m + u < n) dxp_red2(gown + (uint32_t)dst[u], __uint_as_float(p0[u]), __uint_as_float(p1[u]));
              }
            }
          }
        }
        MARK(44);
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&t_empty[rs]);
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&d_empty[ps]);
    }
    MARK(45);
    if (n_my > 0) flush(t_cur);
    MARK(46);
  }
  MARK(50);

  tc_fence_before();
  __syncthreads();
  MARK(51);
  if (CS > 1) dxp_cluster_sync();              // no CTA leaves while its peer may still multicast into it or arrive on its barriers
  if (warp == C::W_MMA) { tc_fence_after(); tmem_dealloc<512>(tmem_base); }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
template <int G, int K, int CS, int NW, int R>
static int launch_dx_pair(TcTailState* s, const TailShape& sh, const int32_t* idx, const void* W, const void* dY, float* dXw,
                          cudaStream_t st) {
  using C = DxPairCfg<G, K, CS, NW, R>;
  static_assert(C::S_MAX >= 8 && C::T_MAX >= 8, "no room for on-chip accumulators");
  static_assert(NW % 16 == 0 && NW <= 64 && 3 * C::JMAX <= 32, "job width");
  auto kern = tc_dx_pair_kernel<G, K, CS, NW, R>;
  const int smem = 232448;
  DxPairParams p;
  p.dXw = dXw; p.idx = idx; p.B = sh.B; p.d = sh.d; p.NT2 = ceil_div(sh.B, 256); p.NG = sh.NG;
  p.U = (int64_t)p.NT2 * sh.NG;
  if ((int64_t)p.NT2 * sh.d * 1024 > 0x7fffffffLL) return HASTE_ERR_UNSUPPORTED;   // list codes are 32-bit byte offsets
  p.Fc = ceil_div(sh.d, CS);
  p.nT = std::min(p.Fc, C::T_MAX);
  p.nS = std::min(p.Fc - p.nT, C::S_MAX);
  cudaLaunchConfig_t cfg = {};
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
#ifdef DXP_FORCE_CL2
  attr[0].val.clusterDim.x = 2;
#else
  attr[0].val.clusterDim.x = CS;
#endif
  attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.blockDim = dim3(C::THREADS); cfg.dynamicSmemBytes = smem; cfg.stream = st; cfg.attrs = attr; cfg.numAttrs = 1;
  if (s->pair_clusters == 0) {   // once per handle: (G, K) are fixed, so is the kernel
    HASTE_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    cfg.gridDim = dim3(CS * (s->num_sms / CS));
    int nc = 0;
    HASTE_CUDA_TRY(cudaOccupancyMaxActiveClusters(&nc, kern, &cfg));
    if (nc < 1) { set_error("tc_dx_pair: no cluster of %d CTAs fits on this device", CS); return HASTE_ERR_UNSUPPORTED; }
    s->pair_clusters = std::min(nc, s->num_sms / CS);
  }
  p.NP = (int)std::min<int64_t>(s->pair_clusters, p.U);
  cfg.gridDim = dim3(CS * p.NP);
#ifdef DXP_FORCE_CL2
  p.NP &= ~1; cfg.gridDim = dim3(p.NP);
#endif
  CUtensorMap tmY, tmW;
  {
    const uint64_t dims[3] = {(uint64_t)G, (uint64_t)sh.B, (uint64_t)sh.NG};
    const uint64_t str[2] = {(uint64_t)G * 2, (uint64_t)sh.B * G * 2};
    const uint32_t box[3] = {(uint32_t)std::min(G, 64), 256 / CS, 1};
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
#ifdef DXP_DEBUG
  static int* dbg_h = nullptr;
  if (!dbg_h) cudaHostAlloc(&dbg_h, 512 * 32 * 4, cudaHostAllocMapped);
  memset(dbg_h, 0, 512 * 32 * 4);
  int* dbg_d = nullptr; cudaHostGetDevicePointer(&dbg_d, dbg_h, 0);
  p.dbg = dbg_d;
#endif
  HASTE_CUDA_TRY(cudaLaunchKernelEx(&cfg, kern, tmY, tmW, p));
#ifdef DXP_DEBUG
  if (cudaStreamSynchronize(st) != cudaSuccess) {
    for (int b = 0; b < 4; ++b) { fprintf(stderr, "cta %d:", b); for (int w = 0; w < 16; ++w) fprintf(stderr, " %d", dbg_h[b * 32 + w]); fprintf(stderr, "\n"); }
  }
#endif
  HASTE_LAUNCH_CHECK();
  return HASTE_OK;
}

bool tc_tail_dx_pair_supported(const TailShape& sh) {
  // one 128-row tile would leave half of every instruction idle: tc_dx_acc.cu is the kernel for small batches
  return sh.B > 128 && (sh.G == 32 || sh.G == 64 || sh.G == 128) && (sh.K == 64 || sh.K == 128) &&
         (int64_t)ceil_div(sh.B, 256) * sh.d * 1024 <= 0x7fffffffLL;
}

int tc_tail_dx_pair(TcTailState* s, const TailShape& sh, const int32_t* idx, const void* W, const void* dY, float* dXw,
                    cudaStream_t st) {
#define HASTE_DXP(G_, K_, NW_, R_) \
  if (sh.G == G_ && sh.K == K_) return launch_dx_pair<G_, K_, DXP_CS, NW_, R_>(s, sh, idx, W, dY, dXw, st)
  HASTE_DXP(64, 128, 48, 2); HASTE_DXP(64, 64, 48, 2); HASTE_DXP(128, 64, 48, 2); HASTE_DXP(128, 128, 48, 2);
  HASTE_DXP(32, 64, 48, 2); HASTE_DXP(32, 128, 48, 2);
#undef HASTE_DXP
  return HASTE_ERR_UNSUPPORTED;
}

}  // namespace haste
