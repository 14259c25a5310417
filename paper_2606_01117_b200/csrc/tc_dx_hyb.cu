// tc_dx_hyb.cu -- input-gradient kernel of the HASTE sparse tail: tc_dx_acc.cu with its TMEM class moved onto the tensor
// cores (sm_100a; bf16 in, fp32 accumulate).
//
//   dX[:, idx_g] += dY_g [B x G] * W_g [G x K]   over all groups g
//
// tc_dx_acc.cu is issue-slot bound, and its TMEM class is the most expensive one (~7 instructions per slot and warp: the
// TMEM address of tcgen05.ld/st has to sit in a uniform register).  Here that class costs no issue slots:
//   T  = [0,  f1)   accumulator columns in TMEM, updated by SCATTER MMAs: ACC[128 x 64 window] += P[:, 8 slots] * S, where
//                   the fp32 P tile in TMEM is read as the tf32 A operand and S [64 x 8] in shared memory is one-hot
//                   (S[n][k] = 1 iff slot k goes to column start + n); see tc_dx_mma.cu / profiles/r01_probe_scatter_mma.txt
//   S0..S3 = [f1, f2) in four quarters: fp32 accumulator rows in shared memory, one owner set of 4 warps each
//   L  = [f2, d)    red.global.add.f32 into dX^T (also every slot of a group whose idx row is not strictly increasing
//                   or whose scatter plan does not fit: the atomic path is correct for any row)
// Per group: TMA loads the dY tile and W_g; the issuing warp computes P^T [128 x K] into one of two TMEM buffers and,
// one group later (P is complete by then: a TMEM A operand is NOT ordered behind the MMA that wrote it), issues that
// group's scatter MMAs; four auxiliary warps turn idx_g into the scatter plan and the S/L destination lists; sixteen
// epilogue warps (4 owner sets x 4 TMEM lane quadrants, a lane owns one batch row) do the S and L classes.
// P is read at tf32 precision by the scatter MMAs (rel. 2^-11 per term of the T class; the product by 1.0 and the fp32
// accumulation are exact; integers below 2048 stay exact).
#include <algorithm>
#include <cstdlib>

#include "tc_common.cuh"
#include "tc_kernels.h"

namespace haste {
using namespace tc;

struct DxHybParams {
  float* dXt;           // [d][Bpad] fp32, zeroed by the caller
  const int32_t* idx;   // [NG][K]
  int B, Bpad, NT, S, d;
  int64_t NG;
  int f1, f2;           // class boundaries (see above): T = [0,f1), S = [f1,f2), L = [f2,d)
};

template <int G, int K, int NST_> struct DxHybCfg {
  static constexpr int NSET = 4;                              // epilogue sets: set s owns the s-th quarter of the shared-memory rows
  static constexpr int NLIST = NSET + 1;                      // + the L list
  static constexpr int Y_BYTES = G * 256;                     // [G/64 k-blocks][128 batch rows][128 B]; G = 32: [128 rows][64 B]
  static constexpr int W_BYTES = G * K * 2;                   // [K/64 slot atoms][G label rows][128 B]
  static constexpr int STAGE = Y_BYTES + W_BYTES;
  static constexpr int NST = NST_;                            // operand stages (dY tile + W_g) in flight
  static constexpr int LIST_LEN = K + 16;                     // entries per list (padding for the last chunk)
  static constexpr int RING_META = 48;                        // lo[5] at 0, n[5] at 20
  static constexpr int RING_BYTES = (RING_META + NLIST * LIST_LEN * 4 + 127) / 128 * 128;
  static constexpr int RD = 4;                                // depth of the destination-list ring = number of auxiliary warps
  static constexpr int TF = 512 - 2 * K;                      // TMEM accumulator columns (T class), next to the two P buffers
  static constexpr int NPL = 2;                               // scatter-plan ring (group i uses slot i mod 2)
  static constexpr int MAXT = 12;                             // scatter MMAs per group; a group that needs more goes to the L class
  static constexpr int S_BYTES = 2048;                        // one S matrix: [64 n][8 k] tf32, K-major, no swizzle
  static constexpr int PLAN_BYTES = MAXT * S_BYTES + 128;     // S matrices, then entries [MAXT] x 4 B at +0 and {n issue, n dirty} at +64
  static constexpr int OFF_RING = NST * STAGE;
  static constexpr int OFF_PLAN = (OFF_RING + RD * RING_BYTES + 1023) / 1024 * 1024;
  static constexpr int OFF_BAR = OFF_PLAN + NPL * PLAN_BYTES;
  static constexpr int NBAR = 2 * NST + 4 + 2 * RD + 3 * NPL + 1;
  static constexpr int OFF_MISC = OFF_BAR + NBAR * 8;
  static constexpr int OFF_ACC = (OFF_MISC + 64 + 511) / 512 * 512;
  static constexpr int NS_MAX = (232448 - 1024 - OFF_ACC) / 512 - 1;   // shared-memory accumulator rows (+1 dummy row)
  static constexpr bool FITS = NS_MAX >= 64;                  // otherwise use fewer stages
  static constexpr int NAUX = RD;                             // auxiliary warps: warp a builds plan and lists of groups i = a (mod NAUX)
  static constexpr int THREADS = (4 * NSET + 2 + NAUX) * 32;
};

__device__ __forceinline__ void dxh_red_add_f32(float* addr, float v) {
  asm volatile("red.global.add.f32 [%0], %1;" ::"l"(addr), "f"(v) : "memory");
}
__device__ __forceinline__ uint32_t dxh_tld1(uint32_t taddr) {
  uint32_t v;
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(v) : "r"(taddr) : "memory");
  return v;
}
__device__ __forceinline__ void dxh_tst1(uint32_t taddr, uint32_t v) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};" ::"r"(taddr), "r"(v) : "memory");
}
__device__ __forceinline__ void dxh_tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ int4 dxh_lds128i(uint32_t addr) {
  int4 v;
  asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
  return v;
}
__device__ __forceinline__ int dxh_lds32i(uint32_t addr) {
  int v;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ float dxh_lds32f(uint32_t addr) {
  float v;
  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ void dxh_sts32f(uint32_t addr, float v) {
  asm volatile("st.shared.f32 [%0], %1;" ::"r"(addr), "f"(v) : "memory");
}
__device__ __forceinline__ void dxh_red_add_f32(const char* addr, float v) {
  asm volatile("red.global.add.f32 [%0], %1;" ::"l"(addr), "f"(v) : "memory");
}
__device__ __forceinline__ void dxh_tmem_ld8(uint32_t taddr, uint32_t (&v)[8]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
               : "r"(taddr)
               : "memory");
}
template <int N> __device__ __forceinline__ void dxh_tmem_ldn(uint32_t taddr, uint32_t (&v)[N]);
template <> __device__ __forceinline__ void dxh_tmem_ldn<16>(uint32_t taddr, uint32_t (&v)[16]) { tmem_ld16(taddr, v); }
template <> __device__ __forceinline__ void dxh_tmem_ldn<8>(uint32_t taddr, uint32_t (&v)[8]) { dxh_tmem_ld8(taddr, v); }
template <> __device__ __forceinline__ void dxh_tmem_ldn<24>(uint32_t taddr, uint32_t (&v)[24]) {
  tmem_ld16(taddr, reinterpret_cast<uint32_t(&)[16]>(v[0]));
  dxh_tmem_ld8(taddr + 16, reinterpret_cast<uint32_t(&)[8]>(v[16]));
}
// N destination codes of one chunk of a list (16-byte aligned)
template <int N> __device__ __forceinline__ void dxh_load_dest(uint32_t addr, int (&dst)[N]) {
#pragma unroll
  for (int i = 0; i < N / 4; ++i) {
    const int4 a = dxh_lds128i(addr + i * 16);
    dst[4 * i] = a.x; dst[4 * i + 1] = a.y; dst[4 * i + 2] = a.z; dst[4 * i + 3] = a.w;
  }
}
// one chunk of N slots of a shared-memory class: acc row (byte offset dst[u]), this thread's word += P column u
template <int N> __device__ __forceinline__ void dxh_chunk_s(uint32_t tp, uint32_t lst, uint32_t sown) {
  uint32_t pv[N];
  float a[N];
  int dst[N];
  dxh_tmem_ldn<N>(tp, pv);
  dxh_load_dest<N>(lst, dst);
#pragma unroll
  for (int u = 0; u < N; ++u) a[u] = dxh_lds32f(sown + dst[u]);
  tmem_ld_wait();
#pragma unroll
  for (int u = 0; u < N; ++u) dxh_sts32f(sown + dst[u], a[u] + __uint_as_float(pv[u]));
}

// 20 warps poll barriers here; a polling loop costs issue slots the working warps need, so back off between polls
// shared-memory matrix descriptor without swizzle (layout type 0): core matrices of 8 rows x 16 B
__device__ __forceinline__ uint64_t dxh_sdesc_none(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr >> 4) & 0x3FFF);
  d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16;
  d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32;
  d |= (uint64_t)1 << 46;
  return d;
}
// ACC[tmem d] += P[tmem a] (tf32, 128 x 8) * S[smem desc] (tf32, 8 x 64)
__device__ __forceinline__ void dxh_umma_scatter(uint32_t d_tmem, uint32_t a_tmem, uint64_t bdesc, uint32_t idesc) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, 1, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}"
      ::"r"(d_tmem), "r"(a_tmem), "l"(bdesc), "r"(idesc)
      : "memory");
}
__device__ __forceinline__ uint4 dxh_lds128u(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ void dxh_tst16z(uint32_t taddr) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1};" ::"r"(taddr),
      "r"(0u)
      : "memory");
}
template <int NS_SLEEP> __device__ __forceinline__ void dxh_wait(uint64_t* bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) __nanosleep(NS_SLEEP);
}

template <int G, int K, int NST>
__global__ void __launch_bounds__(DxHybCfg<G, K, NST>::THREADS, 1)
tc_dx_hyb_kernel(const __grid_constant__ CUtensorMap tmY, const __grid_constant__ CUtensorMap tmW, const DxHybParams p) {
  using C = DxHybCfg<G, K, NST>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const uint32_t sbase = smem_u32(smem);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::OFF_BAR);
  uint64_t* full = bars;                    // [NST] TMA (tx) -> MMA
  uint64_t* empty = bars + C::NST;          // [NST] MMA commit -> TMA
  uint64_t* t_full = bars + 2 * C::NST;     // [2]   P MMA commit -> epilogue warps AND the issuer (before its scatter MMAs)
  uint64_t* t_empty = t_full + 2;           // [2]   16 epilogue warps -> MMA
  uint64_t* d_full = t_empty + 2;           // [RD]  aux warp -> epilogue (destination lists ready)
  uint64_t* d_empty = d_full + C::RD;       // [RD]  16 epilogue warps -> aux warp
  uint64_t* pl_full = d_empty + C::RD;      // [NPL] aux warp -> issuer (scatter plan ready)
  uint64_t* pl_empty = pl_full + C::NPL;    // [NPL][2] scatter MMA commit -> aux warp.  Two aux warps alternate on a plan slot, so the
                                            // uses of a slot alternate between two barriers: each barrier then has ONE waiter, in order
                                            // (with one barrier a warp two uses ahead would pass on the stale parity and deadlock the ring)
  uint64_t* done = pl_empty + 2 * C::NPL;   // [1]   last MMA commit -> flush of the TMEM accumulator
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + C::OFF_MISC);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int bt = blockIdx.x % p.NT, stripe = blockIdx.x / p.NT;
  const int n_my = p.NG > stripe ? (int)((p.NG - stripe + p.S - 1) / p.S) : 0;
  const int NS = p.f2 - p.f1;               // shared-memory accumulator rows in use; row NS is the dummy
  constexpr int EW = 4 * C::NSET;           // epilogue warps

  if (threadIdx.x == 0) {
    for (int i = 0; i < C::NST; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&t_full[i], 1); mbar_init(&t_empty[i], EW); }
    for (int i = 0; i < C::RD; ++i) { mbar_init(&d_full[i], 1); mbar_init(&d_empty[i], EW); }
    for (int i = 0; i < C::NPL; ++i) { mbar_init(&pl_full[i], 1); mbar_init(&pl_empty[2 * i], 1); mbar_init(&pl_empty[2 * i + 1], 1); }
    mbar_init(done, 1);
    fence_barrier_init();
  }
  // every S matrix of the plan ring starts as zeros; {n issue, n dirty} = {0, 0}
  for (int o = threadIdx.x * 16; o < C::NPL * C::PLAN_BYTES; o += blockDim.x * 16) sts128(sbase + C::OFF_PLAN + o, 0u, 0u, 0u, 0u);
  if (warp == EW + 1 && lane == 0) { tma_prefetch_desc(&tmY); tma_prefetch_desc(&tmW); }
  if (warp == EW) tmem_alloc<512>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  if (warp < 4) {                            // zero the T accumulator: columns [2K, 512) of this warp's lane quadrant
    const uint32_t tl = tmem_base + ((uint32_t)(warp * 32) << 16);
    for (int c = 2 * K; c < 512; c += 16) dxh_tst16z(tl + c);
    dxh_tmem_st_wait();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();

  if (warp == EW + 1) {
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
  } else if (warp == EW) {
    // ===================== MMA issuer (whole warp waits, one elected lane issues) =====================
    // queue:  P(0)  P(1)  scatter(0)  P(2)  scatter(1)  ...   scatter(i-1) is issued one group late, after this warp has
    // itself seen P(i-1)'s commit: nothing orders an MMA's read of a TMEM A operand behind the MMA that wrote those columns.
    // P(i+1) reuses P(i-1)'s buffer: it follows scatter(i-1) in issue order, and waits for the epilogue warps' release.
    constexpr uint32_t idesc = make_idesc_bf16(128, K, /*A (dY) K-major*/ 0, /*B (W) MN-major*/ 1);
    constexpr uint32_t idesc_s = (1u << 4) | (2u << 7) | (2u << 10) | ((64u >> 3) << 17) | ((128u >> 4) << 24);   // tf32 x tf32 -> f32, M 128, N 64
    // A = the dY tile, K-major: 128-byte rows (64 labels per k-block) or, for G = 32, 64-byte rows with the 64-byte swizzle
    const uint64_t adesc0 = G >= 64 ? make_sdesc_sw128(sbase, 16, 1024) : make_sdesc_sw64(sbase, 16, 512);
    const uint64_t bdesc0 = make_sdesc_sw128(sbase + C::Y_BYTES, G * 128, 1024);
    const uint64_t sdesc0 = dxh_sdesc_none(sbase + C::OFF_PLAN, 128, 256);
    auto scatter = [&](int j) {               // scatter MMAs of group j (its plan is in slot j mod NPL, its P in buffer j & 1)
      const int ps = j % C::NPL;
      mbar_wait(&t_full[j & 1], (j >> 1) & 1);
      mbar_wait(&pl_full[ps], (j / C::NPL) & 1);
      tc_fence_after();
      const uint32_t plan = sbase + C::OFF_PLAN + ps * C::PLAN_BYTES + C::MAXT * C::S_BYTES;
      const uint32_t n = (uint32_t)dxh_lds32i(plan + 64);
      uint32_t en[C::MAXT];
#pragma unroll
      for (int e = 0; e < C::MAXT; e += 4)
        if ((uint32_t)e < n) { const uint4 v = dxh_lds128u(plan + e * 4); en[e] = v.x; en[e + 1] = v.y; en[e + 2] = v.z; en[e + 3] = v.w; }
      if (elect_one()) {
        const uint64_t sd = sdesc0 + (uint64_t)((ps * C::PLAN_BYTES) >> 4);
        const uint32_t pbuf = tmem_base + (j & 1) * K, acc = tmem_base + 2 * K;
#pragma unroll
        for (int e = 0; e < C::MAXT; ++e)
          if ((uint32_t)e < n) dxh_umma_scatter(acc + (en[e] & 511u), pbuf + (en[e] >> 9) * 8, sd + (uint64_t)((e * C::S_BYTES) >> 4), idesc_s);
        umma_commit(&pl_empty[2 * ps + ((j / C::NPL) & 1)]);
      }
      __syncwarp();
    };
    for (int i = 0; i < n_my; ++i) {
      const int st = i % C::NST, slot = i & 1;
      mbar_wait(&full[st], (i / C::NST) & 1);
      mbar_wait(&t_empty[slot], ((i >> 1) & 1) ^ 1);
      tc_fence_after();
      if (elect_one()) {
        const uint64_t so = (uint64_t)((st * C::STAGE) >> 4);
        const uint32_t d = tmem_base + slot * K;
#pragma unroll
        for (int j = 0; j < G / 16; ++j)
          umma_f16(d, adesc0 + so + (uint64_t)(((j >> 2) * 16384 + (j & 3) * 32) >> 4), bdesc0 + so + (uint64_t)((j * 2048) >> 4),
                   idesc, j ? 1u : 0u);
        umma_commit(&empty[st]);
        umma_commit(&t_full[slot]);
      }
      __syncwarp();
      if (i > 0) scatter(i - 1);
    }
    if (n_my > 0) scatter(n_my - 1);
    if (elect_one()) umma_commit(done);
    __syncwarp();
  } else if (warp >= EW + 2) {
    // ===================== auxiliary warps: idx_g -> scatter plan (T class) + destination lists (S and L classes) =====================
    constexpr int PER = K / 32;
    const int aw = warp - (EW + 2);
    const int f1 = p.f1;
    const int fq0 = f1 + NS / 4, fq1 = f1 + NS / 2, fq2 = f1 + 3 * NS / 4, fq3 = p.f2;   // ends of the four shared-memory quarters
    const bool own = lane < K / 8;            // plan layout: lane l owns the 8-slot block l
    int e_[PER], en_[PER];                    // list layout: lane holds slots j = lane + 32 t
    int4 b0 = make_int4(0, 0, 0, 0), b1 = b0, nb0 = b0, nb1 = b0;
#pragma unroll
    for (int t = 0; t < PER; ++t) { e_[t] = 0; en_[t] = 0; }
    if (aw < n_my) {
      const int32_t* row = p.idx + (stripe + (int64_t)aw * p.S) * K;
#pragma unroll
      for (int t = 0; t < PER; ++t) en_[t] = __ldg(row + lane + 32 * t);
      if (own) { nb0 = __ldg(reinterpret_cast<const int4*>(row + lane * 8)); nb1 = __ldg(reinterpret_cast<const int4*>(row + lane * 8) + 1); }
    }
    for (int i = aw; i < n_my; i += C::NAUX) {
      const int64_t g = stripe + (int64_t)i * p.S;
      const int r = i % C::RD, ps = i % C::NPL;
#pragma unroll
      for (int t = 0; t < PER; ++t) e_[t] = en_[t];
      b0 = nb0; b1 = nb1;
      if (i + C::NAUX < n_my) {
        const int32_t* row = p.idx + (g + (int64_t)C::NAUX * p.S) * K;
#pragma unroll
        for (int t = 0; t < PER; ++t) en_[t] = __ldg(row + lane + 32 * t);
        if (own) { nb0 = __ldg(reinterpret_cast<const int4*>(row + lane * 8)); nb1 = __ldg(reinterpret_cast<const int4*>(row + lane * 8) + 1); }
      }
      // strictly increasing?  (slot j+1 is the next lane's value, or lane 0's value of the next t)
      bool inc = true;
#pragma unroll
      for (int t = 0; t < PER; ++t) {
        int nxt = __shfl_down_sync(0xffffffffu, e_[t], 1);
        const int wrap = __shfl_sync(0xffffffffu, t + 1 < PER ? e_[(t + 1) % PER] : 0x7fffffff, 0);
        if (lane == 31) nxt = wrap;
        inc &= e_[t] < nxt;
      }
      const bool strict = __all_sync(0xffffffffu, inc);

      // ---------------- scatter plan of the T class: one MMA per (8-slot block, 64-column window)
      const int f[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
      uint32_t rem = 0;
      if (own && strict) {
#pragma unroll
        for (int k = 0; k < 8; ++k) rem |= (uint32_t)(f[k] < f1) << k;
      }
      const uint32_t plan = sbase + C::OFF_PLAN + ps * C::PLAN_BYTES;
      const uint32_t pmeta = plan + C::MAXT * C::S_BYTES;
      // The plan is worked out twice: first on registers only, to know whether it fits (the lists depend on that and the
      // epilogue warps wait for the lists), then again with the stores, once the plan slot is free.
      auto rounds = [&](uint32_t rem0, bool write, bool& ovf) -> int {
        uint32_t rem = rem0;
        int base = 0;
        ovf = false;
        for (;;) {
          const uint32_t bal = __ballot_sync(0xffffffffu, rem != 0);
          if (bal == 0) break;
          const int cnt = __popc(bal);
          if (base + cnt > C::MAXT) { ovf = true; break; }
          if (rem != 0) {
            const int e = base + __popc(bal & ((1u << lane) - 1u));
            int fmin = 0x7fffffff;
#pragma unroll
            for (int k = 0; k < 8; ++k) if ((rem >> k) & 1u) fmin = min(fmin, f[k]);
            const int start = min(fmin & ~3, C::TF - 64);
            const uint32_t s_e = plan + e * C::S_BYTES;
#pragma unroll
            for (int k = 0; k < 8; ++k) {
              const int n = f[k] - start;
              if (((rem >> k) & 1u) && n < 64) {          // n >= 0 because start <= fmin
                if (write) sts32(s_e + (n >> 3) * 256 + (k >> 2) * 128 + (n & 7) * 16 + (k & 3) * 4, 0x3f800000u);
                rem &= ~(1u << k);
              }
            }
            if (write) sts32(pmeta + e * 4, (uint32_t)((lane << 9) | start));   // {8-slot block, first accumulator column}; S matrix = entry index
          }
          base += cnt;
        }
        return base;
      };
      bool ovf = false;
      const int n_plan = rounds(rem, false, ovf);
      const bool onchip = strict && !ovf;       // otherwise every slot of the group goes through the L class

      // ---------------- destination lists of the S quarters and of the L class
      int cT = 0, c0 = 0, c1 = 0, c2 = 0, c3 = 0;
#pragma unroll
      for (int t = 0; t < PER; ++t) { cT += e_[t] < f1; c0 += e_[t] < fq0; c1 += e_[t] < fq1; c2 += e_[t] < fq2; c3 += e_[t] < fq3; }
      cT = __reduce_add_sync(0xffffffffu, cT); c0 = __reduce_add_sync(0xffffffffu, c0); c1 = __reduce_add_sync(0xffffffffu, c1);
      c2 = __reduce_add_sync(0xffffffffu, c2); c3 = __reduce_add_sync(0xffffffffu, c3);
      if (!onchip) { cT = 0; c0 = 0; c1 = 0; c2 = 0; c3 = 0; }
      dxh_wait<64>(&d_empty[r], ((i / C::RD) & 1) ^ 1);
      const uint32_t ring = sbase + C::OFF_RING + r * C::RING_BYTES;
      const uint32_t lists = ring + C::RING_META;
      // lists 0..3 = quarters [cT,c0) [c0,c1) [c1,c2) [c2,c3); list 4 = L [c3,K)
      if (lane == 0) {
        sts32(ring + 0, (uint32_t)cT); sts32(ring + 4, (uint32_t)c0); sts32(ring + 8, (uint32_t)c1); sts32(ring + 12, (uint32_t)c2);
        sts32(ring + 16, (uint32_t)c3);
        sts32(ring + 20, (uint32_t)(c0 - cT)); sts32(ring + 24, (uint32_t)(c1 - c0)); sts32(ring + 28, (uint32_t)(c2 - c1));
        sts32(ring + 32, (uint32_t)(c3 - c2)); sts32(ring + 36, (uint32_t)(K - c3));
      }
#pragma unroll
      for (int t = 0; t < PER; ++t) {
        const int j = lane + 32 * t, fj = e_[t];
        if (j >= cT) {
          int l, k, code;
          if (j < c0)      { l = 0; k = j - cT; code = (fj - f1) * 512; }          // byte offset of the accumulator row
          else if (j < c1) { l = 1; k = j - c0; code = (fj - f1) * 512; }
          else if (j < c2) { l = 2; k = j - c1; code = (fj - f1) * 512; }
          else if (j < c3) { l = 3; k = j - c2; code = (fj - f1) * 512; }
          else             { l = 4; k = j - c3; code = fj * p.Bpad * 4; }          // byte offset of the dX^T row
          sts32(lists + (l * C::LIST_LEN + k) * 4, (uint32_t)code);
        }
      }
      // pad the on-chip lists to a whole chunk with the dummy row
      if (lane < 16) {
        sts32(lists + (0 * C::LIST_LEN + (c0 - cT) + lane) * 4, (uint32_t)(NS * 512));
        sts32(lists + (1 * C::LIST_LEN + (c1 - c0) + lane) * 4, (uint32_t)(NS * 512));
        sts32(lists + (2 * C::LIST_LEN + (c2 - c1) + lane) * 4, (uint32_t)(NS * 512));
        sts32(lists + (3 * C::LIST_LEN + (c3 - c2) + lane) * 4, (uint32_t)(NS * 512));
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&d_full[r]);

      // ---------------- now the plan itself
      {                                                       // the scatter MMAs of the slot's previous use have completed
        const int n = i / C::NPL;
        if (n > 0) mbar_wait(&pl_empty[2 * ps + ((n - 1) & 1)], ((n - 1) >> 1) & 1);
      }
      {
        const int ndirty = dxh_lds32i(pmeta + 68);
        for (int e = 0; e < ndirty; ++e) {
          const uint32_t a = plan + e * C::S_BYTES + lane * 64;
          sts128(a, 0u, 0u, 0u, 0u); sts128(a + 16, 0u, 0u, 0u, 0u); sts128(a + 32, 0u, 0u, 0u, 0u); sts128(a + 48, 0u, 0u, 0u, 0u);
        }
      }
      __syncwarp();
      if (onchip) { bool o2; rounds(rem, true, o2); }
      fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) {
        sts32(pmeta + 64, onchip ? (uint32_t)n_plan : 0u);     // scatter MMAs to issue
        sts32(pmeta + 68, onchip ? (uint32_t)n_plan : 0u);     // S matrices that hold ones
        mbar_arrive(&pl_full[ps]);
      }
    }
  } else {
    // ===================== epilogue: set = owner of one quarter of the shared-memory rows, q = TMEM lane quadrant, lane = batch row =====================
    const int set = warp >> 2, q = warp & 3;
    const int row = q * 32 + lane;
    const int b = bt * 128 + row;
    const bool vb = b < p.B;
    const uint32_t tlane = tmem_base + ((uint32_t)(q * 32) << 16);
    const uint32_t sown = sbase + C::OFF_ACC + row * 4;                      // + accumulator row * 512
    float* const gcol = p.dXt + b;                                           // + f * Bpad
    const char* const gbytes = reinterpret_cast<const char*>(gcol);          // + byte offset of the dX^T row (L list code)
    const int c_lo = set == 0 ? 0 : set == 1 ? NS / 4 : set == 2 ? NS / 2 : 3 * NS / 4;      // this set's accumulator rows
    const int c_hi = set == 0 ? NS / 4 : set == 1 ? NS / 2 : set == 2 ? 3 * NS / 4 : NS;
    for (int r = c_lo; r < c_hi; ++r) dxh_sts32f(sown + r * 512, 0.f);
    for (int i = 0; i < n_my; ++i) {
      const int r = i % C::RD, slot = i & 1;
      dxh_wait<64>(&d_full[r], (i / C::RD) & 1);
      const uint32_t ring = sbase + C::OFF_RING + r * C::RING_BYTES;
      const uint32_t lists = ring + C::RING_META;
      const int lo_s = dxh_lds32i(ring + set * 4), n_s = dxh_lds32i(ring + 20 + set * 4);
      const int lo_l = dxh_lds32i(ring + C::NSET * 4), n_l = dxh_lds32i(ring + 20 + C::NSET * 4);
      dxh_wait<64>(&t_full[slot], (i >> 1) & 1);
      tc_fence_after();
      const uint32_t tp = tlane + slot * K;
      const uint32_t lst = lists + set * C::LIST_LEN * 4;
      {
        int m = 0;
#pragma unroll 1
        for (; n_s - m > 16; m += 16) dxh_chunk_s<16>(tp + lo_s + m, lst + m * 4, sown);
        // the rest in ONE pass (8 or 16 slots): a chunk is one latency chain
        if (n_s - m > 8) dxh_chunk_s<16>(tp + lo_s + m, lst + m * 4, sown);
        else if (n_s - m > 0) dxh_chunk_s<8>(tp + lo_s + m, lst + m * 4, sown);
      }
      // the L class: red.global is atomic, so chunks need no owner: dealt round-robin to the sets.  No dummy target here:
      // a shared dummy word in L2 would serialise the reductions of every CTA on one address.
      const uint32_t lstl = lists + C::NSET * C::LIST_LEN * 4;
#pragma unroll 1
      for (int m = ((set + i) & 3) * 16; m < n_l; m += C::NSET * 16) {
        uint32_t pv[16];
        int dst[16];
        tmem_ld16(tp + lo_l + m, pv);
        dxh_load_dest<16>(lstl + m * 4, dst);
        tmem_ld_wait();
        if (vb) {
          if (m + 16 <= n_l) {
#pragma unroll
            for (int u = 0; u < 16; ++u) dxh_red_add_f32(gbytes + (uint32_t)dst[u], __uint_as_float(pv[u]));
          } else {
#pragma unroll
            for (int u = 0; u < 16; ++u)
              if (m + u < n_l) dxh_red_add_f32(gbytes + (uint32_t)dst[u], __uint_as_float(pv[u]));
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) { mbar_arrive(&t_empty[slot]); mbar_arrive(&d_empty[r]); }
    }
    // flush this thread's accumulators (its batch row of every feature this set owns) into dX^T
    if (vb) {
      for (int r = c_lo; r < c_hi; ++r) dxh_red_add_f32(gcol + (size_t)(p.f1 + r) * p.Bpad, dxh_lds32f(sown + r * 512));
    }
    if (set == 0) {                          // and the T accumulator (TMEM columns [2K, 2K + f1)), once the last scatter MMA is done
      mbar_wait(done, 0);
      tc_fence_after();
      for (int c0 = 0; c0 < p.f1; c0 += 16) {
        uint32_t v[16];
        tmem_ld16(tlane + 2 * K + min(c0, C::TF - 16), v);
        tmem_ld_wait();
        if (vb) {
          const int cc = min(c0, C::TF - 16);
#pragma unroll
          for (int u = 0; u < 16; ++u) {
            const int c = cc + u;
            if (c >= c0 && c < p.f1) dxh_red_add_f32(gcol + (size_t)c * p.Bpad, __uint_as_float(v[u]));
          }
        }
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == EW) { tc_fence_after(); tmem_dealloc<512>(tmem_base); }
}

template <int G, int K, int NST>
static int launch_dx_hyb(TcTailState* s, const TailShape& sh, const int32_t* idx, const void* W, const void* dY, float* dXt,
                         cudaStream_t st) {
  using C = DxHybCfg<G, K, NST>;
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
  DxHybParams p;
  p.dXt = dXt; p.idx = idx; p.B = sh.B; p.Bpad = sh.Bpad; p.NT = ceil_div(sh.B, 128); p.NG = sh.NG; p.d = sh.d;
  if (p.NT > s->num_sms) return HASTE_ERR_UNSUPPORTED;
  if ((int64_t)sh.d * sh.Bpad * 4 > 0x7fffffff) return HASTE_ERR_UNSUPPORTED;   // list codes are 32-bit byte offsets
  p.S = (int)std::min<int64_t>(sh.NG, std::max(1, s->num_sms / p.NT));
  // class sizes: what fits (tuning knobs for experiments: HASTE_DX_F1, HASTE_DX_NS)
  int f1 = std::min(sh.d, C::TF) & ~3, ns = C::NS_MAX;
  if (const char* e = getenv("HASTE_DX_F1")) f1 = std::max(0, std::min(f1, atoi(e))) & ~3;
  if (const char* e = getenv("HASTE_DX_NS")) ns = std::max(0, std::min(ns, atoi(e)));
  ns = std::min(ns, sh.d - f1);
  p.f1 = f1; p.f2 = f1 + ns;
  const int smem = C::OFF_ACC + (ns + 1) * 512 + 1024;
  HASTE_CUDA_TRY(cudaFuncSetAttribute(tc_dx_hyb_kernel<G, K, NST>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  tc_dx_hyb_kernel<G, K, NST><<<p.NT * p.S, C::THREADS, smem, st>>>(tmY, tmW, p);
  HASTE_LAUNCH_CHECK();
  return HASTE_OK;
}

int tc_tail_dx_hyb(TcTailState* s, const TailShape& sh, const int32_t* idx, const void* W, const void* dY, float* dXt,
                   cudaStream_t st) {
  // operand stages: as many as leave room for a useful number of shared-memory accumulator rows
  static const int nst_env = getenv("HASTE_DX_NST") ? atoi(getenv("HASTE_DX_NST")) : 0;
#define HASTE_DXH(G_, K_, DEF_)                                                                       \
  if (sh.G == G_ && sh.K == K_) {                                                                     \
    const int nst = nst_env ? nst_env : DEF_;                                                         \
    if constexpr (DxHybCfg<G_, K_, 4>::FITS) if (nst == 4) return launch_dx_hyb<G_, K_, 4>(s, sh, idx, W, dY, dXt, st);  \
    if constexpr (DxHybCfg<G_, K_, 3>::FITS) if (nst == 3) return launch_dx_hyb<G_, K_, 3>(s, sh, idx, W, dY, dXt, st);  \
    return launch_dx_hyb<G_, K_, 2>(s, sh, idx, W, dY, dXt, st);                                       \
  }
  HASTE_DXH(64, 128, 2); HASTE_DXH(64, 64, 2); HASTE_DXH(128, 64, 2); HASTE_DXH(128, 128, 2);
  HASTE_DXH(32, 64, 2); HASTE_DXH(32, 128, 2);
#undef HASTE_DXH
  return HASTE_ERR_UNSUPPORTED;
}

}  // namespace haste
