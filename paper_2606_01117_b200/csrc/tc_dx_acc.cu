// tc_dx_acc.cu -- input-gradient kernel of the HASTE sparse tail with the reduction over groups kept ON CHIP
// (sm_100a; bf16 in, fp32 accumulate).
//
//   dX[:, idx_g] += dY_g [B x G] * W_g [G x K]   over all groups g
//
// Why: the B*NG*K scatter-adds (669 M at config 3) go through L2 reductions at no more than ~1.47 T adds/s
// (profiles/r01_probe_microbench.txt), 3.5x the kernel's HBM floor, and a shared-memory accumulator for all d
// features of a 128-row batch tile does not fit (d * 512 B).  Measured on this B200
// (profiles/r01_probe_onchip_rmw.txt): read-modify-write of a thread-owned word runs at ~12 adds/clk/SM in
// shared memory AND at ~12 adds/clk/SM in tensor memory (tcgen05.ld/st .x1 at a dynamic column); the two, and
// the L2 reduction path, are independent resources.  So the features are split by id into five classes, and
// because an idx row is sorted each class is a contiguous slot range of every group:
//     TA = [0, fa)   TC = [fa, f1)   fp32 accumulator COLUMNS in TMEM (next to the two P buffers)
//     SB = [f1, fb)  SD = [fb, f2)   fp32 accumulator ROWS in shared memory ([f2-f1][128 batch] floats)
//     L  = [f2, d)                   red.global.add.f32 into dX^T, as in the first version (tc_dx.cu)
// A CTA owns (128-row batch tile, stripe of groups).  Per group: TMA loads the dY tile and W_g, one thread
// issues P^T[128 batch x K slots] = dY tile * W_g (tcgen05, fp32 in TMEM, double buffered), an auxiliary
// warp (one of two, alternating groups) turns idx_g into one destination list per class, and 16 epilogue warps (4 sets x 4 TMEM lane
// quadrants; a lane owns one batch row) add column j of P into the destination of slot j.  Set s owns class s
// exclusively, so no two threads ever touch the same accumulator word and nothing on chip is atomic; the L
// chunks (atomic in L2, hence owner-free) are dealt round-robin to the four sets, shared-memory sets first
// (handing them out dynamically through a shared-memory counter was measured slower: 0.319 vs 0.298 ms).  Lists are padded to whole chunks with
// a dummy destination per class (a spare TMEM column, a spare shared-memory row), so the on-chip
// inner loops carry no predicates; only the last L chunk is predicated (a dummy word in L2 would be one address
// hammered by every CTA).  Groups whose idx row is not strictly increasing (duplicates, unsorted:
// legal by DESIGN.md reading R4) take the L path for every slot, which is correct for any index row.
// The accumulators are flushed into dX^T once per CTA.
#include <algorithm>

#include "tc_common.cuh"
#include "tc_kernels.h"

namespace haste {
using namespace tc;

struct DxAccParams {
  float* dXt;           // [d][Bpad] fp32, zeroed by the caller
  const int32_t* idx;   // [NG][K]
  int B, Bpad, NT, S, d;
  int64_t NG;
  int fa, f1, fb, f2;   // class boundaries (see above)
  float* part;          // HASTE_DETERMINISTIC: private partial tiles [grid][d][128] fp32 (zeroed by the caller) instead of
                        // reductions into dXt; null otherwise.  See the note at the L class below.
};

template <int G, int K, int NST_> struct DxAccCfg {
  static constexpr int NSET = 4;                              // epilogue sets: 0 = TA, 1 = SB, 2 = TC, 3 = SD
  static constexpr int NLIST = NSET + 1;                      // + the L list
  // narrow groups: the contraction (over the group's labels) is GP = 16 long, the shortest bf16 MMA.  G = 8: the dY box is
  // 16 labels wide over rows that have 8, so labels 8-15 arrive as zeros, and label rows 8-15 of the W image are zeroed
  // once and never loaded.
  static constexpr int GP = G < 16 ? 16 : G;
  static constexpr int Y_BYTES = GP * 256;                    // [G/64 k-blocks][128 batch rows][128 B]; G = 32: [128 rows][64 B]; G <= 16: [128 rows][32 B]
  static constexpr int W_BYTES = GP * K * 2;                  // [K/64 slot atoms][GP label rows][128 B]
  static constexpr int STAGE = Y_BYTES + W_BYTES;
  static constexpr int TX_BYTES = Y_BYTES + G * K * 2;        // what the TMA boxes of one group bring
  static constexpr int NST = NST_;                            // operand stages (dY tile + W_g) in flight
  static constexpr int LIST_LEN = K + 16;                     // entries per list (padding for the last chunk)
  static constexpr int RING_META = 48;                        // lo[5] at 0, n[5] at 20
  static constexpr int RING_BYTES = (RING_META + NLIST * LIST_LEN * 4 + 127) / 128 * 128;
  static constexpr int RD = 4;                                // depth of the destination-list ring
  static constexpr int TF = 512 - 2 * K - 1;                  // TMEM accumulator columns usable by features
  static constexpr int TDUMMY = 511;                          // dummy TMEM column
  static constexpr int OFF_RING = NST * STAGE;
  static constexpr int OFF_BAR = OFF_RING + RD * RING_BYTES;
  static constexpr int NBAR = 2 * NST + 4 + 2 * RD;
  static constexpr int OFF_MISC = OFF_BAR + NBAR * 8;
  static constexpr int OFF_ACC = (OFF_MISC + 64 + 511) / 512 * 512;
  static constexpr int NS_MAX = (232448 - 1024 - OFF_ACC) / 512 - 1;   // shared-memory accumulator rows (+1 dummy row)
  static constexpr bool FITS = NS_MAX >= 64;                  // otherwise use fewer stages
  static constexpr int NAUX = 2;                              // list-building warps: warp a builds the lists of groups i = a mod NAUX
  static constexpr int THREADS = (4 * NSET + 2 + NAUX) * 32;
};

__device__ __forceinline__ void dxa_red_add_f32(float* addr, float v) {
  asm volatile("red.global.add.f32 [%0], %1;" ::"l"(addr), "f"(v) : "memory");
}
__device__ __forceinline__ uint32_t dxa_tld1(uint32_t taddr) {
  uint32_t v;
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(v) : "r"(taddr) : "memory");
  return v;
}
__device__ __forceinline__ void dxa_tst1(uint32_t taddr, uint32_t v) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};" ::"r"(taddr), "r"(v) : "memory");
}
__device__ __forceinline__ void dxa_tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ int4 dxa_lds128i(uint32_t addr) {
  int4 v;
  asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
  return v;
}
__device__ __forceinline__ int dxa_lds32i(uint32_t addr) {
  int v;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ float dxa_lds32f(uint32_t addr) {
  float v;
  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ void dxa_sts32f(uint32_t addr, float v) {
  asm volatile("st.shared.f32 [%0], %1;" ::"r"(addr), "f"(v) : "memory");
}
__device__ __forceinline__ void dxa_red_add_f32(const char* addr, float v) {
  asm volatile("red.global.add.f32 [%0], %1;" ::"l"(addr), "f"(v) : "memory");
}
__device__ __forceinline__ void dxa_tmem_ld8(uint32_t taddr, uint32_t (&v)[8]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
               : "r"(taddr)
               : "memory");
}
template <int N> __device__ __forceinline__ void dxa_tmem_ldn(uint32_t taddr, uint32_t (&v)[N]);
template <> __device__ __forceinline__ void dxa_tmem_ldn<16>(uint32_t taddr, uint32_t (&v)[16]) { tmem_ld16(taddr, v); }
template <> __device__ __forceinline__ void dxa_tmem_ldn<8>(uint32_t taddr, uint32_t (&v)[8]) { dxa_tmem_ld8(taddr, v); }
template <> __device__ __forceinline__ void dxa_tmem_ldn<24>(uint32_t taddr, uint32_t (&v)[24]) {
  tmem_ld16(taddr, reinterpret_cast<uint32_t(&)[16]>(v[0]));
  dxa_tmem_ld8(taddr + 16, reinterpret_cast<uint32_t(&)[8]>(v[16]));
}
// N destination codes of one chunk of a list (16-byte aligned)
template <int N> __device__ __forceinline__ void dxa_load_dest(uint32_t addr, int (&dst)[N]) {
#pragma unroll
  for (int i = 0; i < N / 4; ++i) {
    const int4 a = dxa_lds128i(addr + i * 16);
    dst[4 * i] = a.x; dst[4 * i + 1] = a.y; dst[4 * i + 2] = a.z; dst[4 * i + 3] = a.w;
  }
}
// one chunk of N slots of a TMEM class: acc column dst[u] += P column u (both in this warp's lane quadrant)
template <int N> __device__ __forceinline__ void dxa_chunk_t(uint32_t tp, uint32_t lst, uint32_t tlane) {
  uint32_t pv[N], a[N];
  int dst[N];
  dxa_tmem_ldn<N>(tp, pv);
  dxa_load_dest<N>(lst, dst);
#pragma unroll
  for (int u = 0; u < N; ++u) a[u] = dxa_tld1(tlane + dst[u]);
  tmem_ld_wait();
#pragma unroll
  for (int u = 0; u < N; u += 2) {            // packed add: two slots per instruction (the kernel is issue-bound)
    uint64_t s2;
    asm("{\n\t.reg .b64 x, y;\n\tmov.b64 x, {%1, %2};\n\tmov.b64 y, {%3, %4};\n\tadd.rn.f32x2 %0, x, y;\n\t}"
        : "=l"(s2) : "r"(a[u]), "r"(a[u + 1]), "r"(pv[u]), "r"(pv[u + 1]));
    dxa_tst1(tlane + dst[u], (uint32_t)s2);
    dxa_tst1(tlane + dst[u + 1], (uint32_t)(s2 >> 32));
  }
}
// one chunk of N slots of a shared-memory class: acc row (byte offset dst[u]), this thread's word += P column u
template <int N> __device__ __forceinline__ void dxa_chunk_s(uint32_t tp, uint32_t lst, uint32_t sown) {
  uint32_t pv[N];
  float a[N];
  int dst[N];
  dxa_tmem_ldn<N>(tp, pv);
  dxa_load_dest<N>(lst, dst);
#pragma unroll
  for (int u = 0; u < N; ++u) a[u] = dxa_lds32f(sown + dst[u]);
  tmem_ld_wait();
#pragma unroll
  for (int u = 0; u < N; u += 2) {            // packed add: two slots per instruction
    uint64_t s2;
    asm("{\n\t.reg .b64 x, y;\n\tmov.b64 x, {%1, %2};\n\tmov.b64 y, {%3, %4};\n\tadd.rn.f32x2 %0, x, y;\n\t}"
        : "=l"(s2) : "f"(a[u]), "f"(a[u + 1]), "r"(pv[u]), "r"(pv[u + 1]));
    dxa_sts32f(sown + dst[u], __uint_as_float((uint32_t)s2));
    dxa_sts32f(sown + dst[u + 1], __uint_as_float((uint32_t)(s2 >> 32)));
  }
}

// 20 warps poll barriers here; a polling loop costs issue slots the working warps need, so back off between polls
template <int NS_SLEEP> __device__ __forceinline__ void dxa_wait(uint64_t* bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) __nanosleep(NS_SLEEP);
}

// wait for two barriers at once: both phase checks are in flight together (a check costs 100-300 cycles even when it succeeds)
__device__ __forceinline__ void dxa_wait2(uint64_t* a, uint32_t pa, uint64_t* b, uint32_t pb) {
  bool da = false, db = false;
  do {
    const bool ta = da || mbar_try_wait(a, pa);
    const bool tb = db || mbar_try_wait(b, pb);
    da = ta; db = tb;
  } while (!(da && db));
}

template <int G, int K, int NST, bool DET>
__global__ void __launch_bounds__(DxAccCfg<G, K, NST>::THREADS, 1)
tc_dx_acc_kernel(const __grid_constant__ CUtensorMap tmY, const __grid_constant__ CUtensorMap tmW, const DxAccParams p) {
  using C = DxAccCfg<G, K, NST>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const uint32_t sbase = smem_u32(smem);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::OFF_BAR);
  uint64_t* full = bars;                    // [NST] TMA (tx) -> MMA
  uint64_t* empty = bars + C::NST;          // [NST] MMA commit -> TMA
  uint64_t* t_full = bars + 2 * C::NST;     // [2]   MMA commit -> epilogue
  uint64_t* t_empty = t_full + 2;           // [2]   16 epilogue warps -> MMA
  uint64_t* d_full = t_empty + 2;           // [RD]  aux warp -> epilogue (destination lists ready)
  uint64_t* d_empty = d_full + C::RD;       // [RD]  16 epilogue warps -> aux warp
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + C::OFF_MISC);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int bt = blockIdx.x % p.NT, stripe = blockIdx.x / p.NT;
  const int n_my = p.NG > stripe ? (int)((p.NG - stripe + p.S - 1) / p.S) : 0;
  const int NS = p.f2 - p.f1;               // shared-memory accumulator rows in use; row NS is the dummy

  if (threadIdx.x == 0) {
    for (int i = 0; i < C::NST; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&t_full[i], 1); mbar_init(&t_empty[i], 4 * C::NSET); }
    for (int i = 0; i < C::RD; ++i) { mbar_init(&d_full[i], 1); mbar_init(&d_empty[i], 4 * C::NSET); }
    fence_barrier_init();
  }
  if (warp == 4 * C::NSET + 1 && lane == 0) { tma_prefetch_desc(&tmY); tma_prefetch_desc(&tmW); }
  if constexpr (G < 16) {               // label rows 8-15 of every W image: zero (see DxAccCfg)
    for (int e = threadIdx.x; e < C::NST * (K / 64) * 64; e += blockDim.x) {
      const int st = e / ((K / 64) * 64), a = (e / 64) % (K / 64), c = e % 64;
      sts128(sbase + st * C::STAGE + C::Y_BYTES + a * (C::GP * 128) + 1024 + c * 16, 0u, 0u, 0u, 0u);
    }
    fence_proxy_async_smem();
  }
  if (warp == 4 * C::NSET) tmem_alloc<512>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  pdl_wait();       // nothing above touches global memory (common.cuh, PDL)
  pdl_trigger();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 4 * C::NSET + 1) {
    // ===================== TMA loader: dY tile + W_g =====================
    if (lane == 0) {
      for (int i = 0; i < n_my; ++i) {
        const int64_t g = stripe + (int64_t)i * p.S;
        const int st = i % C::NST;
        mbar_wait(&empty[st], ((i / C::NST) & 1) ^ 1);
        mbar_arrive_expect_tx(&full[st], C::TX_BYTES);
        uint8_t* s0 = smem + st * C::STAGE;
#pragma unroll
        for (int kb = 0; kb < (G >= 64 ? G / 64 : 1); ++kb) tma_load_3d(s0 + kb * 16384, &tmY, &full[st], kb * 64, bt * 128, (int)g);
#pragma unroll
        for (int a = 0; a < K / 64; ++a) tma_load_2d(s0 + C::Y_BYTES + a * (C::GP * 128), &tmW, &full[st], a * 64, (int)(g * G));
      }
    }
  } else if (warp == 4 * C::NSET) {
    // ===================== MMA issuer =====================
    // whole warp waits, one elected lane issues; descriptors are a per-stage base + compile-time offsets (see tc_tail.cu)
    constexpr uint32_t idesc = make_idesc_bf16(128, K, /*A (dY) K-major*/ 0, /*B (W) MN-major*/ 1);
    // A = the dY tile, K-major: 128-byte rows (64 labels per k-block) or, for G = 32, 64-byte rows with the 64-byte swizzle
    // (G <= 16: 32-byte rows with the 32-byte swizzle)
    const uint64_t adesc0 = G >= 64 ? make_sdesc_sw128(sbase, 16, 1024) : G == 32 ? make_sdesc_sw64(sbase, 16, 512) : make_sdesc_sw32(sbase, 16, 256);
    const uint64_t bdesc0 = make_sdesc_sw128(sbase + C::Y_BYTES, C::GP * 128, 1024);
    for (int i = 0; i < n_my; ++i) {
      const int st = i % C::NST, slot = i & 1;
      dxa_wait2(&full[st], (i / C::NST) & 1, &t_empty[slot], ((i >> 1) & 1) ^ 1);
      tc_fence_after();
      if (elect_one()) {
        const uint64_t so = (uint64_t)((st * C::STAGE) >> 4);
        const uint32_t d = tmem_base + slot * K;
#pragma unroll
        for (int j = 0; j < C::GP / 16; ++j)
          umma_f16(d, adesc0 + so + (uint64_t)(((j >> 2) * 16384 + (j & 3) * 32) >> 4), bdesc0 + so + (uint64_t)((j * 2048) >> 4),
                   idesc, j ? 1u : 0u);
        umma_commit(&empty[st]);
        umma_commit(&t_full[slot]);
      }
      __syncwarp();
    }
  } else if (warp >= 4 * C::NSET + 2) {
    // ===================== auxiliary warps: idx_g -> one destination list per class =====================
    // Lane holds slots j = lane + 32 t.  Slot j belongs to the class whose slot range contains it and is entry
    // j - lo of that class's list, so every lane writes its own PER entries; no gather, no second pass.
    constexpr int PER = K / 32;
    const int aw = warp - (4 * C::NSET + 2);
    const int lrow_bytes = DET ? 512 : p.Bpad * 4;
    int e[PER], en[PER];
#pragma unroll
    for (int t = 0; t < PER; ++t) { e[t] = 0; en[t] = 0; }
    if (aw < n_my) {
#pragma unroll
      for (int t = 0; t < PER; ++t) en[t] = __ldg(p.idx + (stripe + (int64_t)aw * p.S) * K + lane + 32 * t);
    }
    for (int i = aw; i < n_my; i += C::NAUX) {
      const int64_t g = stripe + (int64_t)i * p.S;
      const int r = i % C::RD;
#pragma unroll
      for (int t = 0; t < PER; ++t) e[t] = en[t];
      if (i + C::NAUX < n_my) {
#pragma unroll
        for (int t = 0; t < PER; ++t) en[t] = __ldg(p.idx + (g + (int64_t)C::NAUX * p.S) * K + lane + 32 * t);
      }
      // strictly increasing?  (slot j+1 is the next lane's value, or lane 0's value of the next t)
      bool inc = true;
#pragma unroll
      for (int t = 0; t < PER; ++t) {
        int nxt = __shfl_down_sync(0xffffffffu, e[t], 1);
        const int wrap = __shfl_sync(0xffffffffu, t + 1 < PER ? e[(t + 1) % PER] : 0x7fffffff, 0);
        if (lane == 31) nxt = wrap;
        inc &= e[t] < nxt;
      }
      const bool strict = __all_sync(0xffffffffu, inc);
      // class boundaries as slot counts
      int ca = 0, c1 = 0, cb = 0, c2 = 0;
#pragma unroll
      for (int t = 0; t < PER; ++t) { ca += e[t] < p.fa; c1 += e[t] < p.f1; cb += e[t] < p.fb; c2 += e[t] < p.f2; }
      ca = __reduce_add_sync(0xffffffffu, ca); c1 = __reduce_add_sync(0xffffffffu, c1);
      cb = __reduce_add_sync(0xffffffffu, cb); c2 = __reduce_add_sync(0xffffffffu, c2);
      if (!strict) { ca = 0; c1 = 0; cb = 0; c2 = 0; }
      dxa_wait<64>(&d_empty[r], ((i / C::RD) & 1) ^ 1);
      const uint32_t ring = sbase + C::OFF_RING + r * C::RING_BYTES;
      const uint32_t lists = ring + C::RING_META;
      // lists in ring order: sets 0..3 = TA [0,ca), SB [c1,cb), TC [ca,c1), SD [cb,c2); then L [c2,K)
      if (lane == 0) {
        sts32(ring + 0, 0u); sts32(ring + 4, (uint32_t)c1); sts32(ring + 8, (uint32_t)ca); sts32(ring + 12, (uint32_t)cb);
        sts32(ring + 16, (uint32_t)c2);
        sts32(ring + 20, (uint32_t)ca); sts32(ring + 24, (uint32_t)(cb - c1)); sts32(ring + 28, (uint32_t)(c1 - ca));
        sts32(ring + 32, (uint32_t)(c2 - cb)); sts32(ring + 36, (uint32_t)(K - c2));
        sts32(ring + 40, strict ? 1u : 0u);
      }
#pragma unroll
      for (int t = 0; t < PER; ++t) {
        const int j = lane + 32 * t, f = e[t];
        int l, k, code;
        if (j < ca)      { l = 0; k = j;      code = 2 * K + f; }                 // TMEM column
        else if (j < c1) { l = 2; k = j - ca; code = 2 * K + f; }
        else if (j < cb) { l = 1; k = j - c1; code = (f - p.f1) * 512; }          // byte offset of the accumulator row
        else if (j < c2) { l = 3; k = j - cb; code = (f - p.f1) * 512; }
        else             { l = 4; k = j - c2; code = f * lrow_bytes; }           // byte offset of the dX^T (or private tile) row
        sts32(lists + (l * C::LIST_LEN + k) * 4, (uint32_t)code);
      }
      // pad the on-chip lists to a whole chunk with the class's dummy destination
      if (lane < 16) {
        sts32(lists + (0 * C::LIST_LEN + ca + lane) * 4, (uint32_t)C::TDUMMY);
        sts32(lists + (2 * C::LIST_LEN + (c1 - ca) + lane) * 4, (uint32_t)C::TDUMMY);
        sts32(lists + (1 * C::LIST_LEN + (cb - c1) + lane) * 4, (uint32_t)(NS * 512));
        sts32(lists + (3 * C::LIST_LEN + (c2 - cb) + lane) * 4, (uint32_t)(NS * 512));
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&d_full[r]);
    }
  } else {
    // ===================== epilogue: set = class owner, q = TMEM lane quadrant, lane = batch row =====================
    const int set = warp >> 2, q = warp & 3;
    const bool is_t = (set & 1) == 0;                                        // sets 0, 2: TMEM classes; 1, 3: shared memory
    const int row = q * 32 + lane;
    const int b = bt * 128 + row;
    const bool vb = b < p.B;
    const uint32_t tlane = tmem_base + ((uint32_t)(q * 32) << 16);
    const uint32_t sown = sbase + C::OFF_ACC + row * 4;                      // + accumulator row * 512
    // atomic mode: column b of dX^T (row pitch Bpad); deterministic mode: column `row` of this CTA's private tile (pitch 128)
    constexpr bool det = DET;                                                // a template parameter: the default kernel pays nothing for it
    const size_t gpitch = det ? 128 : (size_t)p.Bpad;
    float* const gcol = det ? p.part + (size_t)blockIdx.x * p.d * 128 + row : p.dXt + b;   // + f * gpitch
    char* const gbytes = reinterpret_cast<char*>(gcol);                      // + byte offset of the row (L list code)
    // this set's own accumulators: [c_lo, c_hi) TMEM columns (relative to the lane base) or shared-memory rows
    const int c_lo = set == 0 ? 2 * K : set == 2 ? 2 * K + p.fa : set == 1 ? 0 : p.fb - p.f1;
    const int c_hi = set == 0 ? 2 * K + p.fa : set == 2 ? 2 * K + p.f1 : set == 1 ? p.fb - p.f1 : NS;
    // L chunks go to the shared-memory sets first: their own chunks cost fewer instructions than the TMEM sets'
    const int l_first = set == 3 ? 0 : set == 1 ? 1 : set == 2 ? 2 : 3;
    if (is_t) {
      for (int c = c_lo; c < c_hi; ++c) dxa_tst1(tlane + c, 0u);
      dxa_tmem_st_wait();
    } else {
      for (int r = c_lo; r < c_hi; ++r) dxa_sts32f(sown + r * 512, 0.f);
    }
    for (int i = 0; i < n_my; ++i) {
      const int r = i % C::RD, slot = i & 1;
      dxa_wait2(&d_full[r], (i / C::RD) & 1, &t_full[slot], (i >> 1) & 1);
      tc_fence_after();
      const uint32_t ring = sbase + C::OFF_RING + r * C::RING_BYTES;
      const uint32_t lists = ring + C::RING_META;
      const int lo_s = dxa_lds32i(ring + set * 4), n_s = dxa_lds32i(ring + 20 + set * 4);
      const int lo_l = dxa_lds32i(ring + C::NSET * 4), n_l = dxa_lds32i(ring + 20 + C::NSET * 4);
      const uint32_t tp = tlane + slot * K;
      const uint32_t lst = lists + set * C::LIST_LEN * 4;
      if (is_t) {
        dxa_tmem_st_wait();                                   // the previous group's stores to these columns have landed
        int m = 0;
#pragma unroll 1
        for (; n_s - m > 24; m += 16) dxa_chunk_t<16>(tp + lo_s + m, lst + m * 4, tlane);
        // the rest in ONE pass (8, 16 or 24 slots): a chunk is one latency chain, so as few chunks as registers allow
        if (n_s - m > 16) dxa_chunk_t<24>(tp + lo_s + m, lst + m * 4, tlane);
        else if (n_s - m > 8) dxa_chunk_t<16>(tp + lo_s + m, lst + m * 4, tlane);
        else if (n_s - m > 0) dxa_chunk_t<8>(tp + lo_s + m, lst + m * 4, tlane);
      } else {
        int m = 0;
#pragma unroll 1
        for (; n_s - m > 24; m += 16) dxa_chunk_s<16>(tp + lo_s + m, lst + m * 4, sown);
        if (n_s - m > 16) dxa_chunk_s<24>(tp + lo_s + m, lst + m * 4, sown);
        else if (n_s - m > 8) dxa_chunk_s<16>(tp + lo_s + m, lst + m * 4, sown);
        else if (n_s - m > 0) dxa_chunk_s<8>(tp + lo_s + m, lst + m * 4, sown);
      }
      // the L class: red.global is atomic, so chunks need no owner.  No dummy
      // target here: a shared dummy word in L2 would serialise the reductions of every CTA on one address.
      const uint32_t lstl = lists + C::NSET * C::LIST_LEN * 4;
#pragma unroll 1
      // Deterministic mode: plain read-modify-write of the private tile.  A word (f, b) must then have ONE writer at a time:
      // set 3 alone takes every L chunk, and the flush below waits for it behind a barrier.  The order of additions into a
      // word is then fixed: groups in order, then the owner's flush, then the stripes in order (reduce kernel).
      for (int m = det ? (set == 3 ? 0 : n_l) : l_first * 16; m < n_l; m += det ? 16 : C::NSET * 16) {
        uint32_t pv[16];
        int dst[16];
        tmem_ld16(tp + lo_l + m, pv);
        dxa_load_dest<16>(lstl + m * 4, dst);
        tmem_ld_wait();
        if (vb && det) {
          if (dxa_lds32i(ring + 40)) {        // strictly increasing row: 16 distinct words, loads first, then stores
            float a[16];
#pragma unroll
            for (int u = 0; u < 16; ++u)
              if (m + u < n_l) asm volatile("ld.global.f32 %0, [%1];" : "=f"(a[u]) : "l"(gbytes + (uint32_t)dst[u]) : "memory");
#pragma unroll
            for (int u = 0; u < 16; ++u)
              if (m + u < n_l) asm volatile("st.global.f32 [%0], %1;" ::"l"(gbytes + (uint32_t)dst[u]), "f"(a[u] + __uint_as_float(pv[u])) : "memory");
          } else {                            // duplicates possible: one word at a time
#pragma unroll
            for (int u = 0; u < 16; ++u)
              if (m + u < n_l) { volatile float* a = reinterpret_cast<volatile float*>(gbytes + (uint32_t)dst[u]); *a = *a + __uint_as_float(pv[u]); }
          }
        } else if (vb) {
          if (m + 16 <= n_l) {
#pragma unroll
            for (int u = 0; u < 16; ++u) dxa_red_add_f32(gbytes + (uint32_t)dst[u], __uint_as_float(pv[u]));
          } else {
#pragma unroll
            for (int u = 0; u < 16; ++u)
              if (m + u < n_l) dxa_red_add_f32(gbytes + (uint32_t)dst[u], __uint_as_float(pv[u]));
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) { mbar_arrive(&t_empty[slot]); mbar_arrive(&d_empty[r]); }
    }
    // flush this thread's accumulators (its batch row of every feature this set owns) into dX^T
    if (det) named_bar_sync(1, 4 * C::NSET * 32);       // set 3 has finished its read-modify-writes of the private tile
    if (is_t) {
      dxa_tmem_st_wait();
      for (int c0 = c_lo; c0 < c_hi; c0 += 16) {
        uint32_t v[16];
#pragma unroll
        for (int u = 0; u < 16; ++u) v[u] = dxa_tld1(tlane + min(c0 + u, 511));
        tmem_ld_wait();
        if (vb) {
#pragma unroll
          for (int u = 0; u < 16; ++u)
            if (c0 + u < c_hi) {
              float* a = gcol + (size_t)(c0 + u - 2 * K) * gpitch;
              if (det) *a += __uint_as_float(v[u]); else dxa_red_add_f32(a, __uint_as_float(v[u]));
            }
        }
      }
    } else if (vb) {
      for (int r = c_lo; r < c_hi; ++r) {
        float* a = gcol + (size_t)(p.f1 + r) * gpitch;
        if (det) *a += dxa_lds32f(sown + r * 512); else dxa_red_add_f32(a, dxa_lds32f(sown + r * 512));
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 4 * C::NSET) { tc_fence_after(); tmem_dealloc<512>(tmem_base); }
}

template <int G, int K, int NST>
static int launch_dx_acc(TcTailState* s, const TailShape& sh, const int32_t* idx, const void* W, const void* dY, float* dXt,
                         float* part, cudaStream_t st) {
  using C = DxAccCfg<G, K, NST>;
  CUtensorMap tmY, tmW;
  {
    const uint64_t dims[3] = {(uint64_t)G, (uint64_t)sh.B, (uint64_t)sh.NG};
    const uint64_t str[2] = {(uint64_t)G * 2, (uint64_t)sh.B * G * 2};
    const uint32_t box[3] = {(uint32_t)std::min(C::GP, 64), 128, 1};
    int rc = encode_tmap(&tmY, 2, dY, 3, dims, str, box, G >= 64 ? 128 : G == 32 ? 64 : 32);
    if (rc) return rc;
  }
  {
    const uint64_t dims[2] = {(uint64_t)K, (uint64_t)sh.L};
    const uint64_t str[1] = {(uint64_t)K * 2};
    const uint32_t box[2] = {64, (uint32_t)G};
    int rc = encode_tmap(&tmW, 2, W, 2, dims, str, box, 128);
    if (rc) return rc;
  }
  DxAccParams p;
  p.dXt = dXt; p.part = part; p.idx = idx; p.B = sh.B; p.Bpad = sh.Bpad; p.NT = ceil_div(sh.B, 128); p.NG = sh.NG; p.d = sh.d;
  if (p.NT > s->num_sms) return HASTE_ERR_UNSUPPORTED;
  if ((int64_t)sh.d * sh.Bpad * 4 > 0x7fffffff) return HASTE_ERR_UNSUPPORTED;   // list codes are 32-bit byte offsets
  p.S = (int)std::min<int64_t>(sh.NG, std::max(1, s->num_sms / p.NT));
  // class sizes: what fits
  const int f1 = std::min(sh.d, C::TF);
  const int ns = std::min(C::NS_MAX, sh.d - f1);
  p.f1 = f1; p.fa = f1 / 2; p.f2 = f1 + ns; p.fb = f1 + ns / 2;
  const int smem = C::OFF_ACC + (ns + 1) * 512 + 1024;
  if (part) {
    HASTE_CUDA_TRY(cudaFuncSetAttribute(tc_dx_acc_kernel<G, K, NST, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    HASTE_CUDA_TRY(launch_pdl(tc_dx_acc_kernel<G, K, NST, true>, dim3(p.NT * p.S), dim3(C::THREADS), smem, st, tmY, tmW, p));
  } else {
    HASTE_CUDA_TRY(cudaFuncSetAttribute(tc_dx_acc_kernel<G, K, NST, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    HASTE_CUDA_TRY(launch_pdl(tc_dx_acc_kernel<G, K, NST, false>, dim3(p.NT * p.S), dim3(C::THREADS), smem, st, tmY, tmW, p));
  }
  HASTE_LAUNCH_CHECK();
  return HASTE_OK;
}

int tc_tail_dx_acc(TcTailState* s, const TailShape& sh, const int32_t* idx, const void* W, const void* dY, float* dXt,
                   float* part, cudaStream_t st) {
  // two operand stages: more were measured to gain nothing and they cost shared-memory accumulator rows
#define HASTE_DXA(G_, K_) \
  if (sh.G == G_ && sh.K == K_) return launch_dx_acc<G_, K_, 2>(s, sh, idx, W, dY, dXt, part, st)
  HASTE_DXA(64, 128); HASTE_DXA(64, 64); HASTE_DXA(128, 64); HASTE_DXA(128, 128);
  HASTE_DXA(32, 64); HASTE_DXA(32, 128);
  HASTE_DXA(16, 64); HASTE_DXA(16, 128); HASTE_DXA(8, 64); HASTE_DXA(8, 128);
#undef HASTE_DXA
  return HASTE_ERR_UNSUPPORTED;
}

}  // namespace haste
