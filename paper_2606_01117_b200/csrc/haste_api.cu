// haste_api.cu -- the C-ABI boundary (include/haste.h): handles, argument checks,
// workspace, kernel-family dispatch.  No arithmetic of the method lives here.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <vector>
#include <new>

#include "kernels.h"
#include "tc_kernels.h"

namespace haste {

static thread_local char g_err[512] = "";
void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}

struct DeviceGuard {
  int prev = -1;
  bool ok = true;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
    if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
  }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

// Optional per-kernel device timing: CUDA events on the caller's stream around each main kernel,
// kept in a ring of `depth` calls per kernel so a benchmark can read a whole timed region afterwards.
struct Profiler {
  static const int NSLOT = 6;
  int depth = 0;
  std::vector<cudaEvent_t> a[NSLOT], b[NSLOT];
  long count[NSLOT] = {};     // completed begin/end pairs per slot
  int enable(int new_depth) {
    if (new_depth < 0 || new_depth > 4096) return HASTE_ERR_INVALID_ARG;
    destroy();
    for (int s = 0; s < NSLOT && new_depth > 0; ++s) {
      a[s].assign(new_depth, nullptr);
      b[s].assign(new_depth, nullptr);
      for (int i = 0; i < new_depth; ++i)
        if (cudaEventCreate(&a[s][i]) != cudaSuccess || cudaEventCreate(&b[s][i]) != cudaSuccess) return HASTE_ERR_CUDA;
    }
    depth = new_depth;
    return HASTE_OK;
  }
  void begin(int s, cudaStream_t st) { if (depth) cudaEventRecord(a[s][count[s] % depth], st); }
  void end(int s, cudaStream_t st) { if (depth) { cudaEventRecord(b[s][count[s] % depth], st); ++count[s]; } }
  int ms(int s, int age, float* out) {
    if (s < 0 || s >= NSLOT || !out || !depth || age < 0 || age >= depth || age >= count[s]) {
      set_error("kernel_ms: profiling is off, or no such recorded call (kernel %d, age %d)", s, age);
      return HASTE_ERR_INVALID_ARG;
    }
    const long i = (count[s] - 1 - age) % depth;
    if (cudaEventSynchronize(b[s][i]) != cudaSuccess || cudaEventElapsedTime(out, a[s][i], b[s][i]) != cudaSuccess) {
      set_error("kernel_ms: %s", cudaGetErrorString(cudaGetLastError()));
      return HASTE_ERR_CUDA;
    }
    return HASTE_OK;
  }
  void destroy() {
    for (int s = 0; s < NSLOT; ++s) {
      for (cudaEvent_t e : a[s]) if (e) cudaEventDestroy(e);
      for (cudaEvent_t e : b[s]) if (e) cudaEventDestroy(e);
      a[s].clear(); b[s].clear(); count[s] = 0;
    }
    depth = 0;
  }
};

static inline size_t esize(haste_dtype_t dt) { return dt == HASTE_F32 ? 4 : 2; }
static inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// ---- scratch of haste_forward_topk_static: the candidate lists of the fused top-k forward in device memory that belongs
// to the library image, so that the call allocates nothing.  [2][TOPK_STATIC_ENTRIES] 32-bit words: candidate logits
// (fp32), then candidate labels (int32), each [CTAs <= 148][4 epilogue sets][128 rows][8 candidates] = 4.625 MiB in all,
// held by every GPU that loads the library until the process exits.  ONE array per device: every call on that device
// shares it (calls that overlap on the GPU race), and it keeps the last call's contents -- nothing in it has to start at
// zero, because the forward kernel writes every list its merge kernel reads (tc_tail.cu, end of the top-k epilogue).
// In host code the NAME below is a host-side stand-in, not a device address: the address is asked for once per device
// (resolve_topk_static, called from haste_create with that device current) and that pointer is what the kernels get.
static constexpr int TOPK_STATIC_MAX_CTAS = 148;
static constexpr size_t TOPK_STATIC_ENTRIES = (size_t)TOPK_STATIC_MAX_CTAS * 4 * 128 * 8;
static __device__ __align__(256) unsigned char g_topk_static[2 * TOPK_STATIC_ENTRIES * 4];
static constexpr int TOPK_STATIC_MAX_DEVICES = 64;
struct TopkStaticDev { void* ptr; cudaError_t err; bool tried; };
static TopkStaticDev g_topk_static_dev[TOPK_STATIC_MAX_DEVICES] = {};
static std::mutex g_topk_static_mu;
// `device` must be the current device.  Never fails the caller: the outcome is kept for haste_forward_topk_static.
static void resolve_topk_static(int device) {
  if (device < 0 || device >= TOPK_STATIC_MAX_DEVICES) return;
  std::lock_guard<std::mutex> lock(g_topk_static_mu);
  TopkStaticDev& e = g_topk_static_dev[device];
  if (e.tried) return;
  void* ptr = nullptr;
  e.err = cudaGetSymbolAddress(&ptr, g_topk_static);
  e.ptr = e.err == cudaSuccess ? ptr : nullptr;
  e.tried = true;
  if (e.err != cudaSuccess) (void)cudaGetLastError();      // not sticky; reported by the entry point that needs it
}

}  // namespace haste

using namespace haste;

struct haste_layer {
  haste_config_t cfg;
  int device;
  int family;       // 0 SIMT, 1 tcgen05
  int64_t NG;
  int Bpad;         // row pitch of Xt / dXt
  void* Xt;         // [d][Bpad] dtype
  float* dXt;       // [d][Bpad] fp32
  bool dxt_clean;   // dXt is all zero (the transpose-out kernel zeroes what it reads; false after a pass that ended early)
  float* dx_part;   // HASTE_DETERMINISTIC: [num_sms][d][128] fp32 private partial tiles of the dX kernel, else null
  double* loss_acc; // device scalar
  float* partials;  // [n_partials] per-CTA loss partials (tcgen05 family)
  int n_partials;
  int* flag;        // validate_index result
  void* rw_ws;      // rewiring workspace (scores, mask, ...; allocated on first use)
  float* topk_val;  // fused top-k candidates [num_SMs][4 sets][128][8] (allocated on first use)
  int* topk_idx;
  TcTailState* tc;  // tcgen05 family state (tensor maps, counters) or NULL
  int last_launches;
  Profiler* prof;
};

struct haste_head {
  int32_t d;
  int64_t L;
  int32_t B_max;
  haste_dtype_t dtype;
  int64_t label_offset;
  float loss_scale;
  uint32_t flags;
  int device;
  int family;
  double* loss_acc;
  float* partials;
  int n_partials;
  TcHeadState* tc;
  int last_launches;
  Profiler* prof;
};

extern "C" {

const char* haste_status_string(int status) {
  switch (status) {
    case HASTE_OK: return "HASTE_OK";
    case HASTE_ERR_INVALID_ARG: return "HASTE_ERR_INVALID_ARG";
    case HASTE_ERR_BAD_INDEX: return "HASTE_ERR_BAD_INDEX";
    case HASTE_ERR_UNSUPPORTED: return "HASTE_ERR_UNSUPPORTED";
    case HASTE_ERR_CUDA: return "HASTE_ERR_CUDA";
    case HASTE_ERR_NOMEM: return "HASTE_ERR_NOMEM";
    default: return "HASTE_ERR_UNKNOWN";
  }
}

const char* haste_last_error(void) { return g_err; }

int haste_create(haste_layer_t** out, const haste_config_t* cfg, int cuda_device) {
  if (!out) { set_error("haste_create: out is NULL"); return HASTE_ERR_INVALID_ARG; }
  *out = nullptr;
  if (!cfg) { set_error("haste_create: cfg is NULL"); return HASTE_ERR_INVALID_ARG; }
  if (cfg->d <= 0 || cfg->L < 0 || cfg->G <= 0 || cfg->K <= 0 || cfg->B_max <= 0) {
    set_error("haste_create: d, G, K, B_max must be positive and L >= 0");
    return HASTE_ERR_INVALID_ARG;
  }
  if ((cfg->dtype != HASTE_F32 && cfg->dtype != HASTE_BF16) || (cfg->dw_dtype != HASTE_F32 && cfg->dw_dtype != HASTE_BF16)) {
    set_error("haste_create: unknown dtype");
    return HASTE_ERR_INVALID_ARG;
  }
  if (cfg->G > 1024 || cfg->K > 4096) {
    set_error("haste_create: G <= 1024 and K <= 1700 are supported");
    return HASTE_ERR_UNSUPPORTED;
  }
  const int64_t NG = (cfg->L + cfg->G - 1) / cfg->G;
  if (NG > 0x7fffffffLL) { set_error("haste_create: too many groups"); return HASTE_ERR_UNSUPPORTED; }
  // limits of the generic CUDA-core family, checked here so that no hot call fails at launch time: its forward stages
  // K x 33 words of shared memory per block (227 KB at most), and its grids put ceil(B/32) into gridDim.y
  if (cfg->K > 1700 || cfg->B_max > 65535 * 32) {
    set_error("haste_create: K <= 1700 and B_max <= 2 097 120 are supported");
    return HASTE_ERR_UNSUPPORTED;
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || cuda_device < 0 || cuda_device >= ndev) {
    cudaGetLastError();
    set_error("haste_create: CUDA device %d not available (no CPU fallback exists)", cuda_device);
    return HASTE_ERR_CUDA;
  }
  DeviceGuard guard(cuda_device);
  if (!guard.ok) { set_error("haste_create: cudaSetDevice failed"); return HASTE_ERR_CUDA; }
  haste_layer* h = new (std::nothrow) haste_layer();
  if (!h) return HASTE_ERR_NOMEM;
  memset(h, 0, sizeof(*h));
  h->cfg = *cfg;
  h->device = cuda_device;
  h->NG = NG;
  h->prof = new (std::nothrow) Profiler();
  if (!h->prof) { delete h; return HASTE_ERR_NOMEM; }
  h->Bpad = round_up(cfg->B_max, 128);
  h->n_partials = 1024;
  const size_t xt_bytes = (size_t)cfg->d * h->Bpad * esize(cfg->dtype);
  const size_t dxt_bytes = (size_t)cfg->d * h->Bpad * 4;
  cudaError_t e = cudaMalloc(&h->Xt, xt_bytes);
  if (e == cudaSuccess) e = cudaMalloc(&h->dXt, dxt_bytes);
  if (e == cudaSuccess) e = cudaMalloc(&h->loss_acc, sizeof(double));
  if (e == cudaSuccess) e = cudaMalloc(&h->partials, h->n_partials * sizeof(float));
  if (e == cudaSuccess) e = cudaMalloc(&h->flag, sizeof(int));
  if (e == cudaSuccess) e = cudaMemset(h->Xt, 0, xt_bytes);
  if (e == cudaSuccess) e = cudaMemset(h->dXt, 0, dxt_bytes);
  h->dxt_clean = (e == cudaSuccess);
  if (e == cudaSuccess) e = cudaMemset(h->partials, 0, h->n_partials * sizeof(float));
  if (e != cudaSuccess) {
    set_error("haste_create: workspace allocation failed: %s", cudaGetErrorString(e));
    haste_destroy(h);
    return e == cudaErrorMemoryAllocation ? HASTE_ERR_NOMEM : HASTE_ERR_CUDA;
  }
  h->family = 0;
  if (!(cfg->flags & HASTE_FORCE_SIMT) && tc_tail_supported(*cfg, cuda_device)) {
    int rc = tc_tail_create(&h->tc, *cfg, h->Bpad, cuda_device);
    if (rc != HASTE_OK) { haste_destroy(h); return rc; }
    h->family = 1;
  }
  if (cfg->flags & HASTE_DETERMINISTIC) {
    // atomic-free dX: only the accumulating tcgen05 kernel has such a variant (private partial tiles + ordered reduction)
    if (h->family != 1) {
      set_error("haste_create: HASTE_DETERMINISTIC needs a shape of the tcgen05 family (bf16, G in {8,16,32,64,128}, K in {64,128})");
      haste_destroy(h);
      return HASTE_ERR_UNSUPPORTED;
    }
    // one private tile per CTA of the dX kernel: its grid is NT * S <= num_SMs, which needs NT = ceil(B/128) <= num_SMs
    if ((cfg->B_max + 127) / 128 > tc_tail_num_sms(h->tc)) {
      set_error("haste_create: HASTE_DETERMINISTIC supports B_max <= %d", 128 * tc_tail_num_sms(h->tc));
      haste_destroy(h);
      return HASTE_ERR_UNSUPPORTED;
    }
    const size_t part_bytes = (size_t)tc_tail_num_sms(h->tc) * cfg->d * 128 * 4;
    if (cudaMalloc(&h->dx_part, part_bytes) != cudaSuccess) {
      set_error("haste_create: allocation of the deterministic dX workspace (%zu bytes) failed", part_bytes);
      haste_destroy(h);
      return HASTE_ERR_NOMEM;
    }
  }
  resolve_topk_static(cuda_device);      // set-up of haste_forward_topk_static (this device is current here)
  *out = h;
  return HASTE_OK;
}

int haste_destroy(haste_layer_t* h) {
  if (!h) return HASTE_OK;
  DeviceGuard guard(h->device);
  if (h->tc) tc_tail_destroy(h->tc);
  if (h->prof) { h->prof->destroy(); delete h->prof; }
  cudaFree(h->Xt); cudaFree(h->dXt); cudaFree(h->dx_part); cudaFree(h->loss_acc); cudaFree(h->partials); cudaFree(h->flag); cudaFree(h->topk_val); cudaFree(h->topk_idx); cudaFree(h->rw_ws);
  delete h;
  return HASTE_OK;
}

size_t haste_dy_bytes(const haste_layer_t* h, int B) {
  if (!h || B < 0) return 0;
  return (size_t)h->NG * (size_t)B * (size_t)h->cfg.G * esize(h->cfg.dtype);
}

int haste_kernel_family(const haste_layer_t* h) { return h ? h->family : -1; }
int haste_last_launch_count(const haste_layer_t* h) { return h ? h->last_launches : 0; }

int haste_validate_index(haste_layer_t* h, const int32_t* idx, void* stream) {
  if (!h || !idx) { set_error("haste_validate_index: NULL argument"); return HASTE_ERR_INVALID_ARG; }
  DeviceGuard guard(h->device);
  cudaStream_t st = (cudaStream_t)stream;
  HASTE_CUDA_TRY(cudaMemsetAsync(h->flag, 0, sizeof(int), st));
  int rc = launch_validate_index(idx, h->NG, h->cfg.K, h->cfg.d, (h->cfg.flags & HASTE_IDX_SORTED_DISTINCT) ? 1 : 0,
                                 h->flag, st);
  if (rc != HASTE_OK) return rc;
  int flag = 0;
  HASTE_CUDA_TRY(cudaMemcpyAsync(&flag, h->flag, sizeof(int), cudaMemcpyDeviceToHost, st));
  HASTE_CUDA_TRY(cudaStreamSynchronize(st));
  if (flag & 1) { set_error("haste_validate_index: value outside [0,d)"); return HASTE_ERR_BAD_INDEX; }
  if (flag & 2) { set_error("haste_validate_index: a row is not strictly ascending"); return HASTE_ERR_BAD_INDEX; }
  return HASTE_OK;
}

static int check_call(const haste_layer_t* h, int B, const char* fn) {
  if (!h) { set_error("%s: handle is NULL", fn); return HASTE_ERR_INVALID_ARG; }
  if (B < 0 || B > h->cfg.B_max) { set_error("%s: B=%d outside [0, B_max=%d]", fn, B, h->cfg.B_max); return HASTE_ERR_INVALID_ARG; }
  return HASTE_OK;
}

static TailShape make_shape(const haste_layer_t* h, int B) {
  TailShape sh;
  sh.d = h->cfg.d; sh.G = h->cfg.G; sh.K = h->cfg.K; sh.B = B; sh.Bpad = h->Bpad;
  sh.L = h->cfg.L; sh.NG = h->NG; sh.label_offset = h->cfg.label_offset;
  sh.s = h->cfg.loss_scale != 0.f ? h->cfg.loss_scale : (B > 0 ? 1.0f / (float)B : 0.f);
  return sh;
}

int haste_forward_loss(haste_layer_t* h, int B, const void* X, const int32_t* idx, const void* W, const float* bias,
                       const int32_t* tgt_rowptr, const int32_t* tgt_col, float* loss, void* dY, float* logits_out,
                       void* stream) {
  int rc = check_call(h, B, "haste_forward_loss");
  if (rc) return rc;
  if (!X || !idx || !W) { set_error("haste_forward_loss: X, idx and W are required"); return HASTE_ERR_INVALID_ARG; }
  if ((tgt_rowptr == nullptr) != (tgt_col == nullptr)) {
    set_error("haste_forward_loss: tgt_rowptr and tgt_col must both be given or both be NULL");
    return HASTE_ERR_INVALID_ARG;
  }
  if (!aligned16(X) || !aligned16(W) || !aligned16(dY) || !aligned16(idx)) {
    set_error("haste_forward_loss: X, W, idx and dY must be 16-byte aligned");
    return HASTE_ERR_INVALID_ARG;
  }
  DeviceGuard guard(h->device);
  cudaStream_t st = (cudaStream_t)stream;
  const TailShape sh = make_shape(h, B);
  Profiler& pf = *h->prof;
  h->last_launches = 0;
  if (B == 0 || h->NG == 0) {
    if (loss) HASTE_CUDA_TRY(cudaMemsetAsync(loss, 0, sizeof(float), st));
    return HASTE_OK;
  }
  pf.begin(HASTE_KERNEL_PREP_FWD, st);
  rc = launch_transpose_pad(h->cfg.dtype, X, h->Xt, B, sh.d, h->Bpad, round_up(B, 128), st);
  if (rc) return rc;
  h->last_launches++;
  pf.end(HASTE_KERNEL_PREP_FWD, st);
  if (h->family == 1) {
    int n = 0;
    pf.begin(HASTE_KERNEL_FORWARD, st);
    rc = tc_tail_forward(h->tc, sh, h->Xt, idx, W, bias, tgt_rowptr, tgt_col, loss ? h->partials : nullptr, loss, dY,
                         logits_out, 0, nullptr, nullptr, nullptr, st, &n);       // the kernel's last CTA writes the loss
    if (rc) return rc;
    pf.end(HASTE_KERNEL_FORWARD, st);
    h->last_launches += n;
    return HASTE_OK;
  }
  if (loss) HASTE_CUDA_TRY(cudaMemsetAsync(h->loss_acc, 0, sizeof(double), st));
  pf.begin(HASTE_KERNEL_FORWARD, st);
  rc = launch_simt_forward(h->cfg.dtype, sh, h->Xt, idx, W, bias, tgt_rowptr, tgt_col, loss ? h->loss_acc : nullptr, dY,
                           logits_out, st);
  if (rc) return rc;
  pf.end(HASTE_KERNEL_FORWARD, st);
  h->last_launches++;
  if (loss) {
    rc = launch_finalize_loss(h->loss_acc, nullptr, 0, sh.s, loss, st);
    if (rc) return rc;
    h->last_launches++;
  }
  return HASTE_OK;
}

int haste_forward_loss_dw(haste_layer_t* h, int B, const void* X, const int32_t* idx, const void* W, const float* bias,
                          const int32_t* tgt_rowptr, const int32_t* tgt_col, float* loss, void* dY, void* dW, float* dbias,
                          void* stream) {
  int rc = check_call(h, B, "haste_forward_loss_dw");
  if (rc) return rc;
  if (!X || !idx || !W || !dY) { set_error("haste_forward_loss_dw: X, idx, W and dY are required"); return HASTE_ERR_INVALID_ARG; }
  if ((tgt_rowptr == nullptr) != (tgt_col == nullptr)) {
    set_error("haste_forward_loss_dw: tgt_rowptr and tgt_col must both be given or both be NULL");
    return HASTE_ERR_INVALID_ARG;
  }
  if (!aligned16(X) || !aligned16(W) || !aligned16(dY) || !aligned16(idx) || !aligned16(dW)) {
    set_error("haste_forward_loss_dw: X, W, idx, dY and dW must be 16-byte aligned");
    return HASTE_ERR_INVALID_ARG;
  }
  if (h->family == 1 && B > 0 && h->NG > 0 && h->cfg.G == 64 && B <= 512 && (dW || dbias)) {
    DeviceGuard guard(h->device);
    cudaStream_t st = (cudaStream_t)stream;
    const TailShape sh = make_shape(h, B);
    Profiler& pf = *h->prof;
    h->last_launches = 0;
    pf.begin(HASTE_KERNEL_PREP_FWD, st);
    rc = launch_transpose_pad(h->cfg.dtype, X, h->Xt, B, sh.d, h->Bpad, round_up(B, 128), st);
    if (rc) return rc;
    h->last_launches++;
    pf.end(HASTE_KERNEL_PREP_FWD, st);
    int n = 0;
    pf.begin(HASTE_KERNEL_FORWARD, st);
    rc = tc_tail_forward_dw(h->tc, sh, h->Xt, idx, W, bias, tgt_rowptr, tgt_col, loss ? h->partials : nullptr, loss, dY, dW, dbias, st, &n);
    if (rc == HASTE_OK) {
      pf.end(HASTE_KERNEL_FORWARD, st);
      h->last_launches += n;
      return HASTE_OK;
    }
    if (rc != HASTE_ERR_UNSUPPORTED) return rc;
  }
  // every other shape: the two calls this one is defined as
  rc = haste_forward_loss(h, B, X, idx, W, bias, tgt_rowptr, tgt_col, loss, dY, nullptr, stream);
  if (rc) return rc;
  const int n_fwd = h->last_launches;
  if (dW || dbias) {
    rc = haste_backward(h, B, X, idx, W, dY, dW, dbias, nullptr, 0, stream);
    if (rc) return rc;
  } else {
    h->last_launches = 0;
  }
  h->last_launches += n_fwd;
  return HASTE_OK;
}

int haste_forward_logits(haste_layer_t* h, int B, const void* X, const int32_t* idx, const void* W, const float* bias, void* Z,
                         void* stream) {
  int rc = check_call(h, B, "haste_forward_logits");
  if (rc) return rc;
  if (!X || !idx || !W || !Z) { set_error("haste_forward_logits: X, idx, W and Z are required"); return HASTE_ERR_INVALID_ARG; }
  if (!aligned16(X) || !aligned16(W) || !aligned16(Z) || !aligned16(idx)) {
    set_error("haste_forward_logits: X, W, idx and Z must be 16-byte aligned");
    return HASTE_ERR_INVALID_ARG;
  }
  if (h->family != 1) {
    set_error("haste_forward_logits: only the tcgen05 kernel family has a logits-only forward (use haste_forward_loss with logits_out)");
    return HASTE_ERR_UNSUPPORTED;
  }
  DeviceGuard guard(h->device);
  cudaStream_t st = (cudaStream_t)stream;
  const TailShape sh = make_shape(h, B);
  Profiler& pf = *h->prof;
  h->last_launches = 0;
  if (B == 0 || h->NG == 0) return HASTE_OK;
  pf.begin(HASTE_KERNEL_PREP_FWD, st);
  rc = launch_transpose_pad(h->cfg.dtype, X, h->Xt, B, sh.d, h->Bpad, round_up(B, 128), st);
  if (rc) return rc;
  h->last_launches++;
  pf.end(HASTE_KERNEL_PREP_FWD, st);
  int n = 0;
  pf.begin(HASTE_KERNEL_FORWARD, st);
  rc = tc_tail_forward(h->tc, sh, h->Xt, idx, W, bias, nullptr, nullptr, nullptr, nullptr, Z, nullptr, 1, nullptr, nullptr, nullptr, st, &n);
  if (rc) return rc;
  pf.end(HASTE_KERNEL_FORWARD, st);
  h->last_launches += n;
  return HASTE_OK;
}

int haste_forward_topk(haste_layer_t* h, int B, const void* X, const int32_t* idx, const void* W, const float* bias, int k,
                       float* out_val, int64_t* out_idx, void* stream) {
  int rc = check_call(h, B, "haste_forward_topk");
  if (rc) return rc;
  if (!X || !idx || !W || !out_val || !out_idx) { set_error("haste_forward_topk: X, idx, W, out_val and out_idx are required"); return HASTE_ERR_INVALID_ARG; }
  if (k < 1 || k > 8) { set_error("haste_forward_topk: k must be in [1, 8]"); return HASTE_ERR_INVALID_ARG; }
  if (!aligned16(X) || !aligned16(W) || !aligned16(idx)) { set_error("haste_forward_topk: X, W and idx must be 16-byte aligned"); return HASTE_ERR_INVALID_ARG; }
  if (h->family != 1) { set_error("haste_forward_topk: only the tcgen05 kernel family has the fused top-k forward"); return HASTE_ERR_UNSUPPORTED; }
  DeviceGuard guard(h->device);
  cudaStream_t st = (cudaStream_t)stream;
  const TailShape sh = make_shape(h, B);
  Profiler& pf = *h->prof;
  h->last_launches = 0;
  if (B == 0) return HASTE_OK;
  if (!h->topk_val) {
    const size_t n = (size_t)tc_tail_num_sms(h->tc) * 4 * 128 * 8;
    if (cudaMalloc(&h->topk_val, n * 4) != cudaSuccess || cudaMalloc(&h->topk_idx, n * 4) != cudaSuccess) {
      set_error("haste_forward_topk: workspace allocation failed");
      return HASTE_ERR_NOMEM;
    }
  }
  if (h->NG == 0) {     // no labels: every slot empty
    HASTE_CUDA_TRY(cudaMemsetAsync(out_idx, 0xff, (size_t)B * k * 8, st));
    HASTE_CUDA_TRY(cudaMemsetAsync(out_val, 0xff, (size_t)B * k * 4, st));
    return HASTE_OK;
  }
  pf.begin(HASTE_KERNEL_PREP_FWD, st);
  rc = launch_transpose_pad(h->cfg.dtype, X, h->Xt, B, sh.d, h->Bpad, round_up(B, 128), st);
  if (rc) return rc;
  pf.end(HASTE_KERNEL_PREP_FWD, st);
  int n = 0;
  TopkGeom geom;
  geom.k = k;
  pf.begin(HASTE_KERNEL_FORWARD, st);
  rc = tc_tail_forward(h->tc, sh, h->Xt, idx, W, bias, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, 2, h->topk_val, h->topk_idx,
                       &geom, st, &n);
  if (rc) return rc;
  rc = launch_topk_merge(h->topk_val, h->topk_idx, geom.NP, geom.S, geom.NSET, ceil_div(B, 128), B, k, h->cfg.label_offset, out_val,
                         out_idx, st);
  if (rc) return rc;
  pf.end(HASTE_KERNEL_FORWARD, st);
  h->last_launches = n + 2;
  return HASTE_OK;
}

int haste_forward_topk_static(haste_layer_t* h, int B, const void* X, const int32_t* idx, const void* W, const float* bias, int k,
                              float* out_val, int64_t* out_idx, void* stream) {
  int rc = check_call(h, B, "haste_forward_topk_static");
  if (rc) return rc;
  if (!X || !idx || !W || !out_val || !out_idx) { set_error("haste_forward_topk_static: X, idx, W, out_val and out_idx are required"); return HASTE_ERR_INVALID_ARG; }
  if (k < 1 || k > 8) { set_error("haste_forward_topk_static: k must be in [1, 8]"); return HASTE_ERR_INVALID_ARG; }
  if (!aligned16(X) || !aligned16(W) || !aligned16(idx)) { set_error("haste_forward_topk_static: X, W and idx must be 16-byte aligned"); return HASTE_ERR_INVALID_ARG; }
  if (h->family != 1) { set_error("haste_forward_topk_static: only the tcgen05 kernel family has the fused top-k forward"); return HASTE_ERR_UNSUPPORTED; }
  // the forward kernel's grid is at most one CTA per SM, four epilogue sets of 128 rows x 8 candidates each
  const size_t need = (size_t)tc_tail_num_sms(h->tc) * 4 * 128 * 8;
  if (need > TOPK_STATIC_ENTRIES) {
    set_error("haste_forward_topk_static: this device has %d SMs, the static scratch holds the candidate lists of at most %d CTAs "
              "(%zu bytes); use haste_forward_topk", tc_tail_num_sms(h->tc), TOPK_STATIC_MAX_CTAS, sizeof(g_topk_static));
    return HASTE_ERR_UNSUPPORTED;
  }
  if (h->device < 0 || h->device >= TOPK_STATIC_MAX_DEVICES) {
    set_error("haste_forward_topk_static: device index %d beyond the %d devices the static scratch is tracked for", h->device, TOPK_STATIC_MAX_DEVICES);
    return HASTE_ERR_UNSUPPORTED;
  }
  float* cand_val = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_topk_static_mu);
    const TopkStaticDev& e = g_topk_static_dev[h->device];
    if (!e.tried || !e.ptr) {
      set_error("haste_forward_topk_static: the address of the static scratch is not known on device %d (cudaGetSymbolAddress: %s)",
                h->device, e.tried ? cudaGetErrorString(e.err) : "not asked for");
      return HASTE_ERR_CUDA;
    }
    cand_val = static_cast<float*>(e.ptr);
  }
  int* cand_idx = reinterpret_cast<int*>(cand_val + TOPK_STATIC_ENTRIES);
  DeviceGuard guard(h->device);
  cudaStream_t st = (cudaStream_t)stream;
  const TailShape sh = make_shape(h, B);
  Profiler& pf = *h->prof;
  h->last_launches = 0;
  if (B == 0) return HASTE_OK;
  if (h->NG == 0) {     // no labels: every slot empty
    HASTE_CUDA_TRY(cudaMemsetAsync(out_idx, 0xff, (size_t)B * k * 8, st));
    HASTE_CUDA_TRY(cudaMemsetAsync(out_val, 0xff, (size_t)B * k * 4, st));
    return HASTE_OK;
  }
  pf.begin(HASTE_KERNEL_PREP_FWD, st);
  rc = launch_transpose_pad(h->cfg.dtype, X, h->Xt, B, sh.d, h->Bpad, round_up(B, 128), st);
  if (rc) return rc;
  pf.end(HASTE_KERNEL_PREP_FWD, st);
  int n = 0;
  TopkGeom geom;
  geom.k = k;
  pf.begin(HASTE_KERNEL_FORWARD, st);
  rc = tc_tail_forward(h->tc, sh, h->Xt, idx, W, bias, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, 2, cand_val, cand_idx,
                       &geom, st, &n);
  if (rc) return rc;
  rc = launch_topk_merge(cand_val, cand_idx, geom.NP, geom.S, geom.NSET, ceil_div(B, 128), B, k, h->cfg.label_offset, out_val,
                         out_idx, st);
  if (rc) return rc;
  pf.end(HASTE_KERNEL_FORWARD, st);
  h->last_launches = n + 2;
  return HASTE_OK;
}

int haste_backward(haste_layer_t* h, int B, const void* X, const int32_t* idx, const void* W, const void* dY, void* dW,
                   float* dbias, float* dX, int accumulate_dX, void* stream) {
  int rc = check_call(h, B, "haste_backward");
  if (rc) return rc;
  if (!X || !idx || !W || !dY) { set_error("haste_backward: X, idx, W and dY are required"); return HASTE_ERR_INVALID_ARG; }
  if (!aligned16(X) || !aligned16(W) || !aligned16(dY) || !aligned16(dW) || !aligned16(idx)) {
    set_error("haste_backward: X, W, idx, dY and dW must be 16-byte aligned");
    return HASTE_ERR_INVALID_ARG;
  }
  DeviceGuard guard(h->device);
  cudaStream_t st = (cudaStream_t)stream;
  const TailShape sh = make_shape(h, B);
  Profiler& pf = *h->prof;
  h->last_launches = 0;
  if (B == 0 || h->NG == 0) {
    if (dW && h->cfg.L > 0)
      HASTE_CUDA_TRY(cudaMemsetAsync(dW, 0, (size_t)h->cfg.L * h->cfg.K * esize(h->cfg.dw_dtype), st));
    if (dbias && h->cfg.L > 0) HASTE_CUDA_TRY(cudaMemsetAsync(dbias, 0, (size_t)h->cfg.L * 4, st));
    if (dX && !accumulate_dX && B > 0) HASTE_CUDA_TRY(cudaMemsetAsync(dX, 0, (size_t)B * sh.d * 4, st));
    return HASTE_OK;
  }
  // The gather operand X^T is rebuilt here: backward must not depend on which forward ran last -- unless the caller
  // promised that it is the forward of the same step (HASTE_XT_FROM_FORWARD).
  pf.begin(HASTE_KERNEL_PREP_BWD, st);
  if ((dW || dbias) && !(h->cfg.flags & HASTE_XT_FROM_FORWARD)) {
    rc = launch_transpose_pad(h->cfg.dtype, X, h->Xt, B, sh.d, h->Bpad, round_up(B, 128), st);
    if (rc) return rc;
    h->last_launches++;
  }
  if (dX) {      // zero already unless an earlier pass ended between its dX kernel and the transpose-out (no memset between kernels: PDL)
    if (!h->dxt_clean) HASTE_CUDA_TRY(cudaMemsetAsync(h->dXt, 0, (size_t)sh.d * h->Bpad * 4, st));
    h->dxt_clean = false;
  }
  pf.end(HASTE_KERNEL_PREP_BWD, st);
  if (dW || dbias) {
    pf.begin(HASTE_KERNEL_DW, st);
    rc = HASTE_ERR_UNSUPPORTED;
    if (h->family == 1) {
      int n = 0;
      rc = tc_tail_dw(h->tc, sh, h->Xt, idx, dY, dW, dbias, st, &n);
      if (rc == HASTE_OK) h->last_launches += n;
    }
    if (rc == HASTE_ERR_UNSUPPORTED) {   // shapes / outputs the tcgen05 dW kernel does not cover run the CUDA-core kernel
      rc = launch_simt_dw(h->cfg.dtype, h->cfg.dw_dtype, sh, h->Xt, idx, dY, dW, dbias, st);
      h->last_launches++;
    }
    if (rc) return rc;
    pf.end(HASTE_KERNEL_DW, st);
  }
  if (dX) {
    pf.begin(HASTE_KERNEL_DX, st);
    rc = HASTE_ERR_UNSUPPORTED;
    if (h->family == 1) {
      int n = 0;
      if (h->dx_part) {
        int NT = 0, S = 0;
        tc_tail_dx_grid(h->tc, sh, &NT, &S);
        if (NT * S > tc_tail_num_sms(h->tc)) { set_error("haste_backward: batch too large for the deterministic dX workspace"); return HASTE_ERR_UNSUPPORTED; }
        HASTE_CUDA_TRY(cudaMemsetAsync(h->dx_part, 0, (size_t)NT * S * sh.d * 128 * 4, st));
        rc = tc_tail_dx(h->tc, sh, idx, W, dY, h->dXt, h->dx_part, st, &n);
        if (rc == HASTE_OK) { rc = launch_reduce_dx_parts(h->dx_part, h->dXt, sh.d, h->Bpad, NT, S, st); ++n; }
        if (rc == HASTE_ERR_UNSUPPORTED) { set_error("haste_backward: no atomic-free dX kernel for this call"); return rc; }
      } else {
        rc = tc_tail_dx(h->tc, sh, idx, W, dY, h->dXt, nullptr, st, &n);
      }
      if (rc == HASTE_OK) h->last_launches += n;
    }
    if (rc == HASTE_ERR_UNSUPPORTED) {
      rc = launch_simt_dx(h->cfg.dtype, sh, idx, W, dY, h->dXt, st);
      h->last_launches++;
    }
    if (rc) return rc;
    pf.end(HASTE_KERNEL_DX, st);
    pf.begin(HASTE_KERNEL_POST_BWD, st);
    rc = launch_untranspose_f32(h->dXt, dX, B, sh.d, h->Bpad, accumulate_dX, st);
    if (rc) return rc;
    h->dxt_clean = true;
    h->last_launches++;
    pf.end(HASTE_KERNEL_POST_BWD, st);
  }
  return HASTE_OK;
}

int haste_backward_sgd(haste_layer_t* h, int B, const void* X, const int32_t* idx, void* W, const void* dY, float* momentum,
                       float* bias, float* bias_momentum, float lr, float mu, float weight_decay, float* dX, int accumulate_dX,
                       void* stream) {
  int rc = check_call(h, B, "haste_backward_sgd");
  if (rc) return rc;
  if (!X || !idx || !W || !dY || !momentum) { set_error("haste_backward_sgd: X, idx, W, dY and momentum are required"); return HASTE_ERR_INVALID_ARG; }
  if ((bias == nullptr) != (bias_momentum == nullptr)) { set_error("haste_backward_sgd: bias and bias_momentum go together"); return HASTE_ERR_INVALID_ARG; }
  if (!aligned16(X) || !aligned16(W) || !aligned16(dY) || !aligned16(momentum) || !aligned16(idx)) {
    set_error("haste_backward_sgd: X, W, idx, dY and momentum must be 16-byte aligned");
    return HASTE_ERR_INVALID_ARG;
  }
  if (h->family != 1 || h->dx_part) {
    set_error("haste_backward_sgd: needs the tcgen05 kernel family (bf16, G in {8,16,32,64,128}, K in {64,128}) without HASTE_DETERMINISTIC");
    return HASTE_ERR_UNSUPPORTED;
  }
  DeviceGuard guard(h->device);
  cudaStream_t st = (cudaStream_t)stream;
  const TailShape sh = make_shape(h, B);
  Profiler& pf = *h->prof;
  h->last_launches = 0;
  if (B == 0 || h->NG == 0) return HASTE_OK;     // an empty batch has a zero gradient: with mu v the step would still move W; defined as a no-op
  pf.begin(HASTE_KERNEL_PREP_BWD, st);
  if (!(h->cfg.flags & HASTE_XT_FROM_FORWARD)) {
    rc = launch_transpose_pad(h->cfg.dtype, X, h->Xt, B, sh.d, h->Bpad, round_up(B, 128), st);
    if (rc) return rc;
    h->last_launches++;
  }
  if (dX) {      // zero already unless an earlier pass ended between its dX kernel and the transpose-out (no memset between kernels: PDL)
    if (!h->dxt_clean) HASTE_CUDA_TRY(cudaMemsetAsync(h->dXt, 0, (size_t)sh.d * h->Bpad * 4, st));
    h->dxt_clean = false;
  }
  pf.end(HASTE_KERNEL_PREP_BWD, st);
  int n = 0;
  if (dX) {        // the input gradient first: it needs W as it was in the forward, the update below overwrites it
    pf.begin(HASTE_KERNEL_DX, st);
    rc = tc_tail_dx(h->tc, sh, idx, W, dY, h->dXt, nullptr, st, &n);
    if (rc == HASTE_ERR_UNSUPPORTED) set_error("haste_backward_sgd: no tcgen05 dX kernel for G = %d, K = %d, B = %d", sh.G, sh.K, B);
    if (rc) return rc;
    h->last_launches += n;
    pf.end(HASTE_KERNEL_DX, st);
    pf.begin(HASTE_KERNEL_POST_BWD, st);
    rc = launch_untranspose_f32(h->dXt, dX, B, sh.d, h->Bpad, accumulate_dX, st);
    if (rc) return rc;
    h->dxt_clean = true;
    h->last_launches++;
    pf.end(HASTE_KERNEL_POST_BWD, st);
  }
  pf.begin(HASTE_KERNEL_DW, st);
  rc = tc_tail_dw_sgd(h->tc, sh, h->Xt, idx, dY, W, momentum, bias, bias_momentum, lr, mu, weight_decay, st, &n);
  if (rc == HASTE_ERR_UNSUPPORTED) set_error("haste_backward_sgd: no fused kernel for G = %d, K = %d", sh.G, sh.K);
  if (rc) return rc;
  h->last_launches += n;
  pf.end(HASTE_KERNEL_DW, st);
  return HASTE_OK;
}

int haste_rewire(haste_layer_t* h, int32_t* idx, void* W, float* momentum, float rho, int init_random, uint64_t seed, int resort,
                 int64_t* n_pruned, void* stream) {
  if (n_pruned) *n_pruned = 0;
  if (!h || !idx || !W) { set_error("haste_rewire: handle, idx and W are required"); return HASTE_ERR_INVALID_ARG; }
  if (!(rho >= 0.f && rho <= 1.f)) { set_error("haste_rewire: rho must be in [0, 1]"); return HASTE_ERR_INVALID_ARG; }
  DeviceGuard guard(h->device);
  const int64_t n = h->NG * h->cfg.K;
  const int64_t m = (int64_t)std::floor((double)n * (double)rho);
  if (n_pruned) *n_pruned = m;
  if (m <= 0) return HASTE_OK;
  if (!h->rw_ws && cudaMalloc(&h->rw_ws, rewire_workspace_bytes(h->NG, h->cfg.K)) != cudaSuccess) {
    set_error("haste_rewire: workspace allocation failed");
    return HASTE_ERR_NOMEM;
  }
  int rc = launch_rewire(h->cfg.dtype, idx, W, momentum, h->cfg.L, h->cfg.G, h->cfg.K, h->cfg.d, m, init_random ? 1 : 0, seed,
                         resort ? 1 : 0, h->rw_ws, (cudaStream_t)stream);
  if (rc == HASTE_ERR_UNSUPPORTED) set_error("haste_rewire: shape not supported (K <= 3000)");
  h->last_launches = 5;
  return rc;
}

int haste_set_profiling(haste_layer_t* h, int depth) {
  if (!h) { set_error("haste_set_profiling: handle is NULL"); return HASTE_ERR_INVALID_ARG; }
  DeviceGuard guard(h->device);
  return h->prof->enable(depth);
}
int haste_kernel_ms(haste_layer_t* h, int kernel, int age, float* ms) {
  if (!h) { set_error("haste_kernel_ms: handle is NULL"); return HASTE_ERR_INVALID_ARG; }
  DeviceGuard guard(h->device);
  return h->prof->ms(kernel, age, ms);
}

int haste_dy_unpack(const haste_layer_t* h, int B, const void* dY, float* out_BL, void* stream) {
  int rc = check_call(h, B, "haste_dy_unpack");
  if (rc) return rc;
  if (!dY || !out_BL) { set_error("haste_dy_unpack: NULL argument"); return HASTE_ERR_INVALID_ARG; }
  DeviceGuard guard(h->device);
  return launch_dy_unpack(h->cfg.dtype, dY, out_BL, B, h->cfg.L, h->cfg.G, (cudaStream_t)stream);
}

int haste_dy_pack(const haste_layer_t* h, int B, const float* in_BL, void* dY, void* stream) {
  int rc = check_call(h, B, "haste_dy_pack");
  if (rc) return rc;
  if (!dY || !in_BL) { set_error("haste_dy_pack: NULL argument"); return HASTE_ERR_INVALID_ARG; }
  DeviceGuard guard(h->device);
  return launch_dy_pack(h->cfg.dtype, in_BL, dY, B, h->cfg.L, h->cfg.G, (cudaStream_t)stream);
}

// ---------------------------------------------------------------------------------
// dense head
// ---------------------------------------------------------------------------------
int haste_head_create(haste_head_t** out, int32_t d, int64_t L_h, int32_t B_max, haste_dtype_t dtype,
                      int64_t label_offset, float loss_scale, uint32_t flags, int cuda_device) {
  if (!out) { set_error("haste_head_create: out is NULL"); return HASTE_ERR_INVALID_ARG; }
  *out = nullptr;
  if (d <= 0 || L_h < 0 || B_max <= 0 || L_h > 0x7fffffffLL || (dtype != HASTE_F32 && dtype != HASTE_BF16)) {
    set_error("haste_head_create: bad sizes or dtype");
    return HASTE_ERR_INVALID_ARG;
  }
  // grids of the generic CUDA-core head kernels put ceil(L_h/64) and ceil(B/64) into gridDim.y
  if (L_h > 65535LL * 64 || B_max > 65535 * 64) {
    set_error("haste_head_create: L_h <= 4 194 240 and B_max <= 4 194 240 are supported");
    return HASTE_ERR_UNSUPPORTED;
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || cuda_device < 0 || cuda_device >= ndev) {
    cudaGetLastError();
    set_error("haste_head_create: CUDA device %d not available (no CPU fallback exists)", cuda_device);
    return HASTE_ERR_CUDA;
  }
  DeviceGuard guard(cuda_device);
  haste_head* h = new (std::nothrow) haste_head();
  if (!h) return HASTE_ERR_NOMEM;
  memset(h, 0, sizeof(*h));
  h->d = d; h->L = L_h; h->B_max = B_max; h->dtype = dtype; h->label_offset = label_offset;
  h->loss_scale = loss_scale; h->flags = flags; h->device = cuda_device;
  h->n_partials = 1024;
  h->prof = new (std::nothrow) Profiler();
  if (!h->prof) { delete h; return HASTE_ERR_NOMEM; }
  cudaError_t e = cudaMalloc(&h->loss_acc, sizeof(double));
  if (e == cudaSuccess) e = cudaMalloc(&h->partials, h->n_partials * sizeof(float));
  if (e == cudaSuccess) e = cudaMemset(h->partials, 0, h->n_partials * sizeof(float));
  if (e != cudaSuccess) {
    set_error("haste_head_create: allocation failed: %s", cudaGetErrorString(e));
    haste_head_destroy(h);
    return HASTE_ERR_CUDA;
  }
  h->family = 0;
  if (!(flags & HASTE_FORCE_SIMT) && tc_head_supported(d, L_h, B_max, dtype, cuda_device)) {
    int rc = tc_head_create(&h->tc, d, L_h, B_max, cuda_device);
    if (rc != HASTE_OK) { haste_head_destroy(h); return rc; }
    h->family = 1;
  }
  *out = h;
  return HASTE_OK;
}

int haste_head_destroy(haste_head_t* h) {
  if (!h) return HASTE_OK;
  DeviceGuard guard(h->device);
  if (h->tc) tc_head_destroy(h->tc);
  if (h->prof) { h->prof->destroy(); delete h->prof; }
  cudaFree(h->loss_acc); cudaFree(h->partials);
  delete h;
  return HASTE_OK;
}

int haste_head_kernel_family(const haste_head_t* h) { return h ? h->family : -1; }
int haste_head_last_launch_count(const haste_head_t* h) { return h ? h->last_launches : 0; }

static HeadShape make_head_shape(const haste_head_t* h, int B) {
  HeadShape sh;
  sh.d = h->d; sh.B = B; sh.L = h->L; sh.label_offset = h->label_offset;
  sh.s = h->loss_scale != 0.f ? h->loss_scale : (B > 0 ? 1.0f / (float)B : 0.f);
  return sh;
}

int haste_head_forward_loss(haste_head_t* h, int B, const void* X, const void* Wh, const float* bias,
                            const int32_t* tgt_rowptr, const int32_t* tgt_col, float* loss, void* dY,
                            float* logits_out, void* stream) {
  if (!h) { set_error("haste_head_forward_loss: handle is NULL"); return HASTE_ERR_INVALID_ARG; }
  if (B < 0 || B > h->B_max) { set_error("haste_head_forward_loss: B=%d outside [0, B_max=%d]", B, h->B_max); return HASTE_ERR_INVALID_ARG; }
  if (!X || !Wh) { set_error("haste_head_forward_loss: X and Wh are required"); return HASTE_ERR_INVALID_ARG; }
  if ((tgt_rowptr == nullptr) != (tgt_col == nullptr)) {
    set_error("haste_head_forward_loss: tgt_rowptr and tgt_col must both be given or both be NULL");
    return HASTE_ERR_INVALID_ARG;
  }
  if (!aligned16(X) || !aligned16(Wh) || !aligned16(dY)) {
    set_error("haste_head_forward_loss: X, Wh and dY must be 16-byte aligned");
    return HASTE_ERR_INVALID_ARG;
  }
  DeviceGuard guard(h->device);
  cudaStream_t st = (cudaStream_t)stream;
  const HeadShape sh = make_head_shape(h, B);
  Profiler& pf = *h->prof;
  h->last_launches = 0;
  if (B == 0 || h->L == 0) {
    if (loss) HASTE_CUDA_TRY(cudaMemsetAsync(loss, 0, sizeof(float), st));
    return HASTE_OK;
  }
  int rc;
  if (h->family == 1) {
    int n = 0;
    pf.begin(HASTE_KERNEL_FORWARD, st);
    rc = tc_head_forward(h->tc, sh, X, Wh, bias, tgt_rowptr, tgt_col, loss ? h->partials : nullptr, loss, dY, logits_out, st, &n);
    if (rc) return rc;
    pf.end(HASTE_KERNEL_FORWARD, st);
    h->last_launches += n;
    return HASTE_OK;
  }
  if (loss) HASTE_CUDA_TRY(cudaMemsetAsync(h->loss_acc, 0, sizeof(double), st));
  pf.begin(HASTE_KERNEL_FORWARD, st);
  rc = launch_simt_head_forward(h->dtype, sh, X, Wh, bias, tgt_rowptr, tgt_col, loss ? h->loss_acc : nullptr, dY,
                                logits_out, st);
  if (rc) return rc;
  pf.end(HASTE_KERNEL_FORWARD, st);
  h->last_launches++;
  if (loss) {
    rc = launch_finalize_loss(h->loss_acc, nullptr, 0, sh.s, loss, st);
    if (rc) return rc;
    h->last_launches++;
  }
  return HASTE_OK;
}

int haste_head_backward(haste_head_t* h, int B, const void* X, const void* Wh, const void* dY, void* dWh, float* dbias,
                        float* dX, int accumulate_dX, void* stream) {
  if (!h) { set_error("haste_head_backward: handle is NULL"); return HASTE_ERR_INVALID_ARG; }
  if (B < 0 || B > h->B_max) { set_error("haste_head_backward: B=%d outside [0, B_max=%d]", B, h->B_max); return HASTE_ERR_INVALID_ARG; }
  if (!X || !Wh || !dY) { set_error("haste_head_backward: X, Wh and dY are required"); return HASTE_ERR_INVALID_ARG; }
  if (!aligned16(X) || !aligned16(Wh) || !aligned16(dY) || !aligned16(dWh)) {
    set_error("haste_head_backward: X, Wh, dY and dWh must be 16-byte aligned");
    return HASTE_ERR_INVALID_ARG;
  }
  DeviceGuard guard(h->device);
  cudaStream_t st = (cudaStream_t)stream;
  const HeadShape sh = make_head_shape(h, B);
  h->last_launches = 0;
  if (B == 0 || h->L == 0) {
    if (dWh && h->L > 0) HASTE_CUDA_TRY(cudaMemsetAsync(dWh, 0, (size_t)h->L * h->d * esize(h->dtype), st));
    if (dbias && h->L > 0) HASTE_CUDA_TRY(cudaMemsetAsync(dbias, 0, (size_t)h->L * 4, st));
    if (dX && !accumulate_dX && B > 0) HASTE_CUDA_TRY(cudaMemsetAsync(dX, 0, (size_t)B * h->d * 4, st));
    return HASTE_OK;
  }
  Profiler& pf = *h->prof;
  pf.begin(HASTE_KERNEL_DW, st);     // the head's backward is timed as one unit (dW, db and dX)
  if (h->family == 1) {
    int n = 0;
    int rc = tc_head_backward(h->tc, sh, X, Wh, dY, dWh, dbias, dX, accumulate_dX, (h->flags & HASTE_DETERMINISTIC) ? 1 : 0, st, &n);
    if (rc) return rc;
    h->last_launches += n;
  } else {
    int rc = launch_simt_head_backward(h->dtype, sh, X, Wh, dY, dWh, dbias, dX, accumulate_dX, st);
    if (rc) return rc;
    h->last_launches += (dWh ? 1 : 0) + (dX ? 1 : 0) + (dbias ? 1 : 0);
  }
  pf.end(HASTE_KERNEL_DW, st);
  return HASTE_OK;
}

int haste_head_set_profiling(haste_head_t* h, int depth) {
  if (!h) { set_error("haste_head_set_profiling: handle is NULL"); return HASTE_ERR_INVALID_ARG; }
  DeviceGuard guard(h->device);
  return h->prof->enable(depth);
}
int haste_head_kernel_ms(haste_head_t* h, int kernel, int age, float* ms) {
  if (!h) { set_error("haste_head_kernel_ms: handle is NULL"); return HASTE_ERR_INVALID_ARG; }
  DeviceGuard guard(h->device);
  return h->prof->ms(kernel, age, ms);
}

}  // extern "C"
