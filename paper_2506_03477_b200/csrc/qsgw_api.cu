// C-ABI layer of include/qsgw.h: context, argument validation, state machine, band-batch loop,
// host-buffer driver.  All arithmetic of the path runs in the kernels of zmel_kernels.cu and
// chi0_*_kernels.cu; there is no CPU fallback.
#include "../../include/qsgw.h"

#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <algorithm>
#include <string>
#include <vector>

#include "kernels.h"

namespace {

enum State { ST_CREATED = 0, ST_READY = 1, ST_Z_BUILT = 2 };

thread_local std::string g_create_error;

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_tiled() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  return fn;
}

inline long long round_up(long long x, long long m) { return (x + m - 1) / m * m; }

}  // namespace

namespace qsgw {

cudaError_t make_zmap(CUtensorMap* out, const double2* base, long long inner, long long outer, long long ld,
                      long long d2, long long s2, long long d3, long long s3, int box_rows) {
  EncodeTiledFn enc = get_encode_tiled();
  if (!enc) return cudaErrorNotSupported;
  if (inner < 1 || outer < 1 || ld < inner || d2 < 1 || d3 < 1) return cudaErrorInvalidValue;
  // a dimension of extent 1 still needs a valid (non-zero, 16-byte multiple) stride
  const unsigned long long plane = (unsigned long long)ld * (unsigned long long)outer * 16ull;
  const unsigned long long st2 = (d2 > 1 && s2 > 0) ? (unsigned long long)s2 * 16ull : plane;
  const unsigned long long st3 = (d3 > 1 && s3 > 0) ? (unsigned long long)s3 * 16ull : (st2 > plane ? st2 : plane) * (unsigned long long)d2;
  const cuuint64_t gdim[4] = {(cuuint64_t)(2 * inner), (cuuint64_t)outer, (cuuint64_t)d2, (cuuint64_t)d3};
  const cuuint64_t gstr[3] = {(cuuint64_t)ld * 16ull, (cuuint64_t)st2, (cuuint64_t)st3};
  const cuuint32_t box[4] = {16, (cuuint32_t)box_rows, 1, 1};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<double2*>(base), gdim, gstr, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

cudaError_t make_hl16_map(CUtensorMap* out, const void* base, long long row_halves, long long rows, long long plane_halves) {
  EncodeTiledFn enc = get_encode_tiled();
  if (!enc) return cudaErrorNotSupported;
  const cuuint64_t gdim[3] = {(cuuint64_t)row_halves, (cuuint64_t)rows, 2};
  const cuuint64_t gstr[2] = {(cuuint64_t)row_halves * 2, (cuuint64_t)plane_halves * 2};
  const cuuint32_t box[3] = {64, 64, 1};
  const cuuint32_t estr[3] = {1, 1, 1};
  CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 3, const_cast<void*>(base), gdim, gstr, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

cudaError_t make_hb8_map(CUtensorMap* out, const void* base, long long row_halves, long long rows, long long plane_halves) {
  EncodeTiledFn enc = get_encode_tiled();
  if (!enc) return cudaErrorNotSupported;
  const cuuint64_t gdim[3] = {(cuuint64_t)row_halves * 2, (cuuint64_t)rows, 2};
  const cuuint64_t gstr[2] = {(cuuint64_t)row_halves * 2, (cuuint64_t)plane_halves * 2};
  const cuuint32_t box[3] = {128, 64, 1};
  const cuuint32_t estr[3] = {1, 1, 1};
  CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<void*>(base), gdim, gstr, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

}  // namespace qsgw

struct qsgw_ctx {
  // problem
  int n_sites = 0, n_b = 0, n_m = 0, b_max = 0, n_freq = 0, n_k = 0;
  int max_n_o = 0, max_n_u = 0, precision = 0;
  double occ_tol = 1e-12;
  std::vector<int> orb, pb;
  std::vector<double> omega;
  cudaStream_t stream = nullptr;
  // derived
  int ncg = 0, n_m_pad = 0, n_tiles = 0, n_tiles_half = 0, n_tiles_quarter = 0;
  long long kpad = 0;           // pair capacity of the z workspace (multiple of 32): several band batches are
  long long fill = 0;           // staged back to back ([0, fill) is pending) and accumulated by ONE stage (b) launch
  // device
  int* d_pb_site = nullptr;
  int* d_pb_off = nullptr;
  int* d_orb_off = nullptr;
  long long* d_p_off = nullptr;
  int4* d_tiles = nullptr;
  double* d_omega = nullptr;
  double2* d_P = nullptr;
  long long p_elems = 0;
  double* d_zws = nullptr;
  double* d_wtab = nullptr;
  float* d_wtab32 = nullptr;    // mixed mode: fp16 weight pieces (same bytes per pair as an FP32 table)
  bool f16 = false;             // QSGW_PREC_MIXED: FP16-split planes (kernels.h "hl16")
  void* d_zhl = nullptr;
  void* d_zhb8 = nullptr;       // B rows of the E5M2-corrected variant: h | e5m2(v) | e5m2(v-h)
  CUtensorMap tmap_hb8;
  double* d_wscale = nullptr;
  float* d_zmax = nullptr;
  // stage (b) runs only the 32-pair stages that carry weight (option "skip_dead_stages"): list, count, flag scratch
  int* d_live = nullptr;
  int* d_n_live = nullptr;
  unsigned char* d_stage_flags = nullptr;
  int skip_dead = 1;            // 0 never | 1 for flushes of >= 4 M staged matrix elements (default) | 2 always
  // mixed, direct stage (a) on tcgen05 (option "zmel_direct"): max_I ||P_I||_F per site, per-batch norm scratch, A operand
  float* d_pmax = nullptr;
  float* d_cnorm = nullptr;
  size_t cnorm_cap = 0;
  __half* d_aop = nullptr;
  size_t aop_cap = 0;
  int zmel_direct = 0;          // 0 never | 1 for launches of >= 8 M matrix elements (default where supported) | 2 always
  qsgw::MixedCtl* d_ctl = nullptr;   // device-side choice of the product variant per flush
  int fp8_mode = 2;             // 0 never | 1 always | 2 chosen on the device (option "mixed_fp8")
  double fp8_thr = 4.0;         // automatic choice: E5M2 when P_eff >= fp8_thr * N_M (measured, DESIGN.md 4b:
                                // 1.2e-5 at P_eff = 4.8 N_M, 1.6e-5 at 2.4 N_M, 2.2e-5 at 0.7 N_M)
  int win = 8;                  // stages per TMEM drain window
  int mixed_pair = 1;           // stage (b) on CTA pairs (cta_group::2) (option "mixed_pair")
  int zmel_kt = 0;              // stage (a) DMMA kernel: padded contraction length (0 = CUDA-core kernel)
  int zmel_kt_avail = 0;        // ... as computed at creation (option "zmel_dmma" switches zmel_kt between 0 and this)
  int device = 0, n_sm = 148;   // device the context lives on
  long long batch_pad = 0;      // padded pairs of the largest band batch
  long long stage_cap = 0;      // staged pairs that trigger a flush (<= kpad; option "stage_batches")
  long long z_off = 0;          // workspace slot of the batch the last zmel_build wrote
  int z_zi = 0;                 // ... and the index of its FP16 scale in d_zmax
  int zslot = 0;                // batches staged since the last flush (next free index of d_zmax)
  int e2e_groups = 4;           // frequency groups of the last flush of qsgw_chi0_run_host
  // binned real-axis path (qsgw_imchi_add_batch; allocated by its first call)
  int* d_rowmap = nullptr;      // [batch_pad] workspace row of every pair of the batch
  int* d_binscratch = nullptr;  // [2 batch_pad + 4 (n_freq + 1)]
  int2* d_ranges = nullptr;     // [n_freq] rows touched by each bin
  const int* cur_row_map = nullptr;   // row map of the stage (a) launch being issued (NULL: natural pair order)
  const int2* flush_ranges = nullptr; // binned path, mixed mode: per-bin row ranges of the flush being issued
  const float* flush_zfold = nullptr; // ... and the batch maximum whose FP16 scale its caller-made weights still lack
  // I^c workspace (qsgw_sigc_imag_accumulate; allocated by its first call)
  double2* d_sz = nullptr;      // z of the batch, complex128 [pairs][N_M]
  double2* d_szw = nullptr;     // ZW^c, same shape
  double* d_sw = nullptr;       // quadrature weights [n_freq][batch_pad]
  __half* d_zk16 = nullptr;     // mixed I^c: z rows as FP16 pieces, K = product functions (sigc_f16_kernels.cu)
  __half* d_w16 = nullptr;      // mixed I^c: (W^c_i)^T rows as FP16 pieces
  unsigned char* d_w8 = nullptr;  // ... and their hb8 copy (E5M2 correction products, option "sigc_fp8")
  int sigc_fp8 = 1;
  float* d_samax = nullptr;     // mixed I^c: max |z|, max |W_i|  [1 + n_freq]
  bool sigc_f64 = false;        // option "sigc_f64": a mixed context runs the FP64 GEMM on its FP32-grade z
  CUtensorMap tmap_h;
  double* d_acc_re = nullptr;
  double* d_acc_im = nullptr;
  size_t device_bytes = 0;
  CUtensorMap tmap_z;
  // state
  int state = ST_CREATED;
  int last_n_o = 0, last_n_u = 0;
  long long launches = 0, pairs = 0;
  std::string err;
  // per-stage event timing (qsgw_set_stage_timing)
  bool timing = false;
  struct EvPair { cudaEvent_t a, b; int stage; };
  std::vector<EvPair> ev_pending;
  std::vector<cudaEvent_t> ev_free;
  double stage_ms[QSGW_N_STAGES] = {0, 0, 0, 0};
  long long stage_n[QSGW_N_STAGES] = {0, 0, 0, 0};
  // device staging buffers of qsgw_chi0_run_host (allocated by its first call)
  struct HostRun {
    double2* dP = nullptr;
    double2* dCk[2] = {nullptr, nullptr};
    double2* dCkq[2] = {nullptr, nullptr};
    double* dE[2] = {nullptr, nullptr};       // eps_k | f_k | eps_kq | f_kq
    double2* dOut = nullptr;
    size_t ck_cap = 0, ckq_cap = 0, e_cap = 0;
    cudaEvent_t done[2] = {nullptr, nullptr};
    cudaEvent_t ready[4] = {nullptr, nullptr, nullptr, nullptr};
    cudaStream_t cp = nullptr;
  } hr;

  int fail(int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof(buf), fmt, ap);
    va_end(ap);
    err = buf;
    return code;
  }
  int cuda_fail(cudaError_t e, const char* what) {
    return fail(QSGW_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
  }
};

namespace {

template <typename T>
cudaError_t dev_alloc(qsgw_ctx* c, T** p, size_t n) {
  cudaError_t e = cudaMalloc(reinterpret_cast<void**>(p), n * sizeof(T));
  if (e == cudaSuccess) c->device_bytes += n * sizeof(T);
  return e;
}

void free_all(qsgw_ctx* c) {
  for (auto& p : c->ev_pending) { cudaEventDestroy(p.a); cudaEventDestroy(p.b); }
  for (auto e : c->ev_free) cudaEventDestroy(e);
  c->ev_pending.clear();
  c->ev_free.clear();
  cudaFree(c->d_pb_site);
  cudaFree(c->d_pb_off);
  cudaFree(c->d_orb_off);
  cudaFree(c->d_p_off);
  cudaFree(c->d_tiles);
  cudaFree(c->d_omega);
  cudaFree(c->d_P);
  cudaFree(c->d_zws);
  cudaFree(c->d_wtab);
  cudaFree(c->d_wtab32);
  cudaFree(c->d_ctl);
  cudaFree(c->hr.dP);
  cudaFree(c->hr.dOut);
  for (int i = 0; i < 2; ++i) {
    cudaFree(c->hr.dCk[i]);
    cudaFree(c->hr.dCkq[i]);
    cudaFree(c->hr.dE[i]);
    if (c->hr.done[i]) cudaEventDestroy(c->hr.done[i]);
  }
  for (int i = 0; i < 4; ++i) if (c->hr.ready[i]) cudaEventDestroy(c->hr.ready[i]);
  if (c->hr.cp) cudaStreamDestroy(c->hr.cp);
  cudaFree(c->d_rowmap);
  cudaFree(c->d_binscratch);
  cudaFree(c->d_ranges);
  cudaFree(c->d_zk16);
  cudaFree(c->d_w16);
  cudaFree(c->d_w8);
  cudaFree(c->d_samax);
  cudaFree(c->d_sz);
  cudaFree(c->d_szw);
  cudaFree(c->d_sw);
  cudaFree(c->d_zhl);
  cudaFree(c->d_zhb8);
  cudaFree(c->d_wscale);
  cudaFree(c->d_zmax);
  cudaFree(c->d_live);
  cudaFree(c->d_n_live);
  cudaFree(c->d_stage_flags);
  cudaFree(c->d_pmax);
  cudaFree(c->d_cnorm);
  cudaFree(c->d_aop);
  cudaFree(c->d_acc_re);
  cudaFree(c->d_acc_im);
}

cudaEvent_t ev_get(qsgw_ctx* c) {
  if (!c->ev_free.empty()) {
    cudaEvent_t e = c->ev_free.back();
    c->ev_free.pop_back();
    return e;
  }
  cudaEvent_t e = nullptr;
  cudaEventCreate(&e);
  return e;
}

// move finished event pairs into the per-stage sums; `block` waits for all of them
void ev_harvest(qsgw_ctx* c, bool block) {
  size_t keep = 0;
  for (size_t i = 0; i < c->ev_pending.size(); ++i) {
    qsgw_ctx::EvPair& p = c->ev_pending[i];
    cudaError_t q = block ? cudaEventSynchronize(p.b) : cudaEventQuery(p.b);
    if (q == cudaSuccess) {
      float ms = 0.f;
      if (cudaEventElapsedTime(&ms, p.a, p.b) == cudaSuccess) {
        c->stage_ms[p.stage] += ms;
        c->stage_n[p.stage] += 1;
      }
      c->ev_free.push_back(p.a);
      c->ev_free.push_back(p.b);
    } else {
      if (q == cudaErrorNotReady) cudaGetLastError();
      c->ev_pending[keep++] = p;
    }
  }
  c->ev_pending.resize(keep);
}

// Brackets one kernel launch with events when stage timing is on.
struct StageScope {
  qsgw_ctx* c;
  cudaEvent_t a = nullptr;
  int stage;
  StageScope(qsgw_ctx* ctx, int st) : c(ctx), stage(st) {
    if (c->timing) {
      if (c->ev_pending.size() > 4096) ev_harvest(c, false);
      a = ev_get(c);
      cudaEventRecord(a, c->stream);
    }
  }
  ~StageScope() {
    if (a) {
      cudaEvent_t b = ev_get(c);
      cudaEventRecord(b, c->stream);
      c->ev_pending.push_back({a, b, stage});
    }
  }
};

int create_fail(qsgw_ctx* c, int code, const std::string& msg) {
  g_create_error = msg;
  if (c) {
    free_all(c);
    delete c;
  }
  return code;
}

int validate_desc(const qsgw_desc* d, std::string& why) {
  if (!d) { why = "desc is NULL"; return QSGW_ERR_INVALID_ARG; }
  if (!d->h_orb_per_site || !d->h_pb_per_site || !d->h_omega) { why = "NULL array in desc"; return QSGW_ERR_INVALID_ARG; }
  if (d->precision != QSGW_PREC_FP64 && d->precision != QSGW_PREC_MIXED) { why = "bad precision enum"; return QSGW_ERR_INVALID_ARG; }
  if (d->n_sites < 1 || d->n_freq < 1 || d->n_k < 1 || d->max_n_o < 1 || d->max_n_u < 1) {
    why = "non-positive extent in desc"; return QSGW_ERR_SHAPE;
  }
  for (int s = 0; s < d->n_sites; ++s)
    if (d->h_orb_per_site[s] < 1 || d->h_pb_per_site[s] < 1) { why = "non-positive b_s or m_s"; return QSGW_ERR_SHAPE; }
  for (int j = 0; j < d->n_freq; ++j) {
    const double w = d->h_omega[j];
    if (!(w >= 0.0) || (j > 0 && !(w > d->h_omega[j - 1]))) {
      why = "omega must be >= 0 and strictly increasing"; return QSGW_ERR_SHAPE;
    }
  }
  return QSGW_OK;
}

}  // namespace

namespace {

// Device ordinal, SM count and compute capability of the current device (cached per device; cheap attribute
// queries instead of cudaGetDeviceProperties).
struct DevInfo { int dev = -1, n_sm = 0, cc_major = 0; };
cudaError_t current_device(DevInfo* out) {
  static std::mutex mu;
  static DevInfo cache[qsgw::kMaxDevices];
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  std::lock_guard<std::mutex> lock(mu);
  if (dev >= 0 && dev < qsgw::kMaxDevices && cache[dev].dev == dev) { *out = cache[dev]; return cudaSuccess; }
  DevInfo d;
  d.dev = dev;
  e = cudaDeviceGetAttribute(&d.n_sm, cudaDevAttrMultiProcessorCount, dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&d.cc_major, cudaDevAttrComputeCapabilityMajor, dev);
  if (e != cudaSuccess) return e;
  if (dev >= 0 && dev < qsgw::kMaxDevices) cache[dev] = d;
  *out = d;
  return cudaSuccess;
}

// Kernel attributes of wc_kernels.cu, set once per device.
cudaError_t wc_configure_device(int dev) {
  static std::mutex mu;
  static bool done[qsgw::kMaxDevices] = {};
  std::lock_guard<std::mutex> lock(mu);
  if (dev >= 0 && dev < qsgw::kMaxDevices && done[dev]) return cudaSuccess;
  cudaError_t e = qsgw::wc_configure();
  if (e == cudaSuccess) e = qsgw::eig_configure();
  if (e == cudaSuccess && dev >= 0 && dev < qsgw::kMaxDevices) done[dev] = true;
  return e;
}

// Stream-ordered workspace of the context-free entry points (W^c, basis rotation: ~3 GB at cfg-4 size) comes from a
// private memory pool per device that keeps its memory between calls: the default pool hands it back to the driver
// at every synchronisation and the next cudaMallocAsync then costs ~17 ms with the GPU idle (measured, cfg 4).
// Option "trim_workspace" returns the memory to the driver.
cudaMemPool_t g_work_pool[qsgw::kMaxDevices] = {};
std::mutex g_work_pool_mu;
cudaError_t work_alloc(int dev, void** p, size_t bytes, cudaStream_t st) {
  cudaMemPool_t pool = nullptr;
  if (dev >= 0 && dev < qsgw::kMaxDevices) {
    std::lock_guard<std::mutex> lock(g_work_pool_mu);
    if (!g_work_pool[dev]) {
      cudaMemPoolProps props;
      memset(&props, 0, sizeof(props));
      props.allocType = cudaMemAllocationTypePinned;
      props.handleTypes = cudaMemHandleTypeNone;
      props.location.type = cudaMemLocationTypeDevice;
      props.location.id = dev;
      cudaMemPool_t np = nullptr;
      if (cudaMemPoolCreate(&np, &props) == cudaSuccess) {
        unsigned long long keep = ~0ull;
        cudaMemPoolSetAttribute(np, cudaMemPoolAttrReleaseThreshold, &keep);
        g_work_pool[dev] = np;
      } else {
        cudaGetLastError();
      }
    }
    pool = g_work_pool[dev];
  }
  return pool ? cudaMallocFromPoolAsync(p, bytes, pool, st) : cudaMallocAsync(p, bytes, st);
}

int g_eig_blocked = 1;  // option "eig_blocked": qsgw_coulomb_eigenbasis with block rounds (1) | element-wise rounds (0)
int g_wc_graph = 1;     // option "wc_graph": 0 plain launches | 1 graph with fallback | 2 graph or fail

// Internal streams (one per device) and in-flight executable graphs of qsgw_wc_from_chi0 (destroyed once their
// event completed).
struct WcGraphs {
  std::mutex mu;
  cudaStream_t stream[qsgw::kMaxDevices] = {};
  struct Item { cudaGraphExec_t exec; cudaEvent_t done; };
  std::vector<Item> pending;
  void sweep() {
    size_t keep = 0;
    for (size_t i = 0; i < pending.size(); ++i) {
      if (cudaEventQuery(pending[i].done) == cudaSuccess) {
        cudaGraphExecDestroy(pending[i].exec);
        cudaEventDestroy(pending[i].done);
      } else {
        cudaGetLastError();
        pending[keep++] = pending[i];
      }
    }
    pending.resize(keep);
  }
};
WcGraphs& wc_graphs() {
  static WcGraphs* g = new WcGraphs();   // never destroyed: no CUDA calls at process exit
  return *g;
}

}  // namespace

extern "C" {

const char* qsgw_version(void) { return "qsgw-chi0 0.2 (sm_100a)"; }
const char* qsgw_last_create_error(void) { return g_create_error.c_str(); }
const char* qsgw_last_error(const qsgw_ctx* ctx) { return ctx ? ctx->err.c_str() : "ctx is NULL"; }
int64_t qsgw_kernel_launches(const qsgw_ctx* ctx) { return ctx ? ctx->launches : 0; }
int64_t qsgw_pairs_accumulated(const qsgw_ctx* ctx) { return ctx ? ctx->pairs : 0; }
size_t qsgw_device_bytes(const qsgw_ctx* ctx) { return ctx ? ctx->device_bytes : 0; }
int32_t qsgw_n_m(const qsgw_ctx* ctx) { return ctx ? ctx->n_m : 0; }
int32_t qsgw_n_b(const qsgw_ctx* ctx) { return ctx ? ctx->n_b : 0; }

int32_t qsgw_probe_peak(int32_t kind, double* out_tflops, double* out_ms) {
  g_create_error.clear();
  if (!out_tflops) { g_create_error = "out_tflops is NULL"; return QSGW_ERR_INVALID_ARG; }
  if (kind < QSGW_PEAK_FP64_MMA || kind > QSGW_PEAK_F16_MMA) { g_create_error = "bad peak kind"; return QSGW_ERR_INVALID_ARG; }
  cudaStream_t st = nullptr;
  cudaError_t e = cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking);
  if (e != cudaSuccess) { cudaGetLastError(); g_create_error = cudaGetErrorString(e); return QSGW_ERR_UNSUPPORTED; }
  if (kind == QSGW_PEAK_FP64_MMA) e = qsgw::probe_fp64_mma(st, out_tflops, out_ms);
  else if (kind == QSGW_PEAK_TF32_MMA) e = qsgw::probe_tf32_mma(st, out_tflops, out_ms);
  else e = qsgw::probe_f16_mma(st, out_tflops, out_ms);
  cudaStreamDestroy(st);
  if (e != cudaSuccess) { cudaGetLastError(); g_create_error = cudaGetErrorString(e); return e == cudaErrorNotSupported ? QSGW_ERR_UNSUPPORTED : QSGW_ERR_CUDA; }
  return QSGW_OK;
}

int32_t qsgw_set_stage_timing(qsgw_ctx* ctx, int32_t enable) {
  if (!ctx) return QSGW_ERR_INVALID_ARG;
  ev_harvest(ctx, true);
  for (int s = 0; s < QSGW_N_STAGES; ++s) {
    ctx->stage_ms[s] = 0.0;
    ctx->stage_n[s] = 0;
  }
  ctx->timing = enable != 0;
  return QSGW_OK;
}

int32_t qsgw_stage_time_ms(qsgw_ctx* ctx, int32_t stage, double* out_ms, int64_t* out_launches) {
  if (!ctx) return QSGW_ERR_INVALID_ARG;
  if (stage < 0 || stage >= QSGW_N_STAGES) return ctx->fail(QSGW_ERR_INVALID_ARG, "bad stage %d", stage);
  ev_harvest(ctx, true);
  if (out_ms) *out_ms = ctx->stage_ms[stage];
  if (out_launches) *out_launches = ctx->stage_n[stage];
  return QSGW_OK;
}

static cudaError_t upload_ctl(qsgw_ctx* c) {
  qsgw::MixedCtl h;
  memset(&h, 0, sizeof(h));
  h.peff_min = 3.0e38f;
  h.peff_min_seen = 3.0e38f;
  h.mode = c->fp8_mode;
  h.use_fp8 = c->fp8_mode == 1;
  h.thr_pairs = (float)(c->fp8_thr * c->n_m);
  // pageable source: the copy is staged before the call returns
  return cudaMemcpyAsync(c->d_ctl, &h, sizeof(h), cudaMemcpyHostToDevice, c->stream);
}

int32_t qsgw_create(const qsgw_desc* desc, void* cuda_stream, qsgw_ctx** out) {
  g_create_error.clear();
  if (!out) return create_fail(nullptr, QSGW_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  std::string why;
  int rc = validate_desc(desc, why);
  if (rc != QSGW_OK) return create_fail(nullptr, rc, why);
  DevInfo di;
  cudaError_t e = current_device(&di);
  if (e != cudaSuccess) { cudaGetLastError(); return create_fail(nullptr, QSGW_ERR_UNSUPPORTED, std::string("no CUDA device: ") + cudaGetErrorString(e)); }
  if (di.cc_major != 10) return create_fail(nullptr, QSGW_ERR_UNSUPPORTED, "kernels are built for sm_100a only");

  qsgw_ctx* c = new (std::nothrow) qsgw_ctx();
  if (!c) return create_fail(nullptr, QSGW_ERR_ALLOC, "host allocation failed");
  c->stream = static_cast<cudaStream_t>(cuda_stream);
  c->device = di.dev;
  c->n_sm = di.n_sm;
  c->n_sites = desc->n_sites;
  c->n_freq = desc->n_freq;
  c->n_k = desc->n_k;
  c->max_n_o = desc->max_n_o;
  c->max_n_u = desc->max_n_u;
  c->precision = desc->precision;
  c->occ_tol = desc->occ_tol < 0 ? 1e-12 : desc->occ_tol;
  c->orb.assign(desc->h_orb_per_site, desc->h_orb_per_site + desc->n_sites);
  c->pb.assign(desc->h_pb_per_site, desc->h_pb_per_site + desc->n_sites);
  c->omega.assign(desc->h_omega, desc->h_omega + desc->n_freq);

  std::vector<int> orb_off(c->n_sites + 1, 0), pb_off(c->n_sites + 1, 0);
  std::vector<long long> p_off(c->n_sites, 0);
  long long pe = 0;
  for (int s = 0; s < c->n_sites; ++s) {
    orb_off[s + 1] = orb_off[s] + c->orb[s];
    pb_off[s + 1] = pb_off[s] + c->pb[s];
    p_off[s] = pe;
    pe += (long long)c->pb[s] * c->orb[s] * c->orb[s];
    if (c->orb[s] > c->b_max) c->b_max = c->orb[s];
  }
  c->n_b = orb_off[c->n_sites];
  c->n_m = pb_off[c->n_sites];
  c->p_elems = pe;
  std::vector<int> pb_site(c->n_m);
  for (int s = 0; s < c->n_sites; ++s)
    for (int I = pb_off[s]; I < pb_off[s + 1]; ++I) pb_site[I] = s;

  c->ncg = (c->n_m + qsgw::kCG - 1) / qsgw::kCG;
  {   // contraction length of the DMMA stage (a) kernel: column groups may straddle sites
    int kt = 0;
    for (int cg = 0; cg < c->ncg; ++cg) {
      int sum = 0, last = -1;
      for (int I = cg * qsgw::kCG; I < c->n_m && I < (cg + 1) * qsgw::kCG; ++I)
        if (pb_site[I] != last) { last = pb_site[I]; sum += (c->orb[last] + 3) & ~3; }
      if (sum > kt) kt = sum;
    }
    if (qsgw::zmel_dmma_smem_bytes(c->b_max, kt) <= 200 * 1024) c->zmel_kt_avail = kt;
    c->zmel_kt = c->zmel_kt_avail;
  }
  const bool mixed = c->precision != QSGW_PREC_FP64;
  c->f16 = mixed;
  const int tile_edge = mixed ? qsgw::kTileMx : qsgw::kTile;
  c->n_m_pad = (int)round_up(c->n_m, tile_edge);
  const long long max_pairs = (long long)c->max_n_o * c->max_n_u;
  // Workspace = room for `mult` padded band batches (32 Ki .. 256 Ki pairs): small batches (few bands, many k-points)
  // are staged back to back and stage (b) runs once per full workspace instead of once per batch.
  c->batch_pad = round_up(max_pairs, qsgw::kPairAlign);
  // at least 32 Ki pairs; for small N_M as many as 1.5 GB of FP64 workspace hold (up to 256 Ki): fewer, longer launches
  long long target = (long long)(1.5e9 / ((double)2 * c->ncg * qsgw::kCG * sizeof(double)));
  target = target < 32768 ? 32768 : (target > 262144 ? 262144 : target);
  long long mult = (target + c->batch_pad - 1) / c->batch_pad;
  {   // ... but beyond 32 Ki pairs never more than the declared k-points need
    const long long mult32k = (32768 + c->batch_pad - 1) / c->batch_pad;
    const long long cap = mult32k > c->n_k ? mult32k : c->n_k;
    if (mult > cap) mult = cap;
  }
  size_t z64_bytes = 0, zhl_bytes = 0, z_bytes = 0;
  for (;; --mult) {
    c->kpad = c->batch_pad * mult;
    z64_bytes = (size_t)2 * c->ncg * c->kpad * qsgw::kCG * sizeof(double);
    zhl_bytes = c->f16 ? (size_t)2 * c->n_m_pad * c->kpad * 2 * sizeof(uint16_t) : 0;
    z_bytes = z64_bytes + 2 * zhl_bytes;
    if (mult == 1 || desc->workspace_bytes == 0 || z_bytes <= desc->workspace_bytes) break;
  }
  c->stage_cap = c->kpad;
  if (desc->workspace_bytes != 0 && z_bytes > desc->workspace_bytes) {
    char buf[256];
    snprintf(buf, sizeof(buf), "z workspace for %d x %d band pairs needs %zu bytes > workspace_bytes cap %zu; "
             "pass smaller max_n_o/max_n_u", c->max_n_o, c->max_n_u, z_bytes, desc->workspace_bytes);
    return create_fail(c, QSGW_ERR_ALLOC, buf);
  }
  const int nt = c->n_m_pad / tile_edge;
  // Work list of the stage (b) kernels.  Mixed mode: the upper 128 x 128 tiles.  FP64 mode (chi0_f64_kernels.cu): full
  // 64 x 64 tiles off the diagonal; 64 x 32 pieces for the last tile column when its last 32 columns are padding (cfg 2:
  // N_M = 600 = 9 x 64 + 24; cfg 4: 2400 = 37 x 64 + 32) and for the right half of every diagonal tile; 32 x 32 pieces for
  // the upper-left block of every diagonal tile (a diagonal tile costs 3/4 of a full one).
  const int rem = c->n_m % tile_edge;
  const bool narrow_last = !mixed && rem >= 1 && rem <= 32;
  std::vector<int4> tiles, tiles_half, tiles_quarter;
  for (int tj = 0; tj < nt; ++tj)
    for (int ti = 0; ti <= tj; ++ti) {
      const bool last_narrow = narrow_last && tj == nt - 1;
      if (mixed) {
        tiles.push_back(make_int4(ti, tj, 0, 0));
      } else if (ti == tj) {
        tiles_quarter.push_back(make_int4(ti, tj, 0, 0));
        if (!last_narrow) tiles_half.push_back(make_int4(ti, tj, 2, 0));
      } else {
        (last_narrow ? tiles_half : tiles).push_back(make_int4(ti, tj, 0, 0));
      }
    }
  c->n_tiles = (int)tiles.size();
  c->n_tiles_half = (int)tiles_half.size();
  c->n_tiles_quarter = (int)tiles_quarter.size();
  tiles.insert(tiles.end(), tiles_half.begin(), tiles_half.end());         // one device array: full, half, quarter
  tiles.insert(tiles.end(), tiles_quarter.begin(), tiles_quarter.end());

#define QSGW_TRY_ALLOC(expr)                                                                     \
  do {                                                                                           \
    cudaError_t _e = (expr);                                                                     \
    if (_e != cudaSuccess) {                                                                     \
      cudaGetLastError();                                                                        \
      return create_fail(c, QSGW_ERR_ALLOC, std::string("device allocation failed: ") + cudaGetErrorString(_e)); \
    }                                                                                            \
  } while (0)
  const size_t acc_elems = (size_t)c->n_freq * c->n_m_pad * c->n_m_pad;
  QSGW_TRY_ALLOC(dev_alloc(c, &c->d_pb_site, (size_t)c->n_m));
  QSGW_TRY_ALLOC(dev_alloc(c, &c->d_pb_off, (size_t)c->n_sites + 1));
  QSGW_TRY_ALLOC(dev_alloc(c, &c->d_orb_off, (size_t)c->n_sites + 1));
  QSGW_TRY_ALLOC(dev_alloc(c, &c->d_p_off, (size_t)c->n_sites));
  QSGW_TRY_ALLOC(dev_alloc(c, &c->d_tiles, tiles.size()));
  QSGW_TRY_ALLOC(dev_alloc(c, &c->d_omega, (size_t)c->n_freq));
  QSGW_TRY_ALLOC(dev_alloc(c, &c->d_P, (size_t)c->p_elems));
  QSGW_TRY_ALLOC(dev_alloc(c, &c->d_zws, z64_bytes / sizeof(double)));
  if (c->f16) {
    QSGW_TRY_ALLOC(dev_alloc(c, &c->d_wtab32, (size_t)c->n_freq * c->kpad));
    QSGW_TRY_ALLOC(dev_alloc(c, reinterpret_cast<unsigned char**>(&c->d_zhl), zhl_bytes));
    QSGW_TRY_ALLOC(dev_alloc(c, reinterpret_cast<unsigned char**>(&c->d_zhb8), zhl_bytes));
    QSGW_TRY_ALLOC(dev_alloc(c, &c->d_wscale, (size_t)c->n_freq));
    QSGW_TRY_ALLOC(dev_alloc(c, &c->d_zmax, (size_t)(c->kpad / qsgw::kPairAlign + 1)));   // one scale per staged batch
    QSGW_TRY_ALLOC(dev_alloc(c, &c->d_ctl, (size_t)1));
    QSGW_TRY_ALLOC(dev_alloc(c, &c->d_pmax, (size_t)c->n_sites));
    c->zmel_direct = qsgw::zmel_umma_supported(c->b_max) ? 1 : 0;
  }
  QSGW_TRY_ALLOC(dev_alloc(c, &c->d_wtab, (size_t)c->n_freq * c->kpad));
  QSGW_TRY_ALLOC(dev_alloc(c, &c->d_live, (size_t)(c->kpad / qsgw::kPairStage + 1)));
  QSGW_TRY_ALLOC(dev_alloc(c, &c->d_n_live, (size_t)1));
  QSGW_TRY_ALLOC(dev_alloc(c, &c->d_stage_flags, (size_t)(c->kpad / qsgw::kPairStage + 1)));
  QSGW_TRY_ALLOC(dev_alloc(c, &c->d_acc_re, acc_elems));
  QSGW_TRY_ALLOC(dev_alloc(c, &c->d_acc_im, acc_elems));
#undef QSGW_TRY_ALLOC

#define QSGW_TRY_CUDA(expr)                                                                      \
  do {                                                                                           \
    cudaError_t _e = (expr);                                                                     \
    if (_e != cudaSuccess) return create_fail(c, QSGW_ERR_CUDA, std::string(#expr ": ") + cudaGetErrorString(_e)); \
  } while (0)
  cudaStream_t st = c->stream;
  // small tables: synchronous copies from pageable host memory are fine at create time
  QSGW_TRY_CUDA(cudaMemcpyAsync(c->d_pb_site, pb_site.data(), sizeof(int) * c->n_m, cudaMemcpyHostToDevice, st));
  QSGW_TRY_CUDA(cudaMemcpyAsync(c->d_pb_off, pb_off.data(), sizeof(int) * (c->n_sites + 1), cudaMemcpyHostToDevice, st));
  QSGW_TRY_CUDA(cudaMemcpyAsync(c->d_orb_off, orb_off.data(), sizeof(int) * (c->n_sites + 1), cudaMemcpyHostToDevice, st));
  QSGW_TRY_CUDA(cudaMemcpyAsync(c->d_p_off, p_off.data(), sizeof(long long) * c->n_sites, cudaMemcpyHostToDevice, st));
  QSGW_TRY_CUDA(cudaMemcpyAsync(c->d_tiles, tiles.data(), sizeof(int4) * tiles.size(), cudaMemcpyHostToDevice, st));
  QSGW_TRY_CUDA(cudaMemcpyAsync(c->d_omega, c->omega.data(), sizeof(double) * c->n_freq, cudaMemcpyHostToDevice, st));
  QSGW_TRY_CUDA(cudaMemsetAsync(c->d_zws, 0, z64_bytes, st));
  if (c->f16) {
    QSGW_TRY_CUDA(cudaMemsetAsync(c->d_wtab32, 0, sizeof(float) * c->n_freq * c->kpad, st));
    QSGW_TRY_CUDA(cudaMemsetAsync(c->d_zhl, 0, zhl_bytes, st));
    QSGW_TRY_CUDA(cudaMemsetAsync(c->d_zhb8, 0, zhl_bytes, st));
    QSGW_TRY_CUDA(cudaMemsetAsync(c->d_wscale, 0, sizeof(double) * c->n_freq, st));
    QSGW_TRY_CUDA(cudaMemsetAsync(c->d_zmax, 0, sizeof(float) * (c->kpad / qsgw::kPairAlign + 1), st));
    QSGW_TRY_CUDA(upload_ctl(c));
    QSGW_TRY_CUDA(qsgw::chi0_f16_configure());
  }
  QSGW_TRY_CUDA(cudaMemsetAsync(c->d_wtab, 0, sizeof(double) * c->n_freq * c->kpad, st));
  QSGW_TRY_CUDA(cudaMemsetAsync(c->d_acc_re, 0, sizeof(double) * acc_elems, st));
  QSGW_TRY_CUDA(cudaMemsetAsync(c->d_acc_im, 0, sizeof(double) * acc_elems, st));
  QSGW_TRY_CUDA(cudaStreamSynchronize(st));   // host vectors above go out of scope
  QSGW_TRY_CUDA(qsgw::chi0_f64_configure());
#undef QSGW_TRY_CUDA

  EncodeTiledFn enc = get_encode_tiled();
  if (!enc) return create_fail(c, QSGW_ERR_UNSUPPORTED, "cuTensorMapEncodeTiled not available from the driver");
  {
    const cuuint64_t gdim[4] = {(cuuint64_t)qsgw::kCG, (cuuint64_t)c->kpad, (cuuint64_t)c->ncg, 2};
    const cuuint64_t gstr[3] = {(cuuint64_t)qsgw::kCG * 8, (cuuint64_t)c->kpad * qsgw::kCG * 8,
                                (cuuint64_t)c->ncg * c->kpad * qsgw::kCG * 8};
    const cuuint32_t box[4] = {(cuuint32_t)qsgw::kCG, (cuuint32_t)qsgw::kChi0F64KP3M, 4, 2};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = enc(&c->tmap_z, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, c->d_zws, gdim, gstr, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
      char buf[128];
      snprintf(buf, sizeof(buf), "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
      return create_fail(c, QSGW_ERR_CUDA, buf);
    }
  }
  if (c->f16) {
    const cuuint64_t gdim[3] = {(cuuint64_t)c->kpad * 2, (cuuint64_t)c->n_m_pad, 2};
    const cuuint64_t gstr[2] = {(cuuint64_t)c->kpad * 4, (cuuint64_t)c->n_m_pad * c->kpad * 4};
    const cuuint32_t box[3] = {64, 64, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = enc(&c->tmap_h, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 3, c->d_zhl, gdim, gstr, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r == CUDA_SUCCESS) {
      const cuuint64_t gdim8[3] = {(cuuint64_t)c->kpad * 4, (cuuint64_t)c->n_m_pad, 2};
      const cuuint32_t box8[3] = {128, 64, 1};
      r = enc(&c->tmap_hb8, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, c->d_zhb8, gdim8, gstr, box8, estr,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    }
    if (r != CUDA_SUCCESS) {
      char buf[128];
      snprintf(buf, sizeof(buf), "cuTensorMapEncodeTiled (mixed, hl16 / hb8 planes) failed with CUresult %d", (int)r);
      return create_fail(c, QSGW_ERR_CUDA, buf);
    }
  }
  c->state = ST_CREATED;
  *out = c;
  return QSGW_OK;
}

void qsgw_destroy(qsgw_ctx* ctx) {
  if (!ctx) return;
  cudaStreamSynchronize(ctx->stream);
  if (ctx->hr.cp) cudaStreamSynchronize(ctx->hr.cp);
  free_all(ctx);
  delete ctx;
}

static int flush_pending(qsgw_ctx* ctx);

int32_t qsgw_set_option(qsgw_ctx* ctx, const char* key, int64_t value) {
  if (!key) return ctx ? ctx->fail(QSGW_ERR_INVALID_ARG, "key is NULL") : QSGW_ERR_INVALID_ARG;
  const std::string k(key);
  if (!ctx) {
    g_create_error.clear();
    if (k == "wc_graph" && value >= 0 && value <= 2) { g_wc_graph = (int)value; return QSGW_OK; }
    if (k == "eig_blocked" && (value == 0 || value == 1)) { g_eig_blocked = (int)value; return QSGW_OK; }
    if (k == "trim_workspace") {     // hand the cached W^c / rotation workspace of every device back to the driver
      std::lock_guard<std::mutex> lock(g_work_pool_mu);
      for (int d = 0; d < qsgw::kMaxDevices; ++d)
        if (g_work_pool[d]) cudaMemPoolTrimTo(g_work_pool[d], (size_t)(value > 0 ? value : 0));
      return QSGW_OK;
    }
    g_create_error = "unknown process-wide option or value out of range: " + k;
    return QSGW_ERR_INVALID_ARG;
  }
  if (ctx->fill != 0) return ctx->fail(QSGW_ERR_STATE, "options can be set only while no band batch is staged");
  if (k == "stage_batches" && value >= 1) {
    const long long cap = ctx->batch_pad * (value > (1LL << 30) ? (1LL << 30) : value);
    ctx->stage_cap = cap < ctx->kpad ? cap : ctx->kpad;
  } else if (k == "skip_dead_stages" && value >= 0 && value <= 2) {
    ctx->skip_dead = (int)value;
  } else if (k == "zmel_dmma" && (value == 0 || value == 1)) {
    if (value == 1 && ctx->zmel_kt_avail == 0)
      return ctx->fail(QSGW_ERR_UNSUPPORTED, "the tensor-pipe stage (a) kernel does not fit this site structure");
    ctx->zmel_kt = value ? ctx->zmel_kt_avail : 0;
  } else if (k == "mixed_fp8" && value >= 0 && value <= 2 && ctx->f16) {
    ctx->fp8_mode = (int)value;
    if (upload_ctl(ctx) != cudaSuccess) return ctx->fail(QSGW_ERR_CUDA, "upload of the mixed-mode control block failed");
  } else if (k == "mixed_fp8_threshold_x100" && value >= 0 && ctx->f16) {
    ctx->fp8_thr = 0.01 * (double)value;
    if (upload_ctl(ctx) != cudaSuccess) return ctx->fail(QSGW_ERR_CUDA, "upload of the mixed-mode control block failed");
  } else if (k == "mixed_window" && value >= 1 && value <= 64 && ctx->f16) {
    ctx->win = (int)value;
  } else if (k == "zmel_direct" && value >= 0 && value <= 2 && ctx->f16) {
    if (value != 0 && !qsgw::zmel_umma_supported(ctx->b_max))
      return ctx->fail(QSGW_ERR_UNSUPPORTED, "the tcgen05 stage (a) kernel holds at most 32 orbitals per site");
    ctx->zmel_direct = (int)value;
  } else if (k == "mixed_pair" && (value == 0 || value == 1) && ctx->f16) {
    ctx->mixed_pair = (int)value;
  } else if (k == "sigc_f64" && (value == 0 || value == 1) && ctx->f16) {
    ctx->sigc_f64 = value != 0;
  } else if (k == "sigc_fp8" && (value == 0 || value == 1) && ctx->f16) {
    ctx->sigc_fp8 = (int)value;
  } else if (k == "e2e_groups" && value >= 1 && value <= 4) {
    ctx->e2e_groups = (int)value;
  } else {
    return ctx->fail(QSGW_ERR_INVALID_ARG, "unknown option, value out of range, or option of the other precision mode: %s", key);
  }
  ctx->err.clear();
  return QSGW_OK;
}

int32_t qsgw_mixed_stats(qsgw_ctx* ctx, int64_t* out_launches, int64_t* out_launches_fp8,
                         double* out_min_effective_pairs) {
  if (!ctx) return QSGW_ERR_INVALID_ARG;
  if (!ctx->f16) return ctx->fail(QSGW_ERR_STATE, "qsgw_mixed_stats: the context is in FP64 mode");
  qsgw::MixedCtl h;
  cudaError_t e = cudaMemcpyAsync(&h, ctx->d_ctl, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
  if (e != cudaSuccess) return ctx->cuda_fail(e, "read of the mixed-mode control block");
  if (out_launches) *out_launches = (int64_t)h.n_flush;
  if (out_launches_fp8) *out_launches_fp8 = (int64_t)h.n_flush_fp8;
  if (out_min_effective_pairs) *out_min_effective_pairs = (double)h.peff_min_seen;
  return QSGW_OK;
}

int32_t qsgw_sync(qsgw_ctx* ctx) {
  if (!ctx) return QSGW_ERR_INVALID_ARG;
  int rc = flush_pending(ctx);     // staged band batches are accumulated before the wait
  if (rc != QSGW_OK) return rc;
  cudaError_t e = cudaStreamSynchronize(ctx->stream);
  if (e != cudaSuccess) return ctx->cuda_fail(e, "cudaStreamSynchronize");
  return QSGW_OK;
}

static qsgw::SiteTables site_tables(const qsgw_ctx* ctx);

int32_t qsgw_set_product_tensor(qsgw_ctx* ctx, const void* d_P) {
  if (!ctx) return QSGW_ERR_INVALID_ARG;
  if (!d_P) return ctx->fail(QSGW_ERR_INVALID_ARG, "d_P is NULL");
  cudaError_t e = cudaMemcpyAsync(ctx->d_P, d_P, sizeof(double2) * ctx->p_elems, cudaMemcpyDeviceToDevice, ctx->stream);
  if (e == cudaSuccess && ctx->d_pmax) e = qsgw::launch_zmel_pnorm(site_tables(ctx), ctx->d_P, ctx->d_pmax, ctx->stream);
  if (e != cudaSuccess) return ctx->cuda_fail(e, "copy of P");
  if (ctx->state == ST_CREATED) ctx->state = ST_READY;
  ctx->err.clear();
  return QSGW_OK;
}

int32_t qsgw_reset(qsgw_ctx* ctx) {
  if (!ctx) return QSGW_ERR_INVALID_ARG;
  const size_t acc_elems = (size_t)ctx->n_freq * ctx->n_m_pad * ctx->n_m_pad;
  cudaError_t e = cudaMemsetAsync(ctx->d_acc_re, 0, sizeof(double) * acc_elems, ctx->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(ctx->d_acc_im, 0, sizeof(double) * acc_elems, ctx->stream);
  if (e == cudaSuccess && ctx->f16) e = upload_ctl(ctx);
  if (e != cudaSuccess) return ctx->cuda_fail(e, "reset");
  if (ctx->state != ST_CREATED) ctx->state = ST_READY;
  ctx->pairs = 0;
  ctx->fill = 0;                   // staged, not yet accumulated batches are dropped with the accumulator
  ctx->zslot = 0;
  ctx->z_off = 0;
  ctx->z_zi = 0;
  ctx->err.clear();
  return QSGW_OK;
}

// hl16 / hb8 rows of the staging slot at pair offset `off` (128 bytes per product function and 32 pairs)
static void* hl_slot(void* base, long long off) {
  return base ? static_cast<unsigned char*>(base) + (off / qsgw::kPairStage) * 128 : nullptr;
}
static int stage_slot(qsgw_ctx* ctx, long long n_pairs, long long* off);

static int check_batch(qsgw_ctx* ctx, int n_o, int n_u) {
  if (n_o < 1 || n_u < 1) return ctx->fail(QSGW_ERR_SHAPE, "band batch must be non-empty (n_o=%d, n_u=%d)", n_o, n_u);
  if (n_o > ctx->max_n_o || n_u > ctx->max_n_u)
    return ctx->fail(QSGW_ERR_SHAPE, "band batch %d x %d exceeds the declared maximum %d x %d", n_o, n_u,
                     ctx->max_n_o, ctx->max_n_u);
  return QSGW_OK;
}

static qsgw::SiteTables site_tables(const qsgw_ctx* ctx) {
  qsgw::SiteTables st;
  st.n_sites = ctx->n_sites;
  st.n_b = ctx->n_b;
  st.n_m = ctx->n_m;
  st.b_max = ctx->b_max;
  st.d_pb_site = ctx->d_pb_site;
  st.d_pb_off = ctx->d_pb_off;
  st.d_orb_off = ctx->d_orb_off;
  st.d_p_off = ctx->d_p_off;
  return st;
}

// Stage (a) for `n_batch` k-points of equal band batch in ONE launch (grid.z = k-point): k-point b reads
// Ck + b*ck_bs, Ckq + b*ckq_bs and fills the workspace slot at pair offset off + b*n_pad with batch-scale index
// zi + b.  The caller has made room ([off, off + n_batch*n_pad) <= kpad).
static int build_batches(qsgw_ctx* ctx, const double2* Ck, long long ld_k, long long ck_bs, const double2* Ckq,
                         long long ld_kq, long long ckq_bs, int n_begin, int n_o, int np_begin, int n_u, int n_batch,
                         long long off, long long n_pad, int zi) {
  qsgw::ZmelArgs a;
  a.st = site_tables(ctx);
  a.P = ctx->d_P;
  a.Ck = Ck;
  a.ld_k = ld_k;
  a.Ckq = Ckq;
  a.ld_kq = ld_kq;
  a.n_begin = n_begin;
  a.n_o = n_o;
  a.np_begin = np_begin;
  a.n_u = n_u;
  a.zws = ctx->d_zws + off * qsgw::kCG;
  a.kpad = ctx->kpad;
  a.ncg = ctx->ncg;
  a.kt = ctx->zmel_kt;
  a.n_sm = ctx->n_sm;
  a.n_batch = n_batch;
  a.row_map = ctx->cur_row_map;
  a.Ck_bs = ck_bs;
  a.Ckq_bs = ckq_bs;
  a.z_bs = n_pad;
  cudaError_t e;
  // small launches keep the two-kernel FP64 path: the tcgen05 path has four launches and a tensor-map encode per call;
  // so does the binned real-axis path, whose row map scatters the 64-byte runs of the epilogue (measured: 16.0 -> 19.7 ms)
  const bool direct = ctx->f16 && (ctx->zmel_direct == 2 ||
                                   (ctx->zmel_direct == 1 && !ctx->cur_row_map && (double)n_batch * n_o * n_u * ctx->n_m >= 8.0e6));
  if (direct) {   // stage (a) on tcgen05, straight into the FP16-split rows (no FP64 z, no conversion pass)
    a.zmax = ctx->d_zmax + zi;
    const size_t need_c = ((size_t)2 * ctx->n_sites + 2) * n_batch, need_a = qsgw::zmel_umma_aop_halves(ctx->n_sites, n_u, n_batch);
    e = qsgw::zmel_umma_configure();
    if (e == cudaSuccess && need_c > ctx->cnorm_cap) {
      cudaStreamSynchronize(ctx->stream);
      cudaFree(ctx->d_cnorm);
      ctx->d_cnorm = nullptr;
      ctx->cnorm_cap = 0;
      e = dev_alloc(ctx, &ctx->d_cnorm, need_c);
      if (e == cudaSuccess) ctx->cnorm_cap = need_c;
    }
    if (e == cudaSuccess && need_a > ctx->aop_cap) {
      cudaStreamSynchronize(ctx->stream);
      cudaFree(ctx->d_aop);
      ctx->d_aop = nullptr;
      ctx->aop_cap = 0;
      e = dev_alloc(ctx, &ctx->d_aop, need_a);
      if (e == cudaSuccess) ctx->aop_cap = need_a;
    }
    if (e != cudaSuccess) { cudaGetLastError(); return ctx->fail(QSGW_ERR_ALLOC, "stage (a) scratch allocation failed: %s", cudaGetErrorString(e)); }
    {
      StageScope ts(ctx, QSGW_STAGE_ZMEL);
      e = qsgw::launch_zmel_umma(a, ctx->d_pmax, ctx->d_cnorm, ctx->d_aop, hl_slot(ctx->d_zhl, off), hl_slot(ctx->d_zhb8, off),
                                 ctx->n_m_pad, round_up((long long)n_o * n_u, qsgw::kPairAlign), ctx->stream);
    }
    if (e != cudaSuccess) return ctx->cuda_fail(e, "zmel (tcgen05, FP16-split rows) kernel launch");
    ctx->launches += 4;
    return QSGW_OK;
  }
  if (ctx->f16) {
    a.zmax = ctx->d_zmax + zi;
    e = cudaMemsetAsync(a.zmax, 0, sizeof(float) * n_batch, ctx->stream);
    if (e != cudaSuccess) return ctx->cuda_fail(e, "reset of the batch maximum");
  }
  {
    StageScope ts(ctx, QSGW_STAGE_ZMEL);
    e = ctx->zmel_kt ? qsgw::launch_zmel_dmma(a, ctx->stream) : qsgw::launch_zmel_f64(a, ctx->stream);
    if (e == cudaSuccess && ctx->f16)
      e = qsgw::launch_z_to_hl16(a.zws, ctx->kpad, ctx->ncg, ctx->n_m, (long long)n_o * n_u,
                                 hl_slot(ctx->d_zhl, off), hl_slot(ctx->d_zhb8, off), ctx->n_m_pad, a.zmax, n_batch,
                                 n_pad, ctx->stream);
  }
  if (e != cudaSuccess) return ctx->cuda_fail(e, "zmel kernel launch");
  ctx->launches += ctx->f16 ? 2 : 1;
  return QSGW_OK;
}

int32_t qsgw_zmel_build(qsgw_ctx* ctx, const void* d_Ck, int64_t ld_k, const void* d_Ckq, int64_t ld_kq,
                        int32_t n_begin, int32_t n_o, int32_t np_begin, int32_t n_u, void* d_z_out) {
  if (!ctx) return QSGW_ERR_INVALID_ARG;
  if (ctx->state == ST_CREATED) return ctx->fail(QSGW_ERR_STATE, "set_product_tensor must precede zmel_build");
  if (!d_Ck || !d_Ckq) return ctx->fail(QSGW_ERR_INVALID_ARG, "d_Ck / d_Ckq is NULL");
  if (ld_k < ctx->n_b || ld_kq < ctx->n_b)
    return ctx->fail(QSGW_ERR_INVALID_ARG, "leading dimension smaller than N_b=%d", ctx->n_b);
  if (n_begin < 0 || np_begin < 0) return ctx->fail(QSGW_ERR_SHAPE, "negative band offset");
  int rc = check_batch(ctx, n_o, n_u);
  if (rc != QSGW_OK) return rc;

  long long off = 0;
  const long long n_pairs = (long long)n_o * n_u;
  rc = stage_slot(ctx, n_pairs, &off);
  if (rc != QSGW_OK) return rc;
  const int zi = ctx->zslot;
  rc = build_batches(ctx, static_cast<const double2*>(d_Ck), ld_k, 0, static_cast<const double2*>(d_Ckq), ld_kq, 0,
                     n_begin, n_o, np_begin, n_u, 1, off, round_up(n_pairs, qsgw::kPairAlign), zi);
  if (rc != QSGW_OK) return rc;
  cudaError_t e;
  if (d_z_out) {
    if (ctx->f16)
      e = qsgw::launch_z_export_hl16(hl_slot(ctx->d_zhl, off), ctx->kpad, ctx->n_m_pad, ctx->n_m, n_pairs,
                                     ctx->d_zmax + zi, static_cast<double2*>(d_z_out), ctx->stream);
    else
      e = qsgw::launch_z_export(ctx->d_zws + off * qsgw::kCG, ctx->kpad, ctx->ncg, ctx->n_m, n_pairs,
                                static_cast<double2*>(d_z_out), ctx->stream);
    if (e != cudaSuccess) return ctx->cuda_fail(e, "z export kernel launch");
    ctx->launches += 1;
  }
  ctx->last_n_o = n_o;
  ctx->last_n_u = n_u;
  ctx->z_off = off;
  ctx->z_zi = zi;
  ctx->state = ST_Z_BUILT;
  ctx->err.clear();
  return QSGW_OK;
}

// Stage (b) over the staged pairs [0, fill): one launch for all band batches accumulated since the last flush.
// (frequencies j0 .. j0+nj-1; `first`/`last` mark the first/last frequency group of one flush: the host-buffer
// driver flushes the last workspace group by group so that the device-to-host copy overlaps the kernels)
static int flush_range(qsgw_ctx* ctx, int j0, int nj, bool first, bool last) {
  if (ctx->fill == 0) return QSGW_OK;
  const long long n_pad = ctx->fill;
  if (last) { ctx->fill = 0; ctx->zslot = 0; }
  cudaError_t e;
  // metals: whole bands fail the occupation filter, their stages carry no weight at any frequency and are skipped
  const bool skip = !ctx->flush_ranges &&
                    (ctx->skip_dead == 2 || (ctx->skip_dead == 1 && (double)n_pad * ctx->n_m >= 4.0e6));
  if (skip && first) {
    StageScope ts(ctx, QSGW_STAGE_WEIGHTS);
    e = qsgw::launch_stage_compaction(ctx->d_wtab, ctx->kpad, n_pad, ctx->n_freq, ctx->d_stage_flags, ctx->d_live,
                                      ctx->d_n_live, ctx->stream);
    if (e != cudaSuccess) return ctx->cuda_fail(e, "stage compaction kernel launch");
    ctx->launches += 2;
  }
  if (ctx->f16) {
    if (first) {
      StageScope ts(ctx, QSGW_STAGE_WEIGHTS);
      e = qsgw::launch_weights_scale_hl16(ctx->d_wtab, ctx->d_wtab32, ctx->d_wscale, ctx->kpad, n_pad, ctx->n_freq,
                                          ctx->d_ctl, ctx->flush_zfold, ctx->stream);
      if (e != cudaSuccess) return ctx->cuda_fail(e, "weight scaling kernel launch");
      ctx->launches += 1;
    }
    qsgw::Chi0F16Args m;
    m.tmap = ctx->tmap_h;
    m.tmap_b = ctx->tmap_hb8;
    m.wtab16 = reinterpret_cast<const __half*>(ctx->d_wtab32);   // same bytes per pair as an FP32 table
    m.wscale = ctx->d_wscale;
    m.win = ctx->win;
    m.pair = ctx->mixed_pair;
    m.kpad = ctx->kpad;
    m.acc_re = ctx->d_acc_re;
    m.acc_im = ctx->d_acc_im;
    m.n_m_pad = ctx->n_m_pad;
    m.n_freq = nj;
    m.j0 = j0;
    m.n_stages = (int)(n_pad / qsgw::kPairStage);
    m.n_sm = ctx->n_sm;
    m.ctl = ctx->d_ctl;
    m.d_ranges = ctx->flush_ranges;
    if (skip) { m.d_live = ctx->d_live; m.d_n_live = ctx->d_n_live; }
    m.d_tiles = ctx->d_tiles;
    m.n_tiles = ctx->n_tiles;
    {
      StageScope ts(ctx, QSGW_STAGE_CHI0);
      e = qsgw::launch_chi0_f16(m, ctx->stream);
    }
    if (e != cudaSuccess) return ctx->cuda_fail(e, "chi0 (mixed, FP16 split) kernel launch");
    ctx->launches += 2;            // both product variants are launched, one of them exits at once
    return QSGW_OK;
  }
  qsgw::Chi0F64Args a;
  a.tmap_z = ctx->tmap_z;
  a.wtab = ctx->d_wtab;
  a.kpad = ctx->kpad;
  a.acc_re = ctx->d_acc_re;
  a.acc_im = ctx->d_acc_im;
  a.n_m_pad = ctx->n_m_pad;
  a.n_freq = nj;
  a.j0 = j0;
  a.n_pairs_padded = n_pad;
  a.n_sm = ctx->n_sm;
  a.d_tiles = ctx->d_tiles;
  a.n_tiles = ctx->n_tiles;
  a.n_tiles_half = ctx->n_tiles_half;
  a.n_tiles_quarter = ctx->n_tiles_quarter;
  if (skip) { a.d_live = ctx->d_live; a.d_n_live = ctx->d_n_live; }
  {
    StageScope ts(ctx, QSGW_STAGE_CHI0);
    e = qsgw::launch_chi0_f64(a, ctx->stream);
  }
  if (e != cudaSuccess) return ctx->cuda_fail(e, "chi0 kernel launch");
  ctx->launches += 1;
  return QSGW_OK;
}

static int flush_pending(qsgw_ctx* ctx) { return flush_range(ctx, 0, ctx->n_freq, true, true); }

// Slot of the next band batch in the workspace; flushes the staged batches first when it would not fit.
static int stage_slot(qsgw_ctx* ctx, long long n_pairs, long long* off) {
  const long long n_pad = round_up(n_pairs, qsgw::kPairAlign);
  if (ctx->fill + n_pad > ctx->stage_cap) {
    int rc = flush_pending(ctx);
    if (rc != QSGW_OK) return rc;
  }
  *off = ctx->fill;
  return QSGW_OK;
}

int32_t qsgw_chi0_accumulate(qsgw_ctx* ctx, const void* d_z, const double* d_eps_k, const double* d_f_k,
                             const double* d_eps_kq, const double* d_f_kq, int32_t n_o, int32_t n_u) {
  if (!ctx) return QSGW_ERR_INVALID_ARG;
  if (ctx->state == ST_CREATED) return ctx->fail(QSGW_ERR_STATE, "set_product_tensor must precede chi0_accumulate");
  if (!d_eps_k || !d_f_k || !d_eps_kq || !d_f_kq) return ctx->fail(QSGW_ERR_INVALID_ARG, "NULL energy/occupation array");
  int rc = check_batch(ctx, n_o, n_u);
  if (rc != QSGW_OK) return rc;
  const long long n_pairs = (long long)n_o * n_u;
  const long long n_pad = round_up(n_pairs, qsgw::kPairAlign);
  long long off = 0;
  int zi = 0;
  cudaError_t e = cudaSuccess;
  if (d_z) {
    rc = stage_slot(ctx, n_pairs, &off);
    if (rc != QSGW_OK) return rc;
    zi = ctx->zslot;
    float* zmax = ctx->f16 ? ctx->d_zmax + zi : nullptr;
    e = ctx->f16 ? cudaMemsetAsync(zmax, 0, sizeof(float), ctx->stream) : cudaSuccess;
    if (e == cudaSuccess)
      e = qsgw::launch_z_import(ctx->d_zws + off * qsgw::kCG, ctx->kpad, ctx->ncg, ctx->n_m, n_pairs,
                                static_cast<const double2*>(d_z), zmax, ctx->stream);
    if (e == cudaSuccess && ctx->f16) {
      e = qsgw::launch_z_to_hl16(ctx->d_zws + off * qsgw::kCG, ctx->kpad, ctx->ncg, ctx->n_m, n_pairs,
                                 hl_slot(ctx->d_zhl, off), hl_slot(ctx->d_zhb8, off), ctx->n_m_pad, zmax, 1, n_pad,
                                 ctx->stream);
      ctx->launches += 1;
    }
    if (e != cudaSuccess) return ctx->cuda_fail(e, "z import kernel launch");
    ctx->launches += 1;
    ctx->last_n_o = n_o;
    ctx->last_n_u = n_u;
  } else {
    if (ctx->state != ST_Z_BUILT) return ctx->fail(QSGW_ERR_STATE, "no z batch: call zmel_build first or pass d_z");
    if (n_o != ctx->last_n_o || n_u != ctx->last_n_u)
      return ctx->fail(QSGW_ERR_SHAPE, "batch %d x %d differs from the last zmel_build (%d x %d)", n_o, n_u,
                       ctx->last_n_o, ctx->last_n_u);
    // The batch sits where zmel_build wrote it.  A qsgw_sync / qsgw_chi0_finalize in between has flushed and
    // released the slots below it: their weights are zeroed so that the rows [0, z_off) of this flush contribute
    // exactly nothing (the z rows there are a stale, already accumulated batch).
    off = ctx->z_off;
    zi = ctx->z_zi;
    if (off != ctx->fill) {
      e = cudaMemset2DAsync(ctx->d_wtab, sizeof(double) * ctx->kpad, 0, sizeof(double) * off, ctx->n_freq, ctx->stream);
      if (e != cudaSuccess) return ctx->cuda_fail(e, "clearing the weights of released workspace slots");
    }
  }
  {
    StageScope ts(ctx, QSGW_STAGE_WEIGHTS);
    e = qsgw::launch_pair_weights(d_eps_k, d_f_k, d_eps_kq, d_f_kq, n_o, n_u, ctx->d_omega, ctx->n_freq,
                                  ctx->occ_tol, ctx->d_wtab + off, ctx->kpad, n_pad,
                                  ctx->f16 ? ctx->d_zmax + zi : nullptr, 1, ctx->stream);
  }
  if (e != cudaSuccess) return ctx->cuda_fail(e, "pair weights kernel launch");
  ctx->launches += 1;
  ctx->pairs += n_pairs;
  ctx->state = ST_READY;   // the batch is staged
  ctx->fill = off + n_pad;
  ctx->zslot = zi + 1;
  ctx->err.clear();
  return QSGW_OK;
}

int32_t qsgw_chi0_add_kpoint(qsgw_ctx* ctx, const void* d_Ck, int64_t ld_k, const void* d_Ckq, int64_t ld_kq,
                             const double* d_eps_k, const double* d_f_k, const double* d_eps_kq,
                             const double* d_f_kq, int32_t n_o_total, int32_t n_u_total) {
  if (!ctx) return QSGW_ERR_INVALID_ARG;
  if (n_o_total < 1 || n_u_total < 1) return ctx->fail(QSGW_ERR_SHAPE, "n_o_total and n_u_total must be positive");
  if (!d_eps_k || !d_f_k || !d_eps_kq || !d_f_kq) return ctx->fail(QSGW_ERR_INVALID_ARG, "NULL energy/occupation array");
  for (int n0 = 0; n0 < n_o_total; n0 += ctx->max_n_o) {
    const int no = (n_o_total - n0 < ctx->max_n_o) ? n_o_total - n0 : ctx->max_n_o;
    for (int u0 = 0; u0 < n_u_total; u0 += ctx->max_n_u) {
      const int nu = (n_u_total - u0 < ctx->max_n_u) ? n_u_total - u0 : ctx->max_n_u;
      int rc = qsgw_zmel_build(ctx, d_Ck, ld_k, d_Ckq, ld_kq, n0, no, u0, nu, nullptr);
      if (rc != QSGW_OK) return rc;
      rc = qsgw_chi0_accumulate(ctx, nullptr, d_eps_k + n0, d_f_k + n0, d_eps_kq + u0, d_f_kq + u0, no, nu);
      if (rc != QSGW_OK) return rc;
    }
  }
  return QSGW_OK;
}

int32_t qsgw_chi0_add_kpoints(qsgw_ctx* ctx, const void* d_Ck, int64_t ld_k, int64_t stride_k, const void* d_Ckq,
                              int64_t ld_kq, int64_t stride_kq, const double* d_eps_k, const double* d_f_k,
                              const double* d_eps_kq, const double* d_f_kq, int32_t n_o_total, int32_t n_u_total,
                              int32_t n_kpoints) {
  if (!ctx) return QSGW_ERR_INVALID_ARG;
  if (ctx->state == ST_CREATED) return ctx->fail(QSGW_ERR_STATE, "set_product_tensor must precede chi0_add_kpoints");
  if (n_o_total < 1 || n_u_total < 1 || n_kpoints < 1)
    return ctx->fail(QSGW_ERR_SHAPE, "n_o_total, n_u_total and n_kpoints must be positive");
  if (!d_Ck || !d_Ckq || !d_eps_k || !d_f_k || !d_eps_kq || !d_f_kq) return ctx->fail(QSGW_ERR_INVALID_ARG, "NULL argument");
  if (ld_k < ctx->n_b || ld_kq < ctx->n_b)
    return ctx->fail(QSGW_ERR_INVALID_ARG, "leading dimension smaller than N_b=%d", ctx->n_b);
  if (stride_k < 0 || stride_kq < 0) return ctx->fail(QSGW_ERR_INVALID_ARG, "negative k-point stride");
  const double2* Ck = static_cast<const double2*>(d_Ck);
  const double2* Ckq = static_cast<const double2*>(d_Ckq);
  const long long n_pairs = (long long)n_o_total * n_u_total;
  const long long n_pad = round_up(n_pairs, qsgw::kPairAlign);
  if (n_o_total > ctx->max_n_o || n_u_total > ctx->max_n_u || n_pad > ctx->stage_cap) {
    // the k-point does not fit one band batch: k-point by k-point through the band-batch loop
    for (int k = 0; k < n_kpoints; ++k) {
      int rc = qsgw_chi0_add_kpoint(ctx, Ck + (long long)k * stride_k, ld_k, Ckq + (long long)k * stride_kq, ld_kq,
                                    d_eps_k + (long long)k * n_o_total, d_f_k + (long long)k * n_o_total,
                                    d_eps_kq + (long long)k * n_u_total, d_f_kq + (long long)k * n_u_total, n_o_total,
                                    n_u_total);
      if (rc != QSGW_OK) return rc;
    }
    return QSGW_OK;
  }
  // groups of k-points that fit the staging workspace: ONE stage (a) launch (+ conversion) and ONE weight launch each
  for (int k0 = 0; k0 < n_kpoints;) {
    if (ctx->fill + n_pad > ctx->stage_cap) {
      int rc = flush_pending(ctx);
      if (rc != QSGW_OK) return rc;
    }
    long long room = (ctx->stage_cap - ctx->fill) / n_pad;
    int g = (int)(room < (long long)(n_kpoints - k0) ? room : (long long)(n_kpoints - k0));
    if (g > 65535) g = 65535;           // grid.z
    const long long off = ctx->fill;
    const int zi = ctx->zslot;
    int rc = build_batches(ctx, Ck + (long long)k0 * stride_k, ld_k, stride_k, Ckq + (long long)k0 * stride_kq, ld_kq,
                           stride_kq, 0, n_o_total, 0, n_u_total, g, off, n_pad, zi);
    if (rc != QSGW_OK) return rc;
    cudaError_t e;
    {
      StageScope ts(ctx, QSGW_STAGE_WEIGHTS);
      e = qsgw::launch_pair_weights(d_eps_k + (long long)k0 * n_o_total, d_f_k + (long long)k0 * n_o_total,
                                    d_eps_kq + (long long)k0 * n_u_total, d_f_kq + (long long)k0 * n_u_total, n_o_total,
                                    n_u_total, ctx->d_omega, ctx->n_freq, ctx->occ_tol, ctx->d_wtab + off, ctx->kpad,
                                    n_pad, ctx->f16 ? ctx->d_zmax + zi : nullptr, g, ctx->stream);
    }
    if (e != cudaSuccess) return ctx->cuda_fail(e, "pair weights kernel launch");
    ctx->launches += 1;
    ctx->pairs += n_pairs * g;
    ctx->fill = off + n_pad * g;
    ctx->zslot = zi + g;
    ctx->last_n_o = n_o_total;
    ctx->last_n_u = n_u_total;
    ctx->z_off = off + n_pad * (g - 1);
    ctx->z_zi = zi + g - 1;
    ctx->state = ST_READY;
    k0 += g;
  }
  ctx->err.clear();
  return QSGW_OK;
}

int32_t qsgw_chi0_finalize(qsgw_ctx* ctx, void* d_chi0_out) {
  if (!ctx) return QSGW_ERR_INVALID_ARG;
  if (ctx->state == ST_CREATED) return ctx->fail(QSGW_ERR_STATE, "nothing accumulated: set_product_tensor not called");
  if (!d_chi0_out) return ctx->fail(QSGW_ERR_INVALID_ARG, "d_chi0_out is NULL");
  int rc = flush_pending(ctx);
  if (rc != QSGW_OK) return rc;
  cudaError_t e;
  {
    StageScope ts(ctx, QSGW_STAGE_FINALIZE);
    e = qsgw::launch_finalize(ctx->d_acc_re, ctx->d_acc_im, ctx->n_m, ctx->n_m_pad, ctx->n_freq,
                              1.0 / (double)ctx->n_k, static_cast<double2*>(d_chi0_out), ctx->stream);
  }
  if (e != cudaSuccess) return ctx->cuda_fail(e, "finalize kernel launch");
  ctx->launches += 1;
  ctx->err.clear();
  return QSGW_OK;
}

int32_t qsgw_imchi_add_batch(qsgw_ctx* ctx, const void* d_Ck, int64_t ld_k, const void* d_Ckq, int64_t ld_kq,
                             int32_t n_begin, int32_t n_o, int32_t np_begin, int32_t n_u, const int32_t* d_bin_ptr,
                             const int32_t* d_pair, const double* d_w, int32_t nnz) {
  if (!ctx) return QSGW_ERR_INVALID_ARG;
  if (ctx->state == ST_CREATED) return ctx->fail(QSGW_ERR_STATE, "set_product_tensor must precede imchi_add_batch");
  if (!d_Ck || !d_Ckq || !d_bin_ptr || (nnz > 0 && (!d_pair || !d_w))) return ctx->fail(QSGW_ERR_INVALID_ARG, "NULL argument");
  if (ld_k < ctx->n_b || ld_kq < ctx->n_b)
    return ctx->fail(QSGW_ERR_INVALID_ARG, "leading dimension smaller than N_b=%d", ctx->n_b);
  if (n_begin < 0 || np_begin < 0 || nnz < 0) return ctx->fail(QSGW_ERR_SHAPE, "negative band offset or entry count");
  int rc = check_batch(ctx, n_o, n_u);
  if (rc != QSGW_OK) return rc;
  rc = flush_pending(ctx);              // the batch uses the whole workspace on its own
  if (rc != QSGW_OK) return rc;
  cudaError_t e;
  if (!ctx->d_ranges) {
    e = dev_alloc(ctx, &ctx->d_rowmap, (size_t)ctx->batch_pad);
    if (e == cudaSuccess) e = dev_alloc(ctx, &ctx->d_binscratch, 2 * (size_t)ctx->batch_pad + 4 * ((size_t)ctx->n_freq + 1));
    if (e == cudaSuccess) e = dev_alloc(ctx, &ctx->d_ranges, (size_t)ctx->n_freq);
    if (e != cudaSuccess) {
      cudaGetLastError();
      cudaFree(ctx->d_rowmap); cudaFree(ctx->d_binscratch); cudaFree(ctx->d_ranges);
      ctx->d_rowmap = ctx->d_binscratch = nullptr; ctx->d_ranges = nullptr;
      return ctx->fail(QSGW_ERR_ALLOC, "workspace of the binned path: %s", cudaGetErrorString(e));
    }
  }
  const long long n_pairs = (long long)n_o * n_u, n_pad = round_up(n_pairs, qsgw::kPairAlign);
  {
    StageScope ts(ctx, QSGW_STAGE_WEIGHTS);
    e = qsgw::launch_bin_setup(d_bin_ptr, d_pair, d_w, nnz, ctx->n_freq, n_pairs, n_pad, ctx->d_rowmap,
                               ctx->d_binscratch, ctx->d_wtab, ctx->kpad, ctx->d_ranges, ctx->stream);
  }
  if (e != cudaSuccess) return ctx->cuda_fail(e, "bin set-up kernels");
  ctx->launches += nnz > 0 ? 6 : 4;
  ctx->cur_row_map = ctx->d_rowmap;
  rc = build_batches(ctx, static_cast<const double2*>(d_Ck), ld_k, 0, static_cast<const double2*>(d_Ckq), ld_kq, 0,
                     n_begin, n_o, np_begin, n_u, 1, 0, n_pad, 0);
  ctx->cur_row_map = nullptr;
  if (rc != QSGW_OK) return rc;
  if (ctx->f16) {
    // mixed mode: the batch (FP16-split rows, scale from its measured maximum) is accumulated at once by the tcgen05
    // kernel over the per-bin row ranges; the caller's weights get the batch's 2^(-2S) when they are split into FP16 pieces
    ctx->fill = n_pad;
    ctx->flush_ranges = ctx->d_ranges;
    ctx->flush_zfold = ctx->d_zmax;
    rc = flush_pending(ctx);
    ctx->flush_ranges = nullptr;
    ctx->flush_zfold = nullptr;
    if (rc != QSGW_OK) return rc;
    ctx->pairs += n_pairs;
    ctx->state = ST_READY;
    ctx->err.clear();
    return QSGW_OK;
  }
  qsgw::Chi0F64Args a;
  a.tmap_z = ctx->tmap_z;
  a.wtab = ctx->d_wtab;
  a.kpad = ctx->kpad;
  a.acc_re = ctx->d_acc_re;
  a.acc_im = ctx->d_acc_im;
  a.n_m_pad = ctx->n_m_pad;
  a.n_freq = ctx->n_freq;
  a.j0 = 0;
  a.n_pairs_padded = n_pad;
  a.n_sm = ctx->n_sm;
  a.d_tiles = ctx->d_tiles;
  a.n_tiles = ctx->n_tiles;
  a.n_tiles_half = ctx->n_tiles_half;
  a.n_tiles_quarter = ctx->n_tiles_quarter;
  a.d_ranges = ctx->d_ranges;
  {
    StageScope ts(ctx, QSGW_STAGE_CHI0);
    e = qsgw::launch_chi0_f64(a, ctx->stream);
  }
  if (e != cudaSuccess) return ctx->cuda_fail(e, "binned accumulation kernel launch");
  ctx->launches += 1;
  ctx->pairs += n_pairs;
  ctx->state = ST_READY;               // the batch is consumed: nothing stays staged
  ctx->err.clear();
  return QSGW_OK;
}

static int32_t hilbert_common(int32_t n_m, int32_t n_bins, const double* d_edges, int32_t n_out, const double* d_omega_out,
                              const void* d_A, void* d_out, void* cuda_stream, int real_axis) {
  g_create_error.clear();
  if (!d_edges || !d_omega_out || !d_A || !d_out) { g_create_error = "NULL argument"; return QSGW_ERR_INVALID_ARG; }
  if (d_A == d_out) { g_create_error = "d_out aliases d_A"; return QSGW_ERR_INVALID_ARG; }
  if (n_m < 1 || n_bins < 1 || n_out < 1) { g_create_error = "n_m, n_bins and n_out must be positive"; return QSGW_ERR_SHAPE; }
  if (n_bins > 384) { g_create_error = "at most 384 bins (the transform matrix is held in shared memory)"; return QSGW_ERR_SHAPE; }
  cudaError_t e = qsgw::launch_hilbert(n_m, n_bins, d_edges, n_out, d_omega_out, static_cast<const double2*>(d_A),
                                       static_cast<double2*>(d_out), real_axis, static_cast<cudaStream_t>(cuda_stream));
  if (e != cudaSuccess) { cudaGetLastError(); g_create_error = std::string("Hilbert transform kernel: ") + cudaGetErrorString(e); return QSGW_ERR_CUDA; }
  return QSGW_OK;
}

int32_t qsgw_hilbert_to_imag_axis(int32_t n_m, int32_t n_bins, const double* d_edges, int32_t n_out,
                                  const double* d_omega_out, const void* d_A, void* d_out, void* cuda_stream) {
  return hilbert_common(n_m, n_bins, d_edges, n_out, d_omega_out, d_A, d_out, cuda_stream, 0);
}

int32_t qsgw_hilbert_to_real_axis(int32_t n_m, int32_t n_bins, const double* d_edges, int32_t n_out,
                                  const double* d_omega_out, const void* d_A, void* d_out, void* cuda_stream) {
  return hilbert_common(n_m, n_bins, d_edges, n_out, d_omega_out, d_A, d_out, cuda_stream, 1);
}

int32_t qsgw_sigc_imag_accumulate(qsgw_ctx* ctx, const void* d_z, const double* d_eps_q, const double* d_eps_qk,
                                  const void* d_wc, int32_t n_all, int32_t n_qp, void* d_sigc) {
  if (!ctx) return QSGW_ERR_INVALID_ARG;
  if (!d_eps_q || !d_eps_qk || !d_wc || !d_sigc) return ctx->fail(QSGW_ERR_INVALID_ARG, "NULL argument");
  int rc = check_batch(ctx, n_all, n_qp);
  if (rc != QSGW_OK) return rc;
  if (!d_z) {
    if (ctx->state != ST_Z_BUILT) return ctx->fail(QSGW_ERR_STATE, "no z batch: call zmel_build first or pass d_z");
    if (n_all != ctx->last_n_o || n_qp != ctx->last_n_u)
      return ctx->fail(QSGW_ERR_SHAPE, "batch %d x %d differs from the last zmel_build (%d x %d)", n_all, n_qp,
                       ctx->last_n_o, ctx->last_n_u);
  }
  cudaError_t e = wc_configure_device(ctx->device);
  if (e != cudaSuccess) return ctx->cuda_fail(e, "kernel attributes");
  if (!ctx->d_szw) {
    const size_t cap = (size_t)ctx->max_n_o * ctx->max_n_u * ctx->n_m;
    e = dev_alloc(ctx, &ctx->d_sz, cap);
    if (e == cudaSuccess) e = dev_alloc(ctx, &ctx->d_sw, (size_t)ctx->n_freq * ctx->batch_pad);
    if (e == cudaSuccess) e = dev_alloc(ctx, &ctx->d_szw, cap);
    if (e == cudaSuccess && ctx->f16) {
      e = dev_alloc(ctx, &ctx->d_zk16, qsgw::sigc_f16_z_halves((long long)ctx->max_n_o * ctx->max_n_u, ctx->n_m));
      if (e == cudaSuccess) e = dev_alloc(ctx, &ctx->d_w16, qsgw::sigc_f16_w_halves(ctx->n_m, ctx->n_freq));
      if (e == cudaSuccess) e = dev_alloc(ctx, &ctx->d_w8, 2 * qsgw::sigc_f16_w_halves(ctx->n_m, ctx->n_freq));
      if (e == cudaSuccess) e = dev_alloc(ctx, &ctx->d_samax, (size_t)ctx->n_freq + 1);
      if (e == cudaSuccess) e = qsgw::sigc_f16_configure();
    }
    if (e != cudaSuccess) {
      cudaGetLastError();
      cudaFree(ctx->d_sz); cudaFree(ctx->d_sw); cudaFree(ctx->d_szw);
      cudaFree(ctx->d_zk16); cudaFree(ctx->d_w16); cudaFree(ctx->d_w8); cudaFree(ctx->d_samax);
      ctx->d_zk16 = ctx->d_w16 = nullptr; ctx->d_w8 = nullptr; ctx->d_samax = nullptr;
      ctx->d_sz = ctx->d_szw = nullptr; ctx->d_sw = nullptr;
      return ctx->fail(QSGW_ERR_ALLOC, "I^c workspace allocation failed: %s", cudaGetErrorString(e));
    }
  }
  const long long n_pairs = (long long)n_all * n_qp;
  const double2* z = static_cast<const double2*>(d_z);
  if (!d_z) {
    if (ctx->f16)
      e = qsgw::launch_z_export_hl16(hl_slot(ctx->d_zhl, ctx->z_off), ctx->kpad, ctx->n_m_pad, ctx->n_m, n_pairs,
                                     ctx->d_zmax + ctx->z_zi, ctx->d_sz, ctx->stream);
    else
      e = qsgw::launch_z_export(ctx->d_zws + ctx->z_off * qsgw::kCG, ctx->kpad, ctx->ncg, ctx->n_m, n_pairs, ctx->d_sz,
                                ctx->stream);
    if (e != cudaSuccess) return ctx->cuda_fail(e, "z export kernel launch");
    ctx->launches += 1;
    z = ctx->d_sz;
  }
  e = qsgw::launch_sigc_weights(d_eps_q, d_eps_qk, n_all, n_qp, ctx->d_omega, ctx->n_freq, ctx->d_sw, ctx->batch_pad,
                                ctx->stream);
  if (e == cudaSuccess && ctx->f16 && !ctx->sigc_f64) {
    // mixed mode: the frequency loop on tcgen05 with FP16-split operands, the closing contraction in FP64
    e = qsgw::launch_sigc_zw_f16(z, static_cast<const double2*>(d_wc), ctx->d_sw, ctx->batch_pad, (int)n_pairs, ctx->n_m,
                                 ctx->n_freq, ctx->d_zk16, ctx->d_w16, ctx->sigc_fp8 ? ctx->d_w8 : nullptr, ctx->d_samax, ctx->d_szw,
                                 ctx->stream);
    if (e == cudaSuccess)
      e = qsgw::launch_sigc_close(z, ctx->d_szw, n_all, n_qp, ctx->n_m, 1.0 / (double)ctx->n_k,
                                  static_cast<double2*>(d_sigc), ctx->n_sm, ctx->stream);
    ctx->launches += 4;
  } else if (e == cudaSuccess) {
    e = qsgw::launch_sigc_imag(z, ctx->d_sw, ctx->batch_pad, static_cast<const double2*>(d_wc), n_all, n_qp, ctx->n_m,
                               ctx->n_freq, 1.0 / (double)ctx->n_k, ctx->d_szw, static_cast<double2*>(d_sigc), ctx->n_sm,
                               ctx->stream);
  }
  if (e != cudaSuccess) return ctx->cuda_fail(e, "I^c kernel launch");
  ctx->launches += 3;
  ctx->err.clear();
  return QSGW_OK;
}

// Common checks of the context-free entry points: an sm_100 device is current, kernel attributes are set.
static int wc_prologue(DevInfo* di) {
  if (current_device(di) != cudaSuccess) {
    cudaGetLastError();
    g_create_error = "no CUDA device";
    return QSGW_ERR_UNSUPPORTED;
  }
  if (di->cc_major != 10) { g_create_error = "kernels are built for sm_100a only"; return QSGW_ERR_UNSUPPORTED; }
  cudaError_t e = wc_configure_device(di->dev);
  if (e != cudaSuccess) { cudaGetLastError(); g_create_error = std::string("kernel attributes: ") + cudaGetErrorString(e); return QSGW_ERR_CUDA; }
  return QSGW_OK;
}

int32_t qsgw_wc_from_chi0(int32_t n_m, int32_t n_freq, const void* d_chi0, const double* d_v, void* d_wc_out,
                          int32_t* d_info, void* cuda_stream) {
  g_create_error.clear();
  if (!d_chi0 || !d_v || !d_wc_out || !d_info) { g_create_error = "NULL argument"; return QSGW_ERR_INVALID_ARG; }
  if (d_chi0 == d_wc_out) { g_create_error = "d_wc_out aliases d_chi0"; return QSGW_ERR_INVALID_ARG; }
  if (n_m < 1 || n_freq < 1) { g_create_error = "n_m and n_freq must be positive"; return QSGW_ERR_SHAPE; }
  DevInfo di;
  int rc = wc_prologue(&di);
  if (rc != QSGW_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  double2* work = nullptr;
  cudaError_t e = work_alloc(di.dev, reinterpret_cast<void**>(&work), sizeof(double2) * qsgw::wc_work_elems(n_m, n_freq), st);
  if (e != cudaSuccess) { cudaGetLastError(); g_create_error = std::string("workspace allocation failed: ") + cudaGetErrorString(e); return QSGW_ERR_ALLOC; }
  // The factorisation is a few hundred small dependent launches: they are captured into a CUDA graph on an
  // internal stream of this device (the caller's stream may be the legacy default stream, which cannot be
  // captured) and launched as one unit between two events, so that a busy host cannot starve the GPU.  A capture
  // failure falls back to plain launches on the caller's stream; a failure AFTER the graph was launched does not
  // (the graph is in flight on `work`): it is reported.
  bool done = false, launched = false;
  if (g_wc_graph != 0 && di.dev >= 0 && di.dev < qsgw::kMaxDevices) {
    WcGraphs& G = wc_graphs();
    std::lock_guard<std::mutex> lock(G.mu);
    G.sweep();
    cudaStream_t& gs = G.stream[di.dev];
    cudaEvent_t ev_in = nullptr, ev_out = nullptr;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    bool ok = gs != nullptr || cudaStreamCreateWithFlags(&gs, cudaStreamNonBlocking) == cudaSuccess;
    ok = ok && cudaEventCreateWithFlags(&ev_in, cudaEventDisableTiming) == cudaSuccess &&
         cudaEventCreateWithFlags(&ev_out, cudaEventDisableTiming) == cudaSuccess;
    ok = ok && cudaEventRecord(ev_in, st) == cudaSuccess && cudaStreamWaitEvent(gs, ev_in, 0) == cudaSuccess;
    if (ok && cudaStreamBeginCapture(gs, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
      const cudaError_t le = qsgw::launch_wc_from_chi0(n_m, n_freq, static_cast<const double2*>(d_chi0), d_v,
                                                       static_cast<double2*>(d_wc_out), work, d_info, gs);
      const cudaError_t ce = cudaStreamEndCapture(gs, &graph);
      ok = le == cudaSuccess && ce == cudaSuccess && graph != nullptr &&
           cudaGraphInstantiate(&exec, graph, 0) == cudaSuccess;
      if (ok) {
        ok = cudaGraphLaunch(exec, gs) == cudaSuccess;
        launched = ok;
      }
    } else {
      ok = false;
    }
    if (graph) cudaGraphDestroy(graph);
    if (launched) {
      done = cudaEventRecord(ev_out, gs) == cudaSuccess && cudaStreamWaitEvent(st, ev_out, 0) == cudaSuccess;
      if (!done) cudaStreamSynchronize(gs);        // the graph still owns `work`: wait for it before anything else
      G.pending.push_back({exec, ev_out});         // destroyed by a later sweep once ev_out has completed
      exec = nullptr;
      ev_out = nullptr;
    }
    if (exec) cudaGraphExecDestroy(exec);
    if (ev_in) cudaEventDestroy(ev_in);
    if (ev_out) cudaEventDestroy(ev_out);
    if (!done) cudaGetLastError();
  }
  e = cudaSuccess;
  if (!done && (launched || g_wc_graph == 2)) {
    cudaFreeAsync(work, st);
    g_create_error = launched ? "ordering the W^c graph after launch failed" : "CUDA graph capture of the W^c launch sequence failed";
    return QSGW_ERR_CUDA;
  }
  if (!done)
    e = qsgw::launch_wc_from_chi0(n_m, n_freq, static_cast<const double2*>(d_chi0), d_v,
                                  static_cast<double2*>(d_wc_out), work, d_info, st);
  cudaFreeAsync(work, st);
  if (e != cudaSuccess) { cudaGetLastError(); g_create_error = std::string("W^c kernels: ") + cudaGetErrorString(e); return QSGW_ERR_CUDA; }
  return QSGW_OK;
}

int32_t qsgw_chi0_to_coulomb_basis(int32_t n_m, int32_t n_freq, const void* d_chi0, const void* d_U, void* d_out,
                                   void* cuda_stream) {
  g_create_error.clear();
  if (!d_chi0 || !d_U || !d_out) { g_create_error = "NULL argument"; return QSGW_ERR_INVALID_ARG; }
  if (d_chi0 == d_out) { g_create_error = "d_out aliases d_chi0"; return QSGW_ERR_INVALID_ARG; }
  if (n_m < 1 || n_freq < 1) { g_create_error = "n_m and n_freq must be positive"; return QSGW_ERR_SHAPE; }
  DevInfo di;
  int rc = wc_prologue(&di);
  if (rc != QSGW_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  double2* work = nullptr;
  cudaError_t e = work_alloc(di.dev, reinterpret_cast<void**>(&work), sizeof(double2) * qsgw::rotate_work_elems(n_m, n_freq), st);
  if (e != cudaSuccess) { cudaGetLastError(); g_create_error = std::string("workspace allocation failed: ") + cudaGetErrorString(e); return QSGW_ERR_ALLOC; }
  e = qsgw::launch_rotate_basis(n_m, n_freq, static_cast<const double2*>(d_chi0), static_cast<const double2*>(d_U),
                                static_cast<double2*>(d_out), work, st);
  cudaFreeAsync(work, st);
  if (e != cudaSuccess) { cudaGetLastError(); g_create_error = std::string("rotation kernels: ") + cudaGetErrorString(e); return QSGW_ERR_CUDA; }
  return QSGW_OK;
}

int32_t qsgw_chi0_to_coulomb_basis_static(int32_t n_m, int32_t n_freq, const void* d_chi0, const void* d_U, void* d_out,
                                          void* cuda_stream) {
  g_create_error.clear();
  if (!d_chi0 || !d_U || !d_out) { g_create_error = "NULL argument"; return QSGW_ERR_INVALID_ARG; }
  if (d_chi0 == d_out) { g_create_error = "d_out aliases d_chi0"; return QSGW_ERR_INVALID_ARG; }
  if (n_m < 1 || n_freq < 1) { g_create_error = "n_m and n_freq must be positive"; return QSGW_ERR_SHAPE; }
  const long long need = (long long)qsgw::rotate_work_elems(n_m, n_freq);
  if (need > qsgw::rotate_static_max_elems()) {
    char buf[256];
    snprintf(buf, sizeof(buf), "(2 n_freq + 1) ceil64(n_m)^2 = %lld complex elements exceed the static scratch of %lld "
             "(e.g. n_m <= 256 at 16 frequencies): use qsgw_chi0_to_coulomb_basis", need, qsgw::rotate_static_max_elems());
    g_create_error = buf;
    return QSGW_ERR_ALLOC;
  }
  DevInfo di;
  int rc = wc_prologue(&di);
  if (rc != QSGW_OK) return rc;
  cudaError_t e = qsgw::launch_rotate_basis_static(n_m, n_freq, static_cast<const double2*>(d_chi0),
                                                   static_cast<const double2*>(d_U), static_cast<double2*>(d_out),
                                                   static_cast<cudaStream_t>(cuda_stream));
  if (e != cudaSuccess) { cudaGetLastError(); g_create_error = std::string("rotation kernels (static scratch): ") + cudaGetErrorString(e); return QSGW_ERR_CUDA; }
  return QSGW_OK;
}

int32_t qsgw_zmel_ipw_build(const int32_t* h_L, const void* d_theta, int32_t n_pw_kq, const int32_t* d_g_kq, int32_t n_pw_k,
                            const int32_t* d_g_k, int32_t n_ipw, const int32_t* d_g_ipw, const void* d_Bk, int64_t ld_k,
                            int32_t n_o, const void* d_Bkq, int64_t ld_kq, int32_t n_u, void* d_z_out, int64_t ld_z,
                            void* cuda_stream) {
  g_create_error.clear();
  if (!h_L || !d_theta || !d_g_kq || !d_g_k || !d_g_ipw || !d_Bk || !d_Bkq || !d_z_out) {
    g_create_error = "NULL argument";
    return QSGW_ERR_INVALID_ARG;
  }
  if (n_pw_kq < 1 || n_pw_k < 1 || n_ipw < 1 || n_o < 1 || n_u < 1) { g_create_error = "counts must be positive"; return QSGW_ERR_SHAPE; }
  if (h_L[0] < 0 || h_L[1] < 0 || h_L[2] < 0) { g_create_error = "negative box half extent"; return QSGW_ERR_SHAPE; }
  if (ld_k < n_pw_k || ld_kq < n_pw_kq || ld_z < n_ipw) { g_create_error = "leading dimension smaller than the row length"; return QSGW_ERR_INVALID_ARG; }
  if ((long long)n_ipw * n_o > 2000000000ll || (long long)n_pw_kq * n_ipw > 2000000000ll) { g_create_error = "block too large for 32-bit GEMM extents"; return QSGW_ERR_SHAPE; }
  DevInfo di;
  int rc = wc_prologue(&di);
  if (rc != QSGW_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int a_chunk = qsgw::ipw_alpha_chunk(n_pw_kq, n_pw_k, n_ipw, n_o, (size_t)1 << 30);
  if ((long long)a_chunk * n_ipw > 2000000000ll) { g_create_error = "block too large for 32-bit GEMM extents"; return QSGW_ERR_SHAPE; }
  double2* work = nullptr;
  cudaError_t e = work_alloc(di.dev, reinterpret_cast<void**>(&work),
                             sizeof(double2) * qsgw::ipw_work_elems(a_chunk, n_pw_k, n_ipw, n_o, n_u), st);
  if (e != cudaSuccess) { cudaGetLastError(); g_create_error = std::string("workspace allocation failed: ") + cudaGetErrorString(e); return QSGW_ERR_ALLOC; }
  const int L[3] = {h_L[0], h_L[1], h_L[2]};
  e = qsgw::launch_zmel_ipw(L, static_cast<const double2*>(d_theta), n_pw_kq, d_g_kq, n_pw_k, d_g_k, n_ipw, d_g_ipw,
                            static_cast<const double2*>(d_Bk), ld_k, n_o, static_cast<const double2*>(d_Bkq), ld_kq, n_u,
                            static_cast<double2*>(d_z_out), ld_z, a_chunk, work, st);
  cudaFreeAsync(work, st);
  if (e != cudaSuccess) { cudaGetLastError(); g_create_error = std::string("IPW block kernels: ") + cudaGetErrorString(e); return QSGW_ERR_CUDA; }
  return QSGW_OK;
}

int32_t qsgw_coulomb_eigenbasis(int32_t n_m, const void* d_v, const void* d_O, double* d_vmu_out, void* d_U_out,
                                int32_t* h_info, int32_t* h_sweeps, void* cuda_stream) {
  g_create_error.clear();
  if (h_info) *h_info = 0;
  if (h_sweeps) *h_sweeps = 0;
  if (!d_v || !d_O || !d_vmu_out || !d_U_out) { g_create_error = "NULL argument"; return QSGW_ERR_INVALID_ARG; }
  if (n_m < 1) { g_create_error = "n_m must be positive"; return QSGW_ERR_SHAPE; }
  DevInfo di;
  int rc = wc_prologue(&di);
  if (rc != QSGW_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int N = (n_m + 63) / 64 * 64;
  const size_t small_bytes = 256 + sizeof(double) * (size_t)n_m + sizeof(int) * (size_t)n_m + 64;
  double2* work = nullptr;
  cudaError_t e = work_alloc(di.dev, reinterpret_cast<void**>(&work),
                             sizeof(double2) * qsgw::eig_work_elems(n_m) + small_bytes, st);
  if (e != cudaSuccess) { cudaGetLastError(); g_create_error = std::string("workspace allocation failed: ") + cudaGetErrorString(e); return QSGW_ERR_ALLOC; }
  unsigned char* sm = reinterpret_cast<unsigned char*>(work + qsgw::eig_work_elems(n_m));
  int* d_info = reinterpret_cast<int*>(sm);
  double* d_norms = reinterpret_cast<double*>(sm + 64);
  double* d_diag = reinterpret_cast<double*>(sm + 256);
  int* d_perm = reinterpret_cast<int*>(sm + 256 + sizeof(double) * (size_t)n_m);
#define QSGW_E(expr, what)                                                                              \
  do {                                                                                                  \
    e = (expr);                                                                                         \
    if (e != cudaSuccess) {                                                                             \
      cudaGetLastError(); cudaFreeAsync(work, st);                                                      \
      g_create_error = std::string(what) + ": " + cudaGetErrorString(e);                                \
      return QSGW_ERR_CUDA;                                                                             \
    }                                                                                                   \
  } while (0)
  QSGW_E(qsgw::launch_eig_reduce(n_m, static_cast<const double2*>(d_v), static_cast<const double2*>(d_O), work, d_info, st),
         "reduction to the standard problem");
  int info = 0;
  QSGW_E(cudaMemcpyAsync(&info, d_info, sizeof(int), cudaMemcpyDeviceToHost, st), "copy of info");
  QSGW_E(cudaStreamSynchronize(st), "stream synchronisation");
  if (info != 0) {                                     // O is not positive definite
    cudaFreeAsync(work, st);
    if (h_info) *h_info = info;
    g_create_error = "the overlap matrix is not positive definite";
    return QSGW_ERR_INVALID_ARG;
  }
  // Jacobi sweeps until the off-diagonal part reaches its rounding floor: quadratic convergence, so once the ratio
  // |off|^2 / |C|^2 is below 1e-18 the next sweep lands on the floor and the one after that no longer improves
  const double floor_ratio = 4e-32 * (double)N * (double)N;
  double prev = 1.0;
  int sweeps = 0;
  bool converged = false;
  for (; sweeps < 60 && !converged;) {
    QSGW_E(qsgw::launch_eig_sweep(n_m, work, d_norms, g_eig_blocked != 0, sweeps == 0, st), "Jacobi sweep");
    double nr[2] = {0.0, 0.0};
    QSGW_E(cudaMemcpyAsync(nr, d_norms, 2 * sizeof(double), cudaMemcpyDeviceToHost, st), "copy of the norms");
    QSGW_E(cudaStreamSynchronize(st), "stream synchronisation");
    ++sweeps;
    const double tot = nr[0] + nr[1];
    const double ratio = tot > 0.0 ? nr[0] / tot : 0.0;
    if (ratio <= floor_ratio || (prev <= 1e-18 && ratio >= 0.25 * prev)) converged = true;
    prev = ratio;
  }
  if (h_sweeps) *h_sweeps = sweeps;
  if (!converged) {
    cudaFreeAsync(work, st);
    if (h_info) *h_info = -1;
    g_create_error = "Jacobi iteration did not converge in 60 sweeps";
    return QSGW_ERR_CUDA;
  }
  // eigenvalues to the host, descending order ("mu = 1 corresponds to the largest eigenvalue")
  std::vector<double> lam((size_t)n_m);
  QSGW_E(qsgw::launch_eig_diag(n_m, work, d_diag, st), "eigenvalue extraction");
  QSGW_E(cudaMemcpyAsync(lam.data(), d_diag, sizeof(double) * (size_t)n_m, cudaMemcpyDeviceToHost, st), "copy of the eigenvalues");
  QSGW_E(cudaStreamSynchronize(st), "stream synchronisation");
  std::vector<int> perm((size_t)n_m);
  for (int i = 0; i < n_m; ++i) perm[(size_t)i] = i;
  std::stable_sort(perm.begin(), perm.end(), [&](int a, int b) { return lam[(size_t)a] > lam[(size_t)b]; });
  std::vector<double> sorted((size_t)n_m);
  for (int i = 0; i < n_m; ++i) sorted[(size_t)i] = lam[(size_t)perm[(size_t)i]];
  QSGW_E(cudaMemcpyAsync(d_perm, perm.data(), sizeof(int) * (size_t)n_m, cudaMemcpyHostToDevice, st), "upload of the order");
  QSGW_E(cudaMemcpyAsync(d_vmu_out, sorted.data(), sizeof(double) * (size_t)n_m, cudaMemcpyHostToDevice, st), "upload of v_mu");
  QSGW_E(qsgw::launch_eig_finish(n_m, work, d_perm, static_cast<double2*>(d_U_out), st), "back transformation");
  QSGW_E(cudaStreamSynchronize(st), "stream synchronisation");     // perm / sorted are host temporaries
#undef QSGW_E
  cudaFreeAsync(work, st);
  return QSGW_OK;
}

int32_t qsgw_chi0_run_host(qsgw_ctx* c, const void* h_P, const void* h_Ck, const void* h_Ckq, const double* h_eps_k,
                           const double* h_f_k, const double* h_eps_kq, const double* h_f_kq, int32_t n_k_points,
                           int32_t n_o, int32_t n_u, void* h_chi0_out, int64_t* out_kernel_launches) {
  if (!c) return QSGW_ERR_INVALID_ARG;
  if (!h_P || !h_Ck || !h_Ckq || !h_eps_k || !h_f_k || !h_eps_kq || !h_f_kq || !h_chi0_out)
    return c->fail(QSGW_ERR_INVALID_ARG, "NULL argument");
  if (n_o < 1 || n_u < 1 || n_k_points < 1) return c->fail(QSGW_ERR_SHAPE, "n_k_points, n_o and n_u must be positive");
  cudaStream_t st = c->stream;
  qsgw_ctx::HostRun& H = c->hr;
  const int nb = c->n_b, nm = c->n_m;
  // k-points travel in groups: as many as one multi-k launch of qsgw_chi0_add_kpoints takes (bounded to 64 MB of
  // staging per array), one k-point at a time when a k-point needs the band-batch loop
  const long long n_pad1 = round_up((long long)n_o * n_u, qsgw::kPairAlign);
  int G = 1;
  if (n_o <= c->max_n_o && n_u <= c->max_n_u && n_pad1 <= c->stage_cap) {
    long long g = c->stage_cap / n_pad1;
    const long long cap = (64ll << 20) / (long long)(sizeof(double2) * (size_t)(n_o > n_u ? n_o : n_u) * nb);
    if (g > cap) g = cap;
    if (g > n_k_points) g = n_k_points;
    G = (int)(g < 1 ? 1 : g);
  }
  const size_t ck_1 = (size_t)n_o * nb, ckq_1 = (size_t)n_u * nb;
  const size_t ck_e = ck_1 * G, ckq_e = ckq_1 * G;
  const size_t e_len = (2 * (size_t)n_o + 2 * (size_t)n_u) * G;
  const size_t out_e = (size_t)c->n_freq * nm * nm;
  const long long launches0 = c->launches;
#define QSGW_H(expr)                                                                   \
  do {                                                                                 \
    cudaError_t _e = (expr);                                                           \
    if (_e != cudaSuccess) { cudaGetLastError(); return c->cuda_fail(_e, #expr); }     \
  } while (0)
  // staging buffers: allocated once, grown when a later call passes larger band counts
  if (!H.dP) QSGW_H(dev_alloc(c, &H.dP, (size_t)c->p_elems));
  if (!H.dOut) QSGW_H(dev_alloc(c, &H.dOut, out_e));
  for (int i = 0; i < 2; ++i) {
    if (H.ck_cap < ck_e) { cudaStreamSynchronize(st); cudaFree(H.dCk[i]); H.dCk[i] = nullptr; QSGW_H(dev_alloc(c, &H.dCk[i], ck_e)); }
    if (H.ckq_cap < ckq_e) { cudaStreamSynchronize(st); cudaFree(H.dCkq[i]); H.dCkq[i] = nullptr; QSGW_H(dev_alloc(c, &H.dCkq[i], ckq_e)); }
    if (H.e_cap < e_len) { cudaStreamSynchronize(st); cudaFree(H.dE[i]); H.dE[i] = nullptr; QSGW_H(dev_alloc(c, &H.dE[i], e_len)); }
    if (!H.done[i]) QSGW_H(cudaEventCreateWithFlags(&H.done[i], cudaEventDisableTiming));
  }
  if (H.ck_cap < ck_e) H.ck_cap = ck_e;
  if (H.ckq_cap < ckq_e) H.ckq_cap = ckq_e;
  if (H.e_cap < e_len) H.e_cap = e_len;
  for (int g = 0; g < 4; ++g)
    if (!H.ready[g]) QSGW_H(cudaEventCreateWithFlags(&H.ready[g], cudaEventDisableTiming));
  if (!H.cp) QSGW_H(cudaStreamCreateWithFlags(&H.cp, cudaStreamNonBlocking));

  int rc = qsgw_reset(c);
  if (rc != QSGW_OK) return rc;
  QSGW_H(cudaMemcpyAsync(H.dP, h_P, sizeof(double2) * c->p_elems, cudaMemcpyHostToDevice, st));
  rc = qsgw_set_product_tensor(c, H.dP);
  if (rc != QSGW_OK) return rc;
  int grp = 0;
  for (int k = 0; k < n_k_points; k += G, ++grp) {
    const int b = grp & 1;
    const size_t g = (size_t)((n_k_points - k < G) ? n_k_points - k : G);
    if (grp >= 2) QSGW_H(cudaEventSynchronize(H.done[b]));   // keeps the host at most two groups ahead
    double* E = H.dE[b];
    double* e_k = E;
    double* f_k = E + g * n_o;
    double* e_kq = E + 2 * g * n_o;
    double* f_kq = E + 2 * g * n_o + g * n_u;
    QSGW_H(cudaMemcpyAsync(H.dCk[b], static_cast<const double2*>(h_Ck) + (size_t)k * ck_1, sizeof(double2) * ck_1 * g, cudaMemcpyHostToDevice, st));
    QSGW_H(cudaMemcpyAsync(H.dCkq[b], static_cast<const double2*>(h_Ckq) + (size_t)k * ckq_1, sizeof(double2) * ckq_1 * g, cudaMemcpyHostToDevice, st));
    QSGW_H(cudaMemcpyAsync(e_k, h_eps_k + (size_t)k * n_o, sizeof(double) * n_o * g, cudaMemcpyHostToDevice, st));
    QSGW_H(cudaMemcpyAsync(f_k, h_f_k + (size_t)k * n_o, sizeof(double) * n_o * g, cudaMemcpyHostToDevice, st));
    QSGW_H(cudaMemcpyAsync(e_kq, h_eps_kq + (size_t)k * n_u, sizeof(double) * n_u * g, cudaMemcpyHostToDevice, st));
    QSGW_H(cudaMemcpyAsync(f_kq, h_f_kq + (size_t)k * n_u, sizeof(double) * n_u * g, cudaMemcpyHostToDevice, st));
    rc = qsgw_chi0_add_kpoints(c, H.dCk[b], nb, (long long)ck_1, H.dCkq[b], nb, (long long)ckq_1, e_k, f_k, e_kq, f_kq, n_o,
                               n_u, (int)g);
    if (rc != QSGW_OK) return rc;
    QSGW_H(cudaEventRecord(H.done[b], st));
  }
  // The batches still staged are accumulated frequency group by frequency group; each group is finalized and
  // copied to the host on a second stream while the next group's kernel runs (the 16 N_M^2 result is the one
  // large transfer of the job).
  {
    const int ng = c->e2e_groups <= c->n_freq ? c->e2e_groups : 1;
    const size_t plane_pad = (size_t)c->n_m_pad * c->n_m_pad, plane_out = (size_t)nm * nm;
    cudaError_t ce = cudaSuccess;
    for (int g = 0; g < ng && rc == QSGW_OK && ce == cudaSuccess; ++g) {
      const int j0 = (int)((long long)c->n_freq * g / ng), j1 = (int)((long long)c->n_freq * (g + 1) / ng);
      rc = flush_range(c, j0, j1 - j0, g == 0, g == ng - 1);
      if (rc != QSGW_OK) break;
      ce = qsgw::launch_finalize(c->d_acc_re + j0 * plane_pad, c->d_acc_im + j0 * plane_pad, nm, c->n_m_pad, j1 - j0,
                                 1.0 / (double)c->n_k, H.dOut + j0 * plane_out, st);
      c->launches += 1;
      if (ce == cudaSuccess) ce = cudaEventRecord(H.ready[g], st);
      if (ce == cudaSuccess) ce = cudaStreamWaitEvent(H.cp, H.ready[g], 0);
      if (ce == cudaSuccess)
        ce = cudaMemcpyAsync(static_cast<double2*>(h_chi0_out) + j0 * plane_out, H.dOut + j0 * plane_out,
                             sizeof(double2) * (j1 - j0) * plane_out, cudaMemcpyDeviceToHost, H.cp);
    }
    cudaError_t se = cudaStreamSynchronize(H.cp);
    if (ce == cudaSuccess) ce = se;
    se = cudaStreamSynchronize(st);
    if (ce == cudaSuccess) ce = se;
    if (rc != QSGW_OK) return rc;
    if (ce != cudaSuccess) { cudaGetLastError(); return c->cuda_fail(ce, "result copy"); }
  }
#undef QSGW_H
  if (out_kernel_launches) *out_kernel_launches = c->launches - launches0;
  c->err.clear();
  return QSGW_OK;
}

}  // extern "C"
