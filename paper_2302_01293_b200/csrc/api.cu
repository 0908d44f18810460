// api.cu -- the C ABI of include/qlp_bls.h: context, workspace and kernel launches.
// Every step of the path runs in the kernels of grid.cuh / prep.cuh / foldscan.cuh / snr_kernel.cuh;
// the host code below only sizes buffers and enqueues work.
#include <math.h>
#include <mutex>
#include <new>
#include <string.h>

#include <vector>

#include <nvtx3/nvToolsExt.h>  // header-only; a no-op unless a profiler injects itself (nsys, ncu --nvtx)

#include "common.cuh"
#include "foldscan.cuh"
#include "grid.cuh"
#include "prep.cuh"
#include "snr_kernel.cuh"
#include "stats.cuh"
#include "fit.cuh"
#include "pink.cuh"

using namespace qlp;

static constexpr int kClassCtr = 8;  // uint64 counters per tile class (5 used), see qlp_bls_fold_class_counters
static constexpr uint32_t kPaperMask = 0xFF8u;  // widths 3..11 (PAPER.md:19, :35 -> DESIGN.md O1.9)

// One NVTX range per C-ABI call (and per sub-batch of the host driver), named after the call: a timeline lines the
// stages up with the kernels they launch, and `ncu --nvtx --nvtx-include "qlp_bls_spectrum/"` picks one stage.
struct NvtxRange {
  explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
  ~NvtxRange() { nvtxRangePop(); }
  NvtxRange(const NvtxRange&) = delete;
  NvtxRange& operator=(const NvtxRange&) = delete;
};

struct DevBuf {
  void* p = nullptr;
  size_t cap = 0;
  int ensure(size_t bytes) {
    if (bytes <= cap) return 0;
    if (p) cudaFree(p);
    p = nullptr; cap = 0;
    size_t want = bytes + bytes / 8 + 256;
    cudaError_t e = cudaMalloc(&p, want);
    if (e != cudaSuccess) { cudaGetLastError(); e = cudaMalloc(&p, bytes); want = bytes; }
    if (e != cudaSuccess) { cudaGetLastError(); p = nullptr; return QLP_BLS_ENOMEM; }
    cap = want;
    return 0;
  }
  void release() { if (p) cudaFree(p); p = nullptr; cap = 0; }
};

struct qlp_bls_ctx {
  qlp_bls_config cfg;
  Params prm;
  int device = 0;
  int n_sm = 148;
  int32_t widths[32];
  int n_widths = 0;
  int32_t force_path = 0;
  int64_t launches = 0;
  // workspace
  DevBuf pts, prep, kb, cnt, off, counters, star_bins, totals_dev, fit_cnt, fit_off, fit_work, fit_chunk, fit_list, class_ctr, star_order;
  // host-API staging
  DevBuf h_row[2], h_t[2], h_y[2], h_dy[2], h_rho[2], h_grid, h_fptr, h_sr, h_best, h_peaks, h_stats, h_fits, h_pink;
  static const int kSide = 3;           // side streams for the independent tile-class launches
  cudaStream_t side[kSide];
  cudaEvent_t side_done[kSide], fork_ev;
  bool fork_ready = false;
  cudaStream_t copy_stream = nullptr;  // H2D of the next sub-batch overlaps the search of the current one
  cudaEvent_t h2d_done[2], set_free[2];
  bool copy_ready = false;
  int64_t* totals_host = nullptr;  // pinned, 8 x int64
  // The prepared point records (S0) in `pts` / `prep` belong to the arrays of the last run_prep call; qlp_bls_snr
  // reuses them only if it is given the same arrays and nothing else wrote the workspace since.
  struct PrepKey {
    const void *row_ptr = nullptr, *t = nullptr, *y = nullptr, *dy = nullptr, *grid = nullptr;
    int64_t n_stars = -1;
    bool operator==(const PrepKey& o) const {
      return row_ptr == o.row_ptr && t == o.t && y == o.y && dy == o.dy && grid == o.grid && n_stars == o.n_stars;
    }
  } prep_key;
  bool prep_valid = false;
  const void* grid_row_ptr = nullptr;  // batch of the last qlp_bls_grid call: only the test-only debug_prep call
  int64_t grid_n_stars = -1;           // reads it (to learn the batch size); no workspace is sized from it
  int64_t* row_tmp[2] = {nullptr, nullptr};   // pinned staging of the rebased row_ptr of a host sub-batch
  size_t row_tmp_cap = 0;
  // optional per-call CUDA-event timing of the fold/scan launches (bench.py's roofline figure)
  static const int kRing = 256;
  bool timing = false;
  cudaEvent_t ev0[kRing], ev1[kRing];
  bool ev_ready = false;
  int64_t ev_calls = 0;
};

#define CUDA_TRY(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { cudaGetLastError(); return QLP_BLS_ECUDA; } } while (0)
#define QLP_TRY(x) do { int r_ = (x); if (r_ != 0) return r_; } while (0)

static int launch_ok(qlp_bls_ctx* ctx) {
  ctx->launches++;
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? 0 : QLP_BLS_ECUDA;
}

extern "C" void qlp_bls_default_config(qlp_bls_config* cfg) {
  if (!cfg) return;
  memset(cfg, 0, sizeof(*cfg));
  cfg->struct_bytes = (uint32_t)sizeof(qlp_bls_config);
  cfg->device = 0;
  cfg->samples_per_peak = 2.0;
  cfg->dlogq = 0.1;
  cfg->noverlap = 3;
  cfg->top_k = 3;
  cfg->qmin_fac = 0.5;
  cfg->qmax_fac = 2.0;
  cfg->a_over_rstar_min = 2.0;
  cfg->sector_days = 27.4;
  cfg->flags = 0;
}

// O1.9: duration ladder in fine bins.
static int build_widths(const qlp_bls_config& c, int32_t* M, int cap) {
  int J = (int)floor(log(c.qmax_fac / c.qmin_fac) / log(1.0 + c.dlogq)) + 1;
  int n = 0;
  double x = 1.0;
  for (int j = 0; j < J; ++j) {
    int m = (int)floor((double)c.noverlap * x + 0.5);
    if (n == 0 || M[n - 1] != m) {
      if (n >= cap) return -1;
      M[n++] = m;
    }
    x = x * (1.0 + c.dlogq);
  }
  return n;
}

extern "C" int qlp_bls_create(const qlp_bls_config* cfg, qlp_bls_ctx** out) {
  if (!cfg || !out) return QLP_BLS_EINVAL;
  *out = nullptr;
  if (cfg->struct_bytes != sizeof(qlp_bls_config)) return QLP_BLS_EINVAL;
  if (!(cfg->samples_per_peak > 0.0) || !(cfg->dlogq > 0.0) || cfg->noverlap < 1 || cfg->noverlap > kMaxWidth ||
      !(cfg->qmin_fac > 0.0) || !(cfg->qmax_fac >= cfg->qmin_fac) || !(cfg->a_over_rstar_min > 0.0) ||
      !(cfg->sector_days > 0.0) || cfg->top_k < 1 || cfg->top_k > kMaxTopK ||
      !(cfg->max_period_days >= 0.0) || cfg->max_freq < 0 || cfg->max_freq == 1 ||
      (cfg->flags & ~3u) != 0u || cfg->reserved_ != 0u)   // reserved bits must be 0, so that they can get a meaning
    return QLP_BLS_EINVAL;
  qlp_bls_ctx* ctx = new (std::nothrow) qlp_bls_ctx();
  if (!ctx) return QLP_BLS_ENOMEM;
  ctx->cfg = *cfg;
  ctx->n_widths = build_widths(*cfg, ctx->widths, 32);
  if (ctx->n_widths <= 0) { delete ctx; return QLP_BLS_EINVAL; }
  Params& p = ctx->prm;
  p.samples_per_peak = cfg->samples_per_peak; p.dlogq = cfg->dlogq; p.qmin_fac = cfg->qmin_fac;
  p.qmax_fac = cfg->qmax_fac; p.a_over_rstar_min = cfg->a_over_rstar_min; p.sector_days = cfg->sector_days;
  p.noverlap = cfg->noverlap; p.top_k = cfg->top_k;
  p.max_period_days = cfg->max_period_days; p.max_freq = cfg->max_freq;
  p.uniform_freq = (cfg->flags & 2u) ? 1 : 0;
  p.wmask = 0; p.max_width = 0; p.min_width = ctx->widths[0];
  for (int i = 0; i < ctx->n_widths; ++i) {
    int m = ctx->widths[i];
    if (m < 1 || m > kMaxWidth) { delete ctx; return QLP_BLS_EINVAL; }
    p.wmask |= 1u << m;
    if (m > p.max_width) p.max_width = m;
    if (m < p.min_width) p.min_width = m;
  }
  // every box must be narrower than the coarsest histogram: nb >= noverlap pi a_min / qmin_fac
  if (!((double)cfg->noverlap * QLP_PI * cfg->a_over_rstar_min / cfg->qmin_fac > (double)p.max_width + 1.0)) {
    delete ctx; return QLP_BLS_EINVAL;
  }
  ctx->device = cfg->device;
  if (cudaSetDevice(ctx->device) != cudaSuccess) { cudaGetLastError(); delete ctx; return QLP_BLS_ECUDA; }
  int n_sm = 0;
  if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, ctx->device) != cudaSuccess || n_sm <= 0) {
    cudaGetLastError(); delete ctx; return QLP_BLS_ECUDA;
  }
  ctx->n_sm = n_sm;
  // each instantiation gets the dynamic shared memory of the largest class that uses it
  auto smem_for_cols = [](int cols) {
    int m = 0;
    for (int c = 0; c < kNumClasses; ++c)
      if (class_cols(c) == cols && class_smem_bytes(c) > m) m = class_smem_bytes(c);
    return m;
  };
  bool attr_ok = true;
#define QLP_ATTR(CT_)                                                                                                \
  attr_ok = attr_ok &&                                                                                               \
            cudaFuncSetAttribute(foldscan_kernel<11, CT_, kPaperMask>, cudaFuncAttributeMaxDynamicSharedMemorySize,  \
                                 smem_for_cols(CT_)) == cudaSuccess &&                                               \
            cudaFuncSetAttribute(foldscan_kernel<16, CT_, 0u>, cudaFuncAttributeMaxDynamicSharedMemorySize,          \
                                 smem_for_cols(CT_)) == cudaSuccess
  attr_ok = attr_ok &&
            cudaFuncSetAttribute(fit_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kFitSmemBytes) == cudaSuccess &&
            cudaFuncSetAttribute(fit_kernel<kFitCluster>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 kFitSmemBytes) == cudaSuccess;
  QLP_ATTR(128); QLP_ATTR(64); QLP_ATTR(32); QLP_ATTR(16); QLP_ATTR(8); QLP_ATTR(4); QLP_ATTR(2); QLP_ATTR(1);
  if (!attr_ok ||
      cudaFuncSetAttribute(snr_kernel<kSnrThreads>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSel * 256 * 4) != cudaSuccess ||
      cudaFuncSetAttribute(snr_kernel<kSnrThreadsLong>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSel * 256 * 4) != cudaSuccess) {
    cudaGetLastError(); delete ctx; return QLP_BLS_ECUDA;
  }
  if (cudaMallocHost((void**)&ctx->totals_host, 8 * sizeof(int64_t)) != cudaSuccess) {
    cudaGetLastError(); delete ctx; return QLP_BLS_ENOMEM;
  }
  if (ctx->totals_dev.ensure(8 * sizeof(int64_t)) != 0) { cudaFreeHost(ctx->totals_host); delete ctx; return QLP_BLS_ENOMEM; }
  *out = ctx;
  return QLP_BLS_OK;
}

extern "C" int qlp_bls_destroy(qlp_bls_ctx* ctx) {
  if (!ctx) return QLP_BLS_OK;
  cudaSetDevice(ctx->device);
  DevBuf* bufs[] = {&ctx->pts, &ctx->prep, &ctx->kb, &ctx->cnt, &ctx->off, &ctx->counters, &ctx->star_bins,
                    &ctx->totals_dev, &ctx->fit_cnt, &ctx->fit_off, &ctx->fit_work, &ctx->fit_chunk, &ctx->fit_list, &ctx->class_ctr, &ctx->star_order, &ctx->h_row[0], &ctx->h_t[0], &ctx->h_y[0], &ctx->h_dy[0], &ctx->h_rho[0],
                    &ctx->h_row[1], &ctx->h_t[1], &ctx->h_y[1], &ctx->h_dy[1], &ctx->h_rho[1], &ctx->h_grid,
                    &ctx->h_fptr, &ctx->h_sr, &ctx->h_best, &ctx->h_peaks, &ctx->h_stats, &ctx->h_fits, &ctx->h_pink};
  for (DevBuf* b : bufs) b->release();
  if (ctx->totals_host) cudaFreeHost(ctx->totals_host);
  for (int i = 0; i < 2; ++i) if (ctx->row_tmp[i]) cudaFreeHost(ctx->row_tmp[i]);
  if (ctx->fork_ready) {
    for (int i = 0; i < qlp_bls_ctx::kSide; ++i) { cudaStreamDestroy(ctx->side[i]); cudaEventDestroy(ctx->side_done[i]); }
    cudaEventDestroy(ctx->fork_ev);
  }
  if (ctx->copy_ready) {
    cudaStreamDestroy(ctx->copy_stream);
    for (int i = 0; i < 2; ++i) { cudaEventDestroy(ctx->h2d_done[i]); cudaEventDestroy(ctx->set_free[i]); }
  }
  if (ctx->ev_ready)
    for (int i = 0; i < qlp_bls_ctx::kRing; ++i) { cudaEventDestroy(ctx->ev0[i]); cudaEventDestroy(ctx->ev1[i]); }
  delete ctx;
  return QLP_BLS_OK;
}

extern "C" const char* qlp_bls_strerror(int code) {
  switch (code) {
    case QLP_BLS_OK: return "ok";
    case QLP_BLS_EINVAL: return "invalid argument";
    case QLP_BLS_ENOMEM: return "out of memory";
    case QLP_BLS_ECUDA: return "CUDA error";
    case QLP_BLS_EUNSUPPORTED: return "unsupported";
    case QLP_BLS_EVALIDATION: return "input validation failed";
    case QLP_BLS_ETOOLARGE: return "batch exceeds the static scratch of the no-allocation entry point";
    default: return "unknown status";
  }
}

extern "C" int64_t qlp_bls_launch_count(const qlp_bls_ctx* ctx) { return ctx ? ctx->launches : 0; }

extern "C" int qlp_bls_widths(const qlp_bls_ctx* ctx, int32_t* m, int32_t cap) {
  if (!ctx || !m) return QLP_BLS_EINVAL;
  int n = ctx->n_widths < cap ? ctx->n_widths : cap;
  for (int i = 0; i < n; ++i) m[i] = ctx->widths[i];
  return ctx->n_widths;
}

extern "C" int qlp_bls_fold_timing(qlp_bls_ctx* ctx, int32_t enable) {
  if (!ctx) return QLP_BLS_EINVAL;
  CUDA_TRY(cudaSetDevice(ctx->device));
  if (enable && !ctx->ev_ready) {
    for (int i = 0; i < qlp_bls_ctx::kRing; ++i) {
      CUDA_TRY(cudaEventCreate(&ctx->ev0[i]));
      CUDA_TRY(cudaEventCreate(&ctx->ev1[i]));
    }
    ctx->ev_ready = true;
  }
  ctx->timing = enable != 0;
  ctx->ev_calls = 0;
  QLP_TRY(ctx->class_ctr.ensure((kNumClasses * kClassCtr + 2) * 8));
  CUDA_TRY(cudaMemset(ctx->class_ctr.p, 0, (kNumClasses * kClassCtr + 2) * 8));
  return QLP_BLS_OK;
}

extern "C" int qlp_bls_fold_class_counters(qlp_bls_ctx* ctx, uint64_t* out) {
  if (!ctx || !out) return QLP_BLS_EINVAL;
  CUDA_TRY(cudaSetDevice(ctx->device));
  if (!ctx->class_ctr.p) { memset(out, 0, kNumClasses * 5 * 8); return QLP_BLS_OK; }
  unsigned long long h[kNumClasses * kClassCtr];
  CUDA_TRY(cudaDeviceSynchronize());
  CUDA_TRY(cudaMemcpy(h, ctx->class_ctr.p, sizeof(h), cudaMemcpyDeviceToHost));
  for (int c = 0; c < kNumClasses; ++c)
    for (int i = 0; i < 5; ++i) out[c * 5 + i] = h[c * kClassCtr + i];
  return QLP_BLS_OK;
}

extern "C" int qlp_bls_fit_work(qlp_bls_ctx* ctx, uint64_t* out) {
  if (!ctx || !out) return QLP_BLS_EINVAL;
  out[0] = out[1] = 0;
  if (!ctx->class_ctr.p) return QLP_BLS_OK;
  CUDA_TRY(cudaSetDevice(ctx->device));
  CUDA_TRY(cudaDeviceSynchronize());
  CUDA_TRY(cudaMemcpy(out, (unsigned long long*)ctx->class_ctr.p + kNumClasses * kClassCtr, 16, cudaMemcpyDeviceToHost));
  return QLP_BLS_OK;
}

extern "C" int qlp_bls_fold_phase_clocks(qlp_bls_ctx* ctx, uint64_t* clocks) {
  if (!ctx || !clocks) return QLP_BLS_EINVAL;
  uint64_t all[kNumClasses * 5];
  QLP_TRY(qlp_bls_fold_class_counters(ctx, all));
  for (int i = 0; i < 3; ++i) {
    clocks[i] = 0;
    for (int c = 0; c < kNumClasses; ++c) clocks[i] += all[c * 5 + i];
  }
  return QLP_BLS_OK;
}

extern "C" int qlp_bls_fold_elapsed_ms(qlp_bls_ctx* ctx, int32_t* n_calls, double* total_ms) {
  if (!ctx || !n_calls || !total_ms || !ctx->ev_ready) return QLP_BLS_EINVAL;
  CUDA_TRY(cudaSetDevice(ctx->device));
  int64_t n = ctx->ev_calls < qlp_bls_ctx::kRing ? ctx->ev_calls : qlp_bls_ctx::kRing;
  double sum = 0.0;
  for (int64_t i = 0; i < n; ++i) {
    float ms = 0.f;
    CUDA_TRY(cudaEventSynchronize(ctx->ev1[i]));
    CUDA_TRY(cudaEventElapsedTime(&ms, ctx->ev0[i], ctx->ev1[i]));
    sum += ms;
  }
  *n_calls = (int32_t)n;
  *total_ms = sum;
  return QLP_BLS_OK;
}

extern "C" int qlp_bls_debug_set_path(qlp_bls_ctx* ctx, int32_t path) {
  if (!ctx || path < 0 || path > kNumClasses) return QLP_BLS_EINVAL;
  ctx->force_path = path;
  return QLP_BLS_OK;
}

// flags bit0: count invalid inputs on the device; one synchronising read-back (totals_host[3])
static int run_validation(qlp_bls_ctx* ctx, int which, int64_t n_stars, const int64_t* row_ptr, const double* t,
                          const double* y, const double* dy, cudaStream_t st) {
  if (!(ctx->cfg.flags & 1u) || n_stars == 0) return 0;
  unsigned long long* bad = (unsigned long long*)ctx->totals_dev.p + 3;
  CUDA_TRY(cudaMemsetAsync(bad, 0, 8, st));
  validate_kernel<<<(unsigned)n_stars, 256, 0, st>>>(which, n_stars, row_ptr, t, y, dy, bad);
  QLP_TRY(launch_ok(ctx));
  CUDA_TRY(cudaMemcpyAsync(ctx->totals_host + 3, bad, 8, cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  return ctx->totals_host[3] != 0 ? QLP_BLS_EVALIDATION : 0;
}

// ---- S1 -----------------------------------------------------------------------------------------
extern "C" int qlp_bls_grid(qlp_bls_ctx* ctx, int64_t n_stars, const int64_t* row_ptr, const double* t,
                            const double* rho, const double* rstar, qlp_bls_star_grid* grid, int64_t* freq_ptr,
                            int64_t* total_freq, int64_t* total_bins, void* cuda_stream) {
  NvtxRange nvtx_range("qlp_bls_grid");
  (void)rstar;  // R* cancels out of a/R* = (G rho P^2 / 3 pi)^(1/3): DESIGN.md reading A8
  if (!ctx || n_stars < 0 || !row_ptr || !freq_ptr || !total_freq || !total_bins) return QLP_BLS_EINVAL;
  if (n_stars > 0 && (!t || !rho || !grid)) return QLP_BLS_EINVAL;
  if (n_stars > 0x7fffffff) return QLP_BLS_EUNSUPPORTED;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  CUDA_TRY(cudaSetDevice(ctx->device));
  QLP_TRY(ctx->star_bins.ensure((size_t)(n_stars + 1) * 8));
  QLP_TRY(run_validation(ctx, 0, n_stars, row_ptr, t, nullptr, nullptr, st));
  if (n_stars > 0) {
    grid_kernel<<<(unsigned)n_stars, 256, 0, st>>>(ctx->prm, n_stars, row_ptr, t, rho, grid,
                                                  (unsigned long long*)ctx->star_bins.p);
    QLP_TRY(launch_ok(ctx));
  }
  int64_t* totals = (int64_t*)ctx->totals_dev.p;
  freq_scan_kernel<<<1, 1024, 0, st>>>(n_stars, grid, (const unsigned long long*)ctx->star_bins.p, freq_ptr, totals);
  QLP_TRY(launch_ok(ctx));
  CUDA_TRY(cudaMemcpyAsync(ctx->totals_host, totals, 2 * sizeof(int64_t), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  *total_freq = ctx->totals_host[0];
  *total_bins = ctx->totals_host[1];
  ctx->grid_row_ptr = row_ptr; ctx->grid_n_stars = n_stars;
  return QLP_BLS_OK;
}

// number of points of the batch: always read from the device (8 bytes, one stream synchronisation).  The workspace
// is sized from it, so nothing cached under a pointer that a caching allocator may hand out again is trusted.
static int batch_points(qlp_bls_ctx* ctx, int64_t n_stars, const int64_t* row_ptr, cudaStream_t st, int64_t* n_points) {
  CUDA_TRY(cudaMemcpyAsync(ctx->totals_host + 2, row_ptr + n_stars, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  *n_points = ctx->totals_host[2];
  return 0;
}

// S0 into the context workspace
static int run_prep(qlp_bls_ctx* ctx, int64_t n_stars, const int64_t* row_ptr, const double* t, const double* y,
                    const double* dy, const qlp_bls_star_grid* grid, cudaStream_t st) {
  int64_t n_points = 0;
  ctx->prep_valid = false;
  QLP_TRY(batch_points(ctx, n_stars, row_ptr, st, &n_points));
  if (n_points < 0) return QLP_BLS_EINVAL;
  QLP_TRY(ctx->pts.ensure((size_t)(n_points + 1) * sizeof(Point)));
  QLP_TRY(ctx->prep.ensure((size_t)(n_stars + 1) * sizeof(StarPrep)));
  prep_kernel<<<(unsigned)n_stars, 256, 0, st>>>(ctx->prm, n_stars, row_ptr, t, y, dy, grid, (Point*)ctx->pts.p,
                                                (StarPrep*)ctx->prep.p);
  QLP_TRY(launch_ok(ctx));
  qlp_bls_ctx::PrepKey k;
  k.row_ptr = row_ptr; k.t = t; k.y = y; k.dy = dy; k.grid = grid; k.n_stars = n_stars;
  ctx->prep_key = k;
  ctx->prep_valid = true;
  return 0;
}

// side streams for launches that are independent of one another (tile classes; large and small fits)
static int ensure_side_streams(qlp_bls_ctx* ctx) {
  if (ctx->fork_ready) return 0;
  for (int i = 0; i < qlp_bls_ctx::kSide; ++i) {
    CUDA_TRY(cudaStreamCreateWithFlags(&ctx->side[i], cudaStreamNonBlocking));
    CUDA_TRY(cudaEventCreateWithFlags(&ctx->side_done[i], cudaEventDisableTiming));
  }
  CUDA_TRY(cudaEventCreateWithFlags(&ctx->fork_ev, cudaEventDisableTiming));
  ctx->fork_ready = true;
  return 0;
}

// ---- S0 + S2 + S3 ---------------------------------------------------------------------------------
extern "C" int qlp_bls_spectrum(qlp_bls_ctx* ctx, int64_t n_stars, const int64_t* row_ptr, const double* t,
                                const double* y, const double* dy, const qlp_bls_star_grid* grid,
                                const int64_t* freq_ptr, float* sr, uint32_t* best, void* cuda_stream) {
  NvtxRange nvtx_range("qlp_bls_spectrum");
  if (!ctx || n_stars < 0 || !row_ptr || !freq_ptr) return QLP_BLS_EINVAL;
  if (n_stars == 0) return QLP_BLS_OK;
  if (!t || !y || !dy || !grid || !sr || !best) return QLP_BLS_EINVAL;
  if (n_stars > 0x7fffffff) return QLP_BLS_EUNSUPPORTED;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  CUDA_TRY(cudaSetDevice(ctx->device));
  QLP_TRY(run_validation(ctx, 1, n_stars, row_ptr, t, y, dy, st));
  QLP_TRY(run_prep(ctx, n_stars, row_ptr, t, y, dy, grid, st));
  QLP_TRY(ctx->kb.ensure((size_t)n_stars * kNumClasses * 8));
  QLP_TRY(ctx->cnt.ensure((size_t)n_stars * kNumClasses * 8));
  QLP_TRY(ctx->off.ensure((size_t)(n_stars + 1) * kNumClasses * 8));
  QLP_TRY(ctx->counters.ensure(kNumClasses * 8));
  int64_t* kb = (int64_t*)ctx->kb.p;
  int64_t* cnt = (int64_t*)ctx->cnt.p;
  int64_t* off = (int64_t*)ctx->off.p;
  unsigned long long* counters = (unsigned long long*)ctx->counters.p;
  CUDA_TRY(cudaMemsetAsync(counters, 0, kNumClasses * 8, st));
  // per-phase clock counters of the fold/scan kernel (only while fold timing is on)
  unsigned long long* phase_base = (ctx->timing && ctx->class_ctr.p) ? (unsigned long long*)ctx->class_ctr.p : nullptr;
  tile_bounds_kernel<<<(unsigned)((n_stars + 127) / 128), 128, 0, st>>>(ctx->prm, n_stars, grid, ctx->force_path, kb, cnt);
  QLP_TRY(launch_ok(ctx));
  tile_scan_kernel<<<kNumClasses, 1024, 0, st>>>(n_stars, cnt, off);
  QLP_TRY(launch_ok(ctx));
  const int slot = (int)(ctx->ev_calls % qlp_bls_ctx::kRing);
  if (ctx->timing) CUDA_TRY(cudaEventRecord(ctx->ev0[slot], st));
  // The class kernels are independent: they go to side streams so that the CTAs of the next class fill the SMs
  // that the tail of the previous one leaves idle (each launch is persistent: any number of resident CTAs works).
  QLP_TRY(ensure_side_streams(ctx));
  CUDA_TRY(cudaEventRecord(ctx->fork_ev, st));
  for (int i = 0; i < qlp_bls_ctx::kSide; ++i) CUDA_TRY(cudaStreamWaitEvent(ctx->side[i], ctx->fork_ev, 0));
  cudaStream_t user_st = st;
  for (int c = 0; c < kNumClasses; ++c) {
    st = (c % (qlp_bls_ctx::kSide + 1) == 0) ? user_st : ctx->side[c % (qlp_bls_ctx::kSide + 1) - 1];
    const size_t smem = (size_t)class_smem_bytes(c);
    const int per_sm = class_ctas_per_sm(c);
    const unsigned nblk = (unsigned)(ctx->n_sm * per_sm);
    const int64_t* off_c = off + (int64_t)c * (n_stars + 1);
    // the paper's ladder {3..11} is compiled in; other ladders and the frequency-uniform comparison grid (O1.10c)
    // run the kernels with the run-time ladder, the only ones that know that grid
    const bool generic = ctx->prm.wmask != kPaperMask || ctx->prm.uniform_freq != 0;
#define QLP_LAUNCH(MW_, CT_, WM_)                                                                                          \
  foldscan_kernel<MW_, CT_, WM_><<<nblk, kThreads, smem, st>>>(ctx->prm, c, n_stars, row_ptr, (const Point*)ctx->pts.p,    \
                                                         (const StarPrep*)ctx->prep.p, grid, freq_ptr, off_c, kb,    \
                                                         counters + c, sr, best,                               \
                                                         phase_base ? phase_base + c * kClassCtr : nullptr)
#define QLP_LAUNCH_MW(CT_) do { if (generic) QLP_LAUNCH(16, CT_, 0u); else QLP_LAUNCH(11, CT_, kPaperMask); } while (0)
    switch (class_cols(c)) {
      case 128: QLP_LAUNCH_MW(128); break;
      case 64: QLP_LAUNCH_MW(64); break;
      case 32: QLP_LAUNCH_MW(32); break;
      case 16: QLP_LAUNCH_MW(16); break;
      case 8: QLP_LAUNCH_MW(8); break;
      case 4: QLP_LAUNCH_MW(4); break;
      case 2: QLP_LAUNCH_MW(2); break;
      default: QLP_LAUNCH_MW(1); break;
    }
    QLP_TRY(launch_ok(ctx));
  }
  st = user_st;
  for (int i = 0; i < qlp_bls_ctx::kSide; ++i) {
    CUDA_TRY(cudaEventRecord(ctx->side_done[i], ctx->side[i]));
    CUDA_TRY(cudaStreamWaitEvent(st, ctx->side_done[i], 0));
  }
  if (ctx->timing) { CUDA_TRY(cudaEventRecord(ctx->ev1[slot], st)); ctx->ev_calls++; }
  return QLP_BLS_OK;
}

// ---- S4 -------------------------------------------------------------------------------------------
extern "C" int qlp_bls_snr(qlp_bls_ctx* ctx, int64_t n_stars, const int64_t* row_ptr, const double* t, const double* y,
                           const double* dy, const qlp_bls_star_grid* grid, const int64_t* freq_ptr, const float* sr,
                           const uint32_t* best, float* snr, qlp_bls_peak* peaks, void* cuda_stream) {
  NvtxRange nvtx_range("qlp_bls_snr");
  if (!ctx || n_stars < 0 || !row_ptr || !freq_ptr) return QLP_BLS_EINVAL;
  if (n_stars == 0) return QLP_BLS_OK;
  if (!t || !y || !dy || !grid || !sr || !best || !peaks) return QLP_BLS_EINVAL;
  if (n_stars > 0x7fffffff) return QLP_BLS_EUNSUPPORTED;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  CUDA_TRY(cudaSetDevice(ctx->device));
  {  // S0 again only if the workspace does not hold these arrays' records (see the header)
    qlp_bls_ctx::PrepKey k;
    k.row_ptr = row_ptr; k.t = t; k.y = y; k.dy = dy; k.grid = grid; k.n_stars = n_stars;
    if (!(ctx->prep_valid && ctx->prep_key == k)) QLP_TRY(run_prep(ctx, n_stars, row_ptr, t, y, dy, grid, st));
  }
  QLP_TRY(ctx->star_order.ensure((size_t)n_stars * sizeof(int32_t)));
  star_order_kernel<<<1, 1024, 0, st>>>(n_stars, grid, (int32_t*)ctx->star_order.p);
  QLP_TRY(launch_ok(ctx));
  // two launches side by side: the long grids with 1,024 threads per star on a side stream, the rest with 256
  QLP_TRY(ensure_side_streams(ctx));
  CUDA_TRY(cudaEventRecord(ctx->fork_ev, st));
  CUDA_TRY(cudaStreamWaitEvent(ctx->side[0], ctx->fork_ev, 0));
  snr_kernel<kSnrThreadsLong><<<(unsigned)n_stars, kSnrThreadsLong, kMaxSel * 256 * 4, ctx->side[0]>>>(
      ctx->prm, n_stars, row_ptr, (const Point*)ctx->pts.p, (const StarPrep*)ctx->prep.p, grid, freq_ptr, sr, best,
      snr, peaks, (const int32_t*)ctx->star_order.p);
  QLP_TRY(launch_ok(ctx));
  snr_kernel<kSnrThreads><<<(unsigned)n_stars, kSnrThreads, kMaxSel * 256 * 4, st>>>(
      ctx->prm, n_stars, row_ptr, (const Point*)ctx->pts.p, (const StarPrep*)ctx->prep.p, grid, freq_ptr, sr, best,
      snr, peaks, (const int32_t*)ctx->star_order.p);
  QLP_TRY(launch_ok(ctx));
  CUDA_TRY(cudaEventRecord(ctx->side_done[0], ctx->side[0]));
  CUDA_TRY(cudaStreamWaitEvent(st, ctx->side_done[0], 0));
  return QLP_BLS_OK;
}

// ---- O7: per-peak statistics --------------------------------------------------------------------------
extern "C" int qlp_bls_peak_stats(qlp_bls_ctx* ctx, int64_t n_stars, const int64_t* row_ptr, const double* t,
                                  const double* y, const double* dy, const qlp_bls_peak* peaks,
                                  qlp_bls_transit_stats* stats, void* cuda_stream) {
  NvtxRange nvtx_range("qlp_bls_peak_stats");
  if (!ctx || n_stars < 0) return QLP_BLS_EINVAL;
  if (n_stars == 0) return QLP_BLS_OK;
  if (!row_ptr || !t || !y || !dy || !peaks || !stats) return QLP_BLS_EINVAL;
  if (n_stars * ctx->prm.top_k > 0x7fffffff) return QLP_BLS_EUNSUPPORTED;
  CUDA_TRY(cudaSetDevice(ctx->device));
  peak_stats_kernel<<<(unsigned)(n_stars * ctx->prm.top_k), 256, 0, (cudaStream_t)cuda_stream>>>(
      n_stars, ctx->prm.top_k, row_ptr, t, y, dy, peaks, stats);
  return launch_ok(ctx);
}

// ---- O8: trapezoid fit of every peak --------------------------------------------------------------------
extern "C" int qlp_bls_trapezoid_fit(qlp_bls_ctx* ctx, int64_t n_stars, const int64_t* row_ptr, const double* t,
                                     const double* y, const double* dy, const qlp_bls_peak* peaks,
                                     qlp_bls_trapezoid* fits, void* cuda_stream) {
  NvtxRange nvtx_range("qlp_bls_trapezoid_fit");
  if (!ctx || n_stars < 0) return QLP_BLS_EINVAL;
  if (n_stars == 0) return QLP_BLS_OK;
  if (!row_ptr || !t || !y || !dy || !peaks || !fits) return QLP_BLS_EINVAL;
  const int64_t n_items = n_stars * ctx->prm.top_k;
  if (n_items > 0x7fffffff) return QLP_BLS_EUNSUPPORTED;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  CUDA_TRY(cudaSetDevice(ctx->device));
  int rc = ctx->fit_cnt.ensure((size_t)n_items * sizeof(int64_t));
  if (rc == 0) rc = ctx->fit_off.ensure((size_t)(n_items + 2) * sizeof(int64_t));
  if (rc == 0) rc = ctx->fit_chunk.ensure((size_t)n_items * kFitCluster * sizeof(int32_t));
  if (rc == 0) rc = ctx->fit_list.ensure((size_t)n_items * 2 * sizeof(int32_t) + 16);
  if (rc != 0) return rc;
  int64_t* cnt = (int64_t*)ctx->fit_cnt.p;
  int64_t* off = (int64_t*)ctx->fit_off.p;
  int32_t* chunk = (int32_t*)ctx->fit_chunk.p;
  int32_t* list = (int32_t*)ctx->fit_list.p;
  // two counters (items per size class) behind the lists, 8-byte aligned
  unsigned long long* list_n = (unsigned long long*)((char*)ctx->fit_list.p + (((size_t)n_items * 2 * sizeof(int32_t) + 7) & ~(size_t)7));
  CUDA_TRY(cudaMemsetAsync(list_n, 0, 16, st));
  fit_count_kernel<<<(unsigned)n_items, kFitCountThreads, 0, st>>>(n_items, ctx->prm.top_k, row_ptr, t, peaks, cnt, chunk, list, list_n);
  rc = launch_ok(ctx);
  if (rc != 0) return rc;
  fit_scan_kernel<<<1, 1024, 0, st>>>(n_items, cnt, off, off + n_items + 1);
  rc = launch_ok(ctx);
  if (rc != 0) return rc;
  CUDA_TRY(cudaMemcpyAsync(ctx->totals_host + 2, off + n_items, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaMemcpyAsync(ctx->totals_host + 4, list_n, 16, cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  const int64_t total = ctx->totals_host[2];
  const int64_t n_single = ctx->totals_host[4], n_cluster = ctx->totals_host[5];
  if (total < 0 || n_single < 0 || n_cluster < 0 || n_single + n_cluster != n_items) return QLP_BLS_ECUDA;
  // a single window never holds more points than its star, and a star is capped at QLP_BLS_MAX_POINTS < 2^31
  rc = ctx->fit_work.ensure((size_t)(total > 0 ? total : 1) * 3 * sizeof(double));
  if (rc != 0) return rc;
  // while fold timing is on, the fit kernels count their work (bench.py's roofline entry): class_ctr[72..73]
  unsigned long long* fit_ctr = (ctx->timing && ctx->class_ctr.p) ? (unsigned long long*)ctx->class_ctr.p + kNumClasses * kClassCtr : nullptr;
  // Large windows first, on a side stream: one cluster of kFitCluster CTAs per item; the single-CTA fits of the small
  // windows run beside them on the caller's stream.  Both grids are exact (the size classes were counted above).
  QLP_TRY(ensure_side_streams(ctx));
  CUDA_TRY(cudaEventRecord(ctx->fork_ev, st));
  CUDA_TRY(cudaStreamWaitEvent(ctx->side[0], ctx->fork_ev, 0));
  if (n_cluster > 0) {
    cudaLaunchConfig_t lc = {};
    lc.gridDim = dim3((unsigned)(n_cluster * kFitCluster));
    lc.blockDim = dim3(kFitThreads);
    lc.dynamicSmemBytes = kFitSmemBytes;
    lc.stream = ctx->side[0];
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = kFitCluster; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    lc.attrs = at; lc.numAttrs = 1;
    CUDA_TRY(cudaLaunchKernelEx(&lc, fit_kernel<kFitCluster>, n_items, (int)ctx->prm.top_k, row_ptr, t, y, dy, peaks,
                                (const int64_t*)off, (const int32_t*)chunk, (const int32_t*)(list + n_items), n_cluster,
                                (double*)ctx->fit_work.p, fits, fit_ctr));
    QLP_TRY(launch_ok(ctx));
  }
  if (n_single > 0) {
    fit_kernel<1><<<(unsigned)n_single, kFitThreads, kFitSmemBytes, st>>>(n_items, ctx->prm.top_k, row_ptr, t, y, dy, peaks,
                                                                        off, chunk, list, n_single,
                                                                        (double*)ctx->fit_work.p, fits, fit_ctr);
    QLP_TRY(launch_ok(ctx));
  }
  CUDA_TRY(cudaEventRecord(ctx->side_done[0], ctx->side[0]));
  CUDA_TRY(cudaStreamWaitEvent(st, ctx->side_done[0], 0));
  return QLP_BLS_OK;
}

// ---- O9: noise estimates, S/N_pink, detection criteria ------------------------------------------------
extern "C" int qlp_bls_pink_noise(qlp_bls_ctx* ctx, int64_t n_stars, const int64_t* row_ptr, const double* t,
                                  const double* y, const qlp_bls_peak* peaks, const qlp_bls_trapezoid* fits,
                                  qlp_bls_pink* pink, void* cuda_stream) {
  NvtxRange nvtx_range("qlp_bls_pink_noise");
  if (!ctx || n_stars < 0) return QLP_BLS_EINVAL;
  if (n_stars == 0) return QLP_BLS_OK;
  if (!row_ptr || !t || !y || !peaks || !fits || !pink) return QLP_BLS_EINVAL;
  if (n_stars * ctx->prm.top_k > 0x7fffffff) return QLP_BLS_EUNSUPPORTED;
  CUDA_TRY(cudaSetDevice(ctx->device));
  pink_kernel<<<(unsigned)(n_stars * ctx->prm.top_k), kPinkThreads, 0, (cudaStream_t)cuda_stream>>>(
      n_stars, ctx->prm.top_k, row_ptr, t, y, peaks, fits, pink);
  return launch_ok(ctx);
}

// ---- whole path from host buffers -------------------------------------------------------------------
// Stars are processed in sub-batches: per sub-batch H2D (row_ptr rebased, t, y, dy, rho) -> grid -> spectrum ->
// snr -> D2H of the peak table only.  The H2D of sub-batch i+1 runs on the context's copy stream into the
// second set of staging buffers while sub-batch i is searched, so with pinned host memory only the first
// sub-batch's copy is exposed.  Sub-batch size: enough points to keep the persistent fold kernels busy, small
// enough for several sub-batches per call, and never more than a point budget that keeps the device copies
// small next to 180 GB of HBM.
static int search_host_impl(qlp_bls_ctx* ctx, int64_t n_stars, const int64_t* row_ptr, const double* t,
                            const double* y, const double* dy, const double* rho, const double* rstar,
                            qlp_bls_peak* peaks, qlp_bls_transit_stats* stats, qlp_bls_trapezoid* fits,
                            qlp_bls_pink* pink, qlp_bls_star_grid* grid_out, int64_t* total_freq, void* cuda_stream) {
  (void)rstar;
  if (!ctx || n_stars < 0 || !row_ptr || !peaks) return QLP_BLS_EINVAL;
  if (n_stars > 0 && (!t || !y || !dy || !rho)) return QLP_BLS_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  CUDA_TRY(cudaSetDevice(ctx->device));
  if (total_freq) *total_freq = 0;
  if (n_stars == 0) return QLP_BLS_OK;
  if (!ctx->copy_ready) {
    CUDA_TRY(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
    for (int i = 0; i < 2; ++i) {
      CUDA_TRY(cudaEventCreateWithFlags(&ctx->h2d_done[i], cudaEventDisableTiming));
      CUDA_TRY(cudaEventCreateWithFlags(&ctx->set_free[i], cudaEventDisableTiming));
    }
    ctx->copy_ready = true;
  }
  const int K = ctx->prm.top_k;
  const int64_t n_points = row_ptr[n_stars] - row_ptr[0];
  if (n_points < 0) return QLP_BLS_EINVAL;
  // Sub-batches grow geometrically: the copy of the first one is the only exposed one, so it is small; the search
  // of sub-batch i has to cover the copy of sub-batch i+1, and a search takes several times longer than the copy
  // of its own input (config 2: 24.5 ms against 5.5 ms for 274 MB), so each sub-batch may hold four times the
  // points of the one before.  Few sub-batches: each costs a synchronising grid call and a kernel tail.
  const int64_t kMinPoints = 1ll << 18, kMaxPoints = 256ll << 20;   // 6 MB ... 4 GiB of point records
  const int64_t kStarBudget = 1 << 20;
  std::vector<int64_t> cut(1, 0);   // sub-batch k = stars [cut[k], cut[k+1])
  int64_t n_sub = 0, max_S = 0, max_np = 0;
  {
    int64_t budget = n_points / 24 + 1;
    for (int64_t s0 = 0; s0 < n_stars;) {
      if (budget < kMinPoints) budget = kMinPoints;
      if (budget > kMaxPoints) budget = kMaxPoints;
      int64_t s1 = s0 + 1;
      while (s1 < n_stars && (row_ptr[s1 + 1] - row_ptr[s0]) <= budget && (s1 - s0) < kStarBudget) ++s1;
      if (row_ptr[s1] < row_ptr[s0]) return QLP_BLS_EINVAL;
      const int64_t np = row_ptr[s1] - row_ptr[s0];
      if (s1 - s0 > max_S) max_S = s1 - s0;
      if (np > max_np) max_np = np;
      cut.push_back(s1);
      budget = 4 * (np > budget ? np : budget);
      ++n_sub; s0 = s1;
    }
  }
  for (int i = 0; i < (n_sub > 1 ? 2 : 1); ++i) {
    QLP_TRY(ctx->h_row[i].ensure((size_t)(max_S + 1) * 8));
    QLP_TRY(ctx->h_t[i].ensure((size_t)(max_np + 1) * 8));
    QLP_TRY(ctx->h_y[i].ensure((size_t)(max_np + 1) * 8));
    QLP_TRY(ctx->h_dy[i].ensure((size_t)(max_np + 1) * 8));
    QLP_TRY(ctx->h_rho[i].ensure((size_t)max_S * 8));
  }
  QLP_TRY(ctx->h_grid.ensure((size_t)max_S * sizeof(qlp_bls_star_grid)));
  QLP_TRY(ctx->h_fptr.ensure((size_t)(max_S + 1) * 8));
  QLP_TRY(ctx->h_peaks.ensure((size_t)max_S * K * sizeof(qlp_bls_peak)));
  if (stats) QLP_TRY(ctx->h_stats.ensure((size_t)max_S * K * sizeof(qlp_bls_transit_stats)));
  if (fits || pink) QLP_TRY(ctx->h_fits.ensure((size_t)max_S * K * sizeof(qlp_bls_trapezoid)));
  if (pink) QLP_TRY(ctx->h_pink.ensure((size_t)max_S * K * sizeof(qlp_bls_pink)));
  // pinned, so that the copy stream's H2D of the rebased row_ptr is asynchronous like the others
  if (ctx->row_tmp_cap < (size_t)(max_S + 1)) {
    for (int i = 0; i < 2; ++i) {
      if (ctx->row_tmp[i]) cudaFreeHost(ctx->row_tmp[i]);
      ctx->row_tmp[i] = nullptr;
    }
    ctx->row_tmp_cap = 0;
    const size_t want = (size_t)(max_S + 1) + (size_t)(max_S + 1) / 8;
    for (int i = 0; i < 2; ++i)
      if (cudaMallocHost((void**)&ctx->row_tmp[i], want * 8) != cudaSuccess) { cudaGetLastError(); return QLP_BLS_ENOMEM; }
    ctx->row_tmp_cap = want;
  }
  int64_t** row_tmp = ctx->row_tmp;
  struct Sub { int64_t s0, s1; };
  int64_t sub_idx = 0;
  auto next_sub = [&](int64_t) { const Sub sb{cut[sub_idx], cut[sub_idx + 1]}; ++sub_idx; return sb; };
  // enqueue the H2D of one sub-batch on the copy stream into staging set `set`
  auto issue_h2d = [&](const Sub& sb, int set, bool wait_free) -> int {
    const int64_t S = sb.s1 - sb.s0, p0 = row_ptr[sb.s0], np = row_ptr[sb.s1] - p0;
    cudaStream_t cs = ctx->copy_stream;
    if (wait_free) CUDA_TRY(cudaStreamWaitEvent(cs, ctx->set_free[set], 0));
    for (int64_t i = 0; i <= S; ++i) row_tmp[set][i] = row_ptr[sb.s0 + i] - p0;  // rebased to zero
    CUDA_TRY(cudaMemcpyAsync(ctx->h_row[set].p, row_tmp[set], (size_t)(S + 1) * 8, cudaMemcpyHostToDevice, cs));
    CUDA_TRY(cudaMemcpyAsync(ctx->h_t[set].p, t + p0, (size_t)np * 8, cudaMemcpyHostToDevice, cs));
    CUDA_TRY(cudaMemcpyAsync(ctx->h_y[set].p, y + p0, (size_t)np * 8, cudaMemcpyHostToDevice, cs));
    CUDA_TRY(cudaMemcpyAsync(ctx->h_dy[set].p, dy + p0, (size_t)np * 8, cudaMemcpyHostToDevice, cs));
    CUDA_TRY(cudaMemcpyAsync(ctx->h_rho[set].p, rho + sb.s0, (size_t)S * 8, cudaMemcpyHostToDevice, cs));
    CUDA_TRY(cudaEventRecord(ctx->h2d_done[set], cs));
    return 0;
  };
  int rc = 0;
  int64_t tf_sum = 0;
  Sub cur = next_sub(0);
  rc = issue_h2d(cur, 0, false);
  for (int64_t i = 0; rc == 0; ++i) {
    const int set = (int)(i & 1);
    const bool has_next = cur.s1 < n_stars;
    Sub nxt = cur;
    if (has_next) {
      nxt = next_sub(cur.s1);
      // the other set was last read by sub-batch i-1 (if any): its set_free event was recorded then
      if ((rc = issue_h2d(nxt, set ^ 1, i >= 1)) != 0) break;
    }
    const int64_t S = cur.s1 - cur.s0;
    if (cudaStreamWaitEvent(st, ctx->h2d_done[set], 0) != cudaSuccess) { cudaGetLastError(); rc = QLP_BLS_ECUDA; break; }
    const int64_t* d_row = (const int64_t*)ctx->h_row[set].p;
    const double* d_t = (const double*)ctx->h_t[set].p;
    const double* d_y = (const double*)ctx->h_y[set].p;
    const double* d_dy = (const double*)ctx->h_dy[set].p;
    int64_t tf = 0, tb = 0;
    NvtxRange nvtx_range("qlp_bls_host_sub_batch");
    ctx->prep_valid = false;  // staging pointers are reused across sub-batches: the records are another sub-batch's
    rc = qlp_bls_grid(ctx, S, d_row, d_t, (const double*)ctx->h_rho[set].p, nullptr,
                      (qlp_bls_star_grid*)ctx->h_grid.p, (int64_t*)ctx->h_fptr.p, &tf, &tb, st);
    if (rc != 0) break;
    tf_sum += tf;
    if ((rc = ctx->h_sr.ensure((size_t)(tf + 1) * 4)) != 0 || (rc = ctx->h_best.ensure((size_t)(tf + 1) * 4)) != 0) break;
    rc = qlp_bls_spectrum(ctx, S, d_row, d_t, d_y, d_dy, (const qlp_bls_star_grid*)ctx->h_grid.p,
                          (const int64_t*)ctx->h_fptr.p, (float*)ctx->h_sr.p, (uint32_t*)ctx->h_best.p, st);
    if (rc == 0)
      rc = qlp_bls_snr(ctx, S, d_row, d_t, d_y, d_dy, (const qlp_bls_star_grid*)ctx->h_grid.p,
                       (const int64_t*)ctx->h_fptr.p, (const float*)ctx->h_sr.p, (const uint32_t*)ctx->h_best.p,
                       nullptr, (qlp_bls_peak*)ctx->h_peaks.p, st);
    if (rc == 0 && stats)
      rc = qlp_bls_peak_stats(ctx, S, d_row, d_t, d_y, d_dy, (const qlp_bls_peak*)ctx->h_peaks.p,
                              (qlp_bls_transit_stats*)ctx->h_stats.p, st);
    if (rc == 0 && (fits || pink))   // synchronises the stream once (workspace sizing); the next H2D is already queued
      rc = qlp_bls_trapezoid_fit(ctx, S, d_row, d_t, d_y, d_dy, (const qlp_bls_peak*)ctx->h_peaks.p,
                                 (qlp_bls_trapezoid*)ctx->h_fits.p, st);
    if (rc == 0 && pink)
      rc = qlp_bls_pink_noise(ctx, S, d_row, d_t, d_y, (const qlp_bls_peak*)ctx->h_peaks.p,
                              (const qlp_bls_trapezoid*)ctx->h_fits.p, (qlp_bls_pink*)ctx->h_pink.p, st);
    if (rc != 0) break;
    cudaError_t e = cudaEventRecord(ctx->set_free[set], st);
    if (e == cudaSuccess && fits)
      e = cudaMemcpyAsync(fits + cur.s0 * K, ctx->h_fits.p, (size_t)S * K * sizeof(qlp_bls_trapezoid),
                          cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && pink)
      e = cudaMemcpyAsync(pink + cur.s0 * K, ctx->h_pink.p, (size_t)S * K * sizeof(qlp_bls_pink),
                          cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && stats)
      e = cudaMemcpyAsync(stats + cur.s0 * K, ctx->h_stats.p, (size_t)S * K * sizeof(qlp_bls_transit_stats),
                          cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess)
      e = cudaMemcpyAsync(peaks + cur.s0 * K, ctx->h_peaks.p, (size_t)S * K * sizeof(qlp_bls_peak),
                          cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && grid_out)
      e = cudaMemcpyAsync(grid_out + cur.s0, ctx->h_grid.p, (size_t)S * sizeof(qlp_bls_star_grid),
                          cudaMemcpyDeviceToHost, st);
    if (e != cudaSuccess) { cudaGetLastError(); rc = QLP_BLS_ECUDA; break; }
    if (!has_next) break;
    cur = nxt;
  }
  // everything enqueued (or failed): drain both streams before the host buffers go out of scope
  cudaError_t e1 = cudaStreamSynchronize(st), e2 = cudaStreamSynchronize(ctx->copy_stream);
  if (rc == 0 && (e1 != cudaSuccess || e2 != cudaSuccess)) { cudaGetLastError(); rc = QLP_BLS_ECUDA; }
  if (rc == 0 && total_freq) *total_freq = tf_sum;
  return rc;
}

extern "C" int qlp_bls_search_host(qlp_bls_ctx* ctx, int64_t n_stars, const int64_t* row_ptr, const double* t,
                                   const double* y, const double* dy, const double* rho, const double* rstar,
                                   qlp_bls_peak* peaks, qlp_bls_transit_stats* stats, qlp_bls_star_grid* grid_out,
                                   int64_t* total_freq, void* cuda_stream) {
  return search_host_impl(ctx, n_stars, row_ptr, t, y, dy, rho, rstar, peaks, stats, nullptr, nullptr, grid_out,
                          total_freq, cuda_stream);
}

extern "C" int qlp_bls_vet_host(qlp_bls_ctx* ctx, int64_t n_stars, const int64_t* row_ptr, const double* t,
                                const double* y, const double* dy, const double* rho, const double* rstar,
                                qlp_bls_peak* peaks, qlp_bls_transit_stats* stats, qlp_bls_trapezoid* fits,
                                qlp_bls_pink* pink, qlp_bls_star_grid* grid_out, int64_t* total_freq,
                                void* cuda_stream) {
  return search_host_impl(ctx, n_stars, row_ptr, t, y, dy, rho, rstar, peaks, stats, fits, pink, grid_out, total_freq,
                          cuda_stream);
}

// ---- check build: violation counters of the guarded accesses (common.cuh QLP_IN_BOUNDS) -------------------------
extern "C" int qlp_bls_debug_violations(qlp_bls_ctx* ctx, uint64_t* out, int32_t reset) {
  if (!ctx || !out) return QLP_BLS_EINVAL;
#ifdef QLP_BOUNDS_CHECK
  CUDA_TRY(cudaSetDevice(ctx->device));
  CUDA_TRY(cudaDeviceSynchronize());
  unsigned long long h[kChkSlots];
  CUDA_TRY(cudaMemcpyFromSymbol(h, g_qlp_violations, sizeof(h)));
  for (int i = 0; i < kChkSlots; ++i) out[i] = h[i];
  if (reset) {
    memset(h, 0, sizeof(h));
    CUDA_TRY(cudaMemcpyToSymbol(g_qlp_violations, h, sizeof(h)));
  }
  return QLP_BLS_OK;
#else
  (void)reset;
  for (int i = 0; i < kChkSlots; ++i) out[i] = 0;
  return QLP_BLS_EUNSUPPORTED;   // the checks are not compiled into this build
#endif
}

// ---- test-only entry points ---------------------------------------------------------------------------
extern "C" int qlp_bls_debug_freqs(qlp_bls_ctx* ctx, const qlp_bls_star_grid* grid, int64_t star, int64_t k0,
                                   int64_t k1, double* f, int32_t* nb, void* cuda_stream) {
  if (!ctx || !grid || star < 0 || k0 < 0 || k1 < k0) return QLP_BLS_EINVAL;
  if (k1 == k0) return QLP_BLS_OK;
  if (!f || !nb) return QLP_BLS_EINVAL;
  CUDA_TRY(cudaSetDevice(ctx->device));
  int64_t nblk = (k1 - k0 + 255) / 256;
  if (nblk > 4096) nblk = 4096;
  debug_freqs_kernel<<<(unsigned)nblk, 256, 0, (cudaStream_t)cuda_stream>>>(ctx->prm, grid, star, k0, k1, f, nb);
  return launch_ok(ctx);
}

extern "C" int qlp_bls_debug_bins(qlp_bls_ctx* ctx, const int64_t* row_ptr, const double* t,
                                  const qlp_bls_star_grid* grid, int64_t star, int64_t k, int32_t* bin_of_point,
                                  void* cuda_stream) {
  if (!ctx || !row_ptr || !t || !grid || !bin_of_point || star < 0 || k < 0) return QLP_BLS_EINVAL;
  CUDA_TRY(cudaSetDevice(ctx->device));
  debug_bins_kernel<<<256, 256, 0, (cudaStream_t)cuda_stream>>>(ctx->prm, row_ptr, t, grid, star, k, bin_of_point);
  return launch_ok(ctx);
}

extern "C" int qlp_bls_debug_prep(qlp_bls_ctx* ctx, const int64_t* row_ptr, const double* t, const double* y,
                                  const double* dy, const qlp_bls_star_grid* grid, int64_t star, double* tau, float* w,
                                  float* wy, void* cuda_stream) {
  if (!ctx || !row_ptr || !t || !y || !dy || !grid || !tau || !w || !wy || star < 0) return QLP_BLS_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  CUDA_TRY(cudaSetDevice(ctx->device));
  // the prep kernel runs over the whole batch; the caller passes the batch size through the grid call
  if (ctx->grid_row_ptr != row_ptr || ctx->grid_n_stars <= star) return QLP_BLS_EINVAL;
  QLP_TRY(run_prep(ctx, ctx->grid_n_stars, row_ptr, t, y, dy, grid, st));
  debug_prep_kernel<<<64, 256, 0, st>>>(row_ptr, (const Point*)ctx->pts.p, (const StarPrep*)ctx->prep.p, star, tau, w, wy);
  return launch_ok(ctx);
}

// ---- S1 without any allocation --------------------------------------------------------------------------
// qlp_bls_grid_noalloc: the grid stage (grid_kernel + freq_scan_kernel, the kernels of qlp_bls_grid) for callers that
// cannot call cudaMalloc.  The one scratch array of the stage -- the per-star sum of nb_k that grid_kernel writes
// and freq_scan_kernel adds up -- lives in the file-scope device array below instead of the context's workspace.
// Every GPU that loads the library holds these (QLP_BLS_NOALLOC_MAX_STARS + 1) x 8 bytes = 2 MiB until exit.
static __device__ __align__(256) unsigned long long g_noalloc_star_bins[QLP_BLS_NOALLOC_MAX_STARS + 1];

// In host code `g_noalloc_star_bins` is only the host-side stand-in of the symbol, not a device address: the
// address the kernels get is resolved with cudaGetSymbolAddress, once per device, with that device current.
static constexpr int kNoAllocMaxDevices = 64;
static unsigned long long* g_noalloc_dev_ptr[kNoAllocMaxDevices] = {};
static std::mutex g_noalloc_mutex;

static int noalloc_scratch(int device, unsigned long long** out) {
  if (device < 0 || device >= kNoAllocMaxDevices) return QLP_BLS_EUNSUPPORTED;
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_dev_ptr[device]) {
    unsigned long long* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void**)&p, g_noalloc_star_bins);   // the current device's copy
    if (e != cudaSuccess || !p) { cudaGetLastError(); return QLP_BLS_ECUDA; }
    g_noalloc_dev_ptr[device] = p;
  }
  *out = g_noalloc_dev_ptr[device];
  return 0;
}

extern "C" int qlp_bls_grid_noalloc(qlp_bls_ctx* ctx, int64_t n_stars, const int64_t* row_ptr, const double* t,
                                    const double* rho, qlp_bls_star_grid* grid, int64_t* freq_ptr, int64_t* totals,
                                    void* cuda_stream) {
  NvtxRange nvtx_range("qlp_bls_grid_noalloc");
  if (!ctx || n_stars < 0 || !row_ptr || !freq_ptr || !totals) return QLP_BLS_EINVAL;
  if (n_stars > 0 && (!t || !rho || !grid)) return QLP_BLS_EINVAL;
  if (n_stars > (int64_t)QLP_BLS_NOALLOC_MAX_STARS) return QLP_BLS_ETOOLARGE;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  CUDA_TRY(cudaSetDevice(ctx->device));
  unsigned long long* star_bins = nullptr;
  QLP_TRY(noalloc_scratch(ctx->device, &star_bins));
  // The array keeps the previous call's contents.  grid_kernel writes every element that freq_scan_kernel reads
  // (one per star), so nothing has to start at zero; the used prefix is cleared all the same, so that a launch
  // that fails half-way cannot hand an earlier batch's sums to the scan.
  CUDA_TRY(cudaMemsetAsync(star_bins, 0, (size_t)(n_stars + 1) * sizeof(unsigned long long), st));
  if (n_stars > 0) {
    grid_kernel<<<(unsigned)n_stars, 256, 0, st>>>(ctx->prm, n_stars, row_ptr, t, rho, grid, star_bins);
    QLP_TRY(launch_ok(ctx));
  }
  freq_scan_kernel<<<1, 1024, 0, st>>>(n_stars, grid, star_bins, freq_ptr, totals);
  return launch_ok(ctx);
}
