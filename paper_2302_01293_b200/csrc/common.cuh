// common.cuh -- shared declarations of the CUDA path (sm_100a only).
//
// Nothing here is shared with oracle/: constants and the deterministic cube root are typed a second
// time on purpose.  Step names (S0..S4, O0..O6) are DESIGN.md's.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/qlp_bls.h"

namespace qlp {

// ---- O0 constants (O0; PAPER.md:19 "stellar density", :7 sector length) -------------
// pi and K_rho = G rho_sun (86400 s/d)^2 = 3 GM_sun/(4 pi R_sun^3) 86400^2 with the IAU nominal
// GM_sun = 1.3271244e20 m^3 s^-2, R_sun = 6.957e8 m  ->  702.3999946673047 d^-2.
#define QLP_PI 3.141592653589793115997963468544185161590576171875
#define QLP_K_RHO 702.399994667304699760279618203639984130859375
#define QLP_TWO52 4503599627370496.0

constexpr int kMaxWidth = 16;     // largest supported box width in fine bins (ladder default: 11)
constexpr int kThreads = 512;     // threads per CTA of the fold/scan kernel
constexpr int kWarps = kThreads / 32;
constexpr int kNumClasses = 9;    // tile classes, see foldscan.cu
constexpr int kMaxTopK = 8;
constexpr uint32_t kScaleW = 4290772992u;  // 2^32 - 2^22: fixed-point unit of the weights

// One light-curve point as the fold kernel reads it: 16 bytes, one LDG.128 / LDS.128.
struct __align__(16) Point {
  double tau;   // t - t_ref (O2)
  uint32_t W;   // round(w * kScaleW), w = dy^-2 / sum dy^-2
  int32_t S;    // round(w * (y - ybar) * scale_s)
};

// Per-star results of S0 that later steps need.
struct StarPrep {
  double ybar;      // weighted mean (O2)
  double wsum;      // sum dy^-2
  double scale_s;   // fixed-point units per unit of w*ytilde (0 if the series is constant)
  float inv_w;      // 1 / kScaleW
  float inv_s;      // 1 / scale_s (0 if scale_s == 0)
  int32_t status;   // 0 ok, 5: too many points for the fixed-point weights
  int32_t pad_;
};

// Resolved search parameters (device copy of qlp_bls_config plus derived values).
struct Params {
  double samples_per_peak, dlogq, qmin_fac, qmax_fac, a_over_rstar_min, sector_days;
  double max_period_days;  // O1.10a: 0 = no period cap
  int64_t max_freq;        // O1.10b: 0 = no cap on the number of frequencies
  int32_t noverlap, top_k;
  uint32_t wmask;     // bit m set <=> width m is on the ladder (O1.9)
  int32_t max_width;  // largest width
  int32_t min_width;  // smallest width (the all-zero answer, O4)
  int32_t uniform_freq;  // O1.10c: comparison grid with equal steps in frequency (flags bit 1); read by grid_kernel only
};


// ---- optional bounds checks (the `check` build: -DQLP_BOUNDS_CHECK -> libqlp_bls_check.so) --------------------
// compute-sanitizer is closed on the GPU pool this library is developed on, so the shared-memory and workspace
// indices of the kernels can be checked by a build of their own: every guarded access tests its index against the
// extent it must stay in, counts a violation (per site class) instead of performing the access, and
// qlp_bls_debug_violations() reads the counters back.  In the normal build the macros cost nothing.
enum { kChkFoldCell = 0, kChkStage = 1, kChkScanBin = 2, kChkFitSlot = 3, kChkSnr = 4, kChkSlots = 8 };
#ifdef QLP_BOUNDS_CHECK
__device__ unsigned long long g_qlp_violations[kChkSlots];
#define QLP_IN_BOUNDS(slot, cond) ((cond) ? true : (atomicAdd(&g_qlp_violations[slot], 1ull), false))
#else
#define QLP_IN_BOUNDS(slot, cond) (true)
#endif

// ---- exact FP64 helpers: never contracted into FMAs (O1/O3: "no fused multiply-add") ---
__device__ __forceinline__ double dmul(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double dadd(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double dsub(double a, double b) { return __dadd_rn(a, -b); }
__device__ __forceinline__ double ddiv(double a, double b) { return __ddiv_rn(a, b); }

// cbrt_det (O0): frexp, exponent split by 3, eight Newton steps from y0 = 0.75 + 0.25 a.
__device__ inline double cbrt_det(double x) {
  int e;
  double mant = frexp(x, &e);
  int q = (e >= 0) ? (e / 3) : -((-e + 2) / 3);
  int r = e - 3 * q;
  double a = ldexp(mant, r);
  double y = dadd(0.75, dmul(0.25, a));
#pragma unroll 1
  for (int it = 0; it < 8; ++it) {
    double y2 = dmul(y, y);
    double d = ddiv(a, y2);
    double s = dmul(2.0, y);
    double n = dadd(s, d);
    y = ddiv(n, 3.0);
  }
  return ldexp(y, q);
}

// O1.8: frequency k of a star and its number of fine bins.  Q = qmin_fac * c_q.
// freq_of_k_cube: the f^(1/3) law alone (h > 0), without the test for the other kind of grid -- what the fold kernels
// compiled for the paper's ladder call, so that their code is the same whether or not the library knows the
// comparison grid.  freq_of_k (below): either kind, by the sign of h; everything else calls that one.
__device__ __forceinline__ void freq_of_k_cube(double u0, double h, double Q, double noverlap, int64_t k,
                                               double& f, int32_t& nb) {
  double u = dadd(u0, dmul((double)k, h));
  double u2 = dmul(u, u);
  f = dmul(u2, u);
  double qlo = dmul(Q, u2);
  nb = (int32_t)ceil(ddiv(noverlap, qlo));
}

__device__ __forceinline__ void freq_of_k(double u0, double h, double Q, double noverlap, int64_t k,
                                          double& f, int32_t& nb) {
  if (h < 0.0) {  // O1.10c: the descriptor of a frequency-uniform grid holds u0 = f_min and h = -df
    f = dadd(u0, dmul((double)k, -h));
    const double uk = cbrt_det(f);
    nb = (int32_t)ceil(ddiv(noverlap, dmul(Q, dmul(uk, uk))));
    return;
  }
  freq_of_k_cube(u0, h, Q, noverlap, k, f, nb);
}

// O3: bin of one point.  p = fl64(f * tau) is the only rounded operation; the bin is
// floor(nb * frac(p)) exactly.  Four FP64 instructions:
//   c' = RD(p + 2^52)           = 2^52 + floor(p)                  (0 <= p < 2^51)
//   A  = fma(-nb, c', (nb+1) 2^52) = 2^52 - nb floor(p)             (exactly representable)
//   v  = RD(fma(p, nb, A))      = 2^52 + floor(nb (p - floor p))   (one rounding, downwards)
// and the low word of v is the bin.  dnb = (double)nb, K = (nb + 1) * 2^52.
__device__ __forceinline__ int32_t bin_of(double f, double tau, double dnb, double K) {
  double p = __dmul_rn(f, tau);
  double c = __dadd_rd(p, QLP_TWO52);
  double A = __fma_rn(-dnb, c, K);
  double v = __fma_rd(p, dnb, A);
  return __double2loint(v);
}

// The same bin from THREE FP64 instructions and integer arithmetic (what the fold kernel uses):
//   I = floor(nb p)  = low word of RD(fma(p, nb, 2^52))      (exact: one rounding, downwards)
//   g = floor(p)     = low word of RD(p + 2^52)
//   floor(nb frac(p)) = I - nb g                              (nb g is an integer, so floor splits exactly)
// The difference is below 2^15, so 32-bit wrap-around arithmetic on I and g is harmless.  The two FP64
// results depend only on p, and the integer part folds into the address computation of the caller.
__device__ __forceinline__ void bin_parts(double f, double tau, double dnb, uint32_t& I, uint32_t& g) {
  const double p = __dmul_rn(f, tau);
  I = (uint32_t)__double2loint(__fma_rd(p, dnb, QLP_TWO52));
  g = (uint32_t)__double2loint(__dadd_rd(p, QLP_TWO52));
}
__device__ __forceinline__ int32_t bin_of3(double f, double tau, double dnb, uint32_t nb) {
  uint32_t I, g;
  bin_parts(f, tau, dnb, I, g);
  return (int32_t)(I - nb * g);
}

// Tile classes of the fold/scan kernel: columns per CTA and the largest nb the class holds.
// shared memory = cols * nbcap * 8 bytes of histograms + kStageBytes of point staging; class 0 fits
// two CTAs per SM, the others one.
__host__ __device__ __forceinline__ int class_cols(int c) {
  return c <= 1 ? 128 : (64 >> (c - 2));
}
__host__ __device__ __forceinline__ int class_nbcap(int c) {
  const int caps[kNumClasses] = {94, 208, 420, 840, 1680, 3360, 6720, 13440, 24576};
  return caps[c];
}
__host__ __device__ __forceinline__ int class_ctas_per_sm(int c) { return c == 0 ? 2 : 1; }
#ifndef QLP_PAIRED_CLASSES
#define QLP_PAIRED_CLASSES 1   /* the 32-column class folds two points per warp, 2 columns per lane (foldscan.cuh) */
#endif
constexpr int kChunk = 512;                                   // points per staged chunk
constexpr int kStageBytes = 2 * kChunk * 16 + 16;             // two buffers + two mbarriers
__host__ __device__ __forceinline__ int class_smem_bytes(int c) {
  return class_cols(c) * class_nbcap(c) * 8 + kStageBytes;
}

}  // namespace qlp
