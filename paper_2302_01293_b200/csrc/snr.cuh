// snr.cuh -- S4: the paper's S/N spectrum and the top peaks (Eq. 1, footnote 3 at
// :65, :44; O5, O6).
//
//   S/N(f) = (SR(f) - trend(f)) / sigma_SR,  trend = linear interpolation through the medians of N
//   equal-width frequency bins (N by Sturges' law),  sigma_SR = 1.4826 MAD(SR).
//
// One CTA per star.  Medians are EXACT order statistics found by a 4-pass, 8-bit-digit radix select
// over the FP32 bit patterns; all 2(N+1) selections (lower and upper middle of every bin and of the
// whole spectrum) advance together, each with its own 256-counter histogram in shared memory.  The
// MAD needs a second round on |SR - median|.  A last pass evaluates S/N, keeps each thread's K best
// local maxima and merges them; K short refolds give depth and epoch of each peak.
#pragma once
#include "common.cuh"

namespace qlp {

constexpr int kSnrThreads = 256;        // threads per CTA (= per star) of the S4 kernel ...
constexpr int kSnrThreadsLong = 1024;   // ... and for stars with at least kSnrLongGrid frequencies (a second launch)
constexpr int64_t kSnrLongGrid = 32768;
constexpr int kMaxSturges = 31;
constexpr int kMaxSel = 2 * (kMaxSturges + 1);

__device__ __forceinline__ uint32_t f2key(float v) {  // order-preserving map float -> uint32
  uint32_t b = __float_as_uint(v);
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float key2f(uint32_t k) {
  uint32_t b = (k & 0x80000000u) ? (k & 0x7fffffffu) : ~k;
  return __uint_as_float(b);
}

struct SnrShared {
  int64_t bstart[kMaxSturges + 2];  // first k of every Sturges bin; bstart[N] = n
  int64_t rank[kMaxSel];            // remaining rank of each selection inside its prefix class
  uint32_t prefix[kMaxSel];         // key bits fixed so far
  int32_t active[kMaxSel];
  double cx[kMaxSturges + 1], cy[kMaxSturges + 1];
  int32_t nk;
  double med, sigma;
  double red_v[kSnrThreadsLong / 32];
  int64_t red_k[kSnrThreadsLong / 32];
  int32_t red_t[kSnrThreadsLong / 32];
  double win_v; int64_t win_k; int32_t win_t;
  int64_t peak_k[kMaxTopK];
  double peak_v[kMaxTopK];
  int32_t n_peaks;
  unsigned long long accW; long long accS;
};

// Runs the radix select for selections [sel0, sel1).  key_of(k) gives the 32-bit key of element k;
// selection `sel` looks at elements [lo(sel), hi(sel)).  On return sh.prefix[sel] is the key of the
// wanted order statistic.
template <int NT, typename KeyFn>
__device__ void radix_select(SnrShared& sh, uint32_t* hist, int n_sel, int64_t n, int N, bool per_bin, KeyFn key_of) {
  const int tid = threadIdx.x;
  for (int pass = 0; pass < 4; ++pass) {
    const int shift = 24 - 8 * pass;
    for (int i = tid; i < n_sel * 256; i += NT) hist[i] = 0u;
    __syncthreads();
    for (int64_t k = tid; k < n; k += NT) {
      const uint32_t key = key_of(k);
      const uint32_t hi = (pass == 0) ? 0u : (key >> (shift + 8));
      const uint32_t dg = (key >> shift) & 255u;
      if (per_bin) {
        int b = 0;  // Sturges bin of k: largest b with bstart[b] <= k
        int lo = 0, hh = N - 1;
        while (lo < hh) { int mid = (lo + hh + 1) >> 1; if (sh.bstart[mid] <= k) lo = mid; else hh = mid - 1; }
        b = lo;
#pragma unroll
        for (int q = 0; q < 2; ++q) {
          const int sel = 2 * b + q;
          if (sh.active[sel] && (pass == 0 || (sh.prefix[sel] >> (shift + 8)) == hi)) atomicAdd(&hist[sel * 256 + dg], 1u);
        }
      }
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        const int sel = (per_bin ? 2 * N : 0) + q;
        if (sh.active[sel] && (pass == 0 || (sh.prefix[sel] >> (shift + 8)) == hi)) atomicAdd(&hist[sel * 256 + dg], 1u);
      }
    }
    __syncthreads();
    if (tid < n_sel && sh.active[tid]) {
      int64_t r = sh.rank[tid];
      uint32_t d = 0;
      for (; d < 255u; ++d) {
        const uint32_t c = hist[tid * 256 + d];
        if (r < (int64_t)c) break;
        r -= c;
      }
      sh.rank[tid] = r;
      sh.prefix[tid] |= d << shift;
    }
    __syncthreads();
  }
}

__device__ __forceinline__ int32_t sturges_bins(int64_t n) {
  int32_t N = (int32_t)floor(dadd(dadd(1.0, dmul(3.322, log10((double)n))), 0.5));
  if (N < 1) N = 1;
  if (N > kMaxSturges) N = kMaxSturges;
  return N;
}

// Trend (O5.4) at frequency x from the kept bin centres; same operation order as the definition.
__device__ __forceinline__ double trend_at(const SnrShared& sh, double x) {
  const int nk = sh.nk;
  if (x <= sh.cx[0]) return sh.cy[0];
  if (x >= sh.cx[nk - 1]) return sh.cy[nk - 1];
  int lo = 0, hi = nk - 2;  // largest seg with cx[seg] <= x
  while (lo < hi) { int mid = (lo + hi + 1) >> 1; if (sh.cx[mid] <= x) lo = mid; else hi = mid - 1; }
  const double slope = ddiv(dsub(sh.cy[lo + 1], sh.cy[lo]), dsub(sh.cx[lo + 1], sh.cx[lo]));
  return dadd(dmul(slope, dsub(x, sh.cx[lo])), sh.cy[lo]);
}

}  // namespace qlp
