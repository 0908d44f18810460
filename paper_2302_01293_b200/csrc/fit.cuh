// fit.cuh -- O8: trapezoid fit of each peak: "a trapezoid model parameterized by
// the orbital period (P), transit epoch (T0), depth, duration divided by orbital period (q), duration of ingress
// divided by transit duration (q_in), and out-of-transit magnitude level (z).  P is fixed to the BLS period while
// other parameters are fit using initial guesses from BLS ... we only fit data within two transit durations of
// the transit center ... bounds on q between 0 and 1, and q_in between 0 ... and 0.5".
//
// Readings (O8): the data of a fit are the points with |dt| <= 2 D0 around the BLS epoch (D0 = (m/nb) P,
// dt as in O7), fixed for the whole fit; for given (c = T0 - T0_bls, q, q_in) the level z and the depth enter
// linearly and are the weighted least-squares solution; (c, q, q_in) are found by a compass search with step
// halving from (0, q0, 0.25).
//
// fit_count_kernel (one warp per (star, peak)) counts the points in the window; after an exclusive scan of the
// counts fit_kernel (one CTA per (star, peak)) compacts (dt, y, w) of its points in time order into its slice of
// the workspace (SoA) and runs the search on them: every chi2 evaluation is one strided pass of the CTA over the
// slice, reduced in a fixed order so that all threads hold identical values and take identical decisions.  The
// first kFitCap points of a fit stay in shared memory (the mean window of a 200-s single-sector star holds about
// 3,400), the rest is re-read from the slice through L1/L2; the loops are unrolled so that several loads are in
// flight per thread.
#pragma once
#include "common.cuh"

namespace qlp {

constexpr int kFitWarps = 4;       // (star, peak) items per CTA of the counting kernel
constexpr int kFitThreads = 256;   // threads of the CTA that fits one (star, peak)
constexpr int kFitCap = 2304;      // points of a fit held in shared memory (54 KB: four CTAs of 64 registers per SM)
constexpr int kFitSmemBytes = 3 * kFitCap * 8;
constexpr int kFitLevels = 24;     // step halvings
constexpr int kFitMaxEval = 600;   // no sweep starts once this many chi2 evaluations are spent
constexpr int kFitMinPoints = 5;

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

struct FitWindow {
  double P, D0, win, t0;
  bool valid;
};
__device__ __forceinline__ FitWindow fit_window(const qlp_bls_peak& pk) {
  FitWindow w;
  w.valid = pk.status == 0 && pk.k >= 0 && pk.nb > 0;
  w.P = ddiv(1.0, pk.freq);
  w.D0 = dmul(ddiv((double)pk.m, (double)pk.nb), w.P);
  w.win = dmul(2.0, w.D0);
  w.t0 = pk.t0;
  return w;
}
// time from the nearest expected mid-transit, operations as O7 (the window test is an integer decision)
__device__ __forceinline__ double fit_dt(double t, const FitWindow& w) {
  const double x = ddiv(dsub(t, w.t0), w.P);
  const double cyc = floor(dadd(x, 0.5));
  return dmul(dsub(x, cyc), w.P);
}

__global__ void __launch_bounds__(kFitWarps * 32) fit_count_kernel(int64_t n_items, int top_k,
                                                                   const int64_t* __restrict__ row_ptr,
                                                                   const double* __restrict__ t,
                                                                   const qlp_bls_peak* __restrict__ peaks,
                                                                   int64_t* __restrict__ count) {
  const int64_t item = (int64_t)blockIdx.x * kFitWarps + (threadIdx.x >> 5);
  if (item >= n_items) return;
  const int lane = threadIdx.x & 31;
  const int64_t s = item / top_k;
  const qlp_bls_peak pk = peaks[item];
  const FitWindow w = fit_window(pk);
  const int64_t a = row_ptr[s], n = w.valid ? row_ptr[s + 1] - a : 0;
  int c = 0;
#pragma unroll 4
  for (int64_t i = lane; i < n; i += 32) c += fabs(fit_dt(t[a + i], w)) <= w.win ? 1 : 0;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
  if (lane == 0) count[item] = c;
}

// Exclusive scan of the counts -> offset[n_items + 1]; offset[n_items] (the total) also goes to total_out.
__global__ void __launch_bounds__(1024) fit_scan_kernel(int64_t n_items, const int64_t* __restrict__ count,
                                                        int64_t* __restrict__ offset, int64_t* __restrict__ total_out) {
  __shared__ int64_t warp_sum_s[32];
  __shared__ int64_t carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int64_t base = 0; base < n_items; base += blockDim.x) {
    const int64_t i = base + threadIdx.x;
    const int64_t v = i < n_items ? count[i] : 0;
    int64_t x = v;
    for (int o = 1; o < 32; o <<= 1) {
      const int64_t y = __shfl_up_sync(0xffffffffu, x, o);
      if (lane >= o) x += y;
    }
    if (lane == 31) warp_sum_s[wid] = x;
    __syncthreads();
    if (wid == 0) {
      int64_t ws = warp_sum_s[lane];
      for (int o = 1; o < 32; o <<= 1) {
        const int64_t y = __shfl_up_sync(0xffffffffu, ws, o);
        if (lane >= o) ws += y;
      }
      warp_sum_s[lane] = ws;
    }
    __syncthreads();
    const int64_t prefix = carry + (wid > 0 ? warp_sum_s[wid - 1] : 0) + x - v;
    if (i < n_items) offset[i] = prefix;
    __syncthreads();
    if (threadIdx.x == blockDim.x - 1) carry = prefix + v;
    __syncthreads();
  }
  if (threadIdx.x == 0) { offset[n_items] = carry; *total_out = carry; }
}

// The data of one fit: the first kFitCap points live in shared memory, the rest in the global workspace slice
// (indexed by the same position, so g_* are only read from kFitCap on).
struct FitData {
  const double *s_dt, *s_wy, *s_w;   // shared: dt, w (y - ybar), w
  const double *g_dt, *g_wy, *g_w;   // global slice
  int n;
  double A, inv_A, ybar, G, P;
};

__device__ __forceinline__ void trap_sums(const double* __restrict__ dt, const double* __restrict__ wy,
                                          const double* __restrict__ w, int begin, int end, double c, double half,
                                          double inv_ing, double (&s)[3]) {
#pragma unroll 4
  for (int i = begin + threadIdx.x; i < end; i += kFitThreads) {
    const double u = fabs(dt[i] - c);
    if (u < half) {
      const double sh = fmin((half - u) * inv_ing, 1.0);
      const double wsh = w[i] * sh;
      s[0] += wsh; s[1] += wsh * sh; s[2] += wy[i] * sh;
    }
  }
}

// Sum of NV values over the CTA, the same bits in every thread: butterfly inside a warp, then the warp partials
// in fixed order.  red is double-buffered ([2][NV][kFitThreads / 32]) so that one barrier per call is enough.
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double* red, int& phase) {
  constexpr int NW = kFitThreads / 32;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < NV; ++k) v[k] = warp_sum(v[k]);
  double* slot = red + phase * (NV * NW);
  if (lane == 0) {
#pragma unroll
    for (int k = 0; k < NV; ++k) slot[k * NW + wid] = v[k];
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < NV; ++k) {
    double a = slot[k * NW];
#pragma unroll
    for (int j = 1; j < NW; ++j) a += slot[k * NW + j];
    v[k] = a;
  }
  phase ^= 1;
}

// The unit trapezoid sh(u): 0 for u >= half, 1 on the flat bottom, linear over the ingress/egress of length
// ing = 1/inv_ing (ing = 0: inv_ing = +inf and every point inside the transit is at 1).

// chi2 at (c, q, q_in) with the linear solution (depth, z); every thread returns the same values.
// One pass: with the series centred (sum w yt = 0) and B = sum w sh, C = sum w sh^2, F = sum w yt sh,
//   V = C - B^2/A,  depth = -F/V,  z - ybar = depth B/A,  chi2 = G - F^2/V   (G = sum w yt^2),
// which is the residual sum of the least-squares solution written out.  Only points inside the transit
// (sh > 0) add to the sums; consecutive points are consecutive in time, so whole warps skip the rest.
__device__ __forceinline__ double trap_chi2(const FitData& fd, double* red3, int& ph3, double c, double q, double qin,
                                            double& depth, double& z) {
  const double D = q * fd.P, half = 0.5 * D, inv_ing = 1.0 / (qin * D);
  double s[3] = {0.0, 0.0, 0.0};
  trap_sums(fd.s_dt, fd.s_wy, fd.s_w, 0, fd.n < kFitCap ? fd.n : kFitCap, c, half, inv_ing, s);
  if (fd.n > kFitCap) trap_sums(fd.g_dt, fd.g_wy, fd.g_w, kFitCap, fd.n, c, half, inv_ing, s);
  block_sum<3>(s, red3, ph3);
  const double B = s[0], C = s[1], F = s[2];
  const double V = C - B * B * fd.inv_A;
  const double dl = V > 1e-9 * fd.A ? -F / V : 0.0;
  depth = dl; z = fd.ybar + dl * B * fd.inv_A;
  const double chi2 = fd.G + dl * F;
  return chi2 > 0.0 ? chi2 : 0.0;
}

__global__ void __launch_bounds__(kFitThreads, 4) fit_kernel(int64_t n_items, int top_k, const int64_t* __restrict__ row_ptr,
                                                          const double* __restrict__ t, const double* __restrict__ y,
                                                          const double* __restrict__ dy,
                                                          const qlp_bls_peak* __restrict__ peaks,
                                                          const int64_t* __restrict__ offset, double* __restrict__ work,
                                                          qlp_bls_trapezoid* __restrict__ fits) {
  constexpr int NW = kFitThreads / 32;
  extern __shared__ __align__(16) double fit_smem[];   // 3 x kFitCap doubles: dt, y -> w (y - ybar), w
  __shared__ double red3[2 * 3 * NW], red2[2 * 2 * NW];
  __shared__ int wcount[2][NW];
  double* sdt = fit_smem;
  double* sy = fit_smem + kFitCap;
  double* sw = fit_smem + 2 * kFitCap;
  const int64_t item = blockIdx.x;
  if (item >= n_items) return;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int64_t s = item / top_k;
  const qlp_bls_peak pk = peaks[item];
  const FitWindow w = fit_window(pk);
  const int64_t a = row_ptr[s], n = w.valid ? row_ptr[s + 1] - a : 0;
  const int64_t off = offset[item];
  const int nf = (int)(offset[item + 1] - off);
  double* dtv = work + 3 * off;
  double* yv = dtv + nf;
  double* wv = yv + nf;
  // ordered compaction of the window points, kFitThreads at a time
  int pos = 0, cb = 0;
  for (int64_t base = 0; base < n; base += kFitThreads) {
    const int64_t i = base + threadIdx.x;
    double dt = 0.0;
    bool in = false;
    if (i < n) { dt = fit_dt(t[a + i], w); in = fabs(dt) <= w.win; }
    const unsigned bal = __ballot_sync(0xffffffffu, in);
    if (lane == 0) wcount[cb][wid] = __popc(bal);
    __syncthreads();
    int before = 0, total = 0;
#pragma unroll
    for (int j = 0; j < NW; ++j) { const int cj = wcount[cb][j]; before += j < wid ? cj : 0; total += cj; }
    if (in) {
      const int p = pos + before + __popc(bal & ((1u << lane) - 1u));
      const double d = dy[a + i];
      const double wi = 1.0 / (d * d);
      if (p < kFitCap) { sdt[p] = dt; sy[p] = y[a + i]; sw[p] = wi; }
      else { dtv[p] = dt; yv[p] = y[a + i]; wv[p] = wi; }
    }
    pos += total;
    cb ^= 1;
  }
  __syncthreads();
  qlp_bls_trapezoid o;
  const double q0 = ddiv((double)pk.m, (double)(pk.nb > 0 ? pk.nb : 1));
  o.t0 = pk.t0; o.depth = 0.0; o.q = w.valid ? q0 : 0.0; o.q_in = 0.25; o.z = 0.0; o.chi2 = 0.0; o.chi2_init = 0.0;
  o.n_fit = nf; o.n_eval = 0; o.status = w.valid ? 0 : 1; o.pad_ = 0;
  if (w.valid && nf < kFitMinPoints) o.status = 2;
  if (o.status == 0) {
    int ph3 = 0, ph2 = 0;
    double ae[2] = {0.0, 0.0};
    for (int i = threadIdx.x; i < nf; i += kFitThreads) {
      const double wi = i < kFitCap ? sw[i] : wv[i], yi = i < kFitCap ? sy[i] : yv[i];
      ae[0] += wi; ae[1] += wi * yi;
    }
    block_sum<2>(ae, red2, ph2);
    const double A = ae[0], ybar = ae[1] / ae[0];
    double gs[2] = {0.0, 0.0};
    for (int i = threadIdx.x; i < nf; i += kFitThreads) {
      double* yp = i < kFitCap ? sy + i : yv + i;
      const double wi = i < kFitCap ? sw[i] : wv[i];
      const double yt = *yp - ybar;
      gs[0] += wi * yt * yt;
      *yp = wi * yt;
    }
    block_sum<2>(gs, red2, ph2);   // its barrier also publishes the rewritten slice
    FitData fd{sdt, sy, sw, dtv, yv, wv, nf, A, 1.0 / A, ybar, gs[0], w.P};
    double th0 = 0.0, th1 = q0, th2 = 0.25;                     // c, q, q_in
    double h0 = 0.25 * w.D0, h1 = 0.25 * q0, h2 = 0.125;
    double dl = 0.0, z = 0.0, best = 0.0;
    int n_eval = 0;
    // every thread holds the same numbers, so the whole CTA takes the same branches.  One call site of the
    // chi2 evaluation (move -1 is the start point) keeps the kernel small enough for the instruction cache.
    for (int level = 0; level < kFitLevels && n_eval < kFitMaxEval; ++level) {
      bool moved = true;
      while (moved && n_eval < kFitMaxEval) {
        moved = false;
#pragma unroll 1
        for (int mv = (n_eval == 0 ? -1 : 0); mv < 6; ++mv) {
          const int d = mv >> 1;                                 // -1: start point
          const double cur = d == 0 ? th0 : d == 1 ? th1 : th2;
          const double step = d == 0 ? h0 : d == 1 ? h1 : h2;
          const double lo = d == 0 ? -w.D0 : 0.0, hi = d == 0 ? w.D0 : d == 1 ? 1.0 : 0.5;
          double v = (mv & 1) ? cur - step : cur + step;
          v = v < lo ? lo : v;
          v = v > hi ? hi : v;
          if (mv >= 0 && v == cur) continue;
          double dl2, z2;
          const double chi = trap_chi2(fd, red3, ph3, d == 0 ? v : th0, d == 1 ? v : th1, d == 2 ? v : th2, dl2, z2);
          ++n_eval;
          if (mv < 0) { best = chi; dl = dl2; z = z2; o.chi2_init = chi; }
          else if (chi < best) {
            best = chi; dl = dl2; z = z2; moved = true;
            th0 = d == 0 ? v : th0; th1 = d == 1 ? v : th1; th2 = d == 2 ? v : th2;
          }
        }
      }
      h0 *= 0.5; h1 *= 0.5; h2 *= 0.5;
    }
    o.t0 = pk.t0 + th0; o.q = th1; o.q_in = th2; o.depth = dl; o.z = z; o.chi2 = best; o.n_eval = n_eval;
  }
  if (threadIdx.x == 0) fits[item] = o;
}

}  // namespace qlp
