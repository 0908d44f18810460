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
// One warp per (star, peak).  fit_count_kernel counts the points in the window; after an exclusive scan of the
// counts fit_kernel compacts (dt, y, w) of its points in time order into its slice of the workspace (SoA) and runs
// the search on them: every chi2 evaluation is two strided passes of the warp over the slice (sums, then
// residuals) with butterfly reductions, so all lanes hold identical values and take identical decisions.
#pragma once
#include "common.cuh"

namespace qlp {

constexpr int kFitWarps = 4;       // (star, peak) items per CTA
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

struct FitData {
  const double* dt;
  const double* yt;   // y - ybar
  const double* w;
  int n;
  double A, ybar, P;
};

__device__ __forceinline__ double trap_shape(double u, double half, double ing) {
  if (u >= half) return 0.0;
  const double d = half - u;
  return d < ing ? d / ing : 1.0;
}

// chi2 at (c, q, q_in) with the linear solution (depth, z); all lanes return the same values.
__device__ __forceinline__ double trap_chi2(const FitData& fd, int lane, double c, double q, double qin, double& depth,
                                            double& z) {
  const double D = q * fd.P, half = 0.5 * D, ing = qin * D;
  double B = 0.0, C = 0.0, F = 0.0;
  for (int i = lane; i < fd.n; i += 32) {
    const double sh = trap_shape(fabs(fd.dt[i] - c), half, ing);
    const double wsh = fd.w[i] * sh;
    B += wsh; C += wsh * sh; F += wsh * fd.yt[i];
  }
  B = warp_sum(B); C = warp_sum(C); F = warp_sum(F);
  const double V = C - B * B / fd.A;
  const double dl = V > 1e-9 * fd.A ? -F / V : 0.0;
  const double zc = dl * B / fd.A;
  double chi2 = 0.0;
  for (int i = lane; i < fd.n; i += 32) {
    const double sh = trap_shape(fabs(fd.dt[i] - c), half, ing);
    const double r = fd.yt[i] - zc + dl * sh;
    chi2 += fd.w[i] * r * r;
  }
  depth = dl; z = fd.ybar + zc;
  return warp_sum(chi2);
}

__global__ void __launch_bounds__(kFitWarps * 32) fit_kernel(int64_t n_items, int top_k,
                                                             const int64_t* __restrict__ row_ptr,
                                                             const double* __restrict__ t, const double* __restrict__ y,
                                                             const double* __restrict__ dy,
                                                             const qlp_bls_peak* __restrict__ peaks,
                                                             const int64_t* __restrict__ offset, double* __restrict__ work,
                                                             qlp_bls_trapezoid* __restrict__ fits) {
  const int64_t item = (int64_t)blockIdx.x * kFitWarps + (threadIdx.x >> 5);
  if (item >= n_items) return;
  const int lane = threadIdx.x & 31;
  const int64_t s = item / top_k;
  const qlp_bls_peak pk = peaks[item];
  const FitWindow w = fit_window(pk);
  const int64_t a = row_ptr[s], n = w.valid ? row_ptr[s + 1] - a : 0;
  const int64_t off = offset[item];
  const int nf = (int)(offset[item + 1] - off);
  double* dtv = work + 3 * off;
  double* yv = dtv + nf;
  double* wv = yv + nf;
  // ordered compaction of the window points
  int pos = 0;
  for (int64_t base = 0; base < n; base += 32) {
    const int64_t i = base + lane;
    double dt = 0.0;
    bool in = false;
    if (i < n) { dt = fit_dt(t[a + i], w); in = fabs(dt) <= w.win; }
    const unsigned bal = __ballot_sync(0xffffffffu, in);
    if (in) {
      const int p = pos + __popc(bal & ((1u << lane) - 1u));
      const double d = dy[a + i];
      dtv[p] = dt; yv[p] = y[a + i]; wv[p] = 1.0 / (d * d);
    }
    pos += __popc(bal);
  }
  __syncwarp();
  qlp_bls_trapezoid o;
  const double q0 = ddiv((double)pk.m, (double)(pk.nb > 0 ? pk.nb : 1));
  o.t0 = pk.t0; o.depth = 0.0; o.q = w.valid ? q0 : 0.0; o.q_in = 0.25; o.z = 0.0; o.chi2 = 0.0; o.chi2_init = 0.0;
  o.n_fit = nf; o.n_eval = 0; o.status = w.valid ? 0 : 1; o.pad_ = 0;
  if (w.valid && nf < kFitMinPoints) o.status = 2;
  if (o.status == 0) {
    double A = 0.0, E = 0.0;
    for (int i = lane; i < nf; i += 32) { A += wv[i]; E += wv[i] * yv[i]; }
    A = warp_sum(A); E = warp_sum(E);
    const double ybar = E / A;
    for (int i = lane; i < nf; i += 32) yv[i] = yv[i] - ybar;
    __syncwarp();
    FitData fd{dtv, yv, wv, nf, A, ybar, w.P};
    double th[3] = {0.0, q0, 0.25};
    double h[3] = {0.25 * w.D0, 0.25 * q0, 0.125};
    const double lo[3] = {-w.D0, 0.0, 0.0}, hi[3] = {w.D0, 1.0, 0.5};
    double dl, z;
    double best = trap_chi2(fd, lane, th[0], th[1], th[2], dl, z);
    int n_eval = 1;
    o.chi2_init = best;
    for (int level = 0; level < kFitLevels && n_eval < kFitMaxEval; ++level) {
      bool moved = true;
      while (moved && n_eval < kFitMaxEval) {
        moved = false;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
#pragma unroll
          for (int sg = 0; sg < 2; ++sg) {
            double v = sg == 0 ? th[d] + h[d] : th[d] - h[d];
            v = v < lo[d] ? lo[d] : v;
            v = v > hi[d] ? hi[d] : v;
            if (v == th[d]) continue;
            double dl2, z2;
            const double chi = trap_chi2(fd, lane, d == 0 ? v : th[0], d == 1 ? v : th[1], d == 2 ? v : th[2], dl2, z2);
            ++n_eval;
            if (chi < best) { best = chi; th[d] = v; dl = dl2; z = z2; moved = true; }
          }
        }
      }
      h[0] *= 0.5; h[1] *= 0.5; h[2] *= 0.5;
    }
    o.t0 = pk.t0 + th[0]; o.q = th[1]; o.q_in = th[2]; o.depth = dl; o.z = z; o.chi2 = best; o.n_eval = n_eval;
  }
  if (lane == 0) fits[item] = o;
}

}  // namespace qlp
