// grid.cuh -- S1: per-star Keplerian frequency / duration grid (O1).
//
// One CTA per star.  The timestamps are scanned once for gaps longer than one sector (PAPER.md:23:
// "the longest continuous stretch of data ... without a gap longer than one sector"); everything
// after that is a handful of FP64 operations done by thread 0 in the order DESIGN.md O1 fixes, with
// +, -, *, /, sqrt, frexp/ldexp, floor/ceil only, so that the descriptor is bit-identical to the
// oracle's.  The CTA then sums nb_k over the star's grid (the "total_bins" figure of the API).
#pragma once
#include "common.cuh"

namespace qlp {

constexpr int kMaxBreaks = 256;

__global__ void __launch_bounds__(256) grid_kernel(Params prm, int64_t n_stars, const int64_t* __restrict__ row_ptr,
                                                   const double* __restrict__ t, const double* __restrict__ rho,
                                                   qlp_bls_star_grid* __restrict__ grid,
                                                   unsigned long long* __restrict__ star_bins) {
  const int64_t s = blockIdx.x;
  if (s >= n_stars) return;
  const int64_t a = row_ptr[s], n = row_ptr[s + 1] - a;
  const double* ts = t + a;
  __shared__ int64_t brk[kMaxBreaks];
  __shared__ int n_brk;
  __shared__ qlp_bls_star_grid g;
  __shared__ unsigned long long bins_acc;
  __shared__ int bad_t;
  if (threadIdx.x == 0) { n_brk = 0; bins_acc = 0ull; bad_t = 0; }
  __syncthreads();
  // O1.2: position i is a break if t[i+1] - t[i] > sector_days (strict).  The same differences show whether
  // the timestamps increase strictly (the contract of the API): a star that breaks it would fold with
  // tau < 0, for which the fold's magic-number floor is not defined, so it is skipped here (status 7)
  // whether or not input validation (flags bit0) is on.
  for (int64_t i = threadIdx.x; i + 1 < n; i += blockDim.x) {
    const double d = dsub(ts[i + 1], ts[i]);
    if (d > prm.sector_days) {
      int slot = atomicAdd(&n_brk, 1);
      if (slot < kMaxBreaks) brk[slot] = i;
    }
    if (!(d > 0.0) || !(d < 1.0e15)) bad_t = 1;   // repeated, decreasing, NaN or infinite timestamps
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    qlp_bls_star_grid q;
    q.t_ref = 0.0; q.baseline = 0.0; q.p_min = 0.0; q.p_max = 0.0; q.c_q = 0.0; q.u0 = 0.0; q.h = 0.0;
    q.n_freq = 0; q.nb_max = 0; q.status = 0;
    double r_in = rho[s];
    double rh = (isfinite(r_in) && r_in > 0.0) ? r_in : 1.0;  // O1.1
    if (n < 2) {
      q.status = 1;
      if (n == 1) q.t_ref = ts[0];
    } else {
      q.t_ref = ts[0];
      double T = dsub(ts[n - 1], ts[0]);
      q.baseline = T;
      double L = 0.0;
      int has_break = n_brk > 0;
      if (n_brk <= kMaxBreaks) {
        // insertion sort of the (few) break positions, then the stretches between them
        int nb_ = n_brk;
        for (int i = 1; i < nb_; ++i) {
          int64_t v = brk[i];
          int j = i - 1;
          while (j >= 0 && brk[j] > v) { brk[j + 1] = brk[j]; --j; }
          brk[j + 1] = v;
        }
        int64_t first = 0;
        for (int i = 0; i < nb_; ++i) {
          double len = dsub(ts[brk[i]], ts[first]);
          if (len > L) L = len;
          first = brk[i] + 1;
        }
        double len = dsub(ts[n - 1], ts[first]);
        if (len > L) L = len;
      } else {
        // more breaks than the list holds: plain sequential scan (pathological input)
        int64_t first = 0;
        for (int64_t i = 0; i + 1 < n; ++i) {
          if (dsub(ts[i + 1], ts[i]) > prm.sector_days) {
            double len = dsub(ts[i], ts[first]);
            if (len > L) L = len;
            first = i + 1;
          }
        }
        double len = dsub(ts[n - 1], ts[first]);
        if (len > L) L = len;
      }
      double p_max = has_break ? L : dmul(0.5, L);
      // O1.10a: period cap of the comparison grid
      if (prm.max_period_days > 0.0 && p_max > prm.max_period_days) p_max = prm.max_period_days;
      q.p_max = p_max;
      // O1.3: a/R* = (G rho P^2 / 3 pi)^(1/3)  =>  P_min = sqrt(3 pi k^3 / (K_rho rho))
      double D = dmul(QLP_K_RHO, rh);
      double k = prm.a_over_rstar_min;
      double c3 = dmul(dmul(k, k), k);
      double three_pi = dmul(3.0, QLP_PI);
      q.p_min = __dsqrt_rn(ddiv(dmul(three_pi, c3), D));
      // O1.4: q_circ(f) = (R*/a)/pi = C_q f^(2/3)
      q.c_q = ddiv(cbrt_det(ddiv(three_pi, D)), QLP_PI);
      if (!(T > 0.0)) q.status = 2;
      else if (!(p_max > 0.0)) q.status = 3;
      else {
        double f_min = ddiv(1.0, p_max), f_max = ddiv(1.0, q.p_min);
        if (!(f_max > f_min)) q.status = 3;
        else {
          // O1.6-7: uniform in u = f^(1/3), step h = qmin_fac C_q / (samples_per_peak T) / 3
          double u0 = cbrt_det(f_min), u1 = cbrt_det(f_max);
          double Q = dmul(prm.qmin_fac, q.c_q);
          double A = ddiv(Q, dmul(prm.samples_per_peak, T));
          double h = ddiv(A, 3.0);
          q.n_freq = (int64_t)floor(ddiv(dsub(u1, u0), h)) + 1;
          // O1.10b: at most max_freq frequencies over the same range in u (under-sampled comparison grid)
          if (prm.max_freq >= 2 && q.n_freq > prm.max_freq) {
            h = ddiv(dsub(u1, u0), (double)(prm.max_freq - 1));
            q.n_freq = prm.max_freq;
          }
          q.u0 = u0; q.h = h;
          double qlo = dmul(Q, dmul(u0, u0));
          q.nb_max = (int32_t)ceil(ddiv((double)prm.noverlap, qlo));
          // O1.10c: equal steps in frequency over the same range; df = the f^(1/3) law's step at f_min (A u0^2),
          // or (f_max - f_min) / (max_freq - 1) when that takes more than max_freq points; u0 <- f_min, h <- -df
          if (prm.uniform_freq) {
            double df = dmul(A, dmul(u0, u0));
            q.n_freq = (int64_t)floor(ddiv(dsub(f_max, f_min), df)) + 1;
            if (prm.max_freq >= 2 && q.n_freq > prm.max_freq) {
              df = ddiv(dsub(f_max, f_min), (double)(prm.max_freq - 1));
              q.n_freq = prm.max_freq;
            }
            if (!(df > dmul(1e-9, f_max))) { q.status = 3; q.n_freq = 0; q.nb_max = 0; q.u0 = 0.0; q.h = 0.0; }
            else { q.u0 = f_min; q.h = -df; }
          }
          if (q.status == 3) { }
          else if (bad_t) { q.status = 7; q.n_freq = 0; }
          else if (q.nb_max > QLP_BLS_MAX_NB || q.nb_max <= 0) { q.status = 4; q.n_freq = 0; }
          else if (n >= (int64_t)QLP_BLS_MAX_POINTS) { q.status = 5; q.n_freq = 0; }  // fixed-point weights
        }
      }
    }
    g = q;
  }
  __syncthreads();
  // total_bins: sum of nb_k over the grid
  if (g.status == 0 && g.n_freq > 0) {
    const double Q = dmul(prm.qmin_fac, g.c_q);
    unsigned long long acc = 0;
    for (int64_t k = threadIdx.x; k < g.n_freq; k += blockDim.x) {
      double f; int32_t nb;
      freq_of_k(g.u0, g.h, Q, (double)prm.noverlap, k, f, nb);
      acc += (unsigned long long)nb;
    }
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) atomicAdd(&bins_acc, acc);
  }
  __syncthreads();
  if (threadIdx.x == 0) { grid[s] = g; star_bins[s] = bins_acc; }
}

// Exclusive scan of n_freq -> freq_ptr[S+1], plus the two totals.  One CTA; S is at most a few 1e5.
__global__ void __launch_bounds__(1024) freq_scan_kernel(int64_t n_stars, const qlp_bls_star_grid* __restrict__ grid,
                                                         const unsigned long long* __restrict__ star_bins,
                                                         int64_t* __restrict__ freq_ptr, int64_t* __restrict__ totals) {
  __shared__ int64_t warp_sum[32];
  __shared__ int64_t carry;
  __shared__ unsigned long long bins_total;
  if (threadIdx.x == 0) { carry = 0; bins_total = 0; }
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  unsigned long long my_bins = 0;
  for (int64_t base = 0; base < n_stars; base += blockDim.x) {
    int64_t i = base + threadIdx.x;
    int64_t v = (i < n_stars) ? grid[i].n_freq : 0;
    if (i < n_stars) my_bins += star_bins[i];
    int64_t x = v;
    for (int o = 1; o < 32; o <<= 1) {
      int64_t y = __shfl_up_sync(0xffffffffu, x, o);
      if (lane >= o) x += y;
    }
    if (lane == 31) warp_sum[wid] = x;
    __syncthreads();
    if (wid == 0) {
      int64_t w = warp_sum[lane];
      for (int o = 1; o < 32; o <<= 1) {
        int64_t y = __shfl_up_sync(0xffffffffu, w, o);
        if (lane >= o) w += y;
      }
      warp_sum[lane] = w;
    }
    __syncthreads();
    int64_t prefix = carry + (wid > 0 ? warp_sum[wid - 1] : 0) + x - v;
    if (i < n_stars) freq_ptr[i] = prefix;
    __syncthreads();
    if (threadIdx.x == blockDim.x - 1) carry = prefix + v;
    __syncthreads();
  }
  for (int o = 16; o > 0; o >>= 1) my_bins += __shfl_down_sync(0xffffffffu, my_bins, o);
  if (lane == 0) atomicAdd(&bins_total, my_bins);
  __syncthreads();
  if (threadIdx.x == 0) {
    freq_ptr[n_stars] = carry;
    totals[0] = carry;
    totals[1] = (int64_t)bins_total;
  }
}

// test-only: f_k, nb_k of one star
__global__ void debug_freqs_kernel(Params prm, const qlp_bls_star_grid* __restrict__ grid, int64_t star, int64_t k0,
                                   int64_t k1, double* __restrict__ f, int32_t* __restrict__ nb) {
  const qlp_bls_star_grid g = grid[star];
  const double Q = dmul(prm.qmin_fac, g.c_q);
  for (int64_t k = k0 + blockIdx.x * (int64_t)blockDim.x + threadIdx.x; k < k1; k += (int64_t)gridDim.x * blockDim.x) {
    double fk; int32_t nbk;
    freq_of_k(g.u0, g.h, Q, (double)prm.noverlap, k, fk, nbk);
    f[k - k0] = fk;
    nb[k - k0] = nbk;
  }
}

}  // namespace qlp
