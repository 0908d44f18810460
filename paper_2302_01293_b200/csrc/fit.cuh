// fit.cuh -- O8: trapezoid fit of each peak: "a trapezoid model parameterized by
// the orbital period (P), transit epoch (T0), depth, duration divided by orbital period (q), duration of ingress
// divided by transit duration (q_in), and out-of-transit magnitude level (z).  P is fixed to the BLS period while
// other parameters are fit using initial guesses from BLS ... we only fit data within two transit durations of
// the transit center ... bounds on q between 0 and 1, and q_in between 0 ... and 0.5".
//
// Readings (O8): the data of a fit are the points with |dt| <= 2 D0 around the BLS epoch (D0 = (m/nb) P,
// dt as in O7), fixed for the whole fit; for given (c = T0 - T0_bls, q, q_in) the level z and the depth enter
// linearly and are the weighted least-squares solution; (c, q, q_in) are found by a compass search with step
// halving from (0, q0, 0.25): a sweep evaluates the (up to) six neighbours theta +- h_d e_d, takes the first one (order
// c+, c-, q+, q-, q_in+, q_in-) whose chi2 is within tol = max(1e-9 chi2_best, 1e-12 G) of the smallest, and moves
// there iff that lowers chi2 by more than tol (G = sum w (y - ybar)^2); chi2 values of two summation orders differ
// by ~1e-15 G, so the path does not depend on how the sums are formed.
//
// fit_count_kernel (one warp per (star, peak)) counts the points in the window, separately for each of kFitCluster
// equal chunks of the star's points; after an exclusive scan of the totals fit_kernel compacts (dt, y, w) of the
// window points in time order and runs the search on them: ONE strided pass over the points evaluates all six
// neighbours of a sweep (18 sums), reduced in a fixed order so that all threads take identical decisions.
// Small windows (<= kFitSingleMax points, the usual case of a single-sector star) are fitted by one CTA (the first
// kFitCap points in shared memory, the rest re-read from the workspace).  Larger windows (a noise peak with q ~ 0.3 takes the whole light curve; 13-sector stars) are fitted
// by a thread-block CLUSTER of kFitCluster CTAs: CTA r compacts and keeps chunk r (up to kFitCap points in its own
// shared memory, the rest in its slice of the workspace), the per-CTA sums of a sweep are exchanged through
// distributed shared memory (one cluster barrier per sweep) and added in rank order by every CTA, so all CTAs of
// the cluster hold the same bits and walk the same path.
#pragma once
#include <cooperative_groups.h>

#include "common.cuh"

namespace qlp {

constexpr int kFitCountThreads = 256;   // threads of the CTA that counts the window points of one (star, peak)
constexpr int kFitThreads = 128;   // threads of one CTA of the fit kernel (128 registers each: four CTAs per SM)
constexpr int kFitCluster = 8;     // CTAs per cluster for large windows (portable cluster size)
constexpr int kFitCap = 2240;      // points of a fit held in one CTA's shared memory (52.5 KB: four CTAs per SM)
constexpr int kFitSingleMax = 4 * kFitCap;   // windows up to this many points are fitted by one CTA (measured best)
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

// chunk r of a star of n points: [n r / kFitCluster, n (r + 1) / kFitCluster)
__device__ __forceinline__ int64_t fit_chunk_begin(int64_t n, int r) { return (n * r) / kFitCluster; }

__global__ void __launch_bounds__(kFitCountThreads) fit_count_kernel(int64_t n_items, int top_k,
                                                                    const int64_t* __restrict__ row_ptr,
                                                                    const double* __restrict__ t,
                                                                    const qlp_bls_peak* __restrict__ peaks,
                                                                    int64_t* __restrict__ count,
                                                                    int32_t* __restrict__ chunk_count,
                                                                    int32_t* __restrict__ list /* [2][n_items] */,
                                                                    unsigned long long* __restrict__ list_n /* [2] */) {
  // one CTA per (star, peak): a 13-sector star has 1.5e5 points, too many for the one warp of round 1
  const int64_t item = blockIdx.x;
  if (item >= n_items) return;
  __shared__ int cnt8[kFitCluster];
  if (threadIdx.x < kFitCluster) cnt8[threadIdx.x] = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const int64_t s = item / top_k;
  const qlp_bls_peak pk = peaks[item];
  const FitWindow w = fit_window(pk);
  const int64_t a = row_ptr[s], n = w.valid ? row_ptr[s + 1] - a : 0;
  for (int r = 0; r < kFitCluster; ++r) {
    const int64_t b = fit_chunk_begin(n, r), e = fit_chunk_begin(n, r + 1);
    int c = 0;
#pragma unroll 4
    for (int64_t i = b + threadIdx.x; i < e; i += kFitCountThreads) c += fabs(fit_dt(t[a + i], w)) <= w.win ? 1 : 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if (lane == 0 && c) atomicAdd(&cnt8[r], c);
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    int64_t total = 0;
    for (int r = 0; r < kFitCluster; ++r) { chunk_count[item * kFitCluster + r] = cnt8[r]; total += cnt8[r]; }
    count[item] = total;
    // size class of the fit: 0 = one CTA (also the items without a valid peak), 1 = one cluster
    const int cls = total > kFitSingleMax ? 1 : 0;
    const unsigned long long slot = atomicAdd(&list_n[cls], 1ull);
    list[(int64_t)cls * n_items + (int64_t)slot] = (int32_t)item;
  }
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

// The six trial points of one sweep.  Candidate k = 2 d + sign moves coordinate d of (c, q, q_in): k = 0, 1 move the
// epoch (they share the duration and ingress of the current point), k = 2, 3 the duration (own half-duration and own
// ingress, since ing = q_in D), k = 4, 5 the ingress fraction (own ingress only).  All six are always summed; a
// candidate that is not tried (its clipped value is the current one) is dropped after the reduction.
struct Trial {
  double c0, c1, cb;            // epochs of candidates 0, 1 and of the current point (candidates 2..5)
  double hb, h2, h3;            // half-durations: current (candidates 0, 1, 4, 5), candidates 2, 3
  double ib, i2, i3, i4, i5;    // 1 / ingress: current (candidates 0, 1), candidates 2..5
  double reach;                 // no candidate's transit reaches further from the current epoch than this
};

// One candidate's contribution of one point: u = |dt - c_k|; inside the transit (u < half) the unit trapezoid is
// sh = min((half - u) / ing, 1) (ing = 0: inv_ing = +inf and every inside point is at 1).
__device__ __forceinline__ void trial_add(double u, double half, double inv_ing, double w, double wy, double& B,
                                          double& C, double& F) {
  // branch-free: the six candidates of a point are six independent dependency chains (a branch per candidate
  // serialises them); outside the transit the select discards whatever (half - u) * inv_ing gave, NaN included
  const double sh = u < half ? fmin((half - u) * inv_ing, 1.0) : 0.0;
  const double wsh = w * sh;
  B += wsh; C = fma(wsh, sh, C); F = fma(wy, sh, F);
}

// Sums B = sum w sh, C = sum w sh^2, F = sum w (y - ybar) sh of all six candidates over points [begin, end) in ONE
// pass.  Only points inside some candidate's transit do any work; consecutive points are consecutive in time, so
// whole warps skip the rest of the window.
template <bool PREFETCH>
__device__ __forceinline__ void trial_sums(const double* __restrict__ dt, const double* __restrict__ wy,
                                           const double* __restrict__ w, int begin, int end, const Trial& tr,
                                           double (&s)[18], unsigned int& in_reach) {
  // PREFETCH (the part of a window that lives in global memory): the records of the next iteration are requested
  // before this one's are used, so the L2 latency of one iteration hides behind the arithmetic of another
  int i = begin + threadIdx.x;
  double d_n = 0.0, w_n = 0.0, wy_n = 0.0;
  if (PREFETCH && i < end) { d_n = dt[i]; w_n = w[i]; wy_n = wy[i]; }
#pragma unroll 1
  for (; i < end; i += kFitThreads) {
    double d, wi, wyi;
    if (PREFETCH) {
      d = d_n; wi = w_n; wyi = wy_n;
      const int j = i + kFitThreads;
      if (j < end) { d_n = dt[j]; w_n = w[j]; wy_n = wy[j]; }
    } else {
      d = dt[i];
    }
    const double u0 = fabs(d - tr.cb);            // candidates 2..5 keep the current epoch
    if (u0 < tr.reach) {
      if (!PREFETCH) { wi = w[i]; wyi = wy[i]; }
      ++in_reach;
      trial_add(fabs(d - tr.c0), tr.hb, tr.ib, wi, wyi, s[0], s[1], s[2]);
      trial_add(fabs(d - tr.c1), tr.hb, tr.ib, wi, wyi, s[3], s[4], s[5]);
      trial_add(u0, tr.h2, tr.i2, wi, wyi, s[6], s[7], s[8]);
      trial_add(u0, tr.h3, tr.i3, wi, wyi, s[9], s[10], s[11]);
      trial_add(u0, tr.hb, tr.i4, wi, wyi, s[12], s[13], s[14]);
      trial_add(u0, tr.hb, tr.i5, wi, wyi, s[15], s[16], s[17]);
    }
  }
}

// Sum of NV values over the CTA -- and, for CS > 1, over the CS CTAs of the cluster.  Butterfly inside each warp,
// warp partials to shared memory (red is double-buffered, [2][NV][kFitThreads / 32]: one barrier per call), then lane
// l < NV of EVERY warp adds up the partials of value l in fixed order.  In a cluster, warp 0 publishes the CTA's
// totals in xchg ([2][18] in its own shared memory), one cluster barrier makes them visible, and lane l of every
// warp of every CTA adds the CS totals of value l in rank order through distributed shared memory.  Returns the
// total of value `lane` (lanes >= NV: 0); all warps of all CTAs hold the same bits.
template <int CS, int NV>
__device__ __forceinline__ double all_sum_to_lanes(double (&v)[NV], double* red, double* xchg, int& phase) {
  constexpr int NW = kFitThreads / 32;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < NV; ++k) v[k] = warp_sum(v[k]);
  double* slot = red + phase * (18 * NW);
  if (lane == 0) {
#pragma unroll
    for (int k = 0; k < NV; ++k) slot[k * NW + wid] = v[k];
  }
  __syncthreads();
  double a = 0.0;
  if (lane < NV) {
    a = slot[lane * NW];
#pragma unroll
    for (int j = 1; j < NW; ++j) a += slot[lane * NW + j];
  }
  if (CS > 1) {
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    double* mine = xchg + phase * 18;
    if (wid == 0 && lane < NV) mine[lane] = a;
    cluster.sync();
    a = 0.0;
    if (lane < NV) {
#pragma unroll
      for (int r = 0; r < CS; ++r) a += cluster.map_shared_rank(mine, r)[lane];
    }
  }
  phase ^= 1;
  return a;
}
// The same for a few values that every thread needs (A, sum w y, G): all threads return the totals.
template <int CS, int NV>
__device__ __forceinline__ void all_sum(double (&v)[NV], double* red, double* xchg, int& phase) {
  const double a = all_sum_to_lanes<CS, NV>(v, red, xchg, phase);
#pragma unroll
  for (int k = 0; k < NV; ++k) v[k] = __shfl_sync(0xffffffffu, a, k);
}

// One sweep: chi2 of the six candidates, each with its linear solution (depth, z).  With the series centred
// (sum w yt = 0):  V = C - B^2/A,  depth = -F/V,  z - ybar = depth B/A,  chi2 = G - F^2/V  (G = sum w yt^2), which
// is the residual sum of the least-squares solution written out.  Lane k < 6 of every warp ends up holding candidate
// k's (chi2, depth, z); the other lanes hold chi2 = +inf.
template <int CS>
__device__ __forceinline__ void trial_chi2(const FitData& fd, double* red, double* xchg, int& ph, const Trial& tr,
                                           double& chi2, double& depth, double& z, unsigned int& in_reach) {
  double s[18];
#pragma unroll
  for (int k = 0; k < 18; ++k) s[k] = 0.0;
  trial_sums<false>(fd.s_dt, fd.s_wy, fd.s_w, 0, fd.n < kFitCap ? fd.n : kFitCap, tr, s, in_reach);
  if (fd.n > kFitCap) trial_sums<true>(fd.g_dt, fd.g_wy, fd.g_w, kFitCap, fd.n, tr, s, in_reach);
  const double tot = all_sum_to_lanes<CS, 18>(s, red, xchg, ph);   // lane l: value l = 3 k + {0: B, 1: C, 2: F}
  const int lane = threadIdx.x & 31;
  const int k3 = lane < 6 ? 3 * lane : 0;
  const double B = __shfl_sync(0xffffffffu, tot, k3);
  const double C = __shfl_sync(0xffffffffu, tot, k3 + 1);
  const double F = __shfl_sync(0xffffffffu, tot, k3 + 2);
  const double V = C - B * B * fd.inv_A;
  const double dl = V > 1e-9 * fd.A ? -F / V : 0.0;
  const double c2 = fd.G + dl * F;
  depth = dl;
  z = fd.ybar + dl * B * fd.inv_A;
  chi2 = lane < 6 ? (c2 > 0.0 ? c2 : 0.0) : __longlong_as_double(0x7ff0000000000000ll);
}

// CS = 1: one CTA per (star, peak), windows of at most kFitSingleMax points (also the items without a valid peak);
// CS = kFitCluster: one cluster per (star, peak), larger windows.  `list` holds the items of the size class.
template <int CS>
__global__ void __launch_bounds__(kFitThreads, 4) fit_kernel(int64_t n_items, int top_k, const int64_t* __restrict__ row_ptr,
                                                          const double* __restrict__ t, const double* __restrict__ y,
                                                          const double* __restrict__ dy,
                                                          const qlp_bls_peak* __restrict__ peaks,
                                                          const int64_t* __restrict__ offset,
                                                          const int32_t* __restrict__ chunk_count,
                                                          const int32_t* __restrict__ list, int64_t n_list,
                                                          double* __restrict__ work,
                                                          qlp_bls_trapezoid* __restrict__ fits,
                                                          unsigned long long* __restrict__ work_ctr /* NULL, or two
                                                          counters: (point, sweep) pairs inside a transit; sweeps */) {
  constexpr int NW = kFitThreads / 32;
  extern __shared__ __align__(16) double fit_smem[];   // 3 x kFitCap doubles: dt, y -> w (y - ybar), w
  __shared__ double red[2 * 18 * NW], xchg[2 * 18];
  __shared__ int wcount[2][NW];
  double* sdt = fit_smem;
  double* sy = fit_smem + kFitCap;
  double* sw = fit_smem + 2 * kFitCap;
  const int64_t li = blockIdx.x / CS;                  // position in this size class's list of items
  const int rank = (int)(blockIdx.x % CS);             // = the CTA's rank in its cluster (clusters tile the grid)
  if (li >= n_list) return;
  const int64_t item = list[li];
  if (item < 0 || item >= n_items) return;
  const int64_t off = offset[item];
  const int nf = (int)(offset[item + 1] - off);        // points in the window of this fit
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int64_t s = item / top_k;
  const qlp_bls_peak pk = peaks[item];
  const FitWindow w = fit_window(pk);
  const int64_t a = row_ptr[s], n = w.valid ? row_ptr[s + 1] - a : 0;
  // this CTA's chunk of the star and its place in the fit's slice of the workspace
  int64_t c_begin = 0, c_end = n;
  int base = 0, cnt = nf;
  if (CS > 1) {
    c_begin = fit_chunk_begin(n, rank); c_end = fit_chunk_begin(n, rank + 1);
    for (int r = 0; r < rank; ++r) base += chunk_count[item * kFitCluster + r];
    cnt = chunk_count[item * kFitCluster + rank];
  }
  double* dtv = work + 3 * off + base;                 // local index i >= kFitCap lives at dtv[i], yv[i], wv[i]
  double* yv = dtv + nf;
  double* wv = yv + nf;
  // ordered compaction of the window points of the chunk, kFitThreads at a time
  int pos = 0, cb = 0;
  for (int64_t b0 = c_begin; b0 < c_end; b0 += kFitThreads) {
    const int64_t i = b0 + threadIdx.x;
    double dt = 0.0;
    bool in = false;
    if (i < c_end) { dt = fit_dt(t[a + i], w); in = fabs(dt) <= w.win; }
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
      // check build: the slot lies inside this CTA's share of the window (the counts of fit_count_kernel)
      if (QLP_IN_BOUNDS(kChkFitSlot, p >= 0 && p < cnt && base + p < nf)) {
        if (p < kFitCap) { sdt[p] = dt; sy[p] = y[a + i]; sw[p] = wi; }
        else { dtv[p] = dt; yv[p] = y[a + i]; wv[p] = wi; }
      }
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
    int ph = 0;
    double ae[2] = {0.0, 0.0};
    for (int i = threadIdx.x; i < cnt; i += kFitThreads) {
      const double wi = i < kFitCap ? sw[i] : wv[i], yi = i < kFitCap ? sy[i] : yv[i];
      ae[0] += wi; ae[1] += wi * yi;
    }
    all_sum<CS, 2>(ae, red, xchg, ph);
    const double A = ae[0], ybar = ae[1] / ae[0];
    double gs[2] = {0.0, 0.0};
    for (int i = threadIdx.x; i < cnt; i += kFitThreads) {
      double* yp = i < kFitCap ? sy + i : yv + i;
      const double wi = i < kFitCap ? sw[i] : wv[i];
      const double yt = *yp - ybar;
      gs[0] += wi * yt * yt;
      *yp = wi * yt;
    }
    all_sum<CS, 2>(gs, red, xchg, ph);   // its barrier also publishes the rewritten slice
    FitData fd{sdt, sy, sw, dtv, yv, wv, cnt, A, 1.0 / A, ybar, gs[0], w.P};
    const double tol_floor = 1e-12 * fd.G;
    const double inf = __longlong_as_double(0x7ff0000000000000ll);
    double th0 = 0.0, th1 = q0, th2 = 0.25;                     // c, q, q_in
    double h0 = 0.25 * w.D0, h1 = 0.25 * q0, h2 = 0.125;
    double dl = 0.0, z = 0.0, best = 0.0;
    int n_eval = 0;
    Trial tr;
    unsigned int in_reach = 0;   // points this thread found inside some candidate's transit, over all sweeps
    // start point: the sweep machinery at zero steps (all six candidates are the start point; lane 2 is read)
    {
      const double D = th1 * fd.P;
      tr.c0 = tr.c1 = tr.cb = th0;
      tr.hb = tr.h2 = tr.h3 = 0.5 * D;
      tr.ib = tr.i2 = tr.i3 = tr.i4 = tr.i5 = 1.0 / (th2 * D);
      tr.reach = tr.hb;
      double chi, d2, z2;
      trial_chi2<CS>(fd, red, xchg, ph, tr, chi, d2, z2, in_reach);
      best = __shfl_sync(0xffffffffu, chi, 2); dl = __shfl_sync(0xffffffffu, d2, 2); z = __shfl_sync(0xffffffffu, z2, 2);
      o.chi2_init = best;
      n_eval = 1;
    }
    // every thread holds the same numbers, so the whole CTA takes the same branches
    for (int level = 0; level < kFitLevels && n_eval < kFitMaxEval; ++level) {
      bool moved = true;
      while (moved && n_eval < kFitMaxEval) {
        moved = false;
        const double tol = fmax(1e-9 * best, tol_floor);
        // the six neighbours, clipped to the bounds; a clipped value equal to the current one is not tried
        const double c_p = fmin(th0 + h0, w.D0), c_m = fmax(th0 - h0, -w.D0);
        const double q_p = fmin(th1 + h1, 1.0), q_m = fmax(th1 - h1, 0.0);
        const double i_p = fmin(th2 + h2, 0.5), i_m = fmax(th2 - h2, 0.0);
        const unsigned have = (c_p != th0 ? 1u : 0u) | (c_m != th0 ? 2u : 0u) | (q_p != th1 ? 4u : 0u) |
                              (q_m != th1 ? 8u : 0u) | (i_p != th2 ? 16u : 0u) | (i_m != th2 ? 32u : 0u);
        if (!have) break;
        const double Db = th1 * fd.P, D2 = q_p * fd.P, D3 = q_m * fd.P;
        tr.c0 = c_p; tr.c1 = c_m; tr.cb = th0;
        tr.hb = 0.5 * Db; tr.h2 = 0.5 * D2; tr.h3 = 0.5 * D3;
        {  // the five reciprocals 1 / ingress, one FP64 division per lane instead of five in every lane
          const double den = lane == 0 ? th2 * Db : lane == 1 ? th2 * D2 : lane == 2 ? th2 * D3
                           : lane == 3 ? i_p * Db : i_m * Db;
          const double inv = 1.0 / den;
          tr.ib = __shfl_sync(0xffffffffu, inv, 0); tr.i2 = __shfl_sync(0xffffffffu, inv, 1);
          tr.i3 = __shfl_sync(0xffffffffu, inv, 2); tr.i4 = __shfl_sync(0xffffffffu, inv, 3);
          tr.i5 = __shfl_sync(0xffffffffu, inv, 4);
        }
        tr.reach = fmax(fmax(tr.h2, tr.h3), tr.hb + fmax(c_p - th0, th0 - c_m));
        double chi, d2, z2;
        trial_chi2<CS>(fd, red, xchg, ph, tr, chi, d2, z2, in_reach);     // lane k < 6: candidate k
        n_eval += __popc(have);
        if (!((have >> lane) & 1u)) chi = inf;            // lanes >= 6 hold +inf already
        double cmin = chi;
#pragma unroll
        for (int o2 = 16; o2 > 0; o2 >>= 1) cmin = fmin(cmin, __shfl_xor_sync(0xffffffffu, cmin, o2));
        // the first candidate (in the order c+, c-, q+, q-, q_in+, q_in-) within tol of the smallest
        const unsigned near = __ballot_sync(0xffffffffu, chi <= cmin + tol) & have;
        const int sel = __ffs(near) - 1;                  // near != 0: the minimum itself qualifies
        const double csel = __shfl_sync(0xffffffffu, chi, sel);
        if (csel < best - tol) {
          best = csel;
          dl = __shfl_sync(0xffffffffu, d2, sel);
          z = __shfl_sync(0xffffffffu, z2, sel);
          th0 = sel == 0 ? c_p : sel == 1 ? c_m : th0;
          th1 = sel == 2 ? q_p : sel == 3 ? q_m : th1;
          th2 = sel == 4 ? i_p : sel == 5 ? i_m : th2;
          moved = true;
        }
      }
      h0 *= 0.5; h1 *= 0.5; h2 *= 0.5;
    }
    o.t0 = pk.t0 + th0; o.q = th1; o.q_in = th2; o.depth = dl; o.z = z; o.chi2 = best; o.n_eval = n_eval;
    if (work_ctr) {   // bench.py's roofline entry of the fit: each such pair is six trapezoid evaluations
#pragma unroll
      for (int o2 = 16; o2 > 0; o2 >>= 1) in_reach += __shfl_xor_sync(0xffffffffu, in_reach, o2);
      if (lane == 0) atomicAdd(&work_ctr[0], (unsigned long long)in_reach);
    }
  }
  if (threadIdx.x == 0 && rank == 0) fits[item] = o;
  if (CS > 1) cooperative_groups::this_cluster().sync();   // no CTA leaves while a neighbour may still read its xchg
}

}  // namespace qlp
