// snr_kernel.cuh -- the S4 kernel itself (helpers in snr.cuh).  DESIGN.md O5, O6.
#pragma once
#include "snr.cuh"

namespace qlp {

// Stars in order of decreasing grid size (by power-of-two bucket of n_freq): snr_kernel is one CTA per star and the
// hardware hands out CTAs in index order, so with the longest grids first a 5e5-frequency star does not end up as a
// lone tail while the other SMs idle.  One CTA: count per bucket, scan, scatter (the order inside a bucket is
// whatever the atomics give -- it only decides which CTA runs when, never a result).
__global__ void __launch_bounds__(1024) star_order_kernel(int64_t n_stars, const qlp_bls_star_grid* __restrict__ grid,
                                                          int32_t* __restrict__ order) {
  __shared__ unsigned int cnt[64], base[64];
  if (threadIdx.x < 64) cnt[threadIdx.x] = 0u;
  __syncthreads();
  auto bucket = [&](int64_t s) {
    const qlp_bls_star_grid g = grid[s];
    const long long n = g.status == 0 ? (long long)g.n_freq : 0;
    return n > 0 ? 63 - __clzll(n) + 1 : 0;               // 0: nothing to do; larger = longer grid
  };
  for (int64_t s = threadIdx.x; s < n_stars; s += blockDim.x) atomicAdd(&cnt[bucket(s)], 1u);
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned int acc = 0;
    for (int b = 63; b >= 0; --b) { base[b] = acc; acc += cnt[b]; }
  }
  __syncthreads();
  for (int64_t s = threadIdx.x; s < n_stars; s += blockDim.x) order[atomicAdd(&base[bucket(s)], 1u)] = (int32_t)s;
}

// NT threads per star: the launch with NT = kSnrThreadsLong takes the stars with at least kSnrLongGrid frequencies, the
// one with NT = kSnrThreads the others (each CTA of the wrong launch leaves at once).  On config 5 the kernel's time
// is set by its longest grids (one CTA makes ~9 passes over up to 3 MB of SR): 14.5 -> 8.8 ms with 1,024 threads for
// those; small grids are faster with 256 (config 2: +0.7 % of a step with 1,024 for all).
template <int NT>
__global__ void __launch_bounds__(NT) snr_kernel(
    Params prm, int64_t n_stars, const int64_t* __restrict__ row_ptr, const Point* __restrict__ pts,
    const StarPrep* __restrict__ prep, const qlp_bls_star_grid* __restrict__ grid,
    const int64_t* __restrict__ freq_ptr, const float* __restrict__ sr, const uint32_t* __restrict__ best,
    float* __restrict__ snr_out, qlp_bls_peak* __restrict__ peaks, const int32_t* __restrict__ order) {
  extern __shared__ __align__(16) uint32_t sel_hist[];  // kMaxSel * 256 counters
  __shared__ SnrShared sh;
  if ((int64_t)blockIdx.x >= n_stars) return;
  const int64_t s = order[blockIdx.x];                   // longest grids first (star_order_kernel)
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int K = prm.top_k;
  const qlp_bls_star_grid g = grid[s];
  const int64_t fo = freq_ptr[s], n = freq_ptr[s + 1] - fo;
  if ((n >= kSnrLongGrid) != (NT == kSnrThreadsLong)) return;  // the other launch's star
  qlp_bls_peak* pk = peaks + s * K;
  for (int i = tid; i < K; i += NT) {
    qlp_bls_peak p;
    p.k = -1; p.freq = 0.0; p.period = 0.0; p.t0 = 0.0; p.sr = 0.f; p.snr = 0.f; p.q = 0.f; p.depth = 0.f;
    p.m = 0; p.j = 0; p.nb = 0; p.status = 1;
    pk[i] = p;
  }
  if (g.status != 0 || n <= 0) return;
  const float* srs = sr + fo;
  const double Q = dmul(prm.qmin_fac, g.c_q), dno = (double)prm.noverlap;
  auto freq_at = [&](int64_t k) { double f; int32_t nb; freq_of_k(g.u0, g.h, Q, dno, k, f, nb); return f; };
  // O5.1-2: Sturges bins, equal width in frequency
  const int N = sturges_bins(n);
  const double f0 = freq_at(0), span = dsub(freq_at(n - 1), f0);
  auto bin_at = [&](int64_t k) {
    int b = 0;
    if (span > 0.0) {
      b = (int)dmul(ddiv(dsub(freq_at(k), f0), span), (double)N);
      if (b > N - 1) b = N - 1;
    }
    return b;
  };
  if (tid <= N) {  // bstart[b] = first k with bin(k) >= b
    int64_t lo = 0, hi = n;
    if (tid == 0) hi = 0;
    while (lo < hi) { int64_t mid = lo + ((hi - lo) >> 1); if (bin_at(mid) >= tid) hi = mid; else lo = mid + 1; }
    sh.bstart[tid] = lo;
  }
  __syncthreads();
  // O5.3 + O5.5 first half: medians of every bin and of the whole spectrum
  const int n_sel = 2 * N + 2;
  if (tid < n_sel) {
    const int b = tid >> 1, q = tid & 1;
    const int64_t c = (b < N) ? sh.bstart[b + 1] - sh.bstart[b] : n;
    sh.active[tid] = c > 0;
    sh.rank[tid] = q ? c / 2 : (c - 1) / 2;
    sh.prefix[tid] = 0u;
  }
  __syncthreads();
  radix_select<NT>(sh, sel_hist, n_sel, n, N, true, [&](int64_t k) { return f2key(srs[k]); });
  if (tid == 0) {
    int nk = 0;
    for (int b = 0; b < N; ++b) {
      if (!sh.active[2 * b]) continue;  // empty bins are dropped
      sh.cx[nk] = dadd(f0, ddiv(dmul(dadd((double)b, 0.5), span), (double)N));
      sh.cy[nk] = dmul(0.5, dadd((double)key2f(sh.prefix[2 * b]), (double)key2f(sh.prefix[2 * b + 1])));
      ++nk;
    }
    sh.nk = nk;
    sh.med = dmul(0.5, dadd((double)key2f(sh.prefix[2 * N]), (double)key2f(sh.prefix[2 * N + 1])));
  }
  __syncthreads();
  // O5.5 second half: sigma = 1.4826 * median |SR - median(SR)|
  const double med = sh.med;
  if (tid < 2) { sh.active[tid] = 1; sh.rank[tid] = tid ? n / 2 : (n - 1) / 2; sh.prefix[tid] = 0u; }
  __syncthreads();
  radix_select<NT>(sh, sel_hist, 2, n, N, false, [&](int64_t k) { return f2key((float)fabs(dsub((double)srs[k], med))); });
  if (tid == 0) sh.sigma = dmul(1.4826, dmul(0.5, dadd((double)key2f(sh.prefix[0]), (double)key2f(sh.prefix[1]))));
  __syncthreads();
  const double sigma = sh.sigma;
  auto snr_at = [&](int64_t k) {
    return (sigma > 0.0) ? ddiv(dsub((double)srs[k], trend_at(sh, freq_at(k))), sigma) : 0.0;
  };
  // O5.6 + O6: S/N, per-thread K best local maxima (descending S/N, ties -> lower k)
  double tv[kMaxTopK]; int64_t tk[kMaxTopK];
#pragma unroll
  for (int i = 0; i < kMaxTopK; ++i) { tv[i] = -1.0e300; tk[i] = -1; }
  // contiguous chunk per thread so that neighbours are mostly the thread's own values
  const int64_t per = (n + NT - 1) / NT;
  const int64_t ka = (int64_t)tid * per, kb_ = (ka + per < n) ? ka + per : n;
  if (ka < kb_) {
    double prev = (ka > 0) ? snr_at(ka - 1) : 0.0;
    double cur = snr_at(ka);
    for (int64_t k = ka; k < kb_; ++k) {
      const double nxt = (k + 1 < n) ? snr_at(k + 1) : 0.0;
      if (snr_out) snr_out[fo + k] = (float)cur;
      bool lm = (k == 0 || cur > prev) && (k == n - 1 || cur >= nxt);
      if (n == 1) lm = true;
      if (lm && cur > tv[kMaxTopK - 1]) {
        // insert (cur, k); k ascends within a thread, so equal values stay behind earlier ones
        double v = cur; int64_t kk = k;
#pragma unroll
        for (int i = 0; i < kMaxTopK; ++i) {
          if (v > tv[i]) { double t0 = tv[i]; int64_t t1 = tk[i]; tv[i] = v; tk[i] = kk; v = t0; kk = t1; }
        }
      }
      prev = cur; cur = nxt;
    }
  }
  // K rounds of block-wide argmax over the heads of the per-thread lists
  int n_found = 0;
  for (int round = 0; round < K; ++round) {
    double v = tv[0]; int64_t kk = tk[0]; int t = tid;
    if (kk < 0) v = -2.0e300;
    for (int o = 16; o > 0; o >>= 1) {
      double v2 = __shfl_down_sync(0xffffffffu, v, o);
      int64_t k2 = __shfl_down_sync(0xffffffffu, kk, o);
      int t2 = __shfl_down_sync(0xffffffffu, t, o);
      if (k2 >= 0 && (kk < 0 || v2 > v || (v2 == v && k2 < kk))) { v = v2; kk = k2; t = t2; }
    }
    if (lane == 0) { sh.red_v[wid] = v; sh.red_k[wid] = kk; sh.red_t[wid] = t; }
    __syncthreads();
    if (tid == 0) {
      double bv = sh.red_v[0]; int64_t bk = sh.red_k[0]; int bt = sh.red_t[0];
      for (int w = 1; w < NT / 32; ++w) {
        double v2 = sh.red_v[w]; int64_t k2 = sh.red_k[w];
        if (k2 >= 0 && (bk < 0 || v2 > bv || (v2 == bv && k2 < bk))) { bv = v2; bk = k2; bt = sh.red_t[w]; }
      }
      sh.win_v = bv; sh.win_k = bk; sh.win_t = bt;
      if (bk >= 0) { sh.peak_k[round] = bk; sh.peak_v[round] = bv; sh.n_peaks = round + 1; }
      else if (round == 0) sh.n_peaks = 0;
    }
    __syncthreads();
    if (sh.win_k < 0) break;
    n_found = round + 1;
    if (tid == sh.win_t) {  // pop the winner's head
#pragma unroll
      for (int i = 0; i + 1 < kMaxTopK; ++i) { tv[i] = tv[i + 1]; tk[i] = tk[i + 1]; }
      tv[kMaxTopK - 1] = -1.0e300; tk[kMaxTopK - 1] = -1;
    }
    __syncthreads();
  }
  // peak records: refold at each peak frequency for (r, s) of its best box (O4 "derived for peaks")
  const int64_t pa = row_ptr[s], np = row_ptr[s + 1] - pa;
  const StarPrep sp = prep[s];
  for (int i = 0; i < n_found; ++i) {
    const int64_t k = sh.peak_k[i];
    double f; int32_t nb;
    freq_of_k(g.u0, g.h, Q, dno, k, f, nb);
    const uint32_t bst = best[fo + k];
    const int m = (int)(bst >> 24), j = (int)(bst & 0xffffffu);
    const double dnb = (double)nb, Kc = (dnb + 1.0) * QLP_TWO52;
    if (tid == 0) { sh.accW = 0ull; sh.accS = 0ll; }
    __syncthreads();
    unsigned long long aw = 0ull; long long as = 0ll;
    for (int64_t p = tid; p < np; p += NT) {
      const Point pt = pts[pa + p];
      int b = bin_of(f, pt.tau, dnb, Kc) - j;
      if (b < 0) b += nb;
      if (b < m) { aw += pt.W; as += pt.S; }
    }
    for (int o = 16; o > 0; o >>= 1) { aw += __shfl_down_sync(0xffffffffu, aw, o); as += __shfl_down_sync(0xffffffffu, as, o); }
    if (lane == 0) { atomicAdd(&sh.accW, aw); atomicAdd((unsigned long long*)&sh.accS, (unsigned long long)as); }
    __syncthreads();
    if (tid == 0) {
      const double r = (double)sh.accW / (double)kScaleW;
      const double sv = (sp.scale_s > 0.0) ? (double)sh.accS / sp.scale_s : 0.0;
      qlp_bls_peak p;
      p.k = k; p.freq = f; p.period = ddiv(1.0, f);
      p.t0 = dadd(g.t_ref, ddiv(ddiv(dadd((double)j, dmul(0.5, (double)m)), dnb), f));
      p.sr = srs[k]; p.snr = (float)sh.peak_v[i];
      p.q = (float)((double)m / dnb);
      p.depth = (r > 0.0 && r < 1.0) ? (float)(-sv / (r * (1.0 - r))) : 0.f;
      p.m = m; p.j = j; p.nb = nb; p.status = 0;
      pk[i] = p;
    }
    __syncthreads();
  }
}

}  // namespace qlp
