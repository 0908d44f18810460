// pink.cuh -- O9: noise estimates, signal-to-pink-noise and the detection criteria
// (PAPER.md:45-51 with Eq. 2, :55).  Readings in DESIGN.md O9 (after Pont et al. 2006; the VARTOOLS recipe is not
// in the paper): residuals of ALL points of the star against the fitted trapezoid; sigma_w = their unweighted rms
// about the mean; bins of one transit duration D counted from the first point; sigma_r^2 = variance of the bin means
// minus the white part sigma_w^2 mean(1/n_b), floored at 0; n_t, N_t as in O7 with the fitted epoch and duration;
// S/N_pink = delta (1 - q_in) / sqrt(sigma_w^2/n_t + sigma_r^2/N_t); detected = N_t >= 2, S/N_pink > 9, S/N > 9.
//
// One CTA per (star, peak).  Timestamps increase, so a bin is a run of consecutive points: every thread walks a
// contiguous chunk of the star, closes the bins that lie inside its chunk itself and hands its first and last
// (possibly shared) bin to thread 0, which stitches the 2 x 256 partial bins in chunk order.  The integer decisions
// (in transit, transit opened, bin index) use the oracle's unfused FP64 operations; the sums are FP64, single pass,
// shifted by the first residual so that the variances do not cancel.
#pragma once
#include "common.cuh"
#include "fit.cuh"

namespace qlp {

constexpr int kPinkThreads = 256;

struct PinkPartial {
  double bin, sum;   // bin index (a whole number held in a double) and sum of shifted residuals
  int cnt, pad;
};

struct PinkAcc {
  double s1 = 0.0, s2 = 0.0, si = 0.0;   // sums over closed bins of m_b, m_b^2, 1/n_b
  int nb = 0;
  __device__ __forceinline__ void close(double sum, int cnt) {
    const double m = sum / (double)cnt;
    s1 += m; s2 += m * m; si += 1.0 / (double)cnt; ++nb;
  }
};

__global__ void __launch_bounds__(kPinkThreads) pink_kernel(int64_t n_stars, int top_k, const int64_t* __restrict__ row_ptr,
                                                            const double* __restrict__ t, const double* __restrict__ y,
                                                            const qlp_bls_peak* __restrict__ peaks,
                                                            const qlp_bls_trapezoid* __restrict__ fits,
                                                            qlp_bls_pink* __restrict__ out) {
  constexpr int NW = kPinkThreads / 32;
  __shared__ PinkPartial head[kPinkThreads], tail[kPinkThreads];
  __shared__ double red[2 * 5 * NW];
  __shared__ int icnt[3];
  const int64_t item = blockIdx.x;
  const int64_t s = item / top_k;
  if (s >= n_stars) return;
  const qlp_bls_peak pk = peaks[item];
  const qlp_bls_trapezoid ft = fits[item];
  const bool valid = pk.status == 0 && pk.k >= 0 && pk.nb > 0 && ft.status == 0;
  const int64_t a = row_ptr[s], n = valid ? row_ptr[s + 1] - a : 0;
  if (threadIdx.x < 3) icnt[threadIdx.x] = 0;
  __syncthreads();
  const double P = ddiv(1.0, pk.freq);
  const double D = dmul(ft.q, P), half = dmul(0.5, D), ing = dmul(ft.q_in, D);
  const bool bins_on = D > 0.0;
  const double t_first = n > 0 ? t[a] : 0.0;
  const double shift = n > 0 ? dsub(y[a], ft.z) : 0.0;   // any constant: the variances do not depend on it
  const int64_t chunk = (n + kPinkThreads - 1) / kPinkThreads;
  const int64_t lo = min((int64_t)threadIdx.x * chunk, n), hi = min(lo + chunk, n);
  double sr = 0.0, sr2 = 0.0;
  int c_in = 0, c_tr = 0;
  PinkAcc acc;
  PinkPartial hd{0.0, 0.0, 0, 0}, tl{0.0, 0.0, 0, 0};
  bool prev_in = false;
  double prev_cyc = 0.0;
  if (lo < hi && lo > 0) {   // state of the predecessor point (another thread's)
    const double xp = ddiv(dsub(t[a + lo - 1], ft.t0), P);
    prev_cyc = floor(dadd(xp, 0.5));
    prev_in = fabs(dmul(dsub(xp, prev_cyc), P)) <= half;
  }
  double cur = 0.0, bsum = 0.0;
  int bcnt = 0, nbins_seen = 0;
  for (int64_t i = lo; i < hi; ++i) {
    const double ti = t[a + i];
    const double x = ddiv(dsub(ti, ft.t0), P);
    const double cyc = floor(dadd(x, 0.5));
    const double u = fabs(dmul(dsub(x, cyc), P));
    double sh = 0.0;
    if (u < half) { const double d = dsub(half, u); sh = d < ing ? ddiv(d, ing) : 1.0; }
    const double r = dsub(dsub(y[a + i], dsub(ft.z, dmul(ft.depth, sh))), shift);
    sr += r; sr2 += r * r;
    const bool in = u <= half;
    if (in) { ++c_in; c_tr += (prev_in && prev_cyc == cyc) ? 0 : 1; }
    prev_in = in; prev_cyc = cyc;
    if (bins_on) {
      const double b = floor(ddiv(dsub(ti, t_first), D));
      if (bcnt > 0 && b != cur) {
        if (nbins_seen == 0) hd = PinkPartial{cur, bsum, bcnt, 0};   // may have begun in an earlier chunk
        else acc.close(bsum, bcnt);
        ++nbins_seen; bsum = 0.0; bcnt = 0;
      }
      cur = b; bsum += r; ++bcnt;
    }
  }
  if (bcnt > 0) {
    if (nbins_seen == 0) hd = PinkPartial{cur, bsum, bcnt, 0};       // the whole chunk is one bin
    else tl = PinkPartial{cur, bsum, bcnt, 0};                      // may continue in a later chunk
  }
  head[threadIdx.x] = hd; tail[threadIdx.x] = tl;
  double v[5] = {sr, sr2, acc.s1, acc.s2, acc.si};
  int ph = 0;
  {  // block sums in fixed order (as fit.cuh's block_sum, for this CTA size)
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < 5; ++k) v[k] = warp_sum(v[k]);
    if (lane == 0) {
#pragma unroll
      for (int k = 0; k < 5; ++k) red[ph * 5 * NW + k * NW + wid] = v[k];
    }
    int ci = c_in, ct = c_tr, cb = acc.nb;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      ci += __shfl_xor_sync(0xffffffffu, ci, o);
      ct += __shfl_xor_sync(0xffffffffu, ct, o);
      cb += __shfl_xor_sync(0xffffffffu, cb, o);
    }
    if (lane == 0) { atomicAdd(&icnt[0], ci); atomicAdd(&icnt[1], ct); atomicAdd(&icnt[2], cb); }
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    double tot[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      double z = 0.0;
      for (int w = 0; w < NW; ++w) z += red[k * NW + w];
      tot[k] = z;
    }
    // stitch the partial bins in chunk order
    PinkAcc st;
    double rb = 0.0, rs = 0.0;
    int rc = 0;
    for (int k = 0; k < kPinkThreads; ++k) {
      const PinkPartial h = head[k], tl2 = tail[k];
      if (h.cnt > 0) {
        if (rc > 0 && h.bin != rb) { st.close(rs, rc); rs = 0.0; rc = 0; }
        rb = h.bin; rs += h.sum; rc += h.cnt;
      }
      if (tl2.cnt > 0) {   // this chunk held at least two bins: its first one is complete now
        if (rc > 0) { st.close(rs, rc); }
        rb = tl2.bin; rs = tl2.sum; rc = tl2.cnt;
      }
    }
    if (rc > 0) st.close(rs, rc);
    qlp_bls_pink o;
    o.sigma_w = 0.0; o.sigma_r = 0.0; o.depth_eff = 0.0; o.snr_pink = 0.0;
    o.n_t = 0; o.n_transits = 0; o.n_bins = 0; o.detected = 0;
    if (valid && n > 0) {
      const double dn = (double)n;
      const double rbar = tot[0] / dn;
      double var_w = tot[1] / dn - rbar * rbar;
      var_w = var_w > 0.0 ? var_w : 0.0;
      const int nbins = icnt[2] + st.nb;
      double var_r = 0.0;
      if (nbins > 0) {
        const double dnb = (double)nbins;
        const double mbar = (tot[2] + st.s1) / dnb;
        double var_bin = (tot[3] + st.s2) / dnb - mbar * mbar;
        var_bin = var_bin > 0.0 ? var_bin : 0.0;
        var_r = var_bin - var_w * ((tot[4] + st.si) / dnb);
        var_r = var_r > 0.0 ? var_r : 0.0;
      }
      o.sigma_w = sqrt(var_w); o.sigma_r = sqrt(var_r);
      o.depth_eff = ft.depth * (1.0 - ft.q_in);
      o.n_t = icnt[0]; o.n_transits = icnt[1]; o.n_bins = nbins;
      double den = 0.0;
      if (o.n_t > 0 && o.n_transits > 0) den = var_w / (double)o.n_t + var_r / (double)o.n_transits;
      o.snr_pink = den > 0.0 ? o.depth_eff / sqrt(den) : 0.0;
      o.detected = (o.n_transits >= 2 && o.snr_pink > 9.0 && pk.snr > 9.0f) ? 1 : 0;
    }
    out[item] = o;
  }
}

}  // namespace qlp
