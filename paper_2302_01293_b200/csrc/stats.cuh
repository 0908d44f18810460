// stats.cuh -- O7: the "other statistics" of each peak: number of points in,
// before and after transit, number of transits (a transit counts only with data within 0.5 transit durations
// of the expected mid-transit time) and the out-of-transit level.
//
// One CTA per (star, peak rank).  Per point, in FP64 with explicitly unfused operations in the order DESIGN.md
// O7 fixes (the classification is an integer decision, so both sides must round identically):
//   x = (t - T0)/P;  n = floor(x + 0.5);  dt = (x - n) P;   in <=> |dt| <= D/2,  D = (m/nb) P.
// Timestamps increase, so the in-transit points of one cycle are adjacent: a point opens a new transit iff it is
// in transit and its predecessor is not in transit of the same cycle.
#pragma once
#include "common.cuh"

namespace qlp {

__global__ void __launch_bounds__(256) peak_stats_kernel(int64_t n_stars, int top_k, const int64_t* __restrict__ row_ptr,
                                                         const double* __restrict__ t, const double* __restrict__ y,
                                                         const double* __restrict__ dy,
                                                         const qlp_bls_peak* __restrict__ peaks,
                                                         qlp_bls_transit_stats* __restrict__ stats) {
  const int64_t s = blockIdx.x / top_k;
  if (s >= n_stars) return;
  const qlp_bls_peak pk = peaks[blockIdx.x];
  __shared__ int cnt[4];
  __shared__ double red[2][8];
  if (threadIdx.x < 4) cnt[threadIdx.x] = 0;
  __syncthreads();
  const bool valid = pk.status == 0 && pk.k >= 0 && pk.nb > 0;
  const int64_t a = row_ptr[s], n = valid ? row_ptr[s + 1] - a : 0;
  const double P = ddiv(1.0, pk.freq);
  const double D = dmul(ddiv((double)pk.m, (double)pk.nb), P);
  const double hD = dmul(0.5, D), wD = dmul(1.5, D);
  int c_in = 0, c_before = 0, c_after = 0, c_tr = 0;
  double sw = 0.0, swy = 0.0;
  for (int64_t i = threadIdx.x; i < n; i += blockDim.x) {
    const double x = ddiv(dsub(t[a + i], pk.t0), P);
    const double cyc = floor(dadd(x, 0.5));
    const double dt = dmul(dsub(x, cyc), P);
    if (fabs(dt) <= hD) {
      ++c_in;
      bool opens = true;
      if (i > 0) {
        const double xp = ddiv(dsub(t[a + i - 1], pk.t0), P);
        const double cp = floor(dadd(xp, 0.5));
        const double dp = dmul(dsub(xp, cp), P);
        opens = !(fabs(dp) <= hD && cp == cyc);
      }
      c_tr += opens ? 1 : 0;
    } else {
      const double d = dy[a + i];
      const double w = 1.0 / (d * d);
      sw += w; swy += w * y[a + i];
      if (dt < -hD && dt >= -wD) ++c_before;
      if (dt > hD && dt <= wD) ++c_after;
    }
  }
  for (int o = 16; o > 0; o >>= 1) {
    c_in += __shfl_down_sync(0xffffffffu, c_in, o);
    c_before += __shfl_down_sync(0xffffffffu, c_before, o);
    c_after += __shfl_down_sync(0xffffffffu, c_after, o);
    c_tr += __shfl_down_sync(0xffffffffu, c_tr, o);
    sw += __shfl_down_sync(0xffffffffu, sw, o);
    swy += __shfl_down_sync(0xffffffffu, swy, o);
  }
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) {
    atomicAdd(&cnt[0], c_in); atomicAdd(&cnt[1], c_before); atomicAdd(&cnt[2], c_after); atomicAdd(&cnt[3], c_tr);
    red[0][wid] = sw; red[1][wid] = swy;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    double tw = 0.0, twy = 0.0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) { tw += red[0][w]; twy += red[1][w]; }  // fixed order
    qlp_bls_transit_stats o;
    o.n_in = cnt[0]; o.n_before = cnt[1]; o.n_after = cnt[2]; o.n_transits = cnt[3];
    o.oot_level = (valid && tw > 0.0) ? twy / tw : 0.0;
    o.duration = valid ? D : 0.0;
    stats[blockIdx.x] = o;
  }
}

}  // namespace qlp
