// prep.cuh -- S0: Kovacs et al. (2002) weights and the centred series (PAPER.md:13, :37 name the
// algorithm; O2), converted to the 16-byte fixed-point point record the fold kernel
// streams.
//
//   W_sum = sum dy^-2;  w_i = dy_i^-2 / W_sum;  ybar = sum w_i y_i;  ytilde_i = y_i - ybar;
//   tau_i = t_i - t_ref.
//
// Fixed point: FP32 atomicAdd on shared memory is a compare-and-swap
// loop on sm_100a (ATOMS.CAST.SPIN), the 32-bit integer add is native (ATOMS.ADD), so the
// histograms are integers:
//   W_i = round(w_i * (2^32 - 2^22))        -> any sum of W_i stays below 2^32 for N < 2^23;
//   S_i = round(w_i ytilde_i * scale_s)     -> scale_s chosen per star so that no phase bin of any
//         grid frequency can overflow int32.  A bin of duration D <= Q/(noverlap u) is visited in at most
//         C = f T + 2 cycles; for ANY spacing threshold d, a window of length D holds at most D/d + 1 points
//         whose spacings are >= d, and every spacing below d adds at most one point to one window, so
//             points per bin <= C (D/d + 1) + #{spacings < d}.
//         The spacings are histogrammed in quarter-octave buckets and the best threshold is taken: a few
//         near-coincident timestamps (overlapping sectors or cameras) cost a few counts, not the bound
//         (with the plain minimum spacing one such pair would degrade the bound to N and cost
//         log2(N / cnt) bits of S resolution on a long star).
// One CTA per star, three passes over its points (the 2nd and 3rd hit L2).
#pragma once
#include "common.cuh"

namespace qlp {

__device__ __forceinline__ double block_sum(double v, double* sh) {
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  __syncthreads();
  if (lane == 0) sh[wid] = v;
  __syncthreads();
  if (wid == 0) {
    v = (lane < (int)(blockDim.x >> 5)) ? sh[lane] : 0.0;
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if (lane == 0) sh[0] = v;
  }
  __syncthreads();
  return sh[0];
}
__device__ __forceinline__ double block_max(double v, double* sh) {
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, o));
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  __syncthreads();
  if (lane == 0) sh[wid] = v;
  __syncthreads();
  if (wid == 0) {
    v = (lane < (int)(blockDim.x >> 5)) ? sh[lane] : -1.0e300;
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, o));
    if (lane == 0) sh[0] = v;
  }
  __syncthreads();
  return sh[0];
}

// Quarter-octave buckets of the spacing between consecutive timestamps, 2^-40 d ... 2^12 d.  The bucket of d is
// (biased exponent, top two mantissa bits) of its FP64 pattern; everything below 2^-40 d (zero, negative and NaN
// spacings too) lands in bucket 0, everything above in the last one.
constexpr int kSpLoExp = 1023 - 40;                    // biased exponent of 2^-40
constexpr int kSpBuckets = 52 * 4;
__device__ __forceinline__ int spacing_bucket(double d) {
  if (!(d > 0.0)) return 0;
  const int idx = (__double2hiint(d) >> 18) - (kSpLoExp << 2);
  return idx < 0 ? 0 : (idx >= kSpBuckets ? kSpBuckets - 1 : idx);
}
__device__ __forceinline__ double spacing_bucket_edge(int b) {   // lower edge of bucket b
  return __hiloint2double((b + (kSpLoExp << 2)) << 18, 0);
}

__global__ void __launch_bounds__(256) prep_kernel(Params prm, int64_t n_stars, const int64_t* __restrict__ row_ptr,
                                                   const double* __restrict__ t, const double* __restrict__ y,
                                                   const double* __restrict__ dy,
                                                   const qlp_bls_star_grid* __restrict__ grid,
                                                   Point* __restrict__ pts, StarPrep* __restrict__ prep) {
  const int64_t s = blockIdx.x;
  if (s >= n_stars) return;
  __shared__ double sh[32];
  const int64_t a = row_ptr[s], n = row_ptr[s + 1] - a;
  const qlp_bls_star_grid g = grid[s];
  const double* ts = t + a;
  const double* ys = y + a;
  const double* ds = dy + a;
  // pass 1: W_sum, sum y/dy^2, histogram of the spacings in quarter-octave buckets
  __shared__ unsigned int sp_hist[kSpBuckets];
  for (int i = threadIdx.x; i < kSpBuckets; i += blockDim.x) sp_hist[i] = 0u;
  __syncthreads();
  double acc_w = 0.0, acc_wy = 0.0;
  for (int64_t i = threadIdx.x; i < n; i += blockDim.x) {
    double d = ds[i];
    double iv = 1.0 / (d * d);
    acc_w += iv;
    acc_wy += iv * ys[i];
    if (i + 1 < n) atomicAdd(&sp_hist[spacing_bucket(ts[i + 1] - ts[i])], 1u);
  }
  const double W = block_sum(acc_w, sh);
  const double WY = block_sum(acc_wy, sh);
  const double ybar = (n > 0) ? WY / W : 0.0;
  // pass 2: max |w ytilde|
  double mx = 0.0;
  for (int64_t i = threadIdx.x; i < n; i += blockDim.x) {
    double d = ds[i];
    double w = (1.0 / (d * d)) / W;
    mx = fmax(mx, fabs(w * (ys[i] - ybar)));
  }
  const double wy_max = block_max(mx, sh);
  // bound on the number of points that can share one phase bin at any grid frequency
  // (thread 0 walks the buckets; the result goes through shared memory so that every thread holds the same bits)
  __shared__ double cnt_sh;
  if (threadIdx.x == 0) {
    double cnt = (double)n;
    if (g.status == 0 && g.n_freq > 0) {
      const double Q = prm.qmin_fac * g.c_q;
      double u_lo = g.u0, u_hi = g.u0 + (double)g.n_freq * g.h;
      if (g.h < 0.0) {  // frequency-uniform grid (O1.10c): u0 = f_min, h = -df
        u_lo = cbrt_det(g.u0);
        u_hi = cbrt_det(g.u0 + (double)g.n_freq * (-g.h));
      }
      const double no = (double)prm.noverlap;
      // sum over cycles of D/d: D = Q/(no u) days per bin and cycle, C = f T + 2 cycles, evaluated at the grid
      // ends (u_hi for the f T part, u_lo for the + 2 part); cycles = C at the highest frequency
      const double span = Q * g.baseline * u_hi * u_hi / no + 2.0 * Q / (no * u_lo);
      const double cycles = u_hi * u_hi * u_hi * g.baseline + 2.0;
      double n_small = 0.0;   // spacings below the lower edge of bucket b
      for (int b = 0; b < kSpBuckets; ++b) {
        const double d = spacing_bucket_edge(b);
        if (b > 0) {          // bucket 0 also holds zero / negative / NaN spacings: no threshold below it
          const double bound = (span / d + cycles) * 1.01 + 2.0 + n_small;
          if (bound < cnt) cnt = bound;
        }
        n_small += (double)sp_hist[b];
      }
    }
    if (cnt < 1.0) cnt = 1.0;
    cnt_sh = cnt;
  }
  __syncthreads();
  const double cnt = cnt_sh;
  double scale_s = 0.0;
  if (wy_max > 0.0 && isfinite(wy_max)) scale_s = (2147483647.0 - cnt - 1.0) / (cnt * wy_max);
  int32_t status = (n >= (1 << 22)) ? 5 : 0;
  if (!(W > 0.0) || !isfinite(W)) status = 6;
  // pass 3: write the point records
  Point* ps = pts + a;
  for (int64_t i = threadIdx.x; i < n; i += blockDim.x) {
    double d = ds[i];
    double w = (1.0 / (d * d)) / W;
    double wy = w * (ys[i] - ybar);
    Point p;
    p.tau = dsub(ts[i], g.t_ref);
    p.W = (status == 0) ? __double2uint_rn(w * (double)kScaleW) : 0u;
    p.S = (status == 0) ? __double2int_rn(wy * scale_s) : 0;
    ps[i] = p;
  }
  if (threadIdx.x == 0) {
    StarPrep sp;
    sp.ybar = ybar; sp.wsum = W; sp.scale_s = scale_s;
    sp.inv_w = (float)(1.0 / (double)kScaleW);
    sp.inv_s = (scale_s > 0.0) ? (float)(1.0 / scale_s) : 0.0f;
    sp.status = status; sp.pad_ = 0;
    prep[s] = sp;
  }
}

// Optional input validation (config flags bit0).  which = 0: t finite and strictly increasing within each star,
// row_ptr non-decreasing; which = 1: y finite, dy finite and > 0.  Counts violations into *bad.
__global__ void validate_kernel(int which, int64_t n_stars, const int64_t* __restrict__ row_ptr,
                                const double* __restrict__ t, const double* __restrict__ y,
                                const double* __restrict__ dy, unsigned long long* __restrict__ bad) {
  const int64_t s = blockIdx.x;
  if (s >= n_stars) return;
  const int64_t a = row_ptr[s], n = row_ptr[s + 1] - a;
  unsigned long long cnt = 0;
  if (n < 0) cnt = 1;
  for (int64_t i = threadIdx.x; i < n; i += blockDim.x) {
    if (which == 0) {
      const double ti = t[a + i];
      if (!isfinite(ti)) ++cnt;
      if (i + 1 < n && !(t[a + i + 1] > ti)) ++cnt;
    } else {
      const double d = dy[a + i];
      if (!isfinite(y[a + i]) || !isfinite(d) || !(d > 0.0)) ++cnt;
    }
  }
  for (int o = 16; o > 0; o >>= 1) cnt += __shfl_down_sync(0xffffffffu, cnt, o);
  if ((threadIdx.x & 31) == 0 && cnt) atomicAdd(bad, cnt);
}

// test-only: S0 outputs of one star as plain arrays
__global__ void debug_prep_kernel(const int64_t* __restrict__ row_ptr, const Point* __restrict__ pts,
                                  const StarPrep* __restrict__ prep, int64_t star, double* __restrict__ tau,
                                  float* __restrict__ w, float* __restrict__ wy) {
  const int64_t a = row_ptr[star], n = row_ptr[star + 1] - a;
  const StarPrep sp = prep[star];
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    Point p = pts[a + i];
    tau[i] = p.tau;
    w[i] = (float)p.W * sp.inv_w;
    wy[i] = (float)p.S * sp.inv_s;
  }
}

// test-only: O3 bin of every point of one star at grid frequency k (same device function as the fold)
__global__ void debug_bins_kernel(Params prm, const int64_t* __restrict__ row_ptr, const double* __restrict__ t,
                                  const qlp_bls_star_grid* __restrict__ grid, int64_t star, int64_t k,
                                  int32_t* __restrict__ out) {
  const int64_t a = row_ptr[star], n = row_ptr[star + 1] - a;
  const qlp_bls_star_grid g = grid[star];
  double f; int32_t nb;
  freq_of_k(g.u0, g.h, dmul(prm.qmin_fac, g.c_q), (double)prm.noverlap, k, f, nb);
  const double dnb = (double)nb;  // the three-instruction form the fold kernel uses
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    double tau = dsub(t[a + i], g.t_ref);
    out[i] = bin_of3(f, tau, dnb, (uint32_t)nb);
  }
}

}  // namespace qlp
