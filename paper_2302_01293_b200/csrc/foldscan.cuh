// foldscan.cuh -- S2 fold-and-bin fused with S3 box-scan (O3, O4; the BLS of Kovacs et
// al. 2002 that PAPER.md:13 and :37 name, on the Keplerian duration ladder of PAPER.md:19, :35).
//
// Work unit ("tile"): one star x `cols` consecutive grid frequencies.  Each frequency owns one
// COLUMN of two integer histograms in shared memory (sum of W and sum of S per phase bin); a lane of
// a warp owns one column, so the 32 lanes of a warp fold the SAME point at 32 different
// frequencies: the point is one broadcast 16-byte load, the 32 accumulations go to 32 different
// banks, and the two accumulations are native ATOMS.ADD (no return value -> no dependent chain).
// The warps of the CTA split the point stream; atomics make their concurrent updates safe.
// After the fold the histograms never leave the SM: the box scan runs on them in place and only
// SR(f) and the best (m, j) go to HBM (8 bytes per frequency).
//
// nb (phase bins) falls from nb_max to ~38 along a star's grid, so tiles come in classes that trade
// columns for bins within the same shared-memory budget (class_cols / class_nbcap in common.cuh).
// In the narrow classes (fewer than 32 columns) the spare lanes of a warp take consecutive points.
// Each class is one persistent launch that pulls tile numbers from an atomic counter; a tile number
// is mapped to (star, k0) by a binary search in the per-class prefix sums built by tile_bounds_kernel
// and tile_scan_kernel, so no tile list is materialised.
#pragma once
#include "common.cuh"

namespace qlp {

// ---- tile bookkeeping -------------------------------------------------------------------------
// kb[s][c] = first k of star s whose nb_k <= class_nbcap(c) (n_freq if none); class c then covers
// k in [kb[s][c], kb[s][c-1]) for c >= 1 and [kb[s][0], n_freq) for c = 0.  nb_k is non-increasing
// in k because every operation of O1.8 is monotone.
__global__ void tile_bounds_kernel(Params prm, int64_t n_stars, const qlp_bls_star_grid* __restrict__ grid,
                                   int32_t force_path, int64_t* __restrict__ kb, int64_t* __restrict__ cnt) {
  int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (s >= n_stars) return;
  const qlp_bls_star_grid g = grid[s];
  const int64_t nf = (g.status == 0) ? g.n_freq : 0;
  const double Q = dmul(prm.qmin_fac, g.c_q);
  int64_t prev_lo = nf;
  for (int c = 0; c < kNumClasses; ++c) {
    int cap = class_nbcap(c);
    int64_t lo = 0, hi = nf;  // answer in [0, nf]
    if (force_path > 0 && c < force_path - 1) lo = nf;  // test hook: nothing below class force_path - 1
    else {
      while (lo < hi) {
        int64_t mid = lo + ((hi - lo) >> 1);
        double f; int32_t nb;
        freq_of_k(g.u0, g.h, Q, (double)prm.noverlap, mid, f, nb);
        if (nb <= cap) hi = mid; else lo = mid + 1;
      }
    }
    if (lo > prev_lo) lo = prev_lo;
    kb[s * kNumClasses + c] = lo;
    int64_t span = prev_lo - lo;
    int cols = class_cols(c);
    cnt[c * n_stars + s] = (span + cols - 1) / cols;
    prev_lo = lo;
  }
}

// One CTA per class: exclusive scan of cnt[c][0..S) -> off[c][0..S].
__global__ void __launch_bounds__(1024) tile_scan_kernel(int64_t n_stars, const int64_t* __restrict__ cnt,
                                                         int64_t* __restrict__ off) {
  const int c = blockIdx.x;
  const int64_t* in = cnt + (int64_t)c * n_stars;
  int64_t* out = off + (int64_t)c * (n_stars + 1);
  __shared__ int64_t warp_sum[32];
  __shared__ int64_t carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int64_t base = 0; base < n_stars; base += blockDim.x) {
    int64_t i = base + threadIdx.x;
    int64_t v = (i < n_stars) ? in[i] : 0;
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
    if (i < n_stars) out[i] = prefix;
    __syncthreads();
    if (threadIdx.x == blockDim.x - 1) carry = prefix + v;
    __syncthreads();
  }
  if (threadIdx.x == 0) out[n_stars] = carry;
}

// ---- TMA bulk-copy staging of the point stream (cp.async.bulk -> SASS UBLKCP) -----------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE;\n"
      "bra WAIT_LOOP;\n"
      "DONE:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_load(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// Value s^2 / (r (1 - r)) of one box for the scan's running maximum, with O4's exclusions folded into the
// arithmetic: d = r (c - r) with c = 1 - 2^-24 is negative for r >= 1 (the value then loses every fmaxf against
// 0), and d = 0 only for r = 0, where s = 0 too and 0 * inf = NaN loses as well.  MUFU.RCP is within 1 ulp; the
// relative change of d by c is 6e-8 / (1 - r).  Explicit _rn intrinsics: the same call gives the same bits.
__device__ __forceinline__ float box_value(float r, float sm) {
  const float t = __fadd_rn(0.99999994f, -r);
  const float d = __fmul_rn(r, t);
  float inv;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(inv) : "f"(d));
  return __fmul_rn(__fmul_rn(sm, sm), inv);
}

struct TileInfo {
  int64_t k0, pt_begin, n_pts, out_base;
  double u0, h, Q;
  float inv_w, inv_s;
  int32_t ncols, nb_tile;
  int32_t valid;
};


// ---- the fused kernel ---------------------------------------------------------------------------
// MW = widest box (window registers), CTOT = columns per CTA of this class (compile time so that the
// two atomics of one evaluation differ by an immediate offset and the row stride is a shift), WM = the
// ladder as a compile-time bit mask (bit m set <=> width m is searched) or 0 = take it from prm.wmask.
// Fold phase: every warp is a slice of the point stream.  With CTOT >= 32 a lane owns R = CTOT/32
// columns (lane, lane+32, ...), so one broadcast LDS.128 of a point feeds R evaluations: the load
// costs two shared-memory wavefronts, the two atomics of an evaluation one each, and the
// shared-memory pipe (one wavefront per clock per SM) is what binds.
// With CTOT < 32 the spare lanes take 32/CTOT consecutive points.
// (f_k, nb_k) inside the fold kernel.  Only the kernels with the run-time ladder (WM == 0) know the
// frequency-uniform comparison grid (O1.10c; the host sends such a context to them): the kernels compiled for the
// paper's ladder keep the branch-free f^(1/3) law, so the comparison grid costs the headline path nothing -- with
// the test inlined into them the 64-column class lost 4.6 % to a different register allocation of its inner loop.
template <bool ANY_GRID>
__device__ __forceinline__ void tile_freq_of_k(double u0, double h, double Q, double noverlap, int64_t k, double& f,
                                               int32_t& nb) {
  if (ANY_GRID) freq_of_k(u0, h, Q, noverlap, k, f, nb);
  else freq_of_k_cube(u0, h, Q, noverlap, k, f, nb);
}

// Register budget of the fold kernels, through __launch_bounds__(T, B): ptxas keeps a kernel within 65536 / (T * B)
// registers per thread (T >= kThreads: the launches use kThreads).  128 columns: 64 registers, the budget of two
// CTAs per SM (class 0).  The other caps are tuning, measured per class on config 5: the
// 32-column (paired) loop is 8 % faster at 56 registers than with the 75 ptxas takes when left alone (0.415 -> 0.449
// of the peak; 64: 0.422, 48: 0.407, 40 with spills: 0.396), the 64-column loop 2 % faster at 72 (70 used; 78
// uncapped: 0.506 -> 0.515; 64: 0.498).  Giving class 1 a build of its own with more than 64 registers made it
// slower (72: 0.572, 94: 0.549, 118 with 8 points in flight: 0.534, against 0.590), and so did every cap tried on
// the 16-column class (71: 0.297, 64: 0.289, 56: 0.286, against 0.307 at 79).
template <int CTOT> constexpr int fold_lb_threads() { return CTOT == 64 ? 832 : (CTOT == 32 ? 576 : kThreads); }
template <int CTOT> constexpr int fold_lb_blocks() { return (CTOT == 128 || CTOT == 32) ? 2 : 1; }
template <int MW, int CTOT, uint32_t WM>
__global__ void __launch_bounds__(fold_lb_threads<CTOT>(), fold_lb_blocks<CTOT>()) foldscan_kernel(
    Params prm, int cls, int64_t n_stars, const int64_t* __restrict__ row_ptr, const Point* __restrict__ pts,
    const StarPrep* __restrict__ prep, const qlp_bls_star_grid* __restrict__ grid,
    const int64_t* __restrict__ freq_ptr, const int64_t* __restrict__ tile_off, const int64_t* __restrict__ kb,
    unsigned long long* __restrict__ counter, float* __restrict__ sr, uint32_t* __restrict__ best,
    unsigned long long* __restrict__ phase /* NULL, or this class's 5 counters: set-up, fold, scan clocks of
                                              thread 0, point x frequency evaluations, tiles */) {
  extern __shared__ __align__(16) unsigned char smem[];
  Point* pbuf = reinterpret_cast<Point*>(smem);                          // [2][kChunk]
  uint64_t* mbar = reinterpret_cast<uint64_t*>(smem + 2 * kChunk * 16);  // [2]
  uint32_t* hist = reinterpret_cast<uint32_t*>(smem + kStageBytes);      // [nb_tile][2 * CTOT]
  __shared__ TileInfo ti;
  __shared__ int64_t s_tile;
  constexpr int STRIDE = 2 * CTOT;              // words per histogram row: [W x CTOT][S x CTOT]
  // Lane layout of the fold.  128 and 64 columns: the 32 lanes own 4 resp. 2 columns each and fold the same point.
  // 32 columns ("paired"): a half-warp owns the columns (2 per lane) and the two half-warps fold two different
  // points, so a point load (2 shared-memory wavefronts whether the lanes read one or two points) feeds 2
  // evaluations per lane instead of 1.  The two half-warps must not meet on a bank: the second one walks its columns
  // in the order r ^ 1, so in every instruction the halves work on columns whose indices differ in bit 4 -- the other
  // half of the banks -- with the same immediate offsets as the wide layouts (measured on config 5: class 3 0.374 ->
  // 0.415 of the peak; the same layout with 4 columns per lane in the 64-column class: 0.506 -> 0.494, not used).
  // 16 columns ("quad"): a quarter-warp owns the columns (2 per lane), four points per warp; quarter-warps 1 and 3 walk
  // their columns in the order r ^ 1 and quarter-warps 2 and 3 add S before W, so the four of them use the four
  // quarters of the banks (W and S words of columns 0-7 and 8-15) in every instruction.
  // 8 columns and fewer: one column per lane, 32 / CTOT points per warp, odd point-lanes add S before W.
  constexpr bool PAIRED = QLP_PAIRED_CLASSES && CTOT == 32;
  constexpr bool QUAD = QLP_PAIRED_CLASSES && CTOT == 16;
  constexpr int CW = QUAD ? 8 : (CTOT < 32 ? CTOT : (PAIRED ? 16 : 32));   // distinct columns across the lanes of a warp
  constexpr int R = CTOT / CW;                  // columns per lane
  constexpr int HPW = 32 / CW;                  // points per warp iteration
  constexpr int STEP = kWarps * HPW;            // points consumed per iteration by the CTA
  constexpr int ITERS = kChunk / STEP;
  // points in flight per lane: 4 (2 and 8 measured slower in every class down to 16 columns); the 8-column class
  // takes its whole chunk share of 8 (0.195 -> 0.214 of the peak)
  constexpr int UW = (CTOT == 8) ? 8 : 4;
  constexpr int U = ITERS < UW ? ITERS : UW;
  static_assert(ITERS >= 1 && ITERS % U == 0, "chunk must be a multiple of the CTA's point step");
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int col0 = lane % CW;                   // first column of this lane in the fold phase
  const int hsub = lane / CW;
  const double dno = (double)prm.noverlap;
  const int64_t n_tiles = tile_off[n_stars];
  uint32_t use0 = 0, use1 = 0;                  // completed uses of each staging buffer (phase parity)
  if (tid == 0) {
    mbar_init(&mbar[0], 1);
    mbar_init(&mbar[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }

  for (;;) {
    __syncthreads();  // previous tile fully written before ti / hist are reused
    const long long clk0 = phase ? clock64() : 0;
    if (tid == 0) s_tile = (int64_t)atomicAdd(counter, 1ull);
    __syncthreads();
    const int64_t tile = s_tile;
    if (tile >= n_tiles) break;
    // star of this tile = last s with tile_off[s] <= tile: a 512-way search, one global latency per level
    int64_t lo = 0, len = n_stars + 1;
    while (len > 1) {
      const int64_t stride = (len + kThreads - 1) / kThreads;
      const int64_t off = (int64_t)tid * stride;
      const int hit = (off < len) && (tile_off[lo + off] <= tile);
      const int c = __syncthreads_count(hit);
      lo += (int64_t)(c - 1) * stride;
      const int64_t rest = len - (int64_t)(c - 1) * stride;
      len = stride < rest ? stride : rest;
    }
    if (tid == 0) {
      TileInfo x;
      x.valid = 1;
      {
        const int64_t s = lo;
        const qlp_bls_star_grid g = grid[s];
        const StarPrep sp = prep[s];
        const int64_t k_lo = kb[s * kNumClasses + cls];
        const int64_t k_hi = (cls == 0) ? g.n_freq : kb[s * kNumClasses + cls - 1];
        x.k0 = k_lo + (tile - tile_off[s]) * CTOT;
        int64_t rem = k_hi - x.k0;
        x.ncols = rem < CTOT ? (int32_t)rem : CTOT;
        x.pt_begin = row_ptr[s];
        x.n_pts = row_ptr[s + 1] - row_ptr[s];
        x.out_base = freq_ptr[s];
        x.u0 = g.u0; x.h = g.h; x.Q = dmul(prm.qmin_fac, g.c_q);
        x.inv_w = sp.inv_w; x.inv_s = sp.inv_s;
        double f; int32_t nb;
        tile_freq_of_k<WM == 0u>(x.u0, x.h, x.Q, dno, x.k0, f, nb);
        x.nb_tile = nb;
        // start streaming the first two chunks of the star's points
        const Point* src = pts + x.pt_begin;
        const int64_t n = x.n_pts;
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        if (n > 0) {
          const uint32_t b0 = (uint32_t)((n < kChunk ? n : kChunk) * 16);
          mbar_expect_tx(&mbar[0], b0);
          bulk_load(pbuf, src, b0, &mbar[0]);
        }
        if (n > kChunk) {
          const int64_t r = n - kChunk;
          const uint32_t b1 = (uint32_t)((r < kChunk ? r : kChunk) * 16);
          mbar_expect_tx(&mbar[1], b1);
          bulk_load(pbuf + kChunk, src + kChunk, b1, &mbar[1]);
        }
      }
      ti = x;
    }
    __syncthreads();
    const int nb_tile = ti.nb_tile;
    {  // zero the histograms of this tile
      const int words = nb_tile * STRIDE;  // multiple of 2; hist is 16-byte aligned
      uint4* h4 = reinterpret_cast<uint4*>(hist);
      for (int i = tid; i < (words >> 2); i += kThreads) h4[i] = make_uint4(0u, 0u, 0u, 0u);
      if (tid < (words & 3)) hist[(words & ~3) + tid] = 0u;
    }
    long long clk1s = 0;
    // ---- S2: fold ----
    {
      // A column beyond the tile's last frequency folds with f = 0, nb = 1 into row 0 of its own
      // (never scanned) column: cheaper than predicating every atomic.
      double f[R], dnb[R];
      uint32_t neg_nb_row[R];  // -(nb * row bytes) mod 2^32
      uint32_t lane_off[R];    // byte offset of the lane's r-th column in a histogram row; where the columns of a
                               // lane are CW apart in a fixed order it is lane_off[0] + an immediate
#pragma unroll
      for (int r = 0; r < R; ++r) {
        const int col = col0 + CW * ((PAIRED || QUAD) ? (r ^ (hsub & 1)) : r);
        lane_off[r] = (uint32_t)((PAIRED || QUAD) ? col : col0) * 4u;
        // lanes that add S first (see below) start CTOT words further: folded into the lane's offset here
        if (HPW > 1 && !PAIRED) lane_off[r] += (uint32_t)(((QUAD ? (hsub & 2) != 0 : (hsub & 1) != 0) ? CTOT : 0) * 4);
        f[r] = 0.0;
        int32_t nbk = 1;
        if (col < ti.ncols) tile_freq_of_k<WM == 0u>(ti.u0, ti.h, ti.Q, dno, ti.k0 + col, f[r], nbk);
        dnb[r] = (double)nbk;
        neg_nb_row[r] = 0u - (uint32_t)nbk * (uint32_t)(STRIDE * 4);
      }
      const int64_t n = ti.n_pts;
      const Point* src = pts + ti.pt_begin;
      const int64_t n_chunks = (n + kChunk - 1) / kChunk;
      const bool swap_ws = (HPW > 1) && !PAIRED && (QUAD ? (hsub & 2) != 0 : (hsub & 1) != 0);
      const uint32_t sel_first = swap_ws ? 0x7654u : 0x3210u, sel_second = swap_ws ? 0x3210u : 0x7654u;  // W,S or S,W
      unsigned char* hbytes = reinterpret_cast<unsigned char*>(hist);
      __syncthreads();  // histograms zeroed
      clk1s = phase ? clock64() : 0;
      for (int64_t c = 0; c < n_chunks; ++c) {
        const int b = (int)(c & 1);
        Point* buf = pbuf + b * kChunk;
        mbar_wait(&mbar[b], (b ? use1 : use0) & 1u);
        if (b) ++use1; else ++use0;
        const int64_t left = n - c * kChunk;
        (void)QLP_IN_BOUNDS(kChkStage, left > 0 && b >= 0 && b < 2);
        if (left < kChunk) {  // pad the tail with weightless points so that every chunk is full
          for (int i = (int)left + tid; i < kChunk; i += kThreads) {
            Point z; z.tau = 0.0; z.W = 0u; z.S = 0;
            buf[i] = z;
          }
          __syncthreads();
        }
        const int4* p4 = reinterpret_cast<const int4*>(buf) + warp * HPW + hsub;
        // the 64-column kernel gains 1.3 % from two iterations per loop trip (the 128-column ones lose 3-6 %)
        constexpr int UNR_IT = (CTOT == 64) ? 2 : 1;
#pragma unroll UNR_IT
        for (int it = 0; it < ITERS; it += U) {
          int4 v[U];
#pragma unroll
          for (int u = 0; u < U; ++u) v[u] = p4[(it + u) * STEP];
          // Order of the U x R evaluations of an iteration (all unrolled; ptxas keeps the atomics in source order).
          // The 128- and 64-column kernels walk a lane's columns in the outer loop and the points in the inner one
          // (measured: class 0 0.662 -> 0.667, class 1 0.590 -> 0.594, class 2 0.515 -> 0.525 of the peak); the paired
          // and quad kernels keep the points outside (the other order: 0.449 -> 0.405 and 0.307 -> 0.303).
          constexpr bool R_MAJOR = CTOT >= 64;
#pragma unroll
          for (int e = 0; e < U * R; ++e) {
            const int u = R_MAJOR ? e % U : e / R;
            const int r = R_MAJOR ? e / U : e % R;
            const double tau = __hiloint2double(v[u].y, v[u].x);
            {
              // byte offset of the bin's row: (I - nb g) * row bytes, as I * row + g * (-nb row) (+ lane)
              uint32_t I, g;
              bin_parts(f[r], tau, dnb[r], I, g);
              const uint32_t off = g * neg_nb_row[r] + (I * (uint32_t)(STRIDE * 4) + lane_off[r]);
              uint32_t* cell = reinterpret_cast<uint32_t*>(hbytes + off) + ((PAIRED || QUAD) ? 0 : CW * r);
              // check build: the cell lies inside this tile's histogram (bin < nb of the column <= nb_tile)
              // (the narrow classes' lanes that add S first start in the S half of the row: up to 2 CTOT words)
              if (!QLP_IN_BOUNDS(kChkFoldCell, off / (uint32_t)(STRIDE * 4) < (uint32_t)nb_tile &&
                                                   (off % (uint32_t)(STRIDE * 4)) / 4u + (uint32_t)((PAIRED || QUAD) ? 0 : CW * r) <
                                                       (uint32_t)((HPW > 1 && !PAIRED) ? STRIDE : CTOT)))
                continue;
              if (HPW == 1 || PAIRED) {
                atomicAdd(cell, (uint32_t)v[u].z);
                atomicAdd(cell + CTOT, (uint32_t)v[u].w);
              } else {
                // Narrow classes: the lanes that share a column fold different points, and with a row of
                // 2*CTOT <= 32 words they would meet on one bank in both atomics.  Odd point-lanes therefore
                // add S first and W second: in each instruction the two parities use different banks.
                // The lane's first word is W or S of its column (lane_off holds which); the other one is CTOT words
                // away in the same row, i.e. the same byte offset with bit log2(4 CTOT) flipped (the row offset is a
                // multiple of 8 CTOT and the lane's part is below it), so the second address costs one instruction.
                uint32_t* cell2 = reinterpret_cast<uint32_t*>(hbytes + (off ^ (uint32_t)(CTOT * 4)));
                // (byte permutes with a per-lane selector: a conditional here is compiled into divergent branches)
                atomicAdd(cell, __byte_perm((uint32_t)v[u].z, (uint32_t)v[u].w, sel_first));
                atomicAdd(cell2, __byte_perm((uint32_t)v[u].z, (uint32_t)v[u].w, sel_second));
              }
            }
          }
        }
        __syncthreads();  // everyone is done with this buffer
        if (tid == 0 && c + 2 < n_chunks) {
          const int64_t rr = n - (c + 2) * kChunk;
          const uint32_t bytes = (uint32_t)((rr < kChunk ? rr : kChunk) * 16);
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          mbar_expect_tx(&mbar[b], bytes);
          bulk_load(buf, src + (c + 2) * kChunk, bytes, &mbar[b]);
        }
      }
    }
    __syncthreads();
    const long long clk2 = phase ? clock64() : 0;
    // ---- S3: box scan, in place ----
    // Each column is scanned by TPC threads, each over a contiguous range of start bins with the last
    // MW bins held in registers (statically indexed ring).  Window sums are formed left to right,
    // exactly as O4 states them.  A candidate costs 8 instructions: two adds, box_value (FADD, 2 FMUL,
    // MUFU.RCP, FMUL) and one FMNMX into the maximum of its start bin; the running maximum over start
    // bins is updated once per start bin, and the width of the winner is recovered afterwards by
    // re-evaluating that one start bin (same instructions, hence the same bits).
    constexpr int TPC = kThreads / CTOT;  // threads per column
    const int scol = tid % CTOT, seg = tid / CTOT;
    float bval = 0.f;
    uint32_t bidx = (uint32_t)prm.min_width << 24;
    const bool scol_on = scol < ti.ncols;
    int32_t nbk = 1;
    if (scol_on) {
      double fk;
      tile_freq_of_k<WM == 0u>(ti.u0, ti.h, ti.Q, dno, ti.k0 + scol, fk, nbk);
      const int per = (nbk + TPC - 1) / TPC;
      const int ja = seg * per;
      const int jb = min(nbk, ja + per);
      const uint32_t* hc = hist + scol;                                  // W words of this column
      const uint32_t* hs = hist + CTOT + scol;                           // S words of this column
      const float inv_w = ti.inv_w;
      const uint32_t wmask = WM ? WM : prm.wmask;
      if (ja < jb) {
        int bj = 0;
        float ww[MW], ss[MW];
#pragma unroll
        for (int l = 0; l < MW - 1; ++l) {
          int e = ja + l;
          if (e >= nbk) e -= nbk;
          ww[l] = (float)hc[e * STRIDE] * inv_w;
          ss[l] = (float)(int32_t)hs[e * STRIDE];
        }
        ww[MW - 1] = 0.f; ss[MW - 1] = 0.f;
        for (int j0 = ja; j0 < jb; j0 += MW) {
#pragma unroll
          for (int jj = 0; jj < MW; ++jj) {
            const int j = j0 + jj;
            if (j < jb) {
              int e = j + MW - 1;
              if (e >= nbk) e -= nbk;
              if (!QLP_IN_BOUNDS(kChkScanBin, e >= 0 && e < nbk && nbk <= nb_tile)) e = 0;
              ww[(jj + MW - 1) % MW] = (float)hc[e * STRIDE] * inv_w;
              ss[(jj + MW - 1) % MW] = (float)(int32_t)hs[e * STRIDE];
              float r = 0.f, sm = 0.f, vj = 0.f;
#pragma unroll
              for (int m = 1; m <= MW; ++m) {
                r = __fadd_rn(r, ww[(jj + m - 1) % MW]);
                sm = __fadd_rn(sm, ss[(jj + m - 1) % MW]);
                if ((wmask >> m) & 1u) vj = fmaxf(vj, box_value(r, sm));
              }
              const bool up = vj > bval;  // strict: the earliest start bin keeps a tie
              bval = up ? vj : bval;
              bj = up ? j : bj;
            }
          }
        }
        bidx = (uint32_t)bj;  // the width is recovered after the reduction, by one thread per column
      }
    }
    // reduce over the TPC threads of a column (scratch = the idle staging buffers), earliest j wins ties
    float* cval = reinterpret_cast<float*>(pbuf);
    uint32_t* cidx = reinterpret_cast<uint32_t*>(pbuf) + kThreads;
    if (TPC > 1) {
      cval[tid] = bval; cidx[tid] = bidx;
      __syncthreads();
    }
    if (seg == 0 && scol_on) {
      for (int g2 = 1; g2 < TPC; ++g2) {
        const float v = cval[g2 * CTOT + scol];
        if (v > bval) { bval = v; bidx = cidx[g2 * CTOT + scol]; }
      }
      int bm = prm.min_width, bj = 0;
      if (bval > 0.f) {
        // width of the winner: the narrowest one that reaches the maximum of its start bin (same
        // instructions as in the scan, hence the same bits)
        bj = (int)(bidx & 0xffffffu);
        {
          const uint32_t* hcw = hist + scol;
          const uint32_t* hsw = hist + CTOT + scol;
          const uint32_t wmask = WM ? WM : prm.wmask;
          float r = 0.f, sm = 0.f;
          bm = 0;
#pragma unroll 1
          for (int m = 1; m <= MW; ++m) {
            int e = bj + m - 1;
            if (e >= nbk) e -= nbk;
            r = __fadd_rn(r, (float)hcw[e * STRIDE] * ti.inv_w);
            sm = __fadd_rn(sm, (float)(int32_t)hsw[e * STRIDE]);
            if (((wmask >> m) & 1u) && bm == 0 && box_value(r, sm) == bval) bm = m;
          }
        }
        // Canonical representative of the winning box (O4 ties: smaller m, then smaller j).  Boxes
        // that hold the same points have the same value; trim the empty bins off both ends, then
        // take the narrowest ladder width that still covers the occupied span and, for it, the
        // smallest start bin whose extra bins are all empty.
        const uint32_t* hc = hist + scol;
        const uint32_t* hs2 = hist + CTOT + scol;
        // a bin is empty only if both words are zero (a point of tiny weight may quantise to W = 0 with S != 0)
        auto empty = [&](int e) {
          e %= nbk; if (e < 0) e += nbk;
          return (hc[e * STRIDE] | hs2[e * STRIDE]) == 0u;
        };
        int a = bj, b = bj + bm - 1;
        while (a < b && empty(a)) ++a;
        while (b > a && empty(b)) --b;
        const int mt = b - a + 1;
        int el = 0, er = 0;  // empty bins next to the occupied span, as far as any box could reach
        while (el < bm - mt && empty(a - 1 - el)) ++el;
        while (er < bm - mt && empty(b + 1 + er)) ++er;
        for (int m2 = mt; m2 <= bm; ++m2) {
          if (!(((WM ? WM : prm.wmask) >> m2) & 1u)) continue;
          const int extra = m2 - mt;
          int best_j = -1;
          for (int x = 0; x <= extra; ++x) {  // x extra bins on the left, extra - x on the right
            if (x > el || extra - x > er) continue;
            int j = (a - x) % nbk;
            if (j < 0) j += nbk;
            if (best_j < 0 || j < best_j) best_j = j;
          }
          if (best_j >= 0) { bm = m2; bj = best_j; break; }
        }
      }
      const int64_t o = ti.out_base + ti.k0 + scol;
      sr[o] = (bval * ti.inv_s) * ti.inv_s;
      best[o] = ((uint32_t)bm << 24) | (uint32_t)bj;
    }
    if (phase && tid == 0) {  // thread 0's clocks: tile set-up + zeroing, fold, scan + reduction + output
      const long long clk3 = clock64();
      atomicAdd(&phase[0], (unsigned long long)(clk1s - clk0));
      atomicAdd(&phase[1], (unsigned long long)(clk2 - clk1s));
      atomicAdd(&phase[2], (unsigned long long)(clk3 - clk2));
      atomicAdd(&phase[3], (unsigned long long)ti.n_pts * (unsigned long long)ti.ncols);
      atomicAdd(&phase[4], 1ull);
    }
  }
}

}  // namespace qlp
