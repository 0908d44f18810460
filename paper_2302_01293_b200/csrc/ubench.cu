// ubench.cu -- on-SM issue-rate ceilings that bound the fold kernel.
// Stand-alone program (built by paper_2302_01293_b200.build as qlp_ubench); prints one JSON line:
//   atoms_lanes_per_clk_sm : conflict-free 32-bit shared-memory ATOMS.ADD lanes per clock per SM
//   fp64_lanes_per_clk_sm  : FP64 pipe lanes (DMUL/DADD/DFMA) per clock per SM
//   bin_evals_per_clk_sm   : the 4-instruction bin sequence of common.cuh alone
// It shares no code with the kernels it bounds, apart from restating the 4-instruction sequence.
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>

extern __shared__ __align__(16) unsigned char smem_raw[];

__global__ void k_atoms(int iters, long long* cyc, unsigned* sink) {
  unsigned* h = reinterpret_cast<unsigned*>(smem_raw);
  const int t = threadIdx.x, lane = t & 31, nt = blockDim.x;
  const int rows = 64;
  for (int i = t; i < rows * 32; i += nt) h[i] = 0;
  __syncthreads();
  unsigned r0 = (t * 7) & (rows - 1);
  long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      atomicAdd(&h[((r0 + u * 5) & (rows - 1)) * 32 + lane], (unsigned)it);
    }
    r0 += 3;
  }
  long long t1 = clock64();
  __syncthreads();
  if (t == 0) cyc[blockIdx.x] = t1 - t0;
  sink[blockIdx.x * nt + t] = h[t % (rows * 32)];
}

__global__ void k_fp64(int iters, long long* cyc, double* sink) {
  const int t = threadIdx.x;
  double a0 = 1.0 + t * 1e-3, a1 = 1.1, a2 = 1.2, a3 = 1.3, a4 = 1.4, a5 = 1.5, a6 = 1.6, a7 = 1.7;
  const double m = 1.0000001, c = 1e-9;
  long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
    a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
    a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
  }
  long long t1 = clock64();
  if (t == 0) cyc[blockIdx.x] = t1 - t0;
  sink[blockIdx.x * blockDim.x + t] = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
}

__global__ void k_bin(int iters, long long* cyc, int* sink) {
  const int t = threadIdx.x;
  const double f = 1.0 + 1e-3 * t, dnb = 100.0, K = (dnb + 1.0) * 4503599627370496.0;
  const double* taus = reinterpret_cast<const double*>(smem_raw);
  double* tw = reinterpret_cast<double*>(smem_raw);
  for (int i = t; i < 1024; i += blockDim.x) tw[i] = 0.37 + 0.0023 * i;
  __syncthreads();
  int acc = 0;
  long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const double tau = taus[(it * 8 + u) & 1023];
      double p = __dmul_rn(f, tau);
      double cc = __dadd_rd(p, 4503599627370496.0);
      double A = __fma_rn(-dnb, cc, K);
      double v = __fma_rd(p, dnb, A);
      acc += __double2loint(v);
    }
  }
  long long t1 = clock64();
  if (t == 0) cyc[blockIdx.x] = t1 - t0;
  sink[blockIdx.x * blockDim.x + t] = acc;
}

// Issue cost next to the FP64 pipe: 4 DFMA per iteration plus NI independent 32-bit logic ops (LOP3).  If the
// logic ops issued in the shadow of the half-rate DFMAs the time would not grow with NI; it does (additively),
// i.e. an FP64 instruction occupies its scheduler for two issue cycles.
template <int NI>
__global__ void k_mix(int iters, long long* cyc, double* sink) {
  const int t = threadIdx.x;
  double a0 = 1.0 + t * 1e-3, a1 = 1.1, a2 = 1.2, a3 = 1.3;
  const double m = 1.0000001, c = 1e-9;
  unsigned i0 = t, i1 = 3, i2 = 5, i3 = 7, i4 = 11, i5 = 13, i6 = 17, i7 = 19;
  const unsigned q = (blockIdx.x << 7) | 0x55u;
  long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
    a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
    if (NI >= 1) i0 = (i0 & q) ^ (unsigned)it;
    if (NI >= 2) i1 = (i1 | q) ^ (unsigned)it;
    if (NI >= 3) i2 = (i2 & q) ^ (unsigned)it;
    if (NI >= 4) i3 = (i3 | q) ^ (unsigned)it;
    if (NI >= 5) i4 = (i4 & q) ^ (unsigned)it;
    if (NI >= 6) i5 = (i5 | q) ^ (unsigned)it;
    if (NI >= 7) i6 = (i6 & q) ^ (unsigned)it;
    if (NI >= 8) i7 = (i7 | q) ^ (unsigned)it;
  }
  long long t1 = clock64();
  if (t == 0) cyc[blockIdx.x] = t1 - t0;
  sink[blockIdx.x * blockDim.x + t] = a0 + a1 + a2 + a3 + (double)(i0 + i1 + i2 + i3 + i4 + i5 + i6 + i7);
}

template <typename F>
static double run(F launch, int nblk, long long* cyc) {
  launch(); launch();
  cudaDeviceSynchronize();
  long long* h = new long long[nblk];
  cudaMemcpy(h, cyc, nblk * sizeof(long long), cudaMemcpyDeviceToHost);
  double s = 0;
  for (int i = 0; i < nblk; ++i) s += (double)h[i];
  delete[] h;
  return s / nblk;
}

int main() {
  int nsm = 0;
  if (cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, 0) != cudaSuccess || nsm <= 0) {
    printf("{\"error\": \"no CUDA device\"}\n");
    return 1;
  }
  long long* cyc; void* sink;
  cudaMalloc(&cyc, nsm * sizeof(long long));
  cudaMalloc(&sink, (size_t)nsm * 1024 * 8);
  const int iters = 4000, threads = 1024;
  double best_atoms = 0, best_fp64 = 0, best_bin = 0;
  for (int th : {256, 512, 1024}) {
    double c = run([&] { k_atoms<<<nsm, th, 64 * 32 * 4>>>(iters, cyc, (unsigned*)sink); }, nsm, cyc);
    double v = (double)th * iters * 8 / c;
    if (v > best_atoms) best_atoms = v;
    c = run([&] { k_fp64<<<nsm, th>>>(iters, cyc, (double*)sink); }, nsm, cyc);
    v = (double)th * iters * 8 / c;
    if (v > best_fp64) best_fp64 = v;
    c = run([&] { k_bin<<<nsm, th, 8192>>>(iters, cyc, (int*)sink); }, nsm, cyc);
    v = (double)th * iters * 8 / c;
    if (v > best_bin) best_bin = v;
  }
  (void)threads;
  // cycles per warp iteration per scheduler (1024 threads = 8 warps per scheduler)
  const double mix0 = run([&] { k_mix<0><<<nsm, 1024>>>(iters, cyc, (double*)sink); }, nsm, cyc) / iters / 8.0;
  const double mix4 = run([&] { k_mix<4><<<nsm, 1024>>>(iters, cyc, (double*)sink); }, nsm, cyc) / iters / 8.0;
  const double mix8 = run([&] { k_mix<8><<<nsm, 1024>>>(iters, cyc, (double*)sink); }, nsm, cyc) / iters / 8.0;
  int clk_khz = 0;
  cudaDeviceGetAttribute(&clk_khz, cudaDevAttrClockRate, 0);
  printf("{\"sms\": %d, \"sm_max_mhz\": %.0f, \"atoms_lanes_per_clk_sm\": %.2f, \"fp64_lanes_per_clk_sm\": %.2f, "
         "\"bin_evals_per_clk_sm\": %.2f, \"issue_cycles_4dfma\": %.2f, \"issue_cycles_4dfma_4lop3\": %.2f, "
         "\"issue_cycles_4dfma_8lop3\": %.2f}\n", nsm, clk_khz / 1000.0, best_atoms, best_fp64, best_bin, mix0, mix4, mix8);
  return cudaGetLastError() == cudaSuccess ? 0 : 2;
}
