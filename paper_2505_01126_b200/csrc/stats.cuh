// On-device turbulence statistics of a velocity field (energy spectra,
// PDFs of the longitudinal velocity gradient and of velocity increments, second- and third-order structure functions),
// device side (sm_100a).  Part of the CUDA product path; off the time-step loop.
//
//   k_stats_increments   sum_x sum_a d^p, p = 2, 3, 4, of the longitudinal increments d = u_a(x + r e_a) - u_a(x)  (L189)
//                        (the central-difference gradient of L183 is the r = 2 increment shifted by one cell, divided by 2)
//   k_stats_pdf          histogram of d / scale over [lo, hi) in nbins bins (values outside are counted in the end bins)
//   k_stats_spectrum     shell sums E(k) = sum_{round|k| = k} w |u^(k)|^2 / (2 N^2) of a real-to-complex transform (the FFT
//                        itself is the caller's: a library primitive), w = 2 for the modes whose conjugates are not stored
// Reductions: per-thread partials -> warp shuffle / shared-memory bins -> one atomic per block and quantity.
#pragma once

namespace acclb {

constexpr int STATS_THREADS = 256;

__global__ void __launch_bounds__(STATS_THREADS) k_stats_increments(Grid G, const double* __restrict__ u, int r,
                                                                     double* __restrict__ acc /* [3]: sums of d^2, d^3, d^4 */) {
  double s2 = 0.0, s3 = 0.0, s4 = 0.0;
  for (unsigned k = blockIdx.x * blockDim.x + threadIdx.x; k < G.n; k += gridDim.x * blockDim.x) {
    const int x = (int)(k % (unsigned)G.nx);
    const unsigned yz = k / (unsigned)G.nx;
    const int y = (int)(yz % (unsigned)G.ny), z = (int)(yz / (unsigned)G.ny);
    const unsigned kx = (yz * (unsigned)G.nx) + (unsigned)((x + r) % G.nx);
    const unsigned ky = ((unsigned)z * (unsigned)G.ny + (unsigned)((y + r) % G.ny)) * (unsigned)G.nx + (unsigned)x;
    const unsigned kz = ((unsigned)((z + r) % G.nz) * (unsigned)G.ny + (unsigned)y) * (unsigned)G.nx + (unsigned)x;
    const double d[3] = {__ldg(u + kx) - __ldg(u + k), __ldg(u + (size_t)G.n + ky) - __ldg(u + (size_t)G.n + k),
                         __ldg(u + 2 * (size_t)G.n + kz) - __ldg(u + 2 * (size_t)G.n + k)};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const double q = d[a] * d[a];
      s2 += q;
      s3 += q * d[a];
      s4 += q * q;
    }
  }
  __shared__ double sh[3][STATS_THREADS / 32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  double v[3] = {s2, s3, s4};
#pragma unroll
  for (int j = 0; j < 3; ++j) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v[j] += __shfl_xor_sync(0xffffffffu, v[j], o);
    if (lane == 0) sh[j][wid] = v[j];
  }
  __syncthreads();
  if (threadIdx.x < 3) {
    double t = 0.0;
    for (int w = 0; w < STATS_THREADS / 32; ++w) t += sh[threadIdx.x][w];
    atomicAdd(acc + threadIdx.x, t);
  }
}

// bin of a value: floor((v - lo) * inv_width), clamped to [0, nbins - 1]
__device__ __forceinline__ int stats_bin(double v, double lo, double inv_width, int nbins) {
  const double b = floor((v - lo) * inv_width);
  return b < 0.0 ? 0 : b >= (double)nbins ? nbins - 1 : (int)b;
}

constexpr int STATS_MAX_BINS = 1024;

__global__ void __launch_bounds__(STATS_THREADS) k_stats_pdf(Grid G, const double* __restrict__ u, int r, double inv_scale,
                                                              double lo, double inv_width, int nbins,
                                                              unsigned long long* __restrict__ counts) {
  __shared__ unsigned int bins[STATS_MAX_BINS];
  for (int b = threadIdx.x; b < nbins; b += blockDim.x) bins[b] = 0u;
  __syncthreads();
  for (unsigned k = blockIdx.x * blockDim.x + threadIdx.x; k < G.n; k += gridDim.x * blockDim.x) {
    const int x = (int)(k % (unsigned)G.nx);
    const unsigned yz = k / (unsigned)G.nx;
    const int y = (int)(yz % (unsigned)G.ny), z = (int)(yz / (unsigned)G.ny);
    const unsigned kx = (yz * (unsigned)G.nx) + (unsigned)((x + r) % G.nx);
    const unsigned ky = ((unsigned)z * (unsigned)G.ny + (unsigned)((y + r) % G.ny)) * (unsigned)G.nx + (unsigned)x;
    const unsigned kz = ((unsigned)((z + r) % G.nz) * (unsigned)G.ny + (unsigned)y) * (unsigned)G.nx + (unsigned)x;
    atomicAdd(&bins[stats_bin((__ldg(u + kx) - __ldg(u + k)) * inv_scale, lo, inv_width, nbins)], 1u);
    atomicAdd(&bins[stats_bin((__ldg(u + (size_t)G.n + ky) - __ldg(u + (size_t)G.n + k)) * inv_scale, lo, inv_width, nbins)], 1u);
    atomicAdd(&bins[stats_bin((__ldg(u + 2 * (size_t)G.n + kz) - __ldg(u + 2 * (size_t)G.n + k)) * inv_scale, lo, inv_width, nbins)], 1u);
  }
  __syncthreads();
  for (int b = threadIdx.x; b < nbins; b += blockDim.x)
    if (bins[b]) atomicAdd(counts + b, (unsigned long long)bins[b]);
}

// uhat: [ncomp][nz][ny][nx/2 + 1] complex (re, im interleaved), the unnormalised real-to-complex transform of ncomp fields.
__global__ void __launch_bounds__(STATS_THREADS) k_stats_spectrum(int nx, int ny, int nz, int ncomp, const double2* __restrict__ uhat,
                                                                   int nshell, double* __restrict__ E) {
  extern __shared__ double shell[];
  for (int b = threadIdx.x; b < nshell; b += blockDim.x) shell[b] = 0.0;
  __syncthreads();
  const int nxh = nx / 2 + 1;
  const size_t nmode = (size_t)nxh * ny * nz;
  const double norm = 0.5 / ((double)nx * ny * nz * ((double)nx * ny * nz));
  for (size_t m = blockIdx.x * (size_t)blockDim.x + threadIdx.x; m < nmode; m += (size_t)gridDim.x * blockDim.x) {
    const int kx = (int)(m % nxh);
    const size_t yz = m / nxh;
    int ky = (int)(yz % ny), kz = (int)(yz / ny);
    if (ky > ny / 2) ky -= ny;
    if (kz > nz / 2) kz -= nz;
    const int ks = (int)floor(sqrt((double)(kx * kx + ky * ky + kz * kz)) + 0.5);
    if (ks >= nshell) continue;
    const double w = (kx == 0 || (nx % 2 == 0 && kx == nx / 2)) ? 1.0 : 2.0;  // the conjugate half is not stored
    double e = 0.0;
    for (int c = 0; c < ncomp; ++c) {
      const double2 v = __ldg(uhat + (size_t)c * nmode + m);
      e += v.x * v.x + v.y * v.y;
    }
    atomicAdd(&shell[ks], w * norm * e);
  }
  __syncthreads();
  for (int b = threadIdx.x; b < nshell; b += blockDim.x)
    if (shell[b] != 0.0) atomicAdd(E + b, shell[b]);
}

}  // namespace acclb
