// libacclb.so -- kernels and C ABI (include/acclb.h) of the accLB per-time-step lattice update on sm_100a.
//
// Written from /root/reference/PAPER.md (arXiv 2505.01126).  One step (rows a1-a8):
//   single-phase   k_lb: pull-stream (a1) -> moments (a2) -> body force (a4) -> u (a5) -> Hermite coefficient (a6) ->
//                  regularized reconstruction + aligned store (a7), one node per thread           PAPER.md:L75-92 (Eqs. 4-7)
//   two-phase      k_lb_tp<MODE_FUSED> + k_seam (twophase.cuh): the same plus phase geometry, forces (a3, a4) and the
//                  conservative Allen-Cahn update (a8) on shared-memory tiles marching along z, TMA / cp.async staging;
//                  u and r never written to HBM                                        PAPER.md:L61-67 (Eq. 3), L100-104 (Eq. 8)
//                  phi_integrator = 1 (SSP-RK3, R32): k_lb_tp<MODE_FUSED_U> (the step + first stage, u(t) written out) +
//                  k_seam, then twice k_lb_tp<MODE_STAGE> + k_seam<SCALED> (the same tiles without the LB half);
//                  variant 1 = the unfused forms (k_lb_tp<MODE_UNFUSED> + k_advect; RK3: + k_geom_r (phase_rk.cuh) and
//                  k_advect per stage), kept so that bench.py / ncu can compare fused and unfused on identical inputs.
//   init, moments, diagnostics of a two-phase context are modes of the same tiled kernel.
// State: post-collision, not yet streamed populations f*_i(x) in SoA [z][i][y][x], double-buffered (A/B), so the
// pull f_i(x,t) = f*_i(x - c_i, t-1) reads shifted rows and every store is aligned; phi double-buffered.
// No CPU fallback, no library kernels: everything the path computes runs in the kernels of this file.
#include <cuda.h>
#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/acclb.h"
#include "d3q27.cuh"
#include "stencils.cuh"

namespace acclb {

// ------------------------------------------------------------------------------------------------ parameters
struct KP {
  Grid G;
  double omega, one_m_omega;  // 1/tau, 1 - 1/tau
  double rho_g, drho;         // rho = rho_g + drho phi
  double sig15w;              // gamma * 3 delta / 2                    PAPER.md:L102 + R8
  double visc_pref;           // nu omega / cs2 = (tau - 1/2)/tau       PAPER.md:L104 (R9)
  int ratio_ne;               // rho_l != rho_g
  double D, kappa;            // D, 4 D / delta
  int force_type;
  double force_amp;
  double nu, eps_pref;        // nu, nu / (2 cs4 tau^2) (R21)
  double grav[3], rho_ref;    // buoyancy F^g = (rho - rho_ref) g       PAPER.md:L193, L203 (R31)
  int buoyant;                // g != 0
  int zlo, zhi;               // diagnostics run over planes [zlo, zhi): all of them, or a slab's own planes (halo_z)
  double rk_a, rk_b;          // Shu-Osher coefficients of the Runge-Kutta stage being launched (k_lb_tp<MODE_STAGE>, k_seam)
};

// population storage: fp64, or fp32 deviation from the lattice weight (R22)
template <typename ST> struct Pop;
template <> struct Pop<double> {
  static __device__ __forceinline__ double from_storage(double v, int) { return v; }
  static __device__ __forceinline__ double load(const double* p, int) { return __ldcs(p); }
  static __device__ __forceinline__ void store(double* p, int, double v) { __stcs(p, v); }
};
template <> struct Pop<float> {
  static __device__ __forceinline__ double from_storage(float v, int i) { return (double)v + w_of(i); }
  static __device__ __forceinline__ double load(const float* p, int i) { return (double)__ldcs(p) + w_of(i); }
  static __device__ __forceinline__ void store(float* p, int i, double v) { __stcs(p, (float)(v - w_of(i))); }
};

__device__ __forceinline__ bool node_of_thread(const Grid& G, unsigned& k, int& x, int& y, int& z) {
  k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= G.n) return false;
  x = (int)(k % (unsigned)G.nx);
  const unsigned yz = k / (unsigned)G.nx;
  y = (int)(yz % (unsigned)G.ny);
  z = (int)(yz / (unsigned)G.ny);
  return true;
}

// R20 body-force density from the per-axis tables tabs = [sin kx x | cos kx x | sin ky y | cos ky y | sin kz z | cos kz z]
__device__ __forceinline__ void body_force(const KP& P, const double* __restrict__ tabs, int x, int y, int z,
                                           double (&Fb)[3]) {
  Fb[0] = Fb[1] = Fb[2] = 0.0;
  if (P.force_type == 0) return;
  const double* sx = tabs;
  const double* cx = sx + P.G.nx;
  const double* sy = cx + P.G.nx;
  const double* cy = sy + P.G.ny;
  const double* sz = cy + P.G.ny;
  const double* cz = sz + P.G.nz;
  if (P.force_type == 1) {  // ABC
    Fb[0] = P.force_amp * (__ldg(sz + z) + __ldg(cy + y));
    Fb[1] = P.force_amp * (__ldg(sx + x) + __ldg(cz + z));
    Fb[2] = P.force_amp * (__ldg(sy + y) + __ldg(cx + x));
  } else {  // sine variant of BASELINE config 2
    Fb[0] = P.force_amp * __ldg(sy + y);
    Fb[1] = P.force_amp * __ldg(sz + z);
    Fb[2] = P.force_amp * __ldg(sx + x);
  }
}

// a1: pull-stream.  f_i(x,t) = f*_i(x - c_i, t-1), periodic wrap.   PAPER.md:L75/L85 (LHS of Eqs. 4, 6), L118
template <typename ST>
__device__ __forceinline__ void pull27(const ST* __restrict__ fin, const Grid& G, const Nbr& nb, double (&f)[Q]) {
  const unsigned plane = (unsigned)G.nx * (unsigned)G.ny;
  const ST* slab[3] = {pop_slab(fin, G, nb.z[0]), pop_slab(fin, G, nb.z[1]), pop_slab(fin, G, nb.z[2])};
#pragma unroll
  for (int i = 0; i < Q; ++i)
    f[i] = Pop<ST>::load(slab[1 - cz_of(i)] + ((unsigned)i * plane + nb.yr[1 - cy_of(i)] + (unsigned)nb.x[1 - cx_of(i)]), i);
}

// a4-a5: total force, acceleration A = F / rho (R3) and density at a node from its interface geometry.
//   g = grad phi, gn = |g|, kc = kappa_c = div n, phi0 = phi(x);  rho = rho_g + drho phi
//   F^s = -gamma (3 delta/2) kappa_c |g| g (L102, R8);  F^p = -p* cs2 grad rho (L102);
//   F^nu = -((tau-1/2)/tau) (Pi - p* cs2 I - ut ut) . grad rho (L104, R9), ut = m + (F^s+F^p+F^b)/(2 rho);
//   F = F^s + F^p + F^nu + F^b (Eq. 8).
//   fs = -gamma (3 delta/2) kappa_c |g| is passed in (F^s = fs g).
__device__ __forceinline__ void accel_from_gc(const KP& P, const Moments& M, const double (&g)[3], double fs, double phi0,
                                              const double (&Fb)[3], bool with_visc, double (&A)[3], double& rho) {
  rho = P.rho_g + P.drho * phi0;
  const double fp = -M.p * (1.0 / 3.0) * P.drho;
  double F[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) F[a] = fs * g[a] + fp * g[a] + Fb[a];
  if (P.buoyant) {  // F^g = (rho - rho_ref) g (R31)
    const double dr = rho - P.rho_ref;
    F[0] += dr * P.grav[0]; F[1] += dr * P.grav[1]; F[2] += dr * P.grav[2];
  }
  if (with_visc && P.ratio_ne) {
    const double h = 0.5 / rho;
    const double ut[3] = {M.m[0] + F[0] * h, M.m[1] + F[1] * h, M.m[2] + F[2] * h};
    const double dr[3] = {P.drho * g[0], P.drho * g[1], P.drho * g[2]};
    const double p3 = M.p * (1.0 / 3.0);
    const double sxx = M.Pi[0] - p3 - ut[0] * ut[0], syy = M.Pi[1] - p3 - ut[1] * ut[1], szz = M.Pi[2] - p3 - ut[2] * ut[2];
    const double sxy = M.Pi[3] - ut[0] * ut[1], sxz = M.Pi[4] - ut[0] * ut[2], syz = M.Pi[5] - ut[1] * ut[2];
    F[0] -= P.visc_pref * (sxx * dr[0] + sxy * dr[1] + sxz * dr[2]);
    F[1] -= P.visc_pref * (sxy * dr[0] + syy * dr[1] + syz * dr[2]);
    F[2] -= P.visc_pref * (sxz * dr[0] + syz * dr[1] + szz * dr[2]);
  }
  const double ir = div_pos(1.0, rho);
  A[0] = F[0] * ir; A[1] = F[1] * ir; A[2] = F[2] * ir;
}

__device__ __forceinline__ void accel_from_geometry(const KP& P, const Moments& M, const double (&g)[3], double gn,
                                                    double kc, double phi0, const double (&Fb)[3], bool with_visc,
                                                    double (&A)[3], double& rho) {
  accel_from_gc(P, M, g, -P.sig15w * kc * gn, phi0, Fb, with_visc, A, rho);
}

// a4-a5 for the one-node-per-thread (single-phase) kernels: rho == 1, A = F^b (+ the uniform (1 - rho_ref) g, R31).
__device__ __forceinline__ void node_accel(const KP& P, const double* __restrict__ tabs, int x, int y, int z, double (&A)[3],
                                           double& rho) {
  double Fb[3];
  body_force(P, tabs, x, y, z, Fb);
  rho = 1.0;
  A[0] = Fb[0]; A[1] = Fb[1]; A[2] = Fb[2];
  if (P.buoyant) {
    const double dr = 1.0 - P.rho_ref;
    A[0] += dr * P.grav[0]; A[1] += dr * P.grav[1]; A[2] += dr * P.grav[2];
  }
}

// a6: a_ab = sum_i (f_i - f_i^eq + S_i/2) H_i,ab (Eq. 7) in closed form (O5'):
//   sum f H = Pi - cs2 p* I,  sum f^eq H = uu,  sum S H = uA + Au.
__device__ __forceinline__ void hermite_coeff(const Moments& M, const double (&u)[3], const double (&A)[3],
                                              double (&a)[6]) {
  const double p3 = M.p * (1.0 / 3.0);
  a[0] = M.Pi[0] - p3 - u[0] * u[0] + u[0] * A[0];
  a[1] = M.Pi[1] - p3 - u[1] * u[1] + u[1] * A[1];
  a[2] = M.Pi[2] - p3 - u[2] * u[2] + u[2] * A[2];
  a[3] = M.Pi[3] - u[0] * u[1] + 0.5 * (u[0] * A[1] + u[1] * A[0]);
  a[4] = M.Pi[4] - u[0] * u[2] + 0.5 * (u[0] * A[2] + u[2] * A[0]);
  a[5] = M.Pi[5] - u[1] * u[2] + 0.5 * (u[1] * A[2] + u[2] * A[1]);
}

// a6-a7: Hermite coefficient (Eq. 7), regularized reconstruction (Eq. 6) as one second-order Hermite-space
// population (see hermite2_populations), aligned store of f*_i(x) into the other buffer.
template <typename ST>
__device__ __forceinline__ void collide_store(const KP& P, const Moments& M, const double (&u)[3], const double (&A)[3],
                                              double (&f)[Q], ST* __restrict__ out0, unsigned plane) {
  double a[6];
  hermite_coeff(M, u, A, a);
  const double U[3] = {u[0] + 0.5 * A[0], u[1] + 0.5 * A[1], u[2] + 0.5 * A[2]};
  double T[6];
  T[0] = u[0] * u[0] + P.one_m_omega * a[0] + u[0] * A[0];
  T[1] = u[1] * u[1] + P.one_m_omega * a[1] + u[1] * A[1];
  T[2] = u[2] * u[2] + P.one_m_omega * a[2] + u[2] * A[2];
  T[3] = u[0] * u[1] + P.one_m_omega * a[3] + 0.5 * (u[0] * A[1] + u[1] * A[0]);
  T[4] = u[0] * u[2] + P.one_m_omega * a[4] + 0.5 * (u[0] * A[2] + u[2] * A[0]);
  T[5] = u[1] * u[2] + P.one_m_omega * a[5] + 0.5 * (u[1] * A[2] + u[2] * A[1]);
  hermite2_populations(M.p, U, T, f);
#pragma unroll
  for (int i = 0; i < Q; ++i) Pop<ST>::store(out0 + (unsigned)i * plane, i, f[i]);  // out0 = f*_0 of this node
}

template <typename ST>
__device__ __forceinline__ void collide_store(const KP& P, const Moments& M, const double (&u)[3], const double (&A)[3],
                                              ST* __restrict__ out0, unsigned plane) {
  double f[Q];
  collide_store<ST>(P, M, u, A, f, out0, plane);
}

// ------------------------------------------------------------------------------------------------ kernels
// The single-phase kernels: one node per thread, scalar 64-bit accesses (at the measured copy bandwidth, DESIGN.md
// section 7).  Two-phase contexts run the tiled kernel of twophase.cuh in all of its modes.

// The fused LB step.
template <typename ST>
__global__ void __launch_bounds__(128) k_lb(KP P, const ST* __restrict__ fin, ST* __restrict__ fout,
                                            const double* __restrict__ tabs) {
  unsigned k; int x, y, z;
  if (!node_of_thread(P.G, k, x, y, z)) return;
  Nbr nb;
  make_nbr(P.G, x, y, z, nb);
  double f[Q];
  pull27<ST>(fin, P.G, nb, f);
  Moments M;
  moments_of(f, M);
  double A[3], rho;
  node_accel(P, tabs, x, y, z, A, rho);
  const double u[3] = {M.m[0] + 0.5 * A[0], M.m[1] + 0.5 * A[1], M.m[2] + 0.5 * A[2]};  // a5, PAPER.md:L88 (R4)
  const unsigned plane = (unsigned)P.G.nx * (unsigned)P.G.ny;
  collide_store<ST>(P, M, u, A, f, pop_slab(fout, P.G, z) + (nb.yr[1] + (unsigned)x), plane);
}

// Initial populations (R15): f_i(x,0) = f_i^eq(p*,u0) - S_i(u0,A)/2 with A = F^b (+ F^g), written "pushed" to x - c_i so
// that the first pull returns them at x.
template <typename ST>
__global__ void __launch_bounds__(128) k_init(KP P, const double* __restrict__ rho_in, const double* __restrict__ u_in,
                                              const double* __restrict__ tabs, ST* __restrict__ fout) {
  unsigned k; int x, y, z;
  if (!node_of_thread(P.G, k, x, y, z)) return;
  Nbr nb;
  make_nbr(P.G, x, y, z, nb);
  double A[3], rho;
  node_accel(P, tabs, x, y, z, A, rho);
  const double p = rho_in[k];
  const double u[3] = {u_in[k], u_in[(size_t)P.G.n + k], u_in[2 * (size_t)P.G.n + k]};  // (3 n may exceed 2^32)
  const double U[3] = {u[0] - 0.5 * A[0], u[1] - 0.5 * A[1], u[2] - 0.5 * A[2]};
  double T[6];
  T[0] = u[0] * u[0] - u[0] * A[0];
  T[1] = u[1] * u[1] - u[1] * A[1];
  T[2] = u[2] * u[2] - u[2] * A[2];
  T[3] = u[0] * u[1] - 0.5 * (u[0] * A[1] + u[1] * A[0]);
  T[4] = u[0] * u[2] - 0.5 * (u[0] * A[2] + u[2] * A[0]);
  T[5] = u[1] * u[2] - 0.5 * (u[1] * A[2] + u[2] * A[1]);
  double f[Q];
  hermite2_populations(p, U, T, f);
#pragma unroll
  for (int i = 0; i < Q; ++i)
    Pop<ST>::store(pop_slab(fout, P.G, nb.z[1 - cz_of(i)]) +
                       ((unsigned)i * ((unsigned)P.G.nx * (unsigned)P.G.ny) + nb.yr[1 - cy_of(i)] + (unsigned)nb.x[1 - cx_of(i)]),
                   i, f[i]);
}

// a9: (p*, u) of the current state; the state is unchanged.
template <typename ST>
__global__ void __launch_bounds__(128) k_moments(KP P, const ST* __restrict__ fin, const double* __restrict__ tabs,
                                                 double* __restrict__ rho_out, double* __restrict__ u_out) {
  unsigned k; int x, y, z;
  if (!node_of_thread(P.G, k, x, y, z)) return;
  Nbr nb;
  make_nbr(P.G, x, y, z, nb);
  double f[Q];
  pull27<ST>(fin, P.G, nb, f);
  Moments M;
  moments_of(f, M);
  double A[3], rho;
  node_accel(P, tabs, x, y, z, A, rho);
  if (rho_out) rho_out[k] = M.p;
  if (u_out) {
    u_out[k] = M.m[0] + 0.5 * A[0];
    u_out[(size_t)P.G.n + k] = M.m[1] + 0.5 * A[1];
    u_out[2 * (size_t)P.G.n + k] = M.m[2] + 0.5 * A[2];
  }
}

// a9: diagnostics (R21).  acc[0..6] += sum (|u|^2/2, eps, 0, p*, m_x, m_y, m_z); acc[7] = max |u| (as ordered bits).
// Grid-stride; per-thread partials -> warp shuffle -> one atomic per block and quantity.
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

constexpr int DIAG_THREADS = 128;

template <typename ST>
__global__ void __launch_bounds__(DIAG_THREADS) k_diagnostics(KP P, const ST* __restrict__ fin,
                                                              const double* __restrict__ tabs, double* __restrict__ acc) {
  double s[7] = {0, 0, 0, 0, 0, 0, 0};
  double umax = 0.0;
  const Grid& G = P.G;
  for (unsigned k = blockIdx.x * blockDim.x + threadIdx.x; k < G.n; k += gridDim.x * blockDim.x) {
    const int x = (int)(k % (unsigned)G.nx);
    const unsigned yz = k / (unsigned)G.nx;
    const int y = (int)(yz % (unsigned)G.ny), z = (int)(yz / (unsigned)G.ny);
    if (z < P.zlo || z >= P.zhi) continue;  // halo planes of a z-slab
    Nbr nb;
    make_nbr(G, x, y, z, nb);
    double f[Q];
    pull27<ST>(fin, G, nb, f);
    Moments M;
    moments_of(f, M);
    double A[3], rho;
    node_accel(P, tabs, x, y, z, A, rho);
    const double u[3] = {M.m[0] + 0.5 * A[0], M.m[1] + 0.5 * A[1], M.m[2] + 0.5 * A[2]};
    double a[6];
    hermite_coeff(M, u, A, a);
    const double uu = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
    const double aa = a[0] * a[0] + a[1] * a[1] + a[2] * a[2] + 2.0 * (a[3] * a[3] + a[4] * a[4] + a[5] * a[5]);
    s[0] += 0.5 * rho * uu;
    s[1] += P.eps_pref * aa;
    s[3] += M.p;
    s[4] += M.m[0];
    s[5] += M.m[1];
    s[6] += M.m[2];
    umax = fmax(umax, sqrt(uu));
  }
  __shared__ double sh[8][DIAG_THREADS / 32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int j = 0; j < 7; ++j) {
    const double r = warp_sum(s[j]);
    if (lane == 0) sh[j][wid] = r;
  }
  {
    const double r = warp_max(umax);
    if (lane == 0) sh[7][wid] = r;
  }
  __syncthreads();
  if (threadIdx.x < 8) {
    const int j = threadIdx.x;
    double r = sh[j][0];
    for (int w = 1; w < DIAG_THREADS / 32; ++w) r = (j < 7) ? r + sh[j][w] : fmax(r, sh[j][w]);
    if (j < 7) atomicAdd(acc + j, r);
    else atomicMax(reinterpret_cast<unsigned long long*>(acc + 7), (unsigned long long)__double_as_longlong(r));  // r >= 0
  }
}

}  // namespace acclb

#include "twophase.cuh"
#include "phase_rk.cuh"
#include "stats.cuh"
#include "momrep.cuh"

// ================================================================================================== host / ABI
using namespace acclb;

struct accLB_ctx {
  accLB_params prm;
  KP kp;
  int nx, ny, nz;
  size_t n;
  cudaStream_t stream;
  // carved from the caller's workspace
  void* f[2];
  double* phi[2];
  double* u;
  double* r;    // D lap phi - kappa div q of the current step (k_lb_tp -> k_advect)
  double* phis; // RK3 only: the second stage field
  double* ms[2]; // moment_storage: the ten fields (p*, u, a) of every node, double-buffered (replaces f[])
  double* tabs;
  double* acc;
  CUtensorMap tmap[2];      // populations A / B as rank-3 tensors (x, y, z * 27 + i) for the TMA pull of k_lb_tp<FAST>,
  CUtensorMap tmap_row[2];  // box TX x TY x 1, and box TX x 1 x 1 (single rows: tiles on the periodic y rim)
  int tmap_ok;              // 0: no FAST path (tile shape does not divide the box, fp32 storage, no driver entry point)
  Seams seams;    // u on the seams of the tile columns (k_lb_tp<FUSED> -> k_seam)
  int lz;         // planes per block of the z-marching kernels
  double* stage;  // [5 n] rho | u(3) | phi, host_staging only
  int cur;        // f[cur], phi[cur] hold the current state
  long long step;
  long long launches;
  int variant;
  int profiling;
  struct Rec { int kind; cudaEvent_t e0, e1; };
  std::vector<Rec> recs;                 // at most REC_MAX pending event pairs; older ones are folded into the totals
  double folded_ms[ACCLB_NKERNELS];
  long long folded_count[ACCLB_NKERNELS];
};

// Selects the context's device for the duration of an ABI call and restores the caller's current device afterwards
// (a multi-GPU process keeps its own current device; "replicas only").
struct DeviceGuard {
  int prev = -1;
  bool ok;
  explicit DeviceGuard(int dev) {
    ok = cudaGetDevice(&prev) == cudaSuccess;
    if (ok && prev != dev) ok = cudaSetDevice(dev) == cudaSuccess;
    else if (ok) prev = -1;  // nothing to restore
  }
  ~DeviceGuard() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};
#define GUARD_DEVICE(s_)                                                                          \
  DeviceGuard guard_((s_)->prm.device);                                                            \
  if (!guard_.ok) return fail(ACCLB_ECUDA, "cannot select device %d", (s_)->prm.device)

constexpr size_t REC_MAX = 4096;
// Waits for the pending event pairs and adds their durations to the per-kernel totals (bounded host memory however long
// profiling stays on).
static void fold_records(accLB_ctx* s) {
  if (s->recs.empty()) return;
  cudaEventSynchronize(s->recs.back().e1);
  for (auto& r : s->recs) {
    float t = 0.f;
    if (cudaEventElapsedTime(&t, r.e0, r.e1) == cudaSuccess && r.kind >= 0 && r.kind < ACCLB_NKERNELS) {
      s->folded_ms[r.kind] += (double)t;
      s->folded_count[r.kind] += 1;
    }
    cudaEventDestroy(r.e0);
    cudaEventDestroy(r.e1);
  }
  s->recs.clear();
}

// Counts a kernel launch and, when profiling is on, brackets it with two events on the context's stream.
struct LaunchScope {
  accLB_ctx* s;
  accLB_ctx::Rec r;
  bool on;
  LaunchScope(accLB_ctx* s_, int kind) : s(s_), on(s_->profiling != 0) {
    r.kind = kind;
    if (on) {
      on = cudaEventCreate(&r.e0) == cudaSuccess && cudaEventCreate(&r.e1) == cudaSuccess;
      if (on) cudaEventRecord(r.e0, s->stream);
    }
  }
  ~LaunchScope() {
    s->launches++;
    if (on) {
      cudaEventRecord(r.e1, s->stream);
      s->recs.push_back(r);
      if (s->recs.size() >= REC_MAX) fold_records(s);
    }
  }
};
enum { KIND_LB = 1, KIND_INIT = 3, KIND_MOMENTS = 4, KIND_DIAG = 5, KIND_LB_TP = 6,
       KIND_SEAM = 7, KIND_ADVECT = 8, KIND_GEOM = 9, KIND_MR = 10, KIND_STAGE = 11 };

static thread_local char g_err[512] = "";

static int fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof g_err, fmt, ap);
  va_end(ap);
  return code;
}

static size_t align256(size_t b) { return (b + 255) & ~(size_t)255; }

static bool valid_args(int nx, int ny, int nz, const accLB_params* p) {
  if (!p) return false;
  if (nx < 4 || ny < 4 || nz < 4 || (nx & 1)) return false;
  if ((double)nx * (double)ny * (double)nz >= 2147483648.0) return false;
  if (27.0 * (double)nx * (double)ny >= 4294967296.0) return false;  // 32-bit offsets inside a [27][ny][nx] slab
  if (!(p->tau > 0.5) || !std::isfinite(p->tau)) return false;
  if (p->force_type < 0 || p->force_type > 2) return false;
  if (!std::isfinite(p->gravity[0]) || !std::isfinite(p->gravity[1]) || !std::isfinite(p->gravity[2]) || !std::isfinite(p->rho_ref)) return false;
  if (p->phi_integrator < 0 || p->phi_integrator > 1) return false;
  if (p->moment_storage < 0 || p->moment_storage > 1) return false;
  if (p->moment_storage && (p->two_phase || p->store_fp32)) return false;  // single-phase fp64 only
  if (p->halo_z < 0) return false;
  if (p->halo_z > 0) {  // one z-slab of a larger periodic domain
    if (p->phi_integrator != 0 || p->moment_storage) return false;
    if (p->halo_z < (p->two_phase ? 3 : 1) || nz < 3 * p->halo_z) return false;
    if (p->nz_global < nz - 2 * p->halo_z) return false;
  }
  if (p->two_phase) {
    if (!(p->rho_l > 0.0) || !(p->rho_g > 0.0) || !(p->width > 0.0) || !(p->mobility >= 0.0)) return false;
  }
  return true;
}

// Tile shapes of the two-phase kernels.
constexpr int STAGE_MINB = 3;  // k_lb_tp<MODE_STAGE> holds no population landing zone: three blocks per SM
constexpr int LBT_TX = 32, LBT_TY = 8, LBT_MINB = 2;  // (32 x 16 tiles, one 512-thread block per SM: measured 11.17 vs 10.52 ms at 512^3)
constexpr int ADV_TX = 32, ADV_TY = 8;

// Planes per block along z: enough blocks to load every SM a few times over, chunks of equal length, and no
// chunk so short that its prologue (4 phi planes, 2 derived planes) dominates.
static int planes_per_block(int nx, int ny, int nz, int tx, int ty) {
  const long long tiles = (long long)((nx + tx - 1) / tx) * ((ny + ty - 1) / ty);
  long long lz = (long long)nz * tiles / (148LL * 12LL);
  if (lz < 8) lz = 8;
  if (lz > LZ_MAX) lz = LZ_MAX;
  if (lz > nz) lz = nz;
  const int chunks = (int)((nz + lz - 1) / lz);
  return (nz + chunks - 1) / chunks;
}

struct Carve {
  size_t f, phi, u, r, tabs, acc, sx, sy, sz, phis, stage, total;
};
static Carve carve(int nx, int ny, int nz, const accLB_params* p) {
  const size_t n = (size_t)nx * ny * nz;
  Carve c;
  c.f = p->moment_storage ? align256(10 * n * 8) : align256(27 * n * (p->store_fp32 ? 4 : 8));
  c.phi = p->two_phase ? align256(n * 8) : 0;
  c.u = p->two_phase ? align256(3 * n * 8) : 0;
  c.r = p->two_phase ? align256(n * 8) : 0;
  c.tabs = align256((size_t)2 * (nx + ny + nz) * 8);
  c.acc = align256(16 * 8);
  const size_t ntx = (nx + LBT_TX - 1) / LBT_TX, nty = (ny + LBT_TY - 1) / LBT_TY;
  const int lz = planes_per_block(nx, ny, nz, LBT_TX, LBT_TY);
  const size_t nchunk = (nz + lz - 1) / lz;
  c.sx = p->two_phase ? align256((size_t)nz * ny * 2 * ntx * 8) : 0;
  c.sy = p->two_phase ? align256((size_t)nz * 2 * nty * nx * 8) : 0;
  c.sz = p->two_phase ? align256(2 * nchunk * (size_t)ny * nx * 8) : 0;
  c.phis = p->two_phase && p->phi_integrator == 1 ? align256(n * 8) : 0;
  c.stage = p->host_staging ? align256(5 * n * 8) : 0;
  c.total = 2 * c.f + 2 * c.phi + c.u + c.r + c.tabs + c.acc + c.sx + c.sy + c.sz + c.phis + c.stage;
  return c;
}

#define CK(call)                                                                                      \
  do {                                                                                                \
    cudaError_t e_ = (call);                                                                          \
    if (e_ != cudaSuccess) return fail(ACCLB_ECUDA, "%s: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
  } while (0)

static unsigned blocks_for(size_t n, int threads) { return (unsigned)((n + threads - 1) / threads); }

// One launch of the tiled two-phase kernel in the given MODE (twophase.cuh) on the state f[c], phi[c]; f[d], phi[d] are the
// targets of a step.  out_u / out_r / in0 / in1: see the MODE list.
// phi_in / phi_out (default: phi[c] / phi[d]) let a Runge-Kutta stage run on the stage fields.
template <typename ST, int MODE, bool FAST>
static int launch_lb_tp(accLB_ctx* s, int c, int d, int kind, double* out_u, double* out_r, const double* in0,
                        const double* in1, const double* phi_in = nullptr, double* phi_out = nullptr) {
  constexpr bool STAGE = MODE == MODE_STAGE;
  using T = GeoTile<ST, LBT_TX, LBT_TY, MODE == MODE_FUSED || MODE == MODE_FUSED_U || STAGE, !STAGE>;
  auto kern = k_lb_tp<ST, LBT_TX, LBT_TY, STAGE ? STAGE_MINB : LBT_MINB, MODE, FAST>;
  static thread_local int configured_device = -1;
  if (configured_device != s->prm.device) {
    CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(T)));
    configured_device = s->prm.device;
  }
  const int lz = s->lz;
  const dim3 grid((s->nx + LBT_TX - 1) / LBT_TX, (s->ny + LBT_TY - 1) / LBT_TY, (s->nz + lz - 1) / lz);
  LaunchScope ls(s, kind);
  kern<<<grid, LBT_TX * LBT_TY, sizeof(T), s->stream>>>(s->kp, (const ST*)s->f[c], (ST*)s->f[d], phi_in ? phi_in : s->phi[c],
                                                        out_u, out_r, phi_out ? phi_out : s->phi[d], s->seams, s->tabs, lz,
                                                        s->tmap[c], s->tmap_row[c], in0, in1);
  return ACCLB_OK;
}

// FAST (all tiles full, TMA pull) when the tensor maps exist and the tile shape divides the box.
template <int MODE>
static int launch_lb_tp_any(accLB_ctx* s, int c, int d, int kind = KIND_LB_TP, double* out_u = nullptr,
                            double* out_r = nullptr, const double* in0 = nullptr, const double* in1 = nullptr) {
  if (MODE == MODE_UNFUSED) { out_u = s->u; out_r = s->r; }
  if (MODE == MODE_FUSED_U) out_u = s->u;
  constexpr bool CAN_FAST = MODE != MODE_INIT;
  if (s->prm.store_fp32) {
    if (CAN_FAST && s->tmap_ok) return launch_lb_tp<float, MODE, CAN_FAST>(s, c, d, kind, out_u, out_r, in0, in1);
    return launch_lb_tp<float, MODE, false>(s, c, d, kind, out_u, out_r, in0, in1);
  }
  if (CAN_FAST && s->tmap_ok) return launch_lb_tp<double, MODE, CAN_FAST>(s, c, d, kind, out_u, out_r, in0, in1);
  return launch_lb_tp<double, MODE, false>(s, c, d, kind, out_u, out_r, in0, in1);
}

// The fluxes through the seam faces of the tile columns (k_seam: one launch for the three directions), after
// k_lb_tp<FUSED> of the same step.
static int launch_seam(accLB_ctx* s, const double* phi_in, double* phi_out, bool scaled = false) {
  SeamGrid g;
  g.lz = s->lz;
  g.nchunk = (s->nz + s->lz - 1) / s->lz;
  g.nfx = (unsigned)((size_t)s->seams.ntx * s->ny * s->nz);
  g.nfy = (unsigned)((size_t)s->nx * s->seams.nty * s->nz);
  g.nfz = (unsigned)((size_t)s->nx * s->ny * g.nchunk);
  g.bx = blocks_for(g.nfx, SEAM_THREADS);
  g.by = blocks_for(g.nfy, SEAM_THREADS);
  g.bz = blocks_for(g.nfz, SEAM_THREADS);
  LaunchScope ls(s, KIND_SEAM);
  if (scaled) k_seam<LBT_TX, LBT_TY, true><<<g.bx + g.by + g.bz, SEAM_THREADS, 0, s->stream>>>(s->kp, phi_in, phi_out, s->seams, g);
  else k_seam<LBT_TX, LBT_TY, false><<<g.bx + g.by + g.bz, SEAM_THREADS, 0, s->stream>>>(s->kp, phi_in, phi_out, s->seams, g);
  return ACCLB_OK;
}

static int launch_advect(accLB_ctx* s, const double* phi_in, double* phi_out, const double* base = nullptr, double ca = 0.0,
                         double cb = 1.0) {
  using T = AdvTile<ADV_TX, ADV_TY>;
  auto kern = k_advect<ADV_TX, ADV_TY>;
  static thread_local int configured_device = -1;
  if (configured_device != s->prm.device) {
    CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(T)));
    configured_device = s->prm.device;
  }
  const int lz = planes_per_block(s->nx, s->ny, s->nz, ADV_TX, ADV_TY);
  const dim3 grid((s->nx + ADV_TX - 1) / ADV_TX, (s->ny + ADV_TY - 1) / ADV_TY, (s->nz + lz - 1) / lz);
  LaunchScope ls(s, KIND_ADVECT);
  kern<<<grid, ADV_TX * ADV_TY, sizeof(T), s->stream>>>(s->kp, phi_in, s->u, s->r, phi_out, lz, base, ca, cb);
  return ACCLB_OK;
}

// One single-phase step in the moment representation (k_mr_step, momrep.cuh).
constexpr int MR_TX = 32, MR_TY = 8, MR_NPT = 1;  // (two nodes per thread, 128-thread blocks: measured 7.27 vs 7.18 ms at 512^3)
template <bool FAST>
static int launch_mr_step_t(accLB_ctx* s, int c, int d) {
  using T = MomTile<MR_TX, MR_TY>;
  auto kern = k_mr_step<MR_TX, MR_TY, MR_NPT, 2, FAST>;
  static thread_local int configured_device = -1;
  if (configured_device != s->prm.device) {
    CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(T)));
    configured_device = s->prm.device;
  }
  const int lz = s->lz;
  const dim3 grid((s->nx + MR_TX - 1) / MR_TX, (s->ny + MR_TY - 1) / MR_TY, (s->nz + lz - 1) / lz);
  LaunchScope ls(s, KIND_MR);
  kern<<<grid, MR_TX * MR_TY / MR_NPT, sizeof(T), s->stream>>>(s->kp, s->ms[c], s->ms[d], s->tabs, lz, s->tmap[c]);
  return ACCLB_OK;
}
static int launch_mr_step(accLB_ctx* s, int c, int d) {
  return s->tmap_ok ? launch_mr_step_t<true>(s, c, d) : launch_mr_step_t<false>(s, c, d);
}

// One later stage of the SSP-RK3 integrator (R32): phi_out = a phi(t) + b (phi_in + L(phi_in; u(t))), the tiled kernel in
// MODE_STAGE and the seam faces after it.  phi(t) = phi[c], u(t) = s->u (written by k_lb_tp<MODE_FUSED_U> of this step).
static int launch_stage(accLB_ctx* s, int c, const double* phi_in, double* phi_out, double a, double b) {
  s->kp.rk_a = a;
  s->kp.rk_b = b;
  int r = s->tmap_ok ? launch_lb_tp<double, MODE_STAGE, true>(s, c, c, KIND_STAGE, nullptr, nullptr, s->phi[c], s->u, phi_in, phi_out)
                     : launch_lb_tp<double, MODE_STAGE, false>(s, c, c, KIND_STAGE, nullptr, nullptr, s->phi[c], s->u, phi_in, phi_out);
  if (!r) r = launch_seam(s, phi_in, phi_out, true);
  s->kp.rk_a = 0.0;
  s->kp.rk_b = 1.0;
  return r;
}

// r = D lap phi - kappa div q of a Runge-Kutta stage field (k_geom_r, phase_rk.cuh).
static int launch_geom_r(accLB_ctx* s, const double* phi_in) {
  using T = GeomTile<LBT_TX, LBT_TY>;
  auto kern = k_geom_r<LBT_TX, LBT_TY>;
  static thread_local int configured_device = -1;
  if (configured_device != s->prm.device) {
    CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(T)));
    configured_device = s->prm.device;
  }
  const int lz = s->lz;
  const dim3 grid((s->nx + LBT_TX - 1) / LBT_TX, (s->ny + LBT_TY - 1) / LBT_TY, (s->nz + lz - 1) / lz);
  LaunchScope ls(s, KIND_GEOM);
  kern<<<grid, LBT_TX * LBT_TY, sizeof(T), s->stream>>>(s->kp, phi_in, s->r, lz);
  return ACCLB_OK;
}

// Tensor maps of the two population buffers for the tiled TMA pull (k_lb_tp): rank 3, (x, y, slab = z * 27 + i), box
// LBT_TX x LBT_TY x 1 (unshifted in x: box starts must be 16-byte aligned), no swizzle, zero fill out of bounds.  Returns 1 on success; 0 (the kernels then use the per-thread
// cp.async pull everywhere) when the driver entry point is missing or the shape violates a tensor-map constraint.
static int make_tensor_maps(accLB_ctx* s) {
  typedef CUresult (*encode_t)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                               const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                               CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
      qres != cudaDriverEntryPointSuccess) {
    cudaGetLastError();
    return 0;
  }
  const size_t es = s->prm.store_fp32 ? 4 : 8;
  const CUtensorMapDataType dt = s->prm.store_fp32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64;
  if (s->nx % LBT_TX != 0 || s->ny % LBT_TY != 0) return 0;  // FAST: every tile full
  const cuuint64_t dims[3] = {(cuuint64_t)s->nx, (cuuint64_t)s->ny, (cuuint64_t)(s->prm.moment_storage ? 10 : 27) * s->nz};
  const cuuint64_t strides[2] = {(cuuint64_t)s->nx * es, (cuuint64_t)s->nx * s->ny * es};
  // two-phase: one box fetches the three populations of a triple (twophase.cuh); moment storage: one field per box
  const cuuint32_t box[3] = {LBT_TX, LBT_TY, s->prm.moment_storage ? 1u : 3u}, row[3] = {LBT_TX, 1, 1}, estr[3] = {1, 1, 1};
  for (int b = 0; b < 2; ++b) {
    CUresult r = ((encode_t)fn)(&s->tmap[b], dt, 3, s->f[b], dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,  // (128 B / 256 B promotion measured: no difference)
                                CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return 0;
    r = ((encode_t)fn)(&s->tmap_row[b], dt, 3, s->f[b], dims, strides, row, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                       CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return 0;
  }
  return 1;
}

extern "C" {

size_t accLB_workspace_bytes(int nx, int ny, int nz, const accLB_params* p) {
  if (!valid_args(nx, ny, nz, p)) return 0;
  return carve(nx, ny, nz, p).total;
}

int accLB_create(accLB_ctx** out, int nx, int ny, int nz, const accLB_params* p, void* workspace,
                 size_t workspace_bytes) {
  if (!out) return fail(ACCLB_EINVAL, "accLB_create: out is NULL");
  *out = nullptr;
  if (!valid_args(nx, ny, nz, p))
    return fail(ACCLB_EINVAL, "accLB_create: invalid grid %dx%dx%d or parameters (need nx,ny,nz >= 4, nx even, "
                              "nodes < 2^31, tau > 0.5, force_type in 0..2, two_phase: rho_l, rho_g, width > 0)",
                nx, ny, nz);
  const Carve c = carve(nx, ny, nz, p);
  if (!workspace || ((size_t)workspace & 255)) return fail(ACCLB_EWORKSPACE, "accLB_create: workspace NULL or not 256-byte aligned");
  if (workspace_bytes < c.total)
    return fail(ACCLB_EWORKSPACE, "accLB_create: workspace of %zu bytes, need %zu", workspace_bytes, c.total);
  int ndev = 0;
  CK(cudaGetDeviceCount(&ndev));
  if (p->device < 0 || p->device >= ndev) return fail(ACCLB_EINVAL, "accLB_create: device %d of %d", p->device, ndev);
  DeviceGuard guard_(p->device);
  if (!guard_.ok) return fail(ACCLB_ECUDA, "accLB_create: cannot select device %d", p->device);

  accLB_ctx* s = new (std::nothrow) accLB_ctx();
  if (!s) return fail(ACCLB_EINVAL, "accLB_create: out of host memory");
  s->prm = *p;
  s->nx = nx; s->ny = ny; s->nz = nz;
  s->n = (size_t)nx * ny * nz;
  s->stream = (cudaStream_t)p->stream;
  char* w = (char*)workspace;
  s->f[0] = w; w += c.f;
  s->f[1] = w; w += c.f;
  s->ms[0] = (double*)s->f[0]; s->ms[1] = (double*)s->f[1];
  s->phi[0] = p->two_phase ? (double*)w : nullptr; w += c.phi;
  s->phi[1] = p->two_phase ? (double*)w : nullptr; w += c.phi;
  s->u = p->two_phase ? (double*)w : nullptr; w += c.u;
  s->r = p->two_phase ? (double*)w : nullptr; w += c.r;
  s->tabs = (double*)w; w += c.tabs;
  s->acc = (double*)w; w += c.acc;
  s->seams.sx = p->two_phase ? (double*)w : nullptr; w += c.sx;
  s->seams.sy = p->two_phase ? (double*)w : nullptr; w += c.sy;
  s->seams.sz = p->two_phase ? (double*)w : nullptr; w += c.sz;
  s->seams.ntx = (nx + LBT_TX - 1) / LBT_TX;
  s->seams.nty = (ny + LBT_TY - 1) / LBT_TY;
  s->lz = planes_per_block(nx, ny, nz, LBT_TX, LBT_TY);
  s->phis = c.phis ? (double*)w : nullptr; w += c.phis;
  s->stage = p->host_staging ? (double*)w : nullptr; w += c.stage;
  s->cur = 0; s->step = 0; s->launches = 0; s->variant = 0; s->profiling = 0;
  for (int k = 0; k < ACCLB_NKERNELS; ++k) { s->folded_ms[k] = 0.0; s->folded_count[k] = 0; }

  KP& k = s->kp;
  k.G.nx = nx; k.G.ny = ny; k.G.nz = nz; k.G.n = (unsigned)s->n;
  k.omega = 1.0 / p->tau;
  k.one_m_omega = 1.0 - k.omega;
  k.rho_g = p->two_phase ? p->rho_g : 1.0;
  k.drho = p->two_phase ? p->rho_l - p->rho_g : 0.0;
  k.sig15w = p->sigma * (1.5 * p->width);
  k.visc_pref = (p->tau - 0.5) / p->tau;
  k.ratio_ne = p->two_phase && p->rho_l != p->rho_g;
  k.D = p->mobility;
  k.kappa = p->two_phase ? 4.0 * p->mobility / p->width : 0.0;
  k.force_type = p->force_type;
  k.force_amp = p->force_amp;
  for (int a = 0; a < 3; ++a) k.grav[a] = p->gravity[a];
  k.rho_ref = p->rho_ref;
  k.buoyant = p->gravity[0] != 0.0 || p->gravity[1] != 0.0 || p->gravity[2] != 0.0;
  k.nu = (p->tau - 0.5) / 3.0;
  k.eps_pref = k.nu / (2.0 * (1.0 / 9.0) * p->tau * p->tau);
  k.rk_a = 0.0; k.rk_b = 1.0;
  k.zlo = p->halo_z;
  k.zhi = nz - p->halo_z;

  // R20: per-axis sin/cos tables, libm on the host, k = 2 pi force_k / N, integer node coordinates
  std::vector<double> t((size_t)2 * (nx + ny + nz));
  const double two_pi = 6.283185307179586476925286766559;
  const int dims[3] = {nx, ny, nz};
  size_t o = 0;
  for (int ax = 0; ax < 3; ++ax) {
    // a z-slab (halo_z > 0) takes the table entries of its own planes out of the whole domain's table: the global
    // coordinate is reduced into [0, nz_global) first so that every slab evaluates sin / cos of the same arguments
    const bool slab = ax == 2 && p->halo_z > 0;
    const int period = slab ? p->nz_global : dims[ax];
    const double kk = two_pi * p->force_k / period;
    for (int j = 0; j < dims[ax]; ++j) {
      int g = j;
      if (slab) g = ((p->z_origin + j) % period + period) % period;
      t[o + j] = sin(kk * (double)g);
      t[o + dims[ax] + j] = cos(kk * (double)g);
    }
    o += (size_t)2 * dims[ax];
  }
  cudaError_t e = cudaMemcpyAsync(s->tabs, t.data(), t.size() * 8, cudaMemcpyHostToDevice, s->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  if (e != cudaSuccess) {
    delete s;
    return fail(ACCLB_ECUDA, "accLB_create: table upload: %s", cudaGetErrorString(e));
  }
  s->tmap_ok = p->two_phase || p->moment_storage ? make_tensor_maps(s) : 0;
  *out = s;
  g_err[0] = 0;
  return ACCLB_OK;
}

int accLB_init(accLB_ctx* s, const double* rho, const double* u, const double* phi) {
  if (!s || !rho || !u) return fail(ACCLB_EINVAL, "accLB_init: NULL argument");
  if (s->prm.two_phase && !phi) return fail(ACCLB_EINVAL, "accLB_init: phi is NULL for a two-phase context");
  GUARD_DEVICE(s);
  s->cur = 0;
  s->step = 0;
  const unsigned nb = blocks_for(s->n, 128);
  if (s->prm.two_phase) {
    // the tiled kernel in MODE_INIT: geometry of phi on shared-memory tiles, f_i pushed to x - c_i
    CK(cudaMemcpyAsync(s->phi[0], phi, s->n * 8, cudaMemcpyDeviceToDevice, s->stream));
    int r = launch_lb_tp_any<MODE_INIT>(s, 0, 0, KIND_INIT, nullptr, nullptr, rho, u);
    if (r) return r;
  } else if (s->prm.moment_storage) {
    LaunchScope ls(s, KIND_INIT);
    k_mr_init<<<blocks_for(s->n, 256), 256, 0, s->stream>>>(s->kp.G, rho, u, s->ms[0]);
  } else {
    LaunchScope ls(s, KIND_INIT);
    if (s->prm.store_fp32)
      k_init<float><<<nb, 128, 0, s->stream>>>(s->kp, rho, u, s->tabs, (float*)s->f[0]);
    else
      k_init<double><<<nb, 128, 0, s->stream>>>(s->kp, rho, u, s->tabs, (double*)s->f[0]);
  }
  CK(cudaGetLastError());
  return ACCLB_OK;
}

int accLB_step(accLB_ctx* s, int nsteps) {
  if (!s || nsteps < 0) return fail(ACCLB_EINVAL, "accLB_step: NULL context or negative nsteps");
  GUARD_DEVICE(s);
  const unsigned nb = blocks_for(s->n, 128);
  for (int it = 0; it < nsteps; ++it) {
    const int c = s->cur, d = c ^ 1;
    if (s->prm.two_phase && s->prm.phi_integrator == 1) {
      // SSP-RK3 for phi (R32), u frozen at time t.  Default: the fused time step is the first stage (it also writes u(t)),
      // the two later stages are the same tiled kernel without its LB half; each is followed by its seam faces.
      // Variant 1: the unfused form (u, r through HBM; k_geom_r + k_advect per stage), kept for comparison.
      int r;
      if (s->variant == 0) {
        if ((r = launch_lb_tp_any<MODE_FUSED_U>(s, c, d))) return r;                               // phi1 -> phi[d]
        if ((r = launch_seam(s, s->phi[c], s->phi[d]))) return r;
        if ((r = launch_stage(s, c, s->phi[d], s->phis, 0.75, 0.25))) return r;                    // phi2 -> phis
        if ((r = launch_stage(s, c, s->phis, s->phi[d], 1.0 / 3.0, 2.0 / 3.0))) return r;          // phi(t+1) -> phi[d]
      } else {
        if ((r = launch_lb_tp_any<MODE_UNFUSED>(s, c, d))) return r;
        if ((r = launch_advect(s, s->phi[c], s->phi[d]))) return r;                                  // phi1 -> phi[d]
        if ((r = launch_geom_r(s, s->phi[d]))) return r;
        if ((r = launch_advect(s, s->phi[d], s->phis, s->phi[c], 0.75, 0.25))) return r;             // phi2 -> phis
        if ((r = launch_geom_r(s, s->phis))) return r;
        if ((r = launch_advect(s, s->phis, s->phi[d], s->phi[c], 1.0 / 3.0, 2.0 / 3.0))) return r;   // phi(t+1) -> phi[d]
      }
    } else if (s->prm.two_phase && s->variant == 0) {
      // default: LB + geometry + advection fused on z-marching tiles (k_lb_tp), then the seam faces (k_seam)
      int r = launch_lb_tp_any<MODE_FUSED>(s, c, d);
      if (r) return r;
      r = launch_seam(s, s->phi[c], s->phi[d]);
      if (r) return r;
    } else if (s->prm.two_phase) {
      // variant 1: the forward-Euler form of the unfused path, u and r through HBM (k_lb_tp<MODE_UNFUSED>, k_advect)
      int r = launch_lb_tp_any<MODE_UNFUSED>(s, c, d);
      if (r) return r;
      r = launch_advect(s, s->phi[c], s->phi[d]);
      if (r) return r;
    } else if (s->prm.moment_storage) {
      int r = launch_mr_step(s, c, d);
      if (r) return r;
    } else {
      LaunchScope ls(s, KIND_LB);
      if (s->prm.store_fp32)
        k_lb<float><<<nb, 128, 0, s->stream>>>(s->kp, (const float*)s->f[c], (float*)s->f[d], s->tabs);
      else
        k_lb<double><<<nb, 128, 0, s->stream>>>(s->kp, (const double*)s->f[c], (double*)s->f[d], s->tabs);
    }
    s->cur = d;
    s->step += 1;
  }
  CK(cudaGetLastError());
  return ACCLB_OK;
}

int accLB_moments(accLB_ctx* s, double* rho, double* u, double* phi) {
  if (!s) return fail(ACCLB_EINVAL, "accLB_moments: NULL context");
  GUARD_DEVICE(s);
  const unsigned nb = blocks_for(s->n, 128);
  const int c = s->cur;
  if (s->prm.two_phase) {
    if (rho || u) {
      int r = launch_lb_tp_any<MODE_MOMENTS>(s, c, c, KIND_MOMENTS, u, rho);
      if (r) return r;
    }
    if (phi) CK(cudaMemcpyAsync(phi, s->phi[c], s->n * 8, cudaMemcpyDeviceToDevice, s->stream));
  } else if (s->prm.moment_storage) {
    LaunchScope ls(s, KIND_MOMENTS);
    k_mr_moments<<<blocks_for(s->n, 256), 256, 0, s->stream>>>(s->kp.G, s->ms[c], rho, u);
  } else {
    LaunchScope ls(s, KIND_MOMENTS);
    if (s->prm.store_fp32)
      k_moments<float><<<nb, 128, 0, s->stream>>>(s->kp, (const float*)s->f[c], s->tabs, rho, u);
    else
      k_moments<double><<<nb, 128, 0, s->stream>>>(s->kp, (const double*)s->f[c], s->tabs, rho, u);
  }
  CK(cudaGetLastError());
  return ACCLB_OK;
}

int accLB_diagnostics(accLB_ctx* s, double* out, int n_out) {
  if (!s || !out || n_out < ACCLB_NDIAG) return fail(ACCLB_EINVAL, "accLB_diagnostics: NULL argument or n_out < %d", ACCLB_NDIAG);
  GUARD_DEVICE(s);
  const int c = s->cur;
  CK(cudaMemsetAsync(s->acc, 0, 16 * 8, s->stream));
  unsigned nb = blocks_for(s->n, DIAG_THREADS);
  const unsigned cap = 148u * 16u;  // a multiple of the SM count; grid-stride beyond that
  if (nb > cap) nb = cap;
  if (s->prm.two_phase) {
    int r = launch_lb_tp_any<MODE_DIAG>(s, c, c, KIND_DIAG, nullptr, s->acc);
    if (r) return r;
  } else if (s->prm.moment_storage) {
    LaunchScope ls(s, KIND_DIAG);
    k_mr_diag<<<nb < 148u * 8u ? nb : 148u * 8u, 256, 0, s->stream>>>(s->kp, s->ms[c], s->tabs, s->acc);
  } else {
    LaunchScope ls(s, KIND_DIAG);
    if (s->prm.store_fp32)
      k_diagnostics<float><<<nb, DIAG_THREADS, 0, s->stream>>>(s->kp, (const float*)s->f[c], s->tabs, s->acc);
    else
      k_diagnostics<double><<<nb, DIAG_THREADS, 0, s->stream>>>(s->kp, (const double*)s->f[c], s->tabs, s->acc);
  }
  CK(cudaGetLastError());
  double h[8];
  CK(cudaMemcpyAsync(h, s->acc, sizeof h, cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  const double inv_n = 1.0 / ((double)s->nx * s->ny * (s->kp.zhi - s->kp.zlo));
  out[0] = h[0] * inv_n;
  out[1] = h[1] * inv_n;
  out[2] = h[2];
  out[3] = h[3];
  out[4] = h[4];
  out[5] = h[5];
  out[6] = h[6];
  out[7] = h[7];
  out[8] = (double)s->step;
  for (int j = 0; j < 8; ++j)
    if (!std::isfinite(out[j])) return fail(ACCLB_ENUMERIC, "accLB_diagnostics: entry %d is not finite", j);
  return ACCLB_OK;
}

int accLB_run_host(accLB_ctx* s, const double* h_rho, const double* h_u, const double* h_phi, int nsteps,
                   double* h_rho_out, double* h_u_out, double* h_phi_out, double* h_diag) {
  if (!s || !h_rho || !h_u || nsteps < 0) return fail(ACCLB_EINVAL, "accLB_run_host: NULL argument or negative nsteps");
  if (!s->stage) return fail(ACCLB_EINVAL, "accLB_run_host: context was created without host_staging");
  if (s->prm.two_phase && !h_phi) return fail(ACCLB_EINVAL, "accLB_run_host: h_phi is NULL for a two-phase context");
  GUARD_DEVICE(s);
  const size_t n = s->n;
  double* d_rho = s->stage;
  double* d_u = s->stage + n;
  double* d_phi = s->stage + 4 * n;
  CK(cudaMemcpyAsync(d_rho, h_rho, n * 8, cudaMemcpyHostToDevice, s->stream));
  CK(cudaMemcpyAsync(d_u, h_u, 3 * n * 8, cudaMemcpyHostToDevice, s->stream));
  if (s->prm.two_phase) CK(cudaMemcpyAsync(d_phi, h_phi, n * 8, cudaMemcpyHostToDevice, s->stream));
  int r = accLB_init(s, d_rho, d_u, s->prm.two_phase ? d_phi : nullptr);
  if (r) return r;
  r = accLB_step(s, nsteps);
  if (r) return r;
  if (h_rho_out || h_u_out || h_phi_out) {
    r = accLB_moments(s, d_rho, d_u, d_phi);
    if (r) return r;
    if (h_rho_out) CK(cudaMemcpyAsync(h_rho_out, d_rho, n * 8, cudaMemcpyDeviceToHost, s->stream));
    if (h_u_out) CK(cudaMemcpyAsync(h_u_out, d_u, 3 * n * 8, cudaMemcpyDeviceToHost, s->stream));
    if (h_phi_out && s->prm.two_phase) CK(cudaMemcpyAsync(h_phi_out, d_phi, n * 8, cudaMemcpyDeviceToHost, s->stream));
  }
  if (h_diag) {
    r = accLB_diagnostics(s, h_diag, ACCLB_NDIAG);
    if (r) return r;
  }
  CK(cudaStreamSynchronize(s->stream));
  return ACCLB_OK;
}

long long accLB_launch_count(const accLB_ctx* s) { return s ? s->launches : 0; }

int accLB_set_variant(accLB_ctx* s, int variant) {
  if (!s) return fail(ACCLB_EINVAL, "accLB_set_variant: NULL context");
  if (variant < 0 || variant > 1) return fail(ACCLB_EINVAL, "accLB_set_variant: unknown variant %d", variant);
  s->variant = variant;
  return ACCLB_OK;
}

static void drop_records(accLB_ctx* s) {
  for (auto& r : s->recs) {
    cudaEventDestroy(r.e0);
    cudaEventDestroy(r.e1);
  }
  s->recs.clear();
}

int accLB_profile(accLB_ctx* s, int enable) {
  if (!s) return fail(ACCLB_EINVAL, "accLB_profile: NULL context");
  s->profiling = enable != 0;
  return ACCLB_OK;
}

int accLB_profile_read(accLB_ctx* s, double* ms, long long* count, int n) {
  if (!s || !ms || !count || n < 1) return fail(ACCLB_EINVAL, "accLB_profile_read: NULL argument");
  GUARD_DEVICE(s);
  CK(cudaStreamSynchronize(s->stream));
  fold_records(s);
  for (int k = 0; k < n && k < ACCLB_NKERNELS; ++k) {
    ms[k] += s->folded_ms[k];
    count[k] += s->folded_count[k];
    s->folded_ms[k] = 0.0;
    s->folded_count[k] = 0;
  }
  return ACCLB_OK;
}

// The byte ranges of the halo exchange of a z-slab (include/acclb.h): whole [ny][nx] planes of consecutive populations of
// one z plane are contiguous in the [z][i][y][x] layout, so every item is one range.
int accLB_halo_chunks(accLB_ctx* s, int full, accLB_halo_chunk* out, int cap) {
  if (!s || !out) return fail(ACCLB_EINVAL, "accLB_halo_chunks: NULL argument");
  const int h = s->prm.halo_z;
  if (h <= 0) return fail(ACCLB_EINVAL, "accLB_halo_chunks: the context is not a z-slab (halo_z = 0)");
  const size_t plane = (size_t)s->nx * s->ny;
  const size_t es = s->prm.store_fp32 ? 4 : 8;
  char* f = (char*)s->f[s->cur];
  const int nz = s->nz;
  int n = 0;
  bool overflow = false;
  auto add = [&](void* ptr, size_t bytes, int side, int dir) {
    if (n >= cap) { overflow = true; return; }
    out[n].ptr = ptr; out[n].bytes = bytes; out[n].side = side; out[n].dir = dir;
    ++n;
  };
  // populations i0 .. i1-1 of plane z
  auto pops = [&](int z, int i0, int i1, int side, int dir) {
    add(f + ((size_t)z * 27 + i0) * plane * es, (size_t)(i1 - i0) * plane * es, side, dir);
  };
  auto phis = [&](int z0, int side, int dir) {
    if (s->prm.two_phase) add(s->phi[s->cur] + (size_t)z0 * plane, (size_t)h * plane * 8, side, dir);
  };
  for (int dir = 0; dir < 2; ++dir) {
    // dir 0: my own boundary planes, sent; dir 1: my halo planes, received.  The planes sent DOWN are the ones the lower
    // neighbour receives into its HIGH halo, and the other way round: the send list towards a side mirrors the receive
    // list from the other side.
    if (full) {
      // low end: halo planes [0, h) received from below | own planes [h, 2h) sent down
      pops(dir ? 0 : h, 0, 27 * h, -1, dir);
      phis(dir ? 0 : h, -1, dir);
      pops(dir ? nz - h : nz - 2 * h, 0, 27 * h, +1, dir);
      phis(dir ? nz - h : nz - 2 * h, +1, dir);
      continue;
    }
    const bool tp = s->prm.two_phase != 0;
    if (dir == 1) {
      // received from below: plane h-1 (c_z >= 0, or c_z = +1 single component), plane h-2 (c_z = +1)
      pops(h - 1, tp ? 9 : 18, 27, -1, 1);
      if (tp) pops(h - 2, 18, 27, -1, 1);
      phis(0, -1, 1);
      // received from above: plane nz-h (c_z <= 0 | c_z = -1), plane nz-h+1 (c_z = -1)
      pops(nz - h, 0, tp ? 18 : 9, +1, 1);
      if (tp) pops(nz - h + 1, 0, 9, +1, 1);
      phis(nz - h, +1, 1);
    } else {
      // sent down (the lower neighbour's "received from above"): my planes h, h+1
      pops(h, 0, tp ? 18 : 9, -1, 0);
      if (tp) pops(h + 1, 0, 9, -1, 0);
      phis(h, -1, 0);
      // sent up (the upper neighbour's "received from below"): my planes nz-h-1, nz-h-2
      pops(nz - h - 1, tp ? 9 : 18, 27, +1, 0);
      if (tp) pops(nz - h - 2, 18, 27, +1, 0);
      phis(nz - 2 * h, +1, 0);
    }
  }
  if (overflow) return fail(ACCLB_EINVAL, "accLB_halo_chunks: cap = %d is too small (ACCLB_MAX_HALO_CHUNKS)", cap);
  return n;
}

int accLB_destroy(accLB_ctx* s) {
  if (!s) return fail(ACCLB_EINVAL, "accLB_destroy: NULL context");
  drop_records(s);
  delete s;
  return ACCLB_OK;
}

const char* accLB_last_error(void) { return g_err; }

// ---------------------------------------------------------------------------------------- turbulence statistics (8(f) #4)
static bool stats_args(const void* u, int nx, int ny, int nz, const void* scratch) {
  return u && scratch && nx >= 1 && ny >= 1 && nz >= 1 && (double)nx * ny * nz < 2147483648.0;
}
static unsigned stats_blocks(size_t n) {
  const size_t b = (n + STATS_THREADS - 1) / STATS_THREADS, cap = 148 * 8;
  return (unsigned)(b < cap ? b : cap);
}

int accLB_stats_increments(const double* u, int nx, int ny, int nz, const int* r, int nr, double* out, void* scratch,
                           size_t scratch_bytes, int device, void* stream) {
  if (!stats_args(u, nx, ny, nz, scratch) || !r || !out || nr < 1) return fail(ACCLB_EINVAL, "accLB_stats_increments: bad argument");
  if (scratch_bytes < (size_t)nr * 3 * sizeof(double) || ((size_t)scratch & 7))
    return fail(ACCLB_EWORKSPACE, "accLB_stats_increments: scratch of %zu bytes, need %zu", scratch_bytes, (size_t)nr * 3 * sizeof(double));
  DeviceGuard guard_(device);
  if (!guard_.ok) return fail(ACCLB_ECUDA, "accLB_stats_increments: cannot select device %d", device);
  cudaStream_t st = (cudaStream_t)stream;
  Grid G{nx, ny, nz, (unsigned)((size_t)nx * ny * nz)};
  double* acc = (double*)scratch;
  CK(cudaMemsetAsync(acc, 0, (size_t)nr * 3 * sizeof(double), st));
  for (int j = 0; j < nr; ++j) {
    if (r[j] < 0) return fail(ACCLB_EINVAL, "accLB_stats_increments: negative separation");
    k_stats_increments<<<stats_blocks(G.n), STATS_THREADS, 0, st>>>(G, u, r[j], acc + 3 * j);
  }
  CK(cudaGetLastError());
  CK(cudaMemcpyAsync(out, acc, (size_t)nr * 3 * sizeof(double), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  const double inv = 1.0 / (3.0 * (double)G.n);
  for (int j = 0; j < 3 * nr; ++j) out[j] *= inv;
  return ACCLB_OK;
}

int accLB_stats_pdf(const double* u, int nx, int ny, int nz, int r, double scale, double lo, double hi, int nbins,
                    unsigned long long* counts, void* scratch, size_t scratch_bytes, int device, void* stream) {
  if (!stats_args(u, nx, ny, nz, scratch) || !counts || r < 0 || !(scale > 0.0) || !(hi > lo) || nbins < 1 || nbins > STATS_MAX_BINS)
    return fail(ACCLB_EINVAL, "accLB_stats_pdf: bad argument (1 <= nbins <= %d, hi > lo, scale > 0)", STATS_MAX_BINS);
  if (scratch_bytes < (size_t)nbins * sizeof(unsigned long long) || ((size_t)scratch & 7))
    return fail(ACCLB_EWORKSPACE, "accLB_stats_pdf: scratch too small");
  DeviceGuard guard_(device);
  if (!guard_.ok) return fail(ACCLB_ECUDA, "accLB_stats_pdf: cannot select device %d", device);
  cudaStream_t st = (cudaStream_t)stream;
  Grid G{nx, ny, nz, (unsigned)((size_t)nx * ny * nz)};
  unsigned long long* c = (unsigned long long*)scratch;
  CK(cudaMemsetAsync(c, 0, (size_t)nbins * sizeof(unsigned long long), st));
  k_stats_pdf<<<stats_blocks(G.n), STATS_THREADS, 0, st>>>(G, u, r, 1.0 / scale, lo, (double)nbins / (hi - lo), nbins, c);
  CK(cudaGetLastError());
  CK(cudaMemcpyAsync(counts, c, (size_t)nbins * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  return ACCLB_OK;
}

int accLB_stats_spectrum(const double* uhat, int nx, int ny, int nz, int ncomp, int nshell, double* E, void* scratch,
                         size_t scratch_bytes, int device, void* stream) {
  if (!stats_args(uhat, nx, ny, nz, scratch) || !E || ncomp < 1 || nshell < 1 || nshell > 4096)
    return fail(ACCLB_EINVAL, "accLB_stats_spectrum: bad argument (1 <= nshell <= 4096)");
  if (scratch_bytes < (size_t)nshell * sizeof(double) || ((size_t)scratch & 7)) return fail(ACCLB_EWORKSPACE, "accLB_stats_spectrum: scratch too small");
  DeviceGuard guard_(device);
  if (!guard_.ok) return fail(ACCLB_ECUDA, "accLB_stats_spectrum: cannot select device %d", device);
  cudaStream_t st = (cudaStream_t)stream;
  double* acc = (double*)scratch;
  CK(cudaMemsetAsync(acc, 0, (size_t)nshell * sizeof(double), st));
  const size_t nmode = (size_t)(nx / 2 + 1) * ny * nz;
  k_stats_spectrum<<<stats_blocks(nmode), STATS_THREADS, (size_t)nshell * sizeof(double), st>>>(nx, ny, nz, ncomp, (const double2*)uhat, nshell, acc);
  CK(cudaGetLastError());
  CK(cudaMemcpyAsync(E, acc, (size_t)nshell * sizeof(double), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  return ACCLB_OK;
}

// ---------------------------------------------------------------------------------------- no-allocation entry point
// Accumulators of accLB_stats_increments_static: device memory that belongs to the library image (one copy per GPU that loads
// it).  In host code `g_stats_static` is only a handle for the runtime, not a device address: the address a kernel can use
// comes from cudaGetSymbolAddress, asked for once per device with that device current.
static __device__ __align__(256) double g_stats_static[3 * ACCLB_STATS_STATIC_MAX_NR];

constexpr int STATIC_MAX_DEVICES = 64;
static double* g_stats_static_ptr[STATIC_MAX_DEVICES];  // per device; nullptr = not asked for yet
static std::mutex g_stats_static_mutex;

// Device address of g_stats_static on `device`, which must be the current device.
static int stats_static_address(int device, double** ptr) {
  if (device < 0 || device >= STATIC_MAX_DEVICES) return fail(ACCLB_EINVAL, "accLB_stats_increments_static: device %d", device);
  std::lock_guard<std::mutex> lock(g_stats_static_mutex);
  if (!g_stats_static_ptr[device]) {
    double* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void**)&p, g_stats_static);
    if (e != cudaSuccess || !p)
      return fail(ACCLB_ECUDA, "accLB_stats_increments_static: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
    g_stats_static_ptr[device] = p;
  }
  *ptr = g_stats_static_ptr[device];
  return ACCLB_OK;
}

int accLB_stats_increments_static(const double* u, int nx, int ny, int nz, const int* r, int nr, double* out, int device,
                                  void* stream) {
  if (!u || !r || !out || nr < 1 || nx < 1 || ny < 1 || nz < 1 || (double)nx * ny * nz >= 2147483648.0)
    return fail(ACCLB_EINVAL, "accLB_stats_increments_static: bad argument");
  if (nr > ACCLB_STATS_STATIC_MAX_NR)
    return fail(ACCLB_EINVAL, "accLB_stats_increments_static: nr = %d separations, the built-in scratch holds at most %d "
                              "(use accLB_stats_increments with a scratch block of your own)", nr, ACCLB_STATS_STATIC_MAX_NR);
  for (int j = 0; j < nr; ++j)
    if (r[j] < 0) return fail(ACCLB_EINVAL, "accLB_stats_increments_static: negative separation");
  DeviceGuard guard_(device);
  if (!guard_.ok) return fail(ACCLB_ECUDA, "accLB_stats_increments_static: cannot select device %d", device);
  double* acc = nullptr;
  int rc = stats_static_address(device, &acc);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  Grid G{nx, ny, nz, (unsigned)((size_t)nx * ny * nz)};
  CK(cudaMemsetAsync(acc, 0, (size_t)nr * 3 * sizeof(double), st));  // the array keeps the last call's sums
  for (int j = 0; j < nr; ++j) k_stats_increments<<<stats_blocks(G.n), STATS_THREADS, 0, st>>>(G, u, r[j], acc + 3 * j);
  CK(cudaGetLastError());
  CK(cudaMemcpyAsync(out, acc, (size_t)nr * 3 * sizeof(double), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  const double inv = 1.0 / (3.0 * (double)G.n);
  for (int j = 0; j < 3 * nr; ++j) out[j] *= inv;
  return ACCLB_OK;
}

}  // extern "C"
