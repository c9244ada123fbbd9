// SSP-RK3 integration of the conservative Allen-Cahn equation within one LB step (PAPER.md:L110 names "time
// integrators" without choosing one; reading R32), device side (sm_100a).  Part of the CUDA product path.
//
//   phi1 = phi + L(phi);  phi2 = 3/4 phi + 1/4 (phi1 + L(phi1));  phi(t+1) = 1/3 phi + 2/3 (phi2 + L(phi2)),
//   L(phi) = -div(u phi) [flux-form WENO5, R12] + D lap phi - kappa div(phi (1 - phi) n(phi))     PAPER.md:L61 (Eq. 3)
// with u = u(t) frozen.  One step is: k_lb_tp<unfused> (LB, writes u(t) and r(phi) = D lap phi - kappa div q), then per
// stage k_advect (twophase.cuh: the fluxes, the combination with the base field), and before stages 2 and 3
// k_geom_r (this file): r of the stage field on shared-memory tiles -- the geometry half of k_lb_tp without the
// populations.  u and r go through HBM here (the three stages need u three times); the fused single-pass kernel is
// the forward-Euler path.
#pragma once

namespace acclb {

template <int TX, int TY>
struct GeomTile {
  static constexpr int PX = TX + 4, PY = TY + 4;  // phi planes: tile + halo 2
  static constexpr int NX = TX + 2, NY = TY + 2;  // q planes: tile + halo 1
  alignas(16) double raw[4][PY][PX];              // ring of raw phi planes zc-1, zc, zc+1 and zc+2 (landing)
  double q[3][NY][NX];                            // q = phi (1 - phi) n of plane zc, n = g / (|g| + 1e-12) (R17)
  unsigned rowt[PY], colt[PX / 2];                // wrapped global offsets of the plane's rows / aligned column pairs
};

// r(z) = D lap phi - kappa div q for every node, marching along z (lz planes per block): per iteration zc the plane
// zc+2 is fetched (cp.async, 16-byte pairs), q is derived on tile + 1 rim from the planes zc-1, zc, zc+1 (separable
// lattice stencils), and the plane sums of q at zc complete div q of plane zc-1.
template <int TX, int TY>
__global__ void __launch_bounds__(TX * TY, 3)
k_geom_r(KP P, const double* __restrict__ phi, double* __restrict__ rout, int lz) {
  using T = GeomTile<TX, TY>;
  extern __shared__ __align__(128) unsigned char smem_lb[];
  T& S = *reinterpret_cast<T*>(smem_lb);
  constexpr int NT = TX * TY, PX = T::PX, NX = T::NX, PSZ = T::PX * T::PY;
  constexpr int RIM1 = T::NX * T::NY - NT, PAIRS = T::PX / 2 * T::PY;
  static_assert(RIM1 <= NT && PAIRS <= NT && T::PX % 2 == 0, "one rim item and one staging pair per thread");
  const Grid& G = P.G;
  const int tid = threadIdx.x, tx = tid % TX, ty = tid / TX;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, z0 = blockIdx.z * lz;
  const int z1 = min(z0 + lz, G.nz);
  const int x = x0 + tx, y = y0 + ty;
  const bool active = x < G.nx && y < G.ny;
  const unsigned plane = (unsigned)G.nx * (unsigned)G.ny;
  if (tid < T::PY) S.rowt[tid] = (unsigned)pmod(y0 - 2 + tid, G.ny) * (unsigned)G.nx;
  if (tid < T::PX / 2) S.colt[tid] = (unsigned)pmod(x0 - 2 + 2 * tid, G.nx);
  __syncthreads();
  const bool stager = tid < PAIRS;
  const unsigned soff = stager ? S.rowt[tid / (T::PX / 2)] + S.colt[tid % (T::PX / 2)] : 0u;
  const unsigned own = (unsigned)pmod(y, G.ny) * (unsigned)G.nx + (unsigned)pmod(x, G.nx);
  auto fetch = [&](int slot, int zz) {  // plane zz (any integer) -> ring slot
    if (stager) cp_async_16(&S.raw[slot][0][0] + 2 * tid, phi + (size_t)pmod(zz, G.nz) * plane + soff);
    cp_async_commit();
  };
  // ring slot of plane p: (p - z0 + 2) mod 4
  fetch(0, z0 - 2);
  fetch(1, z0 - 1);
  fetch(2, z0);
  double Pq = 0.0, Qq = 0.0, lapp = 0.0;  // carried: see k_lb_tp
  for (int zc = z0 - 1; zc <= z1; ++zc) {
    const int sm = (zc - z0 + 1) & 3, sc = (zc - z0 + 2) & 3, sp = (zc - z0 + 3) & 3;  // slots of planes zc-1, zc, zc+1
    fetch((zc - z0) & 3, zc + 2);  // one plane ahead, into the slot of plane zc-2 (last read before the barrier below ... of
                                   // the previous iteration)
    cp_async_wait_but<1>();
    __syncthreads();  // plane zc+1 has landed for everybody; q of the previous iteration has been consumed
    const double* rm = &S.raw[sm][0][0];
    const double* rc = &S.raw[sc][0][0];
    const double* rp = &S.raw[sp][0][0];
    double lapc = 0.0;
    auto derive = [&](int j, int i, bool own_node) {
      const int b = j * PX + i;
      double t[9], d[9], ph = 0.0;
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const int e = b + a * PX + c;
          const double m = rm[e], v = rc[e], p = rp[e];
          t[3 * a + c] = fma(4.0, v, m + p);
          d[3 * a + c] = p - m;
          if (a == 1 && c == 1) ph = v;
        }
      const double gx = (1.0 / 72.0) * fma(4.0, t[5] - t[3], (t[2] - t[0]) + (t[8] - t[6]));
      const double gy = (1.0 / 72.0) * fma(4.0, t[7] - t[1], (t[6] - t[0]) + (t[8] - t[2]));
      const double gz = (1.0 / 72.0) * fma(4.0, fma(4.0, d[4], d[3] + d[5]), fma(4.0, d[1], d[0] + d[2]) + fma(4.0, d[7], d[6] + d[8]));
      const double gn = sqrt_pos(fma(gx, gx, fma(gy, gy, gz * gz)));
      const double pq = ph * (1.0 - ph) * div_pos(1.0, gn + 1e-12);
      S.q[0][j][i] = pq * gx;
      S.q[1][j][i] = pq * gy;
      S.q[2][j][i] = pq * gz;
      if (own_node) {
        const double s0 = fma(4.0, t[1], t[0] + t[2]), s1 = fma(4.0, t[4], t[3] + t[5]), s2 = fma(4.0, t[7], t[6] + t[8]);
        lapc = 6.0 * (fma(4.0, s1, s0 + s2) * (1.0 / 216.0) - ph);  // R7
      }
    };
    derive(ty + 1, tx + 1, true);
    if (tid < RIM1) {
      int j, i;
      if (tid < NX) { j = 0; i = tid; }
      else if (tid < 2 * NX) { j = T::NY - 1; i = tid - NX; }
      else { const int e = tid - 2 * NX; j = 1 + (e >> 1); i = (e & 1) ? NX - 1 : 0; }
      derive(j, i, false);
    }
    __syncthreads();
    // plane sums of q at the own node:  a = Dx Sy q_x + Sx Dy q_y,  b = Sx Sy q_z
    const double* vx = &S.q[0][ty][tx];
    const double* vy = &S.q[1][ty][tx];
    const double* vz = &S.q[2][ty][tx];
    const double ax = fma(4.0, vx[NX + 2] - vx[NX], (vx[2] - vx[0]) + (vx[2 * NX + 2] - vx[2 * NX]));
    const double ay = fma(4.0, vy[2 * NX + 1] - vy[1], (vy[2 * NX] - vy[0]) + (vy[2 * NX + 2] - vy[2]));
    const double aq = ax + ay;
    const double bq = fma(4.0, fma(4.0, vz[NX + 1], vz[NX] + vz[NX + 2]),
                          fma(4.0, vz[1], vz[0] + vz[2]) + fma(4.0, vz[2 * NX + 1], vz[2 * NX] + vz[2 * NX + 2]));
    const int z = zc - 1;
    if (z >= z0 && z < z1 && active) {
      const double divq = (1.0 / 72.0) * (Pq + (aq + bq));
      rout[(size_t)z * plane + own] = P.D * lapp - P.kappa * divq;
    }
    Pq = fma(4.0, aq, Qq);
    Qq = aq - bq;
    lapp = lapc;
  }
}

}  // namespace acclb
