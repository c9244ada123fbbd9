// Two-phase step as ONE persistent kernel: a plane-by-plane software pipeline through L2 (sm_100a).
// Part of the CUDA product path.  DESIGN.md section 7.
//
// One time step t -> t+1 of the two-phase path (rows a1-a8 of DESIGN.md section 1) is four stages per lattice plane z:
//   N(z)    n = grad phi / (|grad phi| + 1e-12)                                     PAPER.md:L61, L104; R17
//   K(z)    g = grad phi, c = -gamma (3 delta/2) (div n) |g|   (F^s = c g)          PAPER.md:L102, L104; R8
//           r = D lap phi - kappa div(phi (1 - phi) n)         (phi-only part of Eq. 3)
//   LB(z)   pull-stream, moments, forces, u, Hermite coefficient, regularized reconstruction, aligned store
//           (Eqs. 4-8), writes u for the advection
//   ADV(z)  phi+ = phi - sum_e (Phi_e(x) - Phi_e(x - e)) + r, Phi = u_f WENO5(phi)   PAPER.md:L61-67 (Eq. 3), R12
// A stage of plane z needs a few planes of the previous stage (K: n at z-1..z+1, LB: g,c at z, ADV: u at z..z+1, r
// at z, the z-face flux of ADV(z-1)).  Instead of one kernel per stage with full-size intermediate arrays in HBM
// (n, g, c, r, u: 12 doubles per node written and read back), the stages run as work items of one persistent kernel,
// ordered plane by plane with a lag of one to three planes between stages, and the intermediates live in ring
// buffers of a few planes that stay resident in the 126 MB L2: HBM sees the populations (27 + 27), phi (1 + 1) and
// little else.  The fp64-ALU-bound stages (N, K, ADV) share the SMs with the HBM-bound LB items and hide under them.
//
// Scheduling.  Blocks take tickets from one global counter; ticket -> (macro step m, stage, item).  Macro step m holds,
// in this order, N(zz = m-2), LB(zz = m-4), K(zz = m-3), ADV(zz = m-6).  zz is the unwrapped plane coordinate,
// z = zz mod nz; N covers zz in [-2, nz+1], K and LB [-1, nz], ADV [0, nz-1]: the two wrap-around planes are simply
// processed twice (LB is idempotent: it reads buffer A and writes buffer B), so the pipeline is linear and the
// periodic wrap needs no special case.  An item waits (one thread spins on an acquire load) until the per-plane
// completion counters of the items it depends on are full.  It only ever waits for items with SMALLER tickets, and a
// ticket is handed out to a block that is already running, so the item with the smallest unfinished ticket can always
// proceed: no deadlock, whatever the number of resident blocks.
// Ring data are written by one SM and read by another inside one launch: they are read with ld.global.cg (L2, never a
// stale L1 line) after an acquire of the counter, and published with __syncthreads + __threadfence + atomicAdd.
#pragma once

namespace acclb {

constexpr int PIPE_THREADS = 256;
constexpr int PIPE_TX = 32, PIPE_TY = 8;  // tile of the N, K, ADV items; LB items are 256 consecutive nodes of a plane
// Planes per ring: just what the schedule keeps live plus one macro step of slack, so that the rings' footprint
// in L2 stays small and a dead plane is overwritten while its lines are still resident (no write-back to HBM).
constexpr int RING_N = 4, RING_GC = 3, RING_R = 4, RING_U = 4, RING_FZ = 3;
constexpr int PIPE_RING_DOUBLES = 3 * RING_N + 4 * RING_GC + RING_R + 3 * RING_U + RING_FZ;  // per node of a plane
// Macro step m holds N(zz = m - 2), LB(zz = m - 2 - LAG_LB), K(zz = m - 2 - LAG_K), ADV(zz = m - 2 - LAG_ADV).
constexpr int LAG_K = 1, LAG_LB = 2, LAG_ADV = 4;
enum { ST_N = 0, ST_LB = 1, ST_K = 2, ST_ADV = 3 };

struct PipeArgs {
  KP P;
  const void* fin;    // populations of time t (post-collision, not yet streamed), [nz][27][ny][nx]
  void* fout;         // populations of time t+1
  const double* phi;  // phi(t), [nz][ny][nx]
  double* phi_new;    // phi(t+1)
  const double* tabs;
  double* ring_n;     // [RING_N][3][ny][nx]
  double* ring_gc;    // [RING_GC][4][ny][nx]  g_x g_y g_z c
  double* ring_r;     // [RING_R][ny][nx]
  double* ring_u;     // [RING_U][3][ny][nx]
  double* ring_fz;    // [RING_FZ][ny][nx]     advective flux through the face (z, z+1)
  int* ticket;        // one counter
  int* done;          // [4][nz + 4] completion counters, index zz + 2
  int tiles_x, tiles_y, tiles;  // tiles of PIPE_TX x PIPE_TY per plane
  int lb_items;                 // ceil(nx ny / 256)
  int per_macro;                // 3 tiles + lb_items
  int total;                    // (nz + 3 + LAG_ADV) per_macro
};

__device__ __forceinline__ int ld_acquire(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
// a + n-periodic wrap for a in [-n, n + anything)
__device__ __forceinline__ int wrapg(int a, int n) {
  if (a < 0) a += n;
  if (a >= n) {
    a -= n;
    if (a >= n) a %= n;
  }
  return a;
}
template <int R>
__device__ __forceinline__ int ring_slot(int zz) { return (zz + 2) % R; }

// 3 x 3 in-plane stencils on a row-major plane of pitch PX, p pointing at the (-1,-1) corner; W = (1,4,1)
template <int PX>
__device__ __forceinline__ double st_DxSy(const double* p) {  // Dx Sy
  return fma(4.0, p[PX + 2] - p[PX], (p[2] - p[0]) + (p[2 * PX + 2] - p[2 * PX]));
}
template <int PX>
__device__ __forceinline__ double st_SxDy(const double* p) {  // Sx Dy
  return fma(4.0, p[2 * PX + 1] - p[1], (p[2 * PX] - p[0]) + (p[2 * PX + 2] - p[2]));
}
template <int PX>
__device__ __forceinline__ double st_SxSy(const double* p) {  // Sx Sy
  const double r0 = fma(4.0, p[1], p[0] + p[2]);
  const double r1 = fma(4.0, p[PX + 1], p[PX] + p[PX + 2]);
  const double r2 = fma(4.0, p[2 * PX + 1], p[2 * PX] + p[2 * PX + 2]);
  return fma(4.0, r1, r0 + r2);
}

// Shared memory of one block: the union of what the stages need.
struct PipeSmem {
  static constexpr int HX = PIPE_TX + 2, HY = PIPE_TY + 2;  // tile + halo 1
  union {
    struct { double Tz[HY][HX], Dz[HY][HX]; } n;            // N: Sz phi, Dz phi
    struct { double f[9][HY][HX]; } k;                      // K: Sz n_x, Sz n_y, Dz n_z, Sz q_x, Sz q_y, Dz q_z, Sz phi, Dz phi, phi
    struct {
      double phi[PIPE_TY + 6][PIPE_TX + 6];                 // plane z with halo 3 along x and y (corners unused)
      double ux[PIPE_TY][PIPE_TX + 2];
      double uy[PIPE_TY + 2][PIPE_TX];
      double fx[PIPE_TY][PIPE_TX + 1];
      double fy[PIPE_TY + 1][PIPE_TX];
    } a;
  };
  int ticket;
};

// ---------------------------------------------------------------------------------------------------- stage N
// n(z) at the tile's own nodes from phi(z-1..z+1): z combinations per column first (Sz = (1,4,1), Dz = (+1,0,-1)),
// then the 3 x 3 in-plane stencils.  Same numbers as the 27-term sums of PAPER.md:L104 up to rounding order.
__device__ __forceinline__ void stage_N(const PipeArgs& a, PipeSmem& S, int zz, int tile) {
  const Grid& G = a.P.G;
  constexpr int HX = PipeSmem::HX, HY = PipeSmem::HY;
  const int tid = threadIdx.x;
  const int x0 = (tile % a.tiles_x) * PIPE_TX, y0 = (tile / a.tiles_x) * PIPE_TY;
  const unsigned plane = (unsigned)G.nx * (unsigned)G.ny;
  const int z = wrapg(zz + G.nz, G.nz);
  const double* pm = a.phi + (size_t)wrap_dec(z, G.nz) * plane;
  const double* pc = a.phi + (size_t)z * plane;
  const double* pp = a.phi + (size_t)wrap_inc(z, G.nz) * plane;
  for (int e = tid; e < HX * HY; e += PIPE_THREADS) {
    const int j = e / HX, i = e - j * HX;
    const unsigned off = (unsigned)wrapg(y0 - 1 + j, G.ny) * (unsigned)G.nx + (unsigned)wrapg(x0 - 1 + i, G.nx);
    const double m = __ldg(pm + off), c = __ldg(pc + off), p = __ldg(pp + off);
    S.n.Tz[j][i] = fma(4.0, c, m + p);
    S.n.Dz[j][i] = p - m;
  }
  __syncthreads();
  const int tx = tid % PIPE_TX, ty = tid / PIPE_TX;
  const int x = x0 + tx, y = y0 + ty;
  if (x < G.nx && y < G.ny) {
    const double gx = (1.0 / 72.0) * st_DxSy<HX>(&S.n.Tz[ty][tx]);
    const double gy = (1.0 / 72.0) * st_SxDy<HX>(&S.n.Tz[ty][tx]);
    const double gz = (1.0 / 72.0) * st_SxSy<HX>(&S.n.Dz[ty][tx]);
    const double inv = 1.0 / (sqrt(fma(gx, gx, fma(gy, gy, gz * gz))) + 1e-12);  // R17
    double* out = a.ring_n + (size_t)ring_slot<RING_N>(zz) * 3 * plane + (unsigned)y * (unsigned)G.nx + (unsigned)x;
    out[0] = gx * inv;
    out[plane] = gy * inv;
    out[2 * plane] = gz * inv;
  }
}

// ---------------------------------------------------------------------------------------------------- stage K
// g, c = -gamma (3 delta/2) kappa_c |g| and r = D lap phi - kappa div q of plane z, kappa_c = div n, q = phi (1-phi) n.
__device__ __forceinline__ void stage_K(const PipeArgs& a, PipeSmem& S, int zz, int tile) {
  const Grid& G = a.P.G;
  constexpr int HX = PipeSmem::HX, HY = PipeSmem::HY;
  const int tid = threadIdx.x;
  const int x0 = (tile % a.tiles_x) * PIPE_TX, y0 = (tile / a.tiles_x) * PIPE_TY;
  const unsigned plane = (unsigned)G.nx * (unsigned)G.ny;
  const int z = wrapg(zz + G.nz, G.nz);
  const double* pm = a.phi + (size_t)wrap_dec(z, G.nz) * plane;
  const double* pc = a.phi + (size_t)z * plane;
  const double* pp = a.phi + (size_t)wrap_inc(z, G.nz) * plane;
  const double* nm = a.ring_n + (size_t)ring_slot<RING_N>(zz - 1) * 3 * plane;
  const double* nc = a.ring_n + (size_t)ring_slot<RING_N>(zz) * 3 * plane;
  const double* np = a.ring_n + (size_t)ring_slot<RING_N>(zz + 1) * 3 * plane;
  for (int e = tid; e < HX * HY; e += PIPE_THREADS) {
    const int j = e / HX, i = e - j * HX;
    const unsigned off = (unsigned)wrapg(y0 - 1 + j, G.ny) * (unsigned)G.nx + (unsigned)wrapg(x0 - 1 + i, G.nx);
    const double fm = __ldg(pm + off), fc = __ldg(pc + off), fp = __ldg(pp + off);
    const double nxm = __ldcg(nm + off), nym = __ldcg(nm + plane + off), nzm = __ldcg(nm + 2 * plane + off);
    const double nxc = __ldcg(nc + off), nyc = __ldcg(nc + plane + off);
    const double nxp = __ldcg(np + off), nyp = __ldcg(np + plane + off), nzp = __ldcg(np + 2 * plane + off);
    const double qm = fm * (1.0 - fm), qc = fc * (1.0 - fc), qp = fp * (1.0 - fp);
    S.k.f[0][j][i] = fma(4.0, nxc, nxm + nxp);
    S.k.f[1][j][i] = fma(4.0, nyc, nym + nyp);
    S.k.f[2][j][i] = nzp - nzm;
    S.k.f[3][j][i] = fma(4.0, qc * nxc, qm * nxm + qp * nxp);
    S.k.f[4][j][i] = fma(4.0, qc * nyc, qm * nym + qp * nyp);
    S.k.f[5][j][i] = qp * nzp - qm * nzm;
    S.k.f[6][j][i] = fma(4.0, fc, fm + fp);
    S.k.f[7][j][i] = fp - fm;
    S.k.f[8][j][i] = fc;
  }
  __syncthreads();
  const int tx = tid % PIPE_TX, ty = tid / PIPE_TX;
  const int x = x0 + tx, y = y0 + ty;
  if (x < G.nx && y < G.ny) {
    const double kc = (1.0 / 72.0) * (st_DxSy<HX>(&S.k.f[0][ty][tx]) + st_SxDy<HX>(&S.k.f[1][ty][tx]) + st_SxSy<HX>(&S.k.f[2][ty][tx]));
    const double dq = (1.0 / 72.0) * (st_DxSy<HX>(&S.k.f[3][ty][tx]) + st_SxDy<HX>(&S.k.f[4][ty][tx]) + st_SxSy<HX>(&S.k.f[5][ty][tx]));
    const double gx = (1.0 / 72.0) * st_DxSy<HX>(&S.k.f[6][ty][tx]);
    const double gy = (1.0 / 72.0) * st_SxDy<HX>(&S.k.f[6][ty][tx]);
    const double gz = (1.0 / 72.0) * st_SxSy<HX>(&S.k.f[7][ty][tx]);
    const double lap = 6.0 * (st_SxSy<HX>(&S.k.f[6][ty][tx]) * (1.0 / 216.0) - S.k.f[8][ty + 1][tx + 1]);  // R7
    const double gn = sqrt(fma(gx, gx, fma(gy, gy, gz * gz)));
    const unsigned o = (unsigned)y * (unsigned)G.nx + (unsigned)x;
    double* gc = a.ring_gc + (size_t)ring_slot<RING_GC>(zz) * 4 * plane + o;
    gc[0] = gx;
    gc[plane] = gy;
    gc[2 * plane] = gz;
    gc[3 * plane] = -a.P.sig15w * kc * gn;  // F^s = c g (R8)
    a.ring_r[(size_t)ring_slot<RING_R>(zz) * plane + o] = a.P.D * lap - a.P.kappa * dq;  // phi-only part of Eq. 3
  }
}

// ---------------------------------------------------------------------------------------------------- stage LB
// The fused LB update of 256 consecutive nodes of plane z (rows a1-a7), geometry g, c from K through the L2 ring.
template <typename ST>
__device__ __forceinline__ void stage_LB(const PipeArgs& a, int zz, int item) {
  const KP& P = a.P;
  const Grid& G = P.G;
  const unsigned plane = (unsigned)G.nx * (unsigned)G.ny;
  const unsigned idx = (unsigned)item * PIPE_THREADS + threadIdx.x;
  if (idx >= plane) return;
  const int z = wrapg(zz + G.nz, G.nz);
  const int y = (int)(idx / (unsigned)G.nx), x = (int)(idx - (unsigned)y * (unsigned)G.nx);
  Nbr nb;
  make_nbr(G, x, y, z, nb);
  const unsigned k = (unsigned)z * plane + idx;
  double f[Q];
  pull27<ST>((const ST*)a.fin, G, nb, f);
  const double* gc = a.ring_gc + (size_t)ring_slot<RING_GC>(zz) * 4 * plane + idx;
  const double g[3] = {__ldcg(gc), __ldcg(gc + plane), __ldcg(gc + 2 * plane)};
  const double c = __ldcg(gc + 3 * plane);
  const double phi0 = __ldg(a.phi + k);
  Moments M;
  moments_of(f, M);
  double Fb[3], A[3], rho;
  body_force(P, a.tabs, x, y, z, Fb);
  accel_from_gc(P, M, g, c, phi0, Fb, true, A, rho);
  const double u[3] = {M.m[0] + 0.5 * A[0], M.m[1] + 0.5 * A[1], M.m[2] + 0.5 * A[2]};  // a5, PAPER.md:L88 (R4)
  double* uo = a.ring_u + (size_t)ring_slot<RING_U>(zz) * 3 * plane + idx;
  uo[0] = u[0];
  uo[plane] = u[1];
  uo[2 * plane] = u[2];
  collide_store<ST>(P, M, u, A, f, pop_slab((ST*)a.fout, G, z) + idx, plane);
}

// ---------------------------------------------------------------------------------------------------- stage ADV
// phi+(z) on one tile: x / y face fluxes once per face through shared memory, the flux through the face (z, z+1)
// computed here and handed to ADV(z+1) through the ring, so every face flux is evaluated once and sum phi is
// conserved to rounding (R12).
__device__ __forceinline__ void stage_ADV(const PipeArgs& a, PipeSmem& S, int zz, int tile) {
  const Grid& G = a.P.G;
  constexpr int TX = PIPE_TX, TY = PIPE_TY;
  static_assert(6 * (TX + TY) <= PIPE_THREADS, "one halo element per thread");
  const int tid = threadIdx.x, tx = tid % TX, ty = tid / TX;
  const int x0 = (tile % a.tiles_x) * TX, y0 = (tile / a.tiles_x) * TY;
  const int x = x0 + tx, y = y0 + ty, z = zz;
  const bool active = x < G.nx && y < G.ny;
  const unsigned plane = (unsigned)G.nx * (unsigned)G.ny;
  const unsigned own = (unsigned)wrapg(y, G.ny) * (unsigned)G.nx + (unsigned)wrapg(x, G.nx);
  const double* uc = a.ring_u + (size_t)ring_slot<RING_U>(zz) * 3 * plane;
  const double* uzp = a.ring_u + (size_t)ring_slot<RING_U>(zz + 1) * 3 * plane + 2 * plane;
  auto zoff = [&](int k) { return (size_t)wrapg(z + k + G.nz, G.nz) * plane; };
  const size_t zo = (size_t)z * plane;

  // phi halo element of this thread (tid < 6 (TX + TY)): rows above/below first, then columns left/right
  if (tid < 6 * TX) {
    const int rr = tid / TX;  // 0..5 -> tile rows -3,-2,-1, TY, TY+1, TY+2
    const int hj = rr < 3 ? rr : TY + rr, hi = 3 + tid % TX;
    S.a.phi[hj][hi] = __ldg(a.phi + zo + (unsigned)wrapg(y0 - 3 + hj, G.ny) * (unsigned)G.nx + (unsigned)wrapg(x0 - 3 + hi, G.nx));
  } else if (tid < 6 * (TX + TY)) {
    const int e = tid - 6 * TX, cc = e % 6;  // 0..5 -> tile columns -3,-2,-1, TX, TX+1, TX+2
    const int hj = 3 + e / 6, hi = cc < 3 ? cc : TX + cc;
    S.a.phi[hj][hi] = __ldg(a.phi + zo + (unsigned)wrapg(y0 - 3 + hj, G.ny) * (unsigned)G.nx + (unsigned)wrapg(x0 - 3 + hi, G.nx));
  }
  // velocity halo element (tid < 2 (TX + TY)): u_y rows -1, TY ; u_x columns -1, TX
  if (tid < 2 * TX) {
    const int vj = tid < TX ? 0 : TY + 1, vi = tid % TX;
    S.a.uy[vj][vi] = __ldcg(uc + plane + (unsigned)wrapg(y0 - 1 + vj, G.ny) * (unsigned)G.nx + (unsigned)wrapg(x0 + vi, G.nx));
  } else if (tid < 2 * (TX + TY)) {
    const int e = tid - 2 * TX, vj = e / 2, vi = (e & 1) ? TX + 1 : 0;
    S.a.ux[vj][vi] = __ldcg(uc + (unsigned)wrapg(y0 + vj, G.ny) * (unsigned)G.nx + (unsigned)wrapg(x0 - 1 + vi, G.nx));
  }
  // column window w[j] = phi(z - 2 + j), j = 0..5, of the z face between z and z + 1
  const double w0 = __ldg(a.phi + zoff(-2) + own), w1 = __ldg(a.phi + zoff(-1) + own), w2 = __ldg(a.phi + zo + own);
  const double w3 = __ldg(a.phi + zoff(1) + own), w4 = __ldg(a.phi + zoff(2) + own), w5 = __ldg(a.phi + zoff(3) + own);
  const double uz0 = __ldcg(uc + 2 * plane + own), uz1 = __ldcg(uzp + own);
  S.a.phi[ty + 3][tx + 3] = w2;
  S.a.ux[ty][tx + 1] = __ldcg(uc + own);
  S.a.uy[ty + 1][tx] = __ldcg(uc + plane + own);
  const double rr = __ldcg(a.ring_r + (size_t)ring_slot<RING_R>(zz) * plane + own);
  double fz_lo;
  if (zz == 0) {  // the first plane of the sweep evaluates its lower face itself (same operations, same bits)
    const double uzm = __ldcg(a.ring_u + (size_t)ring_slot<RING_U>(zz - 1) * 3 * plane + 2 * plane + own);
    fz_lo = face_flux(uzm, uz0, __ldg(a.phi + zoff(-3) + own), w0, w1, w2, w3, w4);
  } else {
    fz_lo = __ldcg(a.ring_fz + (size_t)ring_slot<RING_FZ>(zz - 1) * plane + own);
  }
  __syncthreads();
  for (int e = tid; e < TY * (TX + 1); e += PIPE_THREADS) {  // x faces
    const int j = e / (TX + 1), i = e % (TX + 1);
    const double* p = &S.a.phi[j + 3][i];  // p[0..5] = phi at tile columns i-3 .. i+2 = L-2 .. L+3 with L = i-1
    S.a.fx[j][i] = face_flux(S.a.ux[j][i], S.a.ux[j][i + 1], p[0], p[1], p[2], p[3], p[4], p[5]);
  }
  for (int e = tid; e < (TY + 1) * TX; e += PIPE_THREADS) {  // y faces
    const int j = e / TX, i = e % TX;
    S.a.fy[j][i] = face_flux(S.a.uy[j][i], S.a.uy[j + 1][i], S.a.phi[j][i + 3], S.a.phi[j + 1][i + 3], S.a.phi[j + 2][i + 3],
                             S.a.phi[j + 3][i + 3], S.a.phi[j + 4][i + 3], S.a.phi[j + 5][i + 3]);
  }
  const double fz = face_flux(uz0, uz1, w0, w1, w2, w3, w4, w5);  // face (z, z + 1)
  __syncthreads();
  if (active) {
    double adv = 0.0;
    adv += S.a.fx[ty][tx + 1] - S.a.fx[ty][tx];
    adv += S.a.fy[ty + 1][tx] - S.a.fy[ty][tx];
    adv += fz - fz_lo;
    __stcs(a.phi_new + zo + own, w2 + (-adv + rr));
    a.ring_fz[(size_t)ring_slot<RING_FZ>(zz) * plane + own] = fz;
  }
}

// ---------------------------------------------------------------------------------------------------- the kernel
// j-th thing item (stage, zz) has to wait for: the counter index and the count it must reach.  First the data
// dependencies, then the readers of the ring planes the item is about to overwrite.
__device__ __forceinline__ bool pipe_dep(const PipeArgs& a, int stage, int zz, int j, int& idx, int& cnt) {
  const int nz = a.P.G.nz, npos = nz + 4;
  int st = -1, z = 0;
  if (stage == ST_N) {  // readers of n(zz - RING_N): K(zz - RING_N - 1 .. zz - RING_N + 1)
    if (j < 3) { st = ST_K; z = zz - RING_N - 1 + j; }
  } else if (stage == ST_K) {
    if (j < 3) { st = ST_N; z = zz - 1 + j; }
    else if (j == 3) { st = ST_LB; z = zz - RING_GC; }  // reader of g,c(zz - RING_GC)
    else if (j == 4) { st = ST_ADV; z = zz - RING_R; }  // reader of r(zz - RING_R)
  } else if (stage == ST_LB) {
    if (j == 0) { st = ST_K; z = zz; }
    else if (j == 1 && zz - RING_U >= -1) { st = ST_ADV; z = max(zz - RING_U, 0); }  // readers of u(zz - RING_U): ADV(zz - RING_U - 1), ADV(zz - RING_U); ADV(0) reads u(-1)
  } else {
    if (j == 0) { st = ST_LB; z = zz; }
    else if (j == 1) { st = ST_LB; z = zz + 1; }
    else if (j == 2) { if (zz == 0) { st = ST_LB; z = -1; } else { st = ST_ADV; z = zz - 1; } }  // also frees fz(zz - RING_FZ)
  }
  if (st < 0) return false;
  const bool exists = st == ST_N ? (z >= -2 && z <= nz + 1) : st == ST_ADV ? (z >= 0 && z <= nz - 1) : (z >= -1 && z <= nz);
  if (!exists) return false;
  idx = st * npos + z + 2;
  cnt = st == ST_LB ? a.lb_items : a.tiles;
  return true;
}

template <typename ST, int MINB>
__global__ void __launch_bounds__(PIPE_THREADS, MINB) k_step_tp(const __grid_constant__ PipeArgs a) {
  static_assert(RING_FZ >= 2 && RING_N >= 3 && RING_GC >= 1 && RING_R >= 1 && RING_U >= 2, "ring depths");
  __shared__ PipeSmem S;
  const int tid = threadIdx.x;
  const int nz = a.P.G.nz;
  int next = 0;
  if (tid == 0) next = atomicAdd(a.ticket, 1);
  for (;;) {
    if (tid == 0) S.ticket = next;
    __syncthreads();
    const int t = S.ticket;
    if (t >= a.total) break;
    if (tid == 0) next = atomicAdd(a.ticket, 1);  // the next ticket travels while this item runs
    const int m = t / a.per_macro;
    int r = t - m * a.per_macro;
    int stage, zz;
    if (r < a.tiles) { stage = ST_N; zz = m - 2; }
    else if ((r -= a.tiles) < a.lb_items) { stage = ST_LB; zz = m - 2 - LAG_LB; }
    else if ((r -= a.lb_items) < a.tiles) { stage = ST_K; zz = m - 2 - LAG_K; }
    else { r -= a.tiles; stage = ST_ADV; zz = m - 2 - LAG_ADV; }
    const bool valid = stage == ST_N ? (zz >= -2 && zz <= nz + 1)
                                     : stage == ST_ADV ? (zz >= 0 && zz <= nz - 1) : (zz >= -1 && zz <= nz);
    if (!valid) {
      __syncthreads();
      continue;
    }
    if (tid < 5) {  // each dependency is polled by its own thread: one L2 round trip when all are already satisfied
      int idx, cnt;
      if (pipe_dep(a, stage, zz, tid, idx, cnt))
        while (ld_acquire(a.done + idx) < cnt) __nanosleep(40);
    }
    __syncthreads();
    if (stage == ST_N) stage_N(a, S, zz, r);
    else if (stage == ST_K) stage_K(a, S, zz, r);
    else if (stage == ST_LB) stage_LB<ST>(a, zz, r);
    else stage_ADV(a, S, zz, r);
    __syncthreads();
    if (tid == 0) {
      __threadfence();
      atomicAdd(a.done + stage * (nz + 4) + zz + 2, 1);
    }
  }
}

}  // namespace acclb
