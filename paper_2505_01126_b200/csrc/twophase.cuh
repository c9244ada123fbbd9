// Two-phase hot path on shared-memory tiles, device side (sm_100a).  Part of the CUDA product path.
//
// One two-phase step is two kernels:
//   k_lb_tp     rows a1-a7 + the phi-only part of a8.  A block owns a TX x TY column of nodes and marches along z.
//               Per plane it stages phi (halo 2) in shared memory, derives the interface normal n, the sharpening flux
//               q = phi (1 - phi) n and |grad phi| ONCE per node of the tile + 1 rim (they are needed at the 26
//               neighbours by div n and div q), then every thread does its node: kappa_c = div n,
//               F^s, F^p, F^nu (Eq. 8), pull-stream, moments, Hermite coefficient, regularized reconstruction, aligned
//               store (Eqs. 6-7), and writes u (needed by the advection) and r = D lap phi - kappa div q (Eq. 3).
//   k_advect    the advective part of a8: phi+ = phi + (-sum_e (Phi_e(x) - Phi_e(x - e)) + r), Phi = u_f WENO5(phi) in
//               flux form (R12).  Every face flux is computed once per face (shared memory for x / y
//               faces, a register carried along the z march for z faces), so sum phi is conserved to rounding.
// Periodic boundaries are index wraps when the tiles are filled (PAPER.md:L114's halo exchange is not needed).
#pragma once

namespace acclb {

__device__ __forceinline__ int pmod(int a, int n) {
  int r = a % n;
  return r < 0 ? r + n : r;
}

// (2/cs2) sum_i w_i (Psi(x + c_i) - Psi(x)) through an accessor val(dz, dy, dx); PAPER.md:L104 as repaired by R7.
template <class V>
__device__ __forceinline__ double lattice_laplacian(V val) {
  double acc = 0.0;
#pragma unroll
  for (int a = -1; a <= 1; ++a)
#pragma unroll
    for (int b = -1; b <= 1; ++b) {
      const double row = val(a, b, -1) + 4.0 * val(a, b, 0) + val(a, b, 1);
      acc = fma((a == 0 ? 4.0 : 1.0) * (b == 0 ? 4.0 : 1.0), row, acc);
    }
  return 6.0 * (acc * (1.0 / 216.0) - val(0, 0, 0));
}

template <int TX, int TY>
struct GeoTile {
  static constexpr int PX = TX + 4, PY = TY + 4;  // phi plane with halo 2
  static constexpr int NX = TX + 2, NY = TY + 2;  // derived-field plane with halo 1
  static constexpr int NF = 7;                    // n_x n_y n_z q_x q_y q_z |grad phi|
  double phi[5][PY][PX];                          // ring over z: plane zz lives in slot (zz - z0 + 2) % 5
  double fld[3][NF][NY][NX];                      // ring over z: plane zz lives in slot (zz - z0 + 1) % 3
};

// Fused two-phase LB kernel (see the header of this file).  lz = planes per block along z.
template <typename ST, int TX, int TY, int MINB>
__global__ void __launch_bounds__(TX * TY, MINB)
k_lb_tp(KP P, const ST* __restrict__ fin, ST* __restrict__ fout, const double* __restrict__ phi,
        double* __restrict__ uout, double* __restrict__ rout, const double* __restrict__ tabs, int lz) {
  using T = GeoTile<TX, TY>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T& S = *reinterpret_cast<T*>(smem_raw);
  constexpr int NT = TX * TY;
  const Grid& G = P.G;
  const int tid = threadIdx.x, tx = tid % TX, ty = tid / TX;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, z0 = blockIdx.z * lz;
  const int z1 = min(z0 + lz, G.nz);
  const int x = x0 + tx, y = y0 + ty;
  const bool active = x < G.nx && y < G.ny;
  const unsigned plane = (unsigned)G.nx * (unsigned)G.ny;

  // phi tile elements this thread stages per plane: element e = tid + l NT of the PY x PX tile
  constexpr int NPHI = T::PX * T::PY, LP = (NPHI + NT - 1) / NT;
  unsigned poff[LP];
#pragma unroll
  for (int l = 0; l < LP; ++l) {
    const int e = tid + l * NT;
    const int j = e / T::PX, i = e % T::PX;
    poff[l] = (unsigned)pmod(y0 - 2 + j, G.ny) * (unsigned)G.nx + (unsigned)pmod(x0 - 2 + i, G.nx);
  }
  auto stage_phi = [&](int zz) {  // plane zz (unwrapped) -> ring slot
    const double* src = phi + (size_t)pmod(zz, G.nz) * plane;
    double* dst = &S.phi[(zz - z0 + 2) % 5][0][0];
#pragma unroll
    for (int l = 0; l < LP; ++l) {
      const int e = tid + l * NT;
      if (e < NPHI) dst[e] = __ldg(src + poff[l]);
    }
  };
  // n = g / (|g| + 1e-12) (R17), q = phi (1 - phi) n (Eq. 3), |g|, on the tile + 1 rim of plane zz
  auto derive = [&](int zz) {
    const int sp = (zz - z0 + 2) % 5, sm = (zz - z0 + 1) % 5, sq = (zz - z0 + 3) % 5;
    const int so = (zz - z0 + 1) % 3;
    constexpr int NN = T::NX * T::NY;
    for (int e = tid; e < NN; e += NT) {
      const int j = e / T::NX, i = e % T::NX;
      auto val = [&](int dz, int dy, int dx) {
        return S.phi[dz < 0 ? sm : (dz > 0 ? sq : sp)][j + 1 + dy][i + 1 + dx];
      };
      const double gx = lattice_derivative<0>(val), gy = lattice_derivative<1>(val), gz = lattice_derivative<2>(val);
      const double gn = sqrt(gx * gx + gy * gy + gz * gz);
      const double inv = 1.0 / (gn + 1e-12);
      const double ph = val(0, 0, 0), pq = ph * (1.0 - ph);
      const double nx_ = gx * inv, ny_ = gy * inv, nz_ = gz * inv;
      S.fld[so][0][j][i] = nx_;
      S.fld[so][1][j][i] = ny_;
      S.fld[so][2][j][i] = nz_;
      S.fld[so][3][j][i] = pq * nx_;
      S.fld[so][4][j][i] = pq * ny_;
      S.fld[so][5][j][i] = pq * nz_;
      S.fld[so][6][j][i] = gn;
    }
  };

  // prologue: phi planes z0-2 .. z0+1, derived planes z0-1, z0
  stage_phi(z0 - 2);
  stage_phi(z0 - 1);
  stage_phi(z0);
  stage_phi(z0 + 1);
  __syncthreads();
  derive(z0 - 1);
  derive(z0);

  const int xs[3] = {wrap_dec(x < G.nx ? x : 0, G.nx), x < G.nx ? x : 0, wrap_inc(x < G.nx ? x : 0, G.nx)};
  const int yy = y < G.ny ? y : 0;
  const unsigned yrow[3] = {(unsigned)wrap_dec(yy, G.ny) * (unsigned)G.nx, (unsigned)yy * (unsigned)G.nx,
                            (unsigned)wrap_inc(yy, G.ny) * (unsigned)G.nx};

  for (int z = z0; z < z1; ++z) {
    stage_phi(z + 2);
    __syncthreads();
    derive(z + 1);
    __syncthreads();
    if (!active) continue;  // barriers above are executed by every thread: the loop bounds are block-uniform

    const int fm = (z - z0) % 3, f0 = (z - z0 + 1) % 3, fp = (z - z0 + 2) % 3;
    auto fld = [&](int c, int dz, int dy, int dx) {
      return S.fld[dz < 0 ? fm : (dz > 0 ? fp : f0)][c][ty + 1 + dy][tx + 1 + dx];
    };
    const int pm = (z - z0 + 1) % 5, p0 = (z - z0 + 2) % 5, pp = (z - z0 + 3) % 5;
    auto ph = [&](int dz, int dy, int dx) { return S.phi[dz < 0 ? pm : (dz > 0 ? pp : p0)][ty + 2 + dy][tx + 2 + dx]; };

    // a3: kappa_c = div n, div q, lap phi by the lattice stencils
    const double kc = lattice_derivative<0>([&](int dz, int dy, int dx) { return fld(0, dz, dy, dx); }) +
                      lattice_derivative<1>([&](int dz, int dy, int dx) { return fld(1, dz, dy, dx); }) +
                      lattice_derivative<2>([&](int dz, int dy, int dx) { return fld(2, dz, dy, dx); });
    const double divq = lattice_derivative<0>([&](int dz, int dy, int dx) { return fld(3, dz, dy, dx); }) +
                        lattice_derivative<1>([&](int dz, int dy, int dx) { return fld(4, dz, dy, dx); }) +
                        lattice_derivative<2>([&](int dz, int dy, int dx) { return fld(5, dz, dy, dx); });
    const double lap = lattice_laplacian(ph);
    const double gn = fld(6, 0, 0, 0);
    const double gs = gn + 1e-12;  // g = n (|g| + 1e-12) up to rounding
    const double g[3] = {fld(0, 0, 0, 0) * gs, fld(1, 0, 0, 0) * gs, fld(2, 0, 0, 0) * gs};
    const double phi0 = ph(0, 0, 0);

    const unsigned k = (unsigned)z * plane + yrow[1] + (unsigned)xs[1];
    rout[k] = P.D * lap - P.kappa * divq;  // phi-only part of Eq. 3

    // a1: pull-stream
    Nbr nb;
    nb.x[0] = xs[0]; nb.x[1] = xs[1]; nb.x[2] = xs[2];
    {
      const unsigned zr[3] = {(unsigned)wrap_dec(z, G.nz) * plane, (unsigned)z * plane, (unsigned)wrap_inc(z, G.nz) * plane};
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) nb.row[a][b] = zr[a] + yrow[b];
    }
    double f[Q];
    pull27<ST>(fin, G, nb, f);
    Moments M;
    moments_of(f, M);
    double Fb[3], A[3], rho;
    body_force(P, tabs, x, y, z, Fb);
    accel_from_geometry(P, M, g, gn, kc, phi0, Fb, true, A, rho);
    const double u[3] = {M.m[0] + 0.5 * A[0], M.m[1] + 0.5 * A[1], M.m[2] + 0.5 * A[2]};  // a5, PAPER.md:L88 (R4)
    uout[k] = u[0];
    uout[G.n + k] = u[1];
    uout[2u * G.n + k] = u[2];
    collide_store<ST>(P, M, u, A, f, fout, k);
  }
}

// ---------------------------------------------------------------------------------------------------- advection
template <int TX, int TY>
struct AdvTile {
  double phi[TY + 6][TX + 6];  // plane z with halo 3 along x and y (corners unused)
  double ux[TY][TX + 2];       // u_x with halo 1 along x
  double uy[TY + 2][TX];       // u_y with halo 1 along y
  double fx[TY][TX + 1];       // flux through the x face between tile columns i-1 and i
  double fy[TY + 1][TX];       // flux through the y face between tile rows j-1 and j
};

template <int TX, int TY>
__global__ void __launch_bounds__(TX * TY)
k_advect(KP P, const double* __restrict__ phi, const double* __restrict__ u, const double* __restrict__ r,
         double* __restrict__ phi_new, int lz) {
  using T = AdvTile<TX, TY>;
  __shared__ T S2[2];  // ping-pong over z so that two barriers per plane suffice
  constexpr int NT = TX * TY;
  static_assert(6 * (TX + TY) <= NT && 2 * (TX + TY) <= NT, "one halo element per thread");
  const Grid& G = P.G;
  const int tid = threadIdx.x, tx = tid % TX, ty = tid / TX;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, z0 = blockIdx.z * lz;
  const int z1 = min(z0 + lz, G.nz);
  const int x = x0 + tx, y = y0 + ty;
  const bool active = x < G.nx && y < G.ny;
  const unsigned plane = (unsigned)G.nx * (unsigned)G.ny;
  const unsigned n = G.n;
  const unsigned own = (unsigned)pmod(y, G.ny) * (unsigned)G.nx + (unsigned)pmod(x, G.nx);

  // phi halo element of this thread (tid < 6 (TX + TY)): rows above/below first, then columns left/right
  int hj = -1, hi = -1;
  unsigned hoff = 0;
  if (tid < 6 * TX) {
    const int rr = tid / TX;  // 0..5 -> tile rows -3,-2,-1, TY, TY+1, TY+2
    hj = rr < 3 ? rr : TY + rr;
    hi = 3 + tid % TX;
  } else if (tid < 6 * (TX + TY)) {
    const int e = tid - 6 * TX, cc = e % 6;  // 0..5 -> tile columns -3,-2,-1, TX, TX+1, TX+2
    hj = 3 + e / 6;
    hi = cc < 3 ? cc : TX + cc;
  }
  if (hj >= 0) hoff = (unsigned)pmod(y0 - 3 + hj, G.ny) * (unsigned)G.nx + (unsigned)pmod(x0 - 3 + hi, G.nx);
  // velocity halo element (tid < 2 (TX + TY)): u_y rows -1, TY ; u_x columns -1, TX
  int vkind = 0, vj = 0, vi = 0;  // 1: uy, 2: ux
  unsigned voff = 0;
  if (tid < 2 * TX) {
    vkind = 1;
    vj = tid < TX ? 0 : TY + 1;
    vi = tid % TX;
    voff = n + (unsigned)pmod(y0 - 1 + vj, G.ny) * (unsigned)G.nx + (unsigned)pmod(x0 + vi, G.nx);
  } else if (tid < 2 * (TX + TY)) {
    const int e = tid - 2 * TX;
    vkind = 2;
    vj = e / 2;
    vi = (e & 1) ? TX + 1 : 0;
    voff = (unsigned)pmod(y0 + vj, G.ny) * (unsigned)G.nx + (unsigned)pmod(x0 - 1 + vi, G.nx);
  }

  auto zoff = [&](int zz) { return (size_t)pmod(zz, G.nz) * plane; };
  // column window w[j] = phi(z - 2 + j), j = 0..5, of the z face between z and z + 1
  double w0 = __ldg(phi + zoff(z0 - 3) + own), w1 = __ldg(phi + zoff(z0 - 2) + own), w2 = __ldg(phi + zoff(z0 - 1) + own);
  double w3 = __ldg(phi + zoff(z0) + own), w4 = __ldg(phi + zoff(z0 + 1) + own), w5 = __ldg(phi + zoff(z0 + 2) + own);
  double uz0 = __ldg(u + 2u * n + zoff(z0 - 1) + own), uz1 = __ldg(u + 2u * n + zoff(z0) + own);
  double fz_prev = face_flux(uz0, uz1, w0, w1, w2, w3, w4, w5);  // face (z0 - 1, z0)

  for (int z = z0; z < z1; ++z) {
    T& S = S2[(z - z0) & 1];
    const size_t zo = zoff(z);
    w0 = w1; w1 = w2; w2 = w3; w3 = w4; w4 = w5;
    w5 = __ldg(phi + zoff(z + 3) + own);
    uz0 = uz1;
    uz1 = __ldg(u + 2u * n + zoff(z + 1) + own);
    S.phi[ty + 3][tx + 3] = w2;
    S.ux[ty][tx + 1] = __ldg(u + zo + own);
    S.uy[ty + 1][tx] = __ldg(u + n + zo + own);
    if (hj >= 0) S.phi[hj][hi] = __ldg(phi + zo + hoff);
    if (vkind == 1) S.uy[vj][vi] = __ldg(u + zo + voff);
    else if (vkind == 2) S.ux[vj][vi] = __ldg(u + zo + voff);
    const double rr = active ? __ldg(r + zo + own) : 0.0;
    __syncthreads();
    for (int e = tid; e < TY * (TX + 1); e += NT) {  // x faces
      const int j = e / (TX + 1), i = e % (TX + 1);
      const double* p = &S.phi[j + 3][i];  // p[0..5] = phi at tile columns i-3 .. i+2 = L-2 .. L+3 with L = i-1
      S.fx[j][i] = face_flux(S.ux[j][i], S.ux[j][i + 1], p[0], p[1], p[2], p[3], p[4], p[5]);
    }
    for (int e = tid; e < (TY + 1) * TX; e += NT) {  // y faces
      const int j = e / TX, i = e % TX;
      S.fy[j][i] = face_flux(S.uy[j][i], S.uy[j + 1][i], S.phi[j][i + 3], S.phi[j + 1][i + 3], S.phi[j + 2][i + 3],
                             S.phi[j + 3][i + 3], S.phi[j + 4][i + 3], S.phi[j + 5][i + 3]);
    }
    const double fz = face_flux(uz0, uz1, w0, w1, w2, w3, w4, w5);  // face (z, z + 1)
    __syncthreads();
    if (active) {
      double adv = 0.0;
      adv += S.fx[ty][tx + 1] - S.fx[ty][tx];
      adv += S.fy[ty + 1][tx] - S.fy[ty][tx];
      adv += fz - fz_prev;
      phi_new[zo + own] = w2 + (-adv + rr);
    }
    fz_prev = fz;
  }
}

}  // namespace acclb
