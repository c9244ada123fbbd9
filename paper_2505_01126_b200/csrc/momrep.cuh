// Moment-representation storage of the single-phase step, device side (sm_100a).  Part of the CUDA product path.
//
// the post-collision populations are "reconstructed directly from macroscopic fields, avoiding
// direct access to full distribution functions", which "significantly reduces the memory footprint ... ten recovered
// macroscopic fields".  Taken to its end the step is a closed map on those ten fields: the state is (p*, u, a) of every
// node (10 doubles, double-buffered), and one step
//   f_i(x, t+1) = f_i^eq(p*, u)(y) + (1 - omega) w_i H_i:a(y) / (2 cs4) + S_i(u, A)(y) / 2,  y = x - c_i     Eq. 6 (L85)
//   p* = sum f_i,  m = sum f_i c_i,  Pi = sum f_i c_i c_i,  u = m + A/2,  a = Eq. 7 in closed form (O5')     L88, L92
// moves 80 B read + 80 B written per node instead of 432 (A = F^b + F^g is recomputed from the force tables).  Exactly the
// oracle's two-pass step, so the results are identical to rounding.
//
// k_mr_step: a block owns a TX x TY column of nodes and marches along z.  Iteration p: every thread rebuilds the 27
// post-collision populations of its own node of SOURCE plane p (and of one node of the 1-wide rim: the neighbours of the
// tile edge) from the ten fields (fetched one plane ahead by cp.async into the thread's own slots) and puts them into
// shared memory; after a barrier it pulls its 27 incoming populations from the in-plane neighbours: the nine with
// c_z = -1 complete the moments of consumer plane p-1 (node update, 10 aligned stores), the nine with c_z = 0 and +1 start
// those of planes p and p+1 (carried in registers).
#pragma once

namespace acclb {

constexpr int MR_FIELDS = 10;  // p*, u_x, u_y, u_z, a_xx, a_yy, a_zz, a_xy, a_xz, a_yz

template <int TX, int TY>
struct MomTile {
  static constexpr int NX = TX + 2, NY = TY + 2;
  static constexpr int RIM = NX * NY - TX * TY;
  alignas(128) double stage[MR_FIELDS][TX * TY];  // the ten fields of the next source plane at the thread's own node: ten
                                                  // TMA boxes (FAST), else one cp.async per thread and field (own slots)
  double stage_rim[MR_FIELDS][RIM];     // ... and at its rim item (threads tid < RIM; cp.async: the rim wraps)
  double pop[Q][NY][NX];                // post-collision populations of the source plane, tile + rim 1
  unsigned long long sbar;              // mbarrier of the TMA staging
  double ftx[2][NX], fty[2][NY];  // sin / cos force-table entries of the tile's columns / rows incl. the rim (R20)
  double ftz[2][LZ_MAX + 2];      // ... and of the chunk's planes z0-1 .. z1 (a global load per use would wait for L2)
};

// state slab of plane z: [10][ny][nx]
template <typename T>
__device__ __forceinline__ T* mr_slab(T* s, const Grid& G, int z) {
  T* p = s + (size_t)z * MR_FIELDS * ((size_t)G.nx * (size_t)G.ny);
  asm("" : "+l"(p));
  return p;
}

// moments of the nine populations with c_z = CZ (read through f_of(i), i = 9 (CZ + 1) .. 9 (CZ + 1) + 8), added to M
template <int CZ, class F>
__device__ __forceinline__ void mr_accumulate(F f_of, Moments& M) {
#pragma unroll
  for (int j = 0; j < 9; ++j) {
    const int i = 9 * (CZ + 1) + j;
    const int cx = cx_of(i), cy = cy_of(i);
    const double f = f_of(i);
    M.p += f;
    if (cx == 1) M.m[0] += f;
    if (cx == -1) M.m[0] -= f;
    if (cy == 1) M.m[1] += f;
    if (cy == -1) M.m[1] -= f;
    if (CZ == 1) M.m[2] += f;
    if (CZ == -1) M.m[2] -= f;
    if (cx != 0) M.Pi[0] += f;
    if (cy != 0) M.Pi[1] += f;
    if (CZ != 0) M.Pi[2] += f;
    if (cx * cy == 1) M.Pi[3] += f;
    if (cx * cy == -1) M.Pi[3] -= f;
    if (cx * CZ == 1) M.Pi[4] += f;
    if (cx * CZ == -1) M.Pi[4] -= f;
    if (cy * CZ == 1) M.Pi[5] += f;
    if (cy * CZ == -1) M.Pi[5] -= f;
  }
}
__device__ __forceinline__ void mr_zero(Moments& M) {
  M.p = 0.0;
  M.m[0] = M.m[1] = M.m[2] = 0.0;
#pragma unroll
  for (int j = 0; j < 6; ++j) M.Pi[j] = 0.0;
}

// FAST: the tile shape divides the box and the tensor map exists -- the own-node fields arrive by TMA (ten TX x TY boxes per
// plane, one issuing thread), only the rim items by per-thread cp.async.
// NPT: nodes per thread (rows ty + r TY / NPT of the tile).  Two nodes per thread (two independent chains per thread, half
// the warps per block barrier) were measured and are no faster than one (7.27 vs 7.18 ms at 512^3): the limit is the
// shared-memory traffic of the rebuilt populations, not the issue rate per warp.
template <int TX, int TY, int NPT, int MINB, bool FAST>
__global__ void __launch_bounds__(TX * TY / NPT, MINB)
k_mr_step(KP P, const double* __restrict__ sin_, double* __restrict__ sout, const double* __restrict__ tabs, int lz,
          const __grid_constant__ CUtensorMap tmap_in) {
  using T = MomTile<TX, TY>;
  extern __shared__ __align__(128) unsigned char smem_lb[];
  T& S = *reinterpret_cast<T*>(smem_lb);
  constexpr int NT = TX * TY / NPT, NX = T::NX, NY = T::NY, RIM = NX * NY - TX * TY, RY = TY / NPT;
  static_assert(RIM <= NT && TY % NPT == 0, "at most one rim item per thread");
  const Grid& G = P.G;
  const int tid = threadIdx.x, tx = tid % TX, ty = tid / TX;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, z0 = blockIdx.z * lz;
  const int z1 = min(z0 + lz, G.nz);
  const int x = x0 + tx;
  const unsigned plane = (unsigned)G.nx * (unsigned)G.ny;
  // the two source positions of this thread in the NY x NX plane: its own node, and a rim item (tid < RIM)
  int rj = 0, ri = 0;
  const bool has_rim = tid < RIM;
  // warp 0: the row below the tile (j = 0, i = 1..TX), warp 1: the row above (j = NY-1), then the two columns with the
  // corners (2 NY items): every warp that has rim items runs ONE code path for them
  static_assert(TX == 32 && 2 * TX + 2 * NY == RIM, "rim items: two full warps for the rows, 2 NY lanes for the columns");
  if (has_rim) {
    if (tid < TX) { rj = 0; ri = tid + 1; }
    else if (tid < 2 * TX) { rj = NY - 1; ri = tid - TX + 1; }
    else { const int e = tid - 2 * TX; rj = e >> 1; ri = (e & 1) ? NX - 1 : 0; }
  }
  unsigned off_own[NPT];
  bool active[NPT];
#pragma unroll
  for (int r = 0; r < NPT; ++r) {
    const int y = y0 + ty + r * RY;
    off_own[r] = (unsigned)pmod(y, G.ny) * (unsigned)G.nx + (unsigned)pmod(x, G.nx);
    active[r] = x < G.nx && y < G.ny;
  }
  const unsigned off_rim = (unsigned)pmod(y0 - 1 + rj, G.ny) * (unsigned)G.nx + (unsigned)pmod(x0 - 1 + ri, G.nx);
  // body-force table entries of the tile's columns and rows, rim included
  if (P.force_type != 0) {
    if (tid < NX) { const int xx = pmod(x0 - 1 + tid, G.nx); S.ftx[0][tid] = __ldg(tabs + xx); S.ftx[1][tid] = __ldg(tabs + G.nx + xx); }
    if (tid >= 64 && tid < 64 + NY) {
      const int yy = pmod(y0 - 1 + tid - 64, G.ny);
      S.fty[0][tid - 64] = __ldg(tabs + 2 * G.nx + yy);
      S.fty[1][tid - 64] = __ldg(tabs + 2 * G.nx + G.ny + yy);
    }
    for (int t = tid; t < (z1 - z0) + 2; t += NT) {
      const int zz = pmod(z0 - 1 + t, G.nz);
      S.ftz[0][t] = __ldg(tabs + 2 * (G.nx + G.ny) + zz);
      S.ftz[1][t] = __ldg(tabs + 2 * (G.nx + G.ny) + G.nz + zz);
    }
  }
  auto fetch = [&](int p) {  // the ten fields of source plane p (any integer) into this thread's own slots
    const double* sl = mr_slab(sin_, G, pmod(p, G.nz));
#pragma unroll
    for (int k = 0; k < MR_FIELDS; ++k) {
      if (!FAST) {
#pragma unroll
        for (int r = 0; r < NPT; ++r) cp_async_f64(&S.stage[k][r * NT + tid], sl + (unsigned)k * plane + off_own[r]);
      }
      if (has_rim) cp_async_f64(&S.stage_rim[k][tid], sl + (unsigned)k * plane + off_rim);
    }
    cp_async_commit();
  };
  auto tma_fetch = [&](int p) {  // FAST: the ten own-node boxes of source plane p, by one thread, after a block barrier
    if (tid == NT / 2) {
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      mbar_arrive_expect_tx(&S.sbar, (unsigned)(MR_FIELDS * TX * TY * sizeof(double)));
      const int slab0 = pmod(p, G.nz) * MR_FIELDS;
#pragma unroll
      for (int k = 0; k < MR_FIELDS; ++k) tma_load_box(&S.stage[k][0], &tmap_in, x0, y0, slab0 + k, &S.sbar);
    }
  };
  if (FAST && tid == 0) {
    mbar_init(&S.sbar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  // acceleration A = F^b + F^g of a node of the plane (single component: rho == 1), R20 / R31
  auto accel = [&](int j, int i, int zl, double (&A)[3]) {  // zl = plane - (z0 - 1)
    A[0] = A[1] = A[2] = 0.0;
    if (P.force_type != 0) {
      const double fsz = S.ftz[0][zl], fcz = S.ftz[1][zl];
      const double fsx = S.ftx[0][i], fcx = S.ftx[1][i], fsy = S.fty[0][j], fcy = S.fty[1][j];
      if (P.force_type == 1) { A[0] = P.force_amp * (fsz + fcy); A[1] = P.force_amp * (fsx + fcz); A[2] = P.force_amp * (fsy + fcx); }
      else { A[0] = P.force_amp * fsy; A[1] = P.force_amp * fsz; A[2] = P.force_amp * fsx; }
    }
    if (P.buoyant) {
      const double dr = 1.0 - P.rho_ref;
      A[0] += dr * P.grav[0]; A[1] += dr * P.grav[1]; A[2] += dr * P.grav[2];
    }
  };
  // Eq. 6 at a source node: the 27 post-collision populations from (p*, u, a) and A, into the shared plane
  auto rebuild = [&](int slot, int j, int i, int zl) {  // slot = r (own node of row r) or -1 (rim item)
    double c[MR_FIELDS];
#pragma unroll
    for (int k = 0; k < MR_FIELDS; ++k) c[k] = slot < 0 ? S.stage_rim[k][tid] : S.stage[k][slot * NT + tid];
    double A[3];
    accel(j, i, zl, A);
    const double u[3] = {c[1], c[2], c[3]};
    const double U[3] = {u[0] + 0.5 * A[0], u[1] + 0.5 * A[1], u[2] + 0.5 * A[2]};
    double Tt[6];
    Tt[0] = u[0] * u[0] + P.one_m_omega * c[4] + u[0] * A[0];
    Tt[1] = u[1] * u[1] + P.one_m_omega * c[5] + u[1] * A[1];
    Tt[2] = u[2] * u[2] + P.one_m_omega * c[6] + u[2] * A[2];
    Tt[3] = u[0] * u[1] + P.one_m_omega * c[7] + 0.5 * (u[0] * A[1] + u[1] * A[0]);
    Tt[4] = u[0] * u[2] + P.one_m_omega * c[8] + 0.5 * (u[0] * A[2] + u[2] * A[0]);
    Tt[5] = u[1] * u[2] + P.one_m_omega * c[9] + 0.5 * (u[1] * A[2] + u[2] * A[1]);
    if (slot >= 0) {
      double f[Q];
      hermite2_populations(c[0], U, Tt, f);
#pragma unroll
      for (int q = 0; q < Q; ++q) S.pop[q][j][i] = f[q];
    } else {
      // a rim node only feeds the tile: the nine populations that point into it -- c_y = s (s = +1 from the row below the
      // tile, -1 from the row above) or c_x = s (columns left / right; a corner's three are among its column's nine).
      // One instruction sequence per kind, the side entering as the sign s.
      const double e0 = c[0] - 1.5 * (Tt[0] + Tt[1] + Tt[2]);
      const bool row = tid < 2 * TX;
      const double sgn = row ? (j == 0 ? 1.0 : -1.0) : (i == 0 ? 1.0 : -1.0);
      // fixed direction f (y for a row item, x for a column item), free in-plane direction g, and z
      const double Tf = row ? Tt[1] : Tt[0], Tg = row ? Tt[0] : Tt[1];
      const double Tfg = sgn * Tt[3], Tfz = sgn * (row ? Tt[5] : Tt[4]), Tgz = row ? Tt[4] : Tt[5];
      const double Uf = sgn * (row ? U[1] : U[0]), Ug = row ? U[0] : U[1];
      const int qf = (sgn > 0.0 ? 2 : 0) * (row ? 3 : 1), qg = row ? 1 : 3;  // population index = qf + (cg + 1) qg + 9 (cz + 1)
      double* dst = &S.pop[0][j][i] + (size_t)qf * (NY * NX);
#pragma unroll
      for (int cz = -1; cz <= 1; ++cz)
#pragma unroll
        for (int cg = -1; cg <= 1; ++cg) {
          const int nnz = 1 + (cg != 0) + (cz != 0);
          const double w = nnz == 1 ? 2.0 / 27.0 : nnz == 2 ? 1.0 / 54.0 : 1.0 / 216.0;
          double cct = Tf, cross = 0.0, cu = Uf;
          if (cg != 0) cct += Tg;
          if (cz != 0) cct += Tt[2];
          if (cg == 1) { cross += Tfg; cu += Ug; }
          if (cg == -1) { cross -= Tfg; cu -= Ug; }
          if (cz == 1) { cross += Tfz; cu += U[2]; }
          if (cz == -1) { cross -= Tfz; cu -= U[2]; }
          if (cg * cz == 1) cross += Tgz;
          if (cg * cz == -1) cross -= Tgz;
          cct += 2.0 * cross;
          dst[(size_t)((cg + 1) * qg + 9 * (cz + 1)) * (NY * NX)] = w * (e0 + 4.5 * cct) + (3.0 * w) * cu;
        }
    }
  };
  __syncthreads();
  fetch(z0 - 1);
  if (FAST) tma_fetch(z0 - 1);
  Moments Mo[NPT], Mm[NPT];  // moments of consumer planes p-1 (two of three source planes in) and p (one in)
#pragma unroll
  for (int r = 0; r < NPT; ++r) { mr_zero(Mo[r]); mr_zero(Mm[r]); }
  for (int p = z0 - 1; p <= z1; ++p) {
    cp_async_wait_all();
    if (FAST) mbar_wait(&S.sbar, (unsigned)(p - (z0 - 1)) & 1u);
#pragma unroll
    for (int r = 0; r < NPT; ++r) rebuild(r, ty + r * RY + 1, tx + 1, p - (z0 - 1));
    if (has_rim) rebuild(-1, rj, ri, p - (z0 - 1));
    if (p < z1) fetch(p + 1);  // own slots: free as soon as this thread has read them
    __syncthreads();
    if (FAST && p < z1) tma_fetch(p + 1);  // every thread has read its fields of plane p (barrier above)
    const int z = p - 1;
#pragma unroll
    for (int r = 0; r < NPT; ++r) {
      const int jy = ty + r * RY + 1;
      auto pulled = [&](int i) { return S.pop[i][jy - cy_of(i)][tx + 1 - cx_of(i)]; };
      // c_z = -1: source plane p feeds consumer plane p - 1 = its third and last contribution -> node update
      mr_accumulate<-1>(pulled, Mo[r]);
      if (z >= z0 && z < z1 && active[r]) {
        double A[3];
        accel(jy, tx + 1, z - (z0 - 1), A);
        const double u[3] = {Mo[r].m[0] + 0.5 * A[0], Mo[r].m[1] + 0.5 * A[1], Mo[r].m[2] + 0.5 * A[2]};  // a5 (R4)
        double a[6];
        hermite_coeff(Mo[r], u, A, a);                                                                    // a6, Eq. 7 (O5')
        double* o = mr_slab(sout, G, z) + off_own[r];
        __stcs(o, Mo[r].p);
        __stcs(o + plane, u[0]);
        __stcs(o + 2u * plane, u[1]);
        __stcs(o + 3u * plane, u[2]);
#pragma unroll
        for (int k = 0; k < 6; ++k) __stcs(o + (unsigned)(4 + k) * plane, a[k]);
      }
      Mo[r] = Mm[r];
      mr_accumulate<0>(pulled, Mo[r]);   // consumer plane p: second contribution
      mr_zero(Mm[r]);
      mr_accumulate<1>(pulled, Mm[r]);   // consumer plane p + 1: first contribution
    }
    __syncthreads();                // the shared plane is rebuilt in the next iteration
  }
}

// Initial state (R15): f = f^eq(p*, u0) - S/2 has p* = p*, u = m + A/2 = u0 and a = 0 (its non-equilibrium part is -S/2, which
// Eq. 7 cancels), so the ten fields are (p*, u0, 0).
__global__ void __launch_bounds__(256) k_mr_init(Grid G, const double* __restrict__ rho_in, const double* __restrict__ u_in,
                                                 double* __restrict__ state) {
  const unsigned k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= G.n) return;
  const unsigned plane = (unsigned)G.nx * (unsigned)G.ny;
  const unsigned z = k / plane, o = k - z * plane;
  double* s = mr_slab(state, G, (int)z) + o;
  s[0] = rho_in[k];
  s[plane] = u_in[k];
  s[2u * plane] = u_in[(size_t)G.n + k];
  s[3u * plane] = u_in[2 * (size_t)G.n + k];
#pragma unroll
  for (int j = 4; j < MR_FIELDS; ++j) s[(unsigned)j * plane] = 0.0;
}

// a9: p*, u of the current state (a copy: they are stored)
__global__ void __launch_bounds__(256) k_mr_moments(Grid G, const double* __restrict__ state, double* __restrict__ rho_out,
                                                    double* __restrict__ u_out) {
  const unsigned k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= G.n) return;
  const unsigned plane = (unsigned)G.nx * (unsigned)G.ny;
  const unsigned z = k / plane, o = k - z * plane;
  const double* s = mr_slab(state, G, (int)z) + o;
  if (rho_out) rho_out[k] = s[0];
  if (u_out) {
    u_out[k] = s[plane];
    u_out[(size_t)G.n + k] = s[2u * plane];
    u_out[2 * (size_t)G.n + k] = s[3u * plane];
  }
}

// a9: diagnostics (R21) from the stored fields: KE, dissipation from a, sum p*, sum m (m = u - A/2), max |u|
__global__ void __launch_bounds__(256) k_mr_diag(KP P, const double* __restrict__ state, const double* __restrict__ tabs,
                                                 double* __restrict__ acc) {
  const Grid& G = P.G;
  const unsigned plane = (unsigned)G.nx * (unsigned)G.ny;
  double s[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  for (unsigned k = blockIdx.x * blockDim.x + threadIdx.x; k < G.n; k += gridDim.x * blockDim.x) {
    const unsigned z = k / plane, o = k - z * plane;
    const int y = (int)(o / (unsigned)G.nx), x = (int)(o - (unsigned)y * (unsigned)G.nx);
    const double* c = mr_slab(state, G, (int)z) + o;
    const double u[3] = {c[plane], c[2u * plane], c[3u * plane]};
    double Fb[3];
    body_force(P, tabs, x, y, (int)z, Fb);
    if (P.buoyant) {
      const double dr = 1.0 - P.rho_ref;
      Fb[0] += dr * P.grav[0]; Fb[1] += dr * P.grav[1]; Fb[2] += dr * P.grav[2];
    }
    const double uu = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
    double aa = 0.0;
#pragma unroll
    for (int j = 0; j < 6; ++j) {
      const double a = c[(unsigned)(4 + j) * plane];
      aa += (j < 3 ? 1.0 : 2.0) * a * a;
    }
    s[0] += 0.5 * uu;
    s[1] += P.eps_pref * aa;
    s[3] += c[0];
    s[4] += u[0] - 0.5 * Fb[0];
    s[5] += u[1] - 0.5 * Fb[1];
    s[6] += u[2] - 0.5 * Fb[2];
    s[7] = fmax(s[7], sqrt(uu));
  }
  __shared__ double sh[8][8];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    double v = s[j];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const double w = __shfl_xor_sync(0xffffffffu, v, o);
      v = j < 7 ? v + w : fmax(v, w);
    }
    if (lane == 0) sh[j][wid] = v;
  }
  __syncthreads();
  if (threadIdx.x < 8) {
    const int j = threadIdx.x;
    double r = sh[j][0];
    for (int w = 1; w < 8; ++w) r = j < 7 ? r + sh[j][w] : fmax(r, sh[j][w]);
    if (j < 7) atomicAdd(acc + j, r);
    else atomicMax(reinterpret_cast<unsigned long long*>(acc + 7), (unsigned long long)__double_as_longlong(r));
  }
}

}  // namespace acclb
