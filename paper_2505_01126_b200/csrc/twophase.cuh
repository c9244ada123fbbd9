// Two-phase hot path on shared-memory tiles, device side (sm_100a).  Part of the CUDA product path.
//
// One two-phase step is the tiled kernel k_lb_tp<MODE_FUSED> plus the small seam kernel k_seam:
//   k_lb_tp     rows a1-a8.  A block owns a TX x TY column of nodes and marches along z.
//               Per plane it stages phi (halo 2) in shared memory, derives the interface normal n, the sharpening flux
//               q = phi (1 - phi) n and |grad phi| ONCE per node of the tile + 1 rim (they are needed at the 26
//               neighbours by div n and div q), then every thread does its node: kappa_c = div n,
//               F^s, F^p, F^nu, F^g (Eq. 8, R31), pull-stream, moments, Hermite coefficient, regularized reconstruction,
//               aligned store (Eqs. 6-7), u and r = D lap phi - kappa div q (Eq. 3).
//               MODE_FUSED: u and r never leave the SM.  One plane behind the node update the block evaluates the
//               advective WENO5 fluxes Phi_e = u_f WENO5(phi) (R12) through every face INSIDE its tile
//               column (x faces: neighbour lane; y faces: shared memory; z faces: carried along the march) and writes
//               phi(t+1) = phi + r - sum_e (Phi_e(x) - Phi_e(x - e)) without the faces on the tile's seams, whose second
//               velocity belongs to another block; the velocities on the seams go to three thin strips (2.75 B per node).
//               The other modes reuse the march and the geometry: MODE_UNFUSED (u, r to HBM for k_advect: variant 1 and
//               the SSP-RK3 stages), MODE_MOMENTS, MODE_DIAG, MODE_INIT (accLB_moments / diagnostics / init).
//   k_seam      adds the fluxes through the seam faces (x = multiples of TX, y = multiples of TY, z = multiples of lz:
//               5 % of all faces) to the cells on either side, from the strips and phi(t): one thread per face, one
//               flux per face, added to one cell and subtracted from the other (atomics): sum phi is conserved to
//               rounding (R12).
//   k_advect    the advective part of a8 as a kernel of its own (after k_lb_tp<MODE_UNFUSED>):
//               phi+ = a base + b (phi + (-sum_e (Phi_e(x) - Phi_e(x - e)) + r)); every face flux is computed once per face
//               (shared memory for x / y faces, a register carried along z for z faces).
// Periodic boundaries are index wraps when the tiles are filled (PAPER.md:L114's halo exchange is not needed).
// Staging: FAST instances (tile-divisible boxes, fp64 storage): the 27 pulled populations of the next plane arrive by TMA
// (27 tiled cp.async.bulk.tensor box loads, mbarrier completion; tiles on the periodic y rim row by row); otherwise one
// cp.async per thread and population.  phi planes arrive by 16-byte cp.async one plane ahead.
#pragma once

#include <type_traits>

namespace acclb {

constexpr int LZ_MAX = 64;  // planes per block along z, at most (128 and 256 were measured: no difference)

__device__ __forceinline__ int pmod(int a, int n) {
  int r = a % n;
  return r < 0 ? r + n : r;
}

// cp.async (LDGSTS) of one population from global memory into the issuing thread's own shared-memory slot.  Default L2
// policy on purpose: with an evict-first hint the 32-byte sectors that the x-shifted pulls of two neighbouring tiles share
// were evicted between the two reads (ncu: 36.0 GB read per 512^3 step with the hint, 30.9 GB without; ideal 30.1 GB).
template <int BYTES>
__device__ __forceinline__ void cp_async_pop(void* smem, const void* gmem) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(sa), "l"(gmem), "n"(BYTES) : "memory");
}
// mbarrier + TMA (tiled bulk tensor copy) primitives for the population pull of interior tiles.
__device__ __forceinline__ void mbar_init(unsigned long long* b, int count) {
  asm volatile("mbarrier.init.shared.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long* b, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared.b64 _, [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(b)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* b, unsigned parity) {
  const unsigned a = (unsigned)__cvta_generic_to_shared(b);
  unsigned done;
  do {
    asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
                 : "=r"(done) : "r"(a), "r"(parity) : "memory");
  } while (!done);
}
// One TX x TY x 1 box of a rank-3 tensor (x, y, slab = z * 27 + i) -> shared memory, completion in bytes on the mbarrier.
__device__ __forceinline__ void tma_load_box(void* smem, const void* tmap, int cx, int cy, int cs, unsigned long long* b) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
                   (unsigned)__cvta_generic_to_shared(smem)),
               "l"(tmap), "r"(cx), "r"(cy), "r"(cs), "r"((unsigned)__cvta_generic_to_shared(b))
               : "memory");
}

__device__ __forceinline__ void cp_async_f64(double* smem, const double* gmem) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sa), "l"(gmem) : "memory");
}
// 16 bytes, L2 only (no L1 line is allocated): the staging copies of this file.  With 2 x 100 KB of shared memory per SM the
// L1 is down to 28 KB, and 8-byte cp.async.ca copies that each allocate a 128-byte L1 line (a phi plane's halo columns,
// the edge elements of the pull) thrashed it: 10.9 -> 12.1 ms for 10 KB more shared memory per block (measured).
__device__ __forceinline__ void cp_async_16(void* smem, const void* gmem) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gmem) : "memory");
}
template <int N>
__device__ __forceinline__ void cp_async_wait_but() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// Shared-memory working set of k_lb_tp for one TX x TY column marching along z.
//   The D3Q27 stencil weights factorise, w_i = W(cx) W(cy) W(cz) / 216 with W = (1,4,1), so every lattice stencil of
//   PAPER.md:L104 is evaluated separably: a z combination per (x,y) column first (Sz = (1,4,1), Dz = (+1,0,-1)), then a
//   3 x 3 stencil in the plane.  Same numbers as the 27-term sums up to rounding order.
template <typename ST, int TX, int TY, bool FUSED, bool POP = true>
struct GeoTile {
  // Landing zone of the pulled populations of the next plane.  For interior tiles the TMA writes population i's TX x TY box
  // of rows y0 - c_iy, plane z - c_iz, UNSHIFTED in x (TMA needs 16-byte aligned box starts, and a window widened to the next
  // aligned element costs a 64-byte DRAM fetch per row: measured +4.8 GB per 512^3 step), so thread tx reads element
  // tx - c_ix of its row; the one element per row that lies outside the box (x0 - 1 for c_ix = +1, x0 + TX for c_ix = -1)
  // is fetched by lanes of the row's warp as aligned 16-byte chunks (cp.async) into the tail of the slab.
  // The three populations i = 3 m, 3 m + 1, 3 m + 2 (c_ix = -1, 0, +1; same c_iy, c_iz) are consecutive planes of the
  // [z][i][y][x] layout with the same box origin: ONE TMA box TX x TY x 3 fetches them (9 instead of 27 issues per plane).
  // One slab per triple: the three boxes back to back, then the TY edge chunks of population 3 m, then those of 3 m + 2.
  static constexpr int TAILE = 16 / (int)sizeof(ST) * TY;   // elements of one population's edge chunks
  static constexpr int TRIPLE = 3 * TX * TY + 2 * TAILE;
  static_assert(!POP || (TRIPLE * sizeof(ST)) % 128 == 0, "TMA destinations are 128-byte aligned");
  __host__ __device__ static constexpr int pop_off(int i) { return (i / 3) * TRIPLE + (i % 3) * (TX * TY); }  // box of population i in fpop
  alignas(128) ST fpop[POP ? (Q / 3) * TRIPLE : 16];  // (no landing zone for a kernel mode that pulls no populations)
  unsigned long long fbar;  // mbarrier of the TMA pull
  static constexpr int PX = TX + 4, PY = TY + 4;  // phi planes: tile + halo 2
  static constexpr int NX = TX + 2, NY = TY + 2;  // n, q planes: tile + halo 1
  static constexpr int NR = 5;  // (five also without the fused advection: phi(z) is read after the last barrier of an iteration,
                                // so the slot of plane zc-2 must not be the landing slot of the next iteration's fetch)
  alignas(16) double raw[NR][PY][PX];  // ring of raw phi planes (zc-2,) zc-1, zc, zc+1 and zc+2 (landing, cp.async)
  alignas(16) double2 nq[3][NY][NX];  // (n_c, q_c), c = x, y, z, of plane zc, q = phi (1 - phi) n: one 16-byte access serves both
  double ftab[2][LZ_MAX]; // sin / cos force table entries of this block's planes (lz <= LZ_MAX): the streaming pulls evict
                          // everything from L1, so a per-plane __ldg of the table would wait for L2 every plane
  double ftx[2][TX], fty[2][TY];  // the same for the tile's columns and rows (kept here rather than in 8 registers)
  // FUSED advection (row a8), one plane behind the node update:
  static constexpr int NA = FUSED ? TX * TY : 1;
  double ux[NA], uy[NA];  // u_x, u_y of the plane updated last (read by the neighbour lane / row)
  double fy[NA];          // flux through the y face above the node
  double e[FUSED ? 3 : 1][NA];  // own slots: phi + D lap phi (written when the plane is derived) - kappa div q (added at its
                                // node update) of planes zc-2, zc-1, zc; slot = plane mod 3 (as col)
  double col[3][NA];      // own slots: phi of the three planes older than the ring (z-face window)
  double acc[NA];         // own slot: phi(t+1) of the previous advected plane, still missing its upper z flux
};

// Velocity on the seams of the tile columns, written by k_lb_tp<FUSED> and read by k_seam; layouts (carved in accLB_create):
//   sx[((z ntx + bx) ny + y) 2 + s]   u_x at the first (s = 0) / last (s = 1) column of tile column bx
//   sy[(z 2 nty + 2 by + s) nx + x]   u_y at the first / last row of tile row by
//   sz[((2 bz + s) ny + y) nx + x]    u_z at the first / last plane of z chunk bz
struct Seams {
  double* sx;
  double* sy;
  double* sz;
  int ntx, nty;  // tile columns / rows
};

// Strip velocity of tile bb along DIR at (x, y, z): first (s = 0) or last (s = 1) cell of the tile.
template <int DIR>
__device__ __forceinline__ double seam_vel(const Seams& SM, const Grid& G, int x, int y, int z, int bb, int s) {
  if (DIR == 0) return __ldg(SM.sx + (((size_t)z * SM.ntx + bb) * G.ny + y) * 2 + s);
  if (DIR == 1) return __ldg(SM.sy + ((size_t)z * (size_t)(2 * SM.nty) + 2 * bb + s) * G.nx + x);
  return __ldg(SM.sz + ((size_t)(2 * bb + s) * G.ny + y) * G.nx + x);
}

// Advective flux (R12) through the seam face in front of the cell with coordinate c0 = first cell of tile
// b along DIR, at (x, y, z) (whose DIR component is ignored); bp = the tile behind the face.
template <int DIR>
__device__ __forceinline__ double seam_face_flux(const Grid& G, const double* __restrict__ phi, const Seams& SM, int x, int y,
                                                 int z, int c0, int b, int bp) {
  const size_t plane = (size_t)G.nx * (size_t)G.ny;
  const int n = DIR == 0 ? G.nx : DIR == 1 ? G.ny : G.nz;
  const size_t stride = DIR == 0 ? 1 : DIR == 1 ? (size_t)G.nx : plane;
  const size_t base = (DIR == 2 ? 0 : (size_t)z * plane) + (DIR == 1 ? 0 : (size_t)y * G.nx) + (DIR == 0 ? 0 : x);
  auto ph = [&](int k) { return __ldg(phi + base + (size_t)wrap_add(c0, k, n) * stride); };
  return face_flux(seam_vel<DIR>(SM, G, x, y, z, bp, 1), seam_vel<DIR>(SM, G, x, y, z, b, 0), ph(-3), ph(-2), ph(-1), ph(0),
                   ph(1), ph(2));
}

// Fused two-phase LB kernel (see the header of this file).  lz = planes per block along z.
// Iteration zc: phi(zc+1) has landed, fetch phi(zc+2) | derive n, q (tile + 1) and g, |g|, lap (own node, kept in
// registers) on plane zc from the raw planes zc-1, zc, zc+1; FUSED: advective fluxes of plane zc-2 | plane sums of plane
// zc, then the node update of plane z = zc - 1, whose z combinations need planes zc-2 .. zc (carried in registers).
// The 27 populations a thread pulls for plane z are fetched with TMA / cp.async into shared memory while
// the block is still busy with plane z-1 and with the geometry of plane z: the HBM latency of the pull hides under the
// fp64 work instead of stalling every warp at the top of the node update, and no register holds a load in flight.
// FAST (nx a multiple of TX, ny a multiple of TY, tensor maps available): every tile is full and pulls by
// TMA; no thread is idle and no per-thread wrap tables are kept.  Otherwise every tile pulls with per-thread cp.async.
// MODE: what a node does with its moments and its force -- the march, the staging and the geometry are the same:
//   MODE_FUSED    the time step (default): collide + store, advection fused, seam strips            rows a1-a8
//   MODE_UNFUSED  the time step with u(t) -> uout and r -> rout for k_advect (variant 2, RK3 stages)  rows a1-a7
//   MODE_MOMENTS  accLB_moments: p* -> rout, u -> uout (either may be NULL); the state is not touched   row a9
//   MODE_DIAG     accLB_diagnostics: the sums of R21 -> rout[0..7] (warp shuffle + one atomic per block and quantity)
//   MODE_INIT     accLB_init (R15): no pull; p* = in0, u0 = in1, A from F^s + F^p + F^b + F^g (F^nu := 0),
//                 f_i = f_i^eq(p*, u0) - S_i(u0, A)/2 written "pushed" to x - c_i so that the first pull returns it at x
//   MODE_FUSED_U  MODE_FUSED that also writes u(t) -> uout: the time step + first stage of the SSP-RK3 integrator (R32)
//   MODE_STAGE    a later Runge-Kutta stage: no populations; phi = the stage field, u(t) = in1 (frozen), base = in0 =
//                 phi(t); phi_new = rk_a base + rk_b (phi + L(phi)) but for the seam faces (k_seam<SCALED>)       row a8
enum { MODE_FUSED = 0, MODE_UNFUSED = 1, MODE_MOMENTS = 2, MODE_DIAG = 3, MODE_INIT = 4, MODE_STAGE = 5, MODE_FUSED_U = 6 };

__device__ __forceinline__ double tp_warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

template <typename ST, int TX, int TY, int MINB, int MODE, bool FAST>
__global__ void __launch_bounds__(TX * TY, MINB)
k_lb_tp(KP P, const ST* __restrict__ fin, ST* __restrict__ fout, const double* __restrict__ phi,
        double* __restrict__ uout, double* __restrict__ rout, double* __restrict__ phi_new, Seams SM,
        const double* __restrict__ tabs, int lz, const __grid_constant__ CUtensorMap tmap_fin,
        const __grid_constant__ CUtensorMap tmap_row, const double* __restrict__ in0, const double* __restrict__ in1) {
  constexpr bool LBF = MODE == MODE_FUSED || MODE == MODE_FUSED_U;  // the fused time step
  constexpr bool STAGE = MODE == MODE_STAGE;
  constexpr bool FUSED = LBF || STAGE;                              // the advection runs inside this kernel
  constexpr bool PULL = MODE != MODE_INIT && !STAGE;  // the populations of the current state are needed
  constexpr int EC = 16 / (int)sizeof(ST);  // elements per 16-byte chunk: the edge elements of the TMA pull are fetched as aligned chunks
  static_assert(!(FAST && MODE == MODE_INIT), "the push of the initial state uses the per-thread wrap tables");
  using T = GeoTile<ST, TX, TY, FUSED, !STAGE>;
  extern __shared__ __align__(128) unsigned char smem_lb[];
  T& S = *reinterpret_cast<T*>(smem_lb);
  constexpr int NT = TX * TY;
  constexpr int NR = T::NR;
  constexpr int RIM1 = T::NX * T::NY - NT;  // derive items besides the thread's own node
  static_assert(RIM1 <= NT, "at most one rim item per thread");
  static_assert(TX == 32 || !FUSED, "FUSED: one warp per tile row (x-face fluxes travel by warp shuffle)");
  const Grid& G = P.G;
  const int tid = threadIdx.x, tx = tid % TX, ty = tid / TX;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, z0 = blockIdx.z * lz;
  const int z1 = min(z0 + lz, G.nz);
  const int x = x0 + tx, y = y0 + ty;
  const bool active = FAST || (x < G.nx && y < G.ny);
  const unsigned plane = (unsigned)G.nx * (unsigned)G.ny;

  // staging item of this thread: the tid-th aligned pair of doubles of a PY x PX phi plane (tile + halo 2; x0 and nx are
  // even, so a pair never straddles the periodic wrap), copied with one 16-byte cp.async
  constexpr int PAIRS = T::PX / 2 * T::PY;
  static_assert(PAIRS <= NT && T::PX % 2 == 0, "one staging pair per thread");
  int r2 = -1;  // linear index j * PX + i of the pair's first element
  unsigned r2off = 0;
  if (tid < PAIRS) {
    const int j = tid / (T::PX / 2), i = 2 * (tid % (T::PX / 2));
    r2 = j * T::PX + i;
    r2off = (unsigned)pmod(y0 - 2 + j, G.ny) * (unsigned)G.nx + (unsigned)pmod(x0 - 2 + i, G.nx);
  }
  const int o2 = (ty + 2) * T::PX + (tx + 2);
  const unsigned o2off = (unsigned)pmod(y, G.ny) * (unsigned)G.nx + (unsigned)pmod(x, G.nx);
  // rim item of the derive pass: element (j, i) of the NY x NX plane that is not an own node
  int r1 = -1;  // j * NX + i (one register; j, i are recovered by a constant division where they are needed)
  if (tid < RIM1) {
    int r1j, r1i;
    if (tid < T::NX) { r1j = 0; r1i = tid; }
    else if (tid < 2 * T::NX) { r1j = T::NY - 1; r1i = tid - T::NX; }
    else { const int e = tid - 2 * T::NX; r1j = 1 + (e >> 1); r1i = (e & 1) ? T::NX - 1 : 0; }
    r1 = r1j * T::NX + r1i;
  }

  // a1: pull-stream of plane z, f_i(x,t) = f*_i(x - c_i, t-1).
  // FAST: 9 tiled TMA loads per plane (cp.async.bulk.tensor, one TX x TY x 3 box per triple of populations, issued by
  // lane 0 of the block's warps), completion counted in bytes on an mbarrier; no per-thread copy instructions, no address registers held by
  // copies in flight, no L1 allocation.  Lanes 0..17 of a row fetch the 9 + 9 elements per row outside the boxes.
  // Otherwise: one 8-byte cp.async per thread and population.  Either way population i of thread (tx, ty) is at *slot(i).
  constexpr bool fast = FAST;
  // Tiles on the y rim of the box: the rows shifted by c_iy wrap around, and TMA zero-fills out-of-bounds rows instead of
  // wrapping, so these tiles fetch the populations with c_iy != 0 row by row (TX x 1 boxes, every row wrapped on its own,
  // lanes 0..TY-1 of the issuing warp).
  const bool yrim = FAST && (y0 == 0 || y0 + TY >= G.ny);  // block-uniform
  // wrap tables of the per-thread pull (not FAST)
  int xs[3] = {0, 0, 0};
  unsigned yrow[3] = {0, 0, 0};
  if (!FAST) {
    const int xw = pmod(x, G.nx), yw = pmod(y, G.ny);
    xs[0] = wrap_dec(xw, G.nx); xs[1] = xw; xs[2] = wrap_inc(xw, G.nx);
    yrow[0] = (unsigned)wrap_dec(yw, G.ny) * (unsigned)G.nx; yrow[1] = (unsigned)yw * (unsigned)G.nx;
    yrow[2] = (unsigned)wrap_inc(yw, G.ny) * (unsigned)G.nx;
  }
  // three per-thread bases, one per c_ix, so that slot(i) is base + a compile-time offset
  ST* const sl_c = &S.fpop[ty * TX + tx];
  // (FAST: the slab's tail holds, per tile row, the aligned 16-byte chunk that ends at x0-1 (c_ix = +1) / starts at x0+TX (-1);
  // the edge lanes' bases are chosen so that base + pop_off(i) is the tail element: pop_off(3 m + 2) = m TRIPLE + 2 NT,
  // pop_off(3 m) = m TRIPLE)
  ST* const sl_p = tx == 0 ? &S.fpop[NT + T::TAILE + (fast ? EC * ty + EC - 1 : ty)] : sl_c - 1;  // c_ix = +1: element x - 1
  ST* const sl_m = tx == TX - 1 ? &S.fpop[3 * NT + (fast ? EC * ty : ty)] : sl_c + 1;              // c_ix = -1: element x + 1
  auto slot = [&](int i) -> ST* { return (cx_of(i) == 0 ? sl_c : cx_of(i) == 1 ? sl_p : sl_m) + T::pop_off(i); };
  // The TMA issue is spread over the block's warps (the last warp issues triples 0 and TY, the others one each; the first
  // warps carry the rim items of the derive pass): one thread issuing everything made its warp arrive late at the next
  // barrier in every iteration.  Thread 0 arms the mbarrier with the byte count.
  auto tma_pull = [&](int z) {  // called by lanes 0..TY-1 of every warp, after the block-wide hand-over of the landing zone
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    if (tid == 0) mbar_arrive_expect_tx(&S.fbar, (unsigned)(Q * NT * sizeof(ST)));
    const int zs[3] = {wrap_dec(z, G.nz) * Q, z * Q, wrap_inc(z, G.nz) * Q};
#pragma unroll
    for (int k = 0; k < (Q / 3 + TY - 1) / TY; ++k) {
      const int m = (TY - 1 - ty) + k * TY;  // triple: populations 3 m .. 3 m + 2, c_iy = m % 3 - 1, c_iz = m / 3 - 1
      if (m < Q / 3) {
        const int cy = m % 3 - 1, cz = m / 3 - 1;
        const int slab = (cz < 0 ? zs[2] : cz > 0 ? zs[0] : zs[1]) + 3 * m;
        ST* dst = &S.fpop[m * T::TRIPLE];
        if (yrim && cy != 0) {
          const int yy = pmod(y0 - cy + tx, G.ny);
#pragma unroll
          for (int j = 0; j < 3; ++j) tma_load_box(dst + j * NT + tx * TX, &tmap_row, x0, yy, slab + j, &S.fbar);
        } else if (tx == 0) {
          tma_load_box(dst, &tmap_fin, x0, y0 - cy, slab, &S.fbar);
        }
      }
    }
  };
  if (fast) {
    if (tid == 0) {
      mbar_init(&S.fbar, 1);
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (PULL && tx < TY) tma_pull(z0);
  }
  // FAST: the 9 + 9 elements per tile row that lie outside the unshifted boxes (x0 - 1 for c_ix = +1, x0 + TX for
  // c_ix = -1) are fetched by lanes 0..17 of the row's warp, one 16-byte cp.async each (the aligned pair that holds the
  // element), into the tail of the slabs
  // Carried per lane: the source address of its chunk for the plane pulled next (the calls go z0, z0 + 1, ...: the address
  // advances by one z slab per call and wraps with the lane's source plane z - c_iz), its landing address, and the z at
  // which the source plane wraps -- instead of a 64-bit slab product and the index arithmetic in every iteration.
  const ST* e_src = fin;
  unsigned e_dst = 0;
  int e_zwrap = 0;
  if (fast && tx < 18) {
    const int m = tx < 9 ? tx : tx - 9;  // population 3 m + 2 (c_ix = +1) or 3 m (c_ix = -1), c_iz = m / 3 - 1
    const int e_i = 3 * m + (tx < 9 ? 2 : 0), cy = m % 3 - 1, dz = 1 - m / 3;
    const unsigned e_off = (unsigned)e_i * plane + (unsigned)pmod(y - cy, G.ny) * (unsigned)G.nx +
                           (unsigned)(tx < 9 ? pmod(x0 - EC, G.nx) : pmod(x0 + TX, G.nx));
    e_src = pop_slab(fin, G, pmod(z0 + dz, G.nz)) + e_off;
    e_dst = (unsigned)__cvta_generic_to_shared(&S.fpop[m * T::TRIPLE + 3 * NT + (tx < 9 ? T::TAILE : 0) + EC * ty]);
    e_zwrap = G.nz - 1 - dz;  // the call with this z (or z - nz) fetches the last plane: the next one is plane 0
  }
  auto prefetch_pull = [&](int z) {
    if (fast) {  // the boxes are on their way (after the block-wide hand-over)
      if (tx < 18) {
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(e_dst), "l"(e_src) : "memory");
        const size_t slab = (size_t)Q * plane;
        e_src += slab;
        if (z == e_zwrap || z + G.nz == e_zwrap) e_src -= slab * (size_t)G.nz;
      }
      cp_async_commit();
      return;
    }
    const ST* slab[3] = {pop_slab(fin, G, wrap_dec(z, G.nz)), pop_slab(fin, G, z), pop_slab(fin, G, wrap_inc(z, G.nz))};
#pragma unroll
    for (int i = 0; i < Q; ++i) {
      const unsigned off = (unsigned)i * plane + yrow[1 - cy_of(i)] + (unsigned)xs[1 - cx_of(i)];
      cp_async_pop<(int)sizeof(ST)>(slot(i), slab[1 - cz_of(i)] + off);
    }
    cp_async_commit();
  };
  // Per-thread cp.async groups alternate phi plane | populations, every thread commits both in every iteration (an
  // empty group where it has nothing to fetch), so "all but the newest group" is always the one needed next.
  // phi(zc+2) lands in the ring one iteration before it is combined: its latency hides under plane zc.
  // Ring slots: plane z0 - 2 + j lives in slot j mod NR.
  {
    const double* s2 = phi + (size_t)pmod(z0, G.nz) * plane;
    if (r2 >= 0) cp_async_16(&S.raw[2][0][0] + r2, s2 + r2off);
    cp_async_commit();
  }
  if (PULL && active) prefetch_pull(z0);
  else cp_async_commit();

  // stage raw phi planes z0-2 and z0-1
  {
    const double* s0 = phi + (size_t)pmod(z0 - 2, G.nz) * plane;
    const double* s1 = phi + (size_t)pmod(z0 - 1, G.nz) * plane;
    double* d0 = &S.raw[0][0][0];
    double* d1 = &S.raw[1][0][0];
    if (r2 >= 0) {
      *reinterpret_cast<double2*>(d0 + r2) = __ldg(reinterpret_cast<const double2*>(s0 + r2off));
      *reinterpret_cast<double2*>(d1 + r2) = __ldg(reinterpret_cast<const double2*>(s1 + r2off));
    }
  }
  // div n and div q at plane z = zc-1 are z combinations of the plane sums a, b (see below) of planes zc-2, zc-1, zc:
  //   72 div v = a(zc-2) + 4 a(zc-1) + a(zc) + b(zc) - b(zc-2).  Carried per field: P = 4 a(zc-1) + a(zc-2) - b(zc-2) and
  //   Q = a(zc-1) - b(zc-1), so that 72 div v = P + (a(zc) + b(zc)) and P' = 4 a(zc) + Q, Q' = a(zc) - b(zc).
  double Pn = 0.0, Qn = 0.0, Pq = 0.0, Qq = 0.0;
  double gp[3] = {0.0, 0.0, 0.0}, gnp = 0.0, lapp = 0.0;  // g, |g|, lap phi of the own node at plane zc-1
  // FUSED: u_z at planes zc-3, zc-2; slot of plane zc-5 in the column history S.col (planes zc-5, zc-4, zc-3)
  double uzm = 0.0, uzc = 0.0;
  int cj = 0;
  // x-, y- and z-dependent table entries of the body force (R20) of this tile and chunk
  if (P.force_type != 0) {
    const int xw = pmod(x, G.nx), yw = pmod(y, G.ny);
    if (ty == 0) { S.ftx[0][tx] = __ldg(tabs + xw); S.ftx[1][tx] = __ldg(tabs + G.nx + xw); }
    if (tx == 0) { S.fty[0][ty] = __ldg(tabs + 2 * G.nx + yw); S.fty[1][ty] = __ldg(tabs + 2 * G.nx + G.ny + yw); }
    if (tid < z1 - z0) {
      S.ftab[0][tid] = __ldg(tabs + 2 * (G.nx + G.ny) + z0 + tid);
      S.ftab[1][tid] = __ldg(tabs + 2 * (G.nx + G.ny) + G.nz + z0 + tid);
    }
  }
  __syncthreads();

  int zq2 = pmod(z0 + 1, G.nz);  // wrapped zc + 2, carried (no integer division in the march)
  int sb = 0;                    // element offset of the ring slot of plane zc-1 (slot = it mod NR), carried
  const int zc_last = FUSED ? z1 + 1 : z1;  // FUSED: one more iteration to advect the last plane
  double dsum[8] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};  // MODE_DIAG: this thread's partial sums (7) and max |u|
  // One iteration of the march.  STEADY (FAST only): zc in [z0 + 3, z1 - 1], where every phase is active and no plane is
  // the first or the last of the chunk -- the same code with the chunk-boundary conditions resolved at compile time.
  // MODE_STAGE: the frozen velocity of the plane updated next (loaded one iteration ahead), and the Shu-Osher combination
  // rk_a phi(t) + rk_b (stage field + its increment) applied where a plane of phi_new is written
  double un[3] = {0.0, 0.0, 0.0};
  if (STAGE && active && z0 < z1) {
    const size_t kn = (size_t)z0 * plane + o2off;
    un[0] = __ldg(in1 + kn); un[1] = __ldg(in1 + (size_t)G.n + kn); un[2] = __ldg(in1 + 2 * (size_t)G.n + kn);
  }
  auto rk_out = [&](double v, size_t ko) { return STAGE ? fma(P.rk_b, v, P.rk_a * __ldg(in0 + ko)) : v; };
  auto iteration = [&](const int zc, auto steady_tag) {
    constexpr bool STEADY = decltype(steady_tag)::value;
    // ring planes zc-1+k, k = 0..3 (k = NR-1 is plane zc-2 when FUSED), as element offsets from S.raw; sb is carried
    constexpr int PSZ = T::PX * T::PY;
    auto ring = [&](int k) -> double* {
      int o = sb + k * PSZ;
      if (o >= NR * PSZ) o -= NR * PSZ;
      return &S.raw[0][0][0] + o;
    };
    // ---- phi(zc+1) has landed (this thread's own elements); fetch phi(zc+2)
    {
      cp_async_wait_but<1>();
      double* rn = ring(3);  // plane zc+2: its slot held plane zc+2-NR, last read before the previous iteration's
                             // second barrier
      if (STEADY || zc < z1) {
        const double* src = phi + (size_t)zq2 * plane;
        if (r2 >= 0) cp_async_16(rn + r2, src + r2off);
      }
      cp_async_commit();
      zq2 = wrap_inc(zq2, G.nz);
    }
    __syncthreads();
    // ---- derive n, q (tile + 1 rim) and g, |g|, lap (own node) on plane zc           PAPER.md:L61, L104; R17
    double gc[3] = {0.0, 0.0, 0.0}, gnc = 0.0, lapc = 0.0;
    if (STEADY || !FUSED || zc <= z1) {
      const double* rm = ring(0);  // plane zc-1
      const double* rc = ring(1);  // plane zc
      const double* rp = ring(2);  // plane zc+1
      auto derive = [&](int j, int i, bool own_node) {  // (j, i) in the NY x NX plane; centre (j+1, i+1) in a phi plane
        constexpr int PX = T::PX;
        const int b = j * PX + i;
        // z combinations of the nine columns around the node: t = Sz phi = (1,4,1).phi, d = Dz phi = phi(z+1) - phi(z-1)
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
        const double t00 = t[0], t01 = t[1], t02 = t[2], t10 = t[3], t11 = t[4], t12 = t[5], t20 = t[6], t21 = t[7], t22 = t[8];
        const double gx = (1.0 / 72.0) * fma(4.0, t12 - t10, (t02 - t00) + (t22 - t20));
        const double gy = (1.0 / 72.0) * fma(4.0, t21 - t01, (t20 - t00) + (t22 - t02));
        const double r0 = fma(4.0, d[1], d[0] + d[2]);
        const double r1 = fma(4.0, d[4], d[3] + d[5]);
        const double r2_ = fma(4.0, d[7], d[6] + d[8]);
        const double gz = (1.0 / 72.0) * fma(4.0, r1, r0 + r2_);
        const double gn = sqrt_pos(fma(gx, gx, fma(gy, gy, gz * gz)));
        const double inv = div_pos(1.0, gn + 1e-12);
        const double pq = ph * (1.0 - ph);
        const double nx_ = gx * inv, ny_ = gy * inv, nz_ = gz * inv;
        S.nq[0][j][i] = make_double2(nx_, pq * nx_);
        S.nq[1][j][i] = make_double2(ny_, pq * ny_);
        S.nq[2][j][i] = make_double2(nz_, pq * nz_);
        if (own_node) {
          const double s0 = fma(4.0, t01, t00 + t02), s1 = fma(4.0, t11, t10 + t12), s2 = fma(4.0, t21, t20 + t22);
          gc[0] = gx; gc[1] = gy; gc[2] = gz;
          gnc = gn;
          lapc = 6.0 * (fma(4.0, s1, s0 + s2) * (1.0 / 216.0) - ph);  // R7
          if (FUSED) S.e[cj >= 1 ? cj - 1 : 2][tid] = fma(P.D, lapc, ph);  // slot of plane zc = (cj + 2) mod 3
        }
      };
      derive(ty + 1, tx + 1, true);
      if (r1 >= 0) derive(r1 / T::NX, r1 % T::NX, false);
    }
    // ---- FUSED a8: advective fluxes of plane p = zc - 2 through the faces inside the tile column (R12)
    //   x face (x, x+1): own u_x and the neighbour lane's;  y face (y, y+1): u_y of the row above (shared memory);
    //   z face (p-1, p): u_z carried along the march.  Faces on the tile's seams are left to k_seam.
    const int pz = zc - 2;
    const bool adv = FUSED && (STEADY || pz >= z0);  // block-uniform; pz <= z1 - 1 because zc <= z1 + 1
    double Tp = 0.0;                     // phi(t+1) of plane pz, accumulated
    if (FUSED) {
      const double* rq = ring(NR - 1);                   // plane zc-2 = pz, tile + halo 2
      const double php = rq[o2];
      if (adv) {
        constexpr int PX = T::PX;
        if (LBF && FAST && tid >= NT - 2 * TY) {  // u_x of plane pz on the two x seams of the tile: 2 TY contiguous strip entries
          const int e = tid - (NT - 2 * TY);
          SM.sx[(((unsigned)pz * (unsigned)SM.ntx + blockIdx.x) * (unsigned)G.ny + (unsigned)y0) * 2u + (unsigned)e] =
              S.ux[(e >> 1) * TX + ((e & 1) ? TX - 1 : 0)];
        }
        const bool xseam = tx == TX - 1 || x + 1 >= G.nx;  // the face to the right is a seam (or the thread idle)
        const bool yseam = ty == TY - 1 || y + 1 >= G.ny;
        const double* row = rq + (ty + 2) * PX + tx;       // phi(x-2 .. x+3) of the own row
        double Fx = face_flux(S.ux[tid], S.ux[xseam ? tid : tid + 1], row[0], row[1], row[2], row[3], row[4], row[5]);
        Fx = xseam ? 0.0 : Fx;
        double Fxl = __shfl_up_sync(0xffffffffu, Fx, 1);
        Fxl = tx == 0 ? 0.0 : Fxl;
        const double* col = rq + ty * PX + (tx + 2);       // phi(y-2 .. y+3) of the own column
        double Fy = face_flux(S.uy[tid], S.uy[yseam ? tid : tid + TX], col[0], col[PX], col[2 * PX], col[3 * PX], col[4 * PX],
                              col[5 * PX]);
        Fy = yseam ? 0.0 : Fy;
        S.fy[tid] = Fy;
        // z face (pz-1, pz): phi(pz-3 .. pz+2) = the column history, then planes zc-2, zc-1, zc of the ring
        const int cj1 = cj == 2 ? 0 : cj + 1, cj2 = cj1 == 2 ? 0 : cj1 + 1;
        double Fz = face_flux(uzm, uzc, S.col[cj][tid], S.col[cj1][tid], S.col[cj2][tid], php, ring(0)[o2], ring(1)[o2]);
        if (!STEADY) Fz = pz == z0 ? 0.0 : Fz;
        if (STEADY || (pz > z0 && active)) {  // plane pz-1 is complete
          const size_t ko = (size_t)(pz - 1) * plane + o2off;
          __stcs(phi_new + ko, rk_out(S.acc[tid] - Fz, ko));
        }
        Tp = S.e[cj][tid] - (Fx - Fxl) - Fy + Fz;
      }
      S.col[cj][tid] = php;  // plane zc-2 replaces plane zc-5
      cj = cj == 2 ? 0 : cj + 1;
    }
    // ---- a1-a2 of plane z = zc - 1: the pulled populations have landed in this thread's slots; moments.  Done before the
    // barrier so that ONE barrier both publishes n, q, the y fluxes and hands the landing zone over for the next pull.
    const int z = zc - 1;
    const bool node = STEADY || (z >= z0 && z < z1 && active);
    Moments M;
    if (node && PULL) {
      cp_async_wait_but<1>();
      if (fast) {
        __syncwarp();  // the edge elements were copied by other lanes of this warp
        mbar_wait(&S.fbar, (unsigned)(z - z0) & 1u);
      }
      moments_of([&](int i) { return Pop<ST>::from_storage(*slot(i), i); }, M);
    }
    if (node && MODE == MODE_INIT) {  // p* given, no momentum, no stress (R15)
      M.p = __ldg(in0 + (size_t)z * plane + o2off);
      M.m[0] = M.m[1] = M.m[2] = 0.0;
#pragma unroll
      for (int j = 0; j < 6; ++j) M.Pi[j] = 0.0;
    }
    __syncthreads();
    if (adv) {
      Tp += ty == 0 ? 0.0 : S.fy[tid - TX];
      if (!STEADY && pz == z1 - 1) {  // the face above the chunk's last plane is a seam
        if (active) {
          const size_t ko = (size_t)pz * plane + o2off;
          __stcs(phi_new + ko, rk_out(Tp, ko));
        }
      } else {
        S.acc[tid] = Tp;
      }
    }
    // ---- plane sums of plane zc at the own node:  a = Dx Sy v_x + Sx Dy v_y,  b = Sx Sy v_z
    double an2 = 0.0, bn2 = 0.0, aq2 = 0.0, bq2 = 0.0;
    if (STEADY || !FUSED || zc <= z1) {
      constexpr int NX = T::NX;
      // (n and q together: every shared-memory access fetches the pair (n_c, q_c))
      const double2* vx = &S.nq[0][ty][tx];
      const double2* vy = &S.nq[1][ty][tx];
      const double2* vz = &S.nq[2][ty][tx];
      const double2 x00 = vx[0], x02 = vx[2], x10 = vx[NX], x12 = vx[NX + 2], x20 = vx[2 * NX], x22 = vx[2 * NX + 2];
      const double2 y00 = vy[0], y01 = vy[1], y02 = vy[2], y20 = vy[2 * NX], y21 = vy[2 * NX + 1], y22 = vy[2 * NX + 2];
      const double axn = fma(4.0, x12.x - x10.x, (x02.x - x00.x) + (x22.x - x20.x));
      const double axq = fma(4.0, x12.y - x10.y, (x02.y - x00.y) + (x22.y - x20.y));
      const double ayn = fma(4.0, y21.x - y01.x, (y20.x - y00.x) + (y22.x - y02.x));
      const double ayq = fma(4.0, y21.y - y01.y, (y20.y - y00.y) + (y22.y - y02.y));
      an2 = axn + ayn;
      aq2 = axq + ayq;
      const double2 z00 = vz[0], z01 = vz[1], z02 = vz[2], z10 = vz[NX], z11 = vz[NX + 1], z12 = vz[NX + 2];
      const double2 z20 = vz[2 * NX], z21 = vz[2 * NX + 1], z22 = vz[2 * NX + 2];
      bn2 = fma(4.0, fma(4.0, z11.x, z10.x + z12.x), fma(4.0, z01.x, z00.x + z02.x) + fma(4.0, z21.x, z20.x + z22.x));
      bq2 = fma(4.0, fma(4.0, z11.y, z10.y + z12.y), fma(4.0, z01.y, z00.y + z02.y) + fma(4.0, z21.y, z20.y + z22.y));
    }
    double uz_new = 0.0;
    if (!node) cp_async_commit();
    if (node) {
      // every warp has read its 27 values out of the landing zone (barrier above): refill it for plane z+1
      if (PULL && fast && (STEADY || z + 1 < z1) && tx < TY) tma_pull(z + 1);
      if (PULL && (STEADY || z + 1 < z1)) prefetch_pull(z + 1);
      else cp_async_commit();
      // a3: kappa_c = div n, div q at plane z from the plane sums of z-1, z, z+1
      const double kc = (1.0 / 72.0) * (Pn + (an2 + bn2));
      const double divq = (1.0 / 72.0) * (Pq + (aq2 + bq2));
      const double phi0 = ring(0)[o2];  // plane zc-1 = z

      const unsigned k = (unsigned)z * plane + o2off;
      // phi-only part of Eq. 3: r = D lap phi - kappa div q
      if (FUSED) S.e[cj][tid] -= P.kappa * divq;  // (cj was advanced above: slot of plane z = zc-1)
      else if (MODE == MODE_UNFUSED) rout[k] = P.D * lapp - P.kappa * divq;

      if (STAGE) {  // u(t) is frozen (R32): this plane's was loaded one iteration ago, fetch the next plane's
        S.ux[tid] = un[0];
        S.uy[tid] = un[1];
        uz_new = un[2];
        if (STEADY || z + 1 < z1) {
          const size_t kn = (size_t)k + plane;
          un[0] = __ldg(in1 + kn); un[1] = __ldg(in1 + (size_t)G.n + kn); un[2] = __ldg(in1 + 2 * (size_t)G.n + kn);
        }
      } else {
        // body-force density (R20): the z part of the per-axis tables is the same address for the whole block (L1 hit)
        double Fb[3] = {0.0, 0.0, 0.0};
        if (P.force_type != 0) {
          const double fsz = S.ftab[0][z - z0], fcz = S.ftab[1][z - z0];
          const double fsx = S.ftx[0][tx], fcx = S.ftx[1][tx], fsy = S.fty[0][ty], fcy = S.fty[1][ty];
          if (P.force_type == 1) {  // ABC
            Fb[0] = P.force_amp * (fsz + fcy);
            Fb[1] = P.force_amp * (fsx + fcz);
            Fb[2] = P.force_amp * (fsy + fcx);
          } else {  // sine variant of BASELINE config 2
            Fb[0] = P.force_amp * fsy;
            Fb[1] = P.force_amp * fsz;
            Fb[2] = P.force_amp * fsx;
          }
        }
        double A[3], rho;
        accel_from_geometry(P, M, gp, gnp, kc, phi0, Fb, MODE != MODE_INIT, A, rho);
        const double u[3] = {M.m[0] + 0.5 * A[0], M.m[1] + 0.5 * A[1], M.m[2] + 0.5 * A[2]};  // a5, PAPER.md:L88 (R4)
        if (LBF) {
          S.ux[tid] = u[0];
          S.uy[tid] = u[1];
          uz_new = u[2];
          // velocities on the seams of this tile column (every strip has fewer elements than the grid has nodes: 32-bit
          // indices).  FAST: u_x goes out one iteration later, 2 TY contiguous values from S.ux by one warp (see the
          // advection phase); u_y only by the two warps that own the first and the last row.
          if (!FAST) {
            const unsigned ix = (((unsigned)z * (unsigned)SM.ntx + blockIdx.x) * (unsigned)G.ny + (unsigned)y) * 2u;
            if (tx == 0) SM.sx[ix] = u[0];
            if (tx == TX - 1 || x == G.nx - 1) SM.sx[ix + 1] = u[0];
          }
          if (!FAST || ty == 0 || ty == TY - 1) {
            const unsigned iy = ((unsigned)z * (unsigned)(2 * SM.nty) + 2u * blockIdx.y) * (unsigned)G.nx + (unsigned)x;
            if (ty == 0) SM.sy[iy] = u[1];
            if (ty == TY - 1 || y == G.ny - 1) SM.sy[iy + (unsigned)G.nx] = u[1];
          }
          if (!STEADY && z == z0) SM.sz[(2u * blockIdx.z) * plane + o2off] = u[2];
          if (!STEADY && z == z1 - 1) SM.sz[(2u * blockIdx.z + 1u) * plane + o2off] = u[2];
        }
        if (MODE == MODE_UNFUSED || MODE == MODE_MOMENTS || MODE == MODE_FUSED_U) {
          if (MODE != MODE_MOMENTS || uout) {
            uout[k] = u[0];
            uout[(size_t)G.n + k] = u[1];
            uout[2 * (size_t)G.n + k] = u[2];
          }
          if (MODE == MODE_MOMENTS && rout) rout[k] = M.p;
        }
        if (LBF || MODE == MODE_UNFUSED) collide_store<ST>(P, M, u, A, pop_slab(fout, G, z) + o2off, plane);
        if (MODE == MODE_DIAG && z >= P.zlo && z < P.zhi) {  // R21: rho |u|^2 / 2, nu a:a / (2 cs4 tau^2), phi, p*, m, max |u|;
                                                              // a z-slab sums its own planes only
          double a6[6];
          hermite_coeff(M, u, A, a6);
          const double uu = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
          const double aa = a6[0] * a6[0] + a6[1] * a6[1] + a6[2] * a6[2] + 2.0 * (a6[3] * a6[3] + a6[4] * a6[4] + a6[5] * a6[5]);
          dsum[0] += 0.5 * rho * uu;
          dsum[1] += P.eps_pref * aa;
          dsum[2] += phi0;
          dsum[3] += M.p;
          dsum[4] += M.m[0];
          dsum[5] += M.m[1];
          dsum[6] += M.m[2];
          dsum[7] = fmax(dsum[7], sqrt(uu));
        }
        if (MODE == MODE_INIT) {  // R15: f_i = f_i^eq(p*, u0) - S_i(u0, A)/2, pushed to x - c_i
          const double u0[3] = {__ldg(in1 + k), __ldg(in1 + (size_t)G.n + k), __ldg(in1 + 2 * (size_t)G.n + k)};
          const double U[3] = {u0[0] - 0.5 * A[0], u0[1] - 0.5 * A[1], u0[2] - 0.5 * A[2]};
          double Tt[6];
          Tt[0] = u0[0] * u0[0] - u0[0] * A[0];
          Tt[1] = u0[1] * u0[1] - u0[1] * A[1];
          Tt[2] = u0[2] * u0[2] - u0[2] * A[2];
          Tt[3] = u0[0] * u0[1] - 0.5 * (u0[0] * A[1] + u0[1] * A[0]);
          Tt[4] = u0[0] * u0[2] - 0.5 * (u0[0] * A[2] + u0[2] * A[0]);
          Tt[5] = u0[1] * u0[2] - 0.5 * (u0[1] * A[2] + u0[2] * A[1]);
          double f[Q];
          hermite2_populations(M.p, U, Tt, f);
          ST* slab[3] = {pop_slab(fout, G, wrap_dec(z, G.nz)), pop_slab(fout, G, z), pop_slab(fout, G, wrap_inc(z, G.nz))};
  #pragma unroll
          for (int i = 0; i < Q; ++i)
            Pop<ST>::store(slab[1 - cz_of(i)] + ((unsigned)i * plane + yrow[1 - cy_of(i)] + (unsigned)xs[1 - cx_of(i)]), i, f[i]);
        }
      }
    }
    Pn = fma(4.0, an2, Qn); Qn = an2 - bn2;
    Pq = fma(4.0, aq2, Qq); Qq = aq2 - bq2;
    gp[0] = gc[0]; gp[1] = gc[1]; gp[2] = gc[2]; gnp = gnc; lapp = lapc;
    uzm = uzc; uzc = uz_new;
    sb = sb + PSZ == NR * PSZ ? 0 : sb + PSZ;
  };
  int zc = z0 - 1;
  if (FAST && FUSED) {
    for (; zc < z0 + 3 && zc <= zc_last; ++zc) iteration(zc, std::false_type{});
    for (; zc <= z1 - 1; ++zc) iteration(zc, std::true_type{});
  }
  for (; zc <= zc_last; ++zc) iteration(zc, std::false_type{});
  if (MODE == MODE_DIAG) {  // north-star (e): warp shuffle, then one atomic per block and quantity
    __syncthreads();
    double* sh = reinterpret_cast<double*>(&S.nq[0][0][0]);  // [8][TY]
#pragma unroll
    for (int j = 0; j < 7; ++j) {
      const double r = tp_warp_sum(dsum[j]);
      if (tx == 0) sh[j * TY + ty] = r;
    }
    {
      double v = dsum[7];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
      if (tx == 0) sh[7 * TY + ty] = v;
    }
    __syncthreads();
    if (tid < 8) {
      double r = sh[tid * TY];
      for (int w = 1; w < TY; ++w) r = tid < 7 ? r + sh[tid * TY + w] : fmax(r, sh[tid * TY + w]);
      if (tid < 7) atomicAdd(rout + tid, r);
      else atomicMax(reinterpret_cast<unsigned long long*>(rout + 7), (unsigned long long)__double_as_longlong(r));  // r >= 0
    }
  }
}

// a8 on the seams of the tile columns of k_lb_tp<FUSED> (R12).  A face is a seam when its two cells
// belong to different tile columns / z chunks: x faces in front of x = TX b, y faces in front of y = TY b, z faces in
// front of z = lz b (b = 0 is the periodic wrap).  ONE launch for the three directions, one thread per seam face: it
// evaluates the flux once from the two strip velocities and phi(t) and adds it to phi(t+1) of the cell in front of the
// face (+) and subtracts it from the cell behind (-), so sum phi is conserved to rounding.  The additions are atomic: a
// cell on a tile edge receives fluxes from two or three seams, in an order that is not fixed (last-bit differences from
// run to run in those cells; every other cell is bitwise reproducible).  The blocks of the x faces (latency-bound: their
// cells are a tile width apart) are interleaved with those of the y faces (bandwidth-bound: whole rows) so that the two
// kinds overlap on every SM; lanes run along y for the x faces (the strips u_x[z][bx][y][s] are then contiguous) and
// along x for the y and z faces.
constexpr int SEAM_THREADS = 128;
template <bool SCALED>
__device__ __forceinline__ double seam_scale(const KP& P, double F) { return SCALED ? P.rk_b * F : F; }
struct SeamGrid {
  unsigned nfx, nfy, nfz;  // seam faces per direction
  unsigned bx, by, bz;     // blocks per direction
  int lz, nchunk;
};
// SCALED: the fluxes enter phi_new times rk_b (a Runge-Kutta stage, k_lb_tp<MODE_STAGE>).
template <int TX, int TY, bool SCALED>
__global__ void __launch_bounds__(SEAM_THREADS) k_seam(KP P, const double* __restrict__ phi, double* __restrict__ phi_new,
                                                       Seams SM, SeamGrid SG) {
  const Grid& G = P.G;
  const size_t plane = (size_t)G.nx * (size_t)G.ny;
  // which direction this block serves: x and y blocks interleaved in proportion, z blocks last
  const unsigned i = blockIdx.x, T = SG.bx + SG.by;
  int dir;
  unsigned blk;
  if (i < T) {
    const unsigned y0 = (unsigned)(((unsigned long long)i * SG.by) / T), y1 = (unsigned)(((unsigned long long)(i + 1) * SG.by) / T);
    if (y1 > y0) { dir = 1; blk = y0; }
    else { dir = 0; blk = i - y1; }
  } else {
    dir = 2; blk = i - T;
  }
  const unsigned t = blk * SEAM_THREADS + threadIdx.x;
  if (dir == 0) {
    if (t >= SG.nfx) return;
    const int y = (int)(t % (unsigned)G.ny);
    const unsigned r = t / (unsigned)G.ny;
    const int b = (int)(r % (unsigned)SM.ntx), z = (int)(r / (unsigned)SM.ntx);
    const int c0 = b * TX, bp = b == 0 ? SM.ntx - 1 : b - 1;
    const double F = seam_scale<SCALED>(P, seam_face_flux<0>(G, phi, SM, 0, y, z, c0, b, bp));
    double* row = phi_new + (size_t)z * plane + (size_t)y * G.nx;
    atomicAdd(row + c0, F);
    atomicAdd(row + (c0 == 0 ? G.nx - 1 : c0 - 1), -F);
  } else if (dir == 1) {
    if (t >= SG.nfy) return;
    const int x = (int)(t % (unsigned)G.nx);
    const unsigned r = t / (unsigned)G.nx;
    const int b = (int)(r % (unsigned)SM.nty), z = (int)(r / (unsigned)SM.nty);
    const int c0 = b * TY, bp = b == 0 ? SM.nty - 1 : b - 1;
    const double F = seam_scale<SCALED>(P, seam_face_flux<1>(G, phi, SM, x, 0, z, c0, b, bp));
    double* col = phi_new + (size_t)z * plane + x;
    atomicAdd(col + (size_t)c0 * G.nx, F);
    atomicAdd(col + (size_t)(c0 == 0 ? G.ny - 1 : c0 - 1) * G.nx, -F);
  } else {
    if (t >= SG.nfz) return;
    const int x = (int)(t % (unsigned)G.nx);
    const unsigned r = t / (unsigned)G.nx;
    const int y = (int)(r % (unsigned)G.ny), b = (int)(r / (unsigned)G.ny);
    const int c0 = b * SG.lz, bp = b == 0 ? SG.nchunk - 1 : b - 1;
    const double F = seam_scale<SCALED>(P, seam_face_flux<2>(G, phi, SM, x, y, 0, c0, b, bp));
    double* cell = phi_new + (size_t)y * G.nx + x;
    atomicAdd(cell + (size_t)c0 * plane, F);
    atomicAdd(cell + (size_t)(c0 == 0 ? G.nz - 1 : c0 - 1) * plane, -F);
  }
}

// ---------------------------------------------------------------------------------------------------- advection
// Shared memory of k_advect.  Everything a plane needs is fetched with cp.async one plane ahead (no register holds a
// load in flight); buffers that only their owner thread touches (col, uz, r) need no barrier.
template <int TX, int TY>
struct AdvTile {
  double phi[2][TY + 6][TX + 6];  // plane z (ping-pong) with halo 3 along x and y (corners unused)
  double ux[2][TY][TX + 2];       // u_x with halo 1 along x
  double uy[2][TY + 2][TX];       // u_y with halo 1 along y
  double fx[TY][TX + 1];          // flux through the x face between tile columns i-1 and i
  double fy[TY + 1][TX];          // flux through the y face between tile rows j-1 and j
  double col[2][TX * TY];         // landing slot of the thread's own phi(z+3) (ping-pong); the window lives in registers
  double uz[2][TX * TY];          // landing slot of the thread's own u_z(z+1)
  double r[2][TX * TY];           // r = D lap phi - kappa div q of planes z, z+1
};

template <int TX, int TY>
__global__ void __launch_bounds__(TX * TY, 4)
k_advect(KP P, const double* __restrict__ phi, const double* __restrict__ u, const double* __restrict__ r,
         double* __restrict__ phi_new, int lz, const double* __restrict__ base, double ca, double cb) {
  using T = AdvTile<TX, TY>;
  extern __shared__ __align__(128) unsigned char smem_lb[];
  T& S = *reinterpret_cast<T*>(smem_lb);
  constexpr int NT = TX * TY;
  static_assert(TX == 32 && TY >= 8 && 6 * (TX + TY) <= NT && 2 * (TX + TY) <= NT, "one warp per tile row, one halo element per thread");
  const Grid& G = P.G;
  const int tid = threadIdx.x, tx = tid % TX, ty = tid / TX;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, z0 = blockIdx.z * lz;
  const int z1 = min(z0 + lz, G.nz);
  const int x = x0 + tx, y = y0 + ty;
  const bool active = x < G.nx && y < G.ny;
  const size_t plane = (size_t)G.nx * (size_t)G.ny;
  const size_t n = G.n;
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
  size_t voff = 0;
  if (tid < 2 * TX) {
    vkind = 1;
    vj = tid < TX ? 0 : TY + 1;
    vi = tid % TX;
    voff = n + (size_t)pmod(y0 - 1 + vj, G.ny) * (size_t)G.nx + (size_t)pmod(x0 + vi, G.nx);
  } else if (tid < 2 * (TX + TY)) {
    const int e = tid - 2 * TX;
    vkind = 2;
    vj = e / 2;
    vi = (e & 1) ? TX + 1 : 0;
    voff = (size_t)pmod(y0 + vj, G.ny) * (size_t)G.nx + (size_t)pmod(x0 - 1 + vi, G.nx);
  }

  // asynchronous fetch of what plane zp needs on top of the rings: its tile of phi, u_x, u_y with halos, and r
  auto fetch_plane = [&](int b, int zp) {  // zp already wrapped
    const size_t zo = (size_t)zp * plane;
    cp_async_f64(&S.phi[b][ty + 3][tx + 3], phi + zo + own);
    cp_async_f64(&S.ux[b][ty][tx + 1], u + zo + own);
    cp_async_f64(&S.uy[b][ty + 1][tx], u + n + zo + own);
    cp_async_f64(&S.r[b][tid], r + zo + own);
    if (hj >= 0) cp_async_f64(&S.phi[b][hj][hi], phi + zo + hoff);
    if (vkind == 1) cp_async_f64(&S.uy[b][vj][vi], u + zo + voff);
    else if (vkind == 2) cp_async_f64(&S.ux[b][vj][vi], u + zo + voff);
  };
  // what the first plane needs, fetched asynchronously: its tile, and the newest members of the two z windows
  auto zoff = [&](int zz) { return (size_t)pmod(zz, G.nz) * plane; };
  cp_async_f64(&S.col[0][tid], phi + zoff(z0 + 3) + own);
  cp_async_f64(&S.uz[0][tid], u + 2 * n + zoff(z0 + 1) + own);
  fetch_plane(0, pmod(z0, G.nz));
  cp_async_commit();
  // column window w[j] = phi(z - 2 + j), j = 0..5, of the z face between z and z + 1; here still one plane behind
  double w0, w1 = __ldg(phi + zoff(z0 - 2) + own), w2 = __ldg(phi + zoff(z0 - 1) + own), w3 = __ldg(phi + zoff(z0) + own);
  double w4 = __ldg(phi + zoff(z0 + 1) + own), w5 = __ldg(phi + zoff(z0 + 2) + own);
  double uz0, uz1 = __ldg(u + 2 * n + zoff(z0) + own);
  double fz_prev = face_flux(__ldg(u + 2 * n + zoff(z0 - 1) + own), uz1, __ldg(phi + zoff(z0 - 3) + own), w1, w2, w3, w4, w5);  // face (z0 - 1, z0)
  int zp1 = pmod(z0 + 1, G.nz), zp2 = pmod(z0 + 2, G.nz), zp4 = pmod(z0 + 4, G.nz);

  for (int z = z0; z < z1; ++z) {
    const int b = (z - z0) & 1;
    cp_async_wait_all();
    __syncthreads();  // plane z is in shared memory; the x / y fluxes of plane z-1 have been consumed
    w0 = w1; w1 = w2; w2 = w3; w3 = w4; w4 = w5;
    w5 = S.col[b][tid];
    uz0 = uz1;
    uz1 = S.uz[b][tid];
    if (z + 1 < z1) {  // fetch plane z+1
      cp_async_f64(&S.col[b ^ 1][tid], phi + (size_t)zp4 * plane + own);  // phi(z+4)
      cp_async_f64(&S.uz[b ^ 1][tid], u + 2 * n + (size_t)zp2 * plane + own);  // u_z(z+2)
      fetch_plane(b ^ 1, zp1);
      cp_async_commit();
      zp1 = wrap_inc(zp1, G.nz); zp2 = wrap_inc(zp2, G.nz); zp4 = wrap_inc(zp4, G.nz);
    }
    {  // x face between tile columns tx and tx+1; one warp per tile row
      const double* p = &S.phi[b][ty + 3][tx + 1];  // phi at tile columns tx-2 .. tx+3
      S.fx[ty][tx + 1] = face_flux(S.ux[b][ty][tx + 1], S.ux[b][ty][tx + 2], p[0], p[1], p[2], p[3], p[4], p[5]);
    }
    {  // y face between tile rows ty and ty+1
      const double(*q)[TX + 6] = S.phi[b];
      S.fy[ty + 1][tx] = face_flux(S.uy[b][ty + 1][tx], S.uy[b][ty + 2][tx], q[ty + 1][tx + 3], q[ty + 2][tx + 3], q[ty + 3][tx + 3],
                                   q[ty + 4][tx + 3], q[ty + 5][tx + 3], q[ty + 6][tx + 3]);
    }
    if (ty == 3 && tx < TY) {  // the TY faces on the tile's left edge
      const double* p = &S.phi[b][tx + 3][0];
      S.fx[tx][0] = face_flux(S.ux[b][tx][0], S.ux[b][tx][1], p[0], p[1], p[2], p[3], p[4], p[5]);
    }
    if (ty == TY - 1) {  // the TX faces on the tile's lower edge
      const double(*q)[TX + 6] = S.phi[b];
      S.fy[0][tx] = face_flux(S.uy[b][0][tx], S.uy[b][1][tx], q[0][tx + 3], q[1][tx + 3], q[2][tx + 3], q[3][tx + 3], q[4][tx + 3],
                              q[5][tx + 3]);
    }
    const double fz = face_flux(uz0, uz1, w0, w1, w2, w3, w4, w5);  // face (z, z + 1)
    const double rr = S.r[b][tid];
    __syncthreads();
    if (active) {
      double adv = 0.0;
      adv += S.fx[ty][tx + 1] - S.fx[ty][tx];
      adv += S.fy[ty + 1][tx] - S.fy[ty][tx];
      adv += fz - fz_prev;
      const double euler = w2 + (-adv + rr);
      // a Runge-Kutta stage (phase_rk.cuh) combines the Euler update of the stage field with the base field phi(t)
      __stcs(phi_new + (size_t)z * plane + own, base ? ca * __ldg(base + (size_t)z * plane + own) + cb * euler : euler);
    }
    fz_prev = fz;
  }
}

}  // namespace acclb
