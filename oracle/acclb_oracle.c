/*
 * accLB CPU oracle  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, literal fp64 implementation of the per-time-step lattice update of accLB
 * (arXiv 2505.01126, /root/reference/PAPER.md), written from the paper's equations in the paper's own
 * two-pass "thread-safe" organisation: pass 1 reduces the 27 populations at a node
 * to the ten macroscopic fields p*, u_a, a_ab (+ the acceleration A_a), pass 2 rebuilds the
 * post-collision populations AT THE NEIGHBOUR from those stored fields and pulls them (Eq. 6).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build,
 * load or call this file.  It shares no code, header, table or helper with the CUDA path under
 * paper_2505_01126_b200/csrc, and neither includes the other.
 *
 * Every function cites the passage it follows.  Where PAPER.md is silent or garbled the reading taken is
 * the one listed in DESIGN.md ("Readings", R1..R28, same numbering as SURVEY.md section 8(c)).
 * No blocking, no pair tricks, no closed-form shortcuts: loops over z,y,x and i=0..26, explicit
 * (x+c+N)%N periodic wraps.  Build with -ffp-contract=off so the arithmetic is what is written.
 *
 * Parity-unpinned parts (the paper fixes nothing to pin them against):
 *   - WENO5 variant / epsilon (R12), the choice of phi integrator (R13 forward Euler, R32 SSP-RK3: both pinned as
 *     schemes, the paper names neither), step ordering (R14), the reference density of the buoyancy force (R31).
 *   Pinned since round 2 (tests/test_oracle_physics.py): direction, upwind side and order of the phi advection
 *   (face_flux / pass_allen_cahn), and F^nu (R9) on a prescribed shear against nu (du + du^T).grad rho.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stddef.h>

#define Q 27
#define CS2 (1.0 / 3.0) /* R1: c_s^2 of D3Q27 */
#define CS4 (CS2 * CS2)

typedef struct {
  int nx, ny, nz;
  double tau;      /* PAPER.md:L83  nu = c_s^2 (tau - 1/2), omega = 1/tau */
  int two_phase;   /* 0: single component (rho == 1, F = F^b) ; 1: LB + conservative Allen-Cahn */
  double rho_l;    /* density where phi = 1   PAPER.md:L102, R16 */
  double rho_g;    /* density where phi = 0 */
  double sigma;    /* gamma, surface tension */
  double mobility; /* D, interface diffusivity PAPER.md:L61 */
  double width;    /* delta, interface width; kappa = 4 D / delta */
  int force_type;  /* 0 none | 1 ABC | 2 sine (BASELINE config 2), R20 */
  double force_amp;
  int force_k;         /* forcing wavenumber in units of 2 pi / L */
  int force_period[3]; /* box the forcing is periodic on (0 -> nx,ny,nz); lets a sub-box of a larger */
  int force_origin[3]; /* problem be evaluated: global coordinate of local node (0,0,0)              */
  double gravity[3];   /* buoyancy F^g = (rho(phi) - rho_ref) g   PAPER.md:L193, L203 ("buoyant gas phase"); R31 */
  double rho_ref;      /* reference density of the buoyancy force (the harness sets the mean density: no net force) */
  int phi_rk3;         /* 0: forward Euler (R13) | 1: SSP-RK3 for phi within one LB step   PAPER.md:L110; R32 */
} oracle_params;

typedef struct {
  oracle_params p;
  size_t n;
  long step;
  double *f;            /* [27][n]  post-streaming populations f_i(x,t) */
  double *phi, *phi2;   /* order parameter, and its update target  */
  double *pstar;        /* the ten macroscopic fields of PAPER.md:L118 ...                    */
  double *u;            /* [3][n]                                                             */
  double *a;            /* [6][n]  xx,yy,zz,xy,xz,yz                                          */
  double *A;            /* [3][n]  acceleration F/rho (R3) entering S_i                       */
  double *m;            /* [3][n]  raw first moment sum_i f_i c_i (for diagnostics)           */
  double *g;            /* [3][n]  grad phi                                                   */
  double *nrm;          /* [3][n]  interface normal                                           */
  double *phi_s, *nrm_s; /* RK3 only: stage field and its normal                              */
} oracle_state;

static int C[Q][3];
static double W[Q];
static double HM[Q][3][3]; /* H_i,ab = c_ia c_ib - c_s^2 delta_ab, tabulated */
static int lattice_ready = 0;

/* R1: D3Q27, c_i in {-1,0,1}^3, i = (cx+1) + 3(cy+1) + 9(cz+1); w = 8/27, 2/27, 1/54, 1/216. */
static void lattice_init(void) {
  if (lattice_ready) return;
  for (int i = 0; i < Q; ++i) {
    C[i][0] = i % 3 - 1;
    C[i][1] = (i / 3) % 3 - 1;
    C[i][2] = i / 9 - 1;
    int nnz = abs(C[i][0]) + abs(C[i][1]) + abs(C[i][2]);
    W[i] = nnz == 0 ? 8.0 / 27.0 : nnz == 1 ? 2.0 / 27.0 : nnz == 2 ? 1.0 / 54.0 : 1.0 / 216.0;
    for (int al = 0; al < 3; ++al)
      for (int be = 0; be < 3; ++be) HM[i][al][be] = C[i][al] * C[i][be] - (al == be ? CS2 : 0.0);
  }
  lattice_ready = 1;
}

static inline int wrap(int a, int n) { return ((a % n) + n) % n; }
static inline size_t at(const oracle_state *s, int x, int y, int z) {
  return ((size_t)wrap(z, s->p.nz) * s->p.ny + wrap(y, s->p.ny)) * s->p.nx + wrap(x, s->p.nx);
}
static const int I6[3][3] = {{0, 3, 4}, {3, 1, 5}, {4, 5, 2}}; /* symmetric index: xx,yy,zz,xy,xz,yz */

/* Second-order Hermite polynomial H_i,ab = c_ia c_ib - c_s^2 delta_ab */
static inline double herm(int i, int al, int be) { return HM[i][al][be]; }

/* Pressure-based equilibrium  f_i^eq = w_i (p* + c.u/cs2 + H_i,ab u_a u_b / (2 cs4)) */
static double feq(int i, double pstar, const double u[3]) {
  double cu = 0.0, huu = 0.0;
  for (int al = 0; al < 3; ++al) cu += C[i][al] * u[al];
  for (int al = 0; al < 3; ++al)
    for (int be = 0; be < 3; ++be) huu += herm(i, al, be) * u[al] * u[be];
  return W[i] * (pstar + cu / CS2 + huu / (2.0 * CS4));
}

/* Guo forcing S_i = w_i [ (c_ia - u_a)/cs2 + (c_ib u_b) c_ia / cs4 ] A_a   PAPER.md:L79 (Eq. 5);
 * the "force" is the acceleration A = F/rho because the first moment is a velocity (R3). */
static double guo(int i, const double u[3], const double A[3]) {
  double cu = 0.0, s = 0.0;
  for (int be = 0; be < 3; ++be) cu += C[i][be] * u[be];
  for (int al = 0; al < 3; ++al) s += ((C[i][al] - u[al]) / CS2 + cu * C[i][al] / CS4) * A[al];
  return W[i] * s;
}

/* Hermite-reconstructed non-equilibrium f_i^neq = w_i H_i,ab a_ab / (2 cs4)   PAPER.md:L88 with R5 */
static double fneq_rec(int i, const double a6[6]) {
  double ha = 0.0;
  for (int al = 0; al < 3; ++al)
    for (int be = 0; be < 3; ++be) ha += herm(i, al, be) * a6[I6[al][be]];
  return W[i] * ha / (2.0 * CS4);
}

/* R20 body force density F^b at local node (x,y,z). */
static void body_force(const oracle_params *p, int x, int y, int z, double Fb[3]) {
  Fb[0] = Fb[1] = Fb[2] = 0.0;
  if (p->force_type == 0) return;
  const double two_pi = 6.283185307179586476925286766559;
  int L[3] = {p->force_period[0] ? p->force_period[0] : p->nx, p->force_period[1] ? p->force_period[1] : p->ny,
              p->force_period[2] ? p->force_period[2] : p->nz};
  double X = x + p->force_origin[0], Y = y + p->force_origin[1], Z = z + p->force_origin[2];
  double kx = two_pi * p->force_k / L[0], ky = two_pi * p->force_k / L[1], kz = two_pi * p->force_k / L[2];
  if (p->force_type == 1) { /* ABC */
    Fb[0] = p->force_amp * (sin(kz * Z) + cos(ky * Y));
    Fb[1] = p->force_amp * (sin(kx * X) + cos(kz * Z));
    Fb[2] = p->force_amp * (sin(ky * Y) + cos(kx * X));
  } else { /* sine variant of BASELINE config 2 */
    Fb[0] = p->force_amp * sin(ky * Y);
    Fb[1] = p->force_amp * sin(kz * Z);
    Fb[2] = p->force_amp * sin(kx * X);
  }
}

/* Lattice gradient  d_a Psi = (1/cs2) sum_i w_i Psi(x + c_i) c_ia */
static void grad_at(const oracle_state *s, const double *psi, int x, int y, int z, double out[3]) {
  out[0] = out[1] = out[2] = 0.0;
  for (int i = 0; i < Q; ++i) {
    double v = psi[at(s, x + C[i][0], y + C[i][1], z + C[i][2])];
    for (int al = 0; al < 3; ++al) out[al] += W[i] * v * C[i][al];
  }
  for (int al = 0; al < 3; ++al) out[al] /= CS2;
}

/* Lattice Laplacian  (2/cs2) sum_i w_i (Psi(x+c_i) - Psi(x))   PAPER.md:L104 as repaired by R7 */
static double lap_at(const oracle_state *s, const double *psi, int x, int y, int z) {
  double acc = 0.0, c0 = psi[at(s, x, y, z)];
  for (int i = 0; i < Q; ++i) acc += W[i] * (psi[at(s, x + C[i][0], y + C[i][1], z + C[i][2])] - c0);
  return 2.0 * acc / CS2;
}

/* Jiang-Shu WENO5 face value from the five upwind-ordered cell values (R12, ref [19]). */
static double weno5(double a, double b, double c, double d, double e) {
  const double eps = 1e-6;
  double q0 = (2.0 * a - 7.0 * b + 11.0 * c) / 6.0;
  double q1 = (-b + 5.0 * c + 2.0 * d) / 6.0;
  double q2 = (2.0 * c + 5.0 * d - e) / 6.0;
  double b0 = 13.0 / 12.0 * (a - 2.0 * b + c) * (a - 2.0 * b + c) + 0.25 * (a - 4.0 * b + 3.0 * c) * (a - 4.0 * b + 3.0 * c);
  double b1 = 13.0 / 12.0 * (b - 2.0 * c + d) * (b - 2.0 * c + d) + 0.25 * (b - d) * (b - d);
  double b2 = 13.0 / 12.0 * (c - 2.0 * d + e) * (c - 2.0 * d + e) + 0.25 * (3.0 * c - 4.0 * d + e) * (3.0 * c - 4.0 * d + e);
  double a0 = 0.1 / ((eps + b0) * (eps + b0));
  double a1 = 0.6 / ((eps + b1) * (eps + b1));
  double a2 = 0.3 / ((eps + b2) * (eps + b2));
  return (a0 * q0 + a1 * q1 + a2 * q2) / (a0 + a1 + a2);
}

/* Advective flux of phi through the face between x and x+e along axis ax (R12: flux form, face velocity =
 * arithmetic mean, upwinding by its sign). */
static double face_flux(const oracle_state *s, const double *ph, int ax, int x, int y, int z) {
  int e[3] = {0, 0, 0};
  e[ax] = 1;
  const double *ue = s->u + (size_t)ax * s->n;
#define PH(k) ph[at(s, x + (k)*e[0], y + (k)*e[1], z + (k)*e[2])]
  double uf = 0.5 * (ue[at(s, x, y, z)] + ue[at(s, x + e[0], y + e[1], z + e[2])]);
  double pf;
  if (uf >= 0.0)
    pf = weno5(PH(-2), PH(-1), PH(0), PH(1), PH(2));
  else
    pf = weno5(PH(3), PH(2), PH(1), PH(0), PH(-1));
#undef PH
  return uf * pf;
}

/* ---- O2 (first half): g = grad phi, n = g / (|g| + 1e-12) for every node   PAPER.md:L61, L104; R17 ---- */
static void geometry_of(const oracle_state *s, const double *phi, double *g_out /* may be NULL */, double *nrm_out) {
  const int nx = s->p.nx, ny = s->p.ny, nz = s->p.nz;
  const size_t n = s->n;
#pragma omp parallel for collapse(2) schedule(static)
  for (int z = 0; z < nz; ++z)
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        size_t k = at(s, x, y, z);
        double g[3];
        grad_at(s, phi, x, y, z, g);
        double gn = sqrt(g[0] * g[0] + g[1] * g[1] + g[2] * g[2]);
        for (int al = 0; al < 3; ++al) {
          if (g_out) g_out[al * n + k] = g[al];
          nrm_out[al * n + k] = g[al] / (gn + 1e-12);
        }
      }
}
static void pass_geometry(oracle_state *s) { geometry_of(s, s->phi, s->g, s->nrm); }

/* Total force at a node from phi-geometry and the node's own moments (O2 second half + O3).
 * with_visc = 0 drops F^nu (used by init, R15).  Returns F in F[3] and rho. */
static double total_force(const oracle_state *s, int x, int y, int z, double pstar, const double m[3],
                          const double Pi[6], int with_visc, double F[3]) {
  const oracle_params *p = &s->p;
  double Fb[3];
  body_force(p, x, y, z, Fb);
  if (!p->two_phase) { /* single component: rho == 1, F = F^b (+ the uniform (1 - rho_ref) g, R31) */
    for (int al = 0; al < 3; ++al) F[al] = Fb[al] + (1.0 - p->rho_ref) * p->gravity[al];
    return 1.0;
  }
  const size_t n = s->n, k = at(s, x, y, z);
  double g[3] = {s->g[k], s->g[n + k], s->g[2 * n + k]};
  double gn = sqrt(g[0] * g[0] + g[1] * g[1] + g[2] * g[2]);
  /* curvature kappa_c = div n by the lattice stencil   PAPER.md:L104, R8 */
  double kc = 0.0;
  for (int i = 0; i < Q; ++i) {
    size_t kk = at(s, x + C[i][0], y + C[i][1], z + C[i][2]);
    for (int al = 0; al < 3; ++al) kc += W[i] * C[i][al] * s->nrm[al * n + kk];
  }
  kc /= CS2;
  double rho = p->rho_g + (p->rho_l - p->rho_g) * s->phi[k];
  double drho[3], Fs[3], Fp[3], Fg[3], Fv[3] = {0.0, 0.0, 0.0};
  for (int al = 0; al < 3; ++al) {
    Fg[al] = (rho - p->rho_ref) * p->gravity[al]; /* buoyancy; R31 */
    drho[al] = (p->rho_l - p->rho_g) * g[al];
    Fs[al] = -p->sigma * (1.5 * p->width) * kc * gn * g[al]; /* PAPER.md:L102 + normalisation R8 */
    Fp[al] = -pstar * CS2 * drho[al];
  }
  if (with_visc && p->rho_l != p->rho_g) { /* PAPER.md:L104 read as R9 */
    double ut[3];
    for (int al = 0; al < 3; ++al) ut[al] = m[al] + (Fs[al] + Fp[al] + Fb[al] + Fg[al]) / (2.0 * rho);
    double pref = (p->tau - 0.5) / p->tau; /* nu omega / cs2 */
    for (int al = 0; al < 3; ++al) {
      double acc = 0.0;
      for (int be = 0; be < 3; ++be)
        acc += (Pi[I6[al][be]] - (al == be ? pstar * CS2 : 0.0) - ut[al] * ut[be]) * drho[be];
      Fv[al] = -pref * acc;
    }
  }
  for (int al = 0; al < 3; ++al) F[al] = Fs[al] + Fp[al] + Fv[al] + Fb[al] + Fg[al]; /* Eq. 8, PAPER.md:L100 (+ F^b, F^g) */
  return rho;
}

/* ---- pass 1: O1 moments, O3 forces, O4 velocity, O5 Hermite coefficient; stores the paper's ten fields ---- */
static void pass_moments(oracle_state *s) {
  const int nx = s->p.nx, ny = s->p.ny, nz = s->p.nz;
  const size_t n = s->n;
#pragma omp parallel for collapse(2) schedule(static)
  for (int z = 0; z < nz; ++z)
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        size_t k = at(s, x, y, z);
        /* O1  p* = sum f_i, m = sum f_i c_i, Pi = sum f_i c_i c_i */
        double pstar = 0.0, m[3] = {0, 0, 0}, Pi[6] = {0, 0, 0, 0, 0, 0};
        for (int i = 0; i < Q; ++i) {
          double fi = s->f[(size_t)i * n + k];
          pstar += fi;
          for (int al = 0; al < 3; ++al) m[al] += fi * C[i][al];
          for (int al = 0; al < 3; ++al)
            for (int be = al; be < 3; ++be) Pi[I6[al][be]] += fi * C[i][al] * C[i][be];
        }
        double F[3];
        double rho = total_force(s, x, y, z, pstar, m, Pi, 1, F);
        /* O4  A = F / rho (R3), u = m + A/2 (PAPER.md:L88 read as R4) */
        double A[3], u[3];
        for (int al = 0; al < 3; ++al) {
          A[al] = F[al] / rho;
          u[al] = m[al] + 0.5 * A[al];
        }
        /* O5  a_ab = sum_i (f_i - f_i^eq + S_i/2) H_i,ab   PAPER.md:L83, L92 (Eq. 7) */
        double a6[6] = {0, 0, 0, 0, 0, 0};
        for (int i = 0; i < Q; ++i) {
          double fne = s->f[(size_t)i * n + k] - feq(i, pstar, u) + 0.5 * guo(i, u, A);
          for (int al = 0; al < 3; ++al)
            for (int be = al; be < 3; ++be) a6[I6[al][be]] += fne * herm(i, al, be);
        }
        s->pstar[k] = pstar;
        for (int al = 0; al < 3; ++al) {
          s->u[al * n + k] = u[al];
          s->A[al * n + k] = A[al];
          s->m[al * n + k] = m[al];
        }
        for (int j = 0; j < 6; ++j) s->a[j * n + k] = a6[j];
      }
}

/* ---- pass 2: O6 reconstruction at the source node y = x - c_i and O7 thread-safe pull.
 * f_i(x, t+1) = f_i^eq(y) + (1 - omega) f_i^neq(y) + S_i(y)/2     PAPER.md:L85 (Eq. 6), L118 ---- */
static void pass_reconstruct_stream(oracle_state *s) {
  const int nx = s->p.nx, ny = s->p.ny, nz = s->p.nz;
  const size_t n = s->n;
  const double omega = 1.0 / s->p.tau;
#pragma omp parallel for collapse(2) schedule(static)
  for (int z = 0; z < nz; ++z)
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        size_t k = at(s, x, y, z);
        for (int i = 0; i < Q; ++i) {
          size_t ks = at(s, x - C[i][0], y - C[i][1], z - C[i][2]);
          double u[3] = {s->u[ks], s->u[n + ks], s->u[2 * n + ks]};
          double A[3] = {s->A[ks], s->A[n + ks], s->A[2 * n + ks]};
          double a6[6];
          for (int j = 0; j < 6; ++j) a6[j] = s->a[j * n + ks];
          s->f[(size_t)i * n + k] = feq(i, s->pstar[ks], u) + (1.0 - omega) * fneq_rec(i, a6) + 0.5 * guo(i, u, A);
        }
      }
}

/* ---- pass 3: O8 conservative Allen-Cahn, flux-form WENO5 advection (R12), lattice Laplacian (R7) and lattice divergence
 * of the sharpening flux phi(1-phi)n   PAPER.md:L61 (Eq. 3), L67, L104.
 * One evaluation: out = a * base + b * (phi + L(phi)),  L(phi) = -div(u phi) + D lap phi - kappa div(phi (1 - phi) n),
 * with n = n(phi) given in nrm and u = u(t) of pass 1.  Forward Euler (R13) is a = 0, b = 1. ---- */
static void allen_cahn_stage(const oracle_state *s, const double *phi, const double *nrm, const double *base, double a,
                             double b, double *out) {
  const int nx = s->p.nx, ny = s->p.ny, nz = s->p.nz;
  const size_t n = s->n;
  const double D = s->p.mobility, kappa = 4.0 * s->p.mobility / s->p.width;
#pragma omp parallel for collapse(2) schedule(static)
  for (int z = 0; z < nz; ++z)
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        size_t k = at(s, x, y, z);
        double adv = 0.0;
        adv += face_flux(s, phi, 0, x, y, z) - face_flux(s, phi, 0, x - 1, y, z);
        adv += face_flux(s, phi, 1, x, y, z) - face_flux(s, phi, 1, x, y - 1, z);
        adv += face_flux(s, phi, 2, x, y, z) - face_flux(s, phi, 2, x, y, z - 1);
        double lap = lap_at(s, phi, x, y, z);
        double divq = 0.0;
        for (int i = 0; i < Q; ++i) {
          size_t kk = at(s, x + C[i][0], y + C[i][1], z + C[i][2]);
          double ph = phi[kk];
          for (int al = 0; al < 3; ++al) divq += W[i] * C[i][al] * (ph * (1.0 - ph) * nrm[al * n + kk]);
        }
        divq /= CS2;
        double euler = phi[k] + (-adv + D * lap - kappa * divq);
        out[k] = base ? a * base[k] + b * euler : euler;
      }
}

/* Forward Euler (R13), or the three-stage SSP Runge-Kutta scheme of Shu and Osher (R32; PAPER.md:L110 names "time
 * integrators" without choosing one) with the velocity frozen at u(t):
 *   phi1 = phi + L(phi);  phi2 = 3/4 phi + 1/4 (phi1 + L(phi1));  phi(t+1) = 1/3 phi + 2/3 (phi2 + L(phi2)),
 * the normal recomputed from every stage field. */
static void pass_allen_cahn(oracle_state *s) {
  if (!s->p.phi_rk3) {
    allen_cahn_stage(s, s->phi, s->nrm, NULL, 0.0, 1.0, s->phi2);
  } else {
    allen_cahn_stage(s, s->phi, s->nrm, NULL, 0.0, 1.0, s->phi_s);               /* phi1 */
    geometry_of(s, s->phi_s, NULL, s->nrm_s);
    allen_cahn_stage(s, s->phi_s, s->nrm_s, s->phi, 0.75, 0.25, s->phi2);        /* phi2 */
    geometry_of(s, s->phi2, NULL, s->nrm_s);
    allen_cahn_stage(s, s->phi2, s->nrm_s, s->phi, 1.0 / 3.0, 2.0 / 3.0, s->phi_s); /* phi(t+1) */
    double *t = s->phi_s;
    s->phi_s = s->phi2;
    s->phi2 = t;
  }
  double *t = s->phi;
  s->phi = s->phi2;
  s->phi2 = t;
}

/* =============================== exported C interface (ctypes) =============================== */

oracle_state *oracle_create(const oracle_params *p) {
  lattice_init();
  if (!p || p->nx < 1 || p->ny < 1 || p->nz < 1 || !(p->tau > 0.5)) return NULL;
  oracle_state *s = (oracle_state *)calloc(1, sizeof(oracle_state));
  if (!s) return NULL;
  s->p = *p;
  s->n = (size_t)p->nx * p->ny * p->nz;
  size_t n = s->n;
  s->f = (double *)calloc(Q * n, sizeof(double));
  s->pstar = (double *)calloc(n, sizeof(double));
  s->u = (double *)calloc(3 * n, sizeof(double));
  s->a = (double *)calloc(6 * n, sizeof(double));
  s->A = (double *)calloc(3 * n, sizeof(double));
  s->m = (double *)calloc(3 * n, sizeof(double));
  int ok = s->f && s->pstar && s->u && s->a && s->A && s->m;
  if (p->two_phase) {
    s->phi = (double *)calloc(n, sizeof(double));
    s->phi2 = (double *)calloc(n, sizeof(double));
    s->g = (double *)calloc(3 * n, sizeof(double));
    s->nrm = (double *)calloc(3 * n, sizeof(double));
    ok = ok && s->phi && s->phi2 && s->g && s->nrm;
    if (p->phi_rk3) {
      s->phi_s = (double *)calloc(n, sizeof(double));
      s->nrm_s = (double *)calloc(3 * n, sizeof(double));
      ok = ok && s->phi_s && s->nrm_s;
    }
  }
  if (!ok) {
    free(s->f); free(s->pstar); free(s->u); free(s->a); free(s->A); free(s->m);
    free(s->phi); free(s->phi2); free(s->g); free(s->nrm); free(s->phi_s); free(s->nrm_s); free(s);
    return NULL;
  }
  return s;
}

void oracle_destroy(oracle_state *s) {
  if (!s) return;
  free(s->f); free(s->pstar); free(s->u); free(s->a); free(s->A); free(s->m);
  free(s->phi); free(s->phi2); free(s->g); free(s->nrm); free(s->phi_s); free(s->nrm_s);
  free(s);
}

/* Init (R15): f_i = f_i^eq(p*, u0) - S_i(u0, A)/2 with A from F^s + F^p + F^b (F^nu := 0).
 * rho_in is p* (R19); u_in is [3][nz][ny][nx]; phi_in may be NULL when single-phase. */
int oracle_init(oracle_state *s, const double *rho_in, const double *u_in, const double *phi_in) {
  if (!s || !rho_in || !u_in || (s->p.two_phase && !phi_in)) return -1;
  const int nx = s->p.nx, ny = s->p.ny, nz = s->p.nz;
  const size_t n = s->n;
  if (s->p.two_phase) {
    memcpy(s->phi, phi_in, n * sizeof(double));
    pass_geometry(s);
  }
#pragma omp parallel for collapse(2) schedule(static)
  for (int z = 0; z < nz; ++z)
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        size_t k = at(s, x, y, z);
        double u0[3] = {u_in[k], u_in[n + k], u_in[2 * n + k]};
        double zero3[3] = {0, 0, 0}, zero6[6] = {0, 0, 0, 0, 0, 0}, F[3], A[3];
        double rho = total_force(s, x, y, z, rho_in[k], zero3, zero6, 0, F);
        for (int al = 0; al < 3; ++al) A[al] = F[al] / rho;
        for (int i = 0; i < Q; ++i) s->f[(size_t)i * n + k] = feq(i, rho_in[k], u0) - 0.5 * guo(i, u0, A);
      }
  s->step = 0;
  return 0;
}

/* One or more full steps t -> t+1 in the synchronous order of R14. */
int oracle_step(oracle_state *s, int nsteps) {
  if (!s || nsteps < 0) return -1;
  for (int it = 0; it < nsteps; ++it) {
    if (s->p.two_phase) pass_geometry(s);  /* O2 */
    pass_moments(s);                       /* O1, O3, O4, O5 */
    pass_reconstruct_stream(s);            /* O6, O7 */
    if (s->p.two_phase) pass_allen_cahn(s); /* O8, with u(t), phi(t), n(t) */
    s->step += 1;
  }
  return 0;
}

/* (p*, u, phi) of the current state; the state itself is unchanged (the moment fields are scratch). */
int oracle_moments(oracle_state *s, double *rho_out, double *u_out, double *phi_out) {
  if (!s) return -1;
  if (s->p.two_phase) pass_geometry(s);
  pass_moments(s);
  if (rho_out) memcpy(rho_out, s->pstar, s->n * sizeof(double));
  if (u_out) memcpy(u_out, s->u, 3 * s->n * sizeof(double));
  if (phi_out && s->p.two_phase) memcpy(phi_out, s->phi, s->n * sizeof(double));
  return 0;
}

/* R21: out[0..8] = KE, dissipation, sum phi, sum p*, sum m_x, sum m_y, sum m_z, max|u|, step count. */
int oracle_diagnostics(oracle_state *s, double *out, int n_out) {
  if (!s || !out || n_out < 9) return -1;
  if (s->p.two_phase) pass_geometry(s);
  pass_moments(s);
  const size_t n = s->n;
  const double nu = CS2 * (s->p.tau - 0.5);
  long double ke = 0, eps = 0, sphi = 0, sp = 0, sm[3] = {0, 0, 0};
  double umax = 0.0;
  for (size_t k = 0; k < n; ++k) {
    double rho = s->p.two_phase ? s->p.rho_g + (s->p.rho_l - s->p.rho_g) * s->phi[k] : 1.0;
    double uu = 0.0;
    for (int al = 0; al < 3; ++al) uu += s->u[al * n + k] * s->u[al * n + k];
    ke += 0.5 * rho * uu;
    double aa = 0.0;
    for (int al = 0; al < 3; ++al)
      for (int be = 0; be < 3; ++be) aa += s->a[I6[al][be] * n + k] * s->a[I6[al][be] * n + k];
    eps += nu * aa / (2.0 * CS4 * s->p.tau * s->p.tau);
    if (s->p.two_phase) sphi += s->phi[k];
    sp += s->pstar[k];
    for (int al = 0; al < 3; ++al) sm[al] += s->m[al * n + k];
    if (sqrt(uu) > umax) umax = sqrt(uu);
  }
  out[0] = (double)(ke / (long double)n);
  out[1] = (double)(eps / (long double)n);
  out[2] = (double)sphi;
  out[3] = (double)sp;
  out[4] = (double)sm[0];
  out[5] = (double)sm[1];
  out[6] = (double)sm[2];
  out[7] = umax;
  out[8] = (double)s->step;
  return 0;
}

/* ---- raw access used only by the pin tests ---- */
int oracle_get_populations(const oracle_state *s, double *f_out) {
  if (!s || !f_out) return -1;
  memcpy(f_out, s->f, Q * s->n * sizeof(double));
  return 0;
}
int oracle_set_populations(oracle_state *s, const double *f_in) {
  if (!s || !f_in) return -1;
  memcpy(s->f, f_in, Q * s->n * sizeof(double));
  return 0;
}
/* the stored fields of pass 1 after oracle_moments(): a [6][n], A [3][n], m [3][n], n [3][n] */
int oracle_get_hermite(const oracle_state *s, double *a_out) {
  if (!s || !a_out) return -1;
  memcpy(a_out, s->a, 6 * s->n * sizeof(double));
  return 0;
}
int oracle_get_accel(const oracle_state *s, double *A_out) {
  if (!s || !A_out) return -1;
  memcpy(A_out, s->A, 3 * s->n * sizeof(double));
  return 0;
}

void oracle_lattice(int *c_out /* [27][3] */, double *w_out /* [27] */) {
  lattice_init();
  for (int i = 0; i < Q; ++i) {
    for (int al = 0; al < 3; ++al) c_out[3 * i + al] = C[i][al];
    w_out[i] = W[i];
  }
}
void oracle_feq(double pstar, const double *u, double *out27) {
  lattice_init();
  for (int i = 0; i < Q; ++i) out27[i] = feq(i, pstar, u);
}
void oracle_guo(const double *u, const double *A, double *out27) {
  lattice_init();
  for (int i = 0; i < Q; ++i) out27[i] = guo(i, u, A);
}
void oracle_fneq(const double *a6, double *out27) {
  lattice_init();
  for (int i = 0; i < Q; ++i) out27[i] = fneq_rec(i, a6);
}
double oracle_weno5(double a, double b, double c, double d, double e) { return weno5(a, b, c, d, e); }

/* stencils on a bare periodic field [nz][ny][nx] */
void oracle_gradient(const double *psi, int nx, int ny, int nz, double *out3) {
  lattice_init();
  oracle_state s;
  memset(&s, 0, sizeof s);
  s.p.nx = nx; s.p.ny = ny; s.p.nz = nz;
  s.n = (size_t)nx * ny * nz;
  for (int z = 0; z < nz; ++z)
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        double g[3];
        grad_at(&s, psi, x, y, z, g);
        size_t k = at(&s, x, y, z);
        for (int al = 0; al < 3; ++al) out3[al * s.n + k] = g[al];
      }
}
void oracle_laplacian(const double *psi, int nx, int ny, int nz, double *out) {
  lattice_init();
  oracle_state s;
  memset(&s, 0, sizeof s);
  s.p.nx = nx; s.p.ny = ny; s.p.nz = nz;
  s.n = (size_t)nx * ny * nz;
  for (int z = 0; z < nz; ++z)
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) out[at(&s, x, y, z)] = lap_at(&s, psi, x, y, z);
}
void oracle_body_force(const oracle_params *p, int x, int y, int z, double *F3) { body_force(p, x, y, z, F3); }
