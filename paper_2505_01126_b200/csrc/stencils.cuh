// Periodic neighbour indexing, the lattice-stencil derivative operators of PAPER.md:L104 and the WENO5 face
// reconstruction of PAPER.md:L67 (Jiang-Shu, R12), device side.  Part of the CUDA product path.
//
// The D3Q27 weights factorise, w_i = o(cx) o(cy) o(cz) with o(0) = 2/3, o(+-1) = 1/6, so the stencils
//   d_a Psi  = (1/cs2) sum_i w_i c_ia Psi(x + c_i)
//   lap Psi  = (2/cs2) sum_i w_i (Psi(x + c_i) - Psi(x))        PAPER.md:L104 as repaired by R7
// are evaluated in separable form: a central difference along a, smoothed with (1,4,1)/6 along the two other
// axes.  Same numbers as the 27-term sums up to rounding order.
#pragma once

namespace acclb {

struct Grid {
  int nx, ny, nz;
  unsigned n;  // nodes; n < 2^31 (checked at create)
};

// Wrapped coordinates of the 3x3x3 neighbourhood of a node: periodic boundaries as in-kernel index wrap
// (compare-select, no modulo), replacing the paper's halo exchange.
struct Nbr {
  int x[3];            // x-1, x, x+1 wrapped
  unsigned row[3][3];  // [dz+1][dy+1] -> (zz * ny + yy) * nx   (scalar fields, [z][y][x])
  int z[3];            // z-1, z, z+1 wrapped                    (populations, [z][i][y][x])
  unsigned yr[3];      // yy * nx
  __device__ __forceinline__ unsigned at(int dz, int dy, int dx) const { return row[dz + 1][dy + 1] + x[dx + 1]; }
};

__device__ __forceinline__ int wrap_dec(int a, int n) { return a == 0 ? n - 1 : a - 1; }
__device__ __forceinline__ int wrap_inc(int a, int n) { return a == n - 1 ? 0 : a + 1; }
// a + k for |k| <= 3 on a period n >= 4
__device__ __forceinline__ int wrap_add(int a, int k, int n) {
  int r = a + k;
  if (r < 0) r += n;
  if (r >= n) r -= n;
  return r;
}

__device__ __forceinline__ void make_nbr(const Grid& G, int x, int y, int z, Nbr& nb) {
  nb.x[0] = wrap_dec(x, G.nx); nb.x[1] = x; nb.x[2] = wrap_inc(x, G.nx);
  const int ys[3] = {wrap_dec(y, G.ny), y, wrap_inc(y, G.ny)};
  const int zs[3] = {wrap_dec(z, G.nz), z, wrap_inc(z, G.nz)};
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    nb.z[a] = zs[a];
    nb.yr[a] = (unsigned)ys[a] * (unsigned)G.nx;
#pragma unroll
    for (int b = 0; b < 3; ++b) nb.row[a][b] = ((unsigned)zs[a] * (unsigned)G.ny + (unsigned)ys[b]) * (unsigned)G.nx;
  }
}

// Population storage: [z][i][y][x] -- for every z plane the 27 population planes lie next to each other.  The address of
// f_i at (z, y, x) is base(z) + (i * plane + y * nx + x) with a 64-bit base per z plane and a 32-bit in-slab offset
// (27 * nx * ny < 2^32 is checked at create), which costs two integer instructions per access instead of five for the
// [i][z][y][x] layout (64-bit i * n + offset), and keeps the 27 + 27 streams of a step inside a few 2 MB pages per plane.
template <typename T>
__device__ __forceinline__ T* pop_slab(T* f, const Grid& G, int z) {
  T* p = f + (size_t)z * 27u * ((size_t)G.nx * (size_t)G.ny);
  asm("" : "+l"(p));  // keep the slab base a pointer in a register pair: the compiler otherwise folds it back into a
                      // 64-bit index computation per access
  return p;
}

// sqrt(s) for s >= 0: hardware reciprocal-square-root seed, two Newton steps on y ~ 1/sqrt(s), then s y with one residual
// correction; relative error ~1e-16, a fixed instruction sequence without the library routine's special-case call.
// s = 0 gives 0 (the seed is taken of max(s, 1e-300); below that the result is only needed to be << 1e-12, R17).
__device__ __forceinline__ double sqrt_pos(double s) {
  double y;
  const double sc = fmax(s, 1e-300);
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(sc));
  const double h = 0.5 * sc;
  y = __fma_rn(__fma_rn(-h * y, y, 0.5), y, y);
  y = __fma_rn(__fma_rn(-h * y, y, 0.5), y, y);
  const double r = s * y;
  return __fma_rn(__fma_rn(-r, r, s), 0.5 * y, r);
}

// a / b for b > 0 in the normal range: hardware reciprocal seed (relative error 2^-23), two Newton steps and one
// residual correction of the quotient; within an ulp of the correctly rounded quotient, a fixed instruction sequence
// (so both cells of a face get the same bits), about half the instructions of the IEEE division with its slow path.
__device__ __forceinline__ double div_pos(double a, double b) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(b));
  r = __fma_rn(__fma_rn(-b, r, 1.0), r, r);
  r = __fma_rn(__fma_rn(-b, r, 1.0), r, r);
  const double q = __dmul_rn(a, r);
  return __fma_rn(__fma_rn(-b, q, a), r, q);
}

// Jiang-Shu WENO5 (R12, ref. [19]) at the face downwind of `c`, from the five upwind-ordered cell values
// a..e, written on the four differences d1 = b - a, d2 = c - b, d3 = d - c, d4 = e - d.  Returns face value MINUS c:
//   candidates   q0 - c = (5 d2 - 2 d1)/6,  q1 - c = (d2 + 2 d3)/6,  q2 - c = (4 d3 - d4)/6
//   smoothness   b0 = 13/12 (d2 - d1)^2 + 1/4 (3 d2 - d1)^2,  b1 = 13/12 (d3 - d2)^2 + 1/4 (d2 + d3)^2,
//                b2 = 13/12 (d4 - d3)^2 + 1/4 (d4 - 3 d3)^2
//   weights      d_k / (eps + b_k)^2, d = (.1,.6,.3), eps = 1e-6, normalised.
// The same numbers as the textbook form up to rounding (12 b_k and 12 eps are used: a common factor of the three
// (eps + b_k) drops out of the normalised weights), with a fifth fewer fp64 operations.  The three weight divisions and the
// normalisation are folded into one division (div_pos) by multiplying through with the product of the (eps + b_k)^2.
// Every operation is an explicitly rounded intrinsic so that the two cells sharing a face evaluate bit-identical
// fluxes wherever a face is evaluated twice (k_seam): exact conservation of sum phi, R12.
__device__ __forceinline__ double weno5_minus_c(double d1, double d2, double d3, double d4) {
  const double eps12 = 12.0e-6;
  const double s0 = __dsub_rn(d2, d1), t0 = __fma_rn(3.0, d2, -d1);
  const double s1 = __dsub_rn(d3, d2), t1 = __dadd_rn(d2, d3);
  const double s2 = __dsub_rn(d4, d3), t2 = __fma_rn(-3.0, d3, d4);
  const double r0 = __fma_rn(13.0, __dmul_rn(s0, s0), __fma_rn(3.0, __dmul_rn(t0, t0), eps12));  // 12 (eps + b0)
  const double r1 = __fma_rn(13.0, __dmul_rn(s1, s1), __fma_rn(3.0, __dmul_rn(t1, t1), eps12));
  const double r2 = __fma_rn(13.0, __dmul_rn(s2, s2), __fma_rn(3.0, __dmul_rn(t2, t2), eps12));
  const double e0 = __dmul_rn(r0, r0), e1 = __dmul_rn(r1, r1), e2 = __dmul_rn(r2, r2);
  const double m0 = __dmul_rn(e1, e2), m1 = __dmul_rn(e0, e2), m2 = __dmul_rn(e0, e1);  // weights d_k m_k, d = (.1,.6,.3)
  // numerator and denominator both times 5: every constant is then a multiple of 1/2, which the fp64 instructions take as
  // an immediate operand (0.2, 0.6, 1.2 ... need two uniform-register moves each, at every use)
  const double x0 = __fma_rn(2.5, d2, -d1);                   // 5 * 0.1 * 6 (q0 - c)
  const double x1 = __fma_rn(6.0, d3, __dmul_rn(3.0, d2));    // 5 * 0.6 * 6 (q1 - c)
  const double x2 = __fma_rn(6.0, d3, __dmul_rn(-1.5, d4));   // 5 * 0.3 * 6 (q2 - c)
  const double num = __fma_rn(m2, x2, __fma_rn(m1, x1, __dmul_rn(m0, x0)));
  const double den = __fma_rn(9.0, m2, __fma_rn(18.0, m1, __dmul_rn(3.0, m0)));  // 5 * 6 (0.1 m0 + 0.6 m1 + 0.3 m2)
  return div_pos(num, den);
}

// Advective flux through the face between cells L and R = L + e: u_f = (u_L + u_R)/2, upwinded by its sign
// (R12, R29).  pm2..pp3 are phi at L-2, L-1, L, L+1 (= R), L+2, L+3.
__device__ __forceinline__ double face_flux(double uL, double uR, double pm2, double pm1, double p0, double pp1,
                                            double pp2, double pp3) {
  const double uf = __dmul_rn(0.5, __dadd_rn(uL, uR));
  const bool pos = uf >= 0.0;
  const double a = pos ? pm2 : pp3;
  const double b = pos ? pm1 : pp2;
  const double c = pos ? p0 : pp1;
  const double d = pos ? pp1 : p0;
  const double e = pos ? pp2 : pm1;
  const double w = weno5_minus_c(__dsub_rn(b, a), __dsub_rn(c, b), __dsub_rn(d, c), __dsub_rn(e, d));
  return __dmul_rn(uf, __dadd_rn(c, w));
}

}  // namespace acclb
