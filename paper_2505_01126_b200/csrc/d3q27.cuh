// D3Q27 lattice and the regularized collision algebra, device side (sm_100a).
//
// Written from /root/reference/PAPER.md (arXiv 2505.01126); readings Rnn are listed in DESIGN.md section 2.
// This header is part of the CUDA product path; it shares nothing with oracle/.
//
//   velocity set (R1): c_i in {-1,0,1}^3, i = (cx+1) + 3 (cy+1) + 9 (cz+1), rest = 13,
//   opposite(i) = 26 - i, w = 8/27 | 2/27 | 1/54 | 1/216, c_s^2 = 1/3.
#pragma once

namespace acclb {

constexpr int Q = 27;

__host__ __device__ constexpr int cx_of(int i) { return i % 3 - 1; }
__host__ __device__ constexpr int cy_of(int i) { return (i / 3) % 3 - 1; }
__host__ __device__ constexpr int cz_of(int i) { return i / 9 - 1; }
__host__ __device__ constexpr int nnz_of(int i) {
  return (cx_of(i) != 0) + (cy_of(i) != 0) + (cz_of(i) != 0);
}
__host__ __device__ constexpr double w_of(int i) {
  return nnz_of(i) == 0 ? 8.0 / 27.0 : nnz_of(i) == 1 ? 2.0 / 27.0 : nnz_of(i) == 2 ? 1.0 / 54.0 : 1.0 / 216.0;
}

// The ten raw moments of the populations at a node (row a2):
//   p* = sum f_i, m_a = sum f_i c_ia, Pi_ab = sum f_i c_ia c_ib  (Pi order: xx, yy, zz, xy, xz, yz).
// Evaluated on the 13 opposite pairs: s = f_i + f_j, d = f_i - f_j (j = 26 - i) so that each product with a
// lattice constant folds into an add or a subtract at compile time.
struct Moments {
  double p, m[3], Pi[6];
};

template <class F>
__device__ __forceinline__ void moments_of(F f_of, Moments& M) {  // f_of(i) = f_i, each i asked for once
  double p = f_of(13);
  double mx = 0.0, my = 0.0, mz = 0.0;
  double pxx = 0.0, pyy = 0.0, pzz = 0.0, pxy = 0.0, pxz = 0.0, pyz = 0.0;
#pragma unroll
  for (int i = 0; i < 13; ++i) {
    const int cx = cx_of(i), cy = cy_of(i), cz = cz_of(i);
    const double fa = f_of(i), fb = f_of(26 - i);
    const double s = fa + fb;
    const double d = fa - fb;
    p += s;
    if (cx == 1) mx += d;
    if (cx == -1) mx -= d;
    if (cy == 1) my += d;
    if (cy == -1) my -= d;
    if (cz == 1) mz += d;
    if (cz == -1) mz -= d;
    if (cx != 0) pxx += s;
    if (cy != 0) pyy += s;
    if (cz != 0) pzz += s;
    if (cx * cy == 1) pxy += s;
    if (cx * cy == -1) pxy -= s;
    if (cx * cz == 1) pxz += s;
    if (cx * cz == -1) pxz -= s;
    if (cy * cz == 1) pyz += s;
    if (cy * cz == -1) pyz -= s;
  }
  M.p = p;
  M.m[0] = mx; M.m[1] = my; M.m[2] = mz;
  M.Pi[0] = pxx; M.Pi[1] = pyy; M.Pi[2] = pzz; M.Pi[3] = pxy; M.Pi[4] = pxz; M.Pi[5] = pyz;
}

__device__ __forceinline__ void moments_of(const double (&f)[Q], Moments& M) {
  moments_of([&](int i) { return f[i]; }, M);
}

// Second-order Hermite-space population
//   out_i = w_i [ p + c_i.U / cs2 + H_i,ab T_ab / (2 cs4) ],   H_i,ab = c_ia c_ib - cs2 delta_ab
// With (p, U, T) = (p*, u + A/2, uu + (1-omega) a + (uA + Au)/2) this is Eq. 6:
//   f_i^eq(p*,u) + (1-omega) w_i H_i:a / (2 cs4) + S_i(u,A)/2, because the Guo term of Eq. 5 is
//   S_i = w_i [ c_i.A / cs2 + H_i:(uA + Au) / (2 cs4) ].
// With (p, U, T) = (p*, u - A/2, uu - (uA + Au)/2) it is the initial state f^eq - S/2 (R15).
__device__ __forceinline__ void hermite2_populations(double p, const double (&U)[3], const double (&T)[6],
                                                     double (&out)[Q]) {
  const double trT = T[0] + T[1] + T[2];
  const double e0 = p - 1.5 * trT;  // p - (cs2 trT) / (2 cs4)
  out[13] = w_of(13) * e0;
#pragma unroll
  for (int i = 0; i < 13; ++i) {
    const int cx = cx_of(i), cy = cy_of(i), cz = cz_of(i);
    double cct = 0.0;  // c c : T
    if (cx != 0) cct += T[0];
    if (cy != 0) cct += T[1];
    if (cz != 0) cct += T[2];
    double cross = 0.0;
    if (cx * cy == 1) cross += T[3];
    if (cx * cy == -1) cross -= T[3];
    if (cx * cz == 1) cross += T[4];
    if (cx * cz == -1) cross -= T[4];
    if (cy * cz == 1) cross += T[5];
    if (cy * cz == -1) cross -= T[5];
    cct += 2.0 * cross;
    double cu = 0.0;
    if (cx == 1) cu += U[0];
    if (cx == -1) cu -= U[0];
    if (cy == 1) cu += U[1];
    if (cy == -1) cu -= U[1];
    if (cz == 1) cu += U[2];
    if (cz == -1) cu -= U[2];
    const double even = w_of(i) * (e0 + 4.5 * cct);
    const double odd = (3.0 * w_of(i)) * cu;
    out[i] = even + odd;
    out[26 - i] = even - odd;
  }
}

}  // namespace acclb
