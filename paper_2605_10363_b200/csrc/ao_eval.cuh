// Device evaluation of one contracted Cartesian Gaussian shell at one point (Eq. 2,
// PAPER.md:67).  chi_abc = f_abc (x-Ax)^a (y-Ay)^b (z-Az)^c R(r^2),  R = sum_i cn_i exp(-alpha_i r^2),
// cn_i = coef_i (2 alpha_i/pi)^{3/4} (4 alpha_i)^{l/2} (host, plan.cu), f_abc = 1/sqrt((2a-1)!!(2b-1)!!(2c-1)!!).
// Component order: s | x,y,z | xx,xy,xz,yy,yz,zz.  Gradient: d/dx [x^a R] = a x^{a-1} R + x^{a+1} R2,
// R2 = sum_i (-2 alpha_i) cn_i exp(-alpha_i r^2).
#pragma once
#include "kldi_internal.h"

namespace kldi {

template <bool GRAD>
__device__ __forceinline__ void eval_shell(const ShellTable& T, int s, double px, double py, double pz, double* val,
                                           double* gx, double* gy, double* gz) {
  const int a = T.sh_atom[s];
  const double x = px - T.atom_xyz[3 * a], y = py - T.atom_xyz[3 * a + 1], z = pz - T.atom_xyz[3 * a + 2];
  const double r2 = x * x + y * y + z * z;
  double R = 0.0, R2 = 0.0;
  for (int i = T.sh_prim0[s]; i < T.sh_prim0[s + 1]; ++i) {
    const double al = T.prim_alpha[i];
    const double e = T.prim_cn[i] * exp(-al * r2);
    R += e;
    if (GRAD) R2 -= 2.0 * al * e;
  }
  const int l = T.sh_l[s];
  if (l == 0) {
    val[0] = R;
    if (GRAD) {
      gx[0] = x * R2;
      gy[0] = y * R2;
      gz[0] = z * R2;
    }
  } else if (l == 1) {
    val[0] = x * R;
    val[1] = y * R;
    val[2] = z * R;
    if (GRAD) {
      gx[0] = R + x * x * R2; gy[0] = x * y * R2;     gz[0] = x * z * R2;
      gx[1] = y * x * R2;     gy[1] = R + y * y * R2; gz[1] = y * z * R2;
      gx[2] = z * x * R2;     gy[2] = z * y * R2;     gz[2] = R + z * z * R2;
    }
  } else {
    const double f = 0.57735026918962576451;  // 1/sqrt(3) for xx, yy, zz
    const double Rf = R * f, R2f = R2 * f;
    val[0] = x * x * Rf;
    val[1] = x * y * R;
    val[2] = x * z * R;
    val[3] = y * y * Rf;
    val[4] = y * z * R;
    val[5] = z * z * Rf;
    if (GRAD) {
      // xx
      gx[0] = 2.0 * x * Rf + x * x * x * R2f; gy[0] = x * x * y * R2f;               gz[0] = x * x * z * R2f;
      // xy
      gx[1] = y * R + x * x * y * R2;         gy[1] = x * R + x * y * y * R2;        gz[1] = x * y * z * R2;
      // xz
      gx[2] = z * R + x * x * z * R2;         gy[2] = x * y * z * R2;                gz[2] = x * R + x * z * z * R2;
      // yy
      gx[3] = x * y * y * R2f;                gy[3] = 2.0 * y * Rf + y * y * y * R2f; gz[3] = y * y * z * R2f;
      // yz
      gx[4] = x * y * z * R2;                 gy[4] = z * R + y * y * z * R2;        gz[4] = y * R + y * z * z * R2;
      // zz
      gx[5] = x * z * z * R2f;                gy[5] = y * z * z * R2f;               gz[5] = 2.0 * z * Rf + z * z * z * R2f;
    }
  }
}

// Value-free second derivatives of ONE component (Cartesian powers a, b, c of shell s) at one point, for the GGA nuclear
// gradient: chi = f P(x,y,z) R(r^2), P = x^a y^b z^c, with R1 = sum -2 alpha cn e (d_i R = x_i R1) and
// R2 = sum 4 alpha^2 cn e (d_i R1 = x_i R2):
//     d_i chi     = f [ P_i R + P x_i R1 ]
//     d_i d_j chi = f [ P_ij R + (P_i x_j + P_j x_i) R1 + P (delta_ij R1 + x_i x_j R2) ]
// g[3] = gradient, h[6] = xx, xy, xz, yy, yz, zz.
__device__ __forceinline__ void eval_component_hess(const ShellTable& T, int s, int comp, double px, double py, double pz,
                                                    double (&g)[3], double (&h)[6]) {
  const int at = T.sh_atom[s];
  const double x[3] = {px - T.atom_xyz[3 * at], py - T.atom_xyz[3 * at + 1], pz - T.atom_xyz[3 * at + 2]};
  const double r2 = x[0] * x[0] + x[1] * x[1] + x[2] * x[2];
  double R = 0.0, R1 = 0.0, R2 = 0.0;
  for (int i = T.sh_prim0[s]; i < T.sh_prim0[s + 1]; ++i) {
    const double al = T.prim_alpha[i];
    const double e = T.prim_cn[i] * exp(-al * r2);
    R += e;
    R1 -= 2.0 * al * e;
    R2 += 4.0 * al * al * e;
  }
  const int l = T.sh_l[s];
  int n[3] = {0, 0, 0};  // component order s | x,y,z | xx,xy,xz,yy,yz,zz
  double f = 1.0;
  if (l == 1) {
    n[comp] = 1;
  } else if (l == 2) {
    const int ia = comp < 3 ? 0 : (comp < 5 ? 1 : 2);
    const int ib = comp < 3 ? comp : (comp < 5 ? comp - 2 : 2);
    n[ia] += 1;
    n[ib] += 1;
    if (ia == ib) f = 0.57735026918962576451;
  }
  auto pw = [](double v, int e) { return e <= 0 ? 1.0 : (e == 1 ? v : v * v); };
  // u_d = x_d^{n_d}, first and second derivatives of the monomial factors
  double u[3], u1[3], u2[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    u[d] = pw(x[d], n[d]);
    u1[d] = n[d] == 0 ? 0.0 : n[d] * pw(x[d], n[d] - 1);
    u2[d] = n[d] == 2 ? 2.0 : 0.0;
  }
  const double P = u[0] * u[1] * u[2];
  const double P1[3] = {u1[0] * u[1] * u[2], u[0] * u1[1] * u[2], u[0] * u[1] * u1[2]};
#pragma unroll
  for (int d = 0; d < 3; ++d) g[d] = f * (P1[d] * R + P * x[d] * R1);
  int k = 0;
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = i; j < 3; ++j, ++k) {
      double Pij;
      if (i == j)
        Pij = u2[i] * u[(i + 1) % 3] * u[(i + 2) % 3];
      else
        Pij = u1[i] * u1[j] * u[3 - i - j];
      h[k] = f * (Pij * R + (P1[i] * x[j] + P1[j] * x[i]) * R1 + P * ((i == j ? R1 : 0.0) + x[i] * x[j] * R2));
    }
}

}  // namespace kldi
