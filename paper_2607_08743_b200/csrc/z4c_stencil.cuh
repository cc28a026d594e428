// z4c_stencil.cuh -- finite-difference stencils of the Z4c right-hand side on one field at one point.
//
// SURVEY 8(c) items 3-6 (4th-order centred differences, 4th-order upwind along the shift,
// Kreiss-Oliger dissipation), all in DIFFERENCE FORM: the first operation on any sample is a subtraction
// of a neighbouring sample, so round-off scales with the field's variation, not its magnitude.
//   * the centred first and second derivatives are evaluated in the canonical operation order of SURVEY 8(c)
//     items 3-4 (the library is built with -fmad=false; the FMAs 8a-b and 16p1-p2 have an exact
//     product, so they are bit-identical to the unfused form): D1, D_aa, D_ab are bit-identical to the oracle.
//   * KO and the upwind stencil use explicit FMA chains (one rounding fewer per term than the oracle).
//   * no data-dependent branch or select anywhere: both signs of the shift execute the same instruction
//     stream on mirrored data (bitwise pi-symmetry).
// `Ld` is the sample loader of one field: ld(a, k) = u(x + k h e_a); publish_e / e_y_x / e_z_x / e_z_y exchange the
// inner first differences of the mixed second derivatives between the threads of a tile (z4c_tile.cuh).
#pragma once
#include <cuda_runtime.h>

namespace sacra {

constexpr int NF = 25;
constexpr int NG = 3;
enum Field { F_W = 0, F_G = 1, F_KH = 7, F_A = 8, F_GAM = 14, F_TH = 17, F_ALP = 18, F_BET = 19, F_B = 22 };

// symmetric pair (i,j) -> packed index, xx xy xz yy yz zz
__host__ __device__ __forceinline__ constexpr int sym(int i, int j) {
  return (i <= j) ? (i * 3 - (i * (i - 1)) / 2 + (j - i)) : (j * 3 - (j * (j - 1)) / 2 + (i - j));
}

struct PointCoef {      // per-thread constants of the derivative stage
  double inv12h;        // 1/(12 h)
  double inv12h2;       // 1/(12 h^2)
  double inv144h2;      // 1/(144 h^2)
  double kofac;         // sigma/(64 h)
  double ba[3];         // beta^a / (24 h)    weight of the antisymmetric part of the upwind stencil
  double bs[3];         // |beta^a| / (24 h)  weight of its symmetric part
};

// per-patch constants of the derivative stage, computed once on the host (IEEE double, the same expressions the
// oracle evaluates: identical bits) instead of five divisions per thread and tile
struct GridCoef {
  double inv12h, inv12h2, inv144h2, inv24h, kofac;
};
__host__ __device__ __forceinline__ GridCoef grid_coef(double h, double sigma) {
  GridCoef g;
  g.inv12h = 1.0 / (12.0 * h);
  g.inv12h2 = 1.0 / ((12.0 * h) * h);
  g.inv144h2 = 1.0 / ((144.0 * h) * h);
  g.inv24h = 1.0 / (24.0 * h);
  g.kofac = sigma / (64.0 * h);
  return g;
}
__device__ __forceinline__ void make_coef(const GridCoef& g, const double (&beta)[3], PointCoef& c) {
  c.inv12h = g.inv12h;
  c.inv12h2 = g.inv12h2;
  c.inv144h2 = g.inv144h2;
  c.kofac = g.kofac;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    c.ba[a] = beta[a] * g.inv24h;
    c.bs[a] = fabs(beta[a]) * g.inv24h;
  }
}

struct Stencil {        // derivative bundle of ONE field at one point
  double u0;
  double d1[3];         // centred D_a u                      (if D1)
  double d2[6];         // centred D_ab u, xx xy xz yy yz zz  (if D2)
  double adv;           // beta^a Dup_a u                      (item 5)
  double ko;            // Q u                                 (item 6)
};

// unscaled centred first difference 8 (u+1 - u-1) - (u+2 - u-2)   (item 3)
__device__ __forceinline__ double d1_num(double um2, double um1, double up1, double up2) {
  return fma(8.0, up1 - um1, -(up2 - um2));
}

// Upwind advection without a data-dependent choice of samples. With v_k = u(x + sg k h), sg = sign(beta^a)
// (the tie beta^a = 0 is immaterial: the term is multiplied by 0), the lopsided stencil of item 5 splits
// exactly into an antisymmetric and a symmetric part,
//   beta Dup u = beta [21 a1 - 6 a2 + a3] / (24 h)  +  |beta| [15 s1 - 6 s2 + s3] / (24 h),
//   a_k = u(+k) - u(-k),   s_k = (u(+k) - u0) + (u(-k) - u0),
// and the symmetric bracket IS the Kreiss-Oliger numerator q_a of item 6. Both signs of the shift run the same
// instruction stream on mirrored data (bitwise pi-symmetry): under x -> -x, a_k -> -a_k
// exactly, s_k -> s_k, beta -> -beta. a_k is one subtraction of two samples, so its round-off scales with the
// field's variation like every other difference here. The oracle evaluates item 5 as written; the two agree
// to a few ulp of the advection term.
// AK = false leaves the advection and KO terms out (the constraint monitor needs only the centred derivatives).
template <bool D1, bool D2, bool AK = true, class Ld>
__device__ __forceinline__ void field_derivs(const Ld& ld, const PointCoef& c, Stencil& S) {
  static_assert(D1 || !D2, "the mixed second derivatives reuse the numerators of D_y, D_z");
  const double u0 = ld(0, 0);
  S.u0 = u0;
  double adv = 0.0, q = 0.0, num[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double m2 = ld(a, -2), m1 = ld(a, -1), p1 = ld(a, 1), p2 = ld(a, 2);
    const double a1 = p1 - m1, a2 = p2 - m2;                          // antisymmetric differences
    if (!AK) {
      if (D1) {
        num[a] = fma(8.0, a1, -a2);
        S.d1[a] = num[a] * c.inv12h;
      }
      if (D2) S.d2[sym(a, a)] = fma(16.0, (p1 - u0) + (m1 - u0), -((p2 - u0) + (m2 - u0))) * c.inv12h2;
      continue;
    }
    const double m3 = ld(a, -3), p3 = ld(a, 3);
    const double a3 = p3 - m3;
    if (D1) {
      num[a] = fma(8.0, a1, -a2);                                     // item 3 (8 a1 is exact)
      S.d1[a] = num[a] * c.inv12h;
    }
    double qa;                                                        // item 6: s3 - 6 s2 + 15 s1
    if (D2) {
      // differences to the centre, shared by D_aa, KO and the symmetric part of the upwind stencil: the second
      // derivative of a field that is 1 + O(1e-3) must not see the round-off of the field's magnitude
      const double s1 = (p1 - u0) + (m1 - u0), s2 = (p2 - u0) + (m2 - u0), s3 = (p3 - u0) + (m3 - u0);
      S.d2[sym(a, a)] = fma(16.0, s1, -s2) * c.inv12h2;               // item 4, diagonal (16 s1 is exact)
      qa = fma(15.0, s1, fma(-6.0, s2, s3));
    } else {
      // fields without second derivatives (K-hat, Theta, At_ij, Gt^i, B^i): the bracket only feeds the KO and
      // upwind terms, a few ulp of |u| sigma / (64 h) is far below the tolerance; 6 operations instead of 11
      qa = fma(-20.0, u0, fma(15.0, p1 + m1, fma(-6.0, p2 + m2, p3 + m3)));
    }
    q = (a == 0) ? qa : q + qa;
    const double aa = fma(21.0, a1, fma(-6.0, a2, a3));               // item 5, antisymmetric bracket
    adv = (a == 0) ? fma(c.bs[0], qa, c.ba[0] * aa) : fma(c.bs[a], qa, fma(c.ba[a], aa, adv));
  }
  S.adv = adv;
  S.ko = q * c.kofac;
  if (D2) {
    // item 4, mixed: D_ab = D_a(e_b), a < b, e_b = unscaled inner difference along the later axis b
    ld.publish_e(num[1], num[2]);
    S.d2[sym(0, 1)] = d1_num(ld.e_y_x(-2), ld.e_y_x(-1), ld.e_y_x(1), ld.e_y_x(2)) * c.inv144h2;
    S.d2[sym(0, 2)] = d1_num(ld.e_z_x(-2), ld.e_z_x(-1), ld.e_z_x(1), ld.e_z_x(2)) * c.inv144h2;
    S.d2[sym(1, 2)] = d1_num(ld.e_z_y(-2), ld.e_z_y(-1), ld.e_z_y(1), ld.e_z_y(2)) * c.inv144h2;
  }
}

}  // namespace sacra
