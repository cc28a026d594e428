// z4c_stencil.cuh -- finite-difference stencils of the Z4c right-hand side on one field at one point.
//
// SURVEY 8(c) items 3-6 (4th-order centred differences, 4th-order upwind along the shift,
// Kreiss-Oliger dissipation), all in DIFFERENCE FORM: the first operation on any sample is a subtraction
// of a neighbouring sample, so round-off scales with the field's variation, not its magnitude.
//   * every operator is evaluated in the canonical operation order of SURVEY 8(c) items 3-6, one rounding per
//     written operation (the library is built with -fmad=false). The only FMAs are 8a-b and
//     16p1-p2, where the product is exact, so the fused and unfused results are bit-identical.
//   * the upwind side is chosen by SELECTING mirrored differences, never by branching: both signs of the
//     shift execute the same instruction stream on mirrored data (bitwise pi-symmetry).
// `Ld` is any callable sample loader: ld(a, k) = u(x + k h e_a), ld2(a, ka, b, kb) = u(x + ka h e_a + kb h e_b).
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
  double beta[3];       // shift at the point
  bool pos[3];          // beta^a >= 0 (reading I: the tie goes to +)
};

__device__ __forceinline__ void make_coef(double h, double sigma, const double (&beta)[3], PointCoef& c) {
  c.inv12h = 1.0 / (12.0 * h);
  c.inv12h2 = 1.0 / ((12.0 * h) * h);
  c.inv144h2 = 1.0 / ((144.0 * h) * h);
  c.kofac = sigma / (64.0 * h);
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    c.pos[a] = beta[a] >= 0.0;
    c.beta[a] = beta[a];
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

template <bool D1, bool D2, class Ld>
__device__ __forceinline__ void field_derivs(const Ld& ld, const PointCoef& c, Stencil& S) {
  const double u0 = ld(0, 0);
  S.u0 = u0;
  double adv[3], q = 0.0;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double m3 = ld(a, -3), m2 = ld(a, -2), m1 = ld(a, -1);
    const double p1 = ld(a, 1), p2 = ld(a, 2), p3 = ld(a, 3);
    if (D1) S.d1[a] = d1_num(m2, m1, p1, p2) * c.inv12h;
    // differences to the centre, shared by D_aa, KO and the upwind stencil
    const double dm1 = m1 - u0, dm2 = m2 - u0, dm3 = m3 - u0;
    const double dp1 = p1 - u0, dp2 = p2 - u0, dp3 = p3 - u0;
    const double s1 = dp1 + dm1, s2 = dp2 + dm2, s3 = dp3 + dm3;      // mirror-pair sums
    if (D2) S.d2[sym(a, a)] = fma(16.0, s1, -s2) * c.inv12h2;         // item 4, diagonal
    const double qa = (s3 - 6.0 * s2) + 15.0 * s1;                    // item 6: (p3 - 6 p2) + 15 p1
    q = (a == 0) ? qa : q + qa;
    // item 5: v_k = u(x + sg k h); numerator ((18 (v1-v0) - 3 (v-1-v0)) - 6 (v2-v0)) + (v3-v0)
    const bool ps = c.pos[a];
    const double w1 = ps ? dp1 : dm1, wm = ps ? dm1 : dp1, w2 = ps ? dp2 : dm2, w3 = ps ? dp3 : dm3;
    const double r = ((18.0 * w1 - 3.0 * wm) - 6.0 * w2) + w3;
    adv[a] = c.beta[a] * ((ps ? r : -r) * c.inv12h);                  // beta^a * ((sg r) / (12 h))
  }
  S.adv = (adv[0] + adv[1]) + adv[2];
  S.ko = q * c.kofac;
  if (D2) {
    // item 4, mixed: D_ab = D_a(D_b u), a < b, inner unscaled difference along the later axis b
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = a + 1; b < 3; ++b) {
        double e[4];
#pragma unroll
        for (int t = 0; t < 4; ++t) {
          const int ka = (t < 2) ? t - 2 : t - 1;   // -2 -1 +1 +2
          e[t] = d1_num(ld.mixed(a, ka, b, -2), ld.mixed(a, ka, b, -1), ld.mixed(a, ka, b, 1),
                        ld.mixed(a, ka, b, 2));
        }
        S.d2[sym(a, b)] = d1_num(e[0], e[1], e[2], e[3]) * c.inv144h2;
      }
  }
}

}  // namespace sacra
