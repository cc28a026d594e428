// z4c_point.cuh -- device-side arithmetic of the Z4c right-hand side at one grid point.
//
// Two parts, both FP64 and branch-free across threads:
//   * finite-difference stencils in difference form: written with
//     __dadd_rn/__dmul_rn so that no FMA contraction ever touches them (contraction applied
//     unevenly breaks bitwise pi-symmetry; the difference form keeps round-off at the scale of the field's
//     variation, not its magnitude);
//   * the point-wise algebra (system of Hilditch et al. 2013 cited at PAPER.md:63,
//     gauge Eqs. 6-8).
// Symmetric tensors are stored once (6 components, order xx xy xz yy yz zz).
#pragma once
#include <cuda_runtime.h>

namespace sacra {

constexpr int NF = 25;
constexpr int NG = 3;
enum Field { F_W = 0, F_G = 1, F_KH = 7, F_A = 8, F_GAM = 14, F_TH = 17, F_ALP = 18, F_BET = 19, F_B = 22 };

// symmetric pair (i,j) -> packed index, xx xy xz yy yz zz
__device__ __forceinline__ constexpr int sym(int i, int j) {
  return (i <= j) ? (i * 3 - (i * (i - 1)) / 2 + (j - i)) : (j * 3 - (j * (j - 1)) / 2 + (i - j));
}

struct Coef {          // per-patch stencil scale factors, all computed once per thread in FP64
  double inv12h;       // 1/(12 h)
  double inv12h2;      // 1/(12 h^2)
  double inv144h2;     // 1/(144 h^2)
  double kofac;        // sigma/(64 h)
};

__device__ __forceinline__ Coef make_coef(double h, double sigma) {
  Coef c;
  c.inv12h = 1.0 / __dmul_rn(12.0, h);
  c.inv12h2 = 1.0 / __dmul_rn(__dmul_rn(12.0, h), h);
  c.inv144h2 = 1.0 / __dmul_rn(__dmul_rn(144.0, h), h);
  c.kofac = sigma / __dmul_rn(64.0, h);
  return c;
}

struct Params {        // device copy of sacra_params_t
  double kappa1, kappa2, eta, shift_coef, ko_sigma;
  int lapse_uses_khat;
};

// ---- stencil numerators on already-loaded samples --------------------------------------------------
// item 3: unscaled centred first difference  8 (u+1 - u-1) - (u+2 - u-2)
__device__ __forceinline__ double d1_num(double um2, double um1, double up1, double up2) {
  return __dsub_rn(__dmul_rn(8.0, __dsub_rn(up1, um1)), __dsub_rn(up2, um2));
}
// mirror-pair sums p_k = (u+k - u0) + (u-k - u0), shared by the diagonal second derivative and KO
__device__ __forceinline__ double pair_sum(double um, double u0, double up) {
  return __dadd_rn(__dsub_rn(up, u0), __dsub_rn(um, u0));
}
// item 4: unscaled diagonal second difference 16 p1 - p2
__device__ __forceinline__ double d2_num(double p1, double p2) {
  return __dsub_rn(__dmul_rn(16.0, p1), p2);
}
// item 6: KO numerator along one axis (p3 - 6 p2) + 15 p1
__device__ __forceinline__ double ko_num(double p1, double p2, double p3) {
  return __dadd_rn(__dsub_rn(p3, __dmul_rn(6.0, p2)), __dmul_rn(15.0, p1));
}
// item 5: lopsided upwind numerator; v_k = u(x + sg k h), sg = sign of the shift component (reading I:
// sg = +1 at beta = 0). Returns sg * [((18 (v1-v0) - 3 (v-1-v0)) - 6 (v2-v0)) + (v3-v0)].
__device__ __forceinline__ double up_num(double vm1, double v0, double v1, double v2, double v3,
                                         double sg) {
  double a = __dsub_rn(__dmul_rn(18.0, __dsub_rn(v1, v0)), __dmul_rn(3.0, __dsub_rn(vm1, v0)));
  double b = __dsub_rn(a, __dmul_rn(6.0, __dsub_rn(v2, v0)));
  return __dmul_rn(sg, __dadd_rn(b, __dsub_rn(v3, v0)));
}

// Derivative bundle of one point. Only the entries the algebra uses are ever written.
//   d1 : W, gt(6), K-hat, Gt(3), Theta, alpha, beta(3)            -> slot via d1slot()
//   d2 : W, gt(6), alpha, beta(3), packed xx xy xz yy yz zz        -> slot via d2slot()
struct Derivs {
  double d1[16][3];
  double d2[11][6];
  double adv[NF];
  double ko[NF];
};
__device__ __forceinline__ constexpr int d1slot(int f) {      // -1: no centred first derivative needed
  return (f <= F_KH) ? f : (f < F_GAM) ? -1 : (f <= F_BET + 2) ? (f - 6) : -1;
}
__device__ __forceinline__ constexpr int d2slot(int f) {      // -1: no second derivative needed
  return (f <= F_G + 5) ? f : (f == F_ALP) ? 7 : (f >= F_BET && f < F_BET + 3) ? (8 + f - F_BET) : -1;
}

// ---- items 7-10: the algebra -----------------------------------------------------------------------
// u[25] values at the point, D the derivative bundle, out[25] = RHS + KO. The summation order inside every
// contraction is fixed (index loops in natural order) so that every thread runs the same instruction stream
// (item 13) and the result is reproducible run to run.
__device__ __forceinline__ void z4c_algebra(const double (&u)[NF], const Derivs& D, const Params& P,
                                            double (&out)[NF]) {
  const double half = 0.5, third = 1.0 / 3.0, two3 = 2.0 / 3.0;
  const double W = u[F_W], Kh = u[F_KH], Th = u[F_TH], alp = u[F_ALP];
  const double K = Kh + 2.0 * Th;                                  // item 7
#define G_(i, j) u[F_G + sym(i, j)]
#define A_(i, j) u[F_A + sym(i, j)]

  // true inverse of the conformal metric (item 7; det is not assumed to be 1, reading J)
  const double gxx = G_(0, 0), gxy = G_(0, 1), gxz = G_(0, 2), gyy = G_(1, 1), gyz = G_(1, 2), gzz = G_(2, 2);
  const double det = gxx * (gyy * gzz - gyz * gyz) - gxy * (gxy * gzz - gyz * gxz) + gxz * (gxy * gyz - gyy * gxz);
  double gi[6];
  gi[0] = (gyy * gzz - gyz * gyz) / det;
  gi[1] = (gxz * gyz - gxy * gzz) / det;
  gi[2] = (gxy * gyz - gxz * gyy) / det;
  gi[3] = (gxx * gzz - gxz * gxz) / det;
  gi[4] = (gxy * gxz - gxx * gyz) / det;
  gi[5] = (gxx * gyy - gxy * gxy) / det;
#define GI_(i, j) gi[sym(i, j)]
#define DG_(k, i, j) D.d1[d1slot(F_G + sym(i, j))][k]            /* d_k gt_ij */
#define DDG_(l, m, i, j) D.d2[d2slot(F_G + sym(i, j))][sym(l, m)] /* d_l d_m gt_ij */
#define DW_(k) D.d1[d1slot(F_W)][k]
#define DDW_(i, j) D.d2[d2slot(F_W)][sym(i, j)]
#define DA_(k) D.d1[d1slot(F_ALP)][k]
#define DDA_(i, j) D.d2[d2slot(F_ALP)][sym(i, j)]
#define DB_(k, i) D.d1[d1slot(F_BET + (i))][k]                   /* d_k beta^i */
#define DDB_(k, l, i) D.d2[d2slot(F_BET + (i))][sym(k, l)]        /* d_k d_l beta^i */
#define DGAM_(k, i) D.d1[d1slot(F_GAM + (i))][k]                 /* d_k Gt^i */

  const double divb = (DB_(0, 0) + DB_(1, 1)) + DB_(2, 2);

  // Christoffels: Gl[k][ij] = Gt_kij, Gu[k][ij] = Gt^k_ij, Gd[i] = gt^jk Gt^i_jk
  double Gl[3][6], Gu[3][6], Gd[3];
#pragma unroll
  for (int k = 0; k < 3; ++k)
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = i; j < 3; ++j)
        Gl[k][sym(i, j)] = half * ((DG_(i, k, j) + DG_(j, k, i)) - DG_(k, i, j));
#pragma unroll
  for (int k = 0; k < 3; ++k)
#pragma unroll
    for (int ij = 0; ij < 6; ++ij)
      Gu[k][ij] = (GI_(k, 0) * Gl[0][ij] + GI_(k, 1) * Gl[1][ij]) + GI_(k, 2) * Gl[2][ij];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    double s = 0.0;
#pragma unroll
    for (int j = 0; j < 3; ++j)
#pragma unroll
      for (int k = 0; k < 3; ++k) s += GI_(j, k) * Gu[i][sym(j, k)];
    Gd[i] = s;
  }

  // conformal Ricci tensor Rt_ij (item 7)
  double Rt[6];
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = i; j < 3; ++j) {
      double lap = 0.0;
#pragma unroll
      for (int l = 0; l < 3; ++l)
#pragma unroll
        for (int m = 0; m < 3; ++m) lap += GI_(l, m) * DDG_(l, m, i, j);
      double t2 = 0.0, t3 = 0.0;
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        t2 += G_(k, i) * DGAM_(j, k) + G_(k, j) * DGAM_(i, k);
        t3 += Gd[k] * (Gl[i][sym(j, k)] + Gl[j][sym(i, k)]);
      }
      double t4 = 0.0;
#pragma unroll
      for (int l = 0; l < 3; ++l)
#pragma unroll
        for (int m = 0; m < 3; ++m) {
          double q = 0.0;
#pragma unroll
          for (int k = 0; k < 3; ++k)
            q += (Gu[k][sym(l, i)] * Gl[j][sym(k, m)] + Gu[k][sym(l, j)] * Gl[i][sym(k, m)]) +
                 Gu[k][sym(i, m)] * Gl[k][sym(l, j)];
          t4 += GI_(l, m) * q;
        }
      Rt[sym(i, j)] = ((-half * lap + half * t2) + half * t3) + t4;
    }

  // conformal-factor part: W^2 R_ij and R (item 7)
  double DDW[6];
#pragma unroll
  for (int ij = 0; ij < 6; ++ij) {
    double s = D.d2[d2slot(F_W)][ij];
#pragma unroll
    for (int k = 0; k < 3; ++k) s -= Gu[k][ij] * DW_(k);
    DDW[ij] = s;
  }
  double trDDW = 0.0, dWdW = 0.0, dadW = 0.0;
#pragma unroll
  for (int k = 0; k < 3; ++k)
#pragma unroll
    for (int l = 0; l < 3; ++l) {
      trDDW += GI_(k, l) * DDW[sym(k, l)];
      dWdW += GI_(k, l) * DW_(k) * DW_(l);
    }
#pragma unroll
  for (int k = 0; k < 3; ++k)
#pragma unroll
    for (int l = 0; l < 3; ++l) dadW += GI_(k, l) * DA_(k) * DW_(l);
  double WR[6];
#pragma unroll
  for (int ij = 0; ij < 6; ++ij)
    WR[ij] = W * W * Rt[ij] + (W * (DDW[ij] + u[F_G + ij] * trDDW) - 2.0 * u[F_G + ij] * dWdW);
  double R = 0.0;
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) R += GI_(i, j) * WR[sym(i, j)];

  // W^2 D_i D_j alpha in the physical metric, and D^i D_i alpha (item 7)
  double WDDa[6];
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = i; j < 3; ++j) {
      double s = DDA_(i, j);
#pragma unroll
      for (int k = 0; k < 3; ++k) s -= Gu[k][sym(i, j)] * DA_(k);
      WDDa[sym(i, j)] = W * W * s + W * ((DA_(i) * DW_(j) + DA_(j) * DW_(i)) - G_(i, j) * dadW);
    }
  double lapa = 0.0;
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) lapa += GI_(i, j) * WDDa[sym(i, j)];

  // At^i_j (not symmetric) and At^ij (symmetric up to round-off; stored in full)
  double Aud[3][3], Auu[3][3];
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j)
      Aud[i][j] = (GI_(i, 0) * A_(0, j) + GI_(i, 1) * A_(1, j)) + GI_(i, 2) * A_(2, j);
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j)
      Auu[i][j] = (Aud[i][0] * GI_(0, j) + Aud[i][1] * GI_(1, j)) + Aud[i][2] * GI_(2, j);
  double AA = 0.0;
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) AA += A_(i, j) * Auu[i][j];

  // ---- item 8 ----------------------------------------------------------------------------------------
  double rhs[NF];
  rhs[F_W] = D.adv[F_W] + third * W * (alp * K - divb);
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = i; j < 3; ++j) {
      double s = 0.0;
#pragma unroll
      for (int k = 0; k < 3; ++k) s += G_(i, k) * DB_(j, k) + G_(j, k) * DB_(i, k);
      rhs[F_G + sym(i, j)] = ((-2.0 * alp * A_(i, j) + D.adv[F_G + sym(i, j)]) + s) - two3 * G_(i, j) * divb;
    }
  rhs[F_KH] = ((-lapa + alp * (AA + third * K * K)) + alp * P.kappa1 * (1.0 - P.kappa2) * Th) + D.adv[F_KH];

  double X[6], trX = 0.0;
#pragma unroll
  for (int ij = 0; ij < 6; ++ij) X[ij] = -WDDa[ij] + alp * WR[ij];
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) trX += GI_(i, j) * X[sym(i, j)];
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = i; j < 3; ++j) {
      const double xtf = X[sym(i, j)] - third * G_(i, j) * trX;
      double aa = 0.0, lie = 0.0;
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        aa += A_(i, k) * Aud[k][j];
        lie += A_(i, k) * DB_(j, k) + A_(j, k) * DB_(i, k);
      }
      rhs[F_A + sym(i, j)] =
          (((xtf + alp * (K * A_(i, j) - 2.0 * aa)) + D.adv[F_A + sym(i, j)]) + lie) - two3 * A_(i, j) * divb;
    }

  double gam_noadv[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    double t1 = 0.0, t2 = 0.0, t3 = 0.0, t4 = 0.0, t5 = 0.0, t6 = 0.0, t7 = 0.0;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      t1 += Auu[i][j] * DA_(j);
      t3 += Auu[i][j] * DW_(j);
      t4 += GI_(i, j) * (2.0 * D.d1[d1slot(F_KH)][j] + D.d1[d1slot(F_TH)][j]);
      t7 += Gd[j] * DB_(j, i);
      double dd = 0.0;
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        t2 += Gu[i][sym(j, k)] * Auu[j][k];
        t5 += GI_(j, k) * DDB_(j, k, i);
        dd += DDB_(j, k, k);
      }
      t6 += GI_(i, j) * dd;
    }
    gam_noadv[i] = (((((-2.0 * t1 + 2.0 * alp * ((t2 - 3.0 * t3 / W) - third * t4)) + t5) + third * t6) - t7) +
                    two3 * Gd[i] * divb) -
                   2.0 * alp * P.kappa1 * (u[F_GAM + i] - Gd[i]);
    rhs[F_GAM + i] = gam_noadv[i] + D.adv[F_GAM + i];
  }

  rhs[F_TH] = (half * alp * ((R - AA) + two3 * K * K) - alp * P.kappa1 * (2.0 + P.kappa2) * Th) + D.adv[F_TH];

  // ---- item 9: gauge (Eqs. 6-8) ---------------------------------------------------------------------
  const double Ksrc = P.lapse_uses_khat ? Kh : K;                  // reading C
  rhs[F_ALP] = D.adv[F_ALP] - 2.0 * alp * Ksrc;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    rhs[F_BET + i] = D.adv[F_BET + i] + P.shift_coef * u[F_B + i];
    rhs[F_B + i] = (D.adv[F_B + i] + gam_noadv[i]) - P.eta * u[F_B + i];   // reading H: no KO inside
  }
  // ---- item 10 ------------------------------------------------------------------------------------------
#pragma unroll
  for (int n = 0; n < NF; ++n) out[n] = rhs[n] + D.ko[n];

#undef G_
#undef A_
#undef GI_
#undef DG_
#undef DDG_
#undef DW_
#undef DDW_
#undef DA_
#undef DDA_
#undef DB_
#undef DDB_
#undef DGAM_
}

}  // namespace sacra
