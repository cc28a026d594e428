// z4c_constraints.cuh -- Hamiltonian and momentum constraints at one point.
//
// PAPER.md:182-192, Eqs. 20-21, vacuum:  H = R + K^2 - K_ij K^ij ,  M^i = D_j (K^ij - gamma^ij K), with R and D_j
// those of the physical metric gamma_ij = gt_ij / W^2 and K_ij = (At_ij + gt_ij K / 3) / W^2, K = K-hat + 2 Theta
// (Eqs. 1-4; item 7). Evaluated in the CONFORMAL variables (the oracle goes through the physical
// metric instead), with no assumption det gt = 1 or tr At = 0:
//   Rt    = gt^ij ( d_k Gt^k_ij - d_j Gt^k_ik + Gt^k_kl Gt^l_ij - Gt^k_jl Gt^l_ik )      Ricci scalar of gt_ij
//   R     = W^2 Rt + 4 W Dt^i Dt_i W - 6 Dt^i W Dt_i W                                    (gamma = W^-2 gt, 3 dimensions)
//   B_ij  = At_ij + gt_ij K / 3 = W^2 K_ij ;   K_ij K^ij = gt^ia gt^jb B_ij B_ab
//   M^i   = W^2 { gt^ia gt^jb [ Dt_j B_ab - 2 w_j B_ab - C^c_ja B_cb - C^c_jb B_ac ] - gt^ij d_j K },
//           w_j = d_j W / W,  C^c_ja = -( delta^c_j w_a + delta^c_a w_j - gt_ja gt^cd w_d )   (Gamma - Gt)
// Fields are streamed one at a time like in z4c_fused.cuh (ConStream order: W, gt_ij, K-hat, Theta, At_ij); only centred
// derivatives are needed (no advection, no KO). A diagnostic: written for clarity, every thread runs the same
// instruction stream.
#pragma once
#include "z4c_stencil.cuh"
#include "z4c_tile.cuh"

namespace sacra {

template <class Src, class Emit>
__device__ __forceinline__ void constraints_point(const Src& src, const GridCoef& gc, Emit& emit) {
  Stencil S;
  PointCoef pc;
  {
    const double zero[3] = {0.0, 0.0, 0.0};
    make_coef(gc, zero, pc);
  }
  // ---- centre values first (Tensor Memory strip): metric, its inverse, K, B_ij = At_ij + gt_ij K / 3 ----------------
  double g[6], gi[6], A[6], Kh, Th;
  {
    using namespace tmem;
    Pack4 p0, p8, p12, p16;
    Pack2 p4, p20;
    ld4(src.strip(0), p0); ld2(src.strip(4), p4); ld4(src.strip(8), p8); ld4(src.strip(12), p12);
    ld4(src.strip(16), p16); ld2(src.strip(20), p20);
    wait_ld(p0, p4, p8, p12, p16, p20);
    g[0] = p0.get(0); g[1] = p0.get(1); g[2] = p0.get(2); g[3] = p0.get(3); g[4] = p4.get(0); g[5] = p4.get(1);
    Kh = p8.get(3); Th = p12.get(3);
    A[0] = p16.get(0); A[1] = p16.get(1); A[2] = p16.get(2); A[3] = p16.get(3); A[4] = p20.get(0); A[5] = p20.get(1);
  }
  {
    const double gxx = g[0], gxy = g[1], gxz = g[2], gyy = g[3], gyz = g[4], gzz = g[5];
    const double det = (gxx * (gyy * gzz - gyz * gyz) - gxy * (gxy * gzz - gyz * gxz)) + gxz * (gxy * gyz - gyy * gxz);
    const double rdet = 1.0 / det;
    gi[0] = (gyy * gzz - gyz * gyz) * rdet;
    gi[1] = (gxz * gyz - gxy * gzz) * rdet;
    gi[2] = (gxy * gyz - gxz * gyy) * rdet;
    gi[3] = (gxx * gzz - gxz * gxz) * rdet;
    gi[4] = (gxy * gxz - gxx * gyz) * rdet;
    gi[5] = (gxx * gyy - gxy * gxy) * rdet;
  }
  const double K = Kh + 2.0 * Th;
  double B[6];
#pragma unroll
  for (int n = 0; n < 6; ++n) B[n] = fma(g[n], K * (1.0 / 3.0), A[n]);

  // ---- derivatives, field by field; second derivatives of gt_ij and the gradient of B_ij are folded at once -------
  // the derivatives that are only needed at the very end (d_k W, d_i d_j W, d_k gt_ij) wait in the Tensor Memory
  // strip (slots of z4c_tile.cuh: PK_DB 12 doubles, PK_DG 6 groups of 4), not in registers
  using namespace tmem;
  field_derivs<true, true, false>(src.template field<F_W>(), pc, S);
  const double W = S.u0;
  st4(src.strip(PK_DB), S.d1[0], S.d1[1], S.d1[2], S.d2[0]);
  st4(src.strip(PK_DB + 4), S.d2[1], S.d2[2], S.d2[3], S.d2[4]);
  st1(src.strip(PK_DB + 8), S.d2[5]);

  // second-derivative part of the Ricci scalar of gt:  gt^ij gt^kl ( d_k d_i gt_lj - d_k d_l gt_ij ); the field
  // gt_ab contributes  m_ab [ (gt^.a)^T D2 (gt^.b) - gt^ab tr(gt^-1 D2) ],  m_ab = 1 (a = b) or 2
  double R2 = 0.0;
#define GT_FIELD(A, Bx)                                                                             \
  {                                                                                                 \
    constexpr int N = sym(A, Bx);                                                                   \
    field_derivs<true, true, false>(src.template field<F_G + N>(), pc, S);                          \
    st4(src.strip(PK_DG + 4 * N), S.d1[0], S.d1[1], S.d1[2], 0.0);                                  \
    double q = 0.0, tr = 0.0;                                                                       \
    _Pragma("unroll") for (int i = 0; i < 3; ++i)                                                   \
      _Pragma("unroll") for (int k = 0; k < 3; ++k) {                                               \
        q = fma(gi[sym(i, A)] * gi[sym(k, Bx)], S.d2[sym(i, k)], q);                                \
        tr = fma(gi[sym(i, k)], S.d2[sym(i, k)], tr);                                               \
      }                                                                                             \
    R2 += (A == Bx ? 1.0 : 2.0) * (q - gi[N] * tr);                                                 \
  }
  GT_FIELD(0, 0) GT_FIELD(0, 1) GT_FIELD(0, 2) GT_FIELD(1, 1) GT_FIELD(1, 2) GT_FIELD(2, 2)
#undef GT_FIELD

  wait_st();            // the parked derivatives are read back from here on
  double dK[3];
  field_derivs<true, false, false>(src.template field<F_KH>(), pc, S);
#pragma unroll
  for (int k = 0; k < 3; ++k) dK[k] = S.d1[k];
  field_derivs<true, false, false>(src.template field<F_TH>(), pc, S);
#pragma unroll
  for (int k = 0; k < 3; ++k) dK[k] += 2.0 * S.d1[k];

  // gradient part of the momentum constraint:  gt^ia gt^jb d_j B_ab ; the field B_ab contributes
  // gt^ia v_b + [a != b] gt^ib v_a  with  v_c = gt^jc d_j B_ab
  double M[3] = {0.0, 0.0, 0.0};
#define AT_FIELD(A, Bx)                                                                             \
  {                                                                                                 \
    constexpr int N = sym(A, Bx);                                                                   \
    Pack4 dgn;                                                                                      \
    ld4(src.strip(PK_DG + 4 * N), dgn);                                                             \
    field_derivs<true, false, false>(src.template field<F_A + N>(), pc, S);                         \
    wait_ld(dgn);                                                                                   \
    double dBn[3];                                                                                  \
    _Pragma("unroll") for (int k = 0; k < 3; ++k) dBn[k] = fma(fma(dgn.get(k), K, g[N] * dK[k]), 1.0 / 3.0, S.d1[k]); \
    const double va = (gi[sym(0, A)] * dBn[0] + gi[sym(1, A)] * dBn[1]) + gi[sym(2, A)] * dBn[2];   \
    const double vb = (gi[sym(0, Bx)] * dBn[0] + gi[sym(1, Bx)] * dBn[1]) + gi[sym(2, Bx)] * dBn[2]; \
    _Pragma("unroll") for (int i = 0; i < 3; ++i)                                                   \
      M[i] += (A == Bx) ? gi[sym(i, A)] * va : (gi[sym(i, A)] * vb + gi[sym(i, Bx)] * va);          \
  }
  AT_FIELD(0, 0) AT_FIELD(0, 1) AT_FIELD(0, 2) AT_FIELD(1, 1) AT_FIELD(1, 2) AT_FIELD(2, 2)
#undef AT_FIELD

  // ---- the parked derivatives come back ----------------------------------------------------------------------------
  double dg[3][6], dW[3], ddW[6];
  {
    Pack4 q[6], w0, w4;
    Pack1 w8;
#pragma unroll
    for (int n = 0; n < 6; ++n) ld4(src.strip(PK_DG + 4 * n), q[n]);
    ld4(src.strip(PK_DB), w0); ld4(src.strip(PK_DB + 4), w4); ld1(src.strip(PK_DB + 8), w8);
    wait_ld(q[0], q[1], q[2], q[3], q[4], q[5], w0, w4, w8);
#pragma unroll
    for (int n = 0; n < 6; ++n)
#pragma unroll
      for (int k = 0; k < 3; ++k) dg[k][n] = q[n].get(k);
    dW[0] = w0.get(0); dW[1] = w0.get(1); dW[2] = w0.get(2);
    ddW[0] = w0.get(3); ddW[1] = w4.get(0); ddW[2] = w4.get(1); ddW[3] = w4.get(2); ddW[4] = w4.get(3); ddW[5] = w8.get(0);
  }
  // ---- gradient of the inverse conformal metric: d_l gt^ij = -(gt^-1 d_l gt gt^-1)^ij, two 3 x 3 products per l -------
  double dgi[3][6];
#pragma unroll
  for (int l = 0; l < 3; ++l) {
    double t[3][3];                   // t[i][b] = gt^ia d_l gt_ab
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int bb = 0; bb < 3; ++bb)
        t[i][bb] = fma(gi[sym(i, 2)], dg[l][sym(2, bb)], fma(gi[sym(i, 1)], dg[l][sym(1, bb)], gi[sym(i, 0)] * dg[l][sym(0, bb)]));
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = i; j < 3; ++j)
        dgi[l][sym(i, j)] = -fma(t[i][2], gi[sym(2, j)], fma(t[i][1], gi[sym(1, j)], t[i][0] * gi[sym(0, j)]));
  }
  // ---- Christoffel symbols of gt: Gl[c][ij] first kind, Gu[k][ij] second kind -----------------------------------
  double Gl[3][6], Gu[3][6];
#pragma unroll
  for (int c = 0; c < 3; ++c)
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = i; j < 3; ++j) Gl[c][sym(i, j)] = 0.5 * ((dg[i][sym(c, j)] + dg[j][sym(c, i)]) - dg[c][sym(i, j)]);
#pragma unroll
  for (int k = 0; k < 3; ++k)
#pragma unroll
    for (int n = 0; n < 6; ++n) Gu[k][n] = (gi[sym(k, 0)] * Gl[0][n] + gi[sym(k, 1)] * Gl[1][n]) + gi[sym(k, 2)] * Gl[2][n];

  // ---- Ricci scalar of gt: the folded second-derivative part + the first-derivative terms of
  //      gt^ij ( d_k Gt^k_ij - d_j Gt^k_ik + Gt^k_kl Gt^l_ij - Gt^k_jl Gt^l_ik ),  d gt^kl Gt_l,ij standing for the
  //      part of d Gt^k_ij without second derivatives. Contracted intermediates instead of the four-fold loop:
  //        a_l = d_k gt^kl,  c_l = Gt^k_kl                     ->  sum_l (a_l + ...) of  gt^ij Gt_l,ij  and  gt^ij Gt^l_ij
  //        P[i][k][l] = gt^ij d_j gt^kl,  H[i][k][l] = gt^ij Gt^k_jl   ->  - P[i][k][l] Gt_l,ik  -  H[i][k][l] Gt^l_ik
  double Rt = R2;
  {
    double trl[3], tru[3];            // gt^ij Gt_l,ij ,  gt^ij Gt^l_ij
#pragma unroll
    for (int l = 0; l < 3; ++l) {
      double d = fma(gi[5], Gl[l][5], fma(gi[3], Gl[l][3], gi[0] * Gl[l][0]));
      double o = fma(gi[4], Gl[l][4], fma(gi[2], Gl[l][2], gi[1] * Gl[l][1]));
      trl[l] = fma(2.0, o, d);
      d = fma(gi[5], Gu[l][5], fma(gi[3], Gu[l][3], gi[0] * Gu[l][0]));
      o = fma(gi[4], Gu[l][4], fma(gi[2], Gu[l][2], gi[1] * Gu[l][1]));
      tru[l] = fma(2.0, o, d);
    }
#pragma unroll
    for (int l = 0; l < 3; ++l) {
      const double al = (dgi[0][sym(0, l)] + dgi[1][sym(1, l)]) + dgi[2][sym(2, l)];
      const double cl = (Gu[0][sym(0, l)] + Gu[1][sym(1, l)]) + Gu[2][sym(2, l)];
      Rt = fma(al, trl[l], fma(cl, tru[l], Rt));
    }
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int k = 0; k < 3; ++k)
#pragma unroll
        for (int l = 0; l < 3; ++l) {
          const double Pikl = fma(gi[sym(i, 2)], dgi[2][sym(k, l)], fma(gi[sym(i, 1)], dgi[1][sym(k, l)], gi[sym(i, 0)] * dgi[0][sym(k, l)]));
          const double Hikl = fma(gi[sym(i, 2)], Gu[k][sym(2, l)], fma(gi[sym(i, 1)], Gu[k][sym(1, l)], gi[sym(i, 0)] * Gu[k][sym(0, l)]));
          Rt = fma(-Pikl, Gl[l][sym(i, k)], fma(-Hikl, Gu[l][sym(i, k)], Rt));
        }
  }
  // ---- conformal factor: R = W^2 Rt + 4 W Dt^2 W - 6 |Dt W|^2 -----------------------------------------------------
  double lapW = 0.0, dWdW = 0.0;
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      const int n = sym(i, j);
      lapW += gi[n] * (((ddW[n] - Gu[0][n] * dW[0]) - Gu[1][n] * dW[1]) - Gu[2][n] * dW[2]);
      dWdW += gi[n] * dW[i] * dW[j];
    }
  const double R = W * W * Rt + 4.0 * W * lapW - 6.0 * dWdW;
  // ---- K_ij K^ij = gt^ia gt^jb B_ij B_ab -----------------------------------------------------------------------------
  double Bu[3][3];                    // B^i_b = gt^ia B_ab
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int b = 0; b < 3; ++b)
      Bu[i][b] = (gi[sym(i, 0)] * B[sym(0, b)] + gi[sym(i, 1)] * B[sym(1, b)]) + gi[sym(i, 2)] * B[sym(2, b)];
  double BB = 0.0;
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) BB += Bu[i][j] * Bu[j][i];
  emit.template put<0>(R + K * K - BB, 0.0);

  // ---- momentum constraint ------------------------------------------------------------------------------------------
  double w[3], wu[3];                 // w_j = d_j W / W, w^c = gt^cd w_d
#pragma unroll
  for (int j = 0; j < 3; ++j) w[j] = dW[j] * (1.0 / W);
#pragma unroll
  for (int c = 0; c < 3; ++c) wu[c] = (gi[sym(c, 0)] * w[0] + gi[sym(c, 1)] * w[1]) + gi[sym(c, 2)] * w[2];
  // full connection Gamma^c_ja = Gt^c_ja + C^c_ja ,  C^c_ja = -( delta^c_j w_a + delta^c_a w_j - gt_ja w^c ), formed once;
  // cov_jab = -2 w_j B_ab - Gamma^c_ja B_cb - Gamma^c_jb B_ac (the gradient d_j B_ab is already in M);
  // M^i += gt^ia ( gt^jb cov_jab ): contracted over (j, b) first
  double Gf[3][6];
#pragma unroll
  for (int c = 0; c < 3; ++c)
#pragma unroll
    for (int j = 0; j < 3; ++j)
#pragma unroll
      for (int a = j; a < 3; ++a)
        Gf[c][sym(j, a)] = Gu[c][sym(j, a)] - ((((c == j) ? w[a] : 0.0) + ((c == a) ? w[j] : 0.0)) - g[sym(j, a)] * wu[c]);
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    double va = 0.0;                  // gt^jb cov_jab
#pragma unroll
    for (int j = 0; j < 3; ++j)
#pragma unroll
      for (int b = 0; b < 3; ++b) {
        double cov = -2.0 * w[j] * B[sym(a, b)];
#pragma unroll
        for (int c = 0; c < 3; ++c) cov = fma(-Gf[c][sym(j, a)], B[sym(c, b)], fma(-Gf[c][sym(j, b)], B[sym(a, c)], cov));
        va = fma(gi[sym(j, b)], cov, va);
      }
#pragma unroll
    for (int i = 0; i < 3; ++i) M[i] = fma(gi[sym(i, a)], va, M[i]);
  }
#pragma unroll
  for (int i = 0; i < 3; ++i) M[i] -= (gi[sym(i, 0)] * dK[0] + gi[sym(i, 1)] * dK[1]) + gi[sym(i, 2)] * dK[2];
  emit.template put<1>(W * W * M[0], 0.0);
  emit.template put<2>(W * W * M[1], 0.0);
  emit.template put<3>(W * W * M[2], 0.0);
}

}  // namespace sacra
