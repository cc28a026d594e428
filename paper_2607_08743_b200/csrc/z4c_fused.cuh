// z4c_fused.cuh -- the Z4c right-hand side at one point, evaluated FIELD BY FIELD.
//
// SURVEY 8(c) items 7-10 (system of Hilditch et al. 2013 cited at PAPER.md:63, written in W; gauge Eqs. 6-8,
// PAPER.md:65-71). The derivatives of each field are folded into a small set of running tensors as soon as
// they exist, so that far fewer than the ~190 FP64 values of a one-shot evaluation are live at any time. Each
// field's neighbourhood is visited exactly once and its RHS leaves the thread (emit) as soon as it is complete.
// Order of the fields:
//     beta^i -> Gt^i -> gt_ij -> (Christoffels) -> W -> alpha -> K-hat -> Theta -> (Gt^i out) -> B^i -> At_ij
//
// Numerics policy: -fmad=false. The RHS of the O(1) fields (W, gt_ij, alpha, beta^i) is
// assembled in the oracle's index order, one rounding per operation. Blocks that only feed K-hat, Theta, At_ij,
// Gt^i, B^i use FMA chains and regrouped contractions: the symmetric contractions gi^lm t_lm, the quadratic
// Christoffel block of the conformal Ricci tensor and the running sum of the Gt^i RHS.
// Every thread runs the same instruction stream (no data-dependent branch), which keeps the result bitwise
// pi-symmetric.
//
// `Src` provides   src.derivs<F, D1, D2>(pc, S) -> the derivative bundle S of field F (field_derivs() on its tile,
//                                                  or a bundle computed by the derivative warps)
//                  src.centre(F)   -> value of field F at the point
// `Emit` provides  emit.put<F>(k)  -> consumes the finished RHS value k of field F (KO included)
#pragma once
#include "z4c_stencil.cuh"

namespace sacra {

struct Params {        // device copy of sacra_params_t
  double kappa1, kappa2, eta, shift_coef, ko_sigma;
  int lapse_uses_khat;
};

// contraction gi^lm t_lm of two symmetric tensors (packed): diagonal + 2 x off-diagonal, FMA chains. Every use
// feeds the RHS of K-hat, Theta, At_ij or Gt^i only -- fields whose state is << 1, where a last-bit difference from
// the oracle's index-order sum cannot flip the rounding of an O(1) stage input.
__device__ __forceinline__ double sum9(const double (&gi)[6], const double (&t)[6]) {
  const double d = fma(gi[5], t[5], fma(gi[3], t[3], gi[0] * t[0]));
  const double o = fma(gi[4], t[4], fma(gi[2], t[2], gi[1] * t[1]));
  return fma(2.0, o, d);
}
// sum_j m[i][j] v[j] in index order, m symmetric packed
__device__ __forceinline__ double row3(const double (&m)[6], int i, const double (&v)[3]) {
  return (m[sym(i, 0)] * v[0] + m[sym(i, 1)] * v[1]) + m[sym(i, 2)] * v[2];
}
// FMA contraction of two packed symmetric tensors (used only in the two relaxed blocks)
__device__ __forceinline__ double tr_fma(const double (&a)[6], const double (&b)[6]) {
  const double d = fma(a[5], b[5], fma(a[3], b[3], a[0] * b[0]));
  const double o = fma(a[4], b[4], fma(a[2], b[2], a[1] * b[1]));
  return fma(2.0, o, d);
}

template <class Src, class Emit>
__device__ __forceinline__ void z4c_point(const Src& src, const Params& P, double h, Emit& emit) {
  const double half = 0.5, third = 1.0 / 3.0, two3 = 2.0 / 3.0;
  Stencil S;
  PointCoef pc;
  {
    const double beta[3] = {src.centre(F_BET), src.centre(F_BET + 1), src.centre(F_BET + 2)};
    make_coef(h, P.ko_sigma, beta, pc);
  }

  // ---- centre values and the true inverse conformal metric (item 7; det gt is not assumed to be 1) ------
  double g[6], gi[6];
#pragma unroll
  for (int n = 0; n < 6; ++n) g[n] = src.centre(F_G + n);
  {
    const double gxx = g[0], gxy = g[1], gxz = g[2], gyy = g[3], gyz = g[4], gzz = g[5];
    const double det = (gxx * (gyy * gzz - gyz * gyz) - gxy * (gxy * gzz - gyz * gxz)) + gxz * (gxy * gyz - gyy * gxz);
    gi[0] = (gyy * gzz - gyz * gyz) / det;
    gi[1] = (gxz * gyz - gxy * gzz) / det;
    gi[2] = (gxy * gyz - gxz * gyy) / det;
    gi[3] = (gxx * gzz - gxz * gxz) / det;
    gi[4] = (gxy * gxz - gxx * gyz) / det;
    gi[5] = (gxx * gyy - gxy * gxy) / det;
  }
  const double W = src.centre(F_W), alp = src.centre(F_ALP), Kh = src.centre(F_KH), Th = src.centre(F_TH);
  const double K = Kh + 2.0 * Th;                                        // item 7: K = K-hat + 2 Theta

  double Auu[3][3], AA;   // At^ij and At_ij At^ij: formed at the Christoffel block, where they are first needed

  // ---- beta^i: d_k beta^i; gt^jk d_j d_k beta^i; d_j d_k beta^k; RHS of beta^i (Eq. 7) -------------------
  double db[3][3];      // db[k][i] = d_k beta^i
  double gr[3];         // running RHS of Gt^i without advection (item 8)      [relaxed running sum]
  double dd[3];         // d_j (d_k beta^k)
#define BETA_FIELD(I)                                                                              \
  {                                                                                                \
    src.template derivs<F_BET + I, true, true>(pc, S);                              \
    db[0][I] = S.d1[0]; db[1][I] = S.d1[1]; db[2][I] = S.d1[2];                                    \
    gr[I] = sum9(gi, S.d2);                                                                        \
    if (I == 0) { dd[0] = S.d2[sym(0, 0)]; dd[1] = S.d2[sym(1, 0)]; dd[2] = S.d2[sym(2, 0)]; }     \
    else { dd[0] += S.d2[sym(0, I)]; dd[1] += S.d2[sym(1, I)]; dd[2] += S.d2[sym(2, I)]; }         \
    emit.template put<F_BET + I>((S.adv + P.shift_coef * src.centre(F_B + I)) + S.ko);                          \
  }
  BETA_FIELD(0) BETA_FIELD(1) BETA_FIELD(2)
#undef BETA_FIELD
  const double divb = (db[0][0] + db[1][1]) + db[2][2];
#pragma unroll
  for (int i = 0; i < 3; ++i) gr[i] = fma(third, row3(gi, i, dd), gr[i]);

  // ---- Gt^i: t2_ij = sum_k (gt_ki d_j Gt^k + gt_kj d_i Gt^k); advection and KO of Gt^i kept -------------
  double Rt[6];         // t2_ij, then Rt_ij, then W^2 R_ij, then X_ij
  double advG[3], koG[3];
#define GAM_FIELD(Kx)                                                                              \
  {                                                                                                \
    src.template derivs<F_GAM + Kx, true, false>(pc, S);                            \
    _Pragma("unroll") for (int i = 0; i < 3; ++i)                                                  \
      _Pragma("unroll") for (int j = i; j < 3; ++j) {                                              \
        const double t = g[sym(Kx, i)] * S.d1[j] + g[sym(Kx, j)] * S.d1[i];                        \
        Rt[sym(i, j)] = (Kx == 0) ? t : Rt[sym(i, j)] + t;                                         \
      }                                                                                            \
    advG[Kx] = S.adv; koG[Kx] = S.ko;                                                              \
  }
  GAM_FIELD(0) GAM_FIELD(1) GAM_FIELD(2)
#undef GAM_FIELD

  // ---- gt_ij: first derivatives kept; Rt_ij = -1/2 gt^lm d_l d_m gt_ij + 1/2 t2_ij ; RHS of gt_ij -------
  double dg[3][6];      // dg[k][ij] = d_k gt_ij
#define GT_FIELD(I, J)                                                                             \
  {                                                                                                \
    constexpr int n = sym(I, J);                                                                   \
    src.template derivs<F_G + n, true, true>(pc, S);                                \
    dg[0][n] = S.d1[0]; dg[1][n] = S.d1[1]; dg[2][n] = S.d1[2];                                    \
    Rt[n] = -half * sum9(gi, S.d2) + half * Rt[n];                                                 \
    double lie = g[sym(I, 0)] * db[J][0] + g[sym(J, 0)] * db[I][0];                                \
    lie += g[sym(I, 1)] * db[J][1] + g[sym(J, 1)] * db[I][1];                                      \
    lie += g[sym(I, 2)] * db[J][2] + g[sym(J, 2)] * db[I][2];                                      \
    const double a = -2.0 * alp * src.centre(F_A + n);                                             \
    emit.template put<F_G + n>((((a + S.adv) + lie) - two3 * g[n] * divb) + S.ko);                              \
  }
  GT_FIELD(0, 0) GT_FIELD(0, 1) GT_FIELD(0, 2) GT_FIELD(1, 1) GT_FIELD(1, 2) GT_FIELD(2, 2)
#undef GT_FIELD

  // ---- Christoffels: Gl[k][ij] = Gt_kij, Gu[k][ij] = Gt^k_ij, Gd[k] = gt^ij Gt^k_ij (item 7) --------------
  double Gu[3][6];
  {
    double Gl[3][6], Gd[3];
#pragma unroll
    for (int k = 0; k < 3; ++k)
#pragma unroll
      for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = i; j < 3; ++j)
          Gl[k][sym(i, j)] = half * ((dg[i][sym(k, j)] + dg[j][sym(k, i)]) - dg[k][sym(i, j)]);
#pragma unroll
    for (int k = 0; k < 3; ++k) {
#pragma unroll
      for (int n = 0; n < 6; ++n)
        Gu[k][n] = (gi[sym(k, 0)] * Gl[0][n] + gi[sym(k, 1)] * Gl[1][n]) + gi[sym(k, 2)] * Gl[2][n];
      Gd[k] = sum9(gi, Gu[k]);
    }
    // Rt_ij += 1/2 Gt_d^k (Gt_ijk + Gt_jik)                                          [index order]
    //        + gt^lm ( Gt^k_li Gt_jkm + Gt^k_lj Gt_ikm + Gt^k_im Gt_klj )            [relaxed, regrouped:]
    // with H_i[k][m] = gt^lm Gt^k_li :  T1_ij = H_i[k][m] Gt_jkm ,  T3_ij = H_i[k][l] Gt_klj ,
    // quadratic block = T1_ij + T1_ji + T3_ij.
    // Every piece is added to Rt_ij as soon as it exists (no T1 / T3 arrays: 15 fewer live values at the register
    // peak of the kernel); the diagonal takes T1_ii twice.
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = i; j < 3; ++j) {
        const double t3 = fma(Gd[2], Gl[i][sym(j, 2)] + Gl[j][sym(i, 2)],
                              fma(Gd[1], Gl[i][sym(j, 1)] + Gl[j][sym(i, 1)], Gd[0] * (Gl[i][sym(j, 0)] + Gl[j][sym(i, 0)])));
        Rt[sym(i, j)] = fma(half, t3, Rt[sym(i, j)]);
      }
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      double H[3][3];
#pragma unroll
      for (int k = 0; k < 3; ++k)
#pragma unroll
        for (int m = 0; m < 3; ++m)
          H[k][m] = fma(gi[sym(2, m)], Gu[k][sym(2, i)], fma(gi[sym(1, m)], Gu[k][sym(1, i)], gi[sym(0, m)] * Gu[k][sym(0, i)]));
#pragma unroll
      for (int j = 0; j < 3; ++j) {
        // three partial chains per contraction (k = 0, 1, 2) instead of one chain of nine
        double t[3], t3[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          t[k] = fma(H[k][2], Gl[j][sym(k, 2)], fma(H[k][1], Gl[j][sym(k, 1)], H[k][0] * Gl[j][sym(k, 0)]));
          if (j >= i) t3[k] = fma(H[k][2], Gl[k][sym(2, j)], fma(H[k][1], Gl[k][sym(1, j)], H[k][0] * Gl[k][sym(0, j)]));
        }
        const double T1 = (t[0] + t[1]) + t[2];
        Rt[sym(i, j)] += (i == j) ? 2.0 * T1 : T1;
        if (j >= i) Rt[sym(i, j)] += (t3[0] + t3[1]) + t3[2];
      }
    }
    // At^i_j, At^ij (all nine: the two index orders round differently) and At_ij At^ij
    {
      double A[6], Aud[3][3];
  #pragma unroll
      for (int n = 0; n < 6; ++n) A[n] = src.centre(F_A + n);
  #pragma unroll
      for (int i = 0; i < 3; ++i)
  #pragma unroll
        for (int j = 0; j < 3; ++j)
          Aud[i][j] = (gi[sym(i, 0)] * A[sym(0, j)] + gi[sym(i, 1)] * A[sym(1, j)]) + gi[sym(i, 2)] * A[sym(2, j)];
  #pragma unroll
      for (int i = 0; i < 3; ++i)
  #pragma unroll
        for (int j = 0; j < 3; ++j)
          Auu[i][j] = (Aud[i][0] * gi[sym(0, j)] + Aud[i][1] * gi[sym(1, j)]) + Aud[i][2] * gi[sym(2, j)];
      {   // At_ij At^ij: diagonal + the two index orders of the off-diagonal pairs, FMA tree (feeds K-hat, Theta only)
        const double d = fma(A[5], Auu[2][2], fma(A[3], Auu[1][1], A[0] * Auu[0][0]));
        const double o = fma(A[4], Auu[1][2] + Auu[2][1], fma(A[2], Auu[0][2] + Auu[2][0], A[1] * (Auu[0][1] + Auu[1][0])));
        AA = d + o;
      }
    }
    // Gt^i RHS pieces that need the Christoffels                                      [relaxed running sum]
    //   2 alpha Gt^i_jk At^jk - Gt_d^j d_j beta^i + 2/3 Gt_d^i div beta - 2 alpha kappa1 (Gt^i - Gt_d^i)
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      double t2 = 0.0;
#pragma unroll
      for (int j = 0; j < 3; ++j)
#pragma unroll
        for (int k = 0; k < 3; ++k) t2 = fma(Gu[i][sym(j, k)], Auu[j][k], t2);
      double t = 2.0 * alp * t2;
      t -= fma(Gd[2], db[2][i], fma(Gd[1], db[1][i], Gd[0] * db[0][i]));
      t = fma(two3 * Gd[i], divb, t);
      t -= 2.0 * alp * P.kappa1 * (src.centre(F_GAM + i) - Gd[i]);
      gr[i] += t;
    }
  }

  // ---- W: conformal-factor part of the Ricci tensor; Rt -> W^2 R_ij ; RHS of W ---------------------------
  double dW[3];
  {
    src.template derivs<F_W, true, true>(pc, S);
    dW[0] = S.d1[0]; dW[1] = S.d1[1]; dW[2] = S.d1[2];
    double DDW[6], dW2[6];   // Dt_i Dt_j W and d_i W d_j W (both only feed the Ricci tensor: FMA chains)
#pragma unroll
    for (int n = 0; n < 6; ++n) DDW[n] = fma(-Gu[2][n], dW[2], fma(-Gu[1][n], dW[1], fma(-Gu[0][n], dW[0], S.d2[n])));
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = i; j < 3; ++j) dW2[sym(i, j)] = dW[i] * dW[j];
    const double trDDW = sum9(gi, DDW), dWdW = sum9(gi, dW2);
#pragma unroll
    for (int n = 0; n < 6; ++n)
      Rt[n] = W * W * Rt[n] + (W * (DDW[n] + g[n] * trDDW) - 2.0 * g[n] * dWdW);
    // Gt^i RHS: 2 alpha (-3 At^ij d_j W / W)                                          [relaxed running sum]
    const double f = -6.0 * alp / W;
#pragma unroll
    for (int i = 0; i < 3; ++i)
      gr[i] = fma(f, fma(Auu[i][2], dW[2], fma(Auu[i][1], dW[1], Auu[i][0] * dW[0])), gr[i]);
    emit.template put<F_W>((S.adv + third * W * (alp * K - divb)) + S.ko);
  }
  const double R = sum9(gi, Rt);                                         // R = gt^ij W^2 R_ij

  // ---- alpha: W^2 D_i D_j alpha; Rt -> X_ij = -W^2 D_i D_j alpha + alpha W^2 R_ij ; RHS of alpha (Eq. 6) --
  double lapa;
  {
    src.template derivs<F_ALP, true, true>(pc, S);
    const double (&da)[3] = S.d1;
    const double dadW = fma(da[2], row3(gi, 2, dW), fma(da[1], row3(gi, 1, dW), da[0] * row3(gi, 0, dW)));
    double WDDa[6];
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = i; j < 3; ++j) {
        const int n = sym(i, j);
        const double cov = fma(-Gu[2][n], da[2], fma(-Gu[1][n], da[1], fma(-Gu[0][n], da[0], S.d2[n])));
        WDDa[n] = W * W * cov + W * ((da[i] * dW[j] + da[j] * dW[i]) - g[n] * dadW);
      }
    lapa = sum9(gi, WDDa);
#pragma unroll
    for (int n = 0; n < 6; ++n) Rt[n] = -WDDa[n] + alp * Rt[n];
    // Gt^i RHS: -2 At^ij d_j alpha                                                    [relaxed running sum]
#pragma unroll
    for (int i = 0; i < 3; ++i)
      gr[i] = fma(-2.0, fma(Auu[i][2], da[2], fma(Auu[i][1], da[1], Auu[i][0] * da[0])), gr[i]);
    const double Ksrc = P.lapse_uses_khat ? Kh : K;                      // reading C
    emit.template put<F_ALP>((S.adv - 2.0 * alp * Ksrc) + S.ko);
  }

  // ---- K-hat and Theta: gradient term of Gt^i, and their own RHS ------------------------------------------
  {
    src.template derivs<F_KH, true, false>(pc, S);
    const double f = -2.0 * two3 * alp;                                  // 2 alpha (-1/3) * 2
#pragma unroll
    for (int i = 0; i < 3; ++i) gr[i] = fma(f, row3(gi, i, S.d1), gr[i]);
    const double k = ((-lapa + alp * (AA + third * K * K)) + alp * P.kappa1 * (1.0 - P.kappa2) * Th) + S.adv;
    emit.template put<F_KH>(k + S.ko);
  }
  {
    src.template derivs<F_TH, true, false>(pc, S);
    const double f = -two3 * alp;                                        // 2 alpha (-1/3)
#pragma unroll
    for (int i = 0; i < 3; ++i) gr[i] = fma(f, row3(gi, i, S.d1), gr[i]);
    const double k = (half * alp * ((R - AA) + two3 * K * K) - alp * P.kappa1 * (2.0 + P.kappa2) * Th) + S.adv;
    emit.template put<F_TH>(k + S.ko);
  }

  // ---- Gt^i complete; B^i (Eq. 8; reading H: the Gt^i RHS enters without KO and without advection) --------
  emit.template put<F_GAM + 0>((gr[0] + advG[0]) + koG[0]);
  emit.template put<F_GAM + 1>((gr[1] + advG[1]) + koG[1]);
  emit.template put<F_GAM + 2>((gr[2] + advG[2]) + koG[2]);
#define B_FIELD(I)                                                                                 \
  {                                                                                                \
    src.template derivs<F_B + I, false, false>(pc, S);                              \
    emit.template put<F_B + I>(((S.adv + gr[I]) - P.eta * S.u0) + S.ko);                                        \
  }
  B_FIELD(0) B_FIELD(1) B_FIELD(2)
#undef B_FIELD

  // ---- At_ij: trace-free part of X_ij and the algebraic terms (item 8) ------------------------------------
  {
    const double trX = sum9(gi, Rt);
    double A[6];
#pragma unroll
    for (int n = 0; n < 6; ++n) A[n] = src.centre(F_A + n);
    double Aud[3][3];   // At^k_j
#pragma unroll
    for (int k = 0; k < 3; ++k)
#pragma unroll
      for (int j = 0; j < 3; ++j)
        Aud[k][j] = (gi[sym(k, 0)] * A[sym(0, j)] + gi[sym(k, 1)] * A[sym(1, j)]) + gi[sym(k, 2)] * A[sym(2, j)];
#define AT_FIELD(I, J)                                                                             \
  {                                                                                                \
    constexpr int n = sym(I, J);                                                                   \
    src.template derivs<F_A + n, false, false>(pc, S);                              \
    const double xtf = Rt[n] - third * g[n] * trX;                                                 \
    const double aa = (A[sym(I, 0)] * Aud[0][J] + A[sym(I, 1)] * Aud[1][J]) + A[sym(I, 2)] * Aud[2][J]; \
    double lie = A[sym(I, 0)] * db[J][0] + A[sym(J, 0)] * db[I][0];                                \
    lie += A[sym(I, 1)] * db[J][1] + A[sym(J, 1)] * db[I][1];                                      \
    lie += A[sym(I, 2)] * db[J][2] + A[sym(J, 2)] * db[I][2];                                      \
    const double k = xtf + alp * (K * A[n] - 2.0 * aa);                                            \
    emit.template put<F_A + n>((((k + S.adv) + lie) - two3 * A[n] * divb) + S.ko);                              \
  }
    AT_FIELD(0, 0) AT_FIELD(0, 1) AT_FIELD(0, 2) AT_FIELD(1, 1) AT_FIELD(1, 2) AT_FIELD(2, 2)
#undef AT_FIELD
  }
}

}  // namespace sacra
