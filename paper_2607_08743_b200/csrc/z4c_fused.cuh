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
// Register diet: the tensors that live across many field passes -- d_k beta^i, d_k gt_ij, Gt^k_ij,
// At^ij, the advection / KO terms of Gt^i, and the centre values of all 25 fields -- are PARKED in the thread's Tensor
// Memory strip (z4c_tmem.cuh, slot map in z4c_tile.cuh) and pulled back in aligned groups where a block needs them; the
// loads are issued before the stencils of the field they serve, so their ~55 cycles hide behind the shared-memory work.
//
// `Src` provides   src.derivs<F, D1, D2>(pc, S) -> the derivative bundle S of field F (field_derivs() on its tile)
//                  src.strip(d)    -> Tensor Memory address of double d of this thread's strip
// `Emit` provides  emit.put<F>(k, u0)  -> consumes the finished RHS value k of field F (KO included); u0 = the field's
//                                         value at the point (u_n at RK stage 1)
#pragma once
#include "z4c_stencil.cuh"
#include "z4c_tile.cuh"

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
__device__ __forceinline__ void z4c_point(const Src& src, const Params& P, const GridCoef& gc, Emit& emit) {
  using namespace tmem;
  const double half = 0.5, third = 1.0 / 3.0, two3 = 2.0 / 3.0;
  Stencil S;
  PointCoef pc;

  // ---- centre values (Tensor Memory strip) and the true inverse conformal metric (item 7; det gt is not assumed 1) --
  double g[6], gi[6], alp, W, Kh, Th, Bc[3];
  {
    Pack4 p0, p8, p12;
    Pack2 p4, p6;
    ld4(src.strip(0), p0); ld2(src.strip(4), p4); ld2(src.strip(6), p6); ld4(src.strip(8), p8); ld4(src.strip(12), p12);
    wait_ld(p0, p4, p6, p8, p12);
    g[0] = p0.get(0); g[1] = p0.get(1); g[2] = p0.get(2); g[3] = p0.get(3); g[4] = p4.get(0); g[5] = p4.get(1);
    alp = p6.get(0); W = p6.get(1);
    const double beta[3] = {p8.get(0), p8.get(1), p8.get(2)};
    Kh = p8.get(3);
    Bc[0] = p12.get(0); Bc[1] = p12.get(1); Bc[2] = p12.get(2);
    Th = p12.get(3);
    make_coef(gc, beta, pc);
  }
  {
    const double gxx = g[0], gxy = g[1], gxz = g[2], gyy = g[3], gyz = g[4], gzz = g[5];
    const double det = (gxx * (gyy * gzz - gyz * gyz) - gxy * (gxy * gzz - gyz * gxz)) + gxz * (gxy * gyz - gyy * gxz);
    // one IEEE division, six products: gt^ij feeds only the relaxed fields (K-hat, Theta, At_ij, Gt^i, B^i), where a last-bit
    // difference from the oracle's six divisions is far inside the tolerance
    const double rdet = 1.0 / det;
    gi[0] = (gyy * gzz - gyz * gyz) * rdet;
    gi[1] = (gxz * gyz - gxy * gzz) * rdet;
    gi[2] = (gxy * gyz - gxz * gyy) * rdet;
    gi[3] = (gxx * gzz - gxz * gxz) * rdet;
    gi[4] = (gxy * gxz - gxx * gyz) * rdet;
    gi[5] = (gxx * gyy - gxy * gxy) * rdet;
  }
  const double K = Kh + 2.0 * Th;                                        // item 7: K = K-hat + 2 Theta

  // ---- beta^i: d_k beta^i; gt^jk d_j d_k beta^i; d_j d_k beta^k; RHS of beta^i (Eq. 7) -------------------
  // d_k beta^i is parked k-major: group k = (d_k beta^x, d_k beta^y, d_k beta^z)
  double gr[3];         // running RHS of Gt^i without advection (item 8)      [relaxed running sum]
  double divb;
  {
    double db[3][3];    // db[k][i] = d_k beta^i
    double dd[3];       // d_j (d_k beta^k)
#define BETA_FIELD(I)                                                                              \
  {                                                                                                \
    src.template derivs<F_BET + I, true, true>(pc, S);                                             \
    db[0][I] = S.d1[0]; db[1][I] = S.d1[1]; db[2][I] = S.d1[2];                                    \
    gr[I] = sum9(gi, S.d2);                                                                        \
    if (I == 0) { dd[0] = S.d2[sym(0, 0)]; dd[1] = S.d2[sym(1, 0)]; dd[2] = S.d2[sym(2, 0)]; }     \
    else { dd[0] += S.d2[sym(0, I)]; dd[1] += S.d2[sym(1, I)]; dd[2] += S.d2[sym(2, I)]; }         \
    emit.template put<F_BET + I>((S.adv + P.shift_coef * Bc[I]) + S.ko, S.u0);                     \
  }
    BETA_FIELD(0) BETA_FIELD(1) BETA_FIELD(2)
#undef BETA_FIELD
    divb = (db[0][0] + db[1][1]) + db[2][2];
#pragma unroll
    for (int i = 0; i < 3; ++i) gr[i] = fma(third, row3(gi, i, dd), gr[i]);
#pragma unroll
    for (int k = 0; k < 3; ++k) st4(src.strip(PK_DB + 4 * k), db[k][0], db[k][1], db[k][2], 0.0);
  }

  // ---- Gt^i: t2_ij = sum_k (gt_ki d_j Gt^k + gt_kj d_i Gt^k); advection and KO of Gt^i parked --------------
  double Rt[6];         // t2_ij, then Rt_ij, then W^2 R_ij, then X_ij
#define GAM_FIELD(Kx)                                                                              \
  {                                                                                                \
    src.template derivs<F_GAM + Kx, true, false>(pc, S);                                           \
    _Pragma("unroll") for (int i = 0; i < 3; ++i)                                                  \
      _Pragma("unroll") for (int j = i; j < 3; ++j) {                                              \
        const double t = g[sym(Kx, i)] * S.d1[j] + g[sym(Kx, j)] * S.d1[i];                        \
        Rt[sym(i, j)] = (Kx == 0) ? t : Rt[sym(i, j)] + t;                                         \
      }                                                                                            \
    st2(src.strip(PK_AG + 2 * Kx), S.adv, S.ko);                                                   \
  }
  GAM_FIELD(0) GAM_FIELD(1) GAM_FIELD(2)
#undef GAM_FIELD
  wait_st();            // d_k beta^i is read back from here on

  // ---- gt_ij: first derivatives parked; Rt_ij = -1/2 gt^lm d_l d_m gt_ij + 1/2 t2_ij ; RHS of gt_ij -------
#define GT_FIELD(I, J)                                                                             \
  {                                                                                                \
    constexpr int n = sym(I, J);                                                                   \
    Pack4 dI, dJ;                                                                                  \
    Pack1 an;                                                                                      \
    ld4(src.strip(PK_DB + 4 * I), dI);                                                             \
    ld4(src.strip(PK_DB + 4 * J), dJ);                                                             \
    ld1(src.strip(16 + n), an);                                                                    \
    src.template derivs<F_G + n, true, true>(pc, S);                                               \
    wait_ld(dI, dJ, an);                                                                           \
    st4(src.strip(PK_DG + 4 * n), S.d1[0], S.d1[1], S.d1[2], 0.0);                                 \
    Rt[n] = -half * sum9(gi, S.d2) + half * Rt[n];                                                 \
    double lie = g[sym(I, 0)] * dJ.get(0) + g[sym(J, 0)] * dI.get(0);                              \
    lie += g[sym(I, 1)] * dJ.get(1) + g[sym(J, 1)] * dI.get(1);                                    \
    lie += g[sym(I, 2)] * dJ.get(2) + g[sym(J, 2)] * dI.get(2);                                    \
    const double a = -2.0 * alp * an.get(0);                                                       \
    emit.template put<F_G + n>((((a + S.adv) + lie) - two3 * g[n] * divb) + S.ko, S.u0);           \
  }
  GT_FIELD(0, 0) GT_FIELD(0, 1) GT_FIELD(0, 2) GT_FIELD(1, 1) GT_FIELD(1, 2) GT_FIELD(2, 2)
#undef GT_FIELD

  // ---- Christoffels: Gl[k][ij] = Gt_kij, Gu[k][ij] = Gt^k_ij, Gd[k] = gt^ij Gt^k_ij (item 7) --------------
  // Gt^k_ij goes to the strip as soon as it exists and comes back in the slices the blocks below use, so that the
  // first-kind symbols, one slice and the H matrix are the most that is live at once.
  double AA;            // At_ij At^ij
  {
    double Gd[3];
    {
      double Gl[3][6];
      {
        wait_st();
        Pack4 q[6];
#pragma unroll
        for (int n = 0; n < 6; ++n) ld4(src.strip(PK_DG + 4 * n), q[n]);
        wait_ld(q[0], q[1], q[2], q[3], q[4], q[5]);
        // dg[k][n] = q[n].get(k)
#pragma unroll
        for (int k = 0; k < 3; ++k)
#pragma unroll
          for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = i; j < 3; ++j)
              Gl[k][sym(i, j)] = half * ((q[sym(k, j)].get(i) + q[sym(k, i)].get(j)) - q[sym(i, j)].get(k));
      }
      {
        double Gu[3][6];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
#pragma unroll
          for (int n = 0; n < 6; ++n)
            Gu[k][n] = (gi[sym(k, 0)] * Gl[0][n] + gi[sym(k, 1)] * Gl[1][n]) + gi[sym(k, 2)] * Gl[2][n];
          Gd[k] = sum9(gi, Gu[k]);
        }
#pragma unroll
        for (int n = 0; n < 6; ++n) st4(src.strip(PK_GU + 4 * n), Gu[0][n], Gu[1][n], Gu[2][n], 0.0);
      }
      // Rt_ij += 1/2 Gt_d^k (Gt_ijk + Gt_jik)                                          [index order]
      //        + gt^lm ( Gt^k_li Gt_jkm + Gt^k_lj Gt_ikm + Gt^k_im Gt_klj )            [relaxed, regrouped:]
      // with H_i[k][m] = gt^lm Gt^k_li :  T1_ij = H_i[k][m] Gt_jkm ,  T3_ij = H_i[k][l] Gt_klj ,
      // quadratic block = T1_ij + T1_ji + T3_ij.
      // Every piece is added to Rt_ij as soon as it exists (no T1 / T3 arrays); the diagonal takes T1_ii twice.
#pragma unroll
      for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = i; j < 3; ++j) {
          const double t3 = fma(Gd[2], Gl[i][sym(j, 2)] + Gl[j][sym(i, 2)],
                                fma(Gd[1], Gl[i][sym(j, 1)] + Gl[j][sym(i, 1)], Gd[0] * (Gl[i][sym(j, 0)] + Gl[j][sym(i, 0)])));
          Rt[sym(i, j)] = fma(half, t3, Rt[sym(i, j)]);
        }
      wait_st();
#pragma unroll
      for (int i = 0; i < 3; ++i) {
        Pack4 u0, u1, u2;   // Gt^k_li for l = 0, 1, 2: groups sym(l, i)
        ld4(src.strip(PK_GU + 4 * sym(0, i)), u0); ld4(src.strip(PK_GU + 4 * sym(1, i)), u1);
        ld4(src.strip(PK_GU + 4 * sym(2, i)), u2);
        wait_ld(u0, u1, u2);
        double H[3][3];
#pragma unroll
        for (int k = 0; k < 3; ++k)
#pragma unroll
          for (int m = 0; m < 3; ++m)
            H[k][m] = fma(gi[sym(2, m)], u2.get(k), fma(gi[sym(1, m)], u1.get(k), gi[sym(0, m)] * u0.get(k)));
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
    }
    // At^i_j, At^ij (all nine: the two index orders round differently) and At_ij At^ij; At^ij is parked
    double Auu[3][3];
    Pack4 d0, d1, d2;   // d_k beta^i back for the Gt^i RHS
    Pack4 gq[6];        // Gt^k_n back for the Gt^i RHS
    Pack2 c22;
    Pack1 c24;
    {
      Pack4 a0;
      Pack2 a4;
      ld4(src.strip(16), a0); ld2(src.strip(20), a4);
      ld4(src.strip(PK_DB), d0); ld4(src.strip(PK_DB + 4), d1); ld4(src.strip(PK_DB + 8), d2);
      ld2(src.strip(22), c22); ld1(src.strip(24), c24);
#pragma unroll
      for (int n = 0; n < 6; ++n) ld4(src.strip(PK_GU + 4 * n), gq[n]);
      wait_ld(a0, a4, d0, d1, d2, c22, c24, gq[0], gq[1], gq[2], gq[3], gq[4], gq[5]);
      const double A[6] = {a0.get(0), a0.get(1), a0.get(2), a0.get(3), a4.get(0), a4.get(1)};
      double Aud[3][3];
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
#pragma unroll
      for (int i = 0; i < 3; ++i) st4(src.strip(PK_AUU + 4 * i), Auu[i][0], Auu[i][1], Auu[i][2], 0.0);
    }
    // Gt^i RHS pieces that need the Christoffels                                      [relaxed running sum]
    //   2 alpha Gt^i_jk At^jk - Gt_d^j d_j beta^i + 2/3 Gt_d^i div beta - 2 alpha kappa1 (Gt^i - Gt_d^i)
    const double Gc[3] = {c22.get(0), c22.get(1), c24.get(0)};
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      double t2 = 0.0;
#pragma unroll
      for (int j = 0; j < 3; ++j)
#pragma unroll
        for (int k = 0; k < 3; ++k) t2 = fma(gq[sym(j, k)].get(i), Auu[j][k], t2);
      double t = 2.0 * alp * t2;
      t -= fma(Gd[2], d2.get(i), fma(Gd[1], d1.get(i), Gd[0] * d0.get(i)));
      t = fma(two3 * Gd[i], divb, t);
      t -= 2.0 * alp * P.kappa1 * (Gc[i] - Gd[i]);
      gr[i] += t;
    }
  }
  wait_st();            // Gt^k_ij and At^ij are read back from here on

  // Gt^k_n (group n) and At^ij (group i) back from the strip; issued before a field's stencils, used after them
#define LOAD_GU_AUU()                                                                              \
  Pack4 gq[6], aq[3];                                                                              \
  _Pragma("unroll") for (int n = 0; n < 6; ++n) ld4(src.strip(PK_GU + 4 * n), gq[n]);              \
  _Pragma("unroll") for (int i = 0; i < 3; ++i) ld4(src.strip(PK_AUU + 4 * i), aq[i]);
#define WAIT_GU_AUU() wait_ld(gq[0], gq[1], gq[2], gq[3], gq[4], gq[5], aq[0], aq[1], aq[2]);

  // ---- W: conformal-factor part of the Ricci tensor; Rt -> W^2 R_ij ; RHS of W ---------------------------
  double dW[3];
  {
    LOAD_GU_AUU()
    src.template derivs<F_W, true, true>(pc, S);
    WAIT_GU_AUU()
    dW[0] = S.d1[0]; dW[1] = S.d1[1]; dW[2] = S.d1[2];
    double DDW[6], dW2[6];   // Dt_i Dt_j W and d_i W d_j W (both only feed the Ricci tensor: FMA chains)
#pragma unroll
    for (int n = 0; n < 6; ++n)
      DDW[n] = fma(-gq[n].get(2), dW[2], fma(-gq[n].get(1), dW[1], fma(-gq[n].get(0), dW[0], S.d2[n])));
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
      gr[i] = fma(f, fma(aq[i].get(2), dW[2], fma(aq[i].get(1), dW[1], aq[i].get(0) * dW[0])), gr[i]);
    emit.template put<F_W>((S.adv + third * W * (alp * K - divb)) + S.ko, S.u0);
  }
  const double R = sum9(gi, Rt);                                         // R = gt^ij W^2 R_ij

  // ---- alpha: W^2 D_i D_j alpha; Rt -> X_ij = -W^2 D_i D_j alpha + alpha W^2 R_ij ; RHS of alpha (Eq. 6) --
  double lapa;
  {
    LOAD_GU_AUU()
    src.template derivs<F_ALP, true, true>(pc, S);
    WAIT_GU_AUU()
    const double (&da)[3] = S.d1;
    const double dadW = fma(da[2], row3(gi, 2, dW), fma(da[1], row3(gi, 1, dW), da[0] * row3(gi, 0, dW)));
    double WDDa[6];
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = i; j < 3; ++j) {
        const int n = sym(i, j);
        const double cov = fma(-gq[n].get(2), da[2], fma(-gq[n].get(1), da[1], fma(-gq[n].get(0), da[0], S.d2[n])));
        WDDa[n] = W * W * cov + W * ((da[i] * dW[j] + da[j] * dW[i]) - g[n] * dadW);
      }
    lapa = sum9(gi, WDDa);
#pragma unroll
    for (int n = 0; n < 6; ++n) Rt[n] = -WDDa[n] + alp * Rt[n];
    // Gt^i RHS: -2 At^ij d_j alpha                                                    [relaxed running sum]
#pragma unroll
    for (int i = 0; i < 3; ++i)
      gr[i] = fma(-2.0, fma(aq[i].get(2), da[2], fma(aq[i].get(1), da[1], aq[i].get(0) * da[0])), gr[i]);
    const double Ksrc = P.lapse_uses_khat ? Kh : K;                      // reading C
    emit.template put<F_ALP>((S.adv - 2.0 * alp * Ksrc) + S.ko, S.u0);
  }
#undef LOAD_GU_AUU
#undef WAIT_GU_AUU

  // ---- K-hat and Theta: gradient term of Gt^i, and their own RHS ------------------------------------------
  {
    src.template derivs<F_KH, true, false>(pc, S);
    const double f = -2.0 * two3 * alp;                                  // 2 alpha (-1/3) * 2
#pragma unroll
    for (int i = 0; i < 3; ++i) gr[i] = fma(f, row3(gi, i, S.d1), gr[i]);
    const double k = ((-lapa + alp * (AA + third * K * K)) + alp * P.kappa1 * (1.0 - P.kappa2) * Th) + S.adv;
    emit.template put<F_KH>(k + S.ko, S.u0);
  }
  {
    Pack2 g0, g1, g2;     // advection and KO of Gt^k; its centre values (u_n at RK stage 1)
    Pack2 c22;
    Pack1 c24;
    ld2(src.strip(PK_AG), g0); ld2(src.strip(PK_AG + 2), g1); ld2(src.strip(PK_AG + 4), g2);
    ld2(src.strip(22), c22); ld1(src.strip(24), c24);
    src.template derivs<F_TH, true, false>(pc, S);
    wait_ld(g0, g1, g2, c22, c24);
    const double f = -two3 * alp;                                        // 2 alpha (-1/3)
#pragma unroll
    for (int i = 0; i < 3; ++i) gr[i] = fma(f, row3(gi, i, S.d1), gr[i]);
    const double k = (half * alp * ((R - AA) + two3 * K * K) - alp * P.kappa1 * (2.0 + P.kappa2) * Th) + S.adv;
    emit.template put<F_TH>(k + S.ko, S.u0);
    // ---- Gt^i complete ------------------------------------------------------------------------------------
    emit.template put<F_GAM + 0>((gr[0] + g0.get(0)) + g0.get(1), c22.get(0));
    emit.template put<F_GAM + 1>((gr[1] + g1.get(0)) + g1.get(1), c22.get(1));
    emit.template put<F_GAM + 2>((gr[2] + g2.get(0)) + g2.get(1), c24.get(0));
  }
  // ---- B^i (Eq. 8; reading H: the Gt^i RHS enters without KO and without advection) -----------------------
#define B_FIELD(I)                                                                                 \
  {                                                                                                \
    src.template derivs<F_B + I, false, false>(pc, S);                                             \
    emit.template put<F_B + I>(((S.adv + gr[I]) - P.eta * S.u0) + S.ko, S.u0);                     \
  }
  B_FIELD(0) B_FIELD(1) B_FIELD(2)
#undef B_FIELD

  // ---- At_ij: trace-free part of X_ij and the algebraic terms (item 8) ------------------------------------
  {
    const double trX = sum9(gi, Rt);
    double A[6];
    {
      Pack4 a0;
      Pack2 a4;
      ld4(src.strip(16), a0); ld2(src.strip(20), a4);
      wait_ld(a0, a4);
      A[0] = a0.get(0); A[1] = a0.get(1); A[2] = a0.get(2); A[3] = a0.get(3); A[4] = a4.get(0); A[5] = a4.get(1);
    }
    double Aud[3][3];   // At^k_j
#pragma unroll
    for (int k = 0; k < 3; ++k)
#pragma unroll
      for (int j = 0; j < 3; ++j)
        Aud[k][j] = (gi[sym(k, 0)] * A[sym(0, j)] + gi[sym(k, 1)] * A[sym(1, j)]) + gi[sym(k, 2)] * A[sym(2, j)];
#define AT_FIELD(I, J)                                                                             \
  {                                                                                                \
    constexpr int n = sym(I, J);                                                                   \
    Pack4 dI, dJ;                                                                                  \
    ld4(src.strip(PK_DB + 4 * I), dI);                                                             \
    ld4(src.strip(PK_DB + 4 * J), dJ);                                                             \
    src.template derivs<F_A + n, false, false>(pc, S);                                             \
    wait_ld(dI, dJ);                                                                               \
    const double xtf = Rt[n] - third * g[n] * trX;                                                 \
    const double aa = (A[sym(I, 0)] * Aud[0][J] + A[sym(I, 1)] * Aud[1][J]) + A[sym(I, 2)] * Aud[2][J]; \
    double lie = A[sym(I, 0)] * dJ.get(0) + A[sym(J, 0)] * dI.get(0);                              \
    lie += A[sym(I, 1)] * dJ.get(1) + A[sym(J, 1)] * dI.get(1);                                    \
    lie += A[sym(I, 2)] * dJ.get(2) + A[sym(J, 2)] * dI.get(2);                                    \
    const double k = xtf + alp * (K * A[n] - 2.0 * aa);                                            \
    emit.template put<F_A + n>((((k + S.adv) + lie) - two3 * A[n] * divb) + S.ko, S.u0);           \
  }
    AT_FIELD(0, 0) AT_FIELD(0, 1) AT_FIELD(0, 2) AT_FIELD(1, 1) AT_FIELD(1, 2) AT_FIELD(2, 2)
#undef AT_FIELD
  }
}

}  // namespace sacra
