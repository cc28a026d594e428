// z4c_algebra.hpp -- TEST INFRASTRUCTURE (part of the oracle; see z4c_oracle.hpp).
//
// Point-wise Z4c right-hand side: SURVEY.md 8(c) items 7-10 written out with
// plain loops over tensor indices, no hand CSE. The system is the Z4c
// conformal decomposition of Hilditch et al. 2013 that PAPER.md:63 points to,
// rewritten in W (chi = W^2), with the gauge of Eqs. 6-8.
// Vacuum: all matter sources are zero.
#pragma once
#include "z4c_oracle.hpp"

namespace z4c_oracle {

// u[NF]: field values at the point; D: derivative bundle; out[NF]: RHS
// including KO (item 10). If adv_gam_out != nullptr nothing else changes.
template <class T>
inline void z4c_rhs_point(const T u[NF], const Derivs<T>& D, const Params<T>& P, T out[NF]) {
  const T half = T(1) / T(2), third = T(1) / T(3), two3 = T(2) / T(3);

  // ---- unpack ------------------------------------------------------------
  const T W = u[F_W], Kh = u[F_KH], Th = u[F_TH], alp = u[F_ALP];
  T g[3][3], A[3][3], Gam[3], Bv[3];
  for (int i = 0; i < 3; ++i) {
    for (int j = 0; j < 3; ++j) {
      g[i][j] = u[F_G + SYM[i][j]];
      A[i][j] = u[F_A + SYM[i][j]];
    }
    Gam[i] = u[F_GAM + i];
    Bv[i] = u[F_B + i];
  }
  const T K = Kh + T(2) * Th;                       // item 7: K := K-hat + 2 Theta

  // ---- item 7: true inverse of the conformal metric ----------------------
  const T det = g[0][0] * (g[1][1] * g[2][2] - g[1][2] * g[1][2]) -
                g[0][1] * (g[0][1] * g[2][2] - g[1][2] * g[0][2]) +
                g[0][2] * (g[0][1] * g[1][2] - g[1][1] * g[0][2]);
  T gi[3][3];
  gi[0][0] = (g[1][1] * g[2][2] - g[1][2] * g[1][2]) / det;
  gi[0][1] = (g[0][2] * g[1][2] - g[0][1] * g[2][2]) / det;
  gi[0][2] = (g[0][1] * g[1][2] - g[0][2] * g[1][1]) / det;
  gi[1][1] = (g[0][0] * g[2][2] - g[0][2] * g[0][2]) / det;
  gi[1][2] = (g[0][1] * g[0][2] - g[0][0] * g[1][2]) / det;
  gi[2][2] = (g[0][0] * g[1][1] - g[0][1] * g[0][1]) / det;
  gi[1][0] = gi[0][1]; gi[2][0] = gi[0][2]; gi[2][1] = gi[1][2];

  // ---- derivatives in tensor notation ------------------------------------
  T dg[3][3][3];      // dg[k][i][j]  = d_k gt_ij
  T ddg[3][3][3][3];  // ddg[l][m][i][j] = d_l d_m gt_ij
  T dW[3], ddW[3][3], da[3], dda[3][3];
  T db[3][3];         // db[i][k]  = d_i beta^k
  T ddb[3][3][3];     // ddb[i][j][k] = d_i d_j beta^k
  T dGam[3][3];       // dGam[j][k] = d_j Gt^k
  T dKT[3];           // d_j (2 K-hat + Theta)
  for (int k = 0; k < 3; ++k) {
    dW[k] = D.d1[F_W][k];
    da[k] = D.d1[F_ALP][k];
    dKT[k] = T(2) * D.d1[F_KH][k] + D.d1[F_TH][k];
    for (int i = 0; i < 3; ++i) {
      db[k][i] = D.d1[F_BET + i][k];
      dGam[k][i] = D.d1[F_GAM + i][k];
      ddW[k][i] = D.d2[F_W][SYM[k][i]];
      dda[k][i] = D.d2[F_ALP][SYM[k][i]];
      for (int j = 0; j < 3; ++j) {
        dg[k][i][j] = D.d1[F_G + SYM[i][j]][k];
        ddb[k][i][j] = D.d2[F_BET + j][SYM[k][i]];
        for (int m = 0; m < 3; ++m) ddg[k][m][i][j] = D.d2[F_G + SYM[i][j]][SYM[k][m]];
      }
    }
  }
  T divb = T(0);
  for (int k = 0; k < 3; ++k) divb += db[k][k];

  // ---- item 7: Christoffels ----------------------------------------------
  T Gl[3][3][3];  // Gl[k][i][j] = Gt_kij = 1/2 (d_i gt_kj + d_j gt_ki - d_k gt_ij)
  T Gu[3][3][3];  // Gu[k][i][j] = Gt^k_ij
  T Gd[3];        // Gt_d^i = gt^jk Gt^i_jk
  for (int k = 0; k < 3; ++k)
    for (int i = 0; i < 3; ++i)
      for (int j = 0; j < 3; ++j)
        Gl[k][i][j] = half * (dg[i][k][j] + dg[j][k][i] - dg[k][i][j]);
  for (int k = 0; k < 3; ++k)
    for (int i = 0; i < 3; ++i)
      for (int j = 0; j < 3; ++j) {
        T s = T(0);
        for (int l = 0; l < 3; ++l) s += gi[k][l] * Gl[l][i][j];
        Gu[k][i][j] = s;
      }
  for (int i = 0; i < 3; ++i) {
    T s = T(0);
    for (int j = 0; j < 3; ++j)
      for (int k = 0; k < 3; ++k) s += gi[j][k] * Gu[i][j][k];
    Gd[i] = s;
  }

  // ---- item 7: conformal Ricci tensor Rt_ij -------------------------------
  T Rt[3][3];
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      T lap = T(0);
      for (int l = 0; l < 3; ++l)
        for (int m = 0; m < 3; ++m) lap += gi[l][m] * ddg[l][m][i][j];
      T t2 = T(0), t3 = T(0);
      for (int k = 0; k < 3; ++k) {
        t2 += g[k][i] * dGam[j][k] + g[k][j] * dGam[i][k];
        t3 += Gd[k] * (Gl[i][j][k] + Gl[j][i][k]);
      }
      T t4 = T(0);
      for (int l = 0; l < 3; ++l)
        for (int m = 0; m < 3; ++m) {
          T q = T(0);
          for (int k = 0; k < 3; ++k)
            q += Gu[k][l][i] * Gl[j][k][m] + Gu[k][l][j] * Gl[i][k][m] +
                 Gu[k][i][m] * Gl[k][l][j];
          t4 += gi[l][m] * q;
        }
      Rt[i][j] = -half * lap + half * t2 + half * t3 + t4;
    }

  // ---- item 7: conformal-factor part, W^2 R_ij, R ---------------------------
  T DDW[3][3];
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      T s = ddW[i][j];
      for (int k = 0; k < 3; ++k) s -= Gu[k][i][j] * dW[k];
      DDW[i][j] = s;
    }
  T trDDW = T(0), dWdW = T(0);
  for (int k = 0; k < 3; ++k)
    for (int l = 0; l < 3; ++l) {
      trDDW += gi[k][l] * DDW[k][l];
      dWdW += gi[k][l] * dW[k] * dW[l];
    }
  T WR[3][3];   // W^2 R_ij
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j)
      WR[i][j] = W * W * Rt[i][j] + (W * (DDW[i][j] + g[i][j] * trDDW) - T(2) * g[i][j] * dWdW);
  T R = T(0);
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) R += gi[i][j] * WR[i][j];

  // ---- item 7: lapse Hessian in the physical metric, times W^2 -------------
  T dadW = T(0);
  for (int k = 0; k < 3; ++k)
    for (int l = 0; l < 3; ++l) dadW += gi[k][l] * da[k] * dW[l];
  T WDDa[3][3];  // W^2 D_i D_j alpha
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      T s = dda[i][j];
      for (int k = 0; k < 3; ++k) s -= Gu[k][i][j] * da[k];
      WDDa[i][j] = W * W * s + W * (da[i] * dW[j] + da[j] * dW[i] - g[i][j] * dadW);
    }
  T lapa = T(0);  // D^i D_i alpha
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) lapa += gi[i][j] * WDDa[i][j];

  // ---- item 7: At with raised indices -----------------------------------------
  T Aud[3][3], Auu[3][3];   // At^i_j, At^ij
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      T s = T(0);
      for (int k = 0; k < 3; ++k) s += gi[i][k] * A[k][j];
      Aud[i][j] = s;
    }
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      T s = T(0);
      for (int k = 0; k < 3; ++k) s += Aud[i][k] * gi[k][j];
      Auu[i][j] = s;
    }
  T AA = T(0);
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) AA += A[i][j] * Auu[i][j];

  // ---- item 8: Z4c right-hand sides (before KO) ------------------------------
  T rhs[NF];
  rhs[F_W] = D.adv[F_W] + third * W * (alp * K - divb);

  for (int i = 0; i < 3; ++i)
    for (int j = i; j < 3; ++j) {
      T s = T(0);
      for (int k = 0; k < 3; ++k) s += g[i][k] * db[j][k] + g[j][k] * db[i][k];
      rhs[F_G + SYM[i][j]] =
          -T(2) * alp * A[i][j] + D.adv[F_G + SYM[i][j]] + s - two3 * g[i][j] * divb;
    }

  rhs[F_KH] = -lapa + alp * (AA + third * K * K) + alp * P.kappa1 * (T(1) - P.kappa2) * Th +
              D.adv[F_KH];

  T X[3][3], trX = T(0);
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) X[i][j] = -WDDa[i][j] + alp * WR[i][j];
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) trX += gi[i][j] * X[i][j];
  for (int i = 0; i < 3; ++i)
    for (int j = i; j < 3; ++j) {
      T xtf = X[i][j] - third * g[i][j] * trX;
      T aa = T(0), lie = T(0);
      for (int k = 0; k < 3; ++k) {
        aa += A[i][k] * Aud[k][j];
        lie += A[i][k] * db[j][k] + A[j][k] * db[i][k];
      }
      rhs[F_A + SYM[i][j]] = xtf + alp * (K * A[i][j] - T(2) * aa) + D.adv[F_A + SYM[i][j]] +
                             lie - two3 * A[i][j] * divb;
    }

  T rhsGam_noadv[3];
  for (int i = 0; i < 3; ++i) {
    T t1 = T(0), t2 = T(0), t3 = T(0), t4 = T(0), t5 = T(0), t6 = T(0), t7 = T(0);
    for (int j = 0; j < 3; ++j) {
      t1 += Auu[i][j] * da[j];                     // At^ij d_j alpha
      t3 += Auu[i][j] * dW[j];                     // At^ij d_j W
      t4 += gi[i][j] * dKT[j];                     // gt^ij d_j(2 Kh + Theta)
      t7 += Gd[j] * db[j][i];                      // Gt_d^j d_j beta^i
      T dd = T(0);
      for (int k = 0; k < 3; ++k) {
        t2 += Gu[i][j][k] * Auu[j][k];             // Gt^i_jk At^jk
        t5 += gi[j][k] * ddb[j][k][i];             // gt^jk d_j d_k beta^i
        dd += ddb[j][k][k];                        // d_j d_k beta^k
      }
      t6 += gi[i][j] * dd;
    }
    rhsGam_noadv[i] = -T(2) * t1 + T(2) * alp * (t2 - T(3) * t3 / W - third * t4) + t5 +
                      third * t6 - t7 + two3 * Gd[i] * divb -
                      T(2) * alp * P.kappa1 * (Gam[i] - Gd[i]);
    rhs[F_GAM + i] = rhsGam_noadv[i] + D.adv[F_GAM + i];
  }

  rhs[F_TH] = half * alp * (R - AA + two3 * K * K) - alp * P.kappa1 * (T(2) + P.kappa2) * Th +
              D.adv[F_TH];

  // ---- item 9: gauge (Eqs. 6-8) ---------------------------
  const T Ksrc = P.lapse_uses_khat ? Kh : K;      // reading C
  rhs[F_ALP] = D.adv[F_ALP] - T(2) * alp * Ksrc;
  for (int i = 0; i < 3; ++i) {
    rhs[F_BET + i] = D.adv[F_BET + i] + P.shift_coef * Bv[i];
    // (d_t - beta^j d_j) B^i = (d_t - beta^j d_j) Gt^i - eta B^i ; reading H: no KO inside
    rhs[F_B + i] = D.adv[F_B + i] + rhsGam_noadv[i] - P.eta * Bv[i];
  }

  // ---- item 10: add KO to every field -----------------------------------------
  for (int n = 0; n < NF; ++n) out[n] = rhs[n] + D.ko[n];
}



// ---------------------------------------------------------------------------------------------------
// Constraint monitor (Eqs. 20-21), vacuum:
//   H   = R + K^2 - K_ij K^ij                      (Eq. 20, rho_H = 0)
//   M^i = D_j ( K^ij - gamma^ij K )                (Eq. 21, J_i = 0)
// "R and D_j are the Ricci scalar and covariant derivative of gamma_ij": the oracle takes that
// literally. It rebuilds the PHYSICAL metric and extrinsic curvature and their derivatives from the evolved
// variables by the product rule (Eqs. 1-4: gamma_ij = gt_ij / W^2,
// K_ij = (At_ij + gt_ij K / 3) / W^2, K = K-hat + 2 Theta as in item 7) and then applies the textbook
// definitions (Christoffel symbols, Ricci tensor from their derivatives, covariant divergence). No conformal
// identity, no assumption det gt = 1 or tr At = 0, and nothing shared with the conformal Ricci of z4c_rhs_point.
// out[0] = H, out[1..3] = M^x, M^y, M^z.
template <class T>
inline void constraints_point(const T u[NF], const Derivs<T>& D, T out[4]) {
  const T W = u[F_W], K = u[F_KH] + T(2) * u[F_TH];
  T dW[3], ddW[3][3], dK[3];
  for (int k = 0; k < 3; ++k) {
    dW[k] = D.d1[F_W][k];
    dK[k] = D.d1[F_KH][k] + T(2) * D.d1[F_TH][k];
    for (int l = 0; l < 3; ++l) ddW[k][l] = D.d2[F_W][SYM[k][l]];
  }
  // physical metric gam_ij = gt_ij W^-2 and its first and second derivatives (product rule)
  const T w2 = T(1) / (W * W);                       // W^-2
  T dw2[3], ddw2[3][3];                              // d_k W^-2 = -2 W^-3 d_k W ; d_k d_l W^-2
  for (int k = 0; k < 3; ++k) dw2[k] = -T(2) * w2 / W * dW[k];
  for (int k = 0; k < 3; ++k)
    for (int l = 0; l < 3; ++l)
      ddw2[k][l] = T(6) * w2 / (W * W) * dW[k] * dW[l] - T(2) * w2 / W * ddW[k][l];
  T gam[3][3], dgam[3][3][3], ddgam[3][3][3][3], Kd[3][3], dKd[3][3][3];
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      const int n = SYM[i][j];
      const T gt = u[F_G + n];
      const T B = u[F_A + n] + gt * K / T(3);        // W^2 K_ij
      gam[i][j] = gt * w2;
      Kd[i][j] = B * w2;
      for (int k = 0; k < 3; ++k) {
        const T dgt = D.d1[F_G + n][k];
        dgam[k][i][j] = dgt * w2 + gt * dw2[k];
        const T dB = D.d1[F_A + n][k] + (dgt * K + gt * dK[k]) / T(3);
        dKd[k][i][j] = dB * w2 + B * dw2[k];
        for (int l = 0; l < 3; ++l)
          ddgam[k][l][i][j] = D.d2[F_G + n][SYM[k][l]] * w2 + dgt * dw2[l] + D.d1[F_G + n][l] * dw2[k] +
                              gt * ddw2[k][l];
      }
    }
  // inverse metric and its derivative: d_l gam^ij = - gam^ia gam^jb d_l gam_ab
  const T det = gam[0][0] * (gam[1][1] * gam[2][2] - gam[1][2] * gam[1][2]) -
                gam[0][1] * (gam[0][1] * gam[2][2] - gam[1][2] * gam[0][2]) +
                gam[0][2] * (gam[0][1] * gam[1][2] - gam[1][1] * gam[0][2]);
  T gi[3][3];
  gi[0][0] = (gam[1][1] * gam[2][2] - gam[1][2] * gam[1][2]) / det;
  gi[0][1] = (gam[0][2] * gam[1][2] - gam[0][1] * gam[2][2]) / det;
  gi[0][2] = (gam[0][1] * gam[1][2] - gam[0][2] * gam[1][1]) / det;
  gi[1][1] = (gam[0][0] * gam[2][2] - gam[0][2] * gam[0][2]) / det;
  gi[1][2] = (gam[0][1] * gam[0][2] - gam[0][0] * gam[1][2]) / det;
  gi[2][2] = (gam[0][0] * gam[1][1] - gam[0][1] * gam[0][1]) / det;
  gi[1][0] = gi[0][1]; gi[2][0] = gi[0][2]; gi[2][1] = gi[1][2];
  T dgi[3][3][3];
  for (int l = 0; l < 3; ++l)
    for (int i = 0; i < 3; ++i)
      for (int j = 0; j < 3; ++j) {
        T s = T(0);
        for (int a = 0; a < 3; ++a)
          for (int b = 0; b < 3; ++b) s += gi[i][a] * gi[j][b] * dgam[l][a][b];
        dgi[l][i][j] = -s;
      }
  // Christoffel symbols of gam: first kind Gl[c][i][j], second kind G[k][i][j], and d_l G^k_ij
  T Gl[3][3][3], dGl[3][3][3][3], G[3][3][3], dG[3][3][3][3];
  for (int c = 0; c < 3; ++c)
    for (int i = 0; i < 3; ++i)
      for (int j = 0; j < 3; ++j) {
        Gl[c][i][j] = (dgam[i][c][j] + dgam[j][c][i] - dgam[c][i][j]) / T(2);
        for (int l = 0; l < 3; ++l)
          dGl[l][c][i][j] = (ddgam[l][i][c][j] + ddgam[l][j][c][i] - ddgam[l][c][i][j]) / T(2);
      }
  for (int k = 0; k < 3; ++k)
    for (int i = 0; i < 3; ++i)
      for (int j = 0; j < 3; ++j) {
        T s = T(0);
        for (int c = 0; c < 3; ++c) s += gi[k][c] * Gl[c][i][j];
        G[k][i][j] = s;
        for (int l = 0; l < 3; ++l) {
          T t = T(0);
          for (int c = 0; c < 3; ++c) t += dgi[l][k][c] * Gl[c][i][j] + gi[k][c] * dGl[l][c][i][j];
          dG[l][k][i][j] = t;
        }
      }
  // Ricci tensor R_ij = d_k G^k_ij - d_j G^k_ik + G^k_kl G^l_ij - G^k_jl G^l_ik ; R = gam^ij R_ij
  T R = T(0);
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      T r = T(0);
      for (int k = 0; k < 3; ++k) {
        r += dG[k][k][i][j] - dG[j][k][i][k];
        for (int l = 0; l < 3; ++l) r += G[k][k][l] * G[l][i][j] - G[k][j][l] * G[l][i][k];
      }
      R += gi[i][j] * r;
    }
  // K_ij K^ij and the divergence D_j K^ij = gam^ia gam^jb (d_j K_ab - G^c_ja K_cb - G^c_jb K_ac)
  T KK = T(0);
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j)
      for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) KK += gi[i][a] * gi[j][b] * Kd[i][j] * Kd[a][b];
  out[0] = R + K * K - KK;
  for (int i = 0; i < 3; ++i) {
    T m = T(0);
    for (int j = 0; j < 3; ++j)
      for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) {
          T cov = dKd[j][a][b];
          for (int c = 0; c < 3; ++c) cov -= G[c][j][a] * Kd[c][b] + G[c][j][b] * Kd[a][c];
          m += gi[i][a] * gi[j][b] * cov;
        }
    for (int j = 0; j < 3; ++j) m -= gi[i][j] * dK[j];
    out[1 + i] = m;
  }
}

}  // namespace z4c_oracle
