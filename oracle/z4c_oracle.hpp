// z4c_oracle.hpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, obviously-correct CPU statement of the hot path of SACRA-K's
// spacetime evolution (arxiv/paper_2607_08743): periodic ghost fill, 4th-order
// finite differences, 6th-derivative Kreiss-Oliger dissipation, the Z4c/BSSN
// right-hand side with moving-puncture gauge, and the classical RK4 step.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
// reference leg may build, link, import or execute anything under oracle/.
// It shares no code with paper_2607_08743_b200/ (the CUDA path) and neither
// includes the other.
//
// What the paper fixes (PAPER.md = /root/reference/PAPER.md at authoring time):
//   variables W, gt_ij, K, At_ij, Gt^i      Eqs. 1-5
//   Z4c: extra scalar Theta, kappa1, kappa2 PAPER.md:63 (equations deferred to
//                                           Hilditch et al. 2013; written out in
//                                           SURVEY.md 8(c) items 7-8, restated here)
//   1+log slicing, Gamma driver             Eqs. 6-8
//   evolved set (25 fields)
//   RK4, 4th-order centred FD, 4th-order upwind along the shift,
//   "sixth order" KO dissipation
//   -fno-fast-math, -ffp-contract=off
// Readings of silent / garbled points are listed in DESIGN.md ("Readings").
//
// PARITY UNPINNED with respect to the paper: (C) whether
// Eq. 6's source is K-hat or K-hat+2*Theta (switch lapse_uses_khat); the placement
// of the kappa1/kappa2 coefficients. Both are pinned against SURVEY.md 8(c)'s
// linear-response table (tests/test_oracle_linear_response.py), and the Theta
// coefficient against the constraint monitor; the paper itself prints neither.
//
// Everything is templated on the scalar type so that the same source builds
// as double (the oracle) and as __float128 (round-off referee).
#pragma once
#include <cstdint>
#include <vector>

namespace z4c_oracle {

constexpr int NF = 25;   // PAPER.md:73 : 1+6+1+6+3+1+1+3+3
constexpr int NG = 3;    // ghost zones (BASELINE.json; stencil reach of upwind and KO)

// field indices (order fixed in include/sacra.h; restated, not included)
enum { F_W = 0, F_G = 1 /*xx xy xz yy yz zz*/, F_KH = 7, F_A = 8, F_GAM = 14,
       F_TH = 17, F_ALP = 18, F_BET = 19, F_B = 22 };

// symmetric-pair index: (i,j) -> 0..5 in the order xx xy xz yy yz zz
static const int SYM[3][3] = {{0, 1, 2}, {1, 3, 4}, {2, 4, 5}};

struct Patch {
  int nx, ny, nz;        // active cells
  long pitch;            // doubles per x-row  (>= nx+2*NG)
  long fstride;          // doubles between fields
  long offset;           // doubles from state base to field 0 of this patch
  double dx, dt;
};

template <class T> struct Params {
  T kappa1, kappa2, eta, shift_coef, ko_sigma;
  int lapse_uses_khat;
};

// ---------------------------------------------------------------------------
// Stencils. u points at the centre value, s is the stride (in elements) along
// the axis. Operation order is the canonical one of SURVEY.md 8(c) items 3-6.
// ---------------------------------------------------------------------------

// item 3: centred first derivative, 4th order
//   D_a u = [ 8 (u+1 - u-1) - (u+2 - u-2) ] / (12 h)
template <class T> inline T d1c(const T* u, long s, T inv12h) {
  T a = u[s] - u[-s];
  T b = u[2 * s] - u[-2 * s];
  return (T(8) * a - b) * inv12h;
}

// item 4: centred second derivative, diagonal, 4th order
//   D_aa u = [ 16 ((u+1-u0)+(u-1-u0)) - ((u+2-u0)+(u-2-u0)) ] / (12 h^2)
template <class T> inline T d2c(const T* u, long s, T inv12h2) {
  T u0 = u[0];
  T p1 = (u[s] - u0) + (u[-s] - u0);
  T p2 = (u[2 * s] - u0) + (u[-2 * s] - u0);
  return (T(16) * p1 - p2) * inv12h2;
}

// item 4: mixed second derivative D_ab = D_a(D_b u), a < b; the inner
// (unscaled) difference runs along the LATER axis b.
template <class T> inline T d2m(const T* u, long sa, long sb, T inv144h2) {
  auto e = [&](long o) {
    const T* v = u + o;
    return T(8) * (v[sb] - v[-sb]) - (v[2 * sb] - v[-2 * sb]);
  };
  T a = e(sa) - e(-sa);
  T b = e(2 * sa) - e(-2 * sa);
  return (T(8) * a - b) * inv144h2;
}

// item 5: lopsided 4th-order upwind derivative; bias follows the sign of the
// shift. sg = +1 for beta >= 0 (reading I), v_k = u(x + sg k h).
//   D^up u = sg [ ((18 (v1-v0) - 3 (v-1-v0)) - 6 (v2-v0)) + (v3-v0) ] / (12 h)
template <class T> inline T d1up(const T* u, long s, T beta, T inv12h) {
  long sg = (beta >= T(0)) ? 1 : -1;
  T v0 = u[0];
  T vm1 = u[-sg * s], v1 = u[sg * s], v2 = u[2 * sg * s], v3 = u[3 * sg * s];
  T r = ((T(18) * (v1 - v0) - T(3) * (vm1 - v0)) - T(6) * (v2 - v0)) + (v3 - v0);
  return (T(sg) * r) * inv12h;
}

// item 6: Kreiss-Oliger 6th-derivative numerator along one axis
//   q = (p3 - 6 p2) + 15 p1,  p_k = (u+k - u0) + (u-k - u0)
template <class T> inline T koq(const T* u, long s) {
  T u0 = u[0];
  T p1 = (u[s] - u0) + (u[-s] - u0);
  T p2 = (u[2 * s] - u0) + (u[-2 * s] - u0);
  T p3 = (u[3 * s] - u0) + (u[-3 * s] - u0);
  return (p3 - T(6) * p2) + T(15) * p1;
}

// Per-point derivative bundle handed to the algebra.
template <class T> struct Derivs {
  T d1[NF][3];   // centred D_a f            (used: W, gt, Kh, Gam, Th, alpha, beta)
  T d2[NF][6];   // centred D_ab f, SYM order (used: W, gt, alpha, beta)
  T adv[NF];     // beta^k D^up_k f          (all fields)
  T ko[NF];      // Q f                      (all fields)
};

// Fill a Derivs bundle from a ghost-filled state at storage index c (centre).
template <class T>
inline void derivs_at(const T* const f[NF], long c, long sy, long sz, T h, T sigma,
                      Derivs<T>& D) {
  const long st[3] = {1, sy, sz};
  const T inv12h = T(1) / (T(12) * h);
  const T inv12h2 = T(1) / (T(12) * h * h);
  const T inv144h2 = T(1) / (T(144) * h * h);
  const T kofac = sigma / (T(64) * h);
  T beta[3];
  for (int a = 0; a < 3; ++a) beta[a] = f[F_BET + a][c];
  for (int n = 0; n < NF; ++n) {
    const T* u = f[n] + c;
    for (int a = 0; a < 3; ++a) D.d1[n][a] = d1c(u, st[a], inv12h);
    for (int a = 0; a < 3; ++a)
      for (int b = a; b < 3; ++b)
        D.d2[n][SYM[a][b]] = (a == b) ? d2c(u, st[a], inv12h2)
                                      : d2m(u, st[a], st[b], inv144h2);
    // item 5: A_f = (beta^x Dup_x f + beta^y Dup_y f) + beta^z Dup_z f
    D.adv[n] = (beta[0] * d1up(u, st[0], beta[0], inv12h) +
                beta[1] * d1up(u, st[1], beta[1], inv12h)) +
               beta[2] * d1up(u, st[2], beta[2], inv12h);
    // item 6: Q f = ((q_x + q_y) + q_z) sigma / (64 h)
    D.ko[n] = ((koq(u, st[0]) + koq(u, st[1])) + koq(u, st[2])) * kofac;
  }
}

}  // namespace z4c_oracle
