// z4c_grid.hpp -- TEST INFRASTRUCTURE (part of the oracle; see z4c_oracle.hpp).
//
// Whole-patch drivers: periodic ghost fill, RHS over
// the active cells (items 3-10), classical RK4 (item 11).
// Plain triple loops; OpenMP over z-planes only so that the timed CPU baseline
// uses the host cores (no blocking, no fusion, no reordering).
#pragma once
#include <cmath>
#include "z4c_algebra.hpp"

namespace z4c_oracle {

inline long sy_of(const Patch& p) { return p.pitch; }
inline long sz_of(const Patch& p) { return p.pitch * (long)(p.ny + 2 * NG); }
inline long cell(const Patch& p, int I, int J, int Kk) {  // storage indices
  return ((long)Kk * (p.ny + 2 * NG) + J) * p.pitch + I;
}
inline int wrap(int i, int n) { return ((i % n) + n) % n; }

// item 2: every storage cell with any index outside the active range takes the
// value of the active cell with per-axis wrapped index. Reads active cells only.
template <class T> void fill_ghosts(const Patch& p, T* state) {
  const int sx = p.nx + 2 * NG, sy = p.ny + 2 * NG, sz = p.nz + 2 * NG;
  for (int n = 0; n < NF; ++n) {
    T* f = state + p.offset + (long)n * p.fstride;
#pragma omp parallel for schedule(static)
    for (int Kk = 0; Kk < sz; ++Kk)
      for (int J = 0; J < sy; ++J)
        for (int I = 0; I < sx; ++I) {
          const bool ghost = I < NG || I >= NG + p.nx || J < NG || J >= NG + p.ny || Kk < NG ||
                             Kk >= NG + p.nz;
          if (!ghost) continue;
          const int i = wrap(I - NG, p.nx), j = wrap(J - NG, p.ny), k = wrap(Kk - NG, p.nz);
          f[cell(p, I, J, Kk)] = f[cell(p, i + NG, j + NG, k + NG)];
        }
  }
}

// SURVEY.md 8(f) row f-2 (first half): reflection symmetry as a ghost-fill mode ("we impose reflection
// symmetry with respect to the equatorial plane z = 0"). Per axis a the mode is 0 = periodic (item 2) or 1 = mirror:
// the ghost cell at distance m+1 outside a face takes the value of the active cell at distance m inside it
// (cell-centred grid: the face lies half a cell outside the first active cell), times the parity of the field
// under x^a -> -x^a: -1 for the a-component of a vector (Gt^a, beta^a, B^a) and for tensor components with exactly
// one index a (gt, At), +1 otherwise. A corner cell reflected along several axes takes the product.
inline int field_parity(int f, int axis) {
  auto vec = [&](int f0) { return f >= f0 && f < f0 + 3 ? (f - f0 == axis ? -1 : 1) : 0; };
  auto ten = [&](int f0) {
    if (f < f0 || f >= f0 + 6) return 0;
    static const int IJ[6][2] = {{0, 0}, {0, 1}, {0, 2}, {1, 1}, {1, 2}, {2, 2}};
    const int n = (IJ[f - f0][0] == axis) + (IJ[f - f0][1] == axis);
    return n == 1 ? -1 : 1;
  };
  if (int s = vec(F_GAM)) return s;
  if (int s = vec(F_BET)) return s;
  if (int s = vec(F_B)) return s;
  if (int s = ten(F_G)) return s;
  if (int s = ten(F_A)) return s;
  return 1;   // W, K-hat, Theta, alpha
}
template <class T> void fill_ghosts_bc(const Patch& p, const int mode[3], T* state) {
  const int sx = p.nx + 2 * NG, sy = p.ny + 2 * NG, sz = p.nz + 2 * NG;
  const int nn[3] = {p.nx, p.ny, p.nz};
  for (int n = 0; n < NF; ++n) {
    T* f = state + p.offset + (long)n * p.fstride;
#pragma omp parallel for schedule(static)
    for (int Kk = 0; Kk < sz; ++Kk)
      for (int J = 0; J < sy; ++J)
        for (int I = 0; I < sx; ++I) {
          const int S[3] = {I, J, Kk};
          int src[3], sign = 1;
          bool ghost = false;
          for (int a = 0; a < 3; ++a) {
            const int i = S[a] - NG;
            if (i >= 0 && i < nn[a]) { src[a] = i; continue; }
            ghost = true;
            if (mode[a] == 0) src[a] = wrap(i, nn[a]);
            else { src[a] = i < 0 ? -1 - i : 2 * nn[a] - 1 - i; sign *= field_parity(n, a); }
          }
          if (!ghost) continue;
          f[cell(p, I, J, Kk)] = T(sign) * f[cell(p, src[0] + NG, src[1] + NG, src[2] + NG)];
        }
  }
}

// items 3-10 on every active cell. u is ghost-filled; rhs is written on active
// cells only (ghosts untouched).
template <class T>
void rhs_patch(const Patch& p, const Params<T>& P, const T* u, T* rhs) {
  const T* f[NF];
  for (int n = 0; n < NF; ++n) f[n] = u + p.offset + (long)n * p.fstride;
  const long sy = sy_of(p), sz = sz_of(p);
  const T h = T(p.dx);
#pragma omp parallel for schedule(static)
  for (int k = 0; k < p.nz; ++k)
    for (int j = 0; j < p.ny; ++j)
      for (int i = 0; i < p.nx; ++i) {
        const long c = cell(p, i + NG, j + NG, k + NG);
        Derivs<T> D;
        derivs_at<T>(f, c, sy, sz, h, P.ko_sigma, D);
        T uc[NF], out[NF];
        for (int n = 0; n < NF; ++n) uc[n] = f[n][c];
        z4c_rhs_point<T>(uc, D, P, out);
        for (int n = 0; n < NF; ++n) rhs[p.offset + (long)n * p.fstride + c] = out[n];
      }
}

// f-1: constraints (H, M^x, M^y, M^z) on every active cell of a ghost-filled state; con is a state-shaped buffer
// whose fields 0..3 receive the four constraints on active cells (everything else untouched).
template <class T>
void constraints_patch(const Patch& p, const T* u, T* con) {
  const T* f[NF];
  for (int n = 0; n < NF; ++n) f[n] = u + p.offset + (long)n * p.fstride;
  const long sy = sy_of(p), sz = sz_of(p);
  const T h = T(p.dx);
#pragma omp parallel for schedule(static)
  for (int k = 0; k < p.nz; ++k)
    for (int j = 0; j < p.ny; ++j)
      for (int i = 0; i < p.nx; ++i) {
        const long c = cell(p, i + NG, j + NG, k + NG);
        Derivs<T> D;
        derivs_at<T>(f, c, sy, sz, h, T(0), D);
        T uc[NF], out[4];
        for (int n = 0; n < NF; ++n) uc[n] = f[n][c];
        constraints_point<T>(uc, D, out);
        for (int n = 0; n < 4; ++n) con[p.offset + (long)n * p.fstride + c] = out[n];
      }
}

// Eq. 22: ||C||_2 = sqrt( sum_cells C^2 dV / sum_cells dV ) over all patches, plain loops
template <class T>
void constraint_norms(const Patch* ps, int np, const T* con, T norms[4]) {
  T vol = T(0), acc[4] = {T(0), T(0), T(0), T(0)};
  for (int q = 0; q < np; ++q) {
    const Patch& p = ps[q];
    const T dV = T(p.dx) * T(p.dx) * T(p.dx);
    for (int k = 0; k < p.nz; ++k)
      for (int j = 0; j < p.ny; ++j)
        for (int i = 0; i < p.nx; ++i) {
          const long c = cell(p, i + NG, j + NG, k + NG);
          vol += dV;
          for (int n = 0; n < 4; ++n) {
            const T v = con[p.offset + (long)n * p.fstride + c];
            acc[n] += v * v * dV;
          }
        }
  }
  for (int n = 0; n < 4; ++n) norms[n] = sqrt(acc[n] / vol);
}

// item 11, one substage. k = F(u_in) on active cells; table of item 11:
//   stage 1: u_out = u_n + (dt/2) k ; acc = k
//   stage 2: u_out = u_n + (dt/2) k ; acc = acc + 2k
//   stage 3: u_out = u_n + dt k     ; acc = acc + 2k
//   stage 4: S = (acc + k) c6 ; u_out = u_n + dt S ; acc = S
// Products are formed first, then added (no FMA: built with -ffp-contract=off).
template <class T>
void rk4_substep(const Patch& p, const Params<T>& P, int stage, const T* u_n, const T* u_in,
                 T* u_out, T* acc, T* kbuf /* scratch state */) {
  rhs_patch<T>(p, P, u_in, kbuf);
  const T dt = T(p.dt);
  const T c6 = T(1) / T(6);
  for (int n = 0; n < NF; ++n) {
    const long base = p.offset + (long)n * p.fstride;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < p.nz; ++k)
      for (int j = 0; j < p.ny; ++j)
        for (int i = 0; i < p.nx; ++i) {
          const long c = base + cell(p, i + NG, j + NG, k + NG);
          const T kk = kbuf[c];
          if (stage == 1) {
            T un = u_n[c];
            acc[c] = kk;
            u_out[c] = un + (dt / T(2)) * kk;
          } else if (stage == 2) {
            T un = u_n[c];
            acc[c] = acc[c] + T(2) * kk;
            u_out[c] = un + (dt / T(2)) * kk;
          } else if (stage == 3) {
            T un = u_n[c];
            acc[c] = acc[c] + T(2) * kk;
            u_out[c] = un + dt * kk;
          } else {
            T un = u_n[c];
            const T S = (acc[c] + kk) * c6;
            acc[c] = S;
            u_out[c] = un + dt * S;
          }
        }
  }
}

// item 11, full step: for s=1..4 { fill_ghosts(stage input); substep(s) };
// fill_ghosts(result). u: in state n (active cells), out state n+1, ghosts filled.
// work: 4 states (two stage buffers, acc, k scratch). On return work[2] (acc)
// holds the increment S per unit dt on active cells.
template <class T>
void rk4_step(const Patch* ps, int np, const Params<T>& P, T* u, T* w0, T* w1, T* acc, T* kbuf) {
  for (int q = 0; q < np; ++q) {
    const Patch& p = ps[q];
    fill_ghosts<T>(p, u);
    rk4_substep<T>(p, P, 1, u, u, w0, acc, kbuf);
    fill_ghosts<T>(p, w0);
    rk4_substep<T>(p, P, 2, u, w0, w1, acc, kbuf);
    fill_ghosts<T>(p, w1);
    rk4_substep<T>(p, P, 3, u, w1, w0, acc, kbuf);
    fill_ghosts<T>(p, w0);
    rk4_substep<T>(p, P, 4, u, w0, u, acc, kbuf);   // u_out aliases u_n: centre-only access
    fill_ghosts<T>(p, u);
  }
}

}  // namespace z4c_oracle
