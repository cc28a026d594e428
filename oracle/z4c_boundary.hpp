// z4c_boundary.hpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE (see z4c_oracle.hpp).
//
// Physical boundaries of a patch (section 2.2.2):
//   * the outgoing-wave (Sommerfeld) condition, Eq. 13:  d_t (r Q) + d_r (r Q) = 0  for every evolved variable Q
//     measured relative to its flat-space value, i.e.
//         d_t Q = - ( x^i / r ) d_i Q - Q / r ,     r = |x| ;
//   * reflection symmetry about a face, as in fill_ghosts_bc of z4c_grid.hpp, now per FACE.
//
// The paper gives no discretisation of Eq. 13. Reading ("Sommerfeld"):
//   - a face of a patch has one of four modes: PERIODIC, MIRROR, SOMMERFELD, NONE (ghosts supplied by somebody else,
//     e.g. the prolongation from the parent level);
//   - the BOUNDARY SHELL of a patch is the set of active cells within NG = 3 cells of a SOMMERFELD face. There the
//     right-hand side of ALL 25 evolved fields is the Sommerfeld expression above instead of the Z4c expression (the
//     Z4c stencils reach 3 cells, so no cell outside the shell ever reads a ghost cell behind a SOMMERFELD face);
//   - d_i Q in the shell is a 4th-order difference that uses only cells that exist: the centred stencil of item 3
//     where it fits, else the lopsided stencil of item 5 pointing inwards (-3 -10 18 -6 1)/12h, else the one-sided
//     stencil (-25 48 -36 16 -3)/12h; along an axis whose nearby face is MIRROR, PERIODIC or NONE the ghost cells are
//     valid and the centred stencil always fits. All in difference form (the flat value drops out of d_i Q).
//   - the flat-space values are 1 for W, gt_xx, gt_yy, gt_zz, alpha and 0 for everything else; the wave speed is 1;
//   - no Kreiss-Oliger term in the shell (its 7-point stencil does not fit).
// Coordinates: active cell (i, j, k) of a patch sits at origin + (i, j, k) h.
#pragma once
#include <cmath>
#include "z4c_grid.hpp"

namespace z4c_oracle {

enum { BC_PERIODIC = 0, BC_MIRROR = 1, BC_SOMMERFELD = 2, BC_NONE = 3 };

struct Boundary {
  double origin[3];   // coordinates of the centre of active cell (0, 0, 0)
  int face[6];        // x- x+ y- y+ z- z+
};

inline double sqrt_t(double v) { return std::sqrt(v); }   // built as double only (IEEE square root)
inline bool flat_is_one(int f) { return f == F_W || f == F_G || f == F_G + 3 || f == F_G + 5 || f == F_ALP; }

// Ghost fill with a mode per face. A storage cell outside the active range along one or more axes takes the active
// cell obtained by wrapping (PERIODIC) or reflecting (MIRROR, times the parity of the field) every such axis; if any
// of those axes is SOMMERFELD or NONE on that side, the cell is left alone. PERIODIC must be set on both faces of an axis.
template <class T> void fill_ghosts_faces(const Patch& p, const int face[6], T* state) {
  const int n[3] = {p.nx, p.ny, p.nz};
  for (int f = 0; f < NF; ++f) {
    T* u = state + p.offset + (long)f * p.fstride;
    for (int K = 0; K < p.nz + 2 * NG; ++K)
      for (int J = 0; J < p.ny + 2 * NG; ++J)
        for (int I = 0; I < p.nx + 2 * NG; ++I) {
          int idx[3] = {I - NG, J - NG, K - NG};
          bool ghost = false, skip = false;
          int sign = 1;
          for (int a = 0; a < 3; ++a) {
            if (idx[a] >= 0 && idx[a] < n[a]) continue;
            ghost = true;
            const int m = face[2 * a + (idx[a] < 0 ? 0 : 1)];
            if (m == BC_PERIODIC) idx[a] = wrap(idx[a], n[a]);
            else if (m == BC_MIRROR) { idx[a] = idx[a] < 0 ? -1 - idx[a] : 2 * n[a] - 1 - idx[a]; sign *= field_parity(f, a); }
            else skip = true;
          }
          if (!ghost || skip) continue;
          u[cell(p, I, J, K)] = T(sign) * u[cell(p, idx[0] + NG, idx[1] + NG, idx[2] + NG)];
        }
  }
}

inline bool in_shell(const Patch& p, const Boundary& b, int i, int j, int k) {
  return (b.face[0] == BC_SOMMERFELD && i < NG) || (b.face[1] == BC_SOMMERFELD && i >= p.nx - NG) ||
         (b.face[2] == BC_SOMMERFELD && j < NG) || (b.face[3] == BC_SOMMERFELD && j >= p.ny - NG) ||
         (b.face[4] == BC_SOMMERFELD && k < NG) || (b.face[5] == BC_SOMMERFELD && k >= p.nz - NG);
}

// 4th-order first derivative along one axis at active index i, using only indices in [lo, hi]; u(k) = sample at
// offset k from the point. inv12h = 1/(12 h).
template <class T, class U> T d1_bounded(U u, int i, int lo, int hi, T inv12h) {
  if (i - 2 >= lo && i + 2 <= hi)                                   // item 3
    return (T(8) * (u(1) - u(-1)) - (u(2) - u(-2))) * inv12h;
  const int s = (i - 2 < lo) ? 1 : -1;                              // the side the stencil leans to
  const T u0 = u(0);
  if (i - s >= lo && i - s <= hi)                                   // item 5 with sign s: one cell behind, three ahead
    return T(s) * ((((T(18) * (u(s) - u0) - T(3) * (u(-s) - u0)) - T(6) * (u(2 * s) - u0)) + (u(3 * s) - u0)) * inv12h);
  return T(s) * ((((T(48) * (u(s) - u0) - T(36) * (u(2 * s) - u0)) + T(16) * (u(3 * s) - u0)) - T(3) * (u(4 * s) - u0)) * inv12h);
}

// Eq. 13 on the boundary shell: rhs_f <- -( x^i d_i Q / r + Q / r ) for all 25 fields; cells outside the shell untouched
template <class T> void sommerfeld_rhs_patch(const Patch& p, const Boundary& b, const T* u, T* rhs) {
  const T h = T(p.dx), inv12h = T(1) / (T(12) * h);
  const int n[3] = {p.nx, p.ny, p.nz};
  int lo[3], hi[3];
  for (int a = 0; a < 3; ++a) {
    lo[a] = b.face[2 * a] == BC_SOMMERFELD ? 0 : -NG;
    hi[a] = b.face[2 * a + 1] == BC_SOMMERFELD ? n[a] - 1 : n[a] - 1 + NG;
  }
  const long st[3] = {1, sy_of(p), sz_of(p)};
  for (int f = 0; f < NF; ++f) {
    const T* uf = u + p.offset + (long)f * p.fstride;
    T* rf = rhs + p.offset + (long)f * p.fstride;
    const T flat = flat_is_one(f) ? T(1) : T(0);
    for (int k = 0; k < p.nz; ++k)
      for (int j = 0; j < p.ny; ++j)
        for (int i = 0; i < p.nx; ++i) {
          if (!in_shell(p, b, i, j, k)) continue;
          const long c = cell(p, i + NG, j + NG, k + NG);
          const int idx[3] = {i, j, k};
          T x[3], d[3];
          for (int a = 0; a < 3; ++a) {
            x[a] = T(b.origin[a]) + T(idx[a]) * h;
            const long s = st[a];
            d[a] = d1_bounded<T>([&](int q) { return uf[c + q * s]; }, idx[a], lo[a], hi[a], inv12h);
          }
          const T r = sqrt_t((x[0] * x[0] + x[1] * x[1]) + x[2] * x[2]);
          const T Q = uf[c] - flat;
          rf[c] = -((((x[0] * d[0] + x[1] * d[1]) + x[2] * d[2]) / r) + Q / r);
        }
  }
}

// RK4 substage (item 11 table) with physical boundaries: k = Z4c right-hand side outside the shell, Eq. 13 inside
template <class T>
void rk4_substep_bc(const Patch& p, const Params<T>& P, const Boundary& b, int stage, const T* u_n, const T* u_in,
                    T* u_out, T* acc, T* kbuf) {
  rhs_patch<T>(p, P, u_in, kbuf);               // shell cells: whatever the unfilled ghosts give; overwritten next
  sommerfeld_rhs_patch<T>(p, b, u_in, kbuf);
  const T dt = T(p.dt), c6 = T(1) / T(6);
  for (int n = 0; n < NF; ++n) {
    const long base = p.offset + (long)n * p.fstride;
    for (int k = 0; k < p.nz; ++k)
      for (int j = 0; j < p.ny; ++j)
        for (int i = 0; i < p.nx; ++i) {
          const long c = base + cell(p, i + NG, j + NG, k + NG);
          const T kk = kbuf[c], un = u_n[c];
          if (stage == 1) { acc[c] = kk; u_out[c] = un + (dt / T(2)) * kk; }
          else if (stage == 2) { acc[c] = acc[c] + T(2) * kk; u_out[c] = un + (dt / T(2)) * kk; }
          else if (stage == 3) { acc[c] = acc[c] + T(2) * kk; u_out[c] = un + dt * kk; }
          else { const T S = (acc[c] + kk) * c6; acc[c] = S; u_out[c] = un + dt * S; }
        }
  }
}

template <class T>
void rk4_step_bc(const Patch* ps, const Boundary* bs, int np, const Params<T>& P, T* u, T* w0, T* w1, T* acc, T* kbuf) {
  for (int q = 0; q < np; ++q) {
    const Patch& p = ps[q];
    const Boundary& b = bs[q];
    fill_ghosts_faces<T>(p, b.face, u);
    rk4_substep_bc<T>(p, P, b, 1, u, u, w0, acc, kbuf);
    fill_ghosts_faces<T>(p, b.face, w0);
    rk4_substep_bc<T>(p, P, b, 2, u, w0, w1, acc, kbuf);
    fill_ghosts_faces<T>(p, b.face, w1);
    rk4_substep_bc<T>(p, P, b, 3, u, w1, w0, acc, kbuf);
    fill_ghosts_faces<T>(p, b.face, w0);
    rk4_substep_bc<T>(p, P, b, 4, u, w0, u, acc, kbuf);
    fill_ghosts_faces<T>(p, b.face, u);
  }
}

}  // namespace z4c_oracle
