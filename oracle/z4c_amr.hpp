// z4c_amr.hpp -- TEST INFRASTRUCTURE (part of the oracle; see z4c_oracle.hpp).
//
// SURVEY.md 8(f) row f-3, spatial inter-level operators of the box-in-box hierarchy:
// "Successive levels are related by a 2:1 refinement ratio on a cell centered staggered grid"; prolongation
// "interpolates from the parent level with a sixth order Lagrange interpolation"; restriction "overwrites each
// coarse cell covered by a finer level with a fourth order Lagrange interpolation of the fine data".
// Geometry (reading): along each axis the parent cell with active index org + m holds the child cells
// 2m and 2m+1; its centre lies midway between them. Interpolation is the tensor product of 1-D Lagrange
// interpolation, written out from the textbook basis L_j(s) = prod_{k != j} (s - t_k) / (t_j - t_k) on the nearest
// nodes that are symmetric about the target. Time interpolation and the subcycling driver are not built.
#pragma once
#include "z4c_grid.hpp"

namespace z4c_oracle {

// Lagrange basis on NP consecutive integer nodes t0, t0+1, ... evaluated at s (s, t in units of the node spacing)
template <class T, int NP> inline void lagrange(int t0, T s, T w[NP]) {
  for (int j = 0; j < NP; ++j) {
    T num = T(1), den = T(1);
    for (int k = 0; k < NP; ++k)
      if (k != j) { num = num * (s - T(t0 + k)); den = den * T(j - k); }
    w[j] = num / den;
  }
}

// Restriction: every parent cell (org + m) with 0 <= m < n_child / 2 on all three axes takes the 4-point-per-axis
// Lagrange interpolant of the child data at its centre, s = 1/2 between child cells 2m and 2m+1 (nodes 2m-1 .. 2m+2:
// the child's ghost cells are read at the patch edges and must be valid). All NF fields.
template <class T>
void restrict_patch(const Patch& pp, const Patch& pc, const int org[3], T* u_parent, const T* u_child) {
  T w[4];
  lagrange<T, 4>(-1, T(1) / T(2), w);
  for (int n = 0; n < NF; ++n) {
    T* fp = u_parent + pp.offset + (long)n * pp.fstride;
    const T* fc = u_child + pc.offset + (long)n * pc.fstride;
    for (int mz = 0; mz < pc.nz / 2; ++mz)
      for (int my = 0; my < pc.ny / 2; ++my)
        for (int mx = 0; mx < pc.nx / 2; ++mx) {
          T sz = T(0);
          for (int kz = 0; kz < 4; ++kz) {
            T sy = T(0);
            for (int ky = 0; ky < 4; ++ky) {
              T sx = T(0);
              for (int kx = 0; kx < 4; ++kx)
                sx = sx + w[kx] * fc[cell(pc, 2 * mx - 1 + kx + NG, 2 * my - 1 + ky + NG, 2 * mz - 1 + kz + NG)];
              sy = sy + w[ky] * sx;
            }
            sz = sz + w[kz] * sy;
          }
          fp[cell(pp, org[0] + mx + NG, org[1] + my + NG, org[2] + mz + NG)] = sz;
        }
  }
}

// Prolongation of the refinement-boundary zones: every GHOST cell of the child (all faces, edges, corners) takes the
// 6-point-per-axis Lagrange interpolant of the parent data at its centre. Child cell i (any integer) sits at parent
// coordinate org + floor(i/2) -+ 1/4 (minus for even i, plus for odd i); nodes: the six parent cells symmetric about
// the parent interval that contains it. Parent ghost cells may be read and must be valid. All NF fields.
template <class T> inline void prolong_axis(int i, int org, int& j0, T w[6]) {
  const int m = (i >= 0) ? i / 2 : -((-i + 1) / 2);      // floor(i / 2)
  const bool odd = (i - 2 * m) == 1;
  j0 = org + m + (odd ? -2 : -3);                         // first of the six parent cells (active index)
  lagrange<T, 6>(odd ? -2 : -3, odd ? T(1) / T(4) : -T(1) / T(4), w);
}
template <class T>
void prolong_ghosts(const Patch& pp, const Patch& pc, const int org[3], const T* u_parent, T* u_child) {
  const int sx = pc.nx + 2 * NG, sy = pc.ny + 2 * NG, sz = pc.nz + 2 * NG;
  for (int n = 0; n < NF; ++n) {
    const T* fp = u_parent + pp.offset + (long)n * pp.fstride;
    T* fc = u_child + pc.offset + (long)n * pc.fstride;
    for (int Kk = 0; Kk < sz; ++Kk)
      for (int J = 0; J < sy; ++J)
        for (int I = 0; I < sx; ++I) {
          const int i = I - NG, j = J - NG, k = Kk - NG;
          const bool ghost = i < 0 || i >= pc.nx || j < 0 || j >= pc.ny || k < 0 || k >= pc.nz;
          if (!ghost) continue;
          int x0, y0, z0;
          T wx[6], wy[6], wz[6];
          prolong_axis<T>(i, org[0], x0, wx);
          prolong_axis<T>(j, org[1], y0, wy);
          prolong_axis<T>(k, org[2], z0, wz);
          T az = T(0);
          for (int kz = 0; kz < 6; ++kz) {
            T ay = T(0);
            for (int ky = 0; ky < 6; ++ky) {
              T ax = T(0);
              for (int kx = 0; kx < 6; ++kx)
                ax = ax + wx[kx] * fp[cell(pp, x0 + kx + NG, y0 + ky + NG, z0 + kz + NG)];
              ay = ay + wy[ky] * ax;
            }
            az = az + wz[kz] * ay;
          }
          fc[cell(pc, I, J, Kk)] = az;
        }
  }
}

}  // namespace z4c_oracle
