// z4c_subcycle.hpp -- TEST INFRASTRUCTURE (part of the oracle; see z4c_oracle.hpp).
//
// SURVEY.md 8(f) row f-3, the remaining parts: time interpolation of the refinement-boundary data and the
// Berger-Oliger subcycling step of a parent / child pair.
//   "Each finer level is advanced with a halved time step and therefore takes twice as many substeps per coarse step."
//   "In time, the refinement boundary data needed at the substeps are interpolated between the parent time levels, at
//    first order in the very first time step of a run and at second order thereafter."
// Reading ("Subcycling"), with theta = (t - t_n) / dt_parent:
//   * first order: the straight line through the parent states U^n (theta = 0) and U^{n+1} (theta = 1);
//     second order: the parabola through U^{n-1}, U^n, U^{n+1} (theta = -1, 0, 1), Lagrange basis written out;
//   * the interpolation in time is done first, cell by cell on the parent (every storage cell, ghosts included),
//     the spatial prolongation (z4c_amr.hpp) second;
//   * one step of the pair:  (1) the parent takes one RK4 step t_n -> t_n + dt (its own boundary modes);
//     (2) the child takes two RK4 steps of dt / 2; before EVERY substage of the child the ghost cells of the stage
//     input are prolonged from the parent data interpolated to the substage time (classical RK4 stage times
//     t, t + dt_c/2, t + dt_c/2, t + dt_c), i.e. theta = (m + c_s) / 2, m = 0, 1, c = (0, 1/2, 1/2, 1);
//     (3) the child's ghosts are prolonged from the new parent state (theta = 1; the restriction stencil reads them at
//     the edge of the covered region), the child is restricted onto the parent's covered cells, and the parent's ghosts
//     are refilled.
//   On return `u_parent_prev`, if given, holds the parent state the step started from (the U^{n-1} of the next step).
#pragma once
#include <vector>
#include "z4c_amr.hpp"
#include "z4c_boundary.hpp"

namespace z4c_oracle {

// weights of the parent time levels at theta: n = 2 -> (U^n, U^{n+1}); n = 3 -> (U^{n-1}, U^n, U^{n+1})
template <class T> inline void time_weights(int n, T theta, T w[3]) {
  if (n == 2) { w[0] = T(1) - theta; w[1] = theta; w[2] = T(0); }
  else lagrange<T, 3>(-1, theta, w);
}

// out = (w0 u0 + w1 u1) [+ w2 u2] on every storage cell of the patch (ghosts included), all fields
template <class T> void lincomb_patch(const Patch& p, int n, const T* const u[3], const T w[3], T* out) {
  for (int f = 0; f < NF; ++f)
    for (int K = 0; K < p.nz + 2 * NG; ++K)
      for (int J = 0; J < p.ny + 2 * NG; ++J)
        for (int I = 0; I < p.nx + 2 * NG; ++I) {
          const long c = p.offset + (long)f * p.fstride + cell(p, I, J, K);
          T s = w[0] * u[0][c] + w[1] * u[1][c];
          if (n == 3) s = s + w[2] * u[2][c];
          out[c] = s;
        }
}

template <class T>
void subcycle_step(const Patch& pp, const Patch& pc, const int org[3], const Params<T>& P, const Boundary& bp,
                   T* u_parent, T* u_parent_prev /* U^{n-1} or nullptr */, bool have_prev, T* u_child,
                   long n_parent, long n_child) {
  std::vector<T> old(u_parent, u_parent + n_parent), tmp(n_parent, T(0));
  std::vector<T> wk(4 * n_parent, T(0)), wc(4 * n_child, T(0));
  // (1) parent
  rk4_step_bc<T>(&pp, &bp, 1, P, u_parent, wk.data(), wk.data() + n_parent, wk.data() + 2 * n_parent, wk.data() + 3 * n_parent);
  // (2) child: two steps of dt / 2
  const int nlev = have_prev ? 3 : 2;
  const T* lev[3];
  if (have_prev) { lev[0] = u_parent_prev; lev[1] = old.data(); lev[2] = u_parent; }
  else { lev[0] = old.data(); lev[1] = u_parent; lev[2] = nullptr; }
  T* w0 = wc.data();
  T* w1 = wc.data() + n_child;
  T* acc = wc.data() + 2 * n_child;
  T* kbuf = wc.data() + 3 * n_child;
  const T cs[4] = {T(0), T(1) / T(2), T(1) / T(2), T(1)};
  for (int m = 0; m < 2; ++m) {
    const T* in[4] = {u_child, w0, w1, w0};
    T* out[4] = {w0, w1, w0, u_child};
    for (int s = 0; s < 4; ++s) {
      T w[3];
      time_weights<T>(nlev, (T(m) + cs[s]) / T(2), w);
      lincomb_patch<T>(pp, nlev, lev, w, tmp.data());
      prolong_ghosts<T>(pp, pc, org, tmp.data(), const_cast<T*>(in[s]));
      rk4_substep<T>(pc, P, s + 1, u_child, in[s], out[s], acc, kbuf);
    }
  }
  // (3) child ghosts at the new time (the restriction reads them at the edge of the covered region), restriction,
  // parent ghosts
  prolong_ghosts<T>(pp, pc, org, u_parent, u_child);
  restrict_patch<T>(pp, pc, org, u_parent, u_child);
  fill_ghosts_faces<T>(pp, bp.face, u_parent);
  if (u_parent_prev) for (long i = 0; i < n_parent; ++i) u_parent_prev[i] = old[i];
}

}  // namespace z4c_oracle

// ---- hierarchy of nested levels ("fixed levels, each a single cubic patch"; level l + 1 is the child of
// level l, half its spacing and time step). Recursive Berger-Oliger step, the pair step above applied at every level:
//   step(0):   U_0 takes one RK4 step with its boundary modes.
//   step(l>0): level l takes one RK4 step of dt_l; the ghosts of every substage input are prolonged from the parent's time
//              levels (U^{n-1}, U^n, U^{n+1} of level l - 1; first order while the parent has no U^{n-1} yet) at
//              theta = (m + c_s) / 2, m = 0, 1 the number of this step inside the parent's.
//   after a step of level l: if it has a child, level l > 0 first refills its own ghosts at the time just reached (the
//              child's prolongation box may read them), the child takes two steps (recursively), then the child's ghosts are
//              prolonged from the new U_l, the child is restricted onto U_l and U_l's ghosts are refilled (level 0: its
//              boundary modes; level l > 0: prolongation from its parent at the time just reached -- theta = (m + 1) / 2).
// With two levels this is subcycle_step(), bit for bit.
namespace z4c_oracle {

template <class T> struct Level {
  Patch p;
  int org[3];          // position in the parent (unused for level 0)
  T* u;                // state
  T* prev;             // U^{n-1} of this level (valid when nsteps > 0)
  long n;              // doubles per state
  long nsteps;         // steps this level has taken
  std::vector<T> old;  // U^n during a step
};

template <class T>
void hierarchy_advance(std::vector<Level<T>>& L, int l, const Params<T>& P, const Boundary& b0, int m) {
  Level<T>& me = L[l];
  me.old.assign(me.u, me.u + me.n);
  std::vector<T> wk(4 * me.n, T(0));
  T* w0 = wk.data();
  T* w1 = wk.data() + me.n;
  T* acc = wk.data() + 2 * me.n;
  T* kbuf = wk.data() + 3 * me.n;
  auto parent_ghosts = [&](T theta, T* target) {      // ghosts of `target` from the parent's time levels at theta
    Level<T>& pa = L[l - 1];
    const int nlev = pa.nsteps > 0 ? 3 : 2;
    const T* lev[3];
    if (nlev == 3) { lev[0] = pa.prev; lev[1] = pa.old.data(); lev[2] = pa.u; }
    else { lev[0] = pa.old.data(); lev[1] = pa.u; lev[2] = nullptr; }
    T w[3];
    time_weights<T>(nlev, theta, w);
    std::vector<T> tmp(pa.n, T(0));
    lincomb_patch<T>(pa.p, nlev, lev, w, tmp.data());
    prolong_ghosts<T>(pa.p, me.p, me.org, tmp.data(), target);
  };
  if (l == 0) {
    rk4_step_bc<T>(&me.p, &b0, 1, P, me.u, w0, w1, acc, kbuf);
  } else {
    const T cs[4] = {T(0), T(1) / T(2), T(1) / T(2), T(1)};
    const T* in[4] = {me.u, w0, w1, w0};
    T* out[4] = {w0, w1, w0, me.u};
    for (int s = 0; s < 4; ++s) {
      parent_ghosts((T(m) + cs[s]) / T(2), const_cast<T*>(in[s]));
      rk4_substep<T>(me.p, P, s + 1, me.u, in[s], out[s], acc, kbuf);
    }
  }
  if (l + 1 < (int)L.size()) {
    // An intermediate level refreshes its own ghosts at the time just reached BEFORE its child advances: stage 4
    // wrote active cells only, and the child's time-interpolated prolongation box (parent cells org - 4 ..
    // org + n/2 + 3) reaches into these ghosts when the child sits within 4 cells of this level's edge. (Level 0's
    // rk4_step_bc ends with its own fill.) PAPER.md:109: the child's buffer data come from the parent AT the
    // substage's time, which needs every parent cell the stencil reads to be at U^{n+1}.
    if (l > 0) parent_ghosts((T(m) + T(1)) / T(2), me.u);
    hierarchy_advance<T>(L, l + 1, P, b0, 0);
    hierarchy_advance<T>(L, l + 1, P, b0, 1);
    Level<T>& ch = L[l + 1];
    prolong_ghosts<T>(me.p, ch.p, ch.org, me.u, ch.u);
    restrict_patch<T>(me.p, ch.p, ch.org, me.u, ch.u);
  }
  if (l == 0) fill_ghosts_faces<T>(me.p, b0.face, me.u);
  else parent_ghosts((T(m) + T(1)) / T(2), me.u);
  for (long i = 0; i < me.n; ++i) me.prev[i] = me.old[i];
  me.nsteps += 1;
}

}  // namespace z4c_oracle
