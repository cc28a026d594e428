"""ctypes wrapper of the oracle library (TEST INFRASTRUCTURE; see z4c_oracle.hpp).

May be imported only by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference leg. It takes numpy arrays and plain patch
descriptors (any object with nx ny nz pitch_x field_stride patch_offset dx dt).
"""
from __future__ import annotations

import ctypes as C
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import build as _build  # noqa: E402  (oracle/build.py)

NF = 25


class OrcPatch(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("ng", C.c_int32),
                ("pitch_x", C.c_int64), ("field_stride", C.c_int64), ("patch_offset", C.c_int64),
                ("dx", C.c_double), ("dt", C.c_double)]


class OrcParams(C.Structure):
    _fields_ = [("kappa1", C.c_double), ("kappa2", C.c_double), ("eta", C.c_double),
                ("shift_coef", C.c_double), ("ko_sigma", C.c_double),
                ("lapse_uses_khat", C.c_int32)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def _patches(ps):
    arr = (OrcPatch * len(ps))()
    for a, p in zip(arr, ps):
        a.nx, a.ny, a.nz, a.ng = p.nx, p.ny, p.nz, 3
        a.pitch_x, a.field_stride, a.patch_offset = p.pitch_x, p.field_stride, p.patch_offset
        a.dx, a.dt = p.dx, p.dt
    return arr


def _params(d):
    return OrcParams(d["kappa1"], d["kappa2"], d["eta"], d["shift_coef"], d["ko_sigma"],
                     int(d.get("lapse_uses_khat", 1)))


def _p(a):
    assert a.dtype == np.float64 and a.flags.c_contiguous
    return a.ctypes.data_as(C.POINTER(C.c_double))


def num_threads() -> int:
    return lib().orc_num_threads()


def set_threads(n: int):
    lib().orc_set_threads(int(n))


def fill_ghosts(ps, u):
    lib().orc_fill_ghosts(_patches(ps), len(ps), _p(u))


def z4c_rhs(ps, prm, u, quad=False):
    """RHS (incl. KO) on the active cells of a ghost-filled state; zeros elsewhere."""
    rhs = np.zeros_like(u)
    pr = _params(prm)
    if quad:
        lib().orc_z4c_rhs_q(_patches(ps), len(ps), C.byref(pr), _p(u), _p(rhs), C.c_int64(u.size))
    else:
        lib().orc_z4c_rhs(_patches(ps), len(ps), C.byref(pr), _p(u), _p(rhs))
    return rhs


def rk4_substep(ps, prm, stage, u_n, u_in, u_out, acc):
    kbuf = np.zeros_like(u_in)
    pr = _params(prm)
    lib().orc_rk4_substep(_patches(ps), len(ps), C.byref(pr), int(stage), _p(u_n), _p(u_in),
                          _p(u_out), _p(acc), _p(kbuf))


def rk4_step(ps, prm, u, quad=False):
    """Advance u in place by one RK4 step (ghosts filled on return).
    Returns S, the increment per unit dt, on active cells (zeros elsewhere)."""
    pr = _params(prm)
    n = u.size
    if quad:
        S = np.zeros_like(u)
        lib().orc_rk4_step_q(_patches(ps), len(ps), C.byref(pr), _p(u), _p(S), C.c_int64(n))
        return S
    work = np.zeros(4 * n)
    lib().orc_rk4_step(_patches(ps), len(ps), C.byref(pr), _p(u), _p(work), C.c_int64(n))
    return work[2 * n:3 * n].copy()


def rhs_point(prm, u, d1, d2, adv, ko):
    """Point-wise algebra with caller-supplied derivatives. u[25], d1[25,3], d2[25,6]."""
    u, d1, d2, adv, ko = (np.ascontiguousarray(a, dtype=np.float64) for a in (u, d1, d2, adv, ko))
    assert u.shape == (NF,) and d1.shape == (NF, 3) and d2.shape == (NF, 6)
    out = np.zeros(NF)
    pr = _params(prm)
    lib().orc_rhs_point(C.byref(pr), _p(u), _p(d1), _p(d2), _p(adv), _p(ko), _p(out))
    return out


def derivs_field(p, u, f, i, j, k, sigma):
    """(d1[3], d2[6], adv, ko) of field f at active cell (i,j,k) of patch p."""
    out = np.zeros(11)
    lib().orc_derivs_field(C.byref(_patches([p])[0]), _p(u), int(f), int(i), int(j), int(k),
                           C.c_double(sigma), _p(out))
    return out[0:3], out[3:9], out[9], out[10]


def count_ops():
    """(adds, muls, divs) of the point-wise algebra at one point, and of the oracle's derivative bundle of one
    field (all 3 D1, 6 D2, upwind advection, KO) -- the oracle source instantiated with a counting scalar."""
    c = (C.c_long * 6)()
    lib().orc_count_ops(c)
    return tuple(c[:3]), tuple(c[3:])


def constraints(ps, u):
    """H, M^x, M^y, M^z (Eqs. 20-21, vacuum) on the active cells: a state-shaped buffer, fields 0..3."""
    u = np.ascontiguousarray(u, dtype=np.float64)
    con = np.zeros_like(u)
    lib().orc_constraints(_patches(ps), len(ps), _p(u), _p(con))
    return con


def constraint_norms(ps, con):
    """volume-normalised L2 norms of the four constraints over all patches (Eq. 22)"""
    out = np.zeros(4)
    lib().orc_constraint_norms(_patches(ps), len(ps), _p(np.ascontiguousarray(con, dtype=np.float64)), _p(out))
    return out


def constraints_point(u, d1, d2):
    """constraints at one point from caller-supplied derivatives. u[25], d1[25,3], d2[25,6]."""
    u, d1, d2 = (np.ascontiguousarray(a, dtype=np.float64) for a in (u, d1, d2))
    assert u.shape == (NF,) and d1.shape == (NF, 3) and d2.shape == (NF, 6)
    out = np.zeros(4)
    lib().orc_constraints_point(_p(u), _p(d1), _p(d2), _p(out))
    return out


def fill_ghosts_bc(ps, mode, u):
    """ghost fill with per-axis mode (0 periodic, 1 mirror with field parity), in place; mode = (mx, my, mz)"""
    m = (C.c_int32 * 3)(*[int(v) for v in mode])
    lib().orc_fill_ghosts_bc(_patches(ps), len(ps), m, _p(u))
    return u


def restrict(parent, child, org, u_parent, u_child):
    """4th-order Lagrange restriction of the child's active cells onto the covered parent cells, in place on
    u_parent; org = parent active index of the coarse cell that holds child cells 0, 1 (per axis)."""
    o = (C.c_int32 * 3)(*[int(v) for v in org])
    lib().orc_restrict(C.byref(_patches([parent])[0]), C.byref(_patches([child])[0]), o, _p(u_parent), _p(u_child))
    return u_parent


def prolong_ghosts(parent, child, org, u_parent, u_child):
    """6th-order Lagrange prolongation of the parent onto every ghost cell of the child, in place on u_child"""
    o = (C.c_int32 * 3)(*[int(v) for v in org])
    lib().orc_prolong_ghosts(C.byref(_patches([parent])[0]), C.byref(_patches([child])[0]), o, _p(u_parent),
                             _p(u_child))
    return u_child


# ---- physical boundaries: face modes 0 periodic, 1 mirror, 2 Sommerfeld, 3 none ---------------------
BC_PERIODIC, BC_MIRROR, BC_SOMMERFELD, BC_NONE = 0, 1, 2, 3


class OrcBoundary(C.Structure):
    _fields_ = [("origin", C.c_double * 3), ("face", C.c_int32 * 6)]


def _boundaries(bs):
    """bs: list of (origin[3], face[6]) per patch"""
    arr = (OrcBoundary * len(bs))()
    for a, (o, f) in zip(arr, bs):
        for i in range(3):
            a.origin[i] = float(o[i])
        for i in range(6):
            a.face[i] = int(f[i])
    return arr


def fill_ghosts_faces(ps, bs, u):
    lib().orc_fill_ghosts_faces(_patches(ps), _boundaries(bs), len(ps), _p(u))
    return u


def sommerfeld_rhs(ps, bs, u, rhs=None):
    """Eq. 13 on the boundary shell (active cells within 3 cells of a Sommerfeld face); other cells of rhs untouched"""
    if rhs is None:
        rhs = np.zeros_like(u)
    lib().orc_sommerfeld_rhs(_patches(ps), _boundaries(bs), len(ps), _p(u), _p(rhs))
    return rhs


def d1_bounded(u, i, lo, hi, h):
    lib().orc_d1_bounded.restype = C.c_double
    u = np.ascontiguousarray(u, dtype=np.float64)
    return lib().orc_d1_bounded(_p(u), int(i), int(lo), int(hi), C.c_double(h))


def rk4_substep_bc(ps, bs, prm, stage, u_n, u_in, u_out, acc):
    kbuf = np.zeros_like(u_in)
    pr = _params(prm)
    lib().orc_rk4_substep_bc(_patches(ps), _boundaries(bs), len(ps), C.byref(pr), int(stage), _p(u_n), _p(u_in),
                             _p(u_out), _p(acc), _p(kbuf))


def rk4_step_bc(ps, bs, prm, u):
    """one RK4 step with per-face boundary modes, in place; returns the increment S per unit dt"""
    pr = _params(prm)
    n = u.size
    work = np.zeros(4 * n)
    lib().orc_rk4_step_bc(_patches(ps), _boundaries(bs), len(ps), C.byref(pr), _p(u), _p(work), C.c_int64(n))
    return work[2 * n:3 * n].copy()


# ---- subcycling: time interpolation of the parent levels and one Berger-Oliger step of a pair ----------
def time_weights(n, theta):
    """weights of the parent time levels at theta = (t - t_n)/dt: n = 2 (U^n, U^n+1), n = 3 (U^n-1, U^n, U^n+1)"""
    w = np.zeros(3)
    lib().orc_time_weights(int(n), C.c_double(theta), _p(w))
    return w


def lincomb(p, levels, w):
    """(w0 u0 + w1 u1) [+ w2 u2] on every storage cell of patch p"""
    out = np.zeros_like(levels[0])
    n = len(levels)
    u = list(levels) + [levels[0]] * (3 - n)
    lib().orc_lincomb(C.byref(_patches([p])[0]), n, _p(u[0]), _p(u[1]), _p(u[2]), _p(np.ascontiguousarray(w, dtype=np.float64)),
                      _p(out))
    return out


def subcycle_step(parent, child, org, prm, bnd, u_parent, u_parent_prev, have_prev, u_child):
    """one Berger-Oliger step of a parent / child pair, in place; bnd = (origin, faces) of the parent.
    u_parent_prev: buffer that receives the parent state the step started from (read as U^n-1 if have_prev)."""
    o = (C.c_int32 * 3)(*[int(v) for v in org])
    pr = _params(prm)
    lib().orc_subcycle_step(C.byref(_patches([parent])[0]), C.byref(_patches([child])[0]), o, C.byref(pr),
                            C.byref(_boundaries([bnd])[0]), _p(u_parent), _p(u_parent_prev), int(bool(have_prev)),
                            _p(u_child), C.c_int64(u_parent.size), C.c_int64(u_child.size))


def hierarchy_step(patches, orgs, prm, bnd0, states, prevs, nsteps):
    """one step of level 0 of a hierarchy of nested levels (level l + 1 inside level l at parent index orgs[l + 1]; orgs[0]
    unused), every finer level subcycled; in place on states / prevs (lists of arrays); nsteps: list of ints, updated"""
    n = len(patches)
    o = (C.c_int32 * (3 * n))(*[int(v) for org in orgs for v in org])
    pr = _params(prm)
    PP = C.POINTER(C.c_double)
    us = (PP * n)(*[_p(a) for a in states])
    ps_ = (PP * n)(*[_p(a) for a in prevs])
    nd = (C.c_int64 * n)(*[a.size for a in states])
    ns = (C.c_int64 * n)(*[int(v) for v in nsteps])
    lib().orc_hierarchy_step(_patches(patches), o, n, C.byref(pr), C.byref(_boundaries([bnd0])[0]), us, ps_, nd, ns)
    for i in range(n):
        nsteps[i] = int(ns[i])
