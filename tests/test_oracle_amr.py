"""Pins for the inter-level operators: published Lagrange weights through unit
impulses, exactness on polynomials (degree 3 for the 4-point restriction, degree 5 for the 6-point prolongation, in
all three directions at once), convergence orders, and the geometry of the 2:1 cell-centred staggered grids."""
import os

import numpy as np
import pytest

import orc
from helpers import NF, NG, storage_coords
from paper_2607_08743_b200 import workloads as wl
from test_golden_weights import _golden


def _pair(nc=8, npar=16, org=(4, 5, 3), H=0.2):
    """a parent patch (npar^3, spacing H) and a child (nc^3, spacing H/2) whose cells 0,1 sit in parent cell org"""
    pp, tp = wl.make_layout([(npar, npar, npar)], [H], [0.01], [(0.0, 0.0, 0.0)])
    child_origin = tuple(org[a] * H - 0.25 * H for a in range(3))   # centre of child cell 0 = parent centre - H/4
    pc, tc = wl.make_layout([(nc, nc, nc)], [H / 2], [0.005], [child_origin])
    return pp[0], tp, pc[0], tc


def _fill(p, total, fn):
    u = np.zeros(total)
    Z, Y, X = storage_coords(p)
    w = wl.Workload("x", [p], dict(wl.DEFAULT_PARAMS), u)
    for f in range(NF):
        w.field_view(u, 0, f)[...] = fn(X, Y, Z, f)
    return w, u


def test_geometry_child_cells_straddle_the_parent_centre():
    pp, tp, pc, tc = _pair()
    xp = pp.origin[0] + np.arange(pp.nx) * pp.dx
    xc = pc.origin[0] + np.arange(pc.nx) * pc.dx
    assert np.allclose(0.5 * (xc[0] + xc[1]), xp[4]) and np.allclose(0.5 * (xc[2] + xc[3]), xp[5])


def test_restriction_weights_are_the_published_ones():
    g = _golden()
    den, offs, num = g["restrict4"]
    pp, tp, pc, tc = _pair()
    wc = wl.Workload("c", [pc], dict(wl.DEFAULT_PARAMS), np.zeros(tc))
    for axis in range(3):
        for k, off in enumerate(offs):
            uc = np.zeros(tc)
            idx = [2 + NG, 2 + NG, 2 + NG]          # storage index of child cell 2 (= 2m, m = 1) on the other axes
            idx[2 - axis] = 2 + off + NG             # field_view is (z, y, x)
            wc.field_view(uc, 0, 0)[tuple(idx)] = 1.0
            up = orc.restrict(pp, pc, (4, 5, 3), np.zeros(tp), uc)
            wp = wl.Workload("p", [pp], dict(wl.DEFAULT_PARAMS), up)
            # parent cell org + 1 on every axis; on the two other axes the impulse sits at offset 0 (weight 9/16)
            got = wp.active_view(up, 0, 0)[3 + 1, 5 + 1, 4 + 1]
            assert got == num[k] / den * (9 / 16) ** 2, (axis, off, got)


def test_prolongation_weights_are_the_published_ones():
    g = _golden()
    den, offs, num = g["prolong6"]
    pp, tp, pc, tc = _pair()
    wp = wl.Workload("p", [pp], dict(wl.DEFAULT_PARAMS), np.zeros(tp))
    wc = wl.Workload("c", [pc], dict(wl.DEFAULT_PARAMS), np.zeros(tc))
    # child ghost cell i = -2 (even, m = -1) along x, cells 2 (even, m = 1) along y and z would be active: use a face
    # ghost: i = -2, j = 2, k = 2 -> parent nodes org + m + off; weights multiply across the axes
    for k, off in enumerate(offs):
        up = np.zeros(tp)
        wp.active_view(up, 0, 0)[3 + 1, 5 + 1, 4 - 1 + off] = 1.0   # impulse at x-node `off`, at offset 0 in y and z
        uc = orc.prolong_ghosts(pp, pc, (4, 5, 3), up, np.zeros(tc))
        got = wc.field_view(uc, 0, 0)[2 + NG, 2 + NG, -2 + NG]
        assert got == num[k] / den * (num[offs.index(0)] / den) ** 2, (off, got)
    # an odd cell uses the mirror image: i = -1 (odd, m = -1): nodes -2..3 with the reversed weights
    for k, off in enumerate(offs):
        up = np.zeros(tp)
        wp.active_view(up, 0, 0)[3 + 1, 5 + 1, 4 - 1 - off] = 1.0
        uc = orc.prolong_ghosts(pp, pc, (4, 5, 3), up, np.zeros(tc))
        got = wc.field_view(uc, 0, 0)[2 + NG, 2 + NG, -1 + NG]
        assert got == num[k] / den * (num[offs.index(0)] / den) ** 2, (off, got)


def _poly(deg):
    return lambda X, Y, Z, f: (1 + 0.1 * f) * (0.3 + X) ** deg + (0.7 - Y) ** deg * (1.1 + Z) + (X * Y * Z) ** (deg // 3)


def test_restriction_is_exact_for_cubics_and_fourth_order():
    pp, tp, pc, tc = _pair()
    wcw, uc = _fill(pc, tc, _poly(3))
    wpw, exact = _fill(pp, tp, _poly(3))
    up = orc.restrict(pp, pc, (4, 5, 3), np.zeros(tp), uc)
    for f in (0, 7, 24):
        a = wpw.active_view(up, 0, f)[3:3 + 4, 5:5 + 4, 4:4 + 4]
        b = wpw.active_view(exact, 0, f)[3:3 + 4, 5:5 + 4, 4:4 + 4]
        assert np.max(np.abs(a - b)) < 1e-13 * np.max(np.abs(b))
        assert np.all(wpw.active_view(up, 0, f)[:3] == 0)        # outside the covered cells: untouched
    errs = []
    smooth = lambda X, Y, Z, f: np.sin(1.3 * X + 0.2) * np.cos(0.9 * Y) * np.sin(0.7 * Z + 0.5)
    for H in (0.2, 0.1):
        pp, tp, pc, tc = _pair(H=H)
        _, uc = _fill(pc, tc, smooth)
        wpw, exact = _fill(pp, tp, smooth)
        up = orc.restrict(pp, pc, (4, 5, 3), np.zeros(tp), uc)
        errs.append(np.max(np.abs(wpw.active_view(up, 0, 0)[3:7, 5:9, 4:8] - wpw.active_view(exact, 0, 0)[3:7, 5:9, 4:8])))
    assert 11 < errs[0] / errs[1] < 22, errs


def test_prolongation_is_exact_for_quintics_and_sixth_order():
    pp, tp, pc, tc = _pair()
    _, up = _fill(pp, tp, _poly(5))
    wcw, exact = _fill(pc, tc, _poly(5))
    uc = orc.prolong_ghosts(pp, pc, (4, 5, 3), up, np.full(tc, 7.0))
    n = pc.nx
    for f in (0, 7, 24):
        got, ex = wcw.field_view(uc, 0, f)[:, :, :n + 2 * NG], wcw.field_view(exact, 0, f)[:, :, :n + 2 * NG]
        ghost = np.ones(got.shape, dtype=bool)
        ghost[NG:NG + n, NG:NG + n, NG:NG + n] = False
        assert np.max(np.abs(got[ghost] - ex[ghost])) < 2e-13 * np.max(np.abs(ex))
        assert np.all(got[~ghost] == 7.0)                        # active cells untouched
    errs = []
    smooth = lambda X, Y, Z, f: np.sin(1.3 * X + 0.2) * np.cos(0.9 * Y) * np.sin(0.7 * Z + 0.5)
    for H in (0.2, 0.1):
        pp, tp, pc, tc = _pair(H=H)
        _, up = _fill(pp, tp, smooth)
        wcw, exact = _fill(pc, tc, smooth)
        uc = orc.prolong_ghosts(pp, pc, (4, 5, 3), up, np.zeros(tc))
        got, ex = wcw.field_view(uc, 0, 0)[:NG, :, :n + 2 * NG], wcw.field_view(exact, 0, 0)[:NG, :, :n + 2 * NG]
        errs.append(np.max(np.abs(got - ex)))
    assert 45 < errs[0] / errs[1] < 90, errs                    # 2^6 = 64
