"""Pins for the oracle's constraint monitor (Eqs. 20-22).

The oracle evaluates H and M^i from the textbook definitions on the rebuilt physical metric. Pinned against what the
mathematics fixes, never against itself: flat space -> exactly 0; an exact vacuum solution (Kerr-Schild) -> 0 at 4th
order; closed forms for data that VIOLATE the constraints -- conformally flat time-symmetric data
(R = -8 psi^-5 Laplace(psi)), flat-metric K_ij with a known divergence, and conformally rescaled traceless K_ij
(D_j K^ij = psi^-10 d_j Abar^ij) -- which fix every overall factor, sign and power of W; Eq. 22 against numpy."""
import numpy as np
import pytest

import orc
from helpers import NF, NG, analytic_state, flat
from paper_2607_08743_b200 import workloads as wl
from test_oracle_rhs import kerr_schild

SYM = [[0, 1, 2], [1, 3, 4], [2, 4, 5]]
ORIGIN = (0.3, -0.2, 0.1)


def _constraints(fn, n, L=1.2, origin=ORIGIN):
    h = L / n
    w = analytic_state(n, h, tuple(o + 0.5 * h for o in origin), fn)
    con = orc.constraints(w.patches, w.state)
    p = w.patches[0]
    ax = [p.origin[a] + np.arange(n) * h for a in range(3)]
    Z, Y, X = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
    return [w.active_view(con, 0, c) for c in range(4)], (X, Y, Z), w, con


def _max_err(fn, exact, n):
    got, (X, Y, Z), _, _ = _constraints(fn, n)
    ex = exact(X, Y, Z)
    return np.array([np.max(np.abs(g - e)) for g, e in zip(got, ex)]), np.array([np.max(np.abs(e)) for e in ex])


def _fourth_order(fn, exact, which, n=16):
    e1, scale = _max_err(fn, exact, n)
    e2, _ = _max_err(fn, exact, 2 * n)
    for c in which:
        assert e2[c] < 2e-4 * max(scale[c], 1e-2), (c, e2, scale)
        if e1[c] > 1e-11:                      # a component the stencils represent exactly has no rate
            assert 11 < e1[c] / e2[c] < 22, (c, e1 / e2)
    return e2, scale


def test_flat_space_is_exactly_zero():
    got, _, _, _ = _constraints(lambda X, Y, Z: flat(X.shape), 8)
    assert all(np.all(g == 0.0) for g in got)


def test_kerr_schild_satisfies_the_constraints_at_fourth_order():
    """exact vacuum solution with K != 0, non-flat gt_ij, W != 1: every term of Eqs. 20-21 is exercised"""
    ks_origin = (1.6, 0.9, -0.5)
    errs = []
    for n in (12, 24):
        got, _, _, _ = _constraints(kerr_schild, n, L=1.5, origin=ks_origin)
        errs.append(np.array([np.max(np.abs(g)) for g in got]))
    assert np.all(errs[1] < 2e-5), errs[1]
    ratio = errs[0] / errs[1]
    assert np.all(ratio > 11) and np.all(ratio < 24), ratio


def test_kerr_schild_with_wrong_curvature_violates_them():
    def bad(X, Y, Z):
        v = kerr_schild(X, Y, Z)
        for s in range(6):
            v[wl.F_A + s] = 1.02 * v[wl.F_A + s]
        return v
    got, _, _, _ = _constraints(bad, 24, L=1.5, origin=(1.6, 0.9, -0.5))
    assert max(np.max(np.abs(g)) for g in got) > 1e-4


def _psi(X, Y, Z, a=0.3):
    r2 = X * X + Y * Y + Z * Z
    e = a * np.exp(-r2)
    return 1 + e, (4 * r2 - 6) * e, [-2 * X * e, -2 * Y * e, -2 * Z * e]     # psi, Laplace(psi), grad(psi)


def test_conformally_flat_time_symmetric_data_closed_form():
    """gamma_ij = psi^4 delta_ij, K_ij = 0  =>  H = R = -8 psi^-5 Laplace(psi), M^i = 0 (textbook conformal identity)"""
    def data(X, Y, Z):
        v = flat(X.shape)
        v[wl.F_W] = _psi(X, Y, Z)[0] ** -2
        return v
    def exact(X, Y, Z):
        psi, lap, _ = _psi(X, Y, Z)
        return [-8 * psi ** -5 * lap, 0 * X, 0 * X, 0 * X]
    e2, scale = _fourth_order(data, exact, which=[0])
    assert scale[0] > 1.0 and np.all(e2[1:] < 1e-12)


def test_flat_metric_momentum_constraint_closed_form():
    """gamma = delta: M^i = d_j K^ij - d_i K. K_ij = f delta_ij + (xy: g): M = (-2 f_x + g_y, -2 f_y + g_x, -2 f_z),
    H = K^2 - K_ij K^ij = 9 f^2 - (3 f^2 + 2 g^2)"""
    f = lambda X, Y, Z: 0.2 * np.sin(0.7 * X + 0.3) * np.cos(0.5 * Y) + 0.1 * Z * Z
    g = lambda X, Y, Z: 0.15 * np.cos(0.4 * X - 0.6 * Y + 0.2 * Z)
    def data(X, Y, Z):
        v = flat(X.shape)
        v[wl.F_KH] = 3 * f(X, Y, Z)              # K = trace
        v[wl.F_A + 1] = g(X, Y, Z)               # traceless part: At_xy (W = 1)
        return v
    def exact(X, Y, Z):
        fx = 0.2 * 0.7 * np.cos(0.7 * X + 0.3) * np.cos(0.5 * Y)
        fy = -0.2 * 0.5 * np.sin(0.7 * X + 0.3) * np.sin(0.5 * Y)
        fz = 0.2 * Z
        s = -0.15 * np.sin(0.4 * X - 0.6 * Y + 0.2 * Z)
        gx, gy = 0.4 * s, -0.6 * s
        ff, gg = f(X, Y, Z), g(X, Y, Z)
        return [9 * ff ** 2 - (3 * ff ** 2 + 2 * gg ** 2), -2 * fx + gy, -2 * fy + gx, -2 * fz]
    _fourth_order(data, exact, which=[1, 2, 3])
    e, _ = _max_err(data, exact, 16)
    assert e[0] < 1e-13                           # H is algebraic here (R = 0 exactly for the flat metric)


def test_theta_enters_through_K():
    """item 7: K = K-hat + 2 Theta. The same K split differently between K-hat and Theta gives the same constraints."""
    f = lambda X, Y, Z: 0.2 * np.sin(0.7 * X + 0.3) * np.cos(0.5 * Y)
    def a(X, Y, Z):
        v = flat(X.shape); v[wl.F_KH] = 3 * f(X, Y, Z); return v
    def b(X, Y, Z):
        v = flat(X.shape); v[wl.F_KH] = 1 * f(X, Y, Z); v[wl.F_TH] = f(X, Y, Z); return v
    ga, _, _, _ = _constraints(a, 12)
    gb, _, _, _ = _constraints(b, 12)
    for x, y in zip(ga, gb):
        assert np.max(np.abs(x - y)) < 1e-13 and np.max(np.abs(x)) > 1e-3 or np.max(np.abs(x)) < 1e-13


def test_conformally_rescaled_traceless_curvature_closed_form():
    """gamma_ij = psi^4 delta_ij, K_ij = psi^-2 Abar_ij, Abar traceless (xy, xz components), K = 0:
    M^i = D_j K^ij = psi^-10 d_j Abar^ij (the Bowen-York identity) and H = R - psi^-12 Abar_ij Abar^ij.
    Fixes the powers of W in Eq. 21: At_ij = W^2 K_ij = psi^-6 Abar_ij."""
    g = lambda X, Y, Z: 0.15 * np.cos(0.4 * X - 0.6 * Y + 0.2 * Z)
    q = lambda X, Y, Z: 0.1 * np.sin(0.3 * X + 0.5 * Z)
    def data(X, Y, Z):
        v = flat(X.shape)
        psi = _psi(X, Y, Z)[0]
        v[wl.F_W] = psi ** -2
        v[wl.F_A + 1] = psi ** -6 * g(X, Y, Z)
        v[wl.F_A + 2] = psi ** -6 * q(X, Y, Z)
        return v
    def exact(X, Y, Z):
        psi, lap, _ = _psi(X, Y, Z)
        s = -0.15 * np.sin(0.4 * X - 0.6 * Y + 0.2 * Z)
        gx, gy = 0.4 * s, -0.6 * s
        c = 0.1 * np.cos(0.3 * X + 0.5 * Z)
        qx, qz = 0.3 * c, 0.5 * c
        gg, qq = g(X, Y, Z), q(X, Y, Z)
        H = -8 * psi ** -5 * lap - psi ** -12 * 2 * (gg ** 2 + qq ** 2)
        return [H, psi ** -10 * (gy + qz), psi ** -10 * gx, psi ** -10 * qx]
    _fourth_order(data, exact, which=[0, 1, 2, 3])


def test_norms_are_eq22():
    """Eq. 22 on two patches of different cell size against numpy"""
    ps, total = wl.make_layout([(7, 6, 9), (6, 8, 6)], [0.1, 0.05], [0.01, 0.01], [(0, 0, 0)] * 2)
    w = wl.Workload("norm", ps, dict(wl.DEFAULT_PARAMS), np.zeros(total))
    rng = np.random.default_rng(3)
    con = rng.normal(size=total)
    want = np.zeros(4)
    vol = sum(p.nx * p.ny * p.nz * p.dx ** 3 for p in ps)
    for c in range(4):
        want[c] = np.sqrt(sum(np.sum(w.active_view(con, ip, c) ** 2) * p.dx ** 3 for ip, p in enumerate(ps)) / vol)
    assert np.allclose(orc.constraint_norms(ps, con), want, rtol=1e-13)
