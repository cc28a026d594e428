"""Pins of the oracle's subcycling: time-interpolation weights (published
Lagrange values, exactness on polynomials in time), the linear combination of parent levels (numpy), and the
Berger-Oliger step of a parent / child pair -- flat space stays flat, spatially uniform data follow the ODE (the child
takes TWO RK4 half steps, the covered parent cells take the child's values), and a linearised TT wave is reproduced
on the child with the accuracy of the time-interpolated boundary data."""
import numpy as np
import pytest

import orc
from helpers import NF, NG, storage_coords
from paper_2607_08743_b200 import workloads as wl
from test_golden_weights import _golden

PRM = dict(wl.DEFAULT_PARAMS)
PER = [orc.BC_PERIODIC] * 6


def test_time_weights_published_values_and_exactness():
    g = _golden()
    for name, th in (("time2_q1", 0.25), ("time2_q2", 0.5), ("time2_q3", 0.75)):
        den, offs, num = g[name]
        assert np.array_equal(orc.time_weights(3, th), np.array(num) / den), name
    for th in (0.0, 0.25, 0.5, 0.75, 1.0):
        w2, w3 = orc.time_weights(2, th), orc.time_weights(3, th)
        assert w2[2] == 0.0 and abs(w2.sum() - 1) < 1e-15 and abs(w3.sum() - 1) < 1e-15
        lin = lambda t: 0.3 + 1.7 * t
        quad = lambda t: 0.3 + 1.7 * t - 0.9 * t * t
        assert abs(w2[0] * lin(0) + w2[1] * lin(1) - lin(th)) < 1e-15                      # first order: exact on lines
        assert abs(sum(w3[q] * quad(q - 1) for q in range(3)) - quad(th)) < 1e-15           # second order: on parabolas
    w2 = orc.time_weights(2, 0.5)
    assert abs(w2[0] * 0.3 + w2[1] * (0.3 + 1.7 - 0.9) - (0.3 + 0.85 - 0.225)) > 0.1        # and a line is not a parabola


def test_lincomb_is_the_weighted_sum_on_every_storage_cell():
    rng = np.random.default_rng(1)
    ps, total = wl.make_layout([(7, 6, 9)], [0.1], [0.02], [(0, 0, 0)])
    lev = [rng.normal(size=total) for _ in range(3)]
    w = np.array([-3 / 32, 15 / 16, 5 / 32])
    wk = wl.Workload("x", ps, PRM, lev[0])
    out3, out2 = orc.lincomb(ps[0], lev, w), orc.lincomb(ps[0], lev[:2], w[:2])
    for f in range(NF):
        a, b, c = (wk.field_view(x, 0, f)[:, :, :ps[0].nx + 2 * NG] for x in lev)
        assert np.array_equal(wk.field_view(out3, 0, f)[:, :, :ps[0].nx + 2 * NG], (w[0] * a + w[1] * b) + w[2] * c)
        assert np.array_equal(wk.field_view(out2, 0, f)[:, :, :ps[0].nx + 2 * NG], w[0] * a + w[1] * b)


def _pair(n, fn, h=None):
    """periodic parent of n^3 cells on [0,1)^3 (x_i = i h) and a child covering its central n/2 cells (n cells of h/2)"""
    h = h or 1.0 / n
    org = (n // 4,) * 3
    pp, tp = wl.make_layout([(n, n, n)], [h], [0.25 * h], [(0.0, 0.0, 0.0)])
    o = org[0] * h - 0.25 * h
    pc, tc = wl.make_layout([(n, n, n)], [0.5 * h], [0.125 * h], [(o, o, o)])
    P = wl.Workload("parent", pp, dict(PRM), np.zeros(tp))
    Cw = wl.Workload("child", pc, dict(PRM), np.zeros(tc))
    for w in (P, Cw):
        Z, Y, X = storage_coords(w.patches[0])
        vals = fn(X, Y, Z)
        for f in range(NF):
            w.field_view(w.state, 0, f)[...] = np.broadcast_to(vals[f], w.patches[0].shape)
    return P, Cw, org, ((0.0, 0.0, 0.0), PER)


def _flat(X):
    v = [np.zeros_like(X) for _ in range(NF)]
    for f in (wl.F_W, wl.F_G, wl.F_G + 3, wl.F_G + 5, wl.F_ALP):
        v[f] = np.ones_like(X)
    return v


def test_flat_space_stays_exactly_flat_on_both_levels():
    P, Cw, org, bnd = _pair(12, lambda X, Y, Z: _flat(X))
    up, uc, prev = P.state.copy(), Cw.state.copy(), np.zeros_like(P.state)
    orc.subcycle_step(P.patches[0], Cw.patches[0], org, PRM, bnd, up, prev, False, uc)
    orc.subcycle_step(P.patches[0], Cw.patches[0], org, PRM, bnd, up, prev, True, uc)
    assert np.array_equal(up, P.state) and np.array_equal(uc, Cw.state)


def test_data_linear_in_time_are_reproduced_exactly_on_both_levels():
    """Flat space with a uniform B^i and eta = 0: B^i stays constant and beta^i = beta0 + 3/4 B^i t is uniform in space and
    LINEAR in time; every other field is stationary. RK4 and both time interpolations are exact on such data, so parent
    and child must follow the closed form to round-off -- but only if the ghost data of every child substage is taken
    at the right time: a wrong theta puts a jump between the child's ghosts and its interior, and the shift gradient
    it creates shows up in every field."""
    B0, b0 = np.array([0.3, -0.2, 0.1]), np.array([0.05, 0.02, -0.04])
    def fn(X, Y, Z):
        v = _flat(X)
        for i in range(3):
            v[wl.F_B + i] = np.full_like(X, B0[i]); v[wl.F_BET + i] = np.full_like(X, b0[i])
        return v
    prm = dict(PRM, eta=0.0)
    P, Cw, org, bnd = _pair(12, fn, h=0.5)
    p, c = P.patches[0], Cw.patches[0]
    up, uc, prev = P.state.copy(), Cw.state.copy(), np.zeros_like(P.state)
    for step in (1, 2):                           # the second step interpolates with the parabola
        orc.subcycle_step(p, c, org, prm, bnd, up, prev, step > 1, uc)
        t = step * p.dt
        for w, u in ((P, up), (Cw, uc)):
            for f in range(NF):
                want = w.field_view(w.state, 0, f)[NG, NG, NG]
                if wl.F_BET <= f < wl.F_BET + 3:
                    want = b0[f - wl.F_BET] + 0.75 * B0[f - wl.F_BET] * t
                a = w.field_view(u, 0, f)[:, :, :w.patches[0].nx + 2 * NG]      # ghosts included
                assert np.max(np.abs(a - want)) < 4e-16, (step, wl.FIELD_NAMES[f], np.max(np.abs(a - want)))
    assert abs(P.active_view(up, 0, wl.F_BET)[0, 0, 0] - b0[0]) > 0.01


def test_uniform_data_follow_the_ode_and_the_parent_takes_the_child_values():
    """spatially uniform data with K-hat != 0: every cell follows the same ODE. The child's ghost data (straight line in
    time between the parent levels) differ from its interior RK stage values by O(dt^2); second differences turn that
    jump into an O(dt^2 / h^2) = O(1) error of the right-hand side next to the boundary, O(dt) in the state (the known
    order reduction of time-interpolated refinement boundaries). The child therefore agrees with the ODE solution to
    first order in dt, no better and no worse; the covered parent cells hold the restriction of the child, the others
    the parent's own step."""
    u0 = np.zeros(NF)
    for f in (wl.F_W, wl.F_G, wl.F_G + 3, wl.F_G + 5):
        u0[f] = 1.0
    u0[wl.F_ALP], u0[wl.F_KH], u0[wl.F_TH] = 0.8, 0.4, 0.05
    def fn(X, Y, Z):
        return [np.full_like(X, u0[f]) for f in range(NF)]
    z1, z2 = np.zeros((NF, 3)), np.zeros((NF, 6))
    F = lambda v: orc.rhs_point(PRM, v, z1, z2, np.zeros(NF), np.zeros(NF))
    def rk4(u, dt):
        k1 = F(u); k2 = F(u + 0.5 * dt * k1); k3 = F(u + 0.5 * dt * k2); k4 = F(u + dt * k3)
        return u + dt * (((k1 + 2 * k2) + 2 * k3 + k4) / 6.0)
    errs = []
    for h in (0.2, 0.1):
        P, Cw, org, bnd = _pair(12, fn, h=h)
        p, c = P.patches[0], Cw.patches[0]
        up, uc, prev = P.state.copy(), Cw.state.copy(), np.zeros_like(P.state)
        orc.subcycle_step(p, c, org, PRM, bnd, up, prev, False, uc)
        one = rk4(u0, p.dt)
        n = p.nx
        cov = slice(org[0], org[0] + n // 2)
        e = 0.0
        for f in range(NF):
            e = max(e, np.max(np.abs(Cw.active_view(uc, 0, f) - one[f])))
            pa = P.active_view(up, 0, f).copy()
            rest = pa[cov, cov, cov].copy()
            pa[cov, cov, cov] = one[f]
            assert np.allclose(pa, one[f], rtol=0, atol=3e-15)                 # the parent's own step outside the child
            ch = Cw.active_view(uc, 0, f)
            assert np.max(np.abs(rest - one[f])) <= np.max(np.abs(ch - one[f])) * 1.3 + 1e-15   # restriction of the child
        assert np.array_equal(prev, P.state)                                    # U^n handed back for the next step
        errs.append(e)
    assert 1e-6 < errs[1] < errs[0] < 5e-3 and 1.7 < errs[0] / errs[1] < 2.6, errs   # O(dt)


def _tt_pair(n, eps, t=0.0):
    def fn(X, Y, Z):
        v = _flat(X)
        s, c = np.sin(2 * np.pi * (X - t)), np.cos(2 * np.pi * (X - t))
        v[wl.F_G + 3] = 1 + eps * s; v[wl.F_G + 5] = 1 - eps * s
        v[wl.F_A + 3] = np.pi * eps * c; v[wl.F_A + 5] = -np.pi * eps * c
        return v
    return _pair(n, fn)


def _tt_child_error(n, nsteps):
    eps = 1e-6
    P, Cw, org, bnd = _tt_pair(n, eps)
    prm = dict(PRM, ko_sigma=0.0)
    up, uc, prev = P.state.copy(), Cw.state.copy(), np.zeros_like(P.state)
    for s in range(nsteps):
        orc.subcycle_step(P.patches[0], Cw.patches[0], org, prm, bnd, up, prev, s > 0, uc)
    t = nsteps * P.patches[0].dt
    c = Cw.patches[0]
    x = c.origin[0] + np.arange(c.nx) * c.dx
    exact = 1 + eps * np.sin(2 * np.pi * (x - t))
    return np.max(np.abs(Cw.active_view(uc, 0, wl.F_G + 3) - exact[None, None, :])) / eps


@pytest.mark.parametrize("nsteps", [1, 2])
def test_tt_wave_on_the_child_converges(nsteps):
    """nsteps = 1: first-order time interpolation; 2: the second step uses the parabola through three parent levels.
    The child follows the exact linearised wave; the error is that of the time-interpolated boundary data (second
    order under dt ~ h refinement), far below what a ghost zone frozen over a step (O(omega dt) ~ 1e-1 of the amplitude
    at n = 16) or a wrong substage time would give."""
    e1, e2 = _tt_child_error(16, nsteps), _tt_child_error(32, nsteps)
    assert e1 < 1e-3 and e2 < 2.5e-4, (e1, e2)          # relative to the wave amplitude
    assert 3.3 < e1 / e2 < 5.0, (e1, e2)
