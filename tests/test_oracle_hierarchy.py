"""Pins of the oracle's recursive Berger-Oliger step over a hierarchy of nested levels (
PAPER.md:105-109; oracle/z4c_subcycle.hpp): with two levels it IS the pair step (bitwise); with three, flat space stays
flat, data linear in time are reproduced to round-off on every level (every substage of every level takes its ghost data
at the right time, through two generations of time interpolation), and a linearised TT wave arrives on the finest
level with the accuracy of the interpolated boundary data."""
import numpy as np
import pytest

import orc
from helpers import NF, NG, storage_coords
from paper_2607_08743_b200 import workloads as wl

PRM = dict(wl.DEFAULT_PARAMS)
PER = [orc.BC_PERIODIC] * 6


def _flat(X):
    v = [np.zeros_like(X) for _ in range(NF)]
    for f in (wl.F_W, wl.F_G, wl.F_G + 3, wl.F_G + 5, wl.F_ALP):
        v[f] = np.ones_like(X)
    return v


def hierarchy(n, nlevels, fn, h=None, org=None):
    """level 0: periodic n^3 cells on [0, n h)^3 (x_i = i h); level l + 1 covers n/2 cells of level l per axis, from
    parent cell org[l + 1] on (default n/4: the central ones)"""
    h = h or 1.0 / n
    ws, orgs, o = [], [(0, 0, 0)], 0.0
    for l in range(nlevels):
        hl = h / 2 ** l
        if l > 0:
            og = n // 4 if org is None else org[l]
            o = o + og * (2 * hl) - 0.5 * hl                # first child cell: a quarter parent spacing left of the parent cell
            orgs.append((og,) * 3)
        ps, tot = wl.make_layout([(n, n, n)], [hl], [0.25 * hl], [(o, o, o)])
        w = wl.Workload("level%d" % l, ps, dict(PRM), np.zeros(tot))
        Z, Y, X = storage_coords(ps[0])
        vals = fn(X, Y, Z)
        for f in range(NF):
            w.field_view(w.state, 0, f)[...] = np.broadcast_to(vals[f], ps[0].shape)
        ws.append(w)
    return ws, orgs, ((0.0, 0.0, 0.0), PER)


def _run(ws, orgs, bnd, prm, nsteps):
    states = [w.state.copy() for w in ws]
    prevs = [np.zeros_like(s) for s in states]
    counts = [0] * len(ws)
    for _ in range(nsteps):
        orc.hierarchy_step([w.patches[0] for w in ws], orgs, prm, bnd, states, prevs, counts)
    return states, prevs, counts


def test_two_levels_are_the_pair_step_bitwise():
    rng = np.random.default_rng(3)
    ph = rng.uniform(0, 2 * np.pi, size=(NF, 3))
    def fn(X, Y, Z):
        v = _flat(X)
        for f in range(NF):
            v[f] = v[f] + 5e-3 * np.sin(2 * np.pi * X + ph[f, 0]) * np.sin(2 * np.pi * Y + ph[f, 1]) * np.sin(2 * np.pi * Z + ph[f, 2])
        return v
    ws, orgs, bnd = hierarchy(16, 2, fn)
    states, prevs, counts = _run(ws, orgs, bnd, PRM, 2)
    up, uc, prev = ws[0].state.copy(), ws[1].state.copy(), np.zeros_like(ws[0].state)
    for s in range(2):
        orc.subcycle_step(ws[0].patches[0], ws[1].patches[0], orgs[1], PRM, bnd, up, prev, s > 0, uc)
    assert np.array_equal(states[0], up) and np.array_equal(states[1], uc) and np.array_equal(prevs[0], prev)
    assert counts == [2, 4]


def test_three_levels_flat_and_linear_in_time():
    ws, orgs, bnd = hierarchy(16, 3, lambda X, Y, Z: _flat(X))
    states, _, counts = _run(ws, orgs, bnd, PRM, 2)
    assert all(np.array_equal(s, w.state) for s, w in zip(states, ws)) and counts == [2, 4, 8]
    B0, b0 = np.array([0.3, -0.2, 0.1]), np.array([0.05, 0.02, -0.04])
    def fn(X, Y, Z):
        v = _flat(X)
        for i in range(3):
            v[wl.F_B + i] = np.full_like(X, B0[i]); v[wl.F_BET + i] = np.full_like(X, b0[i])
        return v
    prm = dict(PRM, eta=0.0)
    ws, orgs, bnd = hierarchy(16, 3, fn, h=0.5)
    for nsteps in (1, 2):
        states, _, _ = _run(ws, orgs, bnd, prm, nsteps)
        t = nsteps * ws[0].patches[0].dt
        for w, u in zip(ws, states):
            for f in range(NF):
                want = w.field_view(w.state, 0, f)[NG, NG, NG]
                if wl.F_BET <= f < wl.F_BET + 3:
                    want = b0[f - wl.F_BET] + 0.75 * B0[f - wl.F_BET] * t
                a = w.field_view(u, 0, f)[:, :, :w.patches[0].nx + 2 * NG]          # ghosts included
                assert np.max(np.abs(a - want)) < 6e-16, (nsteps, w.name, wl.FIELD_NAMES[f], np.max(np.abs(a - want)))


@pytest.mark.parametrize("org2", [2, 3, 5, 6])
def test_off_centre_grandchild_sees_its_parents_ghosts_at_the_new_time(org2):
    """The prolongation onto level 2 reads level-1 cells org - 4 .. org + n/2 + 3. With org < 4 (or org + n/2 + 3 > n - 1)
    that box reaches into level 1's GHOST cells, which the RK4 step of level 1 leaves at the old time. They have to be
    refreshed before level 2 advances: data linear in time are then still reproduced to round-off on every level,
    ghosts included (without the refresh: 3e-3 at org 2, 4e-4 at org 3)."""
    B0, b0 = np.array([0.3, -0.2, 0.1]), np.array([0.05, 0.02, -0.04])
    def fn(X, Y, Z):
        v = _flat(X)
        for i in range(3):
            v[wl.F_B + i] = np.full_like(X, B0[i]); v[wl.F_BET + i] = np.full_like(X, b0[i])
        return v
    prm = dict(PRM, eta=0.0)
    ws, orgs, bnd = hierarchy(16, 3, fn, h=0.5, org=[0, 4, org2])
    for nsteps in (1, 2):
        states, _, _ = _run(ws, orgs, bnd, prm, nsteps)
        t = nsteps * ws[0].patches[0].dt
        for w, u in zip(ws, states):
            for i in range(3):
                a = w.field_view(u, 0, wl.F_BET + i)[:, :, :w.patches[0].nx + 2 * NG]
                want = b0[i] + 0.75 * B0[i] * t
                assert np.max(np.abs(a - want)) < 6e-16, (nsteps, w.name, i, np.max(np.abs(a - want)))


def _tt_error(n, nsteps=1, eps=1e-6):
    def fn(X, Y, Z):
        v = _flat(X)
        s, c = np.sin(2 * np.pi * X), np.cos(2 * np.pi * X)
        v[wl.F_G + 3] = 1 + eps * s; v[wl.F_G + 5] = 1 - eps * s
        v[wl.F_A + 3] = np.pi * eps * c; v[wl.F_A + 5] = -np.pi * eps * c
        return v
    ws, orgs, bnd = hierarchy(n, 3, fn)
    states, _, _ = _run(ws, orgs, bnd, dict(PRM, ko_sigma=0.0), nsteps)
    t = nsteps * ws[0].patches[0].dt
    c = ws[2].patches[0]
    x = c.origin[0] + np.arange(c.nx) * c.dx
    exact = 1 + eps * np.sin(2 * np.pi * (x - t))
    return np.max(np.abs(ws[2].active_view(states[2], 0, wl.F_G + 3) - exact[None, None, :])) / eps


def test_tt_wave_on_the_finest_of_three_levels():
    e1, e2 = _tt_error(16), _tt_error(32)
    assert e1 < 1e-3 and e2 < 2.5e-4, (e1, e2)
    assert e1 / e2 > 3.0, (e1, e2)
