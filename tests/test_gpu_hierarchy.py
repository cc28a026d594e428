"""-m gpu: the recursive Berger-Oliger step over nested levels on the CUDA path (sacra_hierarchy_step):
with two levels it equals sacra_subcycle_step bit for bit; with three levels two consecutive coarse steps (2, 4 and 8
steps of the levels; first- and second-order time interpolation at every level) follow the oracle's recursion within a
few times dt x the north_star tolerance, ghosts included."""
import numpy as np
import pytest
import torch

import orc
from gpu_util import dev, host
from helpers import NF, NG
from paper_2607_08743_b200 import sacra
from paper_2607_08743_b200 import workloads as wl
from test_oracle_hierarchy import _flat, hierarchy

pytestmark = pytest.mark.gpu
RTOL, FLOOR = 1e-11, 1e-14


def _data(seed=4, amp=5e-3):
    ph = np.random.default_rng(seed).uniform(0, 2 * np.pi, size=(NF, 3))
    def fn(X, Y, Z):
        v = _flat(X)
        for f in range(NF):
            v[f] = v[f] + amp * np.sin(2 * np.pi * X + ph[f, 0]) * np.sin(2 * np.pi * Y + ph[f, 1]) * np.sin(2 * np.pi * Z + ph[f, 2])
        return v
    return fn


def _gpu_levels(ws):
    st = [dev(w.state) for w in ws]
    pv = [torch.zeros_like(s) for s in st]
    wk = [torch.zeros(5 * s.numel(), dtype=torch.float64, device="cuda") for s in st]
    return st, pv, wk


def test_two_levels_equal_the_pair_step_bitwise():
    ws, orgs, bnd = hierarchy(16, 2, _data())
    ps = [w.patches[0] for w in ws]
    st, pv, wk = _gpu_levels(ws)
    counts = [0, 0]
    up, uc = dev(ws[0].state), dev(ws[1].state)
    prev = torch.zeros_like(up)
    wp, wc = torch.zeros(5 * up.numel(), dtype=torch.float64, device="cuda"), torch.zeros(3 * uc.numel(), dtype=torch.float64, device="cuda")
    for s in range(2):
        sacra.hierarchy_step(ps, orgs, ws[0].params, bnd, st, pv, wk, counts)
        sacra.subcycle_step(ps[0], ps[1], orgs[1], ws[0].params, bnd, up, prev, s > 0, uc, wp, wc)
        assert np.array_equal(host(st[0]), host(up)) and np.array_equal(host(st[1]), host(uc)), s
    assert counts == [2, 4] and np.array_equal(host(pv[0]), host(prev))


@pytest.mark.parametrize("org2", [None, 2, 6])
def test_three_levels_against_the_oracle_recursion(org2):
    """org2 = 2, 6: an off-centre grandchild, whose prolongation box reaches into level 1's ghost cells (they must be at
    the new time before level 2 advances; pinned on the oracle in test_oracle_hierarchy.py)"""
    ws, orgs, bnd = hierarchy(16, 3, _data(seed=6), org=None if org2 is None else [0, 4, org2])
    ps = [w.patches[0] for w in ws]
    prm = ws[0].params
    st, pv, wk = _gpu_levels(ws)
    gcount = [0, 0, 0]
    ref = [w.state.copy() for w in ws]
    rprev = [np.zeros_like(s) for s in ref]
    rcount = [0, 0, 0]
    worst = 0.0
    for step in range(2):
        before = [r.copy() for r in ref]
        orc.hierarchy_step(ps, orgs, prm, bnd, ref, rprev, rcount)
        sacra.hierarchy_step(ps, orgs, prm, bnd, st, pv, wk, gcount)
        assert gcount == rcount
        for l, w in enumerate(ws):
            q = w.patches[0]
            got = host(st[l])
            for f in range(NF):
                a = w.field_view(got, 0, f)[:, :, :q.nx + 2 * NG]
                b = w.field_view(ref[l], 0, f)[:, :, :q.nx + 2 * NG]
                rate = np.max(np.abs(b - w.field_view(before[l], 0, f)[:, :, :q.nx + 2 * NG])) / (q.dt * 2 ** l)
                tol = 16 * (step + 1) * (q.dt * 2 ** l) * RTOL * (rate + FLOOR) + 4 * np.spacing(np.max(np.abs(b)))
                assert np.max(np.abs(a - b)) <= tol, (step, l, wl.FIELD_NAMES[f], np.max(np.abs(a - b)), tol)
                worst = max(worst, np.max(np.abs(a - b)) / tol)
    print("\n[tolerance use] three levels (org2 = %s), 2 coarse steps: worst max|d| / tol = %.3f" % (org2, worst))
    assert np.max(np.abs(ws[2].active_view(ref[2], 0, wl.F_G + 3) - ws[2].active_view(ws[2].state, 0, wl.F_G + 3))) > 1e-6


@pytest.mark.parametrize("org2", [2, 3])
def test_off_centre_grandchild_linear_in_time_on_the_gpu(org2):
    """the oracle's pin of the same name, on the CUDA path: beta^i = b0 + 0.75 B0 t to round-off on all three levels,
    ghosts included (3e-3 at org 2 if level 1's ghosts are still at the old time when level 2 advances)"""
    B0, b0 = np.array([0.3, -0.2, 0.1]), np.array([0.05, 0.02, -0.04])
    def fn(X, Y, Z):
        v = _flat(X)
        for i in range(3):
            v[wl.F_B + i] = np.full_like(X, B0[i]); v[wl.F_BET + i] = np.full_like(X, b0[i])
        return v
    ws, orgs, bnd = hierarchy(16, 3, fn, h=0.5, org=[0, 4, org2])
    prm = dict(ws[0].params, eta=0.0)
    ps = [w.patches[0] for w in ws]
    st, pv, wk = _gpu_levels(ws)
    counts = [0, 0, 0]
    for step in (1, 2):
        sacra.hierarchy_step(ps, orgs, prm, bnd, st, pv, wk, counts)
        t = step * ps[0].dt
        for l, w in enumerate(ws):
            got = host(st[l])
            for i in range(3):
                a = w.field_view(got, 0, wl.F_BET + i)[:, :, :ps[l].nx + 2 * NG]
                want = b0[i] + 0.75 * B0[i] * t
                assert np.max(np.abs(a - want)) < 6e-16, (step, l, i, np.max(np.abs(a - want)))
