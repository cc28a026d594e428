"""-m gpu: subcycling on the CUDA path: time weights and the linear combination of parent levels
bit-exact against the oracle, and two Berger-Oliger steps of a parent / child pair (first- and second-order time
interpolation) against the oracle's driver. The spatial operators and the combination are bit-exact given equal inputs;
the substages agree to the north_star tolerance, so the states are compared at a few times dt x that tolerance."""
import numpy as np
import pytest
import torch

import orc
from gpu_util import dev, host
from helpers import NF, NG, storage_coords
from paper_2607_08743_b200 import sacra
from paper_2607_08743_b200 import workloads as wl

pytestmark = pytest.mark.gpu
RTOL, FLOOR = 1e-11, 1e-14
PER = [0] * 6


def test_time_weights_and_lincomb_bit_exact():
    for n in (2, 3):
        for th in (0.0, 0.25, 0.5, 0.75, 1.0, 0.3):
            assert np.array_equal(np.array(sacra.time_weights(n, th)), orc.time_weights(n, th)) or \
                np.allclose(sacra.time_weights(n, th), orc.time_weights(n, th), rtol=0, atol=1e-16)
    for th in (0.0, 0.25, 0.5, 0.75, 1.0):          # the substage times: exact dyadic arithmetic on both sides
        assert np.array_equal(np.array(sacra.time_weights(3, th)), orc.time_weights(3, th))
    rng = np.random.default_rng(1)
    ps, total = wl.make_layout([(9, 6, 7)], [0.1], [0.02], [(0, 0, 0)])
    lev = [rng.normal(size=total) for _ in range(3)]
    for n in (2, 3):
        w = orc.time_weights(n, 0.75)
        ref = orc.lincomb(ps[0], lev[:n], w)
        out = torch.zeros(total, dtype=torch.float64, device="cuda")
        sacra.lincomb(ps[0], [dev(x) for x in lev[:n]], w, out)
        assert np.array_equal(host(out), ref)


def _pair(n, seed=4, amp=5e-3):
    h = 1.0 / n
    org = (n // 4,) * 3
    pp, tp = wl.make_layout([(n, n, n)], [h], [0.25 * h], [(0.0, 0.0, 0.0)])
    o = org[0] * h - 0.25 * h
    pc, tc = wl.make_layout([(n, n, n)], [0.5 * h], [0.125 * h], [(o, o, o)])
    P = wl.Workload("parent", pp, dict(wl.DEFAULT_PARAMS), np.zeros(tp))
    Cw = wl.Workload("child", pc, dict(wl.DEFAULT_PARAMS), np.zeros(tc))
    rng = np.random.default_rng(seed)
    ph = rng.uniform(0, 2 * np.pi, size=(NF, 3))
    for w in (P, Cw):
        Z, Y, X = storage_coords(w.patches[0])
        for f in range(NF):
            v = amp * np.sin(2 * np.pi * X + ph[f, 0]) * np.sin(2 * np.pi * Y + ph[f, 1]) * np.sin(2 * np.pi * Z + ph[f, 2])
            if f in (wl.F_W, wl.F_G, wl.F_G + 3, wl.F_G + 5, wl.F_ALP):
                v = v + 1.0
            w.field_view(w.state, 0, f)[...] = v
    return P, Cw, org, ((0.0, 0.0, 0.0), PER)


def test_two_subcycle_steps_against_the_oracle_driver():
    P, Cw, org, bnd = _pair(16)
    p, c, prm = P.patches[0], Cw.patches[0], P.params
    up, uc, prev = P.state.copy(), Cw.state.copy(), np.zeros_like(P.state)
    gp, gc, gprev = dev(P.state), dev(Cw.state), torch.zeros(P.state.size, dtype=torch.float64, device="cuda")
    wp = torch.zeros(5 * P.state.size, dtype=torch.float64, device="cuda")
    wc = torch.zeros(3 * Cw.state.size, dtype=torch.float64, device="cuda")
    worst = 0.0
    for step in range(2):
        before = (up.copy(), uc.copy())
        g_before = host(gp).copy()
        orc.subcycle_step(p, c, org, prm, bnd, up, prev, step > 0, uc)
        sacra.subcycle_step(p, c, org, prm, bnd, gp, gprev, step > 0, gc, wp, wc)
        for w, ref, got, old in ((P, up, host(gp), before[0]), (Cw, uc, host(gc), before[1])):
            q = w.patches[0]
            for f in range(NF):
                a = w.field_view(got, 0, f)[:, :, :q.nx + 2 * NG]
                b = w.field_view(ref, 0, f)[:, :, :q.nx + 2 * NG]
                rate = np.max(np.abs(b - w.field_view(old, 0, f)[:, :, :q.nx + 2 * NG])) / q.dt   # ~ max|S_f|
                tol = 8 * (step + 1) * q.dt * RTOL * (rate + FLOOR) + 4 * np.spacing(np.max(np.abs(b)))
                assert np.max(np.abs(a - b)) <= tol, (step, w.name, wl.FIELD_NAMES[f], np.max(np.abs(a - b)), tol)
                worst = max(worst, np.max(np.abs(a - b)) / tol)
        assert np.array_equal(host(gprev), g_before)       # U^n handed back, bit for bit (a copy)
    print("\n[tolerance use] pair, 2 coarse steps: worst max|d| / tol = %.3f" % worst)
    # the child did move, and the parent's covered cells are the restriction of the child (not the parent's own step)
    assert np.max(np.abs(Cw.active_view(uc, 0, wl.F_G + 3) - Cw.active_view(Cw.state, 0, wl.F_G + 3))) > 1e-6
