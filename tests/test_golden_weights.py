"""Oracle stencils against published finite-difference weights (tests/golden/stencil_weights.txt): the response of
each operator to a unit impulse IS its weight row. Catches a wrong coefficient, sign, offset or normalisation."""
import os

import numpy as np
import pytest

import orc
from paper_2607_08743_b200 import workloads as wl

HERE = os.path.dirname(os.path.abspath(__file__))


def _golden():
    rows = {}
    for line in open(os.path.join(HERE, "golden", "stencil_weights.txt")):
        if line.startswith("#") or not line.strip():
            continue
        left, right = line.split(":")
        name, den, *offs = left.split()
        rows[name] = (int(den), [int(o) for o in offs], [int(v) for v in right.split()])
    return rows


def _impulse_response(axis, beta_sign, h=0.5, sigma=0.8, n=12):
    """derivative bundle of field W at every point of a line through a unit impulse at the centre"""
    ps, total = wl.make_layout([(n, n, n)], [h], [0.1], [(0, 0, 0)])
    w = wl.Workload("impulse", ps, dict(wl.DEFAULT_PARAMS), np.zeros(total))
    c = n // 2
    w.active_view(w.state, 0, wl.F_W)[c, c, c] = 1.0
    w.active_view(w.state, 0, wl.F_BET + axis)[...] = beta_sign * 1.0   # unit shift along the axis
    u = w.state.copy()
    orc.fill_ghosts(ps, u)
    out = {}
    for k in range(-3, 4):        # the stencil centred at c - k sees the impulse at offset +k
        idx = [c, c, c]
        idx[axis] = c - k
        out[k] = orc.derivs_field(ps[0], u, wl.F_W, *idx, sigma)
    return out, h, sigma


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_oracle_stencils_reproduce_published_weights(axis):
    g = _golden()
    resp, h, sigma = _impulse_response(axis, +1.0)
    resp_neg, _, _ = _impulse_response(axis, -1.0)
    diag = [0, 3, 5][axis]            # xx, yy, zz in the packed order xx xy xz yy yz zz
    def row(name, pick, scale, r=resp, centre_axes=1):
        den, offs, num = g[name]
        for k in range(-3, 4):
            want = (num[offs.index(k)] / den) * scale if k in offs else 0.0
            if k == 0:
                want *= centre_axes
            got = pick(r[k])
            assert got == pytest.approx(want, rel=1e-14, abs=1e-15), (name, axis, k, got, want)
    row("d1", lambda d: d[0][axis], 1.0 / h)
    row("d2", lambda d: d[1][diag], 1.0 / h ** 2)
    row("up_pos", lambda d: d[2], 1.0 / h)                    # advection = beta * D^up, beta = +1
    row("up_neg", lambda d: d[2], -1.0 / h, r=resp_neg)       # beta = -1
    row("ko", lambda d: d[3], sigma / h, centre_axes=3)   # Q sums the three axes; all see the centre
