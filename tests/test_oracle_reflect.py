"""Pins for the mirror ghost fill: numpy's symmetric padding for the index map, and
the defining property for the parity table -- data that is mirror-symmetric on a periodic domain of twice the size
must give, on the half domain with mirror faces, exactly the right-hand side of the full periodic problem."""
import numpy as np
import pytest

import orc
from helpers import NF, NG
from paper_2607_08743_b200 import workloads as wl

# parity of every field under z -> -z: scalars and xx, xy, yy, zz even; xz, yz and z-components odd
PZ = np.ones(NF)
for f in (wl.F_G + 2, wl.F_G + 4, wl.F_A + 2, wl.F_A + 4, wl.F_GAM + 2, wl.F_BET + 2, wl.F_B + 2):
    PZ[f] = -1.0


def test_mirror_fill_is_numpy_symmetric_padding_times_parity():
    ps, total = wl.make_layout([(7, 8, 6)], [0.1], [0.01], [(0, 0, 0)])
    w = wl.Workload("r", ps, dict(wl.DEFAULT_PARAMS), np.zeros(total))
    rng = np.random.default_rng(1)
    for f in range(NF):
        w.active_view(w.state, 0, f)[...] = rng.normal(size=(6, 8, 7))
    u = orc.fill_ghosts_bc(ps, (0, 0, 1), w.state.copy())       # periodic in x, y; mirror in z
    p = ps[0]
    for f in range(NF):
        a = w.active_view(w.state, 0, f)
        want = np.pad(a, ((0, 0), (NG, NG), (NG, NG)), mode="wrap")
        want = np.pad(want, ((NG, NG), (0, 0), (0, 0)), mode="symmetric")
        want[:NG] *= PZ[f]
        want[-NG:] *= PZ[f]
        assert np.array_equal(w.field_view(u, 0, f)[:, :, :p.nx + 2 * NG], want), wl.FIELD_NAMES[f]


def _mirror_symmetric_full(n, nz2, seed):
    """generic smooth data on n x n x nz2 (periodic) that is symmetric under z -> -z about the middle plane"""
    ps, total = wl.make_layout([(n, n, nz2)], [0.1], [0.025], [(0, 0, 0)])
    w = wl.Workload("full", ps, dict(wl.DEFAULT_PARAMS), np.zeros(total))
    rng = np.random.default_rng(seed)
    half = nz2 // 2
    for f in range(NF):
        top = 0.03 * rng.normal(size=(half, n, n))
        if f in (wl.F_W, wl.F_G, wl.F_G + 3, wl.F_G + 5, wl.F_ALP):
            top = top + 1.0
        v = w.active_view(w.state, 0, f)
        v[half:] = top                             # upper half z >= 0
        v[:half] = PZ[f] * top[::-1]               # lower half: the mirror image with the field's parity
    return w


def test_half_domain_with_mirror_faces_equals_full_periodic_problem():
    n, nz2 = 8, 12
    full = _mirror_symmetric_full(n, nz2, 5)
    uf = full.state.copy()
    orc.fill_ghosts(full.patches, uf)
    rf = orc.z4c_rhs(full.patches, full.params, uf)
    half = nz2 // 2
    ps, total = wl.make_layout([(n, n, half)], [0.1], [0.025], [(0, 0, 0)])
    h = wl.Workload("half", ps, dict(full.params), np.zeros(total))
    for f in range(NF):
        h.active_view(h.state, 0, f)[...] = full.active_view(full.state, 0, f)[half:]
    uh = orc.fill_ghosts_bc(ps, (0, 0, 1), h.state.copy())
    rh = orc.z4c_rhs(ps, h.params, uh)
    for f in range(NF):
        a, b = h.active_view(rh, 0, f), full.active_view(rf, 0, f)[half:]
        assert np.array_equal(a, b), wl.FIELD_NAMES[f]
        assert np.max(np.abs(a)) > 0
    # a wrong parity anywhere breaks it
    bad = h.state.copy()
    orc.fill_ghosts_bc(ps, (0, 0, 1), bad)
    h.field_view(bad, 0, wl.F_BET + 2)[:NG] *= -1.0
    rb = orc.z4c_rhs(ps, h.params, bad)
    assert not np.array_equal(h.active_view(rb, 0, wl.F_BET + 2), full.active_view(rf, 0, wl.F_BET + 2)[half:])
