"""Pins of the oracle's physical boundaries: the Sommerfeld shell of Eq. 13 and
the per-face ghost fill. Against what the mathematics fixes: published one-sided weights, polynomial exactness, an
exact outgoing solution Q = f(t - r)/r (its analytic time derivative at 4th order), the static 1/r tail (RHS -> 0),
flat space (exactly 0), and the mirror property (a half domain with a MIRROR face gives, bit for bit, the shell
values of the full domain with symmetric data)."""
import os

import numpy as np
import pytest

import orc
from helpers import NF, NG, analytic_state, flat
from paper_2607_08743_b200 import workloads as wl
from test_golden_weights import _golden

SOM, MIR, PER, NONE = orc.BC_SOMMERFELD, orc.BC_MIRROR, orc.BC_PERIODIC, orc.BC_NONE
ALL_SOM = [SOM] * 6


def test_bounded_derivative_reproduces_published_one_sided_weights():
    g = _golden()
    h, n = 0.25, 9
    for name, i in (("onesided_0", 0), ("onesided_1", 1)):
        den, offs, num = g[name]
        for k in range(n):
            u = np.zeros(n); u[k] = 1.0
            want = num[offs.index(k - i)] / den / h if (k - i) in offs else 0.0
            assert orc.d1_bounded(u, i, 0, n - 1, h) == pytest.approx(want, rel=1e-14, abs=1e-15), (name, k)
            # upper side: mirror image, opposite sign
            um = u[::-1].copy()
            assert orc.d1_bounded(um, n - 1 - i, 0, n - 1, h) == pytest.approx(-want, rel=1e-14, abs=1e-15), (name, k)
    den, offs, num = g["d1"]
    for k in range(n):                        # interior points: the centred stencil of item 3
        u = np.zeros(n); u[k] = 1.0
        want = num[offs.index(k - 4)] / den / h if (k - 4) in offs else 0.0
        assert orc.d1_bounded(u, 4, 0, n - 1, h) == pytest.approx(want, rel=1e-14, abs=1e-15)


def test_bounded_derivative_is_exact_on_quartics_everywhere():
    rng = np.random.default_rng(2)
    n, h = 11, 0.3
    x = np.arange(n) * h
    c = rng.normal(size=5)
    u = sum(c[q] * x ** q for q in range(5))
    du = sum(q * c[q] * x ** (q - 1) for q in range(1, 5))
    for i in range(n):
        assert orc.d1_bounded(u, i, 0, n - 1, h) == pytest.approx(du[i], rel=1e-11, abs=1e-11), i
    # valid ghosts on the left (lo = -3 relative to an array that starts 3 cells earlier): centred at the first cells
    assert orc.d1_bounded(u, 3, 0, n - 1, h) == pytest.approx(du[3], rel=1e-11)


def _fill(fn, n, origin, L, faces=ALL_SOM, shape=None):
    h = L / n
    w = analytic_state(n, h, origin, fn)
    return w, [(origin, faces)]


def _pulse_fields(t):
    """all 25 fields: flat value + outgoing spherical pulse a_f f(t - r + r0_f) / r, and its time derivative"""
    rng = np.random.default_rng(5)
    amp, r0, wd = rng.uniform(0.5, 1.5, NF) * 1e-2, rng.uniform(5.0, 6.0, NF), rng.uniform(1.5, 2.5, NF)
    def val(X, Y, Z, deriv):
        r = np.sqrt(X * X + Y * Y + Z * Z)
        v = flat(X.shape)
        for f in range(NF):
            s = (t - r + r0[f]) / wd[f]
            g = np.exp(-s * s)
            v[f] = (v[f] if not deriv else 0.0) + amp[f] * (g if not deriv else -2 * s / wd[f] * g) / r
        return v
    return val


def _shell_mask(n, faces):
    i = np.arange(n)
    lo = [faces[2 * a] == SOM for a in range(3)]
    hi = [faces[2 * a + 1] == SOM for a in range(3)]
    m1 = lambda a: (lo[a] & (i < NG)) | (hi[a] & (i >= n - NG))
    return m1(2)[:, None, None] | m1(1)[None, :, None] | m1(0)[None, None, :]


def _pulse_error(n, faces=ALL_SOM):
    origin, L = (3.0, 2.5, 2.0), 3.0
    h = L / n
    o = tuple(c + 0.5 * h for c in origin)
    val = _pulse_fields(0.0)
    w, bs = _fill(lambda X, Y, Z: val(X, Y, Z, False), n, o, L, faces)
    rhs = orc.sommerfeld_rhs(w.patches, bs, w.state, np.full(w.state.size, 7.0))
    ax = [o[a] + np.arange(n) * h for a in range(3)]
    Z, Y, X = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
    exact = val(X, Y, Z, True)
    mask = _shell_mask(n, faces)
    err = np.zeros(NF)
    for f in range(NF):
        got = w.active_view(rhs, 0, f)
        assert np.all(got[~mask] == 7.0)                    # cells outside the shell are not touched
        err[f] = np.max(np.abs(got[mask] - exact[f][mask]))
    scale = np.array([np.max(np.abs(exact[f])) for f in range(NF)])
    return err, scale


def test_outgoing_pulse_is_reproduced_at_fourth_order():
    """Q = f(t - r)/r solves Eq. 13 exactly: the shell RHS must converge to the analytic d_t Q at 4th order, on faces,
    edges and corners, for all 25 fields (those with flat value 1 included)"""
    e1, s = _pulse_error(12)
    e2, _ = _pulse_error(24)
    assert np.all(e2 < 2e-3 * s), (e2, s)
    r = e1 / e2
    assert np.all((r > 10) & (r < 26)), r


def test_static_one_over_r_tail_has_zero_rhs():
    def tail(X, Y, Z):
        r = np.sqrt(X * X + Y * Y + Z * Z)
        v = flat(X.shape)
        for f in range(NF):
            v[f] = v[f] + 0.01 * (f + 1) / r
        return v
    errs = []
    for n in (12, 24):
        h = 3.0 / n
        o = (3.0 + 0.5 * h, 2.5 + 0.5 * h, 2.0 + 0.5 * h)
        w, bs = _fill(tail, n, o, 3.0)
        rhs = orc.sommerfeld_rhs(w.patches, bs, w.state)
        errs.append(np.array([np.max(np.abs(w.active_view(rhs, 0, f))) for f in range(NF)]))
    assert np.all(errs[1] < 1e-6)
    assert np.all(errs[0] / errs[1] > 10)


def test_flat_space_shell_is_exactly_zero():
    w, bs = _fill(lambda X, Y, Z: flat(X.shape), 10, (1.0, 2.0, 3.0), 2.0)
    rhs = orc.sommerfeld_rhs(w.patches, bs, w.state, np.full(w.state.size, 7.0))
    mask = _shell_mask(10, ALL_SOM)
    for f in range(NF):
        assert np.all(w.active_view(rhs, 0, f)[mask] == 0.0)


def test_fill_ghosts_faces_reduces_to_the_per_axis_fill_and_leaves_other_faces_alone():
    rng = np.random.default_rng(8)
    ps, total = wl.make_layout([(9, 7, 8)], [0.1], [0.02], [(0, 0, 0)])
    base = rng.normal(size=total)
    for mode in ((0, 0, 0), (1, 1, 1), (0, 1, 0), (1, 0, 1)):
        a = orc.fill_ghosts_bc(ps, mode, base.copy())
        faces = [m for m in mode for _ in (0, 1)]
        b = orc.fill_ghosts_faces(ps, [((0, 0, 0), faces)], base.copy())
        assert np.array_equal(a, b), mode
    # z- mirror, everything else Sommerfeld / none: only cells that are ghosts in z- alone change
    faces = [SOM, SOM, NONE, SOM, MIR, SOM]
    out = orc.fill_ghosts_faces(ps, [((0, 0, 0), faces)], base.copy())
    p = ps[0]
    w = wl.Workload("x", ps, dict(wl.DEFAULT_PARAMS), base)
    for f in range(NF):
        o, b = w.field_view(out, 0, f), w.field_view(base, 0, f)
        par = -1.0 if f in (wl.F_GAM + 2, wl.F_BET + 2, wl.F_B + 2, wl.F_G + 2, wl.F_G + 4, wl.F_A + 2, wl.F_A + 4) else 1.0
        act = (slice(NG, NG + p.ny), slice(NG, NG + p.nx))
        for m in range(NG):
            assert np.array_equal(o[NG - 1 - m][act], par * b[NG + m][act]), (f, m)
        chk = o.copy()
        chk[:NG, NG:NG + p.ny, NG:NG + p.nx] = b[:NG, NG:NG + p.ny, NG:NG + p.nx]
        assert np.array_equal(chk, b)


def test_mirror_face_half_domain_equals_full_domain_bitwise():
    """data symmetric under z -> -z on a box [-L, L] in z with six Sommerfeld faces; the upper half with a MIRROR face
    at z = 0 must give the same shell values bit for bit (centred z-stencils through the mirror ghosts)"""
    n = 12
    h = 0.25
    rng = np.random.default_rng(4)
    amp = rng.uniform(0.5, 1.5, NF) * 1e-2
    zpar = np.ones(NF)
    for f in (wl.F_GAM + 2, wl.F_BET + 2, wl.F_B + 2, wl.F_G + 2, wl.F_G + 4, wl.F_A + 2, wl.F_A + 4):
        zpar[f] = -1.0
    def fn(X, Y, Z):
        v = flat(X.shape)
        for f in range(NF):
            s = np.sin(0.7 * X + 0.2 * f) * np.cos(0.5 * Y)
            v[f] = v[f] + amp[f] * s * (np.cos(0.9 * Z) if zpar[f] > 0 else np.sin(0.9 * Z))
        return v
    ox, oy = 2.0, 1.5
    # full: 2n cells in z centred on z = 0; built as one n x n x 2n patch
    psF, totF = wl.make_layout([(n, n, 2 * n)], [h], [0.05], [(ox, oy, -(n - 0.5) * h)])
    wF = wl.Workload("full", psF, dict(wl.DEFAULT_PARAMS), np.zeros(totF))
    psH, totH = wl.make_layout([(n, n, n)], [h], [0.05], [(ox, oy, 0.5 * h)])
    wH = wl.Workload("half", psH, dict(wl.DEFAULT_PARAMS), np.zeros(totH))
    from helpers import storage_coords
    for w in (wF, wH):
        Z, Y, X = storage_coords(w.patches[0])
        vals = fn(X, Y, Z)
        for f in range(NF):
            w.field_view(w.state, 0, f)[...] = vals[f]
    # make the full data exactly symmetric (copy the upper half down with parity), the half's z- ghosts come from the fill
    for f in range(NF):
        a = wF.active_view(wF.state, 0, f)
        a[:n] = zpar[f] * a[n:][::-1]
        assert np.array_equal(a[n:], wH.active_view(wH.state, 0, f))
    bF = [((ox, oy, -(n - 0.5) * h), ALL_SOM)]
    facesH = [SOM, SOM, SOM, SOM, MIR, SOM]
    bH = [((ox, oy, 0.5 * h), facesH)]
    uH = orc.fill_ghosts_faces(psH, bH, wH.state.copy())
    rF = orc.sommerfeld_rhs(psF, bF, wF.state)
    rH = orc.sommerfeld_rhs(psH, bH, uH)
    mask = _shell_mask(n, facesH)
    for f in range(NF):
        full_upper = wF.active_view(rF, 0, f)[n:]
        half = wH.active_view(rH, 0, f)
        assert np.array_equal(half[mask], full_upper[mask]), wl.FIELD_NAMES[f]
        assert np.max(np.abs(half[mask])) > 0
