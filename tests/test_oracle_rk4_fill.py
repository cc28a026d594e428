"""Pins for the oracle's ghost fill (item 2) and classical RK4 (item 11)."""
import numpy as np

import orc
from helpers import NF, NG
from paper_2607_08743_b200 import workloads as wl


def test_ghost_fill_matches_numpy_wrap_padding():
    """Brute force: periodic fill == np.pad(mode='wrap') of the active block, faces, edges and corners."""
    rng = np.random.default_rng(3)
    patches, total = wl.make_layout([(7, 6, 9), (6, 8, 6)], [0.1, 0.2], [0.01, 0.02], [(0, 0, 0)] * 2)
    w = wl.Workload("t", patches, dict(wl.DEFAULT_PARAMS), rng.normal(size=total))
    before = w.state.copy()
    orc.fill_ghosts(w.patches, w.state)
    touched = np.zeros(total, dtype=bool)
    for ip, p in enumerate(patches):
        for f in range(NF):
            act = w.active_view(before, ip, f)
            want = np.pad(act, NG, mode="wrap")
            got = w.field_view(w.state, ip, f)[:, :, :p.nx + 2 * NG]
            assert np.array_equal(got, want)
            n = int(np.prod(p.shape)); o = p.patch_offset + f * p.field_stride
            t = touched[o:o + n].reshape(p.shape); t[:, :, :p.nx + 2 * NG] = True
    assert np.array_equal(w.state[~touched], before[~touched])     # pitch padding and gaps untouched


def test_rk4_step_equals_four_substeps_and_stage_table():
    """rk4_step == fill/substep x4 + fill (bitwise), and the stage table of item 11 on a frozen k."""
    w = wl.config0(n=8, eps=1e-3, amp=1e-6)
    ps, prm = w.patches, w.params
    u = w.state.copy(); orc.fill_ghosts(ps, u)
    ref = u.copy(); S = orc.rk4_step(ps, prm, ref)
    un = u.copy(); a = np.zeros_like(u); b = np.zeros_like(u); acc = np.zeros_like(u)
    ks = []
    for stage, (src, dst) in enumerate([(un, a), (a, b), (b, a), (a, None)], start=1):
        orc.fill_ghosts(ps, src)
        ks.append(orc.z4c_rhs(ps, prm, src))
        out = dst if dst is not None else np.zeros_like(u)
        orc.rk4_substep(ps, prm, stage, un, src, out, acc)
        last = out
    orc.fill_ghosts(ps, last)
    dt = ps[0].dt
    for f in range(NF):
        k1, k2, k3, k4 = (w.active_view(k, 0, f) for k in ks)
        Sf = (((k1 + 2 * k2) + 2 * k3) + k4) * (1.0 / 6.0)
        assert np.array_equal(w.active_view(acc, 0, f), Sf)
        assert np.array_equal(w.active_view(S, 0, f), Sf)
        assert np.array_equal(w.active_view(last, 0, f), w.active_view(un, 0, f) + dt * Sf)
        assert np.array_equal(w.field_view(last, 0, f)[:, :, :8 + 2 * NG], w.field_view(ref, 0, f)[:, :, :8 + 2 * NG])
        # stage inputs: u + dt/2 k1, u + dt/2 k2, u + dt k3
        assert np.array_equal(w.active_view(b, 0, f), w.active_view(un, 0, f) + (dt / 2) * k2)


def test_rk4_tt_wave_follows_stability_polynomial():
    """Noise-free TT data: (gt_yy-1, At_yy) amplitudes obey d/dt (g,A) = L (g,A), L=[[q,-2],[-s2/2,q]].
    One RK4 step must equal (I + zL + ... + z^4 L^4/24) to O(eps^2): pins the stage weights 1/2,1/2,1 and
    1/6,2/6,2/6,1/6 (any other choice changes the z^2..z^4 coefficients)."""
    n, sigma = 32, 0.1
    h = 1.0 / n
    th = 2 * np.pi * h
    s2 = (8 * np.cos(th) / 3 - np.cos(2 * th) / 6 - 2.5) / h ** 2
    q = -sigma * np.sin(th / 2) ** 6 / h
    L = np.array([[q, -2.0], [-0.5 * s2, q]])
    dt = 0.25 * h
    P = np.eye(2); term = np.eye(2)
    for m in range(1, 5):
        term = term @ (dt * L) / m
        P = P + term
    x = np.arange(n) * h
    s, c = np.sin(2 * np.pi * x), np.cos(2 * np.pi * x)
    mism = []
    for eps in (1e-3, 5e-4):
        w = wl.config0(n=n, eps=eps, amp=0.0)
        u = w.state.copy()
        orc.rk4_step(w.patches, w.params, u)
        gs, As = P @ np.array([eps, 0.0])         # sine pair
        gc, Ac = P @ np.array([0.0, np.pi * eps])  # cosine pair
        g = gs * s + gc * c
        A = As * s + Ac * c
        exp = {wl.F_G + 3: 1 + g, wl.F_G + 5: 1 - g, wl.F_A + 3: A, wl.F_A + 5: -A,
               wl.F_W: 1 + 0 * x, wl.F_G: 1 + 0 * x, wl.F_ALP: 1 + 0 * x}
        worst = 0.0
        for f in range(NF):
            e = exp.get(f, 0 * x)
            worst = max(worst, np.max(np.abs(w.active_view(u, 0, f) - e[None, None, :])))
        mism.append(worst)
    assert mism[0] < 1.0 * (1e-3) ** 2, mism
    assert 3.5 < mism[0] / mism[1] < 4.5, mism
    # Odd part in eps removes the eps^2 terms: the linear response must then match to O(eps^3), which is
    # below the z^4 term of the stability polynomial (eps * |(dt L)^4/24| ~ 2e-11 at eps = 1e-4).
    eps = 1e-4
    us = []
    for sg in (+1, -1):
        w = wl.config0(n=n, eps=sg * eps, amp=0.0)
        u = w.state.copy()
        orc.rk4_step(w.patches, w.params, u)
        us.append(u)
    gs, As = P @ np.array([eps, 0.0]); gc, Ac = P @ np.array([0.0, np.pi * eps])
    g_odd = 0.5 * (w.active_view(us[0], 0, wl.F_G + 3) - w.active_view(us[1], 0, wl.F_G + 3))[0, 0, :]
    A_odd = 0.5 * (w.active_view(us[0], 0, wl.F_A + 3) - w.active_view(us[1], 0, wl.F_A + 3))[0, 0, :]
    z4 = np.abs(np.linalg.matrix_power(dt * L, 4) / 24) @ np.array([eps, np.pi * eps])
    assert np.max(np.abs(g_odd - (gs * s + gc * c))) < 0.2 * z4[0]
    assert np.max(np.abs(A_odd - (As * s + Ac * c))) < 0.2 * z4[1]
