"""Pins for the oracle's stencils.

Everything here is fixed by mathematics, not by the oracle: polynomial
exactness, Fourier symbols, 4th-order convergence. A dropped term, wrong sign,
wrong offset or transposed axis in any stencil fails one of them.
"""
import numpy as np
import pytest

import orc
from helpers import NF, analytic_state
from paper_2607_08743_b200 import workloads as wl

SYMPAIRS = [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]


def _poly_state(n, h, origin, px, py, pz, beta):
    """field 0 = x^px y^py z^pz; beta fields constant = beta."""
    def fn(X, Y, Z):
        v = [np.zeros_like(X) for _ in range(NF)]
        v[0] = X ** px * Y ** py * Z ** pz
        for a in range(3):
            v[wl.F_BET + a] = np.full_like(X, beta[a])
        return v
    return analytic_state(n, h, origin, fn)


@pytest.mark.parametrize("beta", [(0.7, -0.3, 0.2), (-0.7, 0.3, -0.2), (0.0, 0.0, 0.0)])
@pytest.mark.parametrize("powers", [(4, 0, 0), (0, 4, 0), (0, 0, 4), (3, 1, 0), (1, 1, 2),
                                    (2, 2, 0), (0, 3, 1), (4, 4, 0), (4, 0, 4), (0, 4, 4)])
def test_polynomial_exactness(powers, beta):
    px, py, pz = powers
    n, h, org = 8, 0.125, (0.3, -0.2, 0.55)
    w = _poly_state(n, h, org, px, py, pz, beta)
    p = w.patches[0]
    i, j, k = 3, 4, 2
    x, y, z = (org[0] + i * h, org[1] + j * h, org[2] + k * h)
    d1, d2, adv, ko = orc.derivs_field(p, w.state, 0, i, j, k, sigma=0.4)
    mono = lambda t, q, dq: (np.prod(np.arange(q - dq + 1, q + 1)) * t ** (q - dq)) if q >= dq else 0.0
    c = [(x, px), (y, py), (z, pz)]
    def exact(dq):
        r = 1.0
        for a in range(3):
            r *= mono(c[a][0], c[a][1], dq[a])
        return r
    e1 = [exact(tuple(1 if a == b else 0 for b in range(3))) for a in range(3)]
    scale = max(1.0, abs(exact((0, 0, 0)))) / h ** 2
    np.testing.assert_allclose(d1, e1, rtol=0, atol=2e-13 * scale)
    for s, (a, b) in enumerate(SYMPAIRS):
        dq = [0, 0, 0]; dq[a] += 1; dq[b] += 1
        # diagonal D2 is exact to degree 5, mixed to degree 4 per axis
        assert abs(d2[s] - exact(tuple(dq))) <= 2e-12 * scale, (a, b)
    assert abs(adv - sum(beta[a] * e1[a] for a in range(3))) <= 2e-13 * scale
    assert abs(ko) <= 1e-12 * scale      # Q annihilates degree <= 5


def test_d2_diagonal_exact_degree5_and_ko_sees_degree6():
    n, h, org = 8, 0.25, (0.1, 0.2, 0.3)
    for axis in range(3):
        pw = [0, 0, 0]; pw[axis] = 5
        w = _poly_state(n, h, org, *pw, beta=(0, 0, 0))
        t = org[axis] + 3 * h
        d1, d2, adv, ko = orc.derivs_field(w.patches[0], w.state, 0, 3, 3, 3, sigma=1.0)
        assert abs(d2[[0, 3, 5][axis]] - 20 * t ** 3) < 1e-11
        assert abs(ko) < 1e-10
        # degree 6: (D+D-)^3 x^6 = 720 exactly, so Q x^6 = sigma h^5/64 * 720
        pw[axis] = 6
        w = _poly_state(n, h, org, *pw, beta=(0, 0, 0))
        _, _, _, ko = orc.derivs_field(w.patches[0], w.state, 0, 3, 3, 3, sigma=1.0)
        assert abs(ko - 720 * h ** 5 / 64) < 1e-10


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_fourier_symbols(axis):
    """sin/cos(k x_a) on a periodic grid: D1 -> (4 sin t/3 - sin 2t/6)/h, D2 -> (8cos t/3 - cos2t/6 - 5/2)/h^2,
    Q -> -sigma sin^6(t/2)/h, upwind -> centred symbol + |.|-signed dissipative part."""
    n, m, sigma = 16, 3, 0.3
    h = 1.0 / n
    kk = 2 * np.pi * m
    th = kk * h
    ph = 0.37
    def fn(X, Y, Z):
        v = [np.zeros_like(X) for _ in range(NF)]
        v[0] = np.sin(kk * (X, Y, Z)[axis] + ph)
        v[wl.F_BET + axis] = np.full_like(X, -0.5)
        return v
    w = analytic_state(n, h, (0.0, 0.0, 0.0), fn)
    i = j = k = 5
    t = kk * 5 * h + ph
    d1, d2, adv, ko = orc.derivs_field(w.patches[0], w.state, 0, i, j, k, sigma)
    s1 = (4 * np.sin(th) / 3 - np.sin(2 * th) / 6) / h
    s2 = (8 * np.cos(th) / 3 - np.cos(2 * th) / 6 - 2.5) / h ** 2
    assert abs(d1[axis] - s1 * np.cos(t)) < 1e-11 * abs(s1)
    assert abs(d2[[0, 3, 5][axis]] - s2 * np.sin(t)) < 1e-11 * abs(s2)
    assert abs(ko - (-sigma * np.sin(th / 2) ** 6 / h) * np.sin(t)) < 1e-11 / h
    # upwind symbol for beta<0 (stencil -u-3 +6u-2 -18u-1 +10u0 +3u+1)/(12h) applied to e^{i k x}
    z = np.exp(1j * th)
    sym = (-z ** -3 + 6 * z ** -2 - 18 * z ** -1 + 10 + 3 * z) / (12 * h)
    expect = -0.5 * np.imag(sym * np.exp(1j * t))
    assert abs(adv - expect) < 1e-11 / h
    # off-axis derivatives of a function of one coordinate vanish
    for a in range(3):
        if a != axis:
            assert abs(d1[a]) < 1e-12 / h


def test_mixed_symbol_is_product_and_axis_order():
    """D_ab sin(kx x+ky y+kz z) = -s1(a) s1(b) sin(.), each pair, distinct wavenumbers per axis."""
    n = 16
    h = 1.0 / n
    ks = 2 * np.pi * np.array([1, 2, 3])
    def fn(X, Y, Z):
        v = [np.zeros_like(X) for _ in range(NF)]
        v[0] = np.sin(ks[0] * X + ks[1] * Y + ks[2] * Z + 0.2)
        return v
    w = analytic_state(n, h, (0.0, 0.0, 0.0), fn)
    i, j, k = 2, 7, 11
    t = ks[0] * i * h + ks[1] * j * h + ks[2] * k * h + 0.2
    s1 = (4 * np.sin(ks * h) / 3 - np.sin(2 * ks * h) / 6) / h
    _, d2, _, _ = orc.derivs_field(w.patches[0], w.state, 0, i, j, k, 0.0)
    for s, (a, b) in enumerate(SYMPAIRS):
        if a != b:
            assert abs(d2[s] + s1[a] * s1[b] * np.sin(t)) < 1e-10 * abs(s1[a] * s1[b])


def test_fourth_order_convergence_all_operators():
    """Error ratio between h and h/2 is 16 (+-15%) for D1, D2 (6), upwind (both signs); KO -> 0 as h^5."""
    ph = np.array([0.31, 1.17, 2.03])
    kv = np.array([1.3, 0.9, 1.7])
    def make(n, beta):
        h = 1.0 / n
        def fn(X, Y, Z):
            v = [np.zeros_like(X) for _ in range(NF)]
            v[0] = np.sin(kv[0] * X + ph[0]) * np.sin(kv[1] * Y + ph[1]) * np.sin(kv[2] * Z + ph[2])
            for a in range(3):
                v[wl.F_BET + a] = np.full_like(X, beta[a])
            return v
        return analytic_state(n, h, (0.5, 0.5, 0.5), fn), h
    def exact(x, y, z, beta):
        s = [np.sin(kv[a] * c + ph[a]) for a, c in enumerate((x, y, z))]
        c = [kv[a] * np.cos(kv[a] * cc + ph[a]) for a, cc in enumerate((x, y, z))]
        d1 = np.array([c[0] * s[1] * s[2], s[0] * c[1] * s[2], s[0] * s[1] * c[2]])
        d2 = np.array([-kv[0] ** 2 * s[0] * s[1] * s[2], c[0] * c[1] * s[2], c[0] * s[1] * c[2],
                       -kv[1] ** 2 * s[0] * s[1] * s[2], s[0] * c[1] * c[2], -kv[2] ** 2 * s[0] * s[1] * s[2]])
        return d1, d2, float(np.dot(beta, d1))
    for beta in [(0.6, -0.4, 0.9), (-0.6, 0.4, -0.9)]:
        errs = []
        for n in (8, 16):
            w, h = make(n, beta)
            i = n // 2     # same physical point x = 0.5 + 0.5 = 1.0 at both resolutions
            d1, d2, adv, ko = orc.derivs_field(w.patches[0], w.state, 0, i, i, i, sigma=1.0)
            e1, e2, ea = exact(1.0, 1.0, 1.0, beta)
            errs.append(np.concatenate([d1 - e1, d2 - e2, [adv - ea], [ko]]))
        ratio = np.abs(errs[0]) / np.abs(errs[1])
        assert np.all(ratio[:10] > 13.5) and np.all(ratio[:10] < 18.5), ratio
        assert 27 < ratio[10] < 37, ratio      # KO term itself is O(h^5)
