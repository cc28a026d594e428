"""Pins for the oracle's Z4c right-hand side.

None of these compares the oracle with itself: exact solutions of Einstein's
equations must be stationary (Minkowski exactly, Kerr-Schild and isotropic
Schwarzschild at 4th order), a linearised TT wave has a closed-form time
derivative, Theta must obey the wave equation, pi-symmetry must hold bitwise
(PAPER.md:280), and the algebraic identities hold for any data.
"""
import numpy as np
import pytest

import orc
from helpers import NF, NG, analytic_state, flat, pi_partner
from paper_2607_08743_b200 import workloads as wl

PRM = dict(wl.DEFAULT_PARAMS)
SYM = [[0, 1, 2], [1, 3, 4], [2, 4, 5]]


# --------------------------------------------------------------------------- check (1)
def test_minkowski_rhs_is_exactly_zero():
    n = 8
    w = analytic_state(n, 1.0 / n, (0, 0, 0), lambda X, Y, Z: flat(X.shape))
    rhs = orc.z4c_rhs(w.patches, PRM, w.state)
    assert np.all(rhs == 0.0)
    S = orc.rk4_step(w.patches, PRM, w.state.copy())
    assert np.all(S == 0.0)


# --------------------------------------------------------------------------- exact solutions
def kerr_schild(X, Y, Z, M=1.0):
    """Schwarzschild in Kerr-Schild coordinates in the evolved variables (K_ij from d_t gamma_ij=0)."""
    r = np.sqrt(X * X + Y * Y + Z * Z)
    H = M / r
    l = [X / r, Y / r, Z / r]
    alp = (1 + 2 * H) ** -0.5
    W = (1 + 2 * H) ** (-1.0 / 6.0)
    v = [np.zeros_like(X) for _ in range(NF)]
    v[wl.F_W] = W
    v[wl.F_ALP] = alp
    K = 2 * H * alp / r * (1 + 3 * H) / (1 + 2 * H)
    v[wl.F_KH] = K
    # Gt^i = -(a' + b' + 2 b / r) l^i with gt^ij = a delta^ij + b l^i l^j
    Hp = -M / r ** 2
    a_p = (1.0 / 3.0) * (1 + 2 * H) ** (-2.0 / 3.0) * 2 * Hp
    b = -2 * H * (1 + 2 * H) ** (-2.0 / 3.0)
    b_p = -2 * Hp * (1 + 2 * H) ** (-2.0 / 3.0) + 2 * H * (2.0 / 3.0) * (1 + 2 * H) ** (-5.0 / 3.0) * 2 * Hp
    gfac = -(a_p + b_p + 2 * b / r)
    for i in range(3):
        v[wl.F_BET + i] = 2 * H / (1 + 2 * H) * l[i]
        v[wl.F_GAM + i] = gfac * l[i]
        for j in range(i, 3):
            d = 1.0 if i == j else 0.0
            gij = d + 2 * H * l[i] * l[j]
            Kij = 2 * H * alp / r * (d - (2 + H) * l[i] * l[j])
            v[wl.F_G + SYM[i][j]] = W * W * gij
            v[wl.F_A + SYM[i][j]] = W * W * (Kij - gij * K / 3.0)
    return v


def isotropic_schwarzschild(X, Y, Z, M=1.0):
    r = np.sqrt(X * X + Y * Y + Z * Z)
    v = flat(X.shape)
    v[wl.F_W] = (1 + M / (2 * r)) ** -2
    v[wl.F_ALP] = (1 - M / (2 * r)) / (1 + M / (2 * r))
    return v


GEOM = [wl.F_W] + list(range(wl.F_G, wl.F_G + 6)) + [wl.F_KH] + list(range(wl.F_A, wl.F_A + 6)) + \
       list(range(wl.F_GAM, wl.F_GAM + 3)) + [wl.F_TH]


def _rhs_err(fn, n, fields, prm):
    L = 1.5
    h = L / n
    w = analytic_state(n, h, (1.6 + 0.5 * h, 0.9 + 0.5 * h, -0.5 + 0.5 * h), fn)
    rhs = orc.z4c_rhs(w.patches, prm, w.state)
    return np.array([np.max(np.abs(w.active_view(rhs, 0, f))) for f in fields])


def test_kerr_schild_is_stationary_at_fourth_order():
    """Pins every term of item 8 that is non-zero in vacuum with shift, K != 0 and a non-flat gt_ij."""
    prm = dict(PRM, ko_sigma=0.0, kappa1=0.0)
    e1 = _rhs_err(kerr_schild, 12, GEOM, prm)
    e2 = _rhs_err(kerr_schild, 24, GEOM, prm)
    assert np.all(e2 < 2e-5), e2                    # term scales are 1e-2..1e-1
    ratio = e1 / e2
    assert np.all(ratio > 11) and np.all(ratio < 22), ratio


def test_kerr_schild_wrong_data_does_not_converge():
    """Sanity of the pin itself: a 1% error in K_ij (At) leaves an O(1e-3) residual that does not converge away."""
    def bad(X, Y, Z):
        v = kerr_schild(X, Y, Z)
        for s in range(6):
            v[wl.F_A + s] = 1.01 * v[wl.F_A + s]
        return v
    prm = dict(PRM, ko_sigma=0.0, kappa1=0.0)
    e2 = _rhs_err(bad, 24, GEOM, prm)
    assert np.max(e2) > 1e-4


def test_isotropic_schwarzschild_is_static_at_fourth_order():
    """W-sector of the Ricci tensor and the lapse Hessian: R = 0 and D_iD_j alpha = alpha R_ij."""
    prm = dict(PRM, ko_sigma=0.0)
    fields = GEOM + [wl.F_ALP]
    e1 = _rhs_err(isotropic_schwarzschild, 12, fields, prm)
    e2 = _rhs_err(isotropic_schwarzschild, 24, fields, prm)
    assert np.all(e2 < 1e-5), e2
    nz = e2 > 1e-13                                 # fields whose RHS vanishes identically stay 0
    ratio = e1[nz] / e2[nz]
    assert nz.sum() >= 8
    assert np.all(ratio > 11) and np.all(ratio < 22), ratio


# --------------------------------------------------------------------------- check (3)
def _symbols(n, m=1, sigma=0.1):
    h = 1.0 / n
    th = 2 * np.pi * m * h
    s1 = (4 * np.sin(th) / 3 - np.sin(2 * th) / 6) / h
    s2 = (8 * np.cos(th) / 3 - np.cos(2 * th) / 6 - 2.5) / h ** 2
    q = -sigma * np.sin(th / 2) ** 6 / h
    return s1, s2, q


def _tt_rhs_mismatch(eps, n=32):
    w = wl.config0(n=n, eps=eps, amp=0.0)
    p = w.patches[0]
    orc.fill_ghosts(w.patches, w.state)
    rhs = orc.z4c_rhs(w.patches, w.params, w.state)
    x = np.arange(n) / n
    s, c = np.sin(2 * np.pi * x), np.cos(2 * np.pi * x)
    s1, s2, q = _symbols(n, sigma=w.params["ko_sigma"])
    expect = {wl.F_G + 3: -2 * np.pi * eps * c + q * eps * s,
              wl.F_G + 5: +2 * np.pi * eps * c - q * eps * s,
              wl.F_A + 3: -0.5 * s2 * eps * s + q * np.pi * eps * c,
              wl.F_A + 5: +0.5 * s2 * eps * s - q * np.pi * eps * c}
    worst = 0.0
    for f in range(NF):
        e = expect.get(f, np.zeros(n))
        worst = max(worst, np.max(np.abs(w.active_view(rhs, 0, f) - e[None, None, :])))
    return worst


def test_tt_wave_rhs_matches_closed_form_to_second_order():
    m1 = _tt_rhs_mismatch(1e-3)
    m2 = _tt_rhs_mismatch(5e-4)
    assert m1 < 60 * (1e-3) ** 2            # O(eps^2) with second-derivative-sized coefficients
    assert 3.6 < m1 / m2 < 4.4, (m1, m2)    # halving eps quarters the mismatch
    # continuum values: d_t gt_yy = -2 pi eps cos, d_t At_yy = +2 pi^2 eps sin (s2 ~ -4 pi^2)
    s1, s2, q = _symbols(32)
    assert abs(-0.5 * s2 - 2 * np.pi ** 2) < 2e-3 * 2 * np.pi ** 2


# --------------------------------------------------------------------------- Theta couplings
def test_theta_obeys_unit_speed_wave_equation():
    """Constraint propagation. kappa1 = sigma = 0 and shift frozen (shift_coef = 0), flat data
    plus Theta = eps sin(kx). Linearised item 8 closes on (Theta, W, Gt^x):
        Theta' = 1/2 (D1 Gt^x + 4 D2 W),  W' = 2/3 Theta,  Gt^x' = -2/3 D1 Theta
    so Theta'' = lam Theta with lam = 1/2 (2/3 s1^2 + 8/3 s2) -> -k^2: the unit-speed wave equation. A plain
    BSSN coefficient (-4/3 dK with K = Kh + 2 Theta) or a missing 2 Theta in the W equation changes lam.
    One RK4 step of a linear system gives Theta_1/Theta_0 = 1 + z/2 + z^2/24, z = lam dt^2."""
    n, eps = 32, 1e-5
    h = 1.0 / n
    prm = dict(PRM, kappa1=0.0, ko_sigma=0.0, shift_coef=0.0)
    th = []
    for sgn in (+1.0, -1.0):       # odd part in eps removes the eps^2 terms (1/3 alpha K^2, ...)
        def fn(X, Y, Z):
            v = flat(X.shape)
            v[wl.F_TH] = sgn * eps * np.sin(2 * np.pi * X)
            return v
        w = analytic_state(n, h, (0, 0, 0), fn, dt=0.25 * h)
        u = w.state.copy()
        orc.rk4_step(w.patches, prm, u)
        th.append(w.active_view(u, 0, wl.F_TH)[0, 0, :].copy())
    th = 0.5 * (th[0] - th[1])
    s1, s2, _ = _symbols(n)
    lam = 0.5 * ((2.0 / 3.0) * s1 ** 2 + (8.0 / 3.0) * s2)
    assert abs(lam + (2 * np.pi) ** 2) < 0.01 * (2 * np.pi) ** 2        # continuum limit: -k^2
    z = lam * (0.25 * h) ** 2
    x = np.arange(n) * h
    # round-off floor: W = 1 + O(eps dt) carries 1e-16, amplified by 4 D2 dt ~ 2e2 -> 2e-9 of eps
    assert np.max(np.abs(th / eps - (1 + z / 2 + z * z / 24) * np.sin(2 * np.pi * x))) < 2e-8
    assert abs(z / 2) > 1e-3                                               # the pin has teeth


def test_uniform_theta_decays_at_rate_2_kappa1():
    n = 8
    def fn(X, Y, Z):
        v = flat(X.shape)
        v[wl.F_TH] = np.full_like(X, 1e-6)
        return v
    w = analytic_state(n, 1.0 / n, (0, 0, 0), fn)
    prm = dict(PRM, kappa1=0.05, kappa2=0.0)
    rhs = orc.z4c_rhs(w.patches, prm, w.state)
    th = w.active_view(rhs, 0, wl.F_TH)
    # -alpha kappa1 (2+kappa2) Theta + 1/3 alpha K^2 (K = 2 Theta): second order in Theta
    assert np.allclose(th, -2 * 0.05 * 1e-6, rtol=1e-5)
    kh = w.active_view(rhs, 0, wl.F_KH)
    assert np.allclose(kh, 0.05 * 1e-6, rtol=1e-4)          # + alpha kappa1 (1-kappa2) Theta


# --------------------------------------------------------------------------- invariants on random data
def _random_point(rng):
    u = rng.normal(size=NF) * 0.3
    g = np.eye(3) + 0.2 * rng.normal(size=(3, 3)); g = 0.5 * (g + g.T) + np.eye(3)
    for i in range(3):
        for j in range(i, 3):
            u[wl.F_G + SYM[i][j]] = g[i, j]
    u[wl.F_W] = 0.7; u[wl.F_ALP] = 0.9
    return u, rng.normal(size=(NF, 3)), rng.normal(size=(NF, 6)), rng.normal(size=NF), rng.normal(size=NF)


def test_algebraic_identities_on_random_data():
    rng = np.random.default_rng(7)
    prm = dict(PRM, kappa1=0.3, kappa2=0.2, eta=1.3)
    for _ in range(20):
        u, d1, d2, adv, ko = _random_point(rng)
        out = orc.rhs_point(prm, u, d1, d2, adv, ko)
        g = np.array([[u[wl.F_G + SYM[i][j]] for j in range(3)] for i in range(3)])
        A = np.array([[u[wl.F_A + SYM[i][j]] for j in range(3)] for i in range(3)])
        gi = np.linalg.inv(g)
        full = lambda base, vec: np.array([[vec[base + SYM[i][j]] for j in range(3)] for i in range(3)])
        # gt^ij RHS(gt_ij) = -2 alpha gt^ij At_ij + gt^ij (adv+ko)_ij     (d beta terms cancel)
        lhs = np.sum(gi * full(wl.F_G, out))
        rhs = -2 * u[wl.F_ALP] * np.sum(gi * A) + np.sum(gi * full(wl.F_G, adv + ko))
        assert abs(lhs - rhs) < 1e-11 * (1 + abs(rhs))
        # RHS(B^i) - RHS(Gt^i) + eta B^i = (adv+ko)_B - (adv+ko)_Gt   (KO cancels out of the difference... not inside)
        for i in range(3):
            l = out[wl.F_B + i] - out[wl.F_GAM + i] + prm["eta"] * u[wl.F_B + i]
            r = (adv[wl.F_B + i] + ko[wl.F_B + i]) - (adv[wl.F_GAM + i] + ko[wl.F_GAM + i])
            assert abs(l - r) < 1e-10 * (1 + abs(out[wl.F_GAM + i]))
            assert abs(out[wl.F_BET + i] - (adv[wl.F_BET + i] + ko[wl.F_BET + i] + 0.75 * u[wl.F_B + i])) < 1e-13
        # lapse: -2 alpha K-hat (default) or -2 alpha (K-hat + 2 Theta)
        assert abs(out[wl.F_ALP] - (adv[wl.F_ALP] + ko[wl.F_ALP] - 2 * u[wl.F_ALP] * u[wl.F_KH])) < 1e-13
        out2 = orc.rhs_point(dict(prm, lapse_uses_khat=0), u, d1, d2, adv, ko)
        assert abs(out2[wl.F_ALP] - out[wl.F_ALP] + 4 * u[wl.F_ALP] * u[wl.F_TH]) < 1e-13
        # trace of the At equation with beta-derivatives zeroed and tr At = 0: gt^ij RHS(At_ij) = -2 alpha AtAt
        u2 = u.copy()
        tr = np.sum(gi * A)
        A2 = A - g * tr / 3.0
        for i in range(3):
            for j in range(i, 3):
                u2[wl.F_A + SYM[i][j]] = A2[i, j]
        d1b = d1.copy(); d1b[wl.F_BET:wl.F_BET + 3] = 0.0
        o3 = orc.rhs_point(prm, u2, d1b, d2, 0 * adv, 0 * ko)
        AA = np.einsum("ij,ik,jl,kl->", A2, gi, gi, A2)
        assert abs(np.sum(gi * full(wl.F_A, o3)) + 2 * u[wl.F_ALP] * AA) < 1e-9 * (1 + abs(AA))


# --------------------------------------------------------------------------- check (4)
def test_pi_symmetry_is_bitwise():
    """max abs pair difference is exactly zero. RHS and one full RK4 step (upwinding active
    from stage 3 on, where beta != 0), compared by subtraction with the component signs of PAPER.md:272."""
    w = wl.config2(n=24, half_width=8.0)    # h = 2/3: not a binary fraction on purpose
    u = w.state.copy()
    orc.fill_ghosts(w.patches, u)
    rhs = orc.z4c_rhs(w.patches, w.params, u)
    S = orc.rk4_step(w.patches, w.params, u)
    assert np.max(np.abs(w.active_view(u, 0, wl.F_BET))) > 0          # the shift did switch on
    for buf in (rhs, S, u):
        for f in range(NF):
            a = w.active_view(buf, 0, f)
            assert np.max(np.abs(a - wl.PI_SIGN[f] * pi_partner(a))) == 0.0, wl.FIELD_NAMES[f]
    assert np.max(np.abs(w.active_view(rhs, 0, wl.F_KH))) > 1e-6       # and the data are not trivial
