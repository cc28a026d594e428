"""-m gpu: the inter-level operators (sacra_restrict, sacra_prolong_ghosts) against the oracle, bit for
bit (same weights, same nesting of the sums), on random data; everything outside the target cells untouched."""
import numpy as np
import pytest
import torch

import orc
from gpu_util import dev, host
from helpers import NF, NG
from paper_2607_08743_b200 import sacra
from paper_2607_08743_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _levels(nc=(8, 12, 6), npar=(16, 18, 14), org=(4, 5, 3)):
    pp, tp = wl.make_layout([npar], [0.2], [0.01], [(0.0, 0.0, 0.0)])
    pc, tc = wl.make_layout([nc], [0.1], [0.005], [(0.0, 0.0, 0.0)])
    rng = np.random.default_rng(9)
    return pp[0], rng.normal(size=tp), pc[0], rng.normal(size=tc), org


def test_restrict_bit_exact_and_only_covered_cells_written():
    pp, up, pc, uc, org = _levels()
    ref = orc.restrict(pp, pc, org, up.copy(), uc)
    d = dev(up)
    sacra.restrict(pp, pc, org, d, dev(uc))
    got = host(d)
    assert np.array_equal(got, ref)
    assert np.count_nonzero(got != up) == NF * (pc.nx // 2) * (pc.ny // 2) * (pc.nz // 2)


def test_prolong_ghosts_bit_exact_and_active_cells_untouched():
    pp, up, pc, uc, org = _levels()
    ref = orc.prolong_ghosts(pp, pc, org, up, uc.copy())
    d = dev(uc)
    sacra.prolong_ghosts(pp, pc, org, dev(up), d)
    got = host(d)
    assert np.array_equal(got, ref)
    nghost = (pc.nx + 6) * (pc.ny + 6) * (pc.nz + 6) - pc.nx * pc.ny * pc.nz
    assert np.count_nonzero(got != uc) == NF * nghost


def test_prolong_then_restrict_reproduces_a_cubic():
    """both operators are exact on cubics: parent -> child ghosts and child -> parent agree with the analytic field"""
    from helpers import storage_coords
    pp, tp = wl.make_layout([(16, 16, 16)], [0.2], [0.01], [(0.0, 0.0, 0.0)])
    org = (4, 4, 4)
    pc, tc = wl.make_layout([(8, 8, 8)], [0.1], [0.005], [tuple(o * 0.2 - 0.05 for o in org)])
    f = lambda X, Y, Z: (0.3 + X) ** 3 - (0.2 + Y) * Z ** 2 + X * Y * Z
    up, uc = np.zeros(tp), np.zeros(tc)
    wp = wl.Workload("p", pp, dict(wl.DEFAULT_PARAMS), up)
    wc = wl.Workload("c", pc, dict(wl.DEFAULT_PARAMS), uc)
    Z, Y, X = storage_coords(pp[0])
    Zc, Yc, Xc = storage_coords(pc[0])
    for n in range(NF):
        wp.field_view(up, 0, n)[...] = f(X, Y, Z)
        wc.active_view(uc, 0, n)[...] = f(Xc, Yc, Zc)[NG:-NG, NG:-NG, NG:NG + 8]
    dc = dev(uc)
    sacra.prolong_ghosts(pp[0], pc[0], org, dev(up), dc)
    got = host(dc)
    ex = f(Xc, Yc, Zc)[:, :, :14]
    assert np.max(np.abs(wc.field_view(got, 0, 3)[:, :, :14] - ex)) < 1e-13 * np.max(np.abs(ex))
    dp = dev(np.zeros(tp))
    sacra.restrict(pp[0], pc[0], org, dp, dc)
    back = wp.active_view(host(dp), 0, 3)[4:8, 4:8, 4:8]
    assert np.max(np.abs(back - wp.active_view(up, 0, 3)[4:8, 4:8, 4:8])) < 1e-13 * np.max(np.abs(ex))
