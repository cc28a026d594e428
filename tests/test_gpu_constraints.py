"""-m gpu: the constraint monitor (sacra_constraints, sacra_constraint_norms) against the oracle.
The kernel evaluates Eqs. 20-21 in the conformal variables, the oracle on the rebuilt physical metric: different
routes to the same definition. Tolerance: per constraint max|d| <= 1e-11 (max|ref| + floor); the floor is the
round-off of the cancelling second-derivative terms (1e-16 / h^2), since on a solution the constraint itself is ~0."""
import numpy as np
import pytest
import torch

import orc
from gpu_util import dev, host
from helpers import NF
from paper_2607_08743_b200 import sacra
from paper_2607_08743_b200 import workloads as wl
from test_gpu_parity import _ragged_workload, _smooth_random

pytestmark = pytest.mark.gpu
RTOL = 1e-11


def _gpu_constraints(w, filled):
    u = dev(filled)
    con = torch.full_like(u, float("nan"))
    sacra.constraints(w.patches, u, con)
    return con


def _compare(w, got, ref, what):
    for c in range(4):
        for ip, p in enumerate(w.patches):
            a, b = w.active_view(got, ip, c), w.active_view(ref, ip, c)
            scale = max(np.max(np.abs(w.active_view(ref, q, c))) for q in range(len(w.patches)))
            floor = 50 * 2.2e-16 / p.dx ** 2
            assert np.max(np.abs(a - b)) <= RTOL * scale + floor * RTOL * 1e5, (what, c, ip, np.max(np.abs(a - b)), scale)


def test_constraints_generic_data_ragged_batch():
    """all fields active, non-unit det gt, tr At != 0, several ragged patches; untouched outside fields 0..3"""
    w = _smooth_random(_ragged_workload(dims=[(37, 9, 11), (6, 6, 6), (16, 33, 7)]), 41)
    u = w.state.copy()
    orc.fill_ghosts(w.patches, u)
    ref = orc.constraints(w.patches, u)
    con = _gpu_constraints(w, u)
    got = host(con)
    mask = np.ones(got.size, dtype=bool)
    for ip, p in enumerate(w.patches):
        for c in range(4):
            o = p.patch_offset + c * p.field_stride
            mask[o:o + int(np.prod(p.shape))].reshape(p.shape)[3:3 + p.nz, 3:3 + p.ny, 3:3 + p.nx] = False
    assert np.all(np.isnan(got[mask])), "written outside the active cells of fields 0..3"
    assert not np.any(np.isnan(got[~mask]))
    _compare(w, np.nan_to_num(got), ref, "generic")
    assert max(np.max(np.abs(w.active_view(ref, 0, c))) for c in range(4)) > 1e-2


@pytest.mark.parametrize("idx", [0, 1, 2, 3])
def test_constraints_configs(idx):
    w = wl.make(idx)
    u = w.state.copy()
    orc.fill_ghosts(w.patches, u)
    ref = orc.constraints(w.patches, u)
    got = np.nan_to_num(host(_gpu_constraints(w, u)))
    _compare(w, got, ref, w.name)


def test_norms_match_eq22_and_are_deterministic():
    w = _smooth_random(_ragged_workload(dims=[(13, 8, 9), (8, 8, 8), (9, 6, 21)]), 42)
    u = w.state.copy()
    orc.fill_ghosts(w.patches, u)
    con = _gpu_constraints(w, u)
    scratch = torch.zeros(sacra.constraint_scratch_doubles(w.patches), dtype=torch.float64, device="cuda")
    norms = torch.zeros(4, dtype=torch.float64, device="cuda")
    sacra.constraint_norms(w.patches, con, scratch, norms)
    got = host(norms).copy()
    want = orc.constraint_norms(w.patches, orc.constraints(w.patches, u))
    assert np.allclose(got, want, rtol=1e-11, atol=0.0), (got, want)
    for _ in range(3):                                       # fixed reduction order: bit-identical repeats
        norms.zero_()
        scratch.fill_(7.0)
        sacra.constraint_norms(w.patches, con, scratch, norms)
        assert np.array_equal(host(norms), got)


def test_constraints_after_a_step_stay_at_truncation_level_on_puncture_data():
    """physics sanity through the whole path: on config 1 (a puncture at h = 0.25: ||H|| is the truncation error near
    r = 0) one RK4 step leaves ||H|| where it was, and the momentum constraint, exactly satisfied by the
    time-symmetric initial data, stays below it"""
    w = wl.make(1)
    u = dev(w.state)
    n = u.numel()
    work = torch.zeros(3 * n, dtype=torch.float64, device="cuda")
    scratch = torch.zeros(sacra.constraint_scratch_doubles(w.patches), dtype=torch.float64, device="cuda")
    norms = torch.zeros(4, dtype=torch.float64, device="cuda")
    con = torch.zeros_like(u)
    sacra.fill_ghosts(w.patches, u)
    sacra.constraints(w.patches, u, con)
    sacra.constraint_norms(w.patches, con, scratch, norms)
    before = host(norms).copy()
    sacra.rk4_step(w.patches, w.params, u, work)
    sacra.constraints(w.patches, u, con)
    sacra.constraint_norms(w.patches, con, scratch, norms)
    after = host(norms)
    assert np.all(np.isfinite(after)), after
    assert np.all(before[1:] < 1e-9) and 0.8 * before[0] < after[0] < 1.2 * before[0], (before, after)
    assert np.all(after[1:] < before[0]), (before, after)
