"""-m gpu: physical boundaries of the CUDA path against the oracle: per-face ghost fill (bit-exact),
the Sommerfeld shell of Eq. 13 (bit-exact: same operation order, no FMA contraction), and an RK4 step on a
non-periodic box -- z- mirror, the five other faces Sommerfeld -- within the
north_star tolerance on the increment S, cells of the shell and of the interior alike."""
import numpy as np
import pytest
import torch

import orc
from gpu_util import dev, host
from helpers import NF, NG, parity_report
from paper_2607_08743_b200 import sacra
from paper_2607_08743_b200 import workloads as wl

pytestmark = pytest.mark.gpu
SOM, MIR, PER, NONE = sacra.BC_SOMMERFELD, sacra.BC_MIRROR, sacra.BC_PERIODIC, sacra.BC_NONE
RTOL, FLOOR = 1e-11, 1e-14


def _workload(dims, seed=3, amp=0.02):
    rng = np.random.default_rng(seed)
    hs = [0.2 + 0.05 * q for q in range(len(dims))]
    ps, total = wl.make_layout(dims, hs, [0.25 * h for h in hs], [(0, 0, 0)] * len(dims))
    w = wl.Workload("bc", ps, dict(wl.DEFAULT_PARAMS), rng.normal(size=total) * 1e-3)
    for ip, p in enumerate(ps):
        z, y, x = np.meshgrid(np.arange(p.nz), np.arange(p.ny), np.arange(p.nx), indexing="ij")
        for f in range(NF):
            v = amp * np.sin(0.37 * x + 0.2 * f) * np.cos(0.29 * y - 0.1 * f) * np.cos(0.41 * z + 0.3)
            if f in (wl.F_W, wl.F_G, wl.F_G + 3, wl.F_G + 5, wl.F_ALP):
                v = v + 1.0
            w.active_view(w.state, ip, f)[...] = v
    return w


def _bnd(w, faces_list):
    return [((4.0 + 0.3 * q, 3.0, 0.5 * p.dx if faces_list[q][4] == MIR else 2.5), faces_list[q])
            for q, p in enumerate(w.patches)]


FACES = [[SOM, SOM, SOM, SOM, MIR, SOM], [SOM, SOM, SOM, SOM, SOM, SOM], [PER, PER, MIR, SOM, NONE, SOM]]


def test_fill_ghosts_faces_bit_exact():
    w = _workload([(9, 7, 8), (6, 6, 6), (21, 10, 13)])
    bnd = _bnd(w, FACES)
    ref = orc.fill_ghosts_faces(w.patches, bnd, w.state.copy())
    u = dev(w.state)
    sacra.fill_ghosts_faces(w.patches, bnd, u)
    assert np.array_equal(host(u), ref)


def test_sommerfeld_rhs_bit_exact_and_only_on_the_shell():
    w = _workload([(19, 8, 9), (6, 6, 6), (33, 10, 13)])
    bnd = _bnd(w, FACES)
    u = orc.fill_ghosts_faces(w.patches, bnd, w.state.copy())
    ref = orc.sommerfeld_rhs(w.patches, bnd, u, np.full(u.size, 7.0))
    got = torch.full((u.size,), 7.0, dtype=torch.float64, device="cuda")
    sacra.sommerfeld_rhs(w.patches, bnd, dev(u), got)
    got = host(got)
    assert np.array_equal(got, ref)
    assert np.sum(got != 7.0) > 1000


@pytest.mark.parametrize("flags", [0, 1])
def test_rk4_step_with_mirror_and_sommerfeld_faces(flags):
    w = _workload([(20, 18, 13), (8, 9, 7)], seed=5)
    faces = [[SOM, SOM, SOM, SOM, MIR, SOM], [SOM, NONE, SOM, SOM, SOM, SOM]]
    bnd = _bnd(w, faces)
    ref = w.state.copy()
    S_ref = orc.rk4_step_bc(w.patches, bnd, w.params, ref)
    u = dev(w.state)
    n = u.numel()
    work = torch.zeros(3 * n, dtype=torch.float64, device="cuda")
    sacra.rk4_step_bc(w.patches, dict(w.params, flags=flags), bnd, u, work)
    got, S = host(u), host(work[2 * n:])
    if flags == 0:
        bad = parity_report(w, S, S_ref, RTOL, FLOOR)
        assert not bad, bad
    for ip, p in enumerate(w.patches):
        for f in range(NF):
            a, b = w.active_view(got, ip, f), w.active_view(ref, ip, f)
            tol = p.dt * RTOL * (np.max(np.abs(w.active_view(S_ref, ip, f))) + FLOOR) + np.spacing(np.abs(b))
            assert np.all(np.abs(a - b) <= tol), (ip, wl.FIELD_NAMES[f])
    # ghosts: mirror faces filled like the oracle's; ghosts behind Sommerfeld / none faces untouched (still the input's)
    chk = orc.fill_ghosts_faces(w.patches, bnd, got.copy())
    assert np.array_equal(chk, got)
    p = w.patches[0]
    for f in (0, 5, 20):
        assert np.array_equal(w.field_view(got, 0, f)[:, :, :NG], w.field_view(w.state, 0, f)[:, :, :NG])


def test_substep_bc_stage_table_shell_bitwise():
    """the shell cells follow the stage table with the Sommerfeld k, bit for bit like the oracle's substep"""
    w = _workload([(12, 11, 10)], seed=9)
    bnd = _bnd(w, [[SOM, SOM, SOM, SOM, MIR, SOM]])
    ps, prm = w.patches, w.params
    un = orc.fill_ghosts_faces(ps, bnd, w.state.copy())
    uin = un.copy()
    acc_ref = np.zeros_like(un)
    acc_gpu = torch.zeros(un.size, dtype=torch.float64, device="cuda")
    p = ps[0]
    i = np.arange(p.nx); j = np.arange(p.ny); k = np.arange(p.nz)
    shell = ((i < 3) | (i >= p.nx - 3))[None, None, :] | ((j < 3) | (j >= p.ny - 3))[None, :, None] | (k >= p.nz - 3)[:, None, None]
    for stage in (1, 2, 3, 4):
        out_ref = np.zeros_like(un)
        orc.rk4_substep_bc(ps, bnd, prm, stage, un, uin, out_ref, acc_ref)
        out_gpu = torch.zeros_like(acc_gpu)
        d_un = dev(un)
        sacra.rk4_substep_bc(ps, prm, bnd, stage, d_un, d_un if stage == 1 else dev(uin), out_gpu, acc_gpu)
        for f in range(NF):
            assert np.array_equal(w.active_view(host(out_gpu), 0, f)[shell], w.active_view(out_ref, 0, f)[shell]), (stage, f)
            assert np.array_equal(w.active_view(host(acc_gpu), 0, f)[shell], w.active_view(acc_ref, 0, f)[shell]), (stage, f)
        uin = orc.fill_ghosts_faces(ps, bnd, out_ref.copy())
        acc_gpu = dev(acc_ref)
