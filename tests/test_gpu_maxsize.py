"""-m gpu: a patch near the largest size the GPU holds (two states of 44 GB: 600^3 active cells, 5.6e9 doubles per
state, offsets beyond 2^32 elements), checked on EVERY point without a 600^3 oracle run: the data are a periodic tiling of
a random 40^3 block, so the right-hand side must be the same tiling -- bit for bit, since every point runs the same
instruction stream on the same neighbourhood -- of the right-hand side of the single periodic 40^3 block, which the
oracle checks to the north_star tolerance. Exercises 64-bit offsets, the tile order on a 38 x 150 x 100 tile grid and a
ragged last tile row (600 is not a multiple of 16)."""
import numpy as np
import pytest
import torch

import orc
from helpers import NF, NG, parity_report
from paper_2607_08743_b200 import sacra
from paper_2607_08743_b200 import workloads as wl

pytestmark = pytest.mark.gpu
M, REP = 40, 15


def _need(free, need, what):
    """These tests must not pass by skipping: on a B200 (180 GB; the box the -m gpu suite is for) too little free memory is
    a failure -- something else holds the device. Smaller GPUs skip, since the sizes are chosen for this one."""
    if free >= need:
        return
    name = torch.cuda.get_device_name()
    msg = "%s needs %.0f GB of device memory, %.0f GB free on %s" % (what, need / 1e9, free / 1e9, name)
    if "B200" in name or torch.cuda.get_device_properties(0).total_memory > (150 << 30):
        pytest.fail(msg)
    pytest.skip(msg)


def _release():
    """hand cached blocks of earlier tests back to the driver: these tests ask for most of the device"""
    import gc
    gc.collect()
    torch.cuda.synchronize()
    torch.cuda.empty_cache()


def test_rhs_on_a_600_cubed_patch_is_the_tiling_of_the_block_rhs():
    _release()
    free, _ = torch.cuda.mem_get_info()
    n = M * REP
    ps, total = wl.make_layout([(n, n, n)], [0.1], [0.025], [(0, 0, 0)])
    _need(free, 2 * total * 8 + (4 << 30), "the 600^3 right-hand side")
    assert total > 2 ** 32
    p = ps[0]
    rng = np.random.default_rng(12)
    pb, tb = wl.make_layout([(M, M, M)], [0.1], [0.025], [(0, 0, 0)])
    wb = wl.Workload("block", pb, dict(wl.DEFAULT_PARAMS), np.zeros(tb))
    for f in range(NF):
        v = 0.02 * rng.normal(size=(M, M, M))
        if f in (wl.F_W, wl.F_G, wl.F_G + 3, wl.F_G + 5, wl.F_ALP):
            v += 1.0
        wb.active_view(wb.state, 0, f)[...] = v
    ub = wb.state.copy()
    orc.fill_ghosts(pb, ub)
    ref = orc.z4c_rhs(pb, wb.params, ub)
    # the block on the GPU, against the oracle
    d_ub = torch.from_numpy(ub).cuda()
    d_rb = torch.zeros_like(d_ub)
    sacra.z4c_rhs(pb, wb.params, d_ub, d_rb)
    rb = d_rb.cpu().numpy()
    assert not parity_report(wb, rb, ref)
    # the big patch: every field is the block repeated 15 x 15 x 15
    u = torch.zeros(total, dtype=torch.float64, device="cuda")
    shape = (p.nz + 2 * NG, p.ny + 2 * NG, p.pitch_x)

    def field(t, f):
        o = p.patch_offset + f * p.field_stride
        return t[o:o + shape[0] * shape[1] * shape[2]].view(shape)[NG:-NG, NG:-NG, NG:NG + n]

    for f in range(NF):
        blk = torch.from_numpy(np.ascontiguousarray(wb.active_view(wb.state, 0, f))).cuda()
        field(u, f).copy_(blk.repeat(REP, REP, REP))
    sacra.fill_ghosts(ps, u)
    rhs = torch.full((total,), float("nan"), dtype=torch.float64, device="cuda")
    sacra.z4c_rhs(ps, wb.params, u, rhs)
    torch.cuda.synchronize()
    for f in range(NF):
        want = torch.from_numpy(np.ascontiguousarray(wb.active_view(rb, 0, f))).cuda()
        got = field(rhs, f).reshape(REP, M, REP, M, REP, M)
        assert bool((got == want.view(1, M, 1, M, 1, M)).all()), wl.FIELD_NAMES[f]
    # and nothing was written outside the active cells of the 25 fields
    assert int(torch.isnan(rhs).sum()) == total - NF * n ** 3


def test_rk4_step_on_a_480_cubed_patch_is_the_tiling_of_the_block_step():
    """the same for a whole RK4 step (four states of 23 GB): halo fills, all four substage kernels with their RK rings
    and the stage-4 aliasing u_out = u_n at offsets beyond 2^31 elements"""
    rep = 12
    n = M * rep
    ps, total = wl.make_layout([(n, n, n)], [0.1], [0.025], [(0, 0, 0)])
    _release()
    free, _ = torch.cuda.mem_get_info()
    _need(free, 4 * total * 8 + (4 << 30), "the 480^3 RK4 step")
    assert total > 2 ** 31
    p = ps[0]
    rng = np.random.default_rng(13)
    pb, tb = wl.make_layout([(M, M, M)], [0.1], [0.025], [(0, 0, 0)])
    wb = wl.Workload("block", pb, dict(wl.DEFAULT_PARAMS), np.zeros(tb))
    for f in range(NF):
        v = 0.02 * rng.normal(size=(M, M, M))
        if f in (wl.F_W, wl.F_G, wl.F_G + 3, wl.F_G + 5, wl.F_ALP):
            v += 1.0
        wb.active_view(wb.state, 0, f)[...] = v
    d_ub = torch.from_numpy(wb.state).cuda()
    d_wb = torch.zeros(3 * tb, dtype=torch.float64, device="cuda")
    sacra.rk4_step(pb, wb.params, d_ub, d_wb)
    ub, Sb = d_ub.cpu().numpy(), d_wb[2 * tb:].cpu().numpy()
    # the block step on the GPU, against the oracle (north_star tolerance on S, dt times it on the new state)
    ref = wb.state.copy()
    S_ref = orc.rk4_step(pb, wb.params, ref)
    assert not parity_report(wb, Sb, S_ref)
    for f in range(NF):
        s = np.max(np.abs(wb.active_view(S_ref, 0, f)))
        a, b = wb.active_view(ub, 0, f), wb.active_view(ref, 0, f)
        assert np.all(np.abs(a - b) <= pb[0].dt * 1e-11 * (s + 1e-14) + np.spacing(np.abs(b))), wl.FIELD_NAMES[f]
    u = torch.zeros(total, dtype=torch.float64, device="cuda")
    work = torch.zeros(3 * total, dtype=torch.float64, device="cuda")
    shape = (p.nz + 2 * NG, p.ny + 2 * NG, p.pitch_x)

    def field(t, f):
        o = p.patch_offset + f * p.field_stride
        return t[o:o + shape[0] * shape[1] * shape[2]].view(shape)[NG:-NG, NG:-NG, NG:NG + n]

    for f in range(NF):
        blk = torch.from_numpy(np.ascontiguousarray(wb.active_view(wb.state, 0, f))).cuda()
        field(u, f).copy_(blk.repeat(rep, rep, rep))
    sacra.rk4_step(ps, wb.params, u, work, total)
    torch.cuda.synchronize()
    S = work[2 * total:]
    for f in range(NF):
        for big, small in ((u, ub), (S, Sb)):
            want = torch.from_numpy(np.ascontiguousarray(wb.active_view(small, 0, f))).cuda()
            got = field(big, f).reshape(rep, M, rep, M, rep, M)
            assert bool((got == want.view(1, M, 1, M, 1, M)).all()), wl.FIELD_NAMES[f]
