"""-m gpu: the CUDA path (libsacra through the C ABI) against the CPU oracle, element by element on the same
seeded inputs. Tolerance (BASELINE.json north_star): per field max|d| <= 1e-11 (max|ref_field| + 1e-14) on
RHS-like quantities (k of each stage, the RK4 increment S); integer/copy work (ghost fill) bit-exact; the new
state within dt*tol + 1 ulp (reading G in DESIGN.md)."""
import numpy as np
import pytest
import torch

import orc
from gpu_util import dev, gpu_fill, gpu_rhs, gpu_step, host
from helpers import NF, NG, parity_report, pi_partner
from paper_2607_08743_b200 import sacra
from paper_2607_08743_b200 import workloads as wl

pytestmark = pytest.mark.gpu
RTOL, FLOOR = 1e-11, 1e-14


def _assert_parity(w, got, ref, what):
    bad = parity_report(w, got, ref, RTOL, FLOOR)
    assert not bad, "%s: fields outside 1e-11 (name, max|d|, max|ref|, ratio): %s" % (what, bad)


def _assert_state(w, got, ref, S_ref):
    for ip, p in enumerate(w.patches):
        for f in range(NF):
            a, b = w.active_view(got, ip, f), w.active_view(ref, ip, f)
            tol = p.dt * RTOL * (np.max(np.abs(w.active_view(S_ref, ip, f))) + FLOOR) + np.spacing(np.abs(b))
            assert np.all(np.abs(a - b) <= tol), (ip, wl.FIELD_NAMES[f], np.max(np.abs(a - b)))


def _untouched_outside_active(w, buf, poison_is_nan=True):
    """ghosts and padding of an output buffer must still hold the poison"""
    mask = np.ones(buf.size, dtype=bool)
    for ip, p in enumerate(w.patches):
        for f in range(NF):
            o = p.patch_offset + f * p.field_stride
            m = mask[o:o + int(np.prod(p.shape))].reshape(p.shape)
            m[NG:NG + p.nz, NG:NG + p.ny, NG:NG + p.nx] = False
    return np.all(np.isnan(buf[mask]))


# ------------------------------------------------------------------------------------------- ghost fill
RAGGED = [(7, 6, 9), (6, 8, 6), (37, 6, 11), (33, 65, 6)]


def _ragged_workload(seed=5, dims=RAGGED):
    rng = np.random.default_rng(seed)
    hs = [0.1 + 0.05 * i for i in range(len(dims))]
    patches, total = wl.make_layout(dims, hs, [0.25 * h for h in hs], [(0.3, -0.2, 0.1)] * len(dims))
    return wl.Workload("ragged", patches, dict(wl.DEFAULT_PARAMS), rng.normal(size=total))


def test_fill_ghosts_bit_exact_ragged_batch():
    w = _ragged_workload()
    ref = w.state.copy()
    orc.fill_ghosts(w.patches, ref)
    got = gpu_fill(w, w.state)
    assert np.array_equal(got, ref)          # includes: padding and inter-patch gaps untouched


@pytest.mark.parametrize("idx", [0, 1])
def test_fill_ghosts_bit_exact_configs(idx):
    w = wl.make(idx)
    ref = w.state.copy()
    orc.fill_ghosts(w.patches, ref)
    assert np.array_equal(gpu_fill(w, w.state), ref)


# ------------------------------------------------------------------------------------------- RHS
def _smooth_random(w, seed, amp=0.05):
    """generic data: every field non-trivial (shift of both signs, non-unit det, non-zero Theta ...)"""
    rng = np.random.default_rng(seed)
    for ip, p in enumerate(w.patches):
        z, y, x = np.meshgrid(np.arange(p.nz), np.arange(p.ny), np.arange(p.nx), indexing="ij")
        for f in range(NF):
            k = rng.integers(1, 3, size=3)
            ph = rng.uniform(0, 2 * np.pi, size=3)
            v = amp * np.sin(2 * np.pi * k[0] * x / p.nx + ph[0]) * np.sin(2 * np.pi * k[1] * y / p.ny + ph[1]) * \
                np.sin(2 * np.pi * k[2] * z / p.nz + ph[2])
            if f in (wl.F_W, wl.F_G, wl.F_G + 3, wl.F_G + 5, wl.F_ALP):
                v = v + 1.0
            w.active_view(w.state, ip, f)[...] = v + rng.uniform(-1e-3, 1e-3, size=v.shape)
    return w


def test_rhs_parity_generic_data_ragged_batch():
    """all 25 fields active, shift of both signs (both upwind branches), ragged sizes, several patches"""
    w = _smooth_random(_ragged_workload(dims=[(37, 9, 11), (6, 6, 6), (16, 33, 7)]), 11)
    u = w.state.copy()
    orc.fill_ghosts(w.patches, u)
    ref = orc.z4c_rhs(w.patches, w.params, u)
    got = gpu_rhs(w, u)
    assert _untouched_outside_active(w, got)
    got = np.nan_to_num(got, nan=0.0)
    _assert_parity(w, got, ref, "rhs generic")


def test_rhs_parity_lapse_switch_and_kappa2():
    """reading C switch (lapse_uses_khat=0) and kappa2 != 0 reach the kernel"""
    w = _smooth_random(_ragged_workload(dims=[(12, 10, 8)]), 12)
    w.params.update(kappa2=0.3, lapse_uses_khat=0, eta=1.3, shift_coef=0.6, ko_sigma=0.25, kappa1=0.07)
    u = w.state.copy()
    orc.fill_ghosts(w.patches, u)
    ref = orc.z4c_rhs(w.patches, w.params, u)
    got = np.nan_to_num(gpu_rhs(w, u), nan=0.0)
    _assert_parity(w, got, ref, "rhs params")
    w.params.update(lapse_uses_khat=1)
    ref1 = orc.z4c_rhs(w.patches, w.params, u)
    assert not np.array_equal(ref, ref1)
    _assert_parity(w, np.nan_to_num(gpu_rhs(w, u), nan=0.0), ref1, "rhs params khat")


@pytest.mark.parametrize("idx", [0, 1, 2])
def test_rhs_parity_configs(idx):
    w = wl.make(idx)
    u = w.state.copy()
    orc.fill_ghosts(w.patches, u)
    ref = orc.z4c_rhs(w.patches, w.params, u)
    got = np.nan_to_num(gpu_rhs(w, u), nan=0.0)
    _assert_parity(w, got, ref, w.name)


def test_minkowski_exact_zero_on_gpu():
    ps, total = wl.make_layout([(20, 9, 7)], [0.1], [0.025], [(0, 0, 0)])
    w = wl.Workload("flat", ps, dict(wl.DEFAULT_PARAMS), np.zeros(total))
    for f in range(NF):
        w.active_view(w.state, 0, f)[...] = 1.0 if f in (wl.F_W, wl.F_G, wl.F_G + 3, wl.F_G + 5, wl.F_ALP) else 0.0
    u = gpu_fill(w, w.state)
    got = gpu_rhs(w, u, poison=7.0)
    for f in range(NF):
        assert np.all(w.active_view(got, 0, f) == 0.0)


# ------------------------------------------------------------------------------------------- RK4
@pytest.mark.parametrize("idx", [0, 1, 2, 3])
def test_rk4_step_parity_configs(idx):
    w = wl.make(idx)
    ref = w.state.copy()
    S_ref = orc.rk4_step(w.patches, w.params, ref)
    got, S = gpu_step(w, w.state)
    _assert_parity(w, S, S_ref, w.name + " increment S")
    _assert_state(w, got, ref, S_ref)
    # ghosts of the result are filled
    chk = got.copy()
    orc.fill_ghosts(w.patches, chk)
    assert np.array_equal(chk, got)


def test_rk4_step_equals_nine_call_sequence_bitwise():
    w = _smooth_random(_ragged_workload(dims=[(13, 8, 9), (8, 8, 8)]), 21, amp=0.02)
    got, S = gpu_step(w, w.state)
    u = dev(w.state)
    a, b, acc = torch.zeros_like(u), torch.zeros_like(u), torch.zeros_like(u)
    seq = [(u, a), (a, b), (b, a), (a, u)]
    for stage, (src, dst) in enumerate(seq, start=1):
        sacra.fill_ghosts(w.patches, src)
        sacra.rk4_substep(w.patches, w.params, stage, u, src, dst, acc)
    sacra.fill_ghosts(w.patches, u)
    assert np.array_equal(host(u), got)
    assert np.array_equal(host(acc), S)


def test_substep_stage_table_against_oracle():
    """each stage's u_out and acc, on generic data, against the oracle's substep (item 11 table)"""
    w = _smooth_random(_ragged_workload(dims=[(9, 14, 8)]), 22, amp=0.02)
    ps, prm = w.patches, w.params
    un = w.state.copy(); orc.fill_ghosts(ps, un)
    uin = un.copy()
    acc_ref = np.zeros_like(un)
    acc_gpu = torch.zeros(un.size, dtype=torch.float64, device="cuda")
    for stage in (1, 2, 3, 4):
        out_ref = np.zeros_like(un)
        k_ref = orc.z4c_rhs(ps, prm, uin)
        orc.rk4_substep(ps, prm, stage, un, uin, out_ref, acc_ref)
        out_gpu = torch.zeros_like(acc_gpu)
        acc_in = acc_ref.copy()
        d_un = dev(un)      # stage 1 takes u_n from the stage input: the same buffer
        sacra.rk4_substep(ps, prm, stage, d_un, d_un if stage == 1 else dev(uin), out_gpu, acc_gpu)
        _assert_parity(w, host(acc_gpu), acc_ref, "acc stage %d" % stage)
        _assert_state(w, host(out_gpu), out_ref, k_ref)
        # next stage input: oracle's own (keeps the comparison stage-local)
        uin = out_ref.copy(); orc.fill_ghosts(ps, uin)
        acc_gpu = dev(acc_ref)


def test_substep_leaves_ghosts_and_padding_untouched():
    """sacra.h: u_out and acc are written on active cells only (ragged sizes incl. the minimum 6^3)"""
    w = _smooth_random(_ragged_workload(dims=[(37, 9, 11), (6, 6, 6), (16, 33, 7)]), 31, amp=0.02)
    ps, prm = w.patches, w.params
    un = w.state.copy(); orc.fill_ghosts(ps, un)
    for stage in (1, 4):
        out = torch.full((un.size,), float("nan"), dtype=torch.float64, device="cuda")
        acc = torch.full((un.size,), 0.5, dtype=torch.float64, device="cuda")
        d_un = dev(un)
        sacra.rk4_substep(ps, prm, stage, d_un, d_un, out, acc)
        assert _untouched_outside_active(w, host(out))
        acc_h, out_h = host(acc), host(out)
        for ip in range(len(ps)):
            for f in range(NF):
                assert not np.any(np.isnan(w.active_view(out_h, ip, f)))
                w.active_view(acc_h, ip, f)[...] = 0.5
        assert np.all(acc_h == 0.5), "acc written outside the active cells (stage %d)" % stage


def test_more_patches_than_one_launch_carries():
    dims = [(6 + (q % 3), 6, 6 + (q % 2)) for q in range(19)]
    w = _smooth_random(_ragged_workload(dims=dims), 23, amp=0.02)
    ref = w.state.copy()
    S_ref = orc.rk4_step(w.patches, w.params, ref)
    got, S = gpu_step(w, w.state)
    _assert_parity(w, S, S_ref, "19 patches")


# ------------------------------------------------------------------------------------------- pi symmetry
def test_pi_symmetry_bitwise_on_gpu():
    """max abs pair difference exactly zero, for k1 and for the state after one step."""
    w = wl.make(2, n=64, half_width=8.0)
    u = gpu_fill(w, w.state)
    k1 = np.nan_to_num(gpu_rhs(w, u), nan=0.0)
    new, S = gpu_step(w, w.state)
    for name, buf in (("k1", k1), ("S", S), ("state", new)):
        for f in range(NF):
            a = w.active_view(buf, 0, f)
            assert np.max(np.abs(a - wl.PI_SIGN[f] * pi_partner(a))) == 0.0, (name, wl.FIELD_NAMES[f])
    assert np.max(np.abs(w.active_view(k1, 0, wl.F_W))) > 0


def test_pi_symmetry_with_shift_of_both_signs():
    """symmetrised generic data with beta != 0: partners take opposite upwind branches (item 13)"""
    n = 16
    ps, total = wl.make_layout([(n, n, n)], [0.2], [0.05], [(0, 0, 0)])
    w = _smooth_random(wl.Workload("sym", ps, dict(wl.DEFAULT_PARAMS), np.zeros(total)), 31, amp=0.03)
    for f in range(NF):
        a = w.active_view(w.state, 0, f)
        a[...] = 0.5 * (a + wl.PI_SIGN[f] * pi_partner(a))       # exact: halving and the sign are exact
        assert np.array_equal(a, wl.PI_SIGN[f] * pi_partner(a))
    u = gpu_fill(w, w.state)
    k1 = np.nan_to_num(gpu_rhs(w, u), nan=0.0)
    ref = orc.z4c_rhs(w.patches, w.params, u)
    _assert_parity(w, k1, ref, "sym generic")
    for f in range(NF):
        a = w.active_view(k1, 0, f)
        assert np.max(np.abs(a - wl.PI_SIGN[f] * pi_partner(a))) == 0.0, wl.FIELD_NAMES[f]
    assert np.min(w.active_view(u, 0, wl.F_BET)) < 0 < np.max(w.active_view(u, 0, wl.F_BET))


# ------------------------------------------------------------------------------------------- full size
def test_full_size_config4_sampled_blocks_against_oracle():
    """BASELINE.json configs[4] (256^3) in the launch configuration bench.py times (one sacra_rk4_step call on the
    whole patch). The oracle cannot do 256^3 in seconds, so it recomputes SAMPLED blocks: one RK4 step has a
    domain of dependence of 4 stages x 3 cells, so the 8^3 centre of a 32^3 periodic sub-patch cut out of the
    same data (with wrap-around) is exact. Blocks: the two punctures, the domain corner (periodic wrap), a face,
    and seeded random places. Increment S and new state, same tolerances as everywhere."""
    w = wl.make(4)
    p = w.patches[0]
    got, S = gpu_step(w, w.state)
    rng = np.random.default_rng(404)
    m, core, mar = 32, 8, 12
    c = p.nx // 2
    centres = [(c, c, c + 20), (c, c, c - 20), (0, 0, 0), (c, 3, c), (p.nz - 2, c, 5)]
    centres += [tuple(int(v) for v in rng.integers(0, p.nx, size=3)) for _ in range(3)]
    # pass 1: the oracle on every block. The tolerance scales with max|S_f| over the WHOLE field, which the
    # oracle cannot afford; the maximum over the valid interiors of all sampled blocks (the puncture blocks
    # dominate) is a lower bound of it computed by the oracle alone, so the test is stricter than required.
    blocks = []
    for (kz, jy, ix) in centres:
        ps, total = wl.make_layout([(m, m, m)], [p.dx], [p.dt], [(0.0, 0.0, 0.0)])
        s = wl.Workload("block", ps, dict(w.params), np.zeros(total))
        zi = (np.arange(m) + kz - m // 2) % p.nz
        yi = (np.arange(m) + jy - m // 2) % p.ny
        xi = (np.arange(m) + ix - m // 2) % p.nx
        for f in range(NF):
            s.active_view(s.state, 0, f)[...] = w.active_view(w.state, 0, f)[np.ix_(zi, yi, xi)]
        ref = s.state.copy()
        S_ref = orc.rk4_step(s.patches, s.params, ref)
        blocks.append((s, ref, S_ref, zi, yi, xi))
    sl = slice(mar, mar + core)
    scale = [max(np.max(np.abs(b[0].active_view(b[2], 0, f)[mar:-mar, mar:-mar, mar:-mar])) for b in blocks)
             for f in range(NF)]
    # pass 2: element by element on the exact 8^3 cores
    for (s, ref, S_ref, zi, yi, xi), ctr in zip(blocks, centres):
        for f in range(NF):
            sub = np.ix_(zi[sl], yi[sl], xi[sl])
            a = w.active_view(S, 0, f)[sub]
            b = s.active_view(S_ref, 0, f)[sl, sl, sl]
            assert np.max(np.abs(a - b)) <= RTOL * (scale[f] + FLOOR), (wl.FIELD_NAMES[f], ctr)
            un = w.active_view(got, 0, f)[sub]
            ur = s.active_view(ref, 0, f)[sl, sl, sl]
            assert np.all(np.abs(un - ur) <= p.dt * RTOL * (scale[f] + FLOOR) + np.spacing(np.abs(ur))), \
                (wl.FIELD_NAMES[f], ctr)


def test_rhs_parity_unpadded_pitch():
    """pitch_x == nx + 6 exactly (nx + 6 a multiple of 8): the tensor maps then address one element more than a row
    holds (the first cell of the next row), which the boxes never use"""
    dims = [(10, 10, 10), (42, 6, 6), (26, 7, 9)]
    ps, total = wl.make_layout(dims, [0.1] * 3, [0.025] * 3, [(0, 0, 0)] * 3)
    assert all(p.pitch_x == p.nx + 2 * NG for p in ps)
    w = _smooth_random(wl.Workload("unpadded", ps, dict(wl.DEFAULT_PARAMS), np.zeros(total)), 3)
    u = w.state.copy()
    orc.fill_ghosts(ps, u)
    ref = orc.z4c_rhs(ps, w.params, u)
    got = gpu_rhs(w, u)
    assert _untouched_outside_active(w, got)
    _assert_parity(w, np.nan_to_num(got), ref, "unpadded pitch")
