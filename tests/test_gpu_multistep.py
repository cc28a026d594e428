"""-m gpu: consecutive RK4 steps of the CUDA path beside the CPU oracle (BASELINE.json configs[4]: "ten consecutive
RK4 steps"), the constraint-norm trajectory, the full 256^3 step on ALL points, and the SACRA_FLAG_SKIP_INCREMENT path.

Tolerance over several steps (derived). One step is held to the north_star tolerance
max|dS_f| <= 1e-11 (max|S_f| + 1e-14). Over k steps two things add up:
  (1) the per-step differences accumulate linearly in the state: k dt 1e-11 (max|S_f| + 1e-14) + 1 ulp;
  (2) round-off level differences of the STATE are amplified by the right-hand side: a last-bit flip of an O(1) field
      (gt_ij, W, alpha) enters the Ricci tensor through a second difference, 16 ulp(1) / (12 h^2) ~ 1e3 ulp for h = 1/32.
      Neither implementation can avoid that; its size is measured by the oracle alone: a second oracle trajectory
      started from the same data with every value moved by one unit in the last place (seeded sign) -- the "last-bit
      envelope" env_k(f) = max|u_B - u_A| after k steps.
The CUDA trajectory must stay within (1) + 4 env_k(f) of the oracle's, per field and step. On config 0 the exact
trajectory (the oracle in __float128 arithmetic, state rounded to double after every step) referees: the CUDA state is
as close to it as the double oracle is, within the same bound."""
import numpy as np
import pytest
import torch

import orc
from gpu_util import dev, gpu_step, host
from helpers import NF, NG
from paper_2607_08743_b200 import sacra
from paper_2607_08743_b200 import workloads as wl

pytestmark = pytest.mark.gpu
RTOL, FLOOR = 1e-11, 1e-14


def _last_bit_perturbed(w, seed):
    rng = np.random.default_rng(seed)
    s = w.state.copy()
    for ip in range(len(w.patches)):
        for f in range(NF):
            a = w.active_view(s, ip, f)
            a += np.where(rng.integers(0, 2, size=a.shape) == 1, 1.0, -1.0) * np.spacing(np.abs(a))
    return s


def _gpu_norms(w, u, con, scratch, norms):
    sacra.constraints(w.patches, u, con)
    sacra.constraint_norms(w.patches, con, scratch, norms)
    return host(norms).copy()


@pytest.mark.parametrize("idx,nsteps,quad_steps", [(0, 10, 3), (1, 10, 0), (4, 3, 0)])
def test_ten_consecutive_steps_beside_the_oracle(idx, nsteps, quad_steps):
    """configs 0 and 1: ten steps. Config 4 (256^3, the timed workload): three consecutive steps on ALL points, the
    most the two oracle trajectories allow within a minute of host time; no constraint norms there (the step-by-step
    state comparison covers every field the norms are made of)."""
    w = wl.make(idx)
    ps, prm = w.patches, w.params
    n = w.state.size
    uA, uB = w.state.copy(), _last_bit_perturbed(w, 99 + idx)
    uQ = w.state.copy()
    u = dev(w.state)
    work = torch.zeros(3 * n, dtype=torch.float64, device="cuda")
    con = torch.zeros(n, dtype=torch.float64, device="cuda")
    scratch = torch.zeros(sacra.constraint_scratch_doubles(ps), dtype=torch.float64, device="cuda")
    norms = torch.zeros(4, dtype=torch.float64, device="cuda")
    scale = np.zeros(NF)
    worst = 0.0
    for k in range(1, nsteps + 1):
        S = orc.rk4_step(ps, prm, uA)
        orc.rk4_step(ps, prm, uB)
        sacra.rk4_step(ps, prm, u, work)
        got = host(u)
        assert np.all(np.isfinite(got))
        if k <= quad_steps:
            orc.rk4_step(ps, prm, uQ, quad=True)
        for f in range(NF):
            scale[f] = max(scale[f], max(np.max(np.abs(w.active_view(S, ip, f))) for ip in range(len(ps))))
        for ip, p in enumerate(ps):
            for f in range(NF):
                a, b, c = (w.active_view(x, ip, f) for x in (got, uA, uB))
                env = np.max(np.abs(c - b))
                bound = k * p.dt * RTOL * (scale[f] + FLOOR) + np.spacing(np.max(np.abs(b))) + 4.0 * env
                d = np.max(np.abs(a - b))
                assert d <= bound, (w.name, "step", k, wl.FIELD_NAMES[f], d, bound, env)
                worst = max(worst, d / bound)
                if k <= quad_steps:
                    q = w.active_view(uQ, ip, f)
                    assert np.max(np.abs(a - q)) <= bound + np.max(np.abs(b - q)), (w.name, "quad", k, wl.FIELD_NAMES[f])
        if idx == 4:
            continue
        # constraint monitor on the evolved state: the CUDA norms of the CUDA state against the oracle's norms of its own
        ng = _gpu_norms(w, u, con, scratch, norms)
        no = orc.constraint_norms(ps, orc.constraints(ps, uA))
        nb = orc.constraint_norms(ps, orc.constraints(ps, uB))
        for c in range(4):
            tol = 1e-9 * abs(no[c]) + 4.0 * abs(nb[c] - no[c]) + 1e-15
            assert abs(ng[c] - no[c]) <= tol, (w.name, "norm", k, c, ng[c], no[c], tol)
    assert worst > 0.0 or idx == 0
    print("\n[tolerance use] %s, %d steps: worst max|d| / bound = %.3f" % (w.name, nsteps, worst))


def test_skip_increment_flag_gives_the_same_state_bitwise():
    w = wl.make(1, n=24)
    got, S = gpu_step(w, w.state)
    u = dev(w.state)
    n = u.numel()
    work = torch.full((3 * n,), 7.0, dtype=torch.float64, device="cuda")
    prm = dict(w.params, flags=sacra.FLAG_SKIP_INCREMENT)
    sacra.rk4_step(w.patches, prm, u, work)
    assert np.array_equal(host(u), got)
    # the increment is NOT what acc holds now: it still carries k1 + 2 k2 + 2 k3 of the third stage
    acc = host(work[2 * n:])
    f = wl.F_W
    assert not np.array_equal(w.active_view(acc, 0, f), w.active_view(S, 0, f))


def test_full_size_config4_all_points_against_oracle():
    """BASELINE.json configs[4] (256^3) in the launch configuration bench.py times -- one sacra_rk4_step call on the
    whole patch -- against one oracle step of the WHOLE patch: all 16.8 M points x 25 fields of the increment S and
    of the new state (the oracle takes ~10 s on 16 host cores and ~25 GB of host memory). Falls back to nothing: if
    the host cannot hold the oracle's buffers the test fails, and test_full_size_config4_sampled_blocks... in
    test_gpu_parity.py remains as the sampled version."""
    w = wl.make(4)
    p = w.patches[0]
    got, S = gpu_step(w, w.state)
    ref = w.state.copy()
    S_ref = orc.rk4_step(w.patches, w.params, ref)
    bad = []
    for f in range(NF):
        a, b = w.active_view(S, 0, f), w.active_view(S_ref, 0, f)
        s = np.max(np.abs(b))
        d = np.max(np.abs(a - b))
        if not d <= RTOL * (s + FLOOR):
            bad.append((wl.FIELD_NAMES[f], d, s))
        un, ur = w.active_view(got, 0, f), w.active_view(ref, 0, f)
        assert np.all(np.abs(un - ur) <= p.dt * RTOL * (s + FLOOR) + np.spacing(np.abs(ur))), wl.FIELD_NAMES[f]
    assert not bad, bad
    chk = got.copy()
    orc.fill_ghosts(w.patches, chk)
    assert np.array_equal(chk, got)          # ghosts of the result are filled
    # the step bench.py TIMES sets SACRA_FLAG_SKIP_INCREMENT (stage 4 is k_z4c<5>, not <4>): same size, same launch
    # shape, and the new state must be the one just checked, bit for bit, ghosts and padding included
    u = dev(w.state)
    n = u.numel()
    work = torch.zeros(3 * n, dtype=torch.float64, device="cuda")
    sacra.rk4_step(w.patches, dict(w.params, flags=sacra.FLAG_SKIP_INCREMENT), u, work)
    assert np.array_equal(host(u), got)


def test_repeatable_bit_for_bit_with_guard_bands():
    """compute-sanitizer is closed on this GPU pool (profiles/r02_sanitizer.md), so races and stray accesses are looked
    for directly: the state and the work area sit inside NaN guard bands (a read of a guard cell that reached a result
    would poison it, a write would break the band), a ragged multi-patch batch is stepped 12 times from the same input
    with other launches in between, and every run must give the same bits -- a race between the warps of a tile, between
    a TMA refill and a late reader of a ring slot, or on the e arrays shows up as a changed bit."""
    dims = [(37, 9, 11), (6, 6, 6), (16, 33, 7), (50, 13, 19)]
    hs = [0.1, 0.15, 0.2, 0.12]
    ps, total = wl.make_layout(dims, hs, [0.25 * h for h in hs], [(0.3, -0.2, 0.1)] * len(dims))
    rng = np.random.default_rng(77)
    w = wl.Workload("guard", ps, dict(wl.DEFAULT_PARAMS), np.zeros(total))
    for ip, p in enumerate(ps):
        for f in range(NF):
            v = 0.02 * rng.normal(size=(p.nz, p.ny, p.nx))
            if f in (wl.F_W, wl.F_G, wl.F_G + 3, wl.F_G + 5, wl.F_ALP):
                v += 1.0
            w.active_view(w.state, ip, f)[...] = v
    G = 16384                                   # guard band, doubles (a multiple of 2: 16-byte alignment is kept)
    big = torch.full((G + total + G + 3 * total + G,), float("nan"), dtype=torch.float64, device="cuda")
    u, work = big[G:G + total], big[2 * G + total:2 * G + 4 * total]
    first = None
    other = dev(wl.make(0, n=16).state)
    w0 = wl.make(0, n=16)
    for rep in range(12):
        u.copy_(torch.from_numpy(w.state))
        work.zero_()
        sacra.rk4_step(ps, w.params, u, work, total)
        sacra.fill_ghosts(w0.patches, other)    # unrelated launches in between
        res = (host(u).copy(), host(work[2 * total:]).copy())
        assert np.all(np.isfinite(res[0]))
        if first is None:
            first = res
        else:
            assert np.array_equal(res[0], first[0]) and np.array_equal(res[1], first[1]), rep
        bands = host(torch.cat([big[:G], big[G + total:2 * G + total], big[2 * G + 4 * total:]]))
        assert np.all(np.isnan(bands)), rep
    ref = w.state.copy()
    S_ref = orc.rk4_step(ps, w.params, ref)
    for ip in range(len(ps)):
        for f in range(NF):
            s = np.max(np.abs(w.active_view(S_ref, ip, f)))
            assert np.max(np.abs(w.active_view(first[1], ip, f) - w.active_view(S_ref, ip, f))) <= RTOL * (s + FLOOR)
