"""-m gpu: mirror ghost fill (sacra_fill_ghosts_bc) bit-exact against the oracle, and the defining
property through the CUDA path: the half domain with mirror faces reproduces the full periodic problem bit for bit
(right-hand side and a whole RK4 step built from the substage calls)."""
import numpy as np
import pytest
import torch

import orc
from gpu_util import dev, gpu_rhs, gpu_step, host
from helpers import NF, NG
from paper_2607_08743_b200 import sacra
from paper_2607_08743_b200 import workloads as wl
from test_gpu_parity import _ragged_workload
from test_oracle_reflect import _mirror_symmetric_full

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("mode", [(0, 0, 1), (1, 1, 1), (1, 0, 0), (0, 0, 0)])
def test_fill_bc_bit_exact_ragged_batch(mode):
    w = _ragged_workload()
    ref = orc.fill_ghosts_bc(w.patches, mode, w.state.copy())
    u = dev(w.state)
    sacra.fill_ghosts_bc(w.patches, mode, u)
    assert np.array_equal(host(u), ref)        # includes: padding and inter-patch gaps untouched


def test_half_domain_with_mirror_faces_equals_full_periodic_step_on_gpu():
    n, nz2 = 16, 24
    full = _mirror_symmetric_full(n, nz2, 7)
    half = nz2 // 2
    ps, total = wl.make_layout([(n, n, half)], [0.1], [0.025], [(0, 0, 0)])
    h = wl.Workload("half", ps, dict(full.params), np.zeros(total))
    for f in range(NF):
        h.active_view(h.state, 0, f)[...] = full.active_view(full.state, 0, f)[half:]
    # right-hand side
    uf = full.state.copy(); orc.fill_ghosts(full.patches, uf)
    uh = orc.fill_ghosts_bc(ps, (0, 0, 1), h.state.copy())
    kf, kh = np.nan_to_num(gpu_rhs(full, uf)), np.nan_to_num(gpu_rhs(h, uh))
    for f in range(NF):
        assert np.array_equal(h.active_view(kh, 0, f), full.active_view(kf, 0, f)[half:]), wl.FIELD_NAMES[f]
    # one RK4 step: full domain through sacra_rk4_step, half domain through the substage calls with mirror fills
    got_full, _ = gpu_step(full, full.state)
    u = dev(h.state)
    a, b, acc = torch.zeros_like(u), torch.zeros_like(u), torch.zeros_like(u)
    for stage, (src, dst) in enumerate([(u, a), (a, b), (b, a), (a, u)], start=1):
        sacra.fill_ghosts_bc(ps, (0, 0, 1), src)
        sacra.rk4_substep(ps, h.params, stage, u, src, dst, acc)
    got_half = host(u)
    for f in range(NF):
        assert np.array_equal(h.active_view(got_half, 0, f), full.active_view(got_full, 0, f)[half:]), wl.FIELD_NAMES[f]
