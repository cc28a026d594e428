"""-m gpu: sacra_constraint_norms_static, the constraint norms for callers that cannot allocate device memory.

Some users of libsacra own no free device memory and may not ask for any while they run: an evolution code that
gave the whole GPU to its own arena at start-up, or a time loop in which a cudaMalloc would synchronise the device
and stall the streams that overlap halo exchange and compute. sacra_constraint_norms needs a scratch buffer from
the caller; sacra_constraint_norms_static keeps its partial sums in a fixed 128 KiB array inside the library instead
(at most SACRA_NORMS_STATIC_MAX_PLANES = 4096 active z-planes over all patches; include/sacra.h has the contract).

What is checked: the new call gives the same four norms as the existing call (same kernels and reduction order, so
bit-equal, which is inside the rtol 1e-11 that tests/test_gpu_constraints.py uses against the oracle), on two calls
in a row with different inputs - the second call finds the first call's partial sums still in the shared array and
must not be disturbed by them - and that a batch beyond the limit is refused before anything is launched.

This file sorts last on purpose (pytest -x stops at the first failure; a failure here must not hide other tests).
It depends on nothing the other tests leave behind and leaves nothing behind: it passes alone in a fresh process
(where its first call is the one that looks the array's address up) and after the rest of the suite."""
import numpy as np
import pytest
import torch

from paper_2607_08743_b200 import sacra
from paper_2607_08743_b200 import workloads as wl

pytestmark = pytest.mark.gpu
RTOL = 1e-11   # the tolerance of tests/test_gpu_constraints.py::test_norms_match_eq22_and_are_deterministic


def _norms_both_ways(w, seed):
    """constraints of a seeded state, then the norms through the caller's scratch and through the library's array"""
    rng = np.random.default_rng(seed)
    state = w.state + 1e-3 * rng.standard_normal(w.state.shape)      # constraint-violating: norms well above round-off
    u = torch.from_numpy(state).cuda()
    sacra.fill_ghosts(w.patches, u)
    con = torch.full_like(u, float("nan"))
    sacra.constraints(w.patches, u, con)
    scratch = torch.zeros(sacra.constraint_scratch_doubles(w.patches), dtype=torch.float64, device="cuda")
    want = torch.zeros(4, dtype=torch.float64, device="cuda")
    sacra.constraint_norms(w.patches, con, scratch, want)
    got = torch.full((4,), float("nan"), dtype=torch.float64, device="cuda")
    free_before = torch.cuda.mem_get_info()[0]
    sacra.constraint_norms_static(w.patches, con, got)
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    return got.cpu().numpy(), want.cpu().numpy(), free_before - free_after


def test_static_scratch_norms_equal_the_existing_path_on_two_calls_in_a_row():
    # first call: a batch of 8 patches (128 planes fill the low part of the shared array) ...
    w_big = wl.config3(n=16)
    got1, want1, _ = _norms_both_ways(w_big, 1)
    # ... second call: one small patch, which finds the first call's sums in the array and must ignore them
    w_small = wl.config0(n=16)
    got2, want2, grew = _norms_both_ways(w_small, 2)
    for got, want in ((got1, want1), (got2, want2)):
        assert np.all(np.isfinite(want)) and np.all(want > 0.0), want
        assert np.allclose(got, want, rtol=RTOL, atol=0.0), (got, want)
        assert np.array_equal(got, want), (got, want)                 # same kernels, same order: same bits
    assert not np.array_equal(got1, got2)                             # the two calls really had different answers
    assert grew < (1 << 20), "the call took %d bytes of device memory" % grew   # second call: set-up is long done


def test_static_scratch_refuses_batches_beyond_its_capacity():
    nz = sacra.NORMS_STATIC_MAX_PLANES + 6
    ps, total = wl.make_layout([(6, 6, nz)], [0.125], [0.03125], [(0, 0, 0)])
    con = torch.zeros(total, dtype=torch.float64, device="cuda")
    norms = torch.full((4,), -1.0, dtype=torch.float64, device="cuda")
    with pytest.raises(sacra.SacraError) as e:
        sacra.constraint_norms_static(ps, con, norms)
    assert e.value.code == sacra.ERR_TOOLARGE and "capacity" in str(e.value)
    torch.cuda.synchronize()
    assert np.array_equal(norms.cpu().numpy(), np.full(4, -1.0))      # nothing was launched
    # the largest batch that fits is accepted
    ps, total = wl.make_layout([(6, 6, sacra.NORMS_STATIC_MAX_PLANES)], [0.125], [0.03125], [(0, 0, 0)])
    con = torch.ones(total, dtype=torch.float64, device="cuda")
    sacra.constraint_norms_static(ps, con, norms)
    torch.cuda.synchronize()
    assert np.array_equal(norms.cpu().numpy(), np.ones(4))            # every C = 1, dx a power of two: the norm is 1 exactly
