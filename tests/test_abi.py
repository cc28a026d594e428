"""C ABI of libsacra (include/sacra.h): the library loads, exports every declared symbol, and rejects bad
arguments before touching the GPU (SURVEY 8(b) error list). No compute calls: runs without a device."""
import ctypes as C
import os
import re

import pytest

from paper_2607_08743_b200 import sacra
from paper_2607_08743_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
FAKE = 0x10000  # a non-null, 16-byte aligned "device pointer"; validation must fail before any launch


def _declared():
    txt = open(os.path.join(ROOT, "include", "sacra.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(sacra_[a-z0-9_]+)\s*\(", txt)))


def test_library_exports_every_declared_symbol():
    names = _declared()
    assert set(names) >= {"sacra_fill_ghosts", "sacra_z4c_rhs", "sacra_rk4_substep", "sacra_rk4_step",
                          "sacra_strerror"}
    lib = C.CDLL(sacra.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), n
    assert set(sacra.EXPORTS) == set(names)


def test_struct_layout_matches_header():
    assert C.sizeof(sacra.SacraPatch) == 4 * 4 + 3 * 8 + 2 * 8
    assert C.sizeof(sacra.SacraParams) == 5 * 8 + 2 * 4
    assert sacra.version()


def test_strerror_covers_every_code():
    seen = {sacra.strerror(c) for c in range(0, -7, -1)}
    assert len(seen) == 7 and sacra.strerror(-99) not in seen


def test_static_norms_capacity_is_checked_before_the_device_is_touched():
    """sacra_constraint_norms_static (for callers that cannot allocate): more active z-planes than its fixed array
    holds is SACRA_ERR_TOOLARGE, decided on the host, so it is testable without a GPU"""
    hdr = open(os.path.join(ROOT, "include", "sacra.h")).read()
    assert int(re.search(r"#define SACRA_NORMS_STATIC_MAX_PLANES (\d+)", hdr).group(1)) == sacra.NORMS_STATIC_MAX_PLANES
    ps, _ = wl.make_layout([(6, 6, sacra.NORMS_STATIC_MAX_PLANES + 1)], [0.1], [0.025], [(0, 0, 0)])
    assert _code(sacra.constraint_norms_static, ps, FAKE, FAKE) == sacra.ERR_TOOLARGE
    ps, _ = wl.make_layout([(6, 6, 2048)] * 3, [0.1] * 3, [0.025] * 3, [(0, 0, 0)] * 3)
    assert _code(sacra.constraint_norms_static, ps, FAKE, FAKE) == sacra.ERR_TOOLARGE
    assert _code(sacra.constraint_norms_static, ps, None, FAKE) == sacra.ERR_NULL


def _patch(**kw):
    ps, total = wl.make_layout([(8, 8, 8)], [0.1], [0.025], [(0, 0, 0)])
    p = ps[0]
    for k, v in kw.items():
        setattr(p, k, v)
    return [p], total


def _code(fn, *a):
    with pytest.raises(sacra.SacraError) as e:
        fn(*a, stream=0)
    return e.value.code


PRM = dict(wl.DEFAULT_PARAMS)


def test_null_pointers():
    ps, _ = _patch()
    assert _code(sacra.fill_ghosts, ps, None) == sacra.ERR_NULL
    assert _code(sacra.fill_ghosts, None, FAKE) == sacra.ERR_NULL
    assert _code(sacra.z4c_rhs, ps, None, FAKE, FAKE + 64) == sacra.ERR_NULL
    assert _code(sacra.z4c_rhs, ps, PRM, None, FAKE) == sacra.ERR_NULL
    assert _code(sacra.rk4_substep, ps, PRM, 1, FAKE, FAKE, None, FAKE + 64) == sacra.ERR_NULL
    assert _code(sacra.rk4_step, ps, PRM, FAKE, None, 1024) == sacra.ERR_NULL


def test_bad_arguments():
    assert _code(sacra.fill_ghosts, _patch(ng=2)[0], FAKE) == sacra.ERR_UNSUPPORTED
    assert _code(sacra.fill_ghosts, _patch(nx=5)[0], FAKE) == sacra.ERR_BADARG
    assert _code(sacra.fill_ghosts, _patch(dx=0.0)[0], FAKE) == sacra.ERR_BADARG
    assert _code(sacra.fill_ghosts, _patch(dx=float("nan"))[0], FAKE) == sacra.ERR_BADARG
    assert _code(sacra.fill_ghosts, _patch(pitch_x=12)[0], FAKE) == sacra.ERR_BADARG      # < nx+6
    assert _code(sacra.fill_ghosts, _patch(field_stride=100)[0], FAKE) == sacra.ERR_BADARG
    assert _code(sacra.fill_ghosts, _patch(patch_offset=-3)[0], FAKE) == sacra.ERR_BADARG
    assert _code(sacra.fill_ghosts, [], FAKE) == sacra.ERR_BADARG                          # npatch < 1
    ps, total = _patch()
    for stage in (0, 5, -1):
        assert _code(sacra.rk4_substep, ps, PRM, stage, FAKE, FAKE + 64, FAKE + 128, FAKE + 192) == sacra.ERR_BADARG
    # forbidden aliasing: u_out == u_in, acc == anything, rhs == u
    assert _code(sacra.rk4_substep, ps, PRM, 2, FAKE, FAKE + 64, FAKE + 64, FAKE + 192) == sacra.ERR_BADARG
    assert _code(sacra.rk4_substep, ps, PRM, 2, FAKE, FAKE + 64, FAKE + 128, FAKE) == sacra.ERR_BADARG
    assert _code(sacra.z4c_rhs, ps, PRM, FAKE, FAKE) == sacra.ERR_BADARG
    # state too small for the patch
    assert _code(sacra.rk4_step, ps, PRM, FAKE, FAKE + 64, 1000) == sacra.ERR_BADARG


def test_alignment():
    ps, _ = _patch()
    assert _code(sacra.fill_ghosts, ps, FAKE + 8) == sacra.ERR_ALIGN
    assert _code(sacra.fill_ghosts, _patch(pitch_x=15)[0], FAKE) == sacra.ERR_ALIGN
    assert _code(sacra.fill_ghosts, _patch(patch_offset=4)[0], FAKE) == sacra.ERR_ALIGN    # offset+ng odd
    assert _code(sacra.z4c_rhs, ps, PRM, FAKE, FAKE + 8) == sacra.ERR_ALIGN


def test_constraint_monitor_and_bc_fill_argument_checks():
    ps, _ = _patch()
    assert _code(sacra.constraints, ps, None, FAKE) == sacra.ERR_NULL
    assert _code(sacra.constraints, ps, FAKE, FAKE) == sacra.ERR_BADARG            # con aliases u
    assert _code(sacra.constraints, ps, FAKE, FAKE + 8) == sacra.ERR_ALIGN
    assert _code(sacra.constraints, _patch(ng=2)[0], FAKE, FAKE + 64) == sacra.ERR_UNSUPPORTED
    assert _code(sacra.constraint_norms, ps, FAKE, None, FAKE + 64) == sacra.ERR_NULL
    assert _code(sacra.constraint_norms, ps, FAKE + 8, FAKE, FAKE + 64) == sacra.ERR_ALIGN
    assert sacra.constraint_scratch_doubles(ps) == 4 * 8                            # 4 per active z-plane
    assert _code(sacra.fill_ghosts_bc, ps, (0, 0, 2), FAKE) == sacra.ERR_BADARG     # unknown mode
    assert _code(sacra.fill_ghosts_bc, ps, (0, 0, 1), None) == sacra.ERR_NULL
    assert _code(sacra.fill_ghosts_bc, ps, (0, 1, 1), FAKE + 8) == sacra.ERR_ALIGN


def test_inter_level_argument_checks():
    pp, _ = wl.make_layout([(16, 16, 16)], [0.2], [0.01], [(0, 0, 0)])
    pc, _ = wl.make_layout([(8, 8, 8)], [0.1], [0.005], [(0, 0, 0)])
    odd, _ = wl.make_layout([(7, 8, 8)], [0.1], [0.005], [(0, 0, 0)])
    ok = (4, 4, 4)
    assert _code(sacra.restrict, pp[0], pc[0], ok, None, FAKE) == sacra.ERR_NULL
    assert _code(sacra.restrict, pp[0], pc[0], None, FAKE, FAKE + 64) == sacra.ERR_NULL
    assert _code(sacra.restrict, pp[0], odd[0], ok, FAKE, FAKE + 64) == sacra.ERR_BADARG        # odd child size
    assert _code(sacra.restrict, pp[0], pc[0], (13, 4, 4), FAKE, FAKE + 64) == sacra.ERR_BADARG  # past the parent
    assert _code(sacra.restrict, pp[0], pc[0], (-1, 4, 4), FAKE, FAKE + 64) == sacra.ERR_BADARG
    assert _code(sacra.restrict, pp[0], pc[0], ok, FAKE + 8, FAKE + 64) == sacra.ERR_ALIGN
    assert _code(sacra.prolong_ghosts, pp[0], pc[0], (1, 4, 4), FAKE, FAKE + 64) == sacra.ERR_BADARG   # stencil leaves storage
    assert _code(sacra.prolong_ghosts, pp[0], pc[0], (4, 4, 11), FAKE, FAKE + 64) == sacra.ERR_BADARG
    assert _code(sacra.prolong_ghosts, pp[0], pc[0], ok, FAKE, None) == sacra.ERR_NULL


def test_aliasing_is_checked_on_whole_states():
    """two states are the same buffer where the stage table allows it, or disjoint ranges (sacra.h)"""
    ps, total = _patch()
    far = lambda k: FAKE + 8 * k * (total + 64)            # disjoint states
    near = FAKE + 64                                       # inside the first state: a partial overlap
    assert _code(sacra.z4c_rhs, ps, PRM, FAKE, near) == sacra.ERR_BADARG
    assert _code(sacra.constraints, ps, FAKE, near) == sacra.ERR_BADARG
    # stage 1 takes u_n from the stage input: u_n must be u_in
    assert _code(sacra.rk4_substep, ps, PRM, 1, far(1), FAKE, far(2), far(3)) == sacra.ERR_BADARG
    # partial overlaps of u_out / acc / u_n with anything
    assert _code(sacra.rk4_substep, ps, PRM, 2, FAKE, far(1), far(1) + 64, far(3)) == sacra.ERR_BADARG
    assert _code(sacra.rk4_substep, ps, PRM, 2, FAKE, far(1), far(2), far(2) + 64) == sacra.ERR_BADARG
    assert _code(sacra.rk4_substep, ps, PRM, 2, FAKE, FAKE + 64, far(2), far(3)) == sacra.ERR_BADARG
    assert _code(sacra.rk4_substep, ps, PRM, 3, FAKE, far(1), FAKE + 64, far(3)) == sacra.ERR_BADARG
    # the work area of a step must not contain the state
    assert _code(sacra.rk4_step, ps, PRM, FAKE + 8 * total, FAKE, total) == sacra.ERR_BADARG
    assert _code(sacra.rk4_step, ps, PRM, FAKE, FAKE + 64, total) == sacra.ERR_BADARG


def test_inter_level_spacing_and_overlap():
    pp, tp = wl.make_layout([(16, 16, 16)], [0.2], [0.01], [(0, 0, 0)])
    pc, _ = wl.make_layout([(8, 8, 8)], [0.1], [0.005], [(0, 0, 0)])
    bad, _ = wl.make_layout([(8, 8, 8)], [0.2], [0.005], [(0, 0, 0)])
    far = FAKE + 8 * (tp + 64)
    assert _code(sacra.restrict, pp[0], bad[0], (4, 4, 4), FAKE, far) == sacra.ERR_BADARG       # not 2:1
    assert _code(sacra.prolong_ghosts, pp[0], bad[0], (4, 4, 4), FAKE, far) == sacra.ERR_BADARG
    assert _code(sacra.restrict, pp[0], pc[0], (4, 4, 4), FAKE, FAKE + 64) == sacra.ERR_BADARG   # states overlap


def test_boundary_argument_checks():
    ps, total = _patch()
    ok = [((1.0, 2.0, 3.0), [2, 2, 2, 2, 1, 2])]
    far = FAKE + 8 * (total + 64)
    assert C.sizeof(sacra.SacraBoundary) == 3 * 8 + 6 * 4
    assert _code(sacra.fill_ghosts_faces, ps, None, FAKE) == sacra.ERR_NULL
    assert _code(sacra.fill_ghosts_faces, ps, [((0, 0, 0), [0, 1, 2, 2, 2, 2])], FAKE) == sacra.ERR_BADARG   # half-periodic axis
    assert _code(sacra.fill_ghosts_faces, ps, [((0, 0, 0), [4, 2, 2, 2, 2, 2])], FAKE) == sacra.ERR_BADARG   # unknown mode
    assert _code(sacra.fill_ghosts_faces, ps, [((float("nan"), 0, 0), [2] * 6)], FAKE) == sacra.ERR_BADARG
    assert _code(sacra.sommerfeld_rhs, ps, ok, FAKE, FAKE + 64) == sacra.ERR_BADARG                       # overlap
    assert _code(sacra.sommerfeld_rhs, ps, ok, FAKE, far + 8) == sacra.ERR_ALIGN
    assert _code(sacra.rk4_substep_bc, ps, PRM, ok, 1, far, FAKE, far + 8 * (total + 64), far + 16 * (total + 64)) == sacra.ERR_BADARG
    assert _code(sacra.rk4_substep_bc, ps, PRM, ok, 7, FAKE, FAKE, far, far + 8 * (total + 64)) == sacra.ERR_BADARG
    assert _code(sacra.rk4_step_bc, ps, PRM, ok, FAKE, FAKE + 64, total) == sacra.ERR_BADARG
    assert _code(sacra.rk4_step_bc, ps, PRM, None, FAKE, far, total) == sacra.ERR_NULL


def test_sommerfeld_shell_cell_at_the_coordinate_origin_is_rejected():
    """Eq. 13 divides by r. A cell of a Sommerfeld shell at r = 0 would write NaN without an error, so every call
    that evaluates Eq. 13 refuses it on the host (8^3 patch, dx = 0.1: the shell of the x- face is i < 3)."""
    ps, total = _patch()
    far, som = FAKE + 8 * (total + 64), [2] * 6
    at = lambda i, j, k: (-0.1 * i, -0.1 * j, -0.1 * k)          # origin that puts cell (i, j, k) at x = y = z = 0
    for cell in ((0, 0, 0), (2, 4, 4), (4, 4, 7), (3, 5, 4)):
        assert _code(sacra.sommerfeld_rhs, ps, [(at(*cell), som)], FAKE, far) == sacra.ERR_BADARG, cell
    # the same cell is fine when it is not in a shell: interior cell, or the face it is near is not a Sommerfeld face
    for cell, faces in (((4, 4, 4), som), ((3, 3, 4), som), ((0, 4, 4), [1, 2, 2, 2, 2, 2]), ((4, 4, 4), [1] * 6)):
        assert _code(sacra.sommerfeld_rhs, ps, [(at(*cell), faces)], FAKE, FAKE + 64) == sacra.ERR_BADARG   # reaches the overlap check
        assert _code(sacra.sommerfeld_rhs, ps, [(at(*cell), faces)], FAKE, far + 8) == sacra.ERR_ALIGN      # ... and the alignment check
    # an origin that is merely close to a shell cell is accepted (r > 0)
    assert _code(sacra.sommerfeld_rhs, ps, [((1e-300, 0.0, 0.0), som)], FAKE, far + 8) == sacra.ERR_ALIGN
    bad = [(at(1, 1, 1), som)]
    assert _code(sacra.rk4_substep_bc, ps, PRM, bad, 1, FAKE, FAKE, far, far + 8 * (total + 64)) == sacra.ERR_BADARG
    assert _code(sacra.rk4_step_bc, ps, PRM, bad, FAKE, far, total) == sacra.ERR_BADARG


def test_subcycling_argument_checks():
    pp, tp = wl.make_layout([(16, 16, 16)], [0.2], [0.05], [(0, 0, 0)])
    pc, tc = wl.make_layout([(8, 8, 8)], [0.1], [0.025], [(0, 0, 0)])
    slow, _ = wl.make_layout([(8, 8, 8)], [0.1], [0.05], [(0, 0, 0)])
    assert sacra.time_weights(3, 0.5) == [-0.125, 0.75, 0.375]
    assert sacra.time_weights(2, 0.25) == [0.75, 0.25, 0.0]
    with pytest.raises(sacra.SacraError):
        sacra.time_weights(4, 0.5)
    step = 8 * (tp + 64)
    bufs = [FAKE + k * 6 * step for k in range(5)]
    bnd = ((0.0, 0.0, 0.0), [0] * 6)
    class T:                                   # stand-in for a tensor: the binding only asks for numel() and the pointer
        def __init__(self, ptr, n): self.ptr, self.n = ptr, n
        def numel(self): return self.n
    def call(parent, child, org, a, b, cc, d, e):
        lib = sacra.lib
        o = (C.c_int32 * 3)(*org)
        return lib.sacra_subcycle_step(sacra.make_patches([parent]), sacra.make_patches([child]), o,
                                       C.byref(sacra.make_params(PRM)), sacra.make_boundaries([bnd]), a, b, 0, cc, d, tp, e, tc, 0)
    ok = (4, 4, 4)
    assert call(pp[0], slow[0], ok, *bufs) == sacra.ERR_BADARG                 # the child's step is not dt / 2
    assert call(pp[0], pc[0], (1, 4, 4), *bufs) == sacra.ERR_BADARG            # prolongation stencil leaves the parent
    assert call(pp[0], pc[0], ok, bufs[0], bufs[0] + 64, *bufs[2:]) == sacra.ERR_BADARG   # overlapping buffers
    assert call(pp[0], pc[0], ok, bufs[0], None, *bufs[2:]) == sacra.ERR_NULL
    assert _code(sacra.lincomb, pp[0], [FAKE, FAKE + step], [0.5, 0.5], FAKE + 64) == sacra.ERR_BADARG
    assert _code(sacra.lincomb, pp[0], [FAKE, None], [0.5, 0.5], FAKE + 2 * step) == sacra.ERR_NULL


def test_partial_substep_and_face_buffer_argument_checks():
    ps, total = _patch()
    far = lambda k: FAKE + 8 * k * (total + 64)
    ok = [1] * 6
    assert _code(sacra.rk4_substep_part, ps, PRM, 2, 3, ok, FAKE, far(1), far(2), far(3)) == sacra.ERR_BADARG     # unknown part
    assert _code(sacra.rk4_substep_part, ps, PRM, 5, 1, ok, FAKE, far(1), far(2), far(3)) == sacra.ERR_BADARG
    assert _code(sacra.rk4_substep_part, ps, PRM, 1, 1, ok, far(1), FAKE, far(2), far(3)) == sacra.ERR_BADARG     # stage 1: u_n is u_in
    assert _code(sacra.rk4_substep_part, ps, PRM, 2, 2, None, FAKE, far(1), far(2), far(3)) == sacra.ERR_NULL
    assert _code(sacra.rk4_substep_part, ps, PRM, 2, 2, ok, FAKE, far(1), far(1) + 64, far(3)) == sacra.ERR_BADARG
    assert sacra.face_doubles(ps[0], 0) == 25 * 3 * 14 * 14
    assert _code(sacra.pack_face, ps[0], FAKE, 3, 0, far(1)) == sacra.ERR_BADARG
    assert _code(sacra.pack_face, ps[0], FAKE, 0, 2, far(1)) == sacra.ERR_BADARG
    assert _code(sacra.unpack_face, ps[0], FAKE, 0, 0, FAKE + 64) == sacra.ERR_BADARG                             # buffer inside the state
    assert _code(sacra.unpack_face, ps[0], None, 0, 0, far(1)) == sacra.ERR_NULL


def test_hierarchy_argument_checks():
    assert C.sizeof(sacra.SacraLevel) == 64
    pp, tp = wl.make_layout([(16, 16, 16)], [0.2], [0.05], [(0, 0, 0)])
    pc, tc = wl.make_layout([(8, 8, 8)], [0.1], [0.025], [(0, 0, 0)])
    bnd = ((0.0, 0.0, 0.0), [0] * 6)
    class T:                       # stand-in for a tensor: pointer and size
        def __init__(self, ptr, n): self.ptr, self.n = ptr, n
        def numel(self): return self.n
    def lv(base, n):
        step = 8 * (n + 64)
        return base, base + step, base + 2 * step, base + 8 * step
    a0, a1, a2, nxt = lv(FAKE, tp)
    b0, b1, b2, _ = lv(nxt, tc)
    def call(patches, orgs, bufs, sizes):
        n = len(patches)
        keep = [sacra.make_patches([p]) for p in patches]
        arr = (sacra.SacraLevel * n)()
        for l in range(n):
            arr[l].patch = C.cast(keep[l], C.POINTER(sacra.SacraPatch))
            for a in range(3):
                arr[l].org[a] = orgs[l][a]
            arr[l].u, arr[l].u_prev, arr[l].work = bufs[l]
            arr[l].state_doubles, arr[l].nsteps = sizes[l], 0
        return sacra.lib.sacra_hierarchy_step(arr, n, C.byref(sacra.make_params(PRM)), sacra.make_boundaries([bnd]), 0)
    ok = [(0, 0, 0), (4, 4, 4)]
    assert call([pp[0], pc[0]], ok, [(a0, a1, None), (b0, b1, b2)], [tp, tc]) == sacra.ERR_NULL
    assert call([pp[0], pc[0]], [(0, 0, 0), (1, 4, 4)], [(a0, a1, a2), (b0, b1, b2)], [tp, tc]) == sacra.ERR_BADARG   # geometry
    assert call([pp[0], pc[0]], ok, [(a0, a1, a2), (a0 + 64, b1, b2)], [tp, tc]) == sacra.ERR_BADARG                  # levels overlap
    assert call([pp[0], pc[0]], ok, [(a0, a0 + 64, a2), (b0, b1, b2)], [tp, tc]) == sacra.ERR_BADARG                  # u / u_prev overlap
    assert call([pp[0], pc[0]], ok, [(a0, a1, a2), (b0, b1, b2)], [tp, 100]) == sacra.ERR_BADARG                      # state too small
    assert sacra.lib.sacra_hierarchy_step(None, 2, C.byref(sacra.make_params(PRM)), sacra.make_boundaries([bnd]), 0) == sacra.ERR_NULL
