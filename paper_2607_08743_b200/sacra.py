"""ctypes binding of libsacra (include/sacra.h): argument marshalling only.

Same names as the C ABI. State arguments are torch CUDA float64 tensors (or raw device pointers as
ints); every step of the path runs in the CUDA kernels of libsacra. There is no CPU fallback: if the
library cannot be built or loaded, importing this module raises.

    from paper_2607_08743_b200 import sacra
    sacra.rk4_step(patches, params, u, work)          # enqueues on torch's current CUDA stream
"""
from __future__ import annotations

import ctypes as C
import os

from . import build as _build

NF = 25
NG = 3
OK, ERR_NULL, ERR_BADARG, ERR_UNSUPPORTED, ERR_ALIGN, ERR_CUDA, ERR_TOOLARGE = 0, -1, -2, -3, -4, -5, -6
NORMS_STATIC_MAX_PLANES = 4096
FLAG_SKIP_INCREMENT = 1
EXPORTS = ("sacra_fill_ghosts", "sacra_z4c_rhs", "sacra_rk4_substep", "sacra_rk4_step",
           "sacra_strerror", "sacra_version",
           "sacra_constraints", "sacra_constraint_norms", "sacra_constraint_scratch_doubles",
           "sacra_fill_ghosts_bc", "sacra_restrict", "sacra_prolong_ghosts",
           "sacra_fill_ghosts_faces", "sacra_sommerfeld_rhs", "sacra_rk4_substep_bc", "sacra_rk4_step_bc",
           "sacra_time_weights", "sacra_lincomb", "sacra_subcycle_step",
           "sacra_face_doubles", "sacra_pack_face", "sacra_unpack_face", "sacra_rk4_substep_part",
           "sacra_hierarchy_step", "sacra_constraint_norms_static")


class SacraPatch(C.Structure):
    """sacra_patch_t"""
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("ng", C.c_int32),
                ("pitch_x", C.c_int64), ("field_stride", C.c_int64), ("patch_offset", C.c_int64),
                ("dx", C.c_double), ("dt", C.c_double)]


class SacraParams(C.Structure):
    """sacra_params_t"""
    _fields_ = [("kappa1", C.c_double), ("kappa2", C.c_double), ("eta", C.c_double),
                ("shift_coef", C.c_double), ("ko_sigma", C.c_double),
                ("lapse_uses_khat", C.c_int32), ("flags", C.c_int32)]


class SacraBoundary(C.Structure):
    """sacra_boundary_t"""
    _fields_ = [("origin", C.c_double * 3), ("face", C.c_int32 * 6)]


class SacraLevel(C.Structure):
    """sacra_level_t"""
    _fields_ = [("patch", C.POINTER(SacraPatch)), ("org", C.c_int32 * 3), ("pad_", C.c_int32), ("u", C.c_void_p),
                ("u_prev", C.c_void_p), ("work", C.c_void_p), ("state_doubles", C.c_int64), ("nsteps", C.c_int64)]


class SacraError(RuntimeError):
    def __init__(self, code: int):
        self.code = code
        super().__init__("libsacra: %s (%d)" % (strerror(code), code))


def _load():
    # SACRA_LIB overrides the in-tree library; otherwise (re)build it if its sources changed.
    path = os.environ.get("SACRA_LIB") or _build.build()   # raises if nvcc fails: no silent fallback
    lib = C.CDLL(path)
    vp, dp, i32, i64 = C.c_void_p, C.c_void_p, C.c_int, C.c_int64
    lib.sacra_fill_ghosts.argtypes = [vp, i32, dp, vp]
    lib.sacra_z4c_rhs.argtypes = [vp, i32, vp, dp, dp, vp]
    lib.sacra_rk4_substep.argtypes = [vp, i32, vp, i32, dp, dp, dp, dp, vp]
    lib.sacra_rk4_step.argtypes = [vp, i32, vp, dp, dp, i64, vp]
    lib.sacra_constraints.argtypes = [vp, i32, dp, dp, vp]
    lib.sacra_constraint_norms.argtypes = [vp, i32, dp, dp, dp, vp]
    lib.sacra_constraint_scratch_doubles.argtypes = [vp, i32]
    lib.sacra_constraint_scratch_doubles.restype = C.c_int64
    lib.sacra_fill_ghosts_bc.argtypes = [vp, i32, vp, dp, vp]
    lib.sacra_restrict.argtypes = [vp, vp, vp, dp, dp, vp]
    lib.sacra_prolong_ghosts.argtypes = [vp, vp, vp, dp, dp, vp]
    lib.sacra_fill_ghosts_faces.argtypes = [vp, i32, vp, dp, vp]
    lib.sacra_sommerfeld_rhs.argtypes = [vp, i32, vp, dp, dp, vp]
    lib.sacra_rk4_substep_bc.argtypes = [vp, i32, vp, vp, i32, dp, dp, dp, dp, vp]
    lib.sacra_rk4_step_bc.argtypes = [vp, i32, vp, vp, dp, dp, i64, vp]
    lib.sacra_time_weights.argtypes = [i32, C.c_double, vp]
    lib.sacra_lincomb.argtypes = [vp, i32, dp, dp, dp, vp, dp, vp]
    lib.sacra_subcycle_step.argtypes = [vp, vp, vp, vp, vp, dp, dp, i32, dp, dp, i64, dp, i64, vp]
    lib.sacra_face_doubles.argtypes = [vp, i32]
    lib.sacra_face_doubles.restype = C.c_int64
    lib.sacra_pack_face.argtypes = [vp, dp, i32, i32, dp, vp]
    lib.sacra_unpack_face.argtypes = [vp, dp, i32, i32, dp, vp]
    lib.sacra_rk4_substep_part.argtypes = [vp, i32, vp, i32, i32, vp, dp, dp, dp, dp, vp]
    lib.sacra_hierarchy_step.argtypes = [vp, i32, vp, vp, vp]
    lib.sacra_constraint_norms_static.argtypes = [vp, i32, dp, dp, vp]
    lib.sacra_constraint_norms_static.restype = C.c_int
    for n in EXPORTS[:4] + EXPORTS[6:8] + EXPORTS[9:19] + EXPORTS[20:24]:
        getattr(lib, n).restype = C.c_int
    lib.sacra_strerror.argtypes = [C.c_int]
    lib.sacra_strerror.restype = C.c_char_p
    lib.sacra_version.restype = C.c_char_p
    return lib, path


lib, LIB_PATH = _load()


def strerror(code: int) -> str:
    return lib.sacra_strerror(int(code)).decode()


def version() -> str:
    return lib.sacra_version().decode()


def make_patches(ps):
    """list of objects with nx ny nz pitch_x field_stride patch_offset dx dt [ng] -> (SacraPatch*n)"""
    if isinstance(ps, C.Array):
        return ps
    arr = (SacraPatch * len(ps))()
    for a, p in zip(arr, ps):
        a.nx, a.ny, a.nz, a.ng = p.nx, p.ny, p.nz, getattr(p, "ng", NG)
        a.pitch_x, a.field_stride, a.patch_offset = p.pitch_x, p.field_stride, p.patch_offset
        a.dx, a.dt = p.dx, p.dt
    return arr


def make_params(d):
    if isinstance(d, SacraParams):
        return d
    return SacraParams(d["kappa1"], d["kappa2"], d["eta"], d["shift_coef"], d["ko_sigma"],
                       int(d.get("lapse_uses_khat", 1)), int(d.get("flags", 0)))


def _ptr(t):
    """device pointer of a torch CUDA float64 tensor, or an int/None passed through"""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if not (t.is_cuda and t.dtype.is_floating_point and t.element_size() == 8 and t.is_contiguous()):
        raise TypeError("libsacra takes contiguous CUDA float64 tensors")
    return t.data_ptr()


def _stream(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return stream if isinstance(stream, int) else stream.cuda_stream


def _check(code):
    if code != OK:
        raise SacraError(code)


def _ref(x):
    return C.byref(x) if x is not None else None


def fill_ghosts(patches, u, stream=None):
    ps = make_patches(patches) if patches is not None else None
    _check(lib.sacra_fill_ghosts(ps, len(ps) if ps is not None else 0, _ptr(u), _stream(stream)))


def z4c_rhs(patches, params, u, rhs, stream=None):
    ps = make_patches(patches) if patches is not None else None
    pr = make_params(params) if params is not None else None
    _check(lib.sacra_z4c_rhs(ps, len(ps) if ps is not None else 0, _ref(pr), _ptr(u), _ptr(rhs),
                             _stream(stream)))


def rk4_substep(patches, params, stage, u_n, u_in, u_out, acc, stream=None):
    ps = make_patches(patches) if patches is not None else None
    pr = make_params(params) if params is not None else None
    _check(lib.sacra_rk4_substep(ps, len(ps) if ps is not None else 0, _ref(pr), int(stage), _ptr(u_n),
                                 _ptr(u_in), _ptr(u_out), _ptr(acc), _stream(stream)))


def rk4_step(patches, params, u, work, state_doubles=None, stream=None):
    """work: one tensor of 3*state_doubles; state_doubles defaults to u.numel()."""
    ps = make_patches(patches) if patches is not None else None
    pr = make_params(params) if params is not None else None
    if state_doubles is None:
        state_doubles = u.numel()
    _check(lib.sacra_rk4_step(ps, len(ps) if ps is not None else 0, _ref(pr), _ptr(u), _ptr(work),
                              int(state_doubles), _stream(stream)))


def constraints(patches, u, con, stream=None):
    """H, M^x, M^y, M^z into fields 0..3 of the state-shaped buffer con (Eqs. 20-21)."""
    ps = make_patches(patches) if patches is not None else None
    _check(lib.sacra_constraints(ps, len(ps) if ps is not None else 0, _ptr(u), _ptr(con), _stream(stream)))


def constraint_scratch_doubles(patches) -> int:
    ps = make_patches(patches)
    return int(lib.sacra_constraint_scratch_doubles(ps, len(ps)))


def constraint_norms(patches, con, scratch, norms, stream=None):
    """norms: CUDA float64 tensor of 4 (Eq. 22); scratch: >= constraint_scratch_doubles(patches)."""
    ps = make_patches(patches) if patches is not None else None
    _check(lib.sacra_constraint_norms(ps, len(ps) if ps is not None else 0, _ptr(con), _ptr(scratch), _ptr(norms),
                                      _stream(stream)))


def constraint_norms_static(patches, con, norms, stream=None):
    """constraint_norms without the scratch argument, for callers that cannot allocate device memory (an arena owns
    it all, or a cudaMalloc inside the time loop would stall the device). The partial sums go to a fixed 128 KiB
    array inside libsacra that all calls on a device share: at most NORMS_STATIC_MAX_PLANES active z-planes over all
    patches (SacraError with ERR_TOOLARGE beyond that), and calls that overlap on the GPU race. Same bits in `norms` as
    constraint_norms. The first call on a device looks the array's address up; make it before any stream capture."""
    ps = make_patches(patches) if patches is not None else None
    _check(lib.sacra_constraint_norms_static(ps, len(ps) if ps is not None else 0, _ptr(con), _ptr(norms),
                                             _stream(stream)))


BC_PERIODIC, BC_MIRROR, BC_SOMMERFELD, BC_NONE = 0, 1, 2, 3


def make_boundaries(bs):
    """list of (origin[3], face[6]) per patch -> (SacraBoundary*n)"""
    if bs is None or isinstance(bs, C.Array):
        return bs
    arr = (SacraBoundary * len(bs))()
    for a, (o, f) in zip(arr, bs):
        for i in range(3):
            a.origin[i] = float(o[i])
        for i in range(6):
            a.face[i] = int(f[i])
    return arr


def fill_ghosts_faces(patches, bnd, u, stream=None):
    ps = make_patches(patches) if patches is not None else None
    _check(lib.sacra_fill_ghosts_faces(ps, len(ps) if ps is not None else 0, make_boundaries(bnd), _ptr(u), _stream(stream)))


def sommerfeld_rhs(patches, bnd, u, rhs, stream=None):
    ps = make_patches(patches) if patches is not None else None
    _check(lib.sacra_sommerfeld_rhs(ps, len(ps) if ps is not None else 0, make_boundaries(bnd), _ptr(u), _ptr(rhs),
                                    _stream(stream)))


def rk4_substep_bc(patches, params, bnd, stage, u_n, u_in, u_out, acc, stream=None):
    ps = make_patches(patches) if patches is not None else None
    pr = make_params(params) if params is not None else None
    _check(lib.sacra_rk4_substep_bc(ps, len(ps) if ps is not None else 0, _ref(pr), make_boundaries(bnd), int(stage),
                                    _ptr(u_n), _ptr(u_in), _ptr(u_out), _ptr(acc), _stream(stream)))


def rk4_step_bc(patches, params, bnd, u, work, state_doubles=None, stream=None):
    ps = make_patches(patches) if patches is not None else None
    pr = make_params(params) if params is not None else None
    if state_doubles is None:
        state_doubles = u.numel()
    _check(lib.sacra_rk4_step_bc(ps, len(ps) if ps is not None else 0, _ref(pr), make_boundaries(bnd), _ptr(u), _ptr(work),
                                 int(state_doubles), _stream(stream)))


def fill_ghosts_bc(patches, axis_mode, u, stream=None):
    """halo fill with a mode per axis (BC_PERIODIC / BC_MIRROR for x, y, z)"""
    ps = make_patches(patches) if patches is not None else None
    m = (C.c_int32 * 3)(*[int(v) for v in axis_mode])
    _check(lib.sacra_fill_ghosts_bc(ps, len(ps) if ps is not None else 0, m, _ptr(u), _stream(stream)))


def _one(p):
    return make_patches([p]) if p is not None else None


def restrict(parent, child, org, u_parent, u_child, stream=None):
    """4th-order Lagrange restriction child -> covered parent cells (sacra_restrict)"""
    o = (C.c_int32 * 3)(*[int(v) for v in org]) if org is not None else None
    _check(lib.sacra_restrict(_one(parent), _one(child), o, _ptr(u_parent), _ptr(u_child), _stream(stream)))


def prolong_ghosts(parent, child, org, u_parent, u_child, stream=None):
    """6th-order Lagrange prolongation parent -> ghost cells of the child (sacra_prolong_ghosts)"""
    o = (C.c_int32 * 3)(*[int(v) for v in org]) if org is not None else None
    _check(lib.sacra_prolong_ghosts(_one(parent), _one(child), o, _ptr(u_parent), _ptr(u_child), _stream(stream)))


def time_weights(nlevels, theta):
    """weights of the parent time levels at theta (host function of the library)"""
    w = (C.c_double * 3)()
    _check(lib.sacra_time_weights(int(nlevels), float(theta), w))
    return [w[0], w[1], w[2]]


def lincomb(patch, levels, w, out, stream=None):
    """out = (w0 u0 + w1 u1) [+ w2 u2] on every storage cell of one patch (sacra_lincomb)"""
    n = len(levels)
    u = list(levels) + [None] * (3 - n)
    wv = (C.c_double * 3)(*([float(x) for x in w] + [0.0] * (3 - len(w))))
    _check(lib.sacra_lincomb(_one(patch), n, _ptr(u[0]), _ptr(u[1]), _ptr(u[2]), wv, _ptr(out), _stream(stream)))


def subcycle_step(parent, child, org, params, parent_bnd, u_parent, u_parent_prev, have_prev, u_child, work_parent,
                  work_child, stream=None):
    """one Berger-Oliger step of a parent / child pair (sacra_subcycle_step); work_parent: 5 parent states, work_child: 3"""
    o = (C.c_int32 * 3)(*[int(v) for v in org]) if org is not None else None
    pr = make_params(params) if params is not None else None
    _check(lib.sacra_subcycle_step(_one(parent), _one(child), o, _ref(pr), make_boundaries([parent_bnd]), _ptr(u_parent),
                                   _ptr(u_parent_prev), int(bool(have_prev)), _ptr(u_child), _ptr(work_parent),
                                   int(u_parent.numel()), _ptr(work_child), int(u_child.numel()), _stream(stream)))


def face_doubles(patch, axis) -> int:
    return int(lib.sacra_face_doubles(_one(patch), int(axis)))


def pack_face(patch, u, axis, side, buf, stream=None):
    """buf <- the 3 outermost active layers at a face (sacra_pack_face)"""
    _check(lib.sacra_pack_face(_one(patch), _ptr(u), int(axis), int(side), _ptr(buf), _stream(stream)))


def unpack_face(patch, u, axis, side, buf, stream=None):
    """the 3 ghost layers behind a face <- buf (sacra_unpack_face)"""
    _check(lib.sacra_unpack_face(_one(patch), _ptr(u), int(axis), int(side), _ptr(buf), _stream(stream)))


PART_INTERIOR, PART_SHELL = 1, 2


def rk4_substep_part(patches, params, stage, part, exchange_faces, u_n, u_in, u_out, acc, stream=None):
    """sacra_rk4_substep on the cells that need no exchanged ghost (PART_INTERIOR) or on the others (PART_SHELL)"""
    ps = make_patches(patches) if patches is not None else None
    pr = make_params(params) if params is not None else None
    xf = (C.c_int32 * 6)(*[int(v) for v in exchange_faces]) if exchange_faces is not None else None
    _check(lib.sacra_rk4_substep_part(ps, len(ps) if ps is not None else 0, _ref(pr), int(stage), int(part), xf,
                                      _ptr(u_n), _ptr(u_in), _ptr(u_out), _ptr(acc), _stream(stream)))


def hierarchy_step(patches, orgs, params, bnd0, states, prevs, works, nsteps, stream=None):
    """one step of level 0 of a hierarchy of nested levels, finer levels subcycled (sacra_hierarchy_step). patches, orgs,
    states, prevs, works (5 states each): one entry per level; nsteps: list of ints, updated in place"""
    n = len(patches)
    keep = [make_patches([p]) for p in patches]
    lv = (SacraLevel * n)()
    for l in range(n):
        lv[l].patch = C.cast(keep[l], C.POINTER(SacraPatch))
        for a in range(3):
            lv[l].org[a] = int(orgs[l][a])
        lv[l].u, lv[l].u_prev, lv[l].work = _ptr(states[l]), _ptr(prevs[l]), _ptr(works[l])
        lv[l].state_doubles, lv[l].nsteps = int(states[l].numel()), int(nsteps[l])
    pr = make_params(params) if params is not None else None
    _check(lib.sacra_hierarchy_step(lv, n, _ref(pr), make_boundaries([bnd0]), _stream(stream)))
    for l in range(n):
        nsteps[l] = int(lv[l].nsteps)
