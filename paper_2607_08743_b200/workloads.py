"""Seeded synthetic inputs for the five BASELINE.json configs (numpy, host side).

This module holds NO arithmetic of the method (no stencil, no RHS, no RK4, no
ghost fill): only closed-form initial data, a counter-based noise generator and
the memory layout. It is the one module that both the CUDA path's callers
(tests, bench.py) and the oracle's callers use, so that both see the same bytes.

The paper's own workloads are FUKA binary initial data on a box-in-box AMR
hierarchy; they are not available, so
BASELINE.json's closed-form configs stand in for them ("Inputs").

Field order (include/sacra.h): 0 W; 1-6 gt_xx xy xz yy yz zz; 7 K-hat;
8-13 At_xx..zz; 14-16 Gt^x y z; 17 Theta; 18 alpha; 19-21 beta^i; 22-24 B^i.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

NF = 25
NG = 3
F_W, F_G, F_KH, F_A, F_GAM, F_TH, F_ALP, F_BET, F_B = 0, 1, 7, 8, 14, 17, 18, 19, 22
FIELD_NAMES = ["W", "gt_xx", "gt_xy", "gt_xz", "gt_yy", "gt_yz", "gt_zz", "Khat",
               "At_xx", "At_xy", "At_xz", "At_yy", "At_yz", "At_zz", "Gt_x", "Gt_y", "Gt_z",
               "Theta", "alpha", "beta_x", "beta_y", "beta_z", "B_x", "B_y", "B_z"]
# pi-rotation about z, (x,y,z)->(-x,-y,z): sign of each field
PI_SIGN = np.array([+1, +1, +1, -1, +1, -1, +1, +1, +1, +1, -1, +1, -1, +1, -1, -1, +1,
                    +1, +1, -1, -1, +1, -1, -1, +1], dtype=np.float64)

DEFAULT_PARAMS = dict(kappa1=0.02, kappa2=0.0, eta=2.0, shift_coef=0.75, ko_sigma=0.1,
                      lapse_uses_khat=1)


@dataclass
class Patch:
    """One uniform patch in a state buffer (mirrors sacra_patch_t)."""
    nx: int
    ny: int
    nz: int
    pitch_x: int
    field_stride: int
    patch_offset: int
    dx: float
    dt: float
    origin: tuple = (0.0, 0.0, 0.0)   # coordinate of active cell (0,0,0); not part of the ABI
    ng: int = NG

    @property
    def shape(self):  # storage shape of one field, (z, y, x-pitch)
        return (self.nz + 2 * NG, self.ny + 2 * NG, self.pitch_x)

    @property
    def npoints(self):
        return self.nx * self.ny * self.nz


@dataclass
class Workload:
    name: str
    patches: list
    params: dict
    state: np.ndarray            # flat float64, all patches, ghosts NOT filled (zero)
    nsteps: int = 1
    meta: dict = field(default_factory=dict)

    @property
    def npoints(self):
        return sum(p.npoints for p in self.patches)

    def field_view(self, buf: np.ndarray, ip: int, f: int) -> np.ndarray:
        """(z,y,x-pitch) view of field f of patch ip inside a flat state buffer."""
        p = self.patches[ip]
        n = int(np.prod(p.shape))
        o = p.patch_offset + f * p.field_stride
        return buf[o:o + n].reshape(p.shape)

    def active_view(self, buf: np.ndarray, ip: int, f: int) -> np.ndarray:
        p = self.patches[ip]
        return self.field_view(buf, ip, f)[NG:NG + p.nz, NG:NG + p.ny, NG:NG + p.nx]


def round_up(a: int, m: int) -> int:
    return (a + m - 1) // m * m


def make_layout(dims, dxs, dts, origins, pitch_align=8, lead_pad=5):
    """Patches back to back in one buffer. pitch = roundup(nx+6, pitch_align).

    lead_pad doubles are left before field 0 of the first patch so that active
    cell i=0 (storage index 3) of every row starts on a 64-byte boundary when
    lead_pad = 5 and pitch is a multiple of 8 (3+5 = 8). Returns (patches, total)."""
    patches, off = [], lead_pad
    for (nx, ny, nz), dx, dt, org in zip(dims, dxs, dts, origins):
        pitch = round_up(nx + 2 * NG, pitch_align)
        fs = round_up(pitch * (ny + 2 * NG) * (nz + 2 * NG), 8)
        patches.append(Patch(nx, ny, nz, pitch, fs, off, float(dx), float(dt), tuple(org)))
        off += NF * fs
    return patches, round_up(off + 8, 8)


# ---------------------------------------------------------------------------
# counter-based noise: U = (splitmix64(seed ^ hash(p,f,i,j,k)) >> 11) * 2^-53
# ---------------------------------------------------------------------------
_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(x: np.ndarray) -> np.ndarray:
    with np.errstate(over="ignore"):
        x = (x + np.uint64(0x9E3779B97F4A7C15)) & _M64
        z = x
        z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
        z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
        return z ^ (z >> np.uint64(31))


def noise(seed: int, ip: int, f: int, nz: int, ny: int, nx: int, amp: float) -> np.ndarray:
    """amp*(2U-1) on the active cells of field f of patch ip; shape (nz,ny,nx)."""
    k, j, i = np.meshgrid(np.arange(nz, dtype=np.uint64), np.arange(ny, dtype=np.uint64),
                          np.arange(nx, dtype=np.uint64), indexing="ij")
    with np.errstate(over="ignore"):
        ctr = ((np.uint64(ip) * np.uint64(NF) + np.uint64(f)) << np.uint64(40)) ^ \
              (k << np.uint64(26)) ^ (j << np.uint64(13)) ^ i
        h = _splitmix64(np.uint64(seed) ^ _splitmix64(ctr))
    u = (h >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)
    return amp * (2.0 * u - 1.0)


def _coords(p: Patch, symmetric=False):
    if symmetric:
        # cell-centred box symmetric about the origin: x_i = (2i-(n-1)) (h/2), so that
        # x_{n-1-i} == -x_i bitwise for any h (needed for bitwise pi-symmetric data)
        x = (2 * np.arange(p.nx) - (p.nx - 1)) * (0.5 * p.dx)
        y = (2 * np.arange(p.ny) - (p.ny - 1)) * (0.5 * p.dx)
        z = (2 * np.arange(p.nz) - (p.nz - 1)) * (0.5 * p.dx)
        return np.meshgrid(z, y, x, indexing="ij")
    x = p.origin[0] + np.arange(p.nx) * p.dx
    y = p.origin[1] + np.arange(p.ny) * p.dx
    z = p.origin[2] + np.arange(p.nz) * p.dx
    return np.meshgrid(z, y, x, indexing="ij")  # Z, Y, X each (nz,ny,nx)


def _flat_fields(shape):
    """Minkowski in these variables: W=1, gt=delta, alpha=1, rest 0."""
    one, zero = np.ones(shape), np.zeros(shape)
    v = [zero] * NF
    v[F_W] = one
    v[F_G + 0] = one
    v[F_G + 3] = one
    v[F_G + 5] = one
    v[F_ALP] = one
    return v


def _store(wl: Workload, ip: int, fields, seed, amp):
    p = wl.patches[ip]

    def one(f):
        a = np.array(fields[f], dtype=np.float64, copy=True)
        if amp:
            a = a + noise(seed, ip, f, p.nz, p.ny, p.nx, amp)
        wl.active_view(wl.state, ip, f)[...] = a

    if p.npoints >= 1 << 21:           # large patches: fields in parallel (numpy releases the GIL)
        from concurrent.futures import ThreadPoolExecutor
        with ThreadPoolExecutor(max_workers=8) as ex:
            list(ex.map(one, range(NF)))
    else:
        for f in range(NF):
            one(f)


def _puncture_fields(p: Patch, punctures, symmetric=False):
    """Brill-Lindquist / single-puncture data: psi = 1 + sum m/(2 r); W = alpha = psi^-2."""
    Z, Y, X = _coords(p, symmetric)
    s = None
    for (m, cx, cy, cz) in punctures:
        r = np.sqrt((X - cx) ** 2 + (Y - cy) ** 2 + (Z - cz) ** 2)
        t = m / (2.0 * r)
        s = t if s is None else s + t      # two punctures: commutative inner sum (pi-symmetric)
    psi = 1.0 + s
    W = 1.0 / (psi * psi)
    v = _flat_fields(W.shape)
    v[F_W] = W
    v[F_ALP] = W.copy()
    return v


def config0(n=32, eps=1e-3, amp=1e-10, seed=1234, params=None):
    """Linearised TT plane wave along x on [0,1)^3, x_i = i h (BASELINE.json configs[0])."""
    h = 1.0 / n
    patches, total = make_layout([(n, n, n)], [h], [0.25 * h], [(0.0, 0.0, 0.0)])
    wl = Workload("config0_tt_wave_%d" % n, patches, dict(params or DEFAULT_PARAMS),
                  np.zeros(total), meta=dict(eps=eps, amp=amp, seed=seed))
    Z, Y, X = _coords(patches[0])
    v = _flat_fields(X.shape)
    s, c = np.sin(2 * np.pi * X), np.cos(2 * np.pi * X)
    v[F_G + 3] = 1.0 + eps * s
    v[F_G + 5] = 1.0 - eps * s
    v[F_A + 3] = np.pi * eps * c          # reading O: right-moving wave, At_yy = +pi eps cos
    v[F_A + 5] = -np.pi * eps * c
    _store(wl, 0, v, seed, amp)
    return wl


def config1(n=64, amp=1e-12, seed=1235, params=None, half_width=8.0):
    """Single Schwarzschild puncture M=1, cell-centred on [-8,8]^3 (configs[1])."""
    h = 2.0 * half_width / n
    org = (-half_width + 0.5 * h,) * 3
    patches, total = make_layout([(n, n, n)], [h], [0.25 * h], [org])
    wl = Workload("config1_puncture_%d" % n, patches, dict(params or DEFAULT_PARAMS),
                  np.zeros(total), meta=dict(amp=amp, seed=seed))
    _store(wl, 0, _puncture_fields(patches[0], [(1.0, 0.0, 0.0, 0.0)]), seed, amp)
    return wl


def config2(n=128, half_width=16.0, amp=0.0, seed=1236, params=None, nsteps=1, name=None):
    """Brill-Lindquist binary m1=m2=0.5 at (+-5,0,0); bitwise pi-symmetric (configs[2])."""
    h = 2.0 * half_width / n
    org = (-half_width + 0.5 * h,) * 3
    patches, total = make_layout([(n, n, n)], [h], [0.25 * h], [org])
    wl = Workload(name or "config2_brill_lindquist_%d" % n, patches,
                  dict(params or DEFAULT_PARAMS), np.zeros(total), nsteps=nsteps,
                  meta=dict(amp=amp, seed=seed))
    _store(wl, 0, _puncture_fields(patches[0], [(0.5, 5.0, 0.0, 0.0), (0.5, -5.0, 0.0, 0.0)],
                                   symmetric=True), seed, amp)
    return wl


def config3(n=64, npatch=8, amp=1e-12, seed=1237, params=None):
    """Box-in-box stand-in: 8 independent n^3 patches, 4 at h=0.25 and 4 at h=0.125, each
    sampling the config-1 puncture around its own seeded origin offset (configs[3])."""
    rng = np.random.Generator(np.random.PCG64(seed))
    dims, dxs, dts, orgs = [], [], [], []
    for ip in range(npatch):
        h = 0.25 if ip < npatch // 2 else 0.125
        while True:
            off = rng.uniform(-2.0, 2.0, size=3)
            org = off - 0.5 * n * h + 0.5 * h
            # redraw if a cell centre lands within 1e-3 h of the puncture on every axis
            d = [np.min(np.abs(org[a] + np.arange(n) * h)) for a in range(3)]
            if np.sqrt(sum(x * x for x in d)) > 1e-3 * h:
                break
        dims.append((n, n, n)); dxs.append(h); dts.append(0.25 * h); orgs.append(tuple(org))
    patches, total = make_layout(dims, dxs, dts, orgs)
    wl = Workload("config3_boxes_%dx%d" % (npatch, n), patches, dict(params or DEFAULT_PARAMS),
                  np.zeros(total), meta=dict(amp=amp, seed=seed))
    for ip, p in enumerate(patches):
        _store(wl, ip, _puncture_fields(p, [(1.0, 0.0, 0.0, 0.0)]), seed, amp)
    return wl


def config4(n=256, amp=1e-12, seed=1238, params=None, nsteps=10):
    """Large uniform patch: config-2 data on [-32,32]^3 at h=0.25, ten steps (configs[4])."""
    return config2(n=n, half_width=n * 0.125, amp=amp, seed=seed, params=params, nsteps=nsteps,
                   name="config4_large_%d" % n)


CONFIGS = {0: config0, 1: config1, 2: config2, 3: config3, 4: config4}


def make(idx: int, **kw) -> Workload:
    return CONFIGS[idx](**kw)
