"""Shared test helpers: analytic-filled states and comparison metrics (no method arithmetic)."""
import numpy as np

from paper_2607_08743_b200 import workloads as wl

NF, NG = wl.NF, wl.NG


def storage_coords(p):
    """Coordinates of every storage cell (ghosts included), arrays of shape (sz, sy, pitch)."""
    sz, sy, px = p.shape
    x = p.origin[0] + (np.arange(px) - NG) * p.dx
    y = p.origin[1] + (np.arange(sy) - NG) * p.dx
    z = p.origin[2] + (np.arange(sz) - NG) * p.dx
    return np.meshgrid(z, y, x, indexing="ij")


def analytic_state(n, h, origin, fn, dt=None):
    """One n^3 patch whose whole storage (ghosts too) is filled by fn(X,Y,Z)->list of 25 arrays."""
    patches, total = wl.make_layout([(n, n, n)], [h], [dt if dt else 0.25 * h], [origin])
    w = wl.Workload("analytic", patches, dict(wl.DEFAULT_PARAMS), np.zeros(total))
    Z, Y, X = storage_coords(patches[0])
    vals = fn(X, Y, Z)
    for f in range(NF):
        w.field_view(w.state, 0, f)[...] = np.broadcast_to(vals[f], patches[0].shape)
    return w


def flat(shape):
    one, zero = np.ones(shape), np.zeros(shape)
    v = [zero.copy() for _ in range(NF)]
    for f in (wl.F_W, wl.F_G + 0, wl.F_G + 3, wl.F_G + 5, wl.F_ALP):
        v[f] = one.copy()
    return v


def field_max_abs(w, buf, f):
    return max(np.max(np.abs(w.active_view(buf, ip, f))) for ip in range(len(w.patches)))


def field_max_diff(w, a, b, f):
    return max(np.max(np.abs(w.active_view(a, ip, f) - w.active_view(b, ip, f)))
               for ip in range(len(w.patches)))


def parity_report(w, got, ref, rtol=1e-11, floor=1e-14):
    """north_star metric: per field max|got-ref| <= rtol*(max|ref|+floor). Returns list of failures."""
    bad = []
    for f in range(NF):
        d = field_max_diff(w, got, ref, f)
        s = field_max_abs(w, ref, f)
        if not (d <= rtol * (s + floor)) or not np.isfinite(d):
            bad.append((wl.FIELD_NAMES[f], d, s, d / (s + floor)))
    return bad


def pi_partner(a):
    """(x,y,z)->(-x,-y,z) on an active (nz,ny,nx) array of a grid symmetric about the z axis."""
    return a[:, ::-1, ::-1]
