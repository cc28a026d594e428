"""Helpers for the -m gpu tests: run the CUDA path (through the ctypes binding of the C ABI) on a numpy
state and bring the result back. Holds no arithmetic of the method."""
import numpy as np
import torch

from paper_2607_08743_b200 import sacra


def dev(a: np.ndarray) -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def host(t: torch.Tensor) -> np.ndarray:
    torch.cuda.synchronize()
    return t.cpu().numpy()


def gpu_fill(w, state):
    u = dev(state)
    sacra.fill_ghosts(w.patches, u)
    return host(u)


def gpu_rhs(w, filled_state, poison=np.nan):
    u = dev(filled_state)
    r = torch.full_like(u, poison)
    sacra.z4c_rhs(w.patches, w.params, u, r)
    return host(r)


def gpu_step(w, state):
    """one sacra_rk4_step; returns (new state, S)"""
    u = dev(state)
    n = u.numel()
    work = torch.zeros(3 * n, dtype=torch.float64, device="cuda")
    sacra.rk4_step(w.patches, w.params, u, work)
    return host(u), host(work[2 * n:])
