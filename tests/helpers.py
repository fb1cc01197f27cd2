"""Shared test helpers: tiny hand-made workloads and error norms (reading A17)."""
import numpy as np

from workloads import CGS, blackbody_groups
from workloads.configs import Workload

_GR = {}


def groups(G):
    if G not in _GR:
        _GR[G] = blackbody_groups(1.0e5, (13.6, 1000.0) if G == 1 else (13.6, 24.6, 54.4, 100.0, 1000.0) if G == 4 else (13.6, 24.6, 54.4, 1000.0), n_quad=20001)
    return _GR[G]


def tiny_workload(n, G=1, L=None, c_red=None, bc=(0,) * 6, n0=1e-3, x=1.2e-3, T=100.0, U0=None,
                  chemistry=1, thermal=1, otsa=1, parent=(), n0_lv=None, x_lv=None, T_lv=None,
                  src_pos=None, src_Q=None, courant=0.9):
    """A Workload with constant (or given) fields on an n^3 coarse grid (+ optional refined levels)."""
    gr = groups(G)
    dx = 6.6 * CGS.kpc / 32
    w = Workload("tiny", n, G, (dx * n) if L is None else L, 0.1 * CGS.c if c_red is None else c_red,
                 gr["sigma_N"], gr["sigma_E"], gr["E_mean"], gr["frac"], bc=tuple(bc), otsa=otsa,
                 chemistry=chemistry, thermal=thermal, courant=courant)
    nc = n ** 3
    full = lambda v, m: (np.full(m, v, np.float32) if np.isscalar(v) else np.ascontiguousarray(v, np.float32))
    w.parent = [np.ascontiguousarray(p, np.int64) for p in parent]
    sizes = [nc] + [8 * len(p) for p in w.parent]
    w.n0 = [full(n0, nc)] + [full(a, m) for a, m in zip(n0_lv or [n0] * len(w.parent), sizes[1:])]
    w.x = [full(x, nc)] + [full(a, m) for a, m in zip(x_lv or [x] * len(w.parent), sizes[1:])]
    w.T = [full(T, nc)] + [full(a, m) for a, m in zip(T_lv or [T] * len(w.parent), sizes[1:])]
    if U0 is not None:
        w.U0 = [np.ascontiguousarray(U0[g], np.float32).reshape(nc, 4) for g in range(G)]
    if src_pos is not None:
        w.src_pos = np.asarray(src_pos, np.float64).reshape(-1, 3)
        w.src_Q = np.asarray(src_Q, np.float64).reshape(len(w.src_pos), G)
    return w


def rel_err_N(N, N_ref):
    """A17: abs(dN) / max(abs(N_ref), 1e-12 * max N_ref)."""
    N_ref = np.asarray(N_ref, np.float64)
    floor = 1e-12 * np.abs(N_ref).max()
    return np.abs(np.asarray(N, np.float64) - N_ref) / np.maximum(np.abs(N_ref), max(floor, 1e-300))


def rel_err_F(F, F_ref, N_ref, c):
    """A17: abs(dF_k) / max(c N_ref, floor*c)  (||F|| <= c N is the natural scale)."""
    N_ref = np.asarray(N_ref, np.float64)
    floor = 1e-12 * np.abs(N_ref).max()
    scale = c * np.maximum(np.abs(N_ref), max(floor, 1e-300))
    return np.abs(np.asarray(F, np.float64) - np.asarray(F_ref, np.float64)) / scale[:, None]
