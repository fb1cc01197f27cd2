"""Static AMR meshes with resolution jumps <= 1 for the standard (non-CRTA) AMR transport.

Input recipe only: which cells are split, the densities of the children, the sources.  The paper's marking rule
(PAPER.md:75-81): (i) mark cells by a physical criterion, (ii) "if a cell is marked for refinement, so must be its 26
neighbors", jumps between neighbours never exceed one level.  Here the criterion is the coarse density averaged over
the 27 cells around a cell (S; refinement follows mass on a few-cell scale, so refined regions are patches, not single
cells): a coarse cell is marked when S > thresh1 * nbar and the marks are dilated once over the 26 neighbours (periodic
wrap); a level-1 cell is split when its parent has S > thresh2 * nbar (thresh2 >= thresh1: nested patches) and all its
26 level-1 neighbours exist, which keeps every face jump <= 1 by construction.
"""
import numpy as np

from .configs import SEED_BASE, Workload, _densest, _groups, _leaf_centres_l1, _leaf_centres_l2, _cell_centres
from .constants import CGS
from .fields import lognormal_density


def _dilate26(m):
    out = np.zeros_like(m)
    for dz in (-1, 0, 1):
        for dy in (-1, 0, 1):
            for dx in (-1, 0, 1):
                out |= np.roll(m, (dz, dy, dx), axis=(0, 1, 2))
    return out


def _mean27(a):
    out = np.zeros_like(a, dtype=np.float64)
    for dz in (-1, 0, 1):
        for dy in (-1, 0, 1):
            for dx in (-1, 0, 1):
                out += np.roll(a, (dz, dy, dx), axis=(0, 1, 2))
    return out / 27.0


def _all26(m):
    out = np.ones_like(m)
    for dz in (-1, 0, 1):
        for dy in (-1, 0, 1):
            for dx in (-1, 0, 1):
                out &= np.roll(m, (dz, dy, dx), axis=(0, 1, 2))
    return out


def _children_density(n0_parent, rng):
    """child = parent * exp(0.5 g - 0.125), g ~ N(0,1) in oct order, rescaled to average to the parent (cfg 4 recipe)."""
    g = rng.standard_normal((len(n0_parent), 8))
    ch = n0_parent[:, None].astype(np.float64) * np.exp(0.5 * g - 0.125)
    ch *= (n0_parent.astype(np.float64) / ch.mean(axis=1))[:, None]
    return ch.reshape(-1)


def _morton(i, j, k, bits=11):
    """interleaved bits of (i, j, k): the Z-order key of a cell."""
    key = np.zeros(len(i), np.int64)
    for b in range(bits):
        key |= ((i >> b) & 1).astype(np.int64) << (3 * b)
        key |= ((j >> b) & 1).astype(np.int64) << (3 * b + 1)
        key |= ((k >> b) & 1).astype(np.int64) << (3 * b + 2)
    return key


def balanced_two_level_mesh(n0c, n, nbar, rng, thresh1=2.5, thresh2=4.0, levels=2, order="id"):
    """n0c: float64 [n^3] coarse densities.  Returns (parents, n0_levels): parents = [p1, p2][:levels].
    order: the order of the octs of a level in memory (the C-ABI takes them in the order of the parent list): "id" =
    increasing id of the parent cell; "morton" = along the Z-order curve of the parent cell's coordinates, which keeps
    the octs of a patch, and so the neighbours a kernel reads together, close in memory."""
    S = _mean27(n0c.reshape(n, n, n))
    mark0 = _dilate26(S > thresh1 * nbar)
    p1 = np.flatnonzero(mark0.reshape(-1)).astype(np.int64)
    if order == "morton":
        p1 = p1[np.argsort(_morton(p1 % n, (p1 // n) % n, p1 // (n * n)), kind="stable")]
    n01 = _children_density(n0c[p1], rng)
    if levels == 1 or len(p1) == 0:
        return [p1], [n0c, n01]
    # dense map of the level-1 cells: id1[kz, ky, kx] = oct*8 + child, or -1
    id1 = np.full((2 * n, 2 * n, 2 * n), -1, np.int64)
    I, J, K = p1 % n, (p1 // n) % n, p1 // (n * n)
    for k in range(8):
        kx, ky, kz = k & 1, (k >> 1) & 1, (k >> 2) & 1
        id1[2 * K + kz, 2 * J + ky, 2 * I + kx] = 8 * np.arange(len(p1)) + k
    exist = id1 >= 0
    S1 = np.repeat(np.repeat(np.repeat(S, 2, axis=0), 2, axis=1), 2, axis=2)       # the parent's S on the level-1 grid
    mark1 = exist & (S1 > thresh2 * nbar) & _all26(exist)
    p2 = np.sort(id1[mark1]).astype(np.int64)
    if order == "morton":
        kz, ky, kx = np.nonzero(mark1)
        p2 = id1[kz, ky, kx][np.argsort(_morton(kx, ky, kz), kind="stable")].astype(np.int64)
    n02 = _children_density(n01[p2], rng)
    return [p1, p2], [n0c, n01, n02]


def make_amr_standard(n=16, G=3, levels=2, n_steps=4, n_src=None, sigma_ln=1.5, seed=None, thresh1=2.5, thresh2=4.0,
                      order="id"):
    """Config-4-like box on a jump-balanced mesh, for the standard AMR transport: lognormal density,
    sources in the densest leaves of the finest level, x = 1.2e-3, T = 100 K, N = F = 0, periodic."""
    rng = np.random.default_rng(SEED_BASE + 42 if seed is None else seed)
    gr = _groups(G)
    dx = 4.0 * CGS.kpc
    w = Workload("amr-standard%d" % n, n, G, dx * n, 0.1 * CGS.c, gr["sigma_N"], gr["sigma_E"], gr["E_mean"], gr["frac"])
    nbar = 1e-3
    n0c = lognormal_density(n, nbar, sigma_ln, rng).reshape(-1).astype(np.float64)
    parents, n0s = balanced_two_level_mesh(n0c, n, nbar, rng, thresh1, thresh2, levels, order)
    w.parent = parents
    w.n0 = [a.astype(np.float32) for a in n0s]
    w.x = [np.full(a.shape, 1.2e-3, np.float32) for a in w.n0]
    w.T = [np.full(a.shape, 100.0, np.float32) for a in w.n0]
    ns = n_src or max(1, min(1024, n ** 3 // 512))
    if len(parents) == 2 and len(parents[1]) * 8 >= ns:
        ids = _densest(w.n0[2], ns)
        pos = _leaf_centres_l2(ids, parents[0], parents[1], n)
    elif len(parents[0]) * 8 >= ns:
        leaf1 = np.ones(len(w.n0[1]), bool)
        if len(parents) == 2:
            leaf1[parents[1]] = False
        cand = np.flatnonzero(leaf1)
        ids = cand[_densest(w.n0[1][cand], ns)]
        pos = _leaf_centres_l1(ids, parents[0], n)
    else:
        pos = _cell_centres(_densest(w.n0[0], ns), n)
    w.src_pos = pos
    w.src_Q = (10.0 ** rng.uniform(47.0, 49.0, len(pos)))[:, None] * gr["frac"][None, :]
    w.n_steps = n_steps
    return w
