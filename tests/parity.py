"""GPU-vs-oracle comparison helpers (used by the -m gpu tests; nothing in the product imports this).

Parity protocol: N, F compared with the A17 norms; x, T plain relative.  The "halve dtau until
abs(de) <= 10 %" rule of PAPER.md:312 is a discrete branch: inputs differing by one fp32 ulp may take a different
number of halvings and both results are valid ("several results are correct").  A cell whose sub-cycle signature
(accepted | halvings << 16) differs from the oracle's on some step is a FLIP.  A flip changes that cell's radiation by
O(1e-3), which the transport hands to its neighbours with a factor <= nu/2 per cell and step; measured on config 5
the induced x error falls 1.5e-3 -> 2.7e-4 -> 3.5e-5 -> 5e-6 at L1 distance 0, 1, 2, 3 and is at the background
(~2e-6) beyond.  So the tolerance applies to cells farther than FLIP_RADIUS = 3 coarse cells (L1) from every flip;
flips and the cells inside that radius are counted, reported and held to a looser sanity bound instead.
"""
import numpy as np

import oracle as O
import paper_1508_07888_b200 as E

from .helpers import rel_err_F, rel_err_N

FLIP_RADIUS = 3


def coarse_ancestors(w):
    """anc[l][cell] -> coarse cell id, for every level."""
    anc = [np.arange(w.n ** 3, dtype=np.int64)]
    for l, p in enumerate(w.parent, start=1):
        a_oct = anc[l - 1][np.asarray(p, np.int64)]
        anc.append(np.repeat(a_oct, 8))
    return anc


def run_pair(w, n_steps, track_signatures=True, chemistry=None, thermal=None, otsa=None, bc=None, block=1, fused=None, flux=None):
    """Advance the oracle and the CUDA library side by side.
    Returns (oracle, gpu, flips, diags); flips = list of (step, level, cell, coarse_cell)."""
    kw = dict(chemistry=chemistry, thermal=thermal, otsa=otsa, bc=bc)
    orc = O.Oracle(w, flux=flux, **kw)
    gpu = E.EmmaRT(w, record_subcycles=1 if track_signatures else 0, fused=fused, flux=flux, **kw)
    nl = w.n_levels
    chem_on = (w.chemistry if chemistry is None else chemistry) and (w.thermal if thermal is None else thermal)
    do_track = track_signatures and chem_on
    anc = coarse_ancestors(w) if do_track else None
    flips, diags = [], []
    done = 0
    while done < n_steps:
        k = 1 if do_track else min(block, n_steps - done)
        rco, do = orc.step(w.dt, k)
        rcg, dg = gpu.step(w.dt, k)
        assert rco == O.OK, rco
        assert rcg == E.OK, (rcg, gpu.last_error())
        diags.append((do, dg))
        done += k
        if do_track:
            for l in range(nl + 1):
                so = orc.read(O.F_SUBCYCLES, l).astype(np.int64)
                sg = gpu.read(E.FIELD_SUBCYCLES, l).astype(np.int64)
                for c in np.flatnonzero(so != sg):
                    flips.append((done, l, int(c), int(anc[l][c])))
    return orc, gpu, flips, diags


def clean_masks(w, flips, n_steps, radius=None):
    """Per level: True for cells farther than `radius` (default FLIP_RADIUS; L1, coarse cells, periodic) from every flip.
    A flip of step s has had n_steps - s steps to spread, so its radius is min(radius, n_steps - s).  The L1 balls are grown by
    repeated 6-neighbour dilation of the seed grid (cost independent of the number of flips)."""
    n = w.n
    RM = FLIP_RADIUS if radius is None else int(radius)
    near = np.zeros((n, n, n), bool)                                  # [iz, iy, ix]
    if flips:
        seeds = [np.zeros((n, n, n), bool) for _ in range(RM + 1)]
        for (step, _l, _c, c0) in flips:
            R = max(0, min(RM, n_steps - step))
            seeds[R][c0 // (n * n), (c0 // n) % n, c0 % n] = True
        for R in range(RM, -1, -1):                                   # near = U_R dilate^R(seeds[R])
            if R < RM and near.any():
                grown = near.copy()
                for ax in range(3):
                    grown |= np.roll(near, 1, ax) | np.roll(near, -1, ax)
                near = grown
            near |= seeds[R]
    near = near.reshape(-1)
    anc = coarse_ancestors(w)
    return [~near[a] for a in anc]


def absorption_condition(w, dt):
    """1 + c sigma_g (1-x) n0 dt per coarse cell and group: the condition number of Eq. 43's N^{p+1} with respect to
    the neutral fraction.  A cell of optical depth tau >> 1 per step turns a relative perturbation d of (1-x) into
    tau*d on the transmitted N (N ~ exp(-tau)); fp32 holds 1-x to ~1e-7..1e-6, so the N, F tolerance after a
    COUPLED step is the north_star 1e-5 times this factor (it is 1 for transport and for optically thin cells)."""
    y = 1.0 - w.x[0].astype(np.float64)
    return [1.0 + w.c_red * w.sigma_N[g] * y * w.n0[0].astype(np.float64) * dt for g in range(w.G)]


def flip_distance(w, flips, rmax=12):
    """L1 distance (coarse cells, periodic) of every coarse cell to the nearest flip, capped at rmax + 1."""
    n = w.n
    cur = np.zeros((n, n, n), bool)
    for (_s, _l, _c, c0) in flips:
        cur[c0 // (n * n), (c0 // n) % n, c0 % n] = True
    dist = np.full((n, n, n), rmax + 1, np.int16)
    dist[cur] = 0
    for r in range(1, rmax + 1):
        grown = cur.copy()
        for ax in range(3):
            grown |= np.roll(cur, 1, ax) | np.roll(cur, -1, ax)
        dist[grown & ~cur] = r
        cur = grown
    return dist.reshape(-1)


def compare(orc, gpu, w, flips=None, n_steps=0, nf_floor=1e-12, nf_cond=None, radius=None):
    """Error report.  Keys: N, F (A17 norms, clean coarse cells), x, T, xn (clean cells, all levels), *_near (cells
    within FLIP_RADIUS of a flip), flips, cells, near_cells.  nf_cond: optional per-group arrays dividing the N, F
    errors (see absorption_condition)."""
    clean = clean_masks(w, flips or [], n_steps, radius)
    rep = {"flips": len(flips or []), "cells": int(sum(m.size for m in clean)),
           "near_cells": int(sum((~m).sum() for m in clean))}
    c = w.c_red
    eN = eF = 0.0
    m0 = clean[0]
    for g in range(w.G):
        Uo = orc.read(O.F_U, 0, g)
        Ug = gpu.read(E.FIELD_U, 0, g).astype(np.float64)
        floor = nf_floor * np.abs(Uo[:, 0]).max()
        sc = np.maximum(np.abs(Uo[:, 0]), max(floor, 1e-300))
        rN = np.abs(Ug[:, 0] - Uo[:, 0]) / sc
        rF = np.abs(Ug[:, 1:] - Uo[:, 1:]).max(axis=1) / (c * sc)
        if nf_cond is not None:
            rN = rN / nf_cond[g]
            rF = rF / nf_cond[g]
        if m0.any():
            eN = max(eN, rN[m0].max())
            eF = max(eF, rF[m0].max())
    rep["N"], rep["F"] = eN, eF
    for name, fo, fg in (("x", O.F_X, E.FIELD_X), ("T", O.F_T, E.FIELD_T), ("xn", O.F_XNEUTRAL, E.FIELD_XNEUTRAL)):
        worst_clean = worst_near = 0.0
        for l in range(w.n_levels + 1):
            a = orc.read(fo, l)
            b = gpu.read(fg, l).astype(np.float64)
            r = np.abs(b - a) / np.maximum(np.abs(a), 1e-300)
            m = clean[l]
            if m.any():
                worst_clean = max(worst_clean, r[m].max())
            if (~m).any():
                worst_near = max(worst_near, r[~m].max())
        rep[name] = worst_clean
        rep[name + "_near"] = worst_near
    return rep


def budget_residual(d, prev_total):
    """Relative photon-budget residual of one step (A15)."""
    rhs = d["photons_injected"] - d["photons_absorbed"] + d["photons_recomb_emitted"] - d["photons_outflow"]
    scale = max(abs(d["photons_total"]), abs(d["photons_injected"]), 1e-300)
    return abs((d["photons_total"] - prev_total) - rhs) / scale


def stencil_scale(U0g, n, bc):
    """max of N over the 7-point stencil of every cell (the magnitude of the terms Eq. 30+32 adds up): the forward
    error of an fp32 evaluation is bounded by a few eps32 times THIS, not times the (possibly cancelled) result."""
    N = np.abs(np.asarray(U0g, np.float64)[:, 0]).reshape(n, n, n)
    s = N.copy()
    for axis, (lo, hi) in zip((2, 1, 0), ((bc[0], bc[1]), (bc[2], bc[3]), (bc[4], bc[5]))):
        for sh in (+1, -1):
            r = np.roll(N, sh, axis=axis)
            if lo != 0:                         # non-periodic: the ghost is the cell itself
                sl = [slice(None)] * 3
                sl[axis] = 0 if sh == +1 else n - 1
                r[tuple(sl)] = N[tuple(sl)]
            s = np.maximum(s, r)
    return s.reshape(-1)
