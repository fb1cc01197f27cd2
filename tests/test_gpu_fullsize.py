"""T2 at BASELINE.json's FULL sizes, in the launch configuration bench.py times (the library derives its grids from
n alone): the oracle cannot sweep 512^3 in test time, so it computes SAMPLED outputs one cell at a time through its
stateless pieces -- `orc_transport_stencil` (Eq. 30 + 32) on the cell's seven input values, then `orc_chem_cell`
(Eq. 43-48 sub-cycled), then the children mean for split cells (A14) -- and the CUDA result is compared at those
cells.  Samples cover random interior cells, the box faces / edges / corners (periodic wrap), the borders of the
transport kernel's 32 x 16 tiles and z chunks, and the source cells.  Whole-grid properties that hold at any size
(photon budget, finiteness, x in [0, 1]) are checked on every cell.
"""
import numpy as np
import pytest

import oracle as O
import paper_1508_07888_b200 as E
from workloads import make_config

pytestmark = pytest.mark.gpu

TOL = 1e-5


def _locate_sources(w):
    """A12: NGP into the leaf containing the position.  Returns {(level, cell): S[G]} with S = sum Q / dV_leaf."""
    n = w.n
    out = {}
    dx = w.L / n
    for pos, Q in zip(np.asarray(w.src_pos, np.float64), np.asarray(w.src_Q, np.float64)):
        f = pos * n
        i = np.minimum(np.floor(f).astype(np.int64), n - 1)
        o = f - i
        lvl, cell = 0, int(i[0] + n * (i[1] + n * i[2]))
        while lvl < w.n_levels:
            p = w.parent[lvl]
            k = int(np.searchsorted(p, cell))
            if k >= len(p) or p[k] != cell:
                break
            c = (o >= 0.5).astype(np.int64)
            o = 2 * o - c
            cell = 8 * k + int(c[0] + 2 * c[1] + 4 * c[2])
            lvl += 1
        dV = (dx / 2 ** lvl) ** 3
        out[(lvl, cell)] = out.get((lvl, cell), np.zeros(w.G)) + Q / dV
    return out


def _sample_cells(w, rng, n_random, extra=()):
    n = w.n
    pts = [rng.integers(0, n, (n_random, 3))]
    edge = np.array([0, 1, n - 2, n - 1])
    pts.append(np.stack(np.meshgrid(edge, edge, edge, indexing="ij"), -1).reshape(-1, 3))          # corners / edges
    face = rng.integers(0, n, (96, 3))
    for k in range(96):
        face[k, k % 3] = (0, n - 1)[(k // 3) % 2]                                                   # box faces
    pts.append(face)
    # borders of the transport kernel's tiles (x multiples of 32, y multiples of 16) and of its z chunks (any z)
    tb = rng.integers(0, n, (256, 3))
    tb[:, 0] = (rng.integers(0, max(1, n // 32), 256) * 32 + rng.choice([-1, 0, 31, 32], 256)) % n
    tb[:, 1] = (rng.integers(0, max(1, n // 16), 256) * 16 + rng.choice([-1, 0, 15, 16], 256)) % n
    pts.append(tb)
    zc = rng.integers(0, n, (256, 3))
    zc[:, 2] = (rng.integers(0, max(1, n // 8), 256) * 8 + rng.choice([-1, 0], 256)) % n
    pts.append(zc)
    p = np.concatenate(pts)
    ids = p[:, 0] + n * (p[:, 1] + n * p[:, 2])
    return np.unique(np.concatenate([ids, np.asarray(extra, np.int64)]))


def _stencil_inputs(U0g, cell, n):
    """The cell's value and its -/+ neighbours along x, y, z with periodic wrap, from the fp32 input bytes."""
    ix, iy, iz = cell % n, (cell // n) % n, cell // (n * n)
    idx = lambda a, b, c: (a % n) + n * ((b % n) + n * (c % n))
    Um = [U0g[idx(ix - 1, iy, iz)], U0g[idx(ix, iy - 1, iz)], U0g[idx(ix, iy, iz - 1)]]
    Up = [U0g[idx(ix + 1, iy, iz)], U0g[idx(ix, iy + 1, iz)], U0g[idx(ix, iy, iz + 1)]]
    return U0g[cell].astype(np.float64), np.array(Um, np.float64), np.array(Up, np.float64)


def _mean8(v):
    """A14: pairwise along x, then y, then z."""
    v = np.asarray(v, np.float64)
    return (((v[0] + v[1]) + (v[2] + v[3])) + ((v[4] + v[5]) + (v[6] + v[7]))) / 8.0


def _oracle_cell(w, phys, src, U_in, state, cell, chemistry=True, flux=None):
    """Oracle result of ONE coupled step for coarse cell `cell`.
    Returns dict(U[G,4], leaves={(level, id): (x, T, sig)}, split={(level, id): (x, T)})."""
    n, G, c, dt, dx = w.n, w.G, w.c_red, w.dt, w.L / w.n
    Ustar = np.zeros((G, 4))
    for g in range(G):
        U0, Um, Up = _stencil_inputs(U_in[g], cell, n)
        Ustar[g] = O.transport_stencil(c, dt, dx, U0, Um, Up, flux=flux)
    res = {"leaves": {}, "split": {}}
    if not chemistry:
        S = src.get((0, cell))
        if S is not None:
            Ustar[:, 0] += S * dt
        res["U"] = Ustar
        return res

    def leaf(level, cid):
        n0, x, T = (float(state[k][level][cid]) for k in ("n0", "x", "T"))
        e = O.energy(T, x, n0)
        rc, x1, e1, U1, out = O.chem_cell(phys, dt, n0, x, e, Ustar, src.get((level, cid)))
        assert rc == O.OK
        res["leaves"][(level, cid)] = (x1, O.temperature(e1, x1, n0), min(out.nsub, 65535) | (min(out.nhalv, 65535) << 16))
        res["kmax"] = max(res.get("kmax", 0.0), (1.0 - x) * n0)
        return U1, x1, e1

    def node(level, cid):
        """(U, x, e) of a cell after the step: leaf chemistry, or the mean of its eight children."""
        if level < w.n_levels:
            p = w.parent[level]
            k = int(np.searchsorted(p, cid))
            if k < len(p) and p[k] == cid:
                ch = [node(level + 1, 8 * k + j) for j in range(8)]
                U = np.zeros((G, 4))
                for g in range(G):
                    for q in range(4):
                        U[g, q] = _mean8([u[0][g, q] for u in ch])
                x = _mean8([u[1] for u in ch])
                e = _mean8([u[2] for u in ch])
                res["split"][(level, cid)] = (x, O.temperature(e, x, state["n0r"][level][cid]))
                return U, x, e
        return leaf(level, cid)

    res["U"] = node(0, cell)[0]
    return res


def _restricted_n0(w, n0):
    """Split cells' density = children mean, bottom-up (what emma_rt_init computes), in fp64 from the fp32 input."""
    r = [np.asarray(a, np.float64).copy() for a in n0]
    for l in range(w.n_levels, 0, -1):
        ch = r[l].reshape(-1, 8)
        m = (((ch[:, 0] + ch[:, 1]) + (ch[:, 2] + ch[:, 3])) + ((ch[:, 4] + ch[:, 5]) + (ch[:, 6] + ch[:, 7]))) / 8.0
        r[l - 1][np.asarray(w.parent[l - 1], np.int64)] = m
    return r


def _check_samples(w, gpu, U_in, state, cells, chemistry=True, flux=None):
    """Compare the library's state after ONE step from (U_in, state) with the oracle at the sampled coarse cells."""
    phys = O.make_phys(w.G, w.c_red, w.sigma_N, w.sigma_E, w.E_mean, otsa=w.otsa, thermal=w.thermal, e_tol=w.e_tol,
                       max_halvings=w.max_halvings)
    src = _locate_sources(w) if w.src_pos is not None else {}
    state = dict(state)
    state["n0r"] = _restricted_n0(w, state["n0"])
    Ug = [gpu.read(E.FIELD_U, 0, g) for g in range(w.G)]
    Nmax = [float(np.abs(u[:, 0]).max()) for u in Ug]
    lv = range(w.n_levels + 1)
    xg = [gpu.read(E.FIELD_X, l) for l in lv] if chemistry else None
    Tg = [gpu.read(E.FIELD_T, l) for l in lv] if chemistry else None
    sg = [gpu.read(E.FIELD_SUBCYCLES, l) for l in lv] if chemistry else None
    eN = eF = ex = eT = 0.0
    flips = n_leaves = n_split = 0
    for cell in cells:
        cell = int(cell)
        r = _oracle_cell(w, phys, src, U_in, state, cell, chemistry, flux)
        flipped = False
        for (l, cid), (x1, T1, sig) in r["leaves"].items():
            n_leaves += 1
            if int(sg[l][cid]) != sig:                                  # A9: several results are correct
                flips += 1
                flipped = True
                assert abs(xg[l][cid] - x1) <= 2e-2 * max(x1, 1e-3) and abs(Tg[l][cid] - T1) <= 2e-2 * T1
                continue
            ex = max(ex, abs(float(xg[l][cid]) - x1) / x1)
            eT = max(eT, abs(float(Tg[l][cid]) - T1) / T1)
        if flipped:
            continue
        for (l, cid), (x1, T1) in r["split"].items():
            n_split += 1
            ex = max(ex, abs(float(xg[l][cid]) - x1) / x1)
            eT = max(eT, abs(float(Tg[l][cid]) - T1) / T1)
        for g in range(w.G):
            ref = r["U"][g]
            got = Ug[g][cell].astype(np.float64)
            sc = max(abs(ref[0]), 1e-12 * Nmax[g], 1e-300)
            # coupled step: tolerance x the condition number of Eq. 43 w.r.t. the neutral fraction (tests/parity.py)
            # (for a split cell: of its most opaque leaf)
            cond = 1.0 + w.c_red * w.sigma_N[g] * r["kmax"] * w.dt if chemistry else 1.0
            eN = max(eN, abs(got[0] - ref[0]) / sc / cond)
            eF = max(eF, float(np.abs(got[1:] - ref[1:]).max()) / (w.c_red * sc) / cond)
    return {"N": eN, "F": eF, "x": ex, "T": eT, "flips": flips, "leaves": n_leaves, "split": n_split, "cells": len(cells)}


def _whole_grid_properties(w, gpu):
    for l in range(w.n_levels + 1):
        x = gpu.read(E.FIELD_X, l)
        T = gpu.read(E.FIELD_T, l)
        assert np.isfinite(x).all() and np.isfinite(T).all()
        assert x.min() >= 0.0 and x.max() <= 1.0 and T.min() > 0.0
    for g in range(w.G):
        U = gpu.read(E.FIELD_U, 0, g)
        assert np.isfinite(U).all()
        assert (U[:, 0] >= 0).all()
        # M1 realisability: |F| <= c N up to rounding of an fp32 update
        assert (np.linalg.norm(U[:, 1:].astype(np.float64), axis=1) <= w.c_red * U[:, 0].astype(np.float64) * (1 + 1e-4) + 1e-30).all()


def test_config5_full_512_sampled_and_budget():
    """BASELINE config 5 (b) at 512^3 x 3 groups, the workload and launch configuration of bench.py."""
    w = make_config(5)
    assert w.n == 512 and w.G == 3
    rng = np.random.default_rng(5120)
    src_cells = [c for (l, c) in _locate_sources(w)][:256]
    cells = _sample_cells(w, rng, 3000, extra=src_cells)
    state = {"n0": w.n0, "x": w.x, "T": w.T}

    # (i) transport + sources only: the M1 update whose outputs ARE N and F
    gpu = E.EmmaRT(w, chemistry=0)
    rc, d0 = gpu.step(w.dt, 0)
    rc, d1 = gpu.step(w.dt, 1)
    assert rc == E.OK and d1["n_nonfinite"] == 0
    rep = _check_samples(w, gpu, w.U0, state, cells, chemistry=False)
    print("cfg5 512^3 transport-only, sampled:", rep)
    assert rep["N"] <= TOL and rep["F"] <= TOL, rep
    # periodic box: photons are conserved by the transport to rounding; sources add sum Q dt
    inj = float(np.sum(w.src_Q)) * w.dt
    assert d1["photons_injected"] == pytest.approx(inj, rel=1e-6)
    assert d1["photons_total"] - d0["photons_total"] == pytest.approx(inj, abs=1e-6 * d1["photons_total"])
    gpu.close()

    # (ii) the coupled step
    gpu = E.EmmaRT(w, record_subcycles=1)
    rc, d1 = gpu.step(w.dt, 1)
    assert rc == E.OK, gpu.last_error()
    rep = _check_samples(w, gpu, w.U0, state, cells)
    print("cfg5 512^3 coupled step, sampled:", rep, {k: d1[k] for k in ("subcycles_max", "n_deferred")})
    assert rep["flips"] <= max(2, 1e-3 * rep["leaves"]), rep
    assert rep["N"] <= TOL and rep["F"] <= TOL and rep["x"] <= TOL and rep["T"] <= TOL, rep
    assert d1["subcycles_max"] > 1 and d1["n_deferred"] > 0              # the divergent tail is exercised at this size
    # photon budget of every further step (A15), whole grid, in fp64 on the device
    prev = d1["photons_total"]
    for _ in range(4):
        rc, d = gpu.step(w.dt, 1)
        assert rc == E.OK
        rhs = d["photons_injected"] - d["photons_absorbed"] + d["photons_recomb_emitted"] - d["photons_outflow"]
        assert abs((d["photons_total"] - prev) - rhs) <= 1e-6 * d["photons_total"]
        prev = d["photons_total"]
    _whole_grid_properties(w, gpu)
    gpu.close()


def test_config5_full_512_hll_transport_sampled():
    """The HLL flux (reading A19) at 512^3 x 3 groups, the launch configuration bench.py times as `transport_only_hll`:
    sampled cells against the oracle's HLL stencil, photons conserved on the periodic box."""
    w = make_config(5)
    rng = np.random.default_rng(5121)
    cells = _sample_cells(w, rng, 3000)
    gpu = E.EmmaRT(w, chemistry=0, flux=E.FLUX_HLL)
    rc, d0 = gpu.step(w.dt, 0)
    rc, d1 = gpu.step(w.dt, 1)
    assert rc == E.OK and d1["n_nonfinite"] == 0
    rep = _check_samples(w, gpu, w.U0, {"n0": w.n0, "x": w.x, "T": w.T}, cells, chemistry=False, flux=O.FLUX_HLL)
    print("cfg5 512^3 HLL transport, sampled:", rep)
    assert rep["N"] <= TOL and rep["F"] <= TOL, rep
    inj = float(np.sum(w.src_Q)) * w.dt
    assert d1["photons_total"] - d0["photons_total"] == pytest.approx(inj, abs=1e-6 * d1["photons_total"])
    gpu.close()


def test_config4_full_256_crta_sampled():
    """BASELINE config 4 at full size: 256^3 coarse cells + 2 refined levels (~30 M leaves), 3 groups, CRTA.  The box
    starts dark, so the library first advances 6 steps; its state is read back and ONE further step from exactly that
    state is compared with the oracle at sampled coarse cells (unrefined, split once, split twice, source-hosting)."""
    w = make_config(4)
    assert w.n == 256 and w.n_levels == 2
    assert 2.5e7 < w.n_leaves < 3.5e7
    gpu = E.EmmaRT(w, record_subcycles=1)
    prev = None
    for _ in range(6):
        rc, d = gpu.step(w.dt, 1)
        assert rc == E.OK, gpu.last_error()
        if prev is not None:
            rhs = d["photons_injected"] - d["photons_absorbed"] + d["photons_recomb_emitted"] - d["photons_outflow"]
            assert abs((d["photons_total"] - prev) - rhs) <= 1e-6 * max(d["photons_total"], d["photons_injected"])
        prev = d["photons_total"]
    U_in = [gpu.read(E.FIELD_U, 0, g) for g in range(w.G)]
    state = {"n0": w.n0, "x": [gpu.read(E.FIELD_X, l) for l in range(3)], "T": [gpu.read(E.FIELD_T, l) for l in range(3)]}
    gpu.close()
    w.U0, w.x, w.T = U_in, state["x"], state["T"]

    rng = np.random.default_rng(4256)
    src = _locate_sources(w)
    p1, p2 = (np.asarray(p, np.int64) for p in w.parent)
    src_coarse = np.unique([p1[p2[c // 8] // 8] for (l, c) in src if l == 2])[:48]
    lit = np.flatnonzero(U_in[0][:, 0] > 1e-6 * U_in[0][:, 0].max())     # cells the light has reached
    extra = np.concatenate([src_coarse, rng.choice(p1, 96, replace=False), p1[p2[rng.choice(len(p2), 48)] // 8],
                            rng.choice(lit, min(512, len(lit)), replace=False)])
    cells = _sample_cells(w, rng, 512, extra=extra)
    gpu = E.EmmaRT(w, record_subcycles=1)
    rc, d = gpu.step(w.dt, 1)
    assert rc == E.OK, gpu.last_error()
    rep = _check_samples(w, gpu, U_in, state, cells)
    print("cfg4 256^3 + 2 levels, coupled CRTA step, sampled:", rep, {k: d[k] for k in ("subcycles_max", "n_deferred")})
    assert rep["split"] >= 100 and rep["leaves"] > 2 * rep["cells"]
    assert rep["flips"] <= max(2, 1e-3 * rep["leaves"]), rep
    assert rep["N"] <= TOL and rep["F"] <= TOL and rep["x"] <= TOL and rep["T"] <= TOL, rep
    _whole_grid_properties(w, gpu)
    gpu.close()
