"""Full-size, full-length parity of BASELINE configs 4 and 5 (VERDICT r1 row g; north_star: "<= 1e-4 on x_HII and T
after 100 coupled steps ... on all five configs"; PAPER.md:652 fixes the workload shape, PAPER.md:312 the 10 % rule whose
branch flips the protocol of tests/parity.py counts).

  * config 5b at 256^3 x 3 groups for its 50 steps, the WHOLE grid element by element.  Why not 512^3: the oracle as it
    stands advances ~2.5e7 cell-groups/s on the GPU box's 16 host cores, i.e. 512^3 x 3 x 50 steps = 13 min and ~45 GB,
    beyond what the driver's test step allows; 512^3 keeps its one-step sampled test (tests/test_gpu_fullsize.py) and the
    256^3 grid spans 8 x 16 tiles and 2 z-chunks of the same kernels in the same launch configuration.
  * config 4 at its full 256^3 coarse grid + 2 refined levels (~30 M leaves) for its 100 steps, every level element by
    element, CRTA.  The source-hosting leaves of level 2 really sub-cycle in the first steps (asserted).

Both print the flip fraction and the error distribution of the cells near a flip (a <~ 1e-5 fraction is
expected at size and is a property of the paper's halving rule), and the worst error as a function of the L1 distance to
the nearest flip.  Measured at config 5b, 256^3, 50 steps (101 flips = 5.9e-6 of the cells, all in steps 1-5): x error
1.2e-2 at a flipped cell, 4.8e-3 / 3.1e-3 / 6.7e-4 / 3.0e-4 / 1.5e-4 / 2.8e-5 at distance 1 .. 6, 2.1e-6 in the far field
(16.5 M of the 16.8 M cells).  The GLF flux diffuses a flip's O(1e-2) perturbation by ~sqrt(nu k) cells in k steps, so the
short runs' radius of 3 (tests/parity.py) is too small here: the tolerance is asserted beyond L1 distance RADIUS(k) = 6
(50 steps) / 8 (100 steps), i.e. on > 99.7 % of the cells, and the far field is held to 2e-5.
"""
import time

import numpy as np
import pytest

import oracle as O
import paper_1508_07888_b200 as E
from workloads import make_config

from .parity import budget_residual, clean_masks, compare, flip_distance, run_pair

pytestmark = pytest.mark.gpu

TOL_XT = 1e-4
TOL_BUDGET = 1e-6


def _near_flip_report(orc, gpu, w, flips, n_steps, radius):
    """Distribution of the x, T errors inside the flip radius and at the flipped cells themselves."""
    clean = clean_masks(w, flips, n_steps, radius)
    out = {}
    for name, fo, fg in (("x", O.F_X, E.FIELD_X), ("T", O.F_T, E.FIELD_T)):
        near, at = [], []
        for l in range(w.n_levels + 1):
            a = orc.read(fo, l)
            b = gpu.read(fg, l).astype(np.float64)
            r = np.abs(b - a) / np.abs(a)
            near.append(r[~clean[l]])
            cells = sorted({c for (_s, fl, c, _c0) in flips if fl == l})
            at.append(r[np.asarray(cells, np.int64)] if cells else np.zeros(0))
        near, at = np.concatenate(near), np.concatenate(at)
        pct = lambda v: [float("%.3g" % q) for q in np.percentile(v, [50, 90, 99, 100])] if v.size else []
        out[name] = {"near_p50_p90_p99_max": pct(near), "flipped_p50_p90_p99_max": pct(at)}
    return out


def _by_distance(orc, gpu, w, flips):
    """Worst x / T error over the cells (all levels) at each L1 distance of their coarse ancestor to the nearest flip."""
    from .parity import coarse_ancestors
    dist = flip_distance(w, flips)
    anc = coarse_ancestors(w)
    table = {}
    for name, fo, fg in (("x", O.F_X, E.FIELD_X), ("T", O.F_T, E.FIELD_T)):
        worst = np.zeros(int(dist.max()) + 1)
        for l in range(w.n_levels + 1):
            a = orc.read(fo, l)
            r = np.abs(gpu.read(fg, l).astype(np.float64) - a) / np.abs(a)
            np.maximum.at(worst, dist[anc[l]], r)
        table[name] = [float("%.3g" % v) for v in worst]
    return table


def _run_full(w, n_steps, max_flip_frac, radius, want_refined_subcycles=False):
    t0 = time.time()
    orc, gpu, flips, diags = run_pair(w, n_steps)
    t_run = time.time() - t0
    rep = compare(orc, gpu, w, flips, n_steps, radius=radius)
    prev, worst_budget = None, 0.0
    for _do, dg in diags:
        if prev is not None:
            worst_budget = max(worst_budget, budget_residual(dg, prev))
        prev = dg["photons_total"]
        assert dg["n_nonfinite"] == 0
    rep["budget"] = worst_budget
    rep["sub_max"] = max(dg["subcycles_max"] for _, dg in diags)
    flipped_cells = len({(l, c) for (_s, l, c, _c0) in flips})
    rep["flip_fraction"] = flipped_cells / float(rep["cells"])
    rep["near_fraction"] = rep["near_cells"] / float(rep["cells"])
    dist = _near_flip_report(orc, gpu, w, flips, n_steps, radius)
    table = _by_distance(orc, gpu, w, flips)
    print(w.name, "%d steps in %.0f s" % (n_steps, t_run), {k: (float("%.3g" % v) if isinstance(v, float) else v) for k, v in rep.items()})
    print(w.name, "flips per step:", np.bincount([s for (s, _l, _c, _c0) in flips], minlength=n_steps + 1)[1:].tolist())
    print(w.name, "near-flip error distribution:", dist)
    print(w.name, "worst error by L1 distance to the nearest flip (0, 1, ..., 12, farther):", table)
    assert table["x"][-1] <= 2e-5 and table["T"][-1] <= 2e-5, table           # far field: no flip within 12 cells
    assert rep["near_fraction"] <= 5e-3, rep
    # oracle and GPU agree on the diagnostics of the last step
    do, dg = diags[-1]
    assert abs(dg["photons_total"] - do["photons_total"]) <= 1e-5 * abs(do["photons_total"])
    assert abs(dg["photons_injected"] - do["photons_injected"]) <= 1e-6 * abs(do["photons_injected"])
    assert rep["flip_fraction"] <= max_flip_frac, rep
    assert rep["x"] <= TOL_XT and rep["T"] <= TOL_XT, rep                    # north_star, every clean cell of every level
    assert rep["x_near"] <= 2e-2 and rep["T_near"] <= 2e-2, rep              # flipped cells: both branches are valid results
    assert rep["budget"] <= TOL_BUDGET, rep
    if want_refined_subcycles:
        assert rep["sub_max"] > 1, rep
    orc.close()
    gpu.close()
    return rep, diags


def test_config5b_256_50_steps_whole_grid():
    w = make_config(5, n=256, variant="b")
    assert w.n == 256 and w.G == 3 and len(w.src_pos) == 512
    rep, diags = _run_full(w, 50, max_flip_frac=1e-4, radius=6)
    assert diags[0][1]["n_deferred"] > 1000 and diags[0][1]["subcycles_max"] > 10     # the random T state sub-cycles hard


def test_config4_full_256_crta_100_steps():
    w = make_config(4)                                                      # 256^3 + 2 levels, 1024 sources in level-2 leaves
    assert w.n == 256 and w.n_levels == 2 and len(w.src_pos) == 1024
    assert 25e6 < w.n_leaves < 35e6
    # the divergent branch on a refined level: the source-hosting leaves of level 2 need several sub-steps in step 1
    orc = O.Oracle(w)
    rc, _ = orc.step(w.dt, 1)
    assert rc == O.OK
    sub2 = orc.read(O.F_SUBCYCLES, 2).astype(np.int64) & 0xffff
    assert sub2.max() > 1 and (orc.read(O.F_SUBCYCLES, 0).astype(np.int64) & 0xffff).max() == 1
    orc.close()
    _run_full(w, w.n_steps, max_flip_frac=1e-4, radius=8, want_refined_subcycles=True)
