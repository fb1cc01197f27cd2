"""T2: the two schedules of the coupled step (emma_rt_set_schedule) against the fp64 oracle and against each other.

fused = 1 (default): transport (Eq. 30, 32) and the first trip of the sub-cycle loop (Eq. 43-48) in ONE pass
(csrc/fused.cu); fused = 0: a transport pass followed by a chemistry pass.  Both must meet north_star's tolerances on
the same seeded inputs; every other GPU test runs the default (fused) schedule, this file also pins the unfused one and
the cases that are special to the fused kernel: non-periodic faces WITH chemistry (its boundary-condition variant),
ragged tiles in x and y, one plane per z-chunk, refined coarse cells (CRTA) and every group count.
"""
import os

import numpy as np
import pytest

import paper_1508_07888_b200 as E
from workloads import CGS, make_config

from .helpers import tiny_workload
from .parity import absorption_condition, budget_residual, compare, run_pair
from .test_gpu_parity import _random_U

pytestmark = pytest.mark.gpu

TOL_NF, TOL_XT, TOL_BUDGET = 1e-5, 1e-4, 1e-6
C_RED = 0.1 * CGS.c


def _random_state(n, G, seed, hot=False):
    rng = np.random.default_rng(seed)
    nc = n ** 3
    n0 = (10 ** rng.uniform(-5, -2, nc)).astype(np.float32)
    x = np.minimum(10 ** rng.uniform(-4, 0, nc), 0.999999).astype(np.float32)
    T = (10 ** rng.uniform(2, 4.7 if hot else 4.0, nc)).astype(np.float32)
    pos = rng.random((4, 3))
    Q = 10 ** rng.uniform(47, 49, (4, G))
    return rng, dict(n0=n0, x=x, T=T, U0=_random_U(rng, G, nc, C_RED, fmax=0.9, lo=-7, hi=-2), src_pos=pos, src_Q=Q)


CASES = [(8, 1, (0,) * 6), (20, 2, (1, 2, 0, 0, 2, 1)), (33, 3, (2, 2, 1, 1, 0, 0)), (40, 4, (0,) * 6),
         (50, 1, (1, 1, 1, 1, 1, 1)), (36, 3, (0, 0, 2, 1, 1, 2))]


@pytest.mark.parametrize("fused", [0, 1])
@pytest.mark.parametrize("n,G,bc", CASES)
def test_coupled_one_step_both_schedules(n, G, bc, fused):
    """One coupled step from a random state, every boundary condition, ragged tiles (n not a multiple of 32 / 16)."""
    _, kw = _random_state(n, G, 1000 + 13 * n + G)
    w = tiny_workload(n, G, bc=bc, **kw)
    orc, gpu, flips, diags = run_pair(w, 1, fused=fused)
    rep = compare(orc, gpu, w, flips, 1, nf_cond=absorption_condition(w, w.dt))
    do, dg = diags[0]
    assert rep["flips"] <= max(2, 1e-4 * rep["cells"]), rep
    assert rep["x"] <= TOL_XT and rep["T"] <= TOL_XT and rep["xn"] <= TOL_XT, rep
    assert rep["N"] <= 5e-5 and rep["F"] <= 5e-5, rep
    for k in ("photons_total", "photons_injected", "photons_absorbed"):
        assert dg[k] == pytest.approx(do[k], rel=2e-5), k
    if any(b == 1 for b in bc):
        assert dg["photons_outflow"] == pytest.approx(do["photons_outflow"], rel=1e-4, abs=1e-9 * do["photons_total"])
    assert abs(dg["subcycles_total"] - do["subcycles_total"]) <= 1e-3 * do["subcycles_total"]
    kinds = gpu.profile(False)
    gpu.close()


def test_schedules_launch_what_they_say():
    """fused = 1 launches the fused kernel and no separate transport / chem_main pass; fused = 0 the opposite."""
    _, kw = _random_state(24, 3, 5)
    w = tiny_workload(24, 3, **kw)
    for fused in (0, 1):
        gpu = E.EmmaRT(w, fused=fused)
        gpu.profile(True)
        rc, _ = gpu.step(w.dt, 3)
        assert rc == E.OK
        k = gpu.profile(False)
        if fused:
            assert k["fused"][1] == 3 and k["transport"][1] == 0 and k["chem_main"][1] == 0, k
        else:
            assert k["fused"][1] == 0 and k["transport"][1] == 3 and k["chem_main"][1] == 3, k
        gpu.close()
    gpu = E.EmmaRT(w)
    assert E.lib().emma_rt_set_schedule(gpu.h, 2) == E.EINVAL
    gpu.close()


def test_schedules_agree_with_each_other():
    """Same inputs, both schedules, 20 coupled steps: the same arithmetic in a different summation order -> agreement
    far inside the parity tolerance wherever the sub-cycle signatures agree; identical photon budgets to 1e-6."""
    w = make_config(3, n=40)
    out = []
    for fused in (0, 1):
        gpu = E.EmmaRT(w, record_subcycles=1, fused=fused)
        rc, d = gpu.step(w.dt, 20)
        assert rc == E.OK
        out.append((np.stack([gpu.read(E.FIELD_U, 0, g) for g in range(w.G)]), gpu.read(E.FIELD_X), gpu.read(E.FIELD_T),
                    gpu.read(E.FIELD_SUBCYCLES), d))
        gpu.close()
    (U0, x0, T0, s0, d0), (U1, x1, T1, s1, d1) = out
    same = s0 == s1
    assert same.mean() > 0.999
    assert np.max(np.abs(x1 - x0)[same] / np.maximum(x0[same], 1e-30)) < 2e-5
    assert np.max(np.abs(T1 - T0)[same] / T0[same]) < 2e-5
    assert d1["photons_total"] == pytest.approx(d0["photons_total"], rel=1e-5)
    assert d1["photons_absorbed"] == pytest.approx(d0["photons_absorbed"], rel=1e-5)


@pytest.mark.parametrize("nzc", [0, 40])
def test_fused_z_chunking(nzc):
    """The fused march with many short z-chunks (one plane per CTA at nzc = n) equals the oracle like the default."""
    _, kw = _random_state(40, 2, 77)
    w = tiny_workload(40, 2, bc=(1, 2, 0, 0, 2, 1), **kw)
    old = os.environ.get("EMMA_RT_TUNE_NZC")
    try:
        if nzc:
            os.environ["EMMA_RT_TUNE_NZC"] = str(nzc)
        orc, gpu, flips, diags = run_pair(w, 2, fused=1)
    finally:
        if old is None:
            os.environ.pop("EMMA_RT_TUNE_NZC", None)
        else:
            os.environ["EMMA_RT_TUNE_NZC"] = old
    rep = compare(orc, gpu, w, flips, 2, nf_cond=absorption_condition(w, w.dt))
    assert rep["x"] <= TOL_XT and rep["T"] <= TOL_XT, rep
    assert rep["N"] <= 5e-5 and rep["F"] <= 5e-5, rep


@pytest.mark.parametrize("k,n,steps", [(1, 32, 100), (4, 48, 60)])
def test_configs_unfused_schedule(k, n, steps):
    """Config 1 (Stroemgren) and config 4 (CRTA, refined cells) through the UNFUSED schedule; the default-schedule
    runs of the same configs are in test_gpu_parity.py."""
    w = make_config(k, n=n) if k == 1 else make_config(k, n=n, n_src=8)
    orc, gpu, flips, diags = run_pair(w, steps, fused=0)
    rep = compare(orc, gpu, w, flips, steps)
    prev, worst = None, 0.0
    for do, dg in diags:
        if prev is not None:
            worst = max(worst, budget_residual(dg, prev))
        prev = dg["photons_total"]
    assert rep["flips"] <= max(1, 1e-3 * rep["cells"]), rep
    assert rep["x"] <= TOL_XT and rep["T"] <= TOL_XT, rep
    assert worst <= TOL_BUDGET, worst
