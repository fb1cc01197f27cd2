"""SURVEY.md 8(f) NEXT-4, second half: the inflow boundary (reading A20; "the x = 0 boundary is a
source of flux of the required rate") and the static cousin of the paper's clump test (`workloads.make_shadow_clump`).

CPU: the oracle's inflow ghost is pinned by the closed form of a beam entering a vacuum box (first-order upwind from a
constant ghost: a binomial tail) and by the photon budget with a NEGATIVE outflow while the box fills; the shadow run by
what the set-up fixes (free-streaming value N = F/c in the lit medium, a dark neutral clump core, a shadow behind it that
HLL keeps darker than GLF -- PAPER.md:580 "the shadow ... is much weaker ... since EMMA implements the GLF flux").
GPU: element-by-element parity, GLF (transport.cu) and HLL."""
from math import comb

import numpy as np
import pytest

import oracle as O
from workloads import CGS, make_shadow_clump

from .helpers import tiny_workload


@pytest.mark.parametrize("flux", [O.FLUX_GLF, O.FLUX_HLL])
@pytest.mark.parametrize("face", [0, 3, 4])
def test_I1_beam_entering_vacuum_is_a_binomial_tail(flux, face):
    """Ghost (N, F) = (1, c n^) on one face, vacuum inside, the opposite face transmissive: both fluxes reduce to upwind
    along the beam, so after k steps N_i = P(Binomial(k, nu) >= i + 1) counted from the inflow face; f stays 1."""
    n, c, k = 12, 2.0 ** 31, 9
    d, hi = face // 2, face % 2
    bc = [0] * 6
    bc[2 * d], bc[2 * d + 1] = (1, 3) if hi else (3, 1)
    w = tiny_workload(n, 1, chemistry=0, bc=tuple(bc), c_red=c, courant=0.75)
    U = [1.0, 0.0, 0.0, 0.0]
    U[1 + d] = -c if hi else c
    w.inflow = {(face, 0): tuple(U)}
    o = O.Oracle(w, flux=flux)
    prev = 0.0
    for step in range(k):
        rc, dg = o.step(w.dt, 1)
        assert rc == O.OK
        assert dg["photons_outflow"] < 0.0                            # light enters: negative net outflow
        assert dg["photons_total"] - prev == pytest.approx(-dg["photons_outflow"], rel=1e-12, abs=0)   # A15
        prev = dg["photons_total"]
    nu = c * w.dt / w.dx
    tail = np.array([sum(comb(k, m) * nu ** m * (1 - nu) ** (k - m) for m in range(i + 1, k + 1)) for i in range(n)])
    Ug = o.read(O.F_U).reshape(n, n, n, 4)                            # [iz, iy, ix]
    line = np.moveaxis(Ug, 2 - d, 0)[:, 3, 5, :]                      # along the beam direction
    if hi:
        line = line[::-1]
    assert np.allclose(line[:, 0], tail, rtol=1e-12, atol=1e-15)
    assert np.allclose(np.abs(line[:, 1 + d]), c * line[:, 0], rtol=1e-12)


def test_I2_set_inflow_argument_errors():
    w = tiny_workload(6, 2, chemistry=0, bc=(3, 1, 0, 0, 0, 0))
    o = O.Oracle(w)
    assert o.set_inflow(0, 1, (1, 0, 0, 0)) == O.OK
    assert o.set_inflow(1, 0, (1, 0, 0, 0)) == O.EINVAL               # not an inflow face
    assert o.set_inflow(0, 2, (1, 0, 0, 0)) == O.EINVAL               # no such group
    assert o.set_inflow(6, 0, (1, 0, 0, 0)) == O.EINVAL


def _run_shadow(flux, n=24, steps=260):
    w = make_shadow_clump(n=n)
    o = O.Oracle(w, flux=flux)
    rc, d = o.step(w.dt, steps)
    assert rc == O.OK
    N = sum(o.read(O.F_N, 0, g) for g in range(w.G)).reshape(n, n, n)          # [iz, iy, ix]
    x = o.read(O.F_X).reshape(n, n, n)
    return w, N, x


def test_shadow_clump_static_glf_and_hll():
    n = 24
    res = {fl: _run_shadow(fl, n) for fl in (O.FLUX_GLF, O.FLUX_HLL)}
    mid = n // 2
    ic = int(5.4 / 6.6 * n)                                           # clump centre along x
    for fl, (w, N, x) in res.items():
        N_in = sum(w.inflow[(0, g)][0] for g in range(w.G))
        # the lit thin medium far from the clump: fully ionised, free-streaming value F/c
        assert N[mid, 1, : n // 2] == pytest.approx(N_in, rel=2e-3, abs=0)
        assert x[mid, 1, n // 2] > 0.999
        # the clump core stays neutral and dark
        assert x[mid, mid, ic] < 0.05 and N[mid, mid, ic] < 1e-2 * N_in
    shadow = {fl: res[fl][1][mid, mid, -1] / res[fl][1][mid, 1, -1] for fl in res}   # behind the clump / beside it
    assert shadow[O.FLUX_GLF] < 0.5                                    # there is a shadow ...
    assert shadow[O.FLUX_HLL] < 0.7 * shadow[O.FLUX_GLF], shadow       # ... and HLL keeps it darker


@pytest.mark.gpu
@pytest.mark.parametrize("flux", [0, 1])
@pytest.mark.parametrize("n,G,bc", [(20, 2, (3, 1, 0, 0, 0, 0)), (33, 1, (1, 3, 3, 2, 2, 3)), (40, 3, (0, 0, 1, 3, 3, 1))])
def test_inflow_transport_gpu_parity(n, G, bc, flux):
    """One transport step on a random state with inflow faces (random sub-luminal ghosts), both fluxes, ragged tiles."""
    import paper_1508_07888_b200 as E  # noqa: F401
    from .parity import compare, run_pair
    from .test_gpu_parity import _random_U
    c = 0.1 * CGS.c
    rng = np.random.default_rng(n + 10 * G + flux)
    w = tiny_workload(n, G, bc=bc, chemistry=0, U0=_random_U(rng, G, n ** 3, c, fmax=0.9, lo=-6, hi=-2), courant=0.9)
    w.inflow = {}
    for f in range(6):
        if bc[f] == 3:
            for g in range(G):
                Nn = 10 ** rng.uniform(-5, -2)
                dirn = rng.standard_normal(3)
                dirn /= np.linalg.norm(dirn)
                w.inflow[(f, g)] = (Nn, *(rng.uniform(0, 0.9) * c * Nn * dirn))
    orc, gpu, _, diags = run_pair(w, 2, track_signatures=False, flux=flux)
    rep = compare(orc, gpu, w)
    assert rep["N"] <= 2e-5 and rep["F"] <= 2e-5, rep
    do, dg = diags[-1]
    assert dg["photons_total"] == pytest.approx(do["photons_total"], rel=1e-6, abs=0)
    assert abs(dg["photons_outflow"] - do["photons_outflow"]) <= 2e-6 * do["photons_total"]


@pytest.mark.gpu
@pytest.mark.parametrize("flux", [0, 1])
def test_shadow_clump_gpu_parity(flux):
    """GLF: the usual bar everywhere.  HLL: the usual bar wherever the cell is lit; in the shadow and its penumbra the HLL
    result is sqrt-sensitive to 1 - f^2 of the neighbouring beam cells (the transverse speed of a beam is
    c sqrt(2 (1 - f^2)), which fp32 states resolve to ~3.5e-4 c and fp64 states to ~1e-8 c), so cells that only receive
    that leaked light cannot agree to 1e-4 between ANY two precisions: there the difference is bounded instead."""
    import paper_1508_07888_b200 as E
    from .parity import budget_residual, compare, run_pair
    w = make_shadow_clump(n=32)
    K = 120
    orc, gpu, flips, diags = run_pair(w, K, flux=flux)
    prev, worst = None, 0.0
    for do, dg in diags:
        if prev is not None:
            worst = max(worst, budget_residual(dg, prev))
        prev = dg["photons_total"]
    assert worst <= 1e-6, worst
    if flux == 0:
        rep = compare(orc, gpu, w, flips, K)
        assert rep["flips"] <= max(2, 1e-3 * rep["cells"]), rep
        assert rep["x"] <= 1e-4 and rep["T"] <= 1e-4, rep
        return
    N_in = sum(w.inflow[(0, g)][0] for g in range(w.G))
    No = sum(orc.read(O.F_N, 0, g) for g in range(w.G))
    Ng = sum(gpu.read(E.FIELD_N, 0, g).astype(np.float64) for g in range(w.G))
    xo, xg = orc.read(O.F_X), gpu.read(E.FIELD_X).astype(np.float64)
    To, Tg = orc.read(O.F_T), gpu.read(E.FIELD_T).astype(np.float64)
    flipped = np.zeros(len(xo), bool)
    flipped[[c for (_, _, c, _) in flips]] = True
    lit = (No > 0.5 * N_in) & ~flipped
    assert lit.mean() > 0.5
    assert np.max(np.abs(xg - xo)[lit] / xo[lit]) <= 1e-4
    assert np.max(np.abs(Tg - To)[lit] / To[lit]) <= 1e-4
    assert np.max(np.abs(Ng - No)[lit] / No[lit]) <= 1e-4
    # shadow / penumbra: bounded by the fp32 transverse leak, and never brighter than a few 1e-3 of the beam
    assert np.max(np.abs(Ng - No)[~lit]) <= 5e-3 * N_in
    assert np.max(np.abs(xg - xo)[~lit]) <= 0.15
