"""T2: the HLL interface flux (emma_rt_set_flux, reading A19) against the fp64 oracle.

The oracle's HLL is pinned on the CPU (tests/test_oracle_pins.py H1-H7: eigenvalues of the finite-difference flux
Jacobian, limits, worked example, exact upwind for a beam, brute-force transcription).  Here the CUDA kernel
(csrc/transport_hll.cu) is compared with it element by element: every boundary type, ragged tiles, several z-chunks,
every group count, transport alone and inside the coupled step.
"""
import numpy as np
import pytest

import oracle as O
import paper_1508_07888_b200 as E
from workloads import CGS, make_config

from .helpers import tiny_workload
from .parity import absorption_condition, budget_residual, compare, run_pair
from .test_gpu_parity import BCS, _random_U

pytestmark = pytest.mark.gpu

TOL_NF, TOL_XT, TOL_BUDGET = 1e-5, 1e-4, 1e-6
C_RED = 0.1 * CGS.c
HLL = E.FLUX_HLL


@pytest.mark.parametrize("n,G,bc", BCS + [(36, 4, (2, 1, 1, 2, 0, 0)), (32, 2, (2, 1, 0, 0, 1, 2)), (63, 1, (0,) * 6),
                                          (31, 3, (1, 2, 2, 1, 0, 0)), (62, 1, (2, 2, 0, 0, 0, 0)), (17, 2, (0,) * 6)])
def test_hll_transport_one_step(n, G, bc):
    """One HLL transport step on a config-5b-like state (N over 5 decades, f in [0, 0.9]); north_star tolerance, A17 norms.
    The kernel's tiles are 31 cells wide and a thread owns two rows: n = 31, 62 (exact tiles), 32, 63 (a last tile ONE cell
    wide), 33, 17 (an odd last row: the unpaired-row path), with open, reflective and periodic faces on the tile edges."""
    rng = np.random.default_rng(n * 10 + G + 7)
    w = tiny_workload(n, G, bc=bc, chemistry=0, U0=_random_U(rng, G, n ** 3, C_RED, fmax=0.9, lo=-7, hi=-2), courant=0.9)
    orc, gpu, _, diags = run_pair(w, 1, track_signatures=False, flux=HLL)
    rep = compare(orc, gpu, w)
    assert rep["N"] <= TOL_NF and rep["F"] <= TOL_NF, rep
    do, dg = diags[0]
    assert dg["photons_total"] == pytest.approx(do["photons_total"], rel=1e-6)
    assert abs(dg["photons_outflow"] - do["photons_outflow"]) <= 1e-6 * do["photons_total"]


def test_hll_differs_from_glf_and_flux_is_switchable():
    """The same handle run with GLF and with HLL gives different fields (the option is really taken), each matching
    its own oracle; an unknown flux is rejected."""
    n, G = 24, 2
    rng = np.random.default_rng(3)
    w = tiny_workload(n, G, chemistry=0, U0=_random_U(rng, G, n ** 3, C_RED, fmax=0.9, lo=-5, hi=-2))
    out = {}
    for fl in (E.FLUX_GLF, E.FLUX_HLL):
        orc, gpu, _, _ = run_pair(w, 3, track_signatures=False, flux=fl, block=3)
        rep = compare(orc, gpu, w)
        assert rep["N"] <= 3e-5 and rep["F"] <= 3e-5, rep
        out[fl] = gpu.read(E.FIELD_N, 0, 0)
        assert E.lib().emma_rt_set_flux(gpu.h, 7) == E.EINVAL
        gpu.close()
    assert np.abs(out[E.FLUX_HLL] - out[E.FLUX_GLF]).max() > 1e-3 * out[E.FLUX_GLF].max()


def test_hll_dark_cells_vacuum_and_clipped_flux():
    """Dark cells (N = 0: f = 0, l = -/+ 1/sqrt 3), denormal N, and reduced fluxes above 1 (clip of A2) stay finite and
    match the oracle relative to the magnitude of what is summed (the stencil maximum, as in the GLF adversarial test)."""
    n, G = 20, 1
    rng = np.random.default_rng(9)
    U0 = _random_U(rng, G, n ** 3, C_RED, fmax=1.2)
    dark = rng.random(n ** 3) < 0.3
    U0[0, dark] = 0.0
    U0[0, rng.random(n ** 3) < 0.02] = (1e-41, 0.0, 0.0, 0.0)      # light that has just reached a dark cell (denormal N)
    w = tiny_workload(n, G, chemistry=0, U0=U0, courant=1.0)
    orc, gpu, _, _ = run_pair(w, 1, track_signatures=False, flux=HLL)
    Uo = orc.read(O.F_U, 0, 0)
    Ug = gpu.read(E.FIELD_U, 0, 0).astype(np.float64)
    assert np.isfinite(Ug).all()
    sc = np.abs(U0[0, :, 0]).max()
    assert np.abs(Ug[:, 0] - Uo[:, 0]).max() <= 5e-6 * sc
    assert np.abs(Ug[:, 1:] - Uo[:, 1:]).max() <= 5e-6 * C_RED * sc


def test_hll_beam_is_upwind_on_gpu():
    """H4 on the GPU: F = c N x^ with a power-of-two c (f = 1 exactly in fp32): exact upwind, nothing leaks sideways."""
    n, c, k = 40, 2.0 ** 31, 5
    rng = np.random.default_rng(5)
    prof = rng.uniform(0.5, 2.0, n).astype(np.float32)
    U0 = np.zeros((1, n, n, n, 4), np.float32)
    U0[0, ..., 0] = prof[None, None, :]
    U0[0, ..., 1] = np.float32(c) * prof[None, None, :]
    w = tiny_workload(n, 1, U0=U0.reshape(1, n ** 3, 4), c_red=c, chemistry=0, courant=0.75)
    orc, gpu, _, _ = run_pair(w, k, track_signatures=False, flux=HLL, block=k)
    Uo = orc.read(O.F_U).reshape(n, n, n, 4)
    Ug = gpu.read(E.FIELD_U).reshape(n, n, n, 4).astype(np.float64)
    assert np.abs(Ug[..., 0] - Uo[..., 0]).max() <= 2e-6 * Uo[..., 0].max()
    assert np.abs(Ug[..., 1] - c * Ug[..., 0]).max() <= 2e-6 * c * Uo[..., 0].max()
    assert np.abs(Ug[..., 2:]).max() == 0.0


@pytest.mark.parametrize("n,G,bc", [(24, 3, (0,) * 6), (33, 1, (2, 2, 1, 1, 0, 0))])
def test_hll_coupled_one_step(n, G, bc):
    """HLL transport followed by the chemistry passes (two-pass schedule) on a random state with sources."""
    rng = np.random.default_rng(50 + n)
    nc = n ** 3
    n0 = (10 ** rng.uniform(-5, -2, nc)).astype(np.float32)
    x = np.minimum(10 ** rng.uniform(-4, 0, nc), 0.999999).astype(np.float32)
    T = (10 ** rng.uniform(2, 4.0, nc)).astype(np.float32)
    w = tiny_workload(n, G, bc=bc, n0=n0, x=x, T=T, U0=_random_U(rng, G, nc, C_RED, fmax=0.9, lo=-7, hi=-2),
                      src_pos=rng.random((3, 3)), src_Q=10 ** rng.uniform(47, 49, (3, G)))
    orc, gpu, flips, diags = run_pair(w, 1, flux=HLL)
    rep = compare(orc, gpu, w, flips, 1, nf_cond=absorption_condition(w, w.dt))
    assert rep["flips"] <= max(2, 1e-4 * rep["cells"]), rep
    assert rep["x"] <= TOL_XT and rep["T"] <= TOL_XT, rep
    assert rep["N"] <= 5e-5 and rep["F"] <= 5e-5, rep
    k = gpu.profile(False)


def test_hll_config1_stromgren_60_steps():
    """Config 1 with the HLL flux, 60 coupled steps: x, T within 1e-4, budget within 1e-6 every step."""
    w = make_config(1)
    orc, gpu, flips, diags = run_pair(w, 60, flux=HLL)
    rep = compare(orc, gpu, w, flips, 60)
    prev, worst = None, 0.0
    for do, dg in diags:
        if prev is not None:
            worst = max(worst, budget_residual(dg, prev))
        prev = dg["photons_total"]
    assert rep["flips"] <= max(1, 1e-4 * rep["cells"]), rep
    assert rep["x"] <= TOL_XT and rep["T"] <= TOL_XT, rep
    assert worst <= TOL_BUDGET, worst


def test_hll_config5_recipe_64_20_coupled_steps_whole_grid():
    """The metric's workload shape (config 5b recipe: lognormal density, random x, T, 3 groups, many sources) at 64^3 with the
    HLL flux for 20 coupled steps, every cell against the oracle with the flip protocol: the two-pass schedule around
    transport_hll_kernel (2 x 3 tiles of 31 cells, a ragged 2-cell tile, 4 tile rows) through the sub-cycling transient."""
    w = make_config(5, n=64, variant="b")
    orc, gpu, flips, diags = run_pair(w, 20, flux=HLL)
    rep = compare(orc, gpu, w, flips, 20, radius=4)
    prev, worst = None, 0.0
    for do, dg in diags:
        if prev is not None:
            worst = max(worst, budget_residual(dg, prev))
        prev = dg["photons_total"]
        assert dg["n_nonfinite"] == 0
    print("HLL config 5b 64^3 x 20 steps", {k: (float("%.3g" % v) if isinstance(v, float) else v) for k, v in rep.items()})
    assert diags[0][1]["subcycles_max"] > 10 and diags[0][1]["n_deferred"] > 1000       # the random T state sub-cycles hard
    assert rep["flips"] <= max(2, 1e-3 * rep["cells"]), rep
    assert rep["x"] <= TOL_XT and rep["T"] <= TOL_XT, rep
    assert worst <= TOL_BUDGET, worst
    do, dg = diags[-1]
    assert abs(dg["photons_total"] - do["photons_total"]) <= 1e-5 * abs(do["photons_total"])
