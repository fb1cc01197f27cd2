"""the static cousin of the paper's HII-region test (corner source, reflective
faces at the source, transmissive elsewhere, 3 groups, 15 kpc box) -- `workloads.make_hii_region_corner`.

The paper prints no numbers for this test (figures only, comparison data not in the container), so the CPU test pins the
oracle to what the set-up itself fixes at early times (t << t_rec): every emitted photon is either still in flight, has
left the box, or has ionised one atom (recombinations remove ~t/t_rec of them), and the gas behind the front is hot and
fully ionised.  The GPU test is element-by-element parity on the same run."""
import math

import numpy as np
import pytest

import oracle as O
from workloads import CGS, make_hii_region_corner

X0, NH, Q = 1.2e-3, 1e-3, 5e48


def test_hii_region_photon_count_front_and_temperature():
    n, K = 24, 220
    w = make_hii_region_corner(n=n)
    o = O.Oracle(w)
    rc, d = o.step(w.dt, K)
    assert rc == O.OK
    x = o.read(O.F_X).reshape(n, n, n)
    T = o.read(O.F_T).reshape(n, n, n)
    dV, t = w.dx ** 3, K * w.dt
    emitted = Q * t
    ions = ((x - X0) * NH * dV).sum()
    accounted = (ions + d["photons_total"] + d["photons_outflow"]) / emitted
    t_rec = 1.0 / (2.59e-13 * NH)
    assert 1.0 - 3.0 * t / t_rec <= accounted <= 1.0 + 1e-9, accounted      # only recombinations remove photons
    assert ions / emitted > 0.85
    # ionised volume of the octant -> radius; analytic: (pi/6) r^3 n_H = Q t (1 - in flight - recombined)
    r_V = (6.0 * ((x - X0) / (1 - X0) * dV).sum() / math.pi) ** (1.0 / 3.0)
    r_an = (6.0 * ions / (NH * math.pi)) ** (1.0 / 3.0)
    assert r_V == pytest.approx(r_an, rel=2e-3, abs=0)
    assert r_an == pytest.approx((6.0 * emitted / (NH * math.pi)) ** (1.0 / 3.0), rel=0.06, abs=0)
    # the front is where x = 0.5: along an axis it sits within a cell and a half of the equivalent radius
    ax = x[0, 0, :]
    i_half = int(np.argmax(ax < 0.5))
    assert abs(i_half - r_an / w.dx) <= 1.5, (i_half, r_an / w.dx)
    # behind the front: fully ionised and photo-heated to a few 1e4 K; far ahead: untouched
    assert x[0, 0, 0] > 0.999 and 1.2e4 < T[0, 0, 1] < 4e4
    assert x[-1, -1, -1] == pytest.approx(X0, rel=1e-3, abs=0) and T[-1, -1, -1] == pytest.approx(100.0, rel=1e-3, abs=0)
    # symmetric set-up -> symmetric solution (the three axes are equivalent)
    assert np.allclose(x[0, 0, :8], x[0, :8, 0], rtol=1e-12) and np.allclose(x[0, 0, :8], x[:8, 0, 0], rtol=1e-12)


@pytest.mark.gpu
@pytest.mark.parametrize("flux", [0, 1])
def test_hii_region_gpu_parity(flux):
    import paper_1508_07888_b200 as E  # noqa: F401
    from .parity import budget_residual, compare, run_pair
    w = make_hii_region_corner(n=48)
    K = 150
    orc, gpu, flips, diags = run_pair(w, K, flux=flux)
    rep = compare(orc, gpu, w, flips, K)
    prev, worst = None, 0.0
    for do, dg in diags:
        if prev is not None:
            worst = max(worst, budget_residual(dg, prev))
        prev = dg["photons_total"]
    assert rep["flips"] <= max(1, 1e-4 * rep["cells"]), rep
    assert rep["x"] <= 1e-4 and rep["T"] <= 1e-4, rep
    assert worst <= 1e-6, worst
