"""T3: the standard AMR scheme at the size and launch configuration bench.py --amr-standard times (256^3 + 2 levels x 3
groups).  The oracle's AMR recursion is serial and non-local (a coarse step of this mesh is minutes of CPU work), so at
this size the check is by properties that hold at any size: the A15 photon budget closes every step, every photon that
was injected is Q dt, split cells hold the mean of their children, nothing is negative or non-finite.  Element-by-element
parity with the oracle is tests/test_gpu_amr.py (meshes of 10^3..16^3 coarse cells that span several CTAs per level).
"""
import numpy as np
import pytest

import paper_1508_07888_b200 as E
from workloads.amr import make_amr_standard

from .parity import budget_residual

pytestmark = pytest.mark.gpu


def test_amr_standard_bench_size_properties():
    w = make_amr_standard(n=256, G=3, levels=2)
    gpu = E.EmmaRT(w, amr_transport=1)
    prev = 0.0
    for step in range(4):
        rc, d = gpu.step(w.dt, 1)
        assert rc == E.OK, gpu.last_error()
        assert budget_residual(d, prev) <= 1e-6, (step, d)
        assert d["n_nonfinite"] == 0
        assert d["photons_injected"] == pytest.approx(w.src_Q.sum() * w.dt, rel=1e-6)
        prev = d["photons_total"]
    assert d["photons_absorbed"] > 0
    for g in (0, 2):
        N = [gpu.read(E.FIELD_N, l, g).astype(np.float64) for l in range(3)]
        for l in (0, 1):
            par = np.asarray(w.parent[l], np.int64)
            mean = N[l + 1].reshape(-1, 8).mean(axis=1)
            np.testing.assert_allclose(N[l][par], mean, rtol=2e-6, atol=1e-30)
        for l in range(3):
            assert N[l].min() >= -1e-7 * N[l].max()
    x2 = gpu.read(E.FIELD_X, 2)
    assert x2.max() > 1.2e-3 and x2.min() >= 0.0
    gpu.close()
