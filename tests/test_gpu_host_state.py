"""emma_rt_step_host (include/emma_rt.h): the slab-pipelined coupled step for HOST-resident state must be the same step,
bit for bit, as write(U, X, T) -> step -> read(U, X, T) (the paper's engines work this way, host state in,
host state out), and through the oracle it is held to the usual tolerances."""
import numpy as np
import pytest

import oracle as O
import paper_1508_07888_b200 as E
from workloads import make_config

from .parity import compare

pytestmark = pytest.mark.gpu


def _host_copy(w):
    U = [np.ascontiguousarray(w.U0[g], np.float32).copy() for g in range(w.G)]
    return U, w.x[0].copy(), w.T[0].copy()


@pytest.mark.parametrize("n,bc", [(48, (0,) * 6), (20, (0,) * 6), (36, (1, 2, 0, 0, 2, 1)), (7, (0,) * 6)])
def test_step_host_equals_write_step_read(n, bc):
    """Several slabs (48: 6 of 8 planes), a ragged last slab (20: 8 + 8 + 4; 36), one slab (7), open and reflective faces
    in z; two steps in a row, the second one in place on the host arrays."""
    w = make_config(5, n=n)
    w.bc = tuple(bc)
    ref = E.EmmaRT(w)
    gpu = E.EmmaRT(w)
    U, x, T = _host_copy(w)
    Uo = [np.empty_like(u) for u in U]
    xo, To = np.empty_like(x), np.empty_like(T)
    for step in range(2):
        if step == 0:
            rc, d = gpu.step_host(w.dt, U, x, T, Uo, xo, To)          # separate output arrays
            U, x, T = Uo, xo, To
        else:
            rc, d = gpu.step_host(w.dt, U, x, T)                      # in place
        assert rc == E.OK, gpu.last_error()
        rcr, dr = ref.step(w.dt, 1)
        assert rcr == E.OK
        Ur = [ref.read(E.FIELD_U, 0, g) for g in range(w.G)]
        xr, Tr = ref.read(E.FIELD_X), ref.read(E.FIELD_T)
        # the reference's next step starts from the HOST values too (cgs F, x, T round once on the way out and back in)
        for g in range(w.G):
            assert ref.write(E.FIELD_U, 0, g, Ur[g]) == E.OK
        assert ref.write(E.FIELD_X, 0, 0, xr) == E.OK and ref.write(E.FIELD_T, 0, 0, Tr) == E.OK
        for g in range(w.G):
            assert np.array_equal(U[g], Ur[g]), (step, g)
            assert np.array_equal(gpu.read(E.FIELD_U, 0, g), U[g])    # the device holds the new state too
        assert np.array_equal(x, xr) and np.array_equal(T, Tr)
        assert np.array_equal(gpu.read(E.FIELD_X), x)
        for k in ("photons_total", "photons_absorbed", "photons_injected", "photons_outflow"):
            assert abs(d[k] - dr[k]) <= 1e-12 * max(abs(dr[k]), 1e-300), k
        for k in ("subcycles_total", "subcycles_max", "halvings_total", "n_deferred", "n_nonfinite"):
            assert d[k] == dr[k], k
        assert d["t_sim"] == dr["t_sim"]
    gpu.close()
    ref.close()


def test_step_host_against_the_oracle_and_pinned_tensors():
    import torch
    w = make_config(5, n=40)
    orc = O.Oracle(w)
    gpu = E.EmmaRT(w, record_subcycles=1)
    U = [torch.from_numpy(np.ascontiguousarray(w.U0[g], np.float32).copy()).pin_memory() for g in range(w.G)]
    x = torch.from_numpy(w.x[0].copy()).pin_memory()
    T = torch.from_numpy(w.T[0].copy()).pin_memory()
    flips = []
    for step in range(1, 6):
        rc, d = gpu.step_host(w.dt, U, x, T)
        assert rc == E.OK, gpu.last_error()
        rco, do = orc.step(w.dt, 1)
        assert rco == O.OK
        so = orc.read(O.F_SUBCYCLES, 0).astype(np.int64)
        sg = gpu.read(E.FIELD_SUBCYCLES, 0).astype(np.int64)
        flips += [(step, 0, int(c), int(c)) for c in np.flatnonzero(so != sg)]
    rep = compare(orc, gpu, w, flips, 5)
    print("step_host vs oracle, 5 steps", {k: (float("%.3g" % v) if isinstance(v, float) else v) for k, v in rep.items()})
    assert rep["x"] <= 1e-4 and rep["T"] <= 1e-4 and rep["flips"] <= 1e-3 * rep["cells"]
    a = orc.read(O.F_X, 0)
    assert np.max(np.abs(x.numpy() - a) / a) <= max(rep["x"], rep["x_near"]) * 1.0000001 + 1e-12      # the host arrays ARE the state
    assert abs(d["photons_total"] - do["photons_total"]) <= 1e-5 * do["photons_total"]


def test_step_host_refusals():
    w = make_config(4, n=16, n_src=2)                                   # refined grid: not available
    gpu = E.EmmaRT(w)
    z = np.zeros((16 ** 3, 4), np.float32)
    rc, _ = gpu.step_host(w.dt, [z, z, z], w.x[0].copy(), w.T[0].copy())
    assert rc == E.ESTATE and "uniform" in gpu.last_error()
    gpu.close()
    w = make_config(5, n=12)
    gpu = E.EmmaRT(w)
    U, x, T = _host_copy(w)
    rc, _ = gpu.step_host(10 * w.dt, U, x, T)
    assert rc == E.ECFL
    bad = x.copy()
    bad[5] = 2.0
    rc, _ = gpu.step_host(w.dt, U, bad, T)
    assert rc == E.EINVAL and "invalid" in gpu.last_error()
    gpu.set_schedule(0)
    rc, _ = gpu.step_host(w.dt, U, x, T)
    assert rc == E.ESTATE
    gpu.close()


def test_step_host_256_many_slabs_bit_equal():
    """At size: 256^3 x 3 groups (0.8 GB of radiation each way per step) goes through the device in 32 slabs of 8 planes on
    three streams; two steps in place on pinned host tensors must leave the same bits as write -> step -> read."""
    import torch
    w = make_config(5, n=256, variant="b")
    ref = E.EmmaRT(w)
    gpu = E.EmmaRT(w)
    U = [torch.from_numpy(np.ascontiguousarray(w.U0[g], np.float32).copy()).pin_memory() for g in range(w.G)]
    x = torch.from_numpy(w.x[0].copy()).pin_memory()
    T = torch.from_numpy(w.T[0].copy()).pin_memory()
    for step in range(2):
        rc, d = gpu.step_host(w.dt, U, x, T)
        assert rc == E.OK, gpu.last_error()
        rcr, dr = ref.step(w.dt, 1)
        assert rcr == E.OK
        Ur = [ref.read(E.FIELD_U, 0, g) for g in range(w.G)]
        xr, Tr = ref.read(E.FIELD_X), ref.read(E.FIELD_T)
        for g in range(w.G):
            assert ref.write(E.FIELD_U, 0, g, Ur[g]) == E.OK          # the reference's next step starts from the host values too
        assert ref.write(E.FIELD_X, 0, 0, xr) == E.OK and ref.write(E.FIELD_T, 0, 0, Tr) == E.OK
        for g in range(w.G):
            assert np.array_equal(U[g].numpy(), Ur[g]), (step, g)
        assert np.array_equal(x.numpy(), xr) and np.array_equal(T.numpy(), Tr)
        assert d["subcycles_total"] == dr["subcycles_total"] and d["n_deferred"] == dr["n_deferred"]
        assert abs(d["photons_total"] - dr["photons_total"]) <= 1e-12 * dr["photons_total"]
    assert d["subcycles_max"] > 1                                        # the random initial T: the tail kernel ran on slabs too
    gpu.close()
    ref.close()
