"""emma_rt_photons_total_noalloc (include/emma_rt.h; csrc/noalloc.cu): the photon total of A15 with its scratch in a static
device array -- no cudaMalloc, for callers under CUDA graph capture or in loops that must not allocate.  Checked against the
existing path, the state query emma_rt_step(h, dt, 0, &diag), which sums the same values with the same kernels, grid and order
out of the handle's arena: same bits expected, 1e-12 relative asserted (the tolerance of the diagnostics elsewhere in tests/).
Two calls in a row (the second after the state has moved on, then a much shorter one that must not see the first one's block
sums), the refusals, and that the device's free memory does not move across a call.

This file sorts last on purpose: the suite runs with `pytest -x`, and a failure here must not hide another test."""
import numpy as np
import pytest

import paper_1508_07888_b200 as E
from workloads import make_config

pytestmark = pytest.mark.gpu

TOL = 1e-12


def _gather_U(gpu, w, Ubuf):
    """FIELD_U of every group, one after the other, into the caller's device buffer [G * ncell, 4] (stream-ordered D2D copies)."""
    nc = w.n ** 3
    for g in range(w.G):
        assert gpu.read_into(E.FIELD_U, 0, g, Ubuf[g * nc:(g + 1) * nc]) == E.OK


def test_noalloc_photon_total_matches_the_state_query_twice_in_a_row():
    import torch
    w = make_config(5, n=48)                                           # 48^3 x 3 groups = 331776 records: 1024 blocks, ragged stride
    gpu = E.EmmaRT(w)
    nc = w.n ** 3
    dx = w.L / w.n                                                     # as api.cu: dV = dx * dx * dx in fp64
    dV = dx * dx * dx
    st = torch.cuda.current_stream().cuda_stream
    # everything the caller owns is allocated up front
    Ubuf = torch.empty((w.G * nc, 4), dtype=torch.float32, device="cuda")
    out = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    seen = []
    for call in range(2):
        _gather_U(gpu, w, Ubuf)
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        rc, err = E.emma_rt_photons_total_noalloc(Ubuf.data_ptr(), w.G * nc, dV, out.data_ptr(), st)
        torch.cuda.synchronize()
        free1 = torch.cuda.mem_get_info()[0]
        assert rc == E.OK and err == "", err
        if call > 0:                                                   # (the first call on a device may load the module)
            assert free1 == free0, (free0, free1)
        got = float(out.item())
        rc, d = gpu.step(w.dt, 0)                                      # the existing path: state query, scratch in the arena
        assert rc == E.OK, gpu.last_error()
        ref = d["photons_total"]
        print("call %d: noalloc %.17g  state query %.17g  bit-equal %s" % (call, got, ref, got == ref))
        assert ref > 0 and abs(got - ref) <= TOL * ref
        seen.append(got)
        rc, _ = gpu.step(w.dt, 3)                                      # move the state on between the two calls
        assert rc == E.OK, gpu.last_error()
    assert seen[0] != seen[1]                                          # the sources injected photons in between

    # a much shorter call right after a long one: 1000 records = 4 blocks; slots 4..1023 still hold the long call's sums
    _gather_U(gpu, w, Ubuf)
    rc, err = E.emma_rt_photons_total_noalloc(Ubuf.data_ptr() + 16 * 5, 1000, dV, out.data_ptr(), st)
    assert rc == E.OK, err
    torch.cuda.synchronize()
    N = Ubuf[5:1005, 0].cpu().numpy().astype(np.float64)
    ref = float(N.sum()) * dV
    assert abs(float(out.item()) - ref) <= TOL * abs(ref)
    # n = 0: set-up only, the total is 0
    rc, err = E.emma_rt_photons_total_noalloc(0, 0, dV, out.data_ptr(), st)
    torch.cuda.synchronize()
    assert rc == E.OK and float(out.item()) == 0.0
    gpu.close()


def test_noalloc_refusals_launch_nothing():
    import torch
    U = torch.ones((64, 4), dtype=torch.float32, device="cuda")
    out = torch.full((1,), -7.0, dtype=torch.float64, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    rc, err = E.emma_rt_photons_total_noalloc(U.data_ptr(), E.NOALLOC_MAX_CELLGROUPS + 1, 1.0, out.data_ptr(), st)
    assert rc == E.EINVAL and "EMMA_RT_NOALLOC_MAX_CELLGROUPS" in err and str(E.NOALLOC_MAX_CELLGROUPS) in err
    rc, err = E.emma_rt_photons_total_noalloc(U.data_ptr(), -1, 1.0, out.data_ptr(), st)
    assert rc == E.EINVAL and "negative" in err
    rc, err = E.emma_rt_photons_total_noalloc(U.data_ptr(), 64, 1.0, 0, st)
    assert rc == E.EINVAL and "total_dev" in err
    rc, err = E.emma_rt_photons_total_noalloc(0, 64, 1.0, out.data_ptr(), st)
    assert rc == E.EINVAL and "U_dev" in err
    rc, err = E.emma_rt_photons_total_noalloc(U.data_ptr() + 4, 8, 1.0, out.data_ptr(), st)
    assert rc == E.EINVAL and "aligned" in err
    for bad in (0.0, -1.0, float("inf"), float("nan")):
        rc, err = E.emma_rt_photons_total_noalloc(U.data_ptr(), 64, bad, out.data_ptr(), st)
        assert rc == E.EINVAL and "dV" in err
    torch.cuda.synchronize()
    assert float(out.item()) == -7.0                                   # nothing was launched
    rc, err = E.emma_rt_photons_total_noalloc(U.data_ptr(), 64, 0.5, out.data_ptr(), st)
    torch.cuda.synchronize()
    assert rc == E.OK and float(out.item()) == 32.0
