"""T1 (CPU part): the C-ABI library loads without a GPU and exports every symbol include/emma_rt.h declares;
argument validation that needs no device works.  No compute call is made here."""
import ctypes as C
import os
import re

import pytest

import paper_1508_07888_b200 as E
from paper_1508_07888_b200 import binding as B
from paper_1508_07888_b200 import build as builder

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    builder.build()
    return E.lib()


def test_every_declared_symbol_is_exported(L):
    hdr = open(os.path.join(ROOT, "include", "emma_rt.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(emma_rt_[a-z_]+)\s*\(", hdr))
    assert declared == set(E.EXPORTED_SYMBOLS)
    for s in declared:
        assert hasattr(L, s), s


def test_struct_sizes_match_header(L):
    # a wrong struct_size / abi_version must be rejected -> arena_bytes == 0
    cfg = B.make_config(32, 1, 1e22, 3e9, [1e-18], [1e-18], [4e-11])
    assert L.emma_rt_arena_bytes(C.byref(cfg), None) > 0
    cfg.struct_size += 4
    assert L.emma_rt_arena_bytes(C.byref(cfg), None) == 0
    cfg = B.make_config(32, 1, 1e22, 3e9, [1e-18], [1e-18], [4e-11])
    cfg.abi_version = 99
    assert L.emma_rt_arena_bytes(C.byref(cfg), None) == 0


def test_arena_bytes_validation_and_size(L):
    ok = lambda **kw: E.emma_rt_arena_bytes(B.make_config(**{**dict(n_coarse=32, n_groups=3, box_len_cm=1e22,
                                                                    c_red_cm_s=3e9, sigma_N=[1e-18] * 3,
                                                                    sigma_E=[1e-18] * 3, E_mean=[4e-11] * 3), **kw}))
    base = ok()
    assert base >= 2 * 3 * 32 ** 3 * 16 + 3 * 32 ** 3 * 4            # two radiation buffers + n0, xs, eps
    assert ok(n_groups=5) == 0 and ok(n_groups=0) == 0
    assert ok(n_coarse=1) == 0
    assert ok(bc=(0, 1, 0, 0, 0, 0)) == 0                             # periodic faces come in pairs
    assert ok(bc=(1, 2, 0, 0, 2, 2)) > 0
    assert ok(box_len_cm=-1.0) == 0 and ok(c_red_cm_s=0.0) == 0
    assert ok(record_subcycles=1) >= base + 32 ** 3 * 4
    # config 5 of BASELINE.json fits one B200 (180 GB) with room to spare
    big = ok(n_coarse=512)
    assert 2 * 3 * 512 ** 3 * 16 < big < 20e9


def test_null_amr_arrays_are_refused_not_dereferenced(L):
    """A refined description whose n_octs / parent arrays (or one level's parent list) are NULL is invalid: 0, no crash."""
    cfg = B.make_config(8, 1, 1e22, 3e9, [1e-18], [1e-18], [4e-11])
    a = B.Amr()
    a.n_levels, a.n_octs, a.parent = 1, None, None
    assert L.emma_rt_arena_bytes(C.byref(cfg), C.byref(a)) == 0
    n_octs = (C.c_int64 * 1)(3)
    a.n_octs = C.cast(n_octs, C.POINTER(C.c_int64))
    assert L.emma_rt_arena_bytes(C.byref(cfg), C.byref(a)) == 0
    par = (C.c_void_p * 1)(None)
    a.parent = C.cast(par, C.POINTER(C.c_void_p))
    assert L.emma_rt_arena_bytes(C.byref(cfg), C.byref(a)) == 0      # n_octs[0] = 3 with a NULL parent list
    # init refuses the same without touching a device
    h = C.c_void_p()
    assert L.emma_rt_init(C.byref(h), C.byref(cfg), C.byref(a), None, None, 0) == E.EINVAL and not h.value


def test_step_reads_no_environment(L):
    """The tuning variables are read once, at init (include/emma_rt.h): no getenv outside emma_rt_init's helper."""
    src = open(os.path.join(ROOT, "paper_1508_07888_b200", "csrc", "api.cu")).read()
    assert src.count("getenv(") == 1
    for f in os.listdir(os.path.join(ROOT, "paper_1508_07888_b200", "csrc")):
        if f != "api.cu":
            assert "getenv(" not in open(os.path.join(ROOT, "paper_1508_07888_b200", "csrc", f)).read(), f
    hdr = open(os.path.join(ROOT, "include", "emma_rt.h")).read()
    for v in re.findall(r'env_int\("(EMMA_RT_TUNE_[A-Z]+)"', src):
        assert v in hdr, v


def test_null_handle_calls_fail_cleanly(L):
    assert L.emma_rt_step(None, 1.0, 1, None) == E.EINVAL
    assert L.emma_rt_set_sources(None, 0, None, None) == E.EINVAL
    assert L.emma_rt_level_cells(None, 0) == -1
    assert L.emma_rt_kernel_launches(None) == 0
    L.emma_rt_free(None)


def test_no_cpu_fallback_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from workloads import make_config
    with pytest.raises(E.EmmaRTError) as ei:
        E.EmmaRT(make_config(1, n=4))
    assert ei.value.code == E.ECUDA
