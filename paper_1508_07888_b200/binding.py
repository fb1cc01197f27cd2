"""ctypes binding of include/emma_rt.h -- argument marshalling only; every step of the path runs in the CUDA kernels.

Module-level functions carry the C names (`emma_rt_init`, `emma_rt_set_sources`, `emma_rt_step`, `emma_rt_read`, ...);
`EmmaRT` is a convenience wrapper that allocates the arena with torch and keeps it alive.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libemma_rt.so")

MAX_GROUPS, MAX_LEVELS, ABI_VERSION = 4, 4, 2
OK, EINVAL, ENOMEM, ECUDA, ENONFINITE, ESTATE, ECFL, ESUBCYCLE = 0, -1, -2, -3, -4, -5, -6, -7
FIELD_U, FIELD_N, FIELD_F, FIELD_X, FIELD_T, FIELD_E, FIELD_N0, FIELD_SUBCYCLES, FIELD_XNEUTRAL = range(9)
_FIELD_SHAPE = {FIELD_U: (4, np.float32), FIELD_F: (3, np.float32), FIELD_SUBCYCLES: (1, np.uint32)}

EXPORTED_SYMBOLS = ["emma_rt_arena_bytes", "emma_rt_init", "emma_rt_set_sources", "emma_rt_dt_cfl", "emma_rt_step",
                    "emma_rt_step_host", "emma_rt_read", "emma_rt_write", "emma_rt_level_cells", "emma_rt_kernel_launches",
                    "emma_rt_profile", "emma_rt_set_schedule", "emma_rt_set_flux", "emma_rt_set_inflow", "emma_rt_last_error", "emma_rt_free",
                    "emma_rt_photons_total_noalloc"]
NOALLOC_MAX_CELLGROUPS = 1 << 33              # EMMA_RT_NOALLOC_MAX_CELLGROUPS
FLUX_GLF, FLUX_HLL = 0, 1
BC_PERIODIC, BC_TRANSMISSIVE, BC_REFLECTIVE, BC_INFLOW = 0, 1, 2, 3
KERNEL_KINDS = ["transport", "chem_main", "chem_tail", "chem_refined", "finalize", "other", "fused", "amr_transport", "amr_chem"]


class EmmaRTError(RuntimeError):
    def __init__(self, code, msg=""):
        super().__init__("emma_rt error %d: %s" % (code, msg))
        self.code = code


class Config(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("abi_version", C.c_uint32), ("n_coarse", C.c_int32),
                ("n_groups", C.c_int32), ("bc", C.c_int32 * 6), ("otsa", C.c_int32), ("chemistry", C.c_int32),
                ("thermal", C.c_int32), ("record_subcycles", C.c_int32), ("max_halvings", C.c_int32),
                ("device", C.c_int32), ("max_source_cells", C.c_int64), ("box_len_cm", C.c_double),
                ("c_red_cm_s", C.c_double), ("sigma_N", C.c_double * MAX_GROUPS), ("sigma_E", C.c_double * MAX_GROUPS),
                ("E_mean", C.c_double * MAX_GROUPS), ("e_tol", C.c_double), ("stream", C.c_void_p),
                ("amr_transport", C.c_int32), ("reserved0", C.c_int32)]


class Amr(C.Structure):
    _fields_ = [("n_levels", C.c_int32), ("n_octs", C.POINTER(C.c_int64)), ("parent", C.POINTER(C.c_void_p))]


class Fields(C.Structure):
    _fields_ = [("U0", C.POINTER(C.c_void_p)), ("n0", C.POINTER(C.c_void_p)), ("x", C.POINTER(C.c_void_p)),
                ("T", C.POINTER(C.c_void_p))]


class HostState(C.Structure):
    _fields_ = [("U", C.POINTER(C.c_void_p)), ("x", C.c_void_p), ("T", C.c_void_p)]


class Diag(C.Structure):
    _fields_ = [("photons_total", C.c_double), ("photons_injected", C.c_double), ("photons_absorbed", C.c_double),
                ("photons_recomb_emitted", C.c_double), ("photons_outflow", C.c_double), ("dtau_min", C.c_double),
                ("subcycles_total", C.c_int64), ("subcycles_max", C.c_int64), ("halvings_total", C.c_int64),
                ("n_nonfinite", C.c_int64), ("n_deferred", C.c_int64), ("t_sim", C.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_lib = None


def lib_path():
    return _LIB_PATH


def lib():
    """Load libemma_rt.so (built in-tree by paper_1508_07888_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise EmmaRTError(ECUDA, "libemma_rt.so is not built (run `python -m paper_1508_07888_b200.build`); "
                                 "there is no CPU fallback")
    L = C.CDLL(_LIB_PATH)
    L.emma_rt_arena_bytes.restype = C.c_size_t
    L.emma_rt_arena_bytes.argtypes = [C.POINTER(Config), C.POINTER(Amr)]
    L.emma_rt_init.restype = C.c_int
    L.emma_rt_init.argtypes = [C.POINTER(C.c_void_p), C.POINTER(Config), C.POINTER(Amr), C.POINTER(Fields),
                               C.c_void_p, C.c_size_t]
    L.emma_rt_set_sources.restype = C.c_int
    L.emma_rt_set_sources.argtypes = [C.c_void_p, C.c_int64, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    L.emma_rt_dt_cfl.restype = C.c_double
    L.emma_rt_dt_cfl.argtypes = [C.c_void_p, C.c_double]
    L.emma_rt_step.restype = C.c_int
    L.emma_rt_step.argtypes = [C.c_void_p, C.c_double, C.c_int32, C.POINTER(Diag)]
    L.emma_rt_step_host.restype = C.c_int
    L.emma_rt_step_host.argtypes = [C.c_void_p, C.c_double, C.POINTER(HostState), C.POINTER(HostState), C.POINTER(Diag)]
    L.emma_rt_read.restype = C.c_int
    L.emma_rt_read.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.c_size_t, C.c_int32]
    L.emma_rt_write.restype = C.c_int
    L.emma_rt_write.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.c_size_t, C.c_int32]
    L.emma_rt_level_cells.restype = C.c_int64
    L.emma_rt_level_cells.argtypes = [C.c_void_p, C.c_int32]
    L.emma_rt_kernel_launches.restype = C.c_int64
    L.emma_rt_kernel_launches.argtypes = [C.c_void_p]
    L.emma_rt_profile.restype = C.c_int
    L.emma_rt_profile.argtypes = [C.c_void_p, C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
    L.emma_rt_set_schedule.restype = C.c_int
    L.emma_rt_set_schedule.argtypes = [C.c_void_p, C.c_int32]
    L.emma_rt_set_inflow.restype = C.c_int
    L.emma_rt_set_inflow.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.POINTER(C.c_double)]
    L.emma_rt_set_flux.restype = C.c_int
    L.emma_rt_set_flux.argtypes = [C.c_void_p, C.c_int32]
    L.emma_rt_last_error.restype = C.c_char_p
    L.emma_rt_last_error.argtypes = [C.c_void_p]
    L.emma_rt_photons_total_noalloc.restype = C.c_int
    L.emma_rt_photons_total_noalloc.argtypes = [C.c_void_p, C.c_int64, C.c_double, C.c_void_p, C.c_void_p, C.c_char_p, C.c_size_t]
    L.emma_rt_free.restype = None
    L.emma_rt_free.argtypes = [C.c_void_p]
    _lib = L
    return L


def make_config(n_coarse, n_groups, box_len_cm, c_red_cm_s, sigma_N, sigma_E, E_mean, bc=(0,) * 6, otsa=1, chemistry=1,
                thermal=1, record_subcycles=0, max_halvings=60, device=0, max_source_cells=0, e_tol=0.1, stream=0,
                amr_transport=0):
    c = Config()
    c.struct_size, c.abi_version = C.sizeof(Config), ABI_VERSION
    c.n_coarse, c.n_groups = int(n_coarse), int(n_groups)
    for i in range(6):
        c.bc[i] = int(bc[i])
    c.otsa, c.chemistry, c.thermal, c.record_subcycles = int(otsa), int(chemistry), int(thermal), int(record_subcycles)
    c.max_halvings, c.device, c.max_source_cells = int(max_halvings), int(device), int(max_source_cells)
    c.box_len_cm, c.c_red_cm_s, c.e_tol = float(box_len_cm), float(c_red_cm_s), float(e_tol)
    for g in range(max(0, min(int(n_groups), MAX_GROUPS, len(sigma_N)))):
        c.sigma_N[g], c.sigma_E[g], c.E_mean[g] = float(sigma_N[g]), float(sigma_E[g]), float(E_mean[g])
    c.stream = stream
    c.amr_transport, c.reserved0 = int(amr_transport), 0
    return c


def _ptrs(arrs):
    pa = (C.c_void_p * max(1, len(arrs)))()
    for i, a in enumerate(arrs):
        pa[i] = a.ctypes.data if a is not None else None
    return pa


def _make_amr(parent):
    keep = [np.ascontiguousarray(p, np.int64) for p in parent]
    a = Amr()
    a.n_levels = len(keep)
    n_octs = (C.c_int64 * max(1, len(keep)))(*[len(p) for p in keep])
    a.n_octs = C.cast(n_octs, C.POINTER(C.c_int64))
    par = _ptrs(keep)
    a.parent = C.cast(par, C.POINTER(C.c_void_p))
    return a, (keep, n_octs, par)


# ---- functions with the C names --------------------------------------------------------------------------------
def emma_rt_arena_bytes(cfg, parent=()):
    amr, _keep = _make_amr(parent)
    return lib().emma_rt_arena_bytes(C.byref(cfg), C.byref(amr))


def emma_rt_init(cfg, parent, U0, n0, x, T, arena_ptr, arena_bytes):
    """Returns (rc, handle).  U0: list of G float32 [n^3,4] arrays or None; n0/x/T: per-level float32 arrays."""
    amr, _keep = _make_amr(parent)
    f32 = lambda a: np.ascontiguousarray(a, np.float32)
    U0k = [f32(u) if u is not None else None for u in U0] if U0 is not None else None
    n0k, xk, Tk = [f32(a) for a in n0], [f32(a) for a in x], [f32(a) for a in T]
    fl = Fields()
    pU = _ptrs(U0k) if U0k is not None else None
    pn, px, pT = _ptrs(n0k), _ptrs(xk), _ptrs(Tk)
    fl.U0 = C.cast(pU, C.POINTER(C.c_void_p)) if pU is not None else None
    fl.n0, fl.x, fl.T = (C.cast(p, C.POINTER(C.c_void_p)) for p in (pn, px, pT))
    h = C.c_void_p()
    rc = lib().emma_rt_init(C.byref(h), C.byref(cfg), C.byref(amr), C.byref(fl), C.c_void_p(arena_ptr), arena_bytes)
    return rc, h


def emma_rt_set_sources(h, pos_box, Q):
    pos = np.ascontiguousarray(pos_box, np.float64).reshape(-1, 3)
    Q = np.ascontiguousarray(Q, np.float64)
    Q = Q.reshape(len(pos), -1) if len(pos) else Q.reshape(0, 1)
    dp = C.POINTER(C.c_double)
    return lib().emma_rt_set_sources(h, len(pos), pos.ctypes.data_as(dp), Q.ctypes.data_as(dp))


def emma_rt_dt_cfl(h, courant):
    return lib().emma_rt_dt_cfl(h, float(courant))


def emma_rt_step(h, dt, n_steps, want_diag=True):
    """Returns (rc, diag dict or None)."""
    if want_diag:
        d = Diag()
        rc = lib().emma_rt_step(h, float(dt), int(n_steps), C.byref(d))
        return rc, d.as_dict()
    return lib().emma_rt_step(h, float(dt), int(n_steps), None), None


def emma_rt_read(h, field, level, group, dst_ptr, nbytes, dst_is_device):
    return lib().emma_rt_read(h, field, level, group, C.c_void_p(dst_ptr), nbytes, int(dst_is_device))


def emma_rt_write(h, field, level, group, src_ptr, nbytes, src_is_device):
    return lib().emma_rt_write(h, field, level, group, C.c_void_p(src_ptr), nbytes, int(src_is_device))


def emma_rt_free(h):
    lib().emma_rt_free(h)


def emma_rt_photons_total_noalloc(U_dev_ptr, n_cellgroups, dV, total_dev_ptr, stream=0):
    """dV * sum of N over n_cellgroups (N, Fx, Fy, Fz) float records at the DEVICE address U_dev_ptr -> the double at the DEVICE
    address total_dev_ptr, stream-ordered, without any allocation (include/emma_rt.h).  Returns (rc, error text)."""
    err = C.create_string_buffer(256)
    rc = lib().emma_rt_photons_total_noalloc(C.c_void_p(U_dev_ptr), int(n_cellgroups), float(dV), C.c_void_p(total_dev_ptr),
                                             C.c_void_p(stream), err, len(err))
    return rc, err.value.decode()


# ---- convenience wrapper ---------------------------------------------------------------------------------------
class EmmaRT:
    """Owns the torch arena and the handle.  `w` is any object with the attributes of workloads.Workload."""

    def __init__(self, w, device=0, record_subcycles=0, chemistry=None, thermal=None, otsa=None, bc=None,
                 max_source_cells=0, stream=None, fused=None, flux=None, amr_transport=0):
        import torch
        if not torch.cuda.is_available():
            raise EmmaRTError(ECUDA, "no CUDA device: this library has no CPU fallback")
        self._torch = torch
        self.w = w
        self.G = w.G
        self.device = device
        st = torch.cuda.current_stream(device).cuda_stream if stream is None else stream
        self.cfg = make_config(w.n, w.G, w.L, w.c_red, w.sigma_N, w.sigma_E, w.E_mean,
                               bc=w.bc if bc is None else bc, otsa=w.otsa if otsa is None else otsa,
                               chemistry=w.chemistry if chemistry is None else chemistry,
                               thermal=w.thermal if thermal is None else thermal,
                               record_subcycles=record_subcycles, max_halvings=w.max_halvings, device=device,
                               max_source_cells=max_source_cells, e_tol=w.e_tol, stream=st,
                               amr_transport=amr_transport)
        nbytes = emma_rt_arena_bytes(self.cfg, w.parent)
        if nbytes == 0:
            raise EmmaRTError(EINVAL, "invalid configuration")
        self.arena_bytes = nbytes
        self.arena = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda:%d" % device)
        ptr = (self.arena.data_ptr() + 255) // 256 * 256
        rc, self.h = emma_rt_init(self.cfg, w.parent, w.U0, w.n0, w.x, w.T, ptr, nbytes)
        self._check(rc)
        if fused is not None:
            self.set_schedule(fused)
        if flux is not None:
            self._check(lib().emma_rt_set_flux(self.h, int(flux)))
        for (face, group), U in (getattr(w, "inflow", None) or {}).items():
            self.set_inflow(face, group, U)
        if w.src_pos is not None and len(w.src_pos):
            self._check(emma_rt_set_sources(self.h, w.src_pos, w.src_Q))

    def _check(self, rc):
        if rc != OK:
            msg = lib().emma_rt_last_error(self.h).decode() if self.h else ""
            raise EmmaRTError(rc, msg)

    def last_error(self):
        return lib().emma_rt_last_error(self.h).decode()

    def set_sources(self, pos, Q):
        return emma_rt_set_sources(self.h, pos, Q)

    def step(self, dt, n_steps=1, diag=True):
        return emma_rt_step(self.h, dt, n_steps, diag)

    def step_host(self, dt, U, x, T, U_out=None, x_out=None, T_out=None, diag=True):
        """One coupled step on HOST state (emma_rt_step_host): U = list of G arrays [n^3, 4], x, T = [n^3]; numpy arrays or
        (pinned) torch CPU tensors, float32, contiguous.  Outputs default to the inputs (in place).  Returns (rc, diag)."""
        def ptr(a):
            if isinstance(a, np.ndarray):
                assert a.dtype == np.float32 and a.flags["C_CONTIGUOUS"]
                return a.ctypes.data
            assert a.dtype == self._torch.float32 and a.is_contiguous() and not a.is_cuda
            return a.data_ptr()

        def state(Us, xs, Ts):
            hs = HostState()
            arr = (C.c_void_p * self.G)(*[ptr(u) for u in Us])
            hs.U, hs.x, hs.T = C.cast(arr, C.POINTER(C.c_void_p)), ptr(xs), ptr(Ts)
            return hs, arr
        si, keep_i = state(U, x, T)
        so, keep_o = state(U if U_out is None else U_out, x if x_out is None else x_out, T if T_out is None else T_out)
        d = Diag()
        rc = lib().emma_rt_step_host(self.h, float(dt), C.byref(si), C.byref(so), C.byref(d) if diag else None)
        return rc, (d.as_dict() if diag else None)

    def level_cells(self, level):
        return lib().emma_rt_level_cells(self.h, level)

    def kernel_launches(self):
        return lib().emma_rt_kernel_launches(self.h)

    def set_inflow(self, face, group, U):
        """Ghost state (N, Fx, Fy, Fz) [cgs] of a BC_INFLOW face (0..5 = -x,+x,-y,+y,-z,+z)."""
        a = (C.c_double * 4)(*[float(v) for v in U])
        self._check(lib().emma_rt_set_inflow(self.h, int(face), int(group), a))

    def set_schedule(self, fused):
        """fused=1 (default): single-pass transport + chemistry; 0: separate passes."""
        self._check(lib().emma_rt_set_schedule(self.h, int(fused)))

    def profile(self, enable):
        """Per-kernel CUDA-event times [ms] and launch counts since the last call; then switch recording on/off."""
        ms = (C.c_double * len(KERNEL_KINDS))()
        cnt = (C.c_int64 * len(KERNEL_KINDS))()
        self._check(lib().emma_rt_profile(self.h, int(enable), ms, cnt))
        return {k: (ms[i], cnt[i]) for i, k in enumerate(KERNEL_KINDS)}

    def read(self, field, level=0, group=0):
        """Host numpy copy of a field."""
        nc = self.level_cells(level)
        per, dt = _FIELD_SHAPE.get(field, (1, np.float32))
        out = np.empty((nc, per) if per > 1 else (nc,), dt)
        self._check(emma_rt_read(self.h, field, level, group, out.ctypes.data, out.nbytes, 0))
        return out

    def read_into(self, field, level, group, tensor_or_array):
        """Read into a pre-allocated torch tensor (device or pinned host) or numpy array."""
        t = tensor_or_array
        if isinstance(t, np.ndarray):
            return emma_rt_read(self.h, field, level, group, t.ctypes.data, t.nbytes, 0)
        return emma_rt_read(self.h, field, level, group, t.data_ptr(), t.numel() * t.element_size(), int(t.is_cuda))

    def write(self, field, level, group, arr):
        if isinstance(arr, np.ndarray):
            a = np.ascontiguousarray(arr, np.float32)
            return emma_rt_write(self.h, field, level, group, a.ctypes.data, a.nbytes, 0)
        return emma_rt_write(self.h, field, level, group, arr.data_ptr(), arr.numel() * arr.element_size(), int(arr.is_cuda))

    def close(self):
        if getattr(self, "h", None):
            self._torch.cuda.synchronize(self.device)
            emma_rt_free(self.h)
            self.h = None
            self.arena = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
