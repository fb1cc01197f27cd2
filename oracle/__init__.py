"""ctypes front-end of the fp64 CPU oracle (oracle/emma_rt_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / `--impl reference` legs may import this package.  It imports nothing from
paper_1508_07888_b200/ and shares no code with it.

`build()` compiles the C file with gcc (building the checker is not using it).
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "emma_rt_oracle.c")
_HDR = os.path.join(_HERE, "emma_rt_oracle.h")
_LIB = os.path.join(_HERE, "libemma_rt_oracle.so")

MAX_GROUPS = 4
OK, EINVAL, ENOMEM, ENONFINITE, ECFL, ESUBCYCLE = 0, -1, -2, -4, -6, -7
F_U, F_N, F_F, F_X, F_T, F_E, F_N0, F_SUBCYCLES, F_XNEUTRAL = range(9)
FLUX_GLF, FLUX_HLL = 0, 1
BC_PERIODIC, BC_TRANSMISSIVE, BC_REFLECTIVE, BC_INFLOW = 0, 1, 2, 3


def build(force=False):
    """gcc -O2 -fopenmp -shared; rebuilt when the source is newer than the library."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))):
        return _LIB
    cmd = ["gcc", "-std=c99", "-O2", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
           "-o", _LIB, _SRC, "-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


class Phys(C.Structure):
    _fields_ = [("G", C.c_int), ("otsa", C.c_int), ("thermal", C.c_int), ("c", C.c_double),
                ("sigN", C.c_double * MAX_GROUPS), ("sigE", C.c_double * MAX_GROUPS),
                ("Emean", C.c_double * MAX_GROUPS), ("e_tol", C.c_double), ("max_halvings", C.c_int)]


class Diag(C.Structure):
    _fields_ = [("photons_total", C.c_double), ("photons_injected", C.c_double),
                ("photons_absorbed", C.c_double), ("photons_recomb_emitted", C.c_double),
                ("photons_outflow", C.c_double), ("dtau_min", C.c_double),
                ("subcycles_total", C.c_int64), ("subcycles_max", C.c_int64),
                ("halvings_total", C.c_int64), ("n_nonfinite", C.c_int64), ("t_sim", C.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class ChemOut(C.Structure):
    _fields_ = [("absorbed", C.c_double), ("injected", C.c_double), ("recomb", C.c_double),
                ("dtau_min", C.c_double), ("nsub", C.c_int), ("nhalv", C.c_int)]


_lib = None


def lib():
    global _lib
    if _lib is not None:
        return _lib
    L = C.CDLL(build())
    dp = C.POINTER(C.c_double)
    L.orc_chi.restype = C.c_double
    L.orc_chi.argtypes = [C.c_double]
    L.orc_closure.restype = None
    L.orc_closure.argtypes = [dp, C.c_double, dp]
    L.orc_rates.restype = None
    L.orc_rates.argtypes = [C.c_double] + [dp] * 6
    L.orc_temperature.restype = C.c_double
    L.orc_temperature.argtypes = [C.c_double] * 3
    L.orc_energy.restype = C.c_double
    L.orc_energy.argtypes = [C.c_double] * 3
    L.orc_transport_stencil.restype = None
    L.orc_transport_stencil.argtypes = [C.c_double, C.c_double, C.c_double, dp, dp, dp, dp]
    L.orc_chem_cell.restype = C.c_int
    L.orc_transport_stencil_flux.restype = None
    L.orc_transport_stencil_flux.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, dp, dp, dp, dp]
    L.orc_m1_wavespeeds.restype = None
    L.orc_m1_wavespeeds.argtypes = [dp, C.c_double, C.c_int, dp, dp]
    L.orc_set_inflow.restype = C.c_int
    L.orc_set_inflow.argtypes = [C.c_void_p, C.c_int, C.c_int, dp]
    L.orc_set_flux.restype = C.c_int
    L.orc_set_flux.argtypes = [C.c_void_p, C.c_int]
    L.orc_chem_cell.argtypes = [C.POINTER(Phys), C.c_double, C.c_double, dp, dp, dp, dp, C.POINTER(ChemOut)]
    L.orc_create.restype = C.c_void_p
    L.orc_create.argtypes = [C.c_int, C.POINTER(C.c_int), C.c_int, C.POINTER(Phys), C.c_double, C.c_int,
                             C.POINTER(C.c_int64), C.POINTER(C.c_void_p), C.POINTER(C.c_void_p),
                             C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), C.POINTER(C.c_void_p)]
    L.orc_set_sources.restype = C.c_int
    L.orc_set_sources.argtypes = [C.c_void_p, C.c_int64, dp, dp]
    L.orc_step.restype = C.c_int
    L.orc_step.argtypes = [C.c_void_p, C.c_double, C.c_int, C.POINTER(Diag)]
    L.orc_read.restype = C.c_int
    L.orc_read.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, dp, C.c_int64]
    L.orc_level_cells.restype = C.c_int64
    L.orc_level_cells.argtypes = [C.c_void_p, C.c_int]
    L.orc_source_cell.restype = C.c_int64
    L.orc_source_cell.argtypes = [C.c_void_p, C.c_int64, C.POINTER(C.c_int)]
    L.orc_threads.restype = C.c_int
    L.orc_counters.restype = None
    L.orc_counters.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    L.orc_free.restype = None
    L.orc_free.argtypes = [C.c_void_p]
    L.orc_set_amr_transport.restype = C.c_int
    L.orc_set_amr_transport.argtypes = [C.c_void_p, C.c_int]
    L.orc_write_U.restype = C.c_int
    L.orc_write_U.argtypes = [C.c_void_p, C.c_int, C.c_int, dp]
    L.orc_amr_ghost.restype = C.c_int
    L.orc_amr_ghost.argtypes = [C.c_void_p, C.c_int, C.c_int, C.POINTER(C.c_int), C.c_int64, dp]
    L.orc_restrict_U.restype = C.c_int
    L.orc_restrict_U.argtypes = [C.c_void_p]
    _lib = L
    return L


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def make_phys(G, c, sigma_N, sigma_E, E_mean, otsa=1, thermal=1, e_tol=0.1, max_halvings=60):
    p = Phys()
    p.G, p.otsa, p.thermal, p.c, p.e_tol, p.max_halvings = G, otsa, thermal, c, e_tol, max_halvings
    for g in range(G):
        p.sigN[g], p.sigE[g], p.Emean[g] = float(sigma_N[g]), float(sigma_E[g]), float(E_mean[g])
    return p


# ---- stateless pieces -------------------------------------------------------------------------
def chi(f):
    return lib().orc_chi(float(f))


def closure(U, c):
    U = np.ascontiguousarray(U, np.float64)
    P = np.zeros(9)
    lib().orc_closure(_dp(U), float(c), _dp(P))
    return P.reshape(3, 3)


def rates(T):
    """dict(alphaA, alphaB, beta, cool_HI, cool_HII_A, cool_HII_B) at temperature T [K]."""
    v = [C.c_double() for _ in range(6)]
    lib().orc_rates(float(T), *[C.byref(q) for q in v])
    return dict(zip(("alphaA", "alphaB", "beta", "cool_HI", "cool_HII_A", "cool_HII_B"), [q.value for q in v]))


def temperature(e, x, n0):
    return lib().orc_temperature(float(e), float(x), float(n0))


def energy(T, x, n0):
    return lib().orc_energy(float(T), float(x), float(n0))


def transport_stencil(c, dt, dx, U0, Um, Up, flux=None):
    """One cell of Eq. 30+32 from its own state U0[4] and its -/+ neighbours Um[3,4], Up[3,4]
    (flux = FLUX_HLL: the HLL interface flux of reading A19 instead of Eq. 32)."""
    U0 = np.ascontiguousarray(U0, np.float64)
    Um = np.ascontiguousarray(Um, np.float64)
    Up = np.ascontiguousarray(Up, np.float64)
    out = np.zeros(4)
    if flux is None:
        lib().orc_transport_stencil(float(c), float(dt), float(dx), _dp(U0), _dp(Um), _dp(Up), _dp(out))
    else:
        lib().orc_transport_stencil_flux(int(flux), float(c), float(dt), float(dx), _dp(U0), _dp(Um), _dp(Up), _dp(out))
    return out


def m1_wavespeeds(U, c, d):
    """(lmin, lmax): extreme eigenvalues of dF~_d/dU of the M1 system in direction d (reading A19)."""
    U = np.ascontiguousarray(U, np.float64)
    lo, hi = np.zeros(1), np.zeros(1)
    lib().orc_m1_wavespeeds(_dp(U), float(c), int(d), _dp(lo), _dp(hi))
    return float(lo[0]), float(hi[0])


def chem_cell(phys, dt, n0, x, e, U, S=None):
    """Sub-cycled Eq. 43-48 for one cell.  Returns (rc, x, e, U[G,4], ChemOut)."""
    U = np.array(U, np.float64).reshape(phys.G, 4).copy()
    xx, ee = C.c_double(float(x)), C.c_double(float(e))
    out = ChemOut()
    Sp = None
    if S is not None:
        S = np.ascontiguousarray(S, np.float64)
        Sp = _dp(S)
    rc = lib().orc_chem_cell(C.byref(phys), float(dt), float(n0), C.byref(xx), C.byref(ee), _dp(U), Sp, C.byref(out))
    return rc, xx.value, ee.value, U, out


# ---- stateful driver --------------------------------------------------------------------------
def _ptr_array(arrs):
    pa = (C.c_void_p * max(1, len(arrs)))()
    for i, a in enumerate(arrs):
        pa[i] = a.ctypes.data if a is not None else None
    return pa


class Oracle:
    """Same call shape as the library: init(config, amr, fields) / set_sources / step / read."""

    def __init__(self, w, chemistry=None, thermal=None, otsa=None, bc=None, flux=None):
        L = lib()
        self.w = w
        self.G = w.G
        self.phys = make_phys(w.G, w.c_red, w.sigma_N, w.sigma_E, w.E_mean,
                              otsa=w.otsa if otsa is None else otsa,
                              thermal=w.thermal if thermal is None else thermal,
                              e_tol=w.e_tol, max_halvings=w.max_halvings)
        bc_a = (C.c_int * 6)(*(w.bc if bc is None else bc))
        nl = w.n_levels
        n_octs = (C.c_int64 * max(1, nl))(*[len(p) for p in w.parent])
        self._keep = [np.ascontiguousarray(p, np.int64) for p in w.parent]
        par = _ptr_array(self._keep)
        f32 = lambda a: np.ascontiguousarray(a, np.float32)
        U0 = [f32(u) for u in w.U0] if w.U0 is not None else None
        n0 = [f32(a) for a in w.n0]
        x = [f32(a) for a in w.x]
        T = [f32(a) for a in w.T]
        self._keep += [U0, n0, x, T]
        self.h = L.orc_create(w.n, bc_a, w.chemistry if chemistry is None else chemistry, C.byref(self.phys),
                              float(w.L), nl, n_octs, par,
                              _ptr_array(U0) if U0 is not None else None,
                              _ptr_array(n0), _ptr_array(x), _ptr_array(T))
        if not self.h:
            raise ValueError("orc_create failed (invalid arguments or out of memory)")
        for (face, group), U in (getattr(w, "inflow", None) or {}).items():
            if self.set_inflow(face, group, U) != OK:
                raise ValueError("orc_set_inflow(face=%d, group=%d) rejected" % (face, group))
        if flux is not None and L.orc_set_flux(self.h, int(flux)) != OK:
            raise ValueError("orc_set_flux: unknown flux %r" % (flux,))
        if w.src_pos is not None and len(w.src_pos):
            rc = self.set_sources(w.src_pos, w.src_Q)
            if rc != OK:
                raise ValueError("orc_set_sources rc=%d" % rc)

    def set_inflow(self, face, group, U):
        """Ghost state (N, Fx, Fy, Fz) [cgs] of a BC_INFLOW face (0..5 = -x,+x,-y,+y,-z,+z), reading A20."""
        U = np.ascontiguousarray(U, np.float64).reshape(4)
        return lib().orc_set_inflow(self.h, int(face), int(group), _dp(U))

    def set_amr_transport(self, on=True):
        """Standard (non-CRTA) AMR transport of reading A21."""
        return lib().orc_set_amr_transport(self.h, int(bool(on)))

    def write_U(self, level, group, U):
        U = np.ascontiguousarray(U, np.float64).reshape(self.level_cells(level), 4)
        return lib().orc_write_U(self.h, int(level), int(group), _dp(U))

    def amr_ghost(self, level, group, v, coarse_cell):
        """Interpolated state of the virtual level-`level` cell at integer coordinates v inside the coarser leaf (A21)."""
        vv = (C.c_int * 3)(*[int(t) for t in v])
        out = np.zeros(4)
        rc = lib().orc_amr_ghost(self.h, int(level), int(group), vv, int(coarse_cell), _dp(out))
        if rc != OK:
            raise ValueError("orc_amr_ghost rc=%d" % rc)
        return out

    def restrict_U(self):
        return lib().orc_restrict_U(self.h)

    def set_sources(self, pos, Q):
        pos = np.ascontiguousarray(pos, np.float64).reshape(-1, 3)
        Q = np.ascontiguousarray(Q, np.float64).reshape(len(pos), self.G)
        return lib().orc_set_sources(self.h, len(pos), _dp(pos), _dp(Q))

    def step(self, dt, n_steps=1):
        d = Diag()
        rc = lib().orc_step(self.h, float(dt), int(n_steps), C.byref(d))
        return rc, d.as_dict()

    def level_cells(self, level):
        return lib().orc_level_cells(self.h, level)

    def source_cell(self, i):
        lvl = C.c_int()
        cell = lib().orc_source_cell(self.h, i, C.byref(lvl))
        return lvl.value, cell

    def read(self, field, level=0, group=0):
        nc = self.level_cells(level)
        per = {F_U: 4, F_F: 3}.get(field, 1)
        out = np.empty(nc * per, np.float64)
        rc = lib().orc_read(self.h, field, level, group, _dp(out), out.size)
        if rc != OK:
            raise ValueError("orc_read rc=%d" % rc)
        return out.reshape(nc, per) if per > 1 else out

    def counters(self):
        a, b = (C.c_int64 * 8)(), (C.c_int64 * 8)()
        lib().orc_counters(self.h, a, b)
        return list(a), list(b)

    def close(self):
        if self.h:
            lib().orc_free(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
