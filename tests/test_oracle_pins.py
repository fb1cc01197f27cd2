"""T0: pins of the fp64 oracle against what the paper and the mathematics fix.

None of the expected values below comes from the CUDA path.  Each test names the reading(s) of
DESIGN.md it would catch if wrong.  CPU only.
"""
import math
import os
from math import comb

import numpy as np
import pytest

import oracle as O
from workloads import CGS, make_config

from . import brute
from .helpers import groups, tiny_workload

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")) as fh:
    for line in fh:
        line = line.split("#")[0].strip()
        if "=" in line:
            k, v = [s.strip() for s in line.split("=", 1)]
            GOLD[k] = v

C_RED = 0.1 * CGS.c


# ---------------------------------------------------------------- closure (A1, A2, A3)
def test_chi_limits_paper():
    """chi = 1/3 (diffusive) ... 1 (transport); monotone in between."""
    assert O.chi(0.0) == pytest.approx(float(GOLD["chi_diffusive"]), abs=1e-15)
    assert O.chi(1.0) == pytest.approx(float(GOLD["chi_transport"]), abs=1e-15)
    f = np.linspace(0, 1, 201)
    c = np.array([O.chi(v) for v in f])
    assert np.all(np.diff(c) > 0)


def test_closure_trace_and_limits():
    """A1: tr D = 1 (so tr P = N) for any F; D = I/3 at f = 0; D = n(x)n at f = 1."""
    rng = np.random.default_rng(1)
    for _ in range(50):
        N = 10 ** rng.uniform(-8, 2)
        n = rng.standard_normal(3)
        n /= np.linalg.norm(n)
        f = rng.uniform(0, 1.3)                       # > 1 exercises the clip
        P = O.closure([N, *(f * C_RED * N * n)], C_RED)
        assert np.trace(P) == pytest.approx(N, rel=1e-14, abs=0)
        assert np.allclose(P, P.T, rtol=0, atol=1e-16 * N)
        # eigen-structure: n is an eigenvector with eigenvalue chi N
        chi = O.chi(min(f, 1.0))
        assert np.allclose(P @ n, chi * N * n, rtol=1e-12, atol=1e-15 * N)
    P = O.closure([2.0, 0, 0, 0], C_RED)
    assert np.allclose(P, np.eye(3) * 2.0 / 3.0, rtol=1e-15)
    n = np.array([0.6, 0.0, -0.8])
    P = O.closure([1.5, *(C_RED * 1.5 * n)], C_RED)
    assert np.allclose(P, 1.5 * np.outer(n, n), rtol=1e-12, atol=1e-15)
    assert np.all(O.closure([0.0, 0, 0, 0], C_RED) == 0.0)


# ---------------------------------------------------------------- P1 invariance
def test_P1_uniform_zero_flux_is_invariant_bitwise(oracle_mod):
    n = 6
    U0 = np.zeros((1, n ** 3, 4), np.float32)
    U0[0, :, 0] = 3.25e-4
    w = tiny_workload(n, 1, U0=U0, chemistry=0)
    o = O.Oracle(w)
    before = o.read(O.F_U)
    rc, _ = o.step(w.dt, 5)
    assert rc == O.OK
    assert np.array_equal(o.read(O.F_U), before)


# ---------------------------------------------------------------- P2 single-cell worked example
def test_P2_single_cell_worked_example(oracle_mod):
    """One cell N0, rest 0, F = 0.  After one step: centre (1-3nu)N0; each face neighbour N = nu N0/2 and an
    outward normal flux nu c N0/6 (c^2 P_dd = c^2 N0/3 at f = 0); everything else 0; sum N conserved.
    Catches: sign of Eq. 30/32, the factor 1/2, A1 at f = 0 (isotropic 1/3), unsplit sum (A4)."""
    n, N0 = 7, 2.0
    c = n // 2
    U0 = np.zeros((1, n, n, n, 4), np.float32)
    U0[0, c, c, c, 0] = N0
    w = tiny_workload(n, 1, U0=U0.reshape(1, -1, 4), chemistry=0, courant=0.6)
    nu = w.c_red * w.dt / w.dx
    assert nu == pytest.approx(0.2)
    o = O.Oracle(w)
    rc, d = o.step(w.dt, 1)
    assert rc == O.OK
    U = o.read(O.F_U).reshape(n, n, n, 4)              # [z, y, x, q]
    exp = np.zeros_like(U)
    exp[c, c, c, 0] = (1 - 3 * nu) * N0
    fl = nu * w.c_red * N0 / 6
    for d_, (dz, dy, dx) in enumerate(((0, 0, 1), (0, 1, 0), (1, 0, 0))):
        for s in (+1, -1):
            exp[c + s * dz, c + s * dy, c + s * dx, 0] = nu * N0 / 2
            exp[c + s * dz, c + s * dy, c + s * dx, 1 + d_] = s * fl
    assert np.allclose(U[..., 0], exp[..., 0], rtol=1e-14, atol=0)
    assert np.allclose(U[..., 1:], exp[..., 1:], rtol=1e-14, atol=1e-14 * fl)
    assert U[..., 0].sum() == pytest.approx(N0, rel=1e-14, abs=0)
    # reduced flux of the neighbours is 1/3
    assert abs(U[c, c, c + 1, 1]) / (w.c_red * U[c, c, c + 1, 0]) == pytest.approx(1 / 3, rel=1e-13, abs=0)


# ---------------------------------------------------------------- P3 free-streaming beam
def test_P3_free_streaming_beam_binomial(oracle_mod):
    """F = c N x^: GLF reduces to first-order upwind at speed c~ (A3), f stays 1 (chi = 1 branch of A1):
    N_i^k = sum_j C(k,j) nu^j (1-nu)^(k-j) N^0_{i-j}; centroid moves nu cells per step."""
    n, k = 16, 6
    prof = np.zeros(n)
    prof[3:6] = [1.0, 2.5, 0.5]
    U0 = np.zeros((1, n, n, n, 4), np.float32)
    U0[0, :, :, :, 0] = prof[None, None, :]
    w = tiny_workload(n, 1, U0=U0.reshape(1, -1, 4), chemistry=0, courant=0.75)
    # F must equal c*N exactly in fp64 after the fp32 input rounding: build it from the rounded N
    U0[0, ..., 1] = 0
    o = O.Oracle(w)
    # overwrite Fx = c N in fp64 by re-creating with exact product is not possible through fp32 inputs;
    # instead choose c so that c*N is exactly representable: use a power-of-two speed.
    w2 = tiny_workload(n, 1, c_red=2.0 ** 31, chemistry=0, courant=0.75,
                       U0=np.concatenate([U0[0, ..., :1], U0[0, ..., :1] * np.float32(2.0 ** 31),
                                          np.zeros_like(U0[0, ..., :2])], axis=-1).reshape(1, -1, 4))
    nu = w2.c_red * w2.dt / w2.dx
    assert nu == pytest.approx(0.25)
    o = O.Oracle(w2)
    rc, _ = o.step(w2.dt, k)
    assert rc == O.OK
    U = o.read(O.F_U).reshape(n, n, n, 4)
    exp = np.zeros(n)
    for i in range(n):
        exp[i] = sum(comb(k, j) * nu ** j * (1 - nu) ** (k - j) * prof[(i - j) % n] for j in range(k + 1))
    assert np.allclose(U[5, 7, :, 0], exp, rtol=1e-13, atol=1e-15)
    assert np.allclose(U[..., 1], w2.c_red * U[..., 0], rtol=1e-13, atol=1e-6)       # stays free-streaming
    assert np.all(U[..., 2:] == 0)
    x = np.arange(n)
    cen0 = (prof * x).sum() / prof.sum()
    cen = (U[0, 0, :, 0] * x).sum() / U[0, 0, :, 0].sum()
    assert cen - cen0 == pytest.approx(k * nu, rel=1e-12, abs=0)                           # speed = c~


# ---------------------------------------------------------------- P4 photon budget
@pytest.mark.parametrize("case", ["cfg1", "transmissive", "crta", "non_otsa"])
def test_P4_photon_budget_closes_every_step(oracle_mod, case):
    """A5, A12, A15: d(sum N dV) = injected - absorbed + recomb_emitted - outflow, every step, to rounding."""
    if case == "cfg1":
        w = make_config(1, n=12, n_steps=12)
    elif case == "transmissive":
        w = make_config(1, n=8, n_steps=30)
        w.bc = (1, 1, 2, 1, 1, 2)
    elif case == "non_otsa":
        w = make_config(1, n=8, n_steps=12)
        w.otsa = 0
    else:
        w = make_config(4, n=8, n_steps=8, n_src=3)
        assert w.n_levels == 2 and len(w.parent[1]) > 0
    o = O.Oracle(w)
    rc, d = o.step(w.dt, 0)
    prev = d["photons_total"]
    saw_out = False
    for s in range(w.n_steps):
        rc, d = o.step(w.dt, 1)
        assert rc == O.OK
        rhs = d["photons_injected"] - d["photons_absorbed"] + d["photons_recomb_emitted"] - d["photons_outflow"]
        scale = max(d["photons_total"], d["photons_injected"])
        assert abs((d["photons_total"] - prev) - rhs) <= 1e-12 * scale
        assert d["photons_injected"] == pytest.approx(w.src_Q.sum() * w.dt, rel=1e-13, abs=0)   # A12: sum Q dt exactly
        saw_out |= d["photons_outflow"] > 0
        if case == "non_otsa":
            assert d["photons_recomb_emitted"] > 0
        prev = d["photons_total"]
    if case == "transmissive":
        assert saw_out


# ---------------------------------------------------------------- P5 decay / A5
def test_P5_absorption_decay_and_dtau_to_zero(oracle_mod):
    """A5: backward Euler of Eq. 33-34 with x^p in the sink: N1 = N0/(1 + c sigma (1-x^p) n0 dtau), F likewise;
    dtau -> 0 gives the identity (the printed denominator without dtau would not)."""
    gr = groups(1)
    ph = O.make_phys(1, C_RED, gr["sigma_N"], gr["sigma_E"], gr["E_mean"], thermal=0)
    n0, x, T = 0.5, 0.25, 1.0e4
    e = O.energy(T, x, n0)
    U = np.array([[3e-3, 1e6, -2e6, 5e5]])
    dt = 3.0e8
    for _ in range(5):
        rc, x1, e1, U1, out = O.chem_cell(ph, dt, n0, x, e, U)
        assert rc == O.OK and out.nsub == 1 and out.nhalv == 0
        den = 1 + C_RED * gr["sigma_N"][0] * (1 - x) * n0 * dt
        assert np.allclose(U1, U / den, rtol=1e-15)
        assert out.absorbed == pytest.approx((U[0, 0] - U1[0, 0]), rel=1e-12, abs=0)       # sink counts what N lost
        assert O.temperature(e1, x1, n0) == pytest.approx(T, rel=1e-14, abs=0)            # isothermal mode holds T
        x, e, U = x1, e1, U1
    rc, x1, e1, U1, out = O.chem_cell(ph, 1e-9, n0, x, e, U)
    assert np.allclose(U1, U, rtol=1e-14) and x1 == pytest.approx(x, rel=1e-14, abs=0)


# ---------------------------------------------------------------- P6 collisional equilibrium
@pytest.mark.parametrize("otsa", [1, 0])
def test_P6_collisional_ionisation_equilibrium(oracle_mod, otsa):
    """Eq. 45 without radiation, T held: fixed point x = beta/(alpha+beta), independent of dtau
    (backward-Euler fixed point).  alpha = alpha_B under OTSA, alpha_A otherwise."""
    gr = groups(1)
    T = 2.0e4
    r = O.rates(T)
    al = r["alphaB"] if otsa else r["alphaA"]
    xeq = r["beta"] / (al + r["beta"])
    for dt in (1e13, 3e14):
        # otsa = 0: recombination photons (A6) would re-ionise within the same sub-step; a zero cross-section
        # keeps radiation out of Eq. 45 so the textbook fixed point with alpha_A applies
        sig = gr["sigma_N"] if otsa else [0.0]
        ph = O.make_phys(1, C_RED, sig, gr["sigma_E"], gr["E_mean"], thermal=0, otsa=otsa)
        n0, x = 1.0, 0.3
        e = O.energy(T, x, n0)
        U = np.zeros((1, 4))
        for _ in range(400):
            rc, x, e, U, out = O.chem_cell(ph, dt, n0, x, e, U)
            U[:] = 0.0
        assert x == pytest.approx(xeq, rel=1e-10, abs=0)


# ---------------------------------------------------------------- P7 photo-ionisation equilibrium
def test_P7_photoionisation_equilibrium(oracle_mod):
    """Eq. 43 + 45 coupled, uniform S, T held, OTSA:
    (alpha_B+beta) n0^2 x^2 - beta n0^2 x - S = 0  and  N = S/(c sigma (1-x) n0)."""
    gr = groups(1)
    T, n0 = 1.0e4, 1.0e-2
    r = O.rates(T)
    a, b = r["alphaB"], r["beta"]
    S = 0.4 * a * n0 * n0
    xeq = (b * n0 ** 2 + math.sqrt(b ** 2 * n0 ** 4 + 4 * (a + b) * n0 ** 2 * S)) / (2 * (a + b) * n0 ** 2)
    Neq = S / (C_RED * gr["sigma_N"][0] * (1 - xeq) * n0)
    ph = O.make_phys(1, C_RED, gr["sigma_N"], gr["sigma_E"], gr["E_mean"], thermal=0)
    x, U = 0.1, np.zeros((1, 4))
    e = O.energy(T, x, n0)
    for _ in range(3000):
        rc, x, e, U, out = O.chem_cell(ph, 2e13, n0, x, e, U, S=[S])
    assert x == pytest.approx(xeq, rel=1e-9, abs=0)
    assert U[0, 0] == pytest.approx(Neq, rel=1e-9, abs=0)
    assert 0 < xeq < 1


# ---------------------------------------------------------------- P8 Stroemgren sphere
def _stromgren_numbers(n0=1e-3, Q=5e48, T=1e4):
    aB = O.rates(T)["alphaB"]
    Rs = (3 * Q / (4 * math.pi * n0 ** 2 * aB)) ** (1 / 3)
    return Rs, 1.0 / (aB * n0)


def test_P8_stromgren_textbook_numbers(oracle_mod):
    """north_star: R_s = (3Q / 4 pi n_H^2 alpha_B)^(1/3); with alpha_B(1e4 K) = 2.59e-13 (textbook) this is 5.4 kpc."""
    Rs, trec = _stromgren_numbers()
    assert O.rates(1e4)["alphaB"] == pytest.approx(2.59e-13, rel=2e-3, abs=0)       # Osterbrock's case-B value
    assert O.rates(1e4)["alphaA"] == pytest.approx(4.18e-13, rel=4e-2, abs=0)       # Osterbrock's case-A value
    assert Rs / CGS.kpc == pytest.approx(5.4, abs=0.05)
    assert trec / CGS.Myr == pytest.approx(122.3, abs=0.5)


@pytest.mark.slow
def test_P8_ionised_radius_converges_to_stromgren(oracle_mod):
    """Whole coupled scheme, isothermal 1e4 K, OTSA, 16^3 box of 16 kpc, c~ = 0.01 c, run to 4 t_rec.
    The Stroemgren balance Q = alpha_B n^2 sum x^2 dV fixes the recombination-weighted radius
    r_rec = (3 sum x^2 dV / 4 pi)^(1/3) -> R_s (1-exp(-t/t_rec))^(1/3); the plain ionised radius
    r_I = (3 sum x dV / 4 pi)^(1/3) lies above it by the (thick, GLF-diffused, 1 kpc cells) front: x > x^2 there."""
    n = 16
    w = tiny_workload(n, 1, L=16 * CGS.kpc, c_red=0.01 * CGS.c, n0=1e-3, x=1e-6, T=1e4, thermal=0,
                      src_pos=[[0.5 + 0.5 / n] * 3], src_Q=[[5e48]], bc=(1,) * 6)
    Rs, trec = _stromgren_numbers()
    o = O.Oracle(w)
    done = 0
    for frac in (0.5, 1.0, 2.0, 4.0):
        target = int(frac * trec / w.dt)
        rc, d = o.step(w.dt, target - done)
        done = target
        assert rc == O.OK
        x = o.read(O.F_X)
        r_I = (3 * x.sum() * w.dx ** 3 / (4 * math.pi)) ** (1 / 3)
        r_rec = (3 * (x * x).sum() * w.dx ** 3 / (4 * math.pi)) ** (1 / 3)
        ana = Rs * (1 - math.exp(-frac)) ** (1 / 3)
        assert r_rec == pytest.approx(ana, rel=0.09, abs=0), (frac, r_rec / ana)
        assert 0.98 * ana < r_I < 1.12 * ana, (frac, r_I / ana)
    assert r_rec / Rs == pytest.approx(0.994, abs=0.03)          # (1 - e^-4)^(1/3) = 0.994
    assert done > 1000


def test_P8_early_time_config1(oracle_mod):
    """Config 1 itself (100 steps): r_I(t) ~ R_s(1-exp(-t/t_rec))^(1/3), plus the initial x = 1.2e-3 volume."""
    w = make_config(1)
    o = O.Oracle(w)
    rc, d = o.step(w.dt, w.n_steps)
    assert rc == O.OK
    x = o.read(O.F_X)
    T = o.read(O.F_T)
    V_ion = x.sum() * w.dx ** 3
    # analytic growth at the gas temperature behind the front (~2.4e4 K), plus the initial ionised volume
    aB = O.rates(float(np.median(T[x > 0.9])))["alphaB"]
    Rs = (3 * 5e48 / (4 * math.pi * 1e-6 * aB)) ** (1 / 3)
    t = d["t_sim"]
    V_ana = 4 * math.pi / 3 * Rs ** 3 * (1 - math.exp(-t * aB * 1e-3)) + 1.2e-3 * w.L ** 3
    assert V_ion == pytest.approx(V_ana, rel=0.08, abs=0)
    # P9: no-cooling temperature bound  T <= (Sigma_E/sigma_N) / (3 k_B)   (A8, A10)
    SigE = w.sigma_E[0] * w.E_mean[0] - w.sigma_N[0] * 13.6 * CGS.eV
    Tmax = SigE / w.sigma_N[0] / (3 * CGS.k_B)
    assert Tmax == pytest.approx(24447, rel=2e-3, abs=0)
    assert T.max() <= Tmax and T.max() > 0.97 * Tmax


# ---------------------------------------------------------------- A10 round trip
def test_A10_temperature_energy_roundtrip(oracle_mod):
    rng = np.random.default_rng(3)
    for _ in range(100):
        T, x, n0 = 10 ** rng.uniform(1, 6), rng.uniform(0, 1), 10 ** rng.uniform(-6, 2)
        assert O.temperature(O.energy(T, x, n0), x, n0) == pytest.approx(T, rel=1e-15, abs=0)
    # fully ionised hydrogen: e = 3 n k T (two particles per atom)
    assert O.energy(1e4, 1.0, 1.0) == pytest.approx(3 * CGS.k_B * 1e4, rel=1e-15, abs=0)


# ---------------------------------------------------------------- A9: the 10 % rule
def test_A9_energy_step_rule(oracle_mod):
    """Every accepted sub-step changes e by <= 10 %: after k accepted sub-steps
    e_final/e_initial lies in [0.9^k, 1.1^k]; a strongly photo-heated cold cell needs >= ln(ratio)/ln(1.1)."""
    gr = groups(1)
    ph = O.make_phys(1, C_RED, gr["sigma_N"], gr["sigma_E"], gr["E_mean"])
    n0, x, T = 1e-3, 1.2e-3, 100.0
    e = O.energy(T, x, n0)
    rc, x1, e1, U1, out = O.chem_cell(ph, 6.4e10, n0, x, e, np.array([[1e-3, 0, 0, 0]]))
    assert rc == O.OK
    assert out.nsub >= math.log(e1 / e) / math.log(1 + float(GOLD["energy_variation_max"]))
    assert out.nhalv >= 1
    assert e1 / e <= 1.1 ** out.nsub
    # no heating, no cooling to speak of: one sub-step of the full dt
    rc, x2, e2, U2, out2 = O.chem_cell(ph, 6.4e10, n0, x, e, np.zeros((1, 4)))
    assert out2.nsub == 1 and out2.nhalv == 0


# ---------------------------------------------------------------- P10 reflective octant symmetry (A13)
def test_P10_reflective_octant_symmetry(oracle_mod):
    """Corner source + reflective on the 3 adjacent faces == one octant of the mirrored 2n box with the 8 central
    cells emitting (PAPER.md:436 'flux inversion' = face-normal component)."""
    n = 6
    q = 1.0 / (2 * n)
    wa = tiny_workload(n, 1, bc=(2, 1, 2, 1, 2, 1), src_pos=[[q, q, q]], src_Q=[[5e48]], courant=0.9)
    pos = [[0.5 + sx * q / 2, 0.5 + sy * q / 2, 0.5 + sz * q / 2] for sx in (-1, 1) for sy in (-1, 1) for sz in (-1, 1)]
    wb = tiny_workload(2 * n, 1, bc=(1,) * 6, src_pos=pos, src_Q=[[5e48]] * 8, courant=0.9)
    assert wa.dx == pytest.approx(wb.dx)
    oa, ob = O.Oracle(wa), O.Oracle(wb)
    oa.step(wa.dt, 10)
    ob.step(wb.dt, 10)
    Ua = oa.read(O.F_U).reshape(n, n, n, 4)
    Ub = ob.read(O.F_U).reshape(2 * n, 2 * n, 2 * n, 4)[n:, n:, n:]
    assert Ua[..., 0].max() > 0
    assert np.allclose(Ua, Ub, rtol=1e-11, atol=1e-11 * np.abs(Ub).max())
    xa = oa.read(O.F_X).reshape(n, n, n)
    xb = ob.read(O.F_X).reshape(2 * n, 2 * n, 2 * n)[n:, n:, n:]
    assert np.allclose(xa, xb, rtol=1e-11)


# ---------------------------------------------------------------- P11 CRTA degeneracy (A14)
def test_P11_crta_uniform_refined_patch_equals_unrefined(oracle_mod):
    """A refined patch whose leaves all carry the parent's state must reproduce the unrefined run bit for bit."""
    n = 6
    rng = np.random.default_rng(5)
    n0 = (1e-3 * np.exp(rng.standard_normal(n ** 3))).astype(np.float32)
    src = dict(src_pos=[[0.08, 0.08, 0.08]], src_Q=[[3e48, 1e48, 2e47]])
    p1 = np.array([40, 41, 100, 215], np.int64)                    # coarse cells to split (source cell 0 is not)
    p2 = np.array([3, 8 * 2 + 5], np.int64)                        # level-1 cells to split
    n01 = np.repeat(n0[p1], 8)
    n02 = np.repeat(n01[p2], 8)
    wu = tiny_workload(n, 3, n0=n0, **src)
    wr = tiny_workload(n, 3, n0=n0, parent=[p1, p2], n0_lv=[n01, n02], **src)
    ou, orf = O.Oracle(wu), O.Oracle(wr)
    ou.step(wu.dt, 15)
    orf.step(wr.dt, 15)
    for g in range(3):
        assert np.array_equal(ou.read(O.F_U, 0, g), orf.read(O.F_U, 0, g))
    assert np.array_equal(ou.read(O.F_X), orf.read(O.F_X))
    assert np.array_equal(ou.read(O.F_T), orf.read(O.F_T))
    assert np.array_equal(orf.read(O.F_X, 1)[:8], np.repeat(ou.read(O.F_X)[40], 8))
    assert ou.read(O.F_X).max() > 0.5                              # something actually happened


def test_A14_restriction_is_children_mean_and_source_in_leaf(oracle_mod):
    """Split cells hold the mean of their 8 children for n0, x, e after every step; a source inside a refined
    cell lands in the leaf containing it (A12) with S = Q / dV_leaf, and the photon budget uses leaf volumes."""
    w = make_config(4, n=8, n_steps=3, n_src=2)
    o = O.Oracle(w)
    lvl, cell = o.source_cell(0)
    assert lvl == 2
    rc, d = o.step(w.dt, 3)
    assert rc == O.OK
    for l in (1, 2):
        for f in (O.F_X, O.F_E, O.F_N0):
            ch = o.read(f, l).reshape(-1, 8).mean(axis=1)
            assert np.allclose(o.read(f, l - 1)[w.parent[l - 1]], ch, rtol=1e-14)
    # the leaf hosting source 0 ionises first
    x2 = o.read(O.F_X, 2)
    assert x2[cell] == x2.max()


# ---------------------------------------------------------------- P12 Fig. 6 call counts
def test_P12_fig6_crta_engine_call_counts(oracle_mod):
    """Fig. 6 / PAPER.md:455: dt_dyn = 4 dt_rad with 2 refined levels => 4 transport calls (coarse level only)
    and 12 chemistry calls (3 levels x 4).  Counted here as engine sweeps over the cells of a level."""
    w = make_config(4, n=8, n_steps=4, n_src=1)
    o = O.Oracle(w)
    k = int(GOLD["fig6_dyn_over_rad"])
    o.step(w.dt, k)
    tr, ch = o.counters()
    n_leaf = [w.n ** 3 - len(w.parent[0]), 8 * len(w.parent[0]) - len(w.parent[1]), 8 * len(w.parent[1])]
    transport_calls = sum(1 for l in range(3) if tr[l]) * k
    assert tr[0] == k * w.n ** 3 and tr[1] == 0 and tr[2] == 0
    assert transport_calls == int(GOLD["fig6_crta_transport_calls"])
    assert [ch[l] for l in range(3)] == [k * m for m in n_leaf]
    chem_calls = sum(ch[l] // n_leaf[l] for l in range(3))
    assert chem_calls == int(GOLD["fig6_crta_chemistry_calls"])


# ---------------------------------------------------------------- P13 brute force
@pytest.mark.parametrize("n,G,seed", [(4, 1, 0), (5, 3, 1), (8, 3, 2)])
def test_P13_bruteforce_transcription(oracle_mod, n, G, seed):
    """Oracle vs the independent numpy transcription in tests/brute.py: random states, sources, 2 coupled steps."""
    rng = np.random.default_rng(100 + seed)
    gr = groups(G)
    nc = n ** 3
    c = C_RED
    U0 = np.zeros((G, nc, 4))
    for g in range(G):
        N = 10 ** rng.uniform(-6, -2, nc)
        d = rng.standard_normal((nc, 3))
        d /= np.linalg.norm(d, axis=1)[:, None]
        U0[g, :, 0] = N
        U0[g, :, 1:] = (rng.uniform(0, 1.0, nc) * c * N)[:, None] * d
    U0 = U0.astype(np.float32)
    n0 = (10 ** rng.uniform(-4, -1, nc)).astype(np.float32)
    x = (10 ** rng.uniform(-4, 0, nc)).astype(np.float32).clip(max=0.9999)
    T = (10 ** rng.uniform(2, 4.5, nc)).astype(np.float32)
    pos = rng.random((2, 3))
    Q = 10 ** rng.uniform(47, 48.5, (2, G))
    w = tiny_workload(n, G, n0=n0, x=x, T=T, U0=U0, src_pos=pos, src_Q=Q)
    o = O.Oracle(w)
    # brute-force side
    Ub = U0.astype(np.float64).reshape(G, n, n, n, 4)
    xb = x.astype(np.float64).copy()
    eb = 1.5 * (1 + xb) * n0.astype(np.float64) * brute.K_B * T.astype(np.float64)
    S = np.zeros((nc, G))
    for s in range(2):
        ijk = np.floor(pos[s] * n).astype(int)
        S[ijk[0] + n * (ijk[1] + n * ijk[2])] += Q[s] / w.dx ** 3
    nsub_b = np.zeros(nc, int)
    for step in range(2):
        Ub = np.stack([brute.transport_periodic(Ub[g], c, w.dt, w.dx) for g in range(G)])
        flat = Ub.reshape(G, nc, 4)
        for i in range(nc):
            Ui, xb[i], eb[i], nacc, nh = brute.chem_cell(flat[:, i, :], float(n0[i]), xb[i], eb[i], S[i], w.dt, c,
                                                         gr["sigma_N"], gr["sigma_E"], gr["E_mean"])
            flat[:, i, :] = Ui
            nsub_b[i] = nacc | (nh << 16)
        Ub = flat.reshape(G, n, n, n, 4)
    rc, d = o.step(w.dt, 2)
    assert rc == O.OK
    for g in range(G):
        Uo = o.read(O.F_U, 0, g)
        ref = Ub[g].reshape(nc, 4)
        assert np.allclose(Uo[:, 0], ref[:, 0], rtol=1e-10, atol=0)
        assert np.allclose(Uo[:, 1:], ref[:, 1:], rtol=1e-9, atol=1e-10 * c * ref[:, 0].max())
    assert np.allclose(o.read(O.F_X), xb, rtol=1e-10)
    assert np.allclose(o.read(O.F_E), eb, rtol=1e-10)
    assert np.array_equal(o.read(O.F_SUBCYCLES).astype(np.int64), nsub_b)
    assert (nsub_b & 0xFFFF).max() > 1                               # the sub-cycling branch was exercised


# ---------------------------------------------------------------- boundary / error behaviour of the driver
def test_cfl_and_argument_errors(oracle_mod):
    w = make_config(1, n=4)
    o = O.Oracle(w)
    rc, _ = o.step(1.01 * w.dx / (3 * w.c_red), 1)
    assert rc == O.ECFL                                              # A4: dt <= dx/(3c)
    assert o.step(w.dx / (3 * w.c_red), 1)[0] == O.OK
    assert o.set_sources([[1.0, 0.5, 0.5]], [[1e48]]) == O.EINVAL
    assert o.set_sources([[0.5, 0.5, 0.5]], [[-1.0]]) == O.EINVAL


def test_thread_count_does_not_change_results(oracle_mod):
    """The OpenMP loops reorder nothing: 1 thread and all threads give identical bits."""
    import subprocess
    import sys
    code = ("import numpy as np, oracle as O; from workloads import make_config;"
            "w=make_config(4,n=8,n_steps=3,n_src=2); o=O.Oracle(w); rc,d=o.step(w.dt,3);"
            "print(repr((d['photons_total'],d['photons_absorbed'],float(o.read(O.F_X).sum()),float(o.read(O.F_U,0,1).sum()))))")
    outs = []
    for nt in ("1", "4"):
        env = dict(os.environ, OMP_NUM_THREADS=nt)
        outs.append(subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True,
                                   cwd=os.path.dirname(os.path.dirname(__file__)), check=True).stdout)
    assert outs[0] == outs[1]


# ------------------------------------------------------------------------------------------------------------
# HLL interface flux (PAPER.md:250 names it, prints nothing: DESIGN.md reading A19)
# ------------------------------------------------------------------------------------------------------------
def _flux_vec(U, c, d):
    P = O.closure(U, c)
    return np.array([U[1 + d], c * c * P[d, 0], c * c * P[d, 1], c * c * P[d, 2]])


def test_H1_wavespeeds_are_the_extreme_eigenvalues_of_the_flux_jacobian(oracle_mod):
    """lmin/lmax of A19 against the eigenvalues of a central-difference Jacobian of F~_d(U) built from orc_closure:
    the mathematics (the closure of Eq. 22-23) fixes them, whatever formula the oracle uses."""
    rng = np.random.default_rng(19)
    c = 1.0
    worst = 0.0
    for _ in range(300):
        f = rng.uniform(0.0, 0.995)
        dirn = rng.standard_normal(3)
        dirn /= np.linalg.norm(dirn)
        U = np.array([1.0, *(f * c * dirn)])
        for d in range(3):
            J = np.zeros((4, 4))
            h = 1e-6
            for k in range(4):
                e = np.zeros(4)
                e[k] = h
                J[:, k] = (_flux_vec(U + e, c, d) - _flux_vec(U - e, c, d)) / (2 * h)
            ev = np.linalg.eigvals(J)
            assert np.abs(ev.imag).max() < 1e-6                       # hyperbolic
            lo, hi = O.m1_wavespeeds(U, c, d)
            worst = max(worst, abs(ev.real.min() - lo), abs(ev.real.max() - hi))
    assert worst < 2e-7, worst


def test_H2_wavespeed_limits_and_scaling(oracle_mod):
    c = C_RED
    lo, hi = O.m1_wavespeeds([2.0, 0, 0, 0], c, 1)
    assert lo == pytest.approx(-c / math.sqrt(3), rel=1e-14, abs=0) and hi == pytest.approx(c / math.sqrt(3), rel=1e-14, abs=0)
    assert O.m1_wavespeeds([1.0, c, 0, 0], c, 0) == pytest.approx((c, c), rel=1e-14, abs=0)        # free streaming along d
    assert O.m1_wavespeeds([1.0, c, 0, 0], c, 2) == pytest.approx((0.0, 0.0), abs=1e-9 * c)  # ... across d
    assert O.m1_wavespeeds([1.0, -3 * c, 0, 0], c, 0) == pytest.approx((-c, -c), rel=1e-14, abs=0)  # f clipped to 1
    assert O.m1_wavespeeds([0.0, 1.0, 0, 0], c, 0) == pytest.approx((-c / math.sqrt(3), c / math.sqrt(3)))  # N<=0: f=0
    # |l| <= c always, lmin <= lmax, and the pair agrees with the independent cancellation-free transcription
    rng = np.random.default_rng(3)
    U = np.concatenate([10 ** rng.uniform(-6, -2, (500, 1)), np.zeros((500, 3))], axis=1)
    dirn = rng.standard_normal((500, 3))
    dirn /= np.linalg.norm(dirn, axis=1)[:, None]
    U[:, 1:] = rng.uniform(0, 1.2, (500, 1)) * c * U[:, :1] * dirn
    for d in range(3):
        blo, bhi = brute.wavespeeds(U, c, d)
        for i in range(500):
            lo, hi = O.m1_wavespeeds(U[i], c, d)
            assert -c * (1 + 1e-12) <= lo <= hi <= c * (1 + 1e-12)
            assert lo == pytest.approx(blo[i], abs=2e-8 * c) and hi == pytest.approx(bhi[i], abs=2e-8 * c)


def test_H3_hll_single_cell_worked_example(oracle_mod):
    """One hot cell in the dark, F = 0: every state has f = 0, so l = -/+ c/sqrt(3) and HLL is Eq. 32 with c/sqrt(3)
    as its dissipation speed: centre (1 - sqrt(3) nu) N0, face neighbours nu N0/(2 sqrt 3), outward flux nu c N0/6."""
    n, c = 8, C_RED
    U0 = np.zeros((1, n ** 3, 4), np.float32)
    ctr = 3 + n * (4 + n * 2)
    U0[0, ctr, 0] = 1.0
    w = tiny_workload(n, 1, U0=U0, chemistry=0)
    o = O.Oracle(w, flux=O.FLUX_HLL)
    rc, _ = o.step(w.dt, 1)
    assert rc == O.OK
    U = o.read(O.F_U).reshape(n, n, n, 4)
    nu = c * w.dt / w.dx
    assert U[2, 4, 3, 0] == pytest.approx(1 - math.sqrt(3) * nu, rel=1e-13, abs=0)
    for (dz, dy, dx_), comp in (((0, 0, 1), 1), ((0, 0, -1), 1), ((0, 1, 0), 2), ((0, -1, 0), 2), ((1, 0, 0), 3), ((-1, 0, 0), 3)):
        v = U[2 + dz, 4 + dy, 3 + dx_]
        sgn = dz + dy + dx_
        assert v[0] == pytest.approx(nu / (2 * math.sqrt(3)), rel=1e-13, abs=0)
        assert v[comp] == pytest.approx(sgn * nu * c / 6, rel=1e-13, abs=0)
        assert np.abs(np.delete(v[1:], comp - 1)).max() == 0.0
    assert U[..., 0].sum() == pytest.approx(1.0, rel=1e-13, abs=0)


def test_H4_hll_free_streaming_beam_is_exact_upwind(oracle_mod):
    """F = c N x^ (f = 1 along x): l+ = c, l- = 0, so HLL is first-order upwind: the binomial closed form of P3, F = cN
    kept, and NOTHING leaks through the transverse faces (l = 0 there)."""
    n, c, k = 16, 2.0 ** 31, 6                  # power-of-two speed: c N is exact in fp32, so f = 1 exactly (as in P3)
    rng = np.random.default_rng(5)
    prof = rng.uniform(0.5, 2.0, n).astype(np.float32)
    U0 = np.zeros((1, n, n, n, 4), np.float32)
    U0[0, ..., 0] = prof[None, None, :]
    U0[0, ..., 1] = np.float32(c) * prof[None, None, :]
    U0 = U0.reshape(1, n ** 3, 4)
    w = tiny_workload(n, 1, U0=U0, c_red=c, chemistry=0, courant=0.75)
    o = O.Oracle(w, flux=O.FLUX_HLL)
    rc, _ = o.step(w.dt, k)
    assert rc == O.OK
    nu = c * w.dt / w.dx
    p0 = prof.astype(np.float64)
    expect = sum(comb(k, m) * nu ** m * (1 - nu) ** (k - m) * np.roll(p0, m) for m in range(k + 1))
    U = o.read(O.F_U).reshape(n, n, n, 4)
    assert np.allclose(U[3, 7, :, 0], expect, rtol=1e-12)
    assert np.allclose(U[..., 1], c * U[..., 0], rtol=1e-12) and np.abs(U[..., 2:]).max() == 0.0


@pytest.mark.parametrize("n,G,seed", [(4, 1, 0), (6, 3, 1), (8, 2, 2)])
def test_H5_hll_bruteforce_transcription_and_conservation(oracle_mod, n, G, seed):
    """Oracle HLL transport vs the independent numpy transcription (tests/brute.py), random states incl. f > 1 and dark
    cells, 3 steps; sum N conserved to rounding on the periodic box."""
    rng = np.random.default_rng(200 + seed)
    nc, c = n ** 3, C_RED
    U0 = np.zeros((G, nc, 4))
    for g in range(G):
        N = 10 ** rng.uniform(-6, -2, nc)
        N[rng.random(nc) < 0.1] = 0.0
        d = rng.standard_normal((nc, 3))
        d /= np.linalg.norm(d, axis=1)[:, None]
        U0[g, :, 0] = N
        U0[g, :, 1:] = (rng.uniform(0, 1.1, nc) * c * N)[:, None] * d
    U0 = U0.astype(np.float32)
    w = tiny_workload(n, G, U0=U0, chemistry=0)
    o = O.Oracle(w, flux=O.FLUX_HLL)
    Ub = U0.astype(np.float64).reshape(G, n, n, n, 4)
    for _ in range(3):
        Ub = np.stack([brute.transport_periodic_hll(Ub[g], c, w.dt, w.dx) for g in range(G)])
    rc, _ = o.step(w.dt, 3)
    assert rc == O.OK
    for g in range(G):
        U = o.read(O.F_U, 0, g).reshape(n, n, n, 4)
        scale = np.abs(Ub[g][..., 0]).max()
        # 1e-8: at f -> 1 (the limiter of A19 puts states there) the speeds are sqrt-sensitive, the two algebraic forms of the
        # radicand differ by ~sqrt(eps)
        assert np.abs(U[..., 0] - Ub[g][..., 0]).max() <= 1e-8 * scale
        assert np.abs(U[..., 1:] - Ub[g][..., 1:]).max() <= 1e-8 * c * scale
        assert U[..., 0].sum() == pytest.approx(U0[g, :, 0].astype(np.float64).sum(), rel=1e-12, abs=0)


def test_H6_hll_is_less_diffusive_than_glf(oracle_mod):
    """HLL is 'less diffusive' than GLF, whose weak shadows come from light leaking sideways.  A beam
    of finite width along x: after 10 steps the photons found outside the beam's own rows are far fewer with HLL."""
    n, c = 16, 2.0 ** 31                        # power-of-two speed: F = c N is exact in fp32, so f = 1, not 1 + 1e-8
    U0 = np.zeros((1, n, n, n, 4))              # (a non-realizable f > 1 would take the -/+c bounds of A19)
    U0[0, 6:10, 6:10, :, 0] = 1.0
    U0[0, 6:10, 6:10, :, 1] = c
    U0 = U0.reshape(1, n ** 3, 4).astype(np.float32)
    w = tiny_workload(n, 1, U0=U0, c_red=c, chemistry=0)
    leak = {}
    for name, fl in (("glf", O.FLUX_GLF), ("hll", O.FLUX_HLL)):
        o = O.Oracle(w, flux=fl)
        rc, _ = o.step(w.dt, 10)
        assert rc == O.OK
        N = o.read(O.F_N).reshape(n, n, n)
        inside = N[6:10, 6:10, :].sum()
        leak[name] = 1.0 - inside / N.sum()
        assert N.sum() == pytest.approx(16.0 * n, rel=1e-12, abs=0)
    assert leak["hll"] < 0.6 * leak["glf"], leak


def test_H7_hll_budget_with_open_and_reflective_faces(oracle_mod):
    """A15 with the HLL flux: photons_total changes by injected - outflow (chemistry off), transmissive + reflective."""
    n = 8
    rng = np.random.default_rng(11)
    U0 = np.zeros((1, n ** 3, 4))
    U0[0, :, 0] = 10 ** rng.uniform(-5, -3, n ** 3)
    d = rng.standard_normal((n ** 3, 3))
    d /= np.linalg.norm(d, axis=1)[:, None]
    U0[0, :, 1:] = (rng.uniform(0, 0.9, n ** 3) * C_RED * U0[0, :, 0])[:, None] * d
    w = tiny_workload(n, 1, U0=U0.astype(np.float32), chemistry=0, bc=(1, 1, 2, 2, 1, 2),
                      src_pos=[[0.5, 0.5, 0.5]], src_Q=[[1e48]])
    o = O.Oracle(w, flux=O.FLUX_HLL)
    prev = o.step(w.dt, 0)[1]["photons_total"] if False else float(U0[0, :, 0].astype(np.float32).astype(np.float64).sum() * w.dx ** 3)
    for _ in range(5):
        rc, dg = o.step(w.dt, 1)
        assert rc == O.OK
        resid = dg["photons_total"] - prev - dg["photons_injected"] + dg["photons_outflow"]
        assert abs(resid) <= 1e-12 * dg["photons_total"]
        assert dg["photons_outflow"] != 0.0
        prev = dg["photons_total"]
