"""Pins of the oracle's standard (non-CRTA) AMR transport, reading A21.  CPU only.

M1  a fully refined level is the uniform fine grid advanced by two (four) half (quarter) steps -- bitwise
M2  photons are conserved across resolution jumps (periodic), and the budget closes with open faces
M3  a uniform field with zero flux is invariant on any mesh
M4  brute force: an independent dict-based transcription (tests/brute_amr.py) on tiny meshes
M5  Fig. 6 call counts of the standard scheme: 4 coarse steps with 2 refined levels = 4 + 24 engine calls
M6  a resolution jump of 2 across a face is refused
M7  a beam crossing a refined slab keeps its photons and its speed
M9  the ghost of a linear field is the field at the centre of the virtual fine cell, all 8 positions
M8  PAPER.md:556: the CRTA front follows the standard scheme's (static HII region with a refined shell)
"""
import numpy as np
import pytest

import oracle
from workloads import CGS
from workloads.amr import make_amr_standard

from .brute_amr import Mesh
from .helpers import tiny_workload


def coords_of(n, parents):
    """integer cell coordinates [ncell_l, 3] per level (child index = ix + 2 iy + 4 iz)."""
    ids = np.arange(n ** 3)
    out = [np.stack([ids % n, (ids // n) % n, ids // (n * n)], axis=1)]
    for p in parents:
        pc = out[-1][np.asarray(p, np.int64)]
        k = np.arange(8)
        off = np.stack([k & 1, (k >> 1) & 1, (k >> 2) & 1], axis=1)
        out.append((2 * pc[:, None, :] + off[None, :, :]).reshape(-1, 3))
    return out


def full_refinement(n, levels):
    parents, m = [], n ** 3
    for _ in range(levels):
        parents.append(np.arange(m, dtype=np.int64))
        m *= 8
    return parents


def random_state(rng, m, c, fmax=0.8):
    U = np.empty((m, 4))
    U[:, 0] = 10.0 ** rng.uniform(-6, -3, m)
    v = rng.standard_normal((m, 3))
    v /= np.linalg.norm(v, axis=1)[:, None]
    U[:, 1:] = v * (rng.uniform(0, fmax, m) * c * U[:, 0])[:, None]
    return U.astype(np.float32).astype(np.float64)


def fine_to_uniform(co, nf):
    """position of each fine cell in the x-fastest uniform grid of nf cells per side."""
    return co[:, 0] + nf * (co[:, 1] + nf * co[:, 2])


@pytest.mark.parametrize("levels,flux", [(1, oracle.FLUX_GLF), (2, oracle.FLUX_GLF), (1, oracle.FLUX_HLL)])
def test_M1_full_refinement_is_the_uniform_fine_grid(levels, flux):
    n, G = 4, 2
    nf = n << levels
    rng = np.random.default_rng(11 + levels)
    parents = full_refinement(n, levels)
    co = coords_of(n, parents)
    pos = fine_to_uniform(co[levels], nf)
    n0f = (1e-3 * np.exp(rng.standard_normal(nf ** 3))).astype(np.float32)          # uniform-grid order
    xf = rng.uniform(0.01, 0.9, nf ** 3).astype(np.float32)
    Tf = (10.0 ** rng.uniform(2, 4.3, nf ** 3)).astype(np.float32)
    src = np.array([[0.3, 0.6, 0.1], [0.77, 0.2, 0.52]])
    Q = np.array([[3e46, 1e46], [1e45, 5e46]])
    lv = lambda a: [np.zeros(8 * len(p), np.float32) for p in parents[:-1]] + [a[pos]]
    wa = tiny_workload(n, G=2, parent=parents, n0_lv=lv(n0f), x_lv=lv(xf), T_lv=lv(Tf), src_pos=src, src_Q=Q)
    wu = tiny_workload(nf, G=2, L=wa.L, n0=n0f, x=xf, T=Tf, src_pos=src, src_Q=Q)
    oa, ou = oracle.Oracle(wa, flux=flux), oracle.Oracle(wu, flux=flux)
    assert oa.set_amr_transport(True) == oracle.OK
    Uf = [random_state(rng, nf ** 3, wa.c_red) for _ in range(G)]
    for g in range(G):
        assert oa.write_U(levels, g, Uf[g][pos]) == oracle.OK
        wu.U0 = None
    assert oa.restrict_U() == oracle.OK
    ou.close()
    wu.U0 = [u.astype(np.float32) for u in Uf]
    ou = oracle.Oracle(wu, flux=flux)
    rc, da = oa.step(wa.dt, 2)
    assert rc == oracle.OK
    rc, du = ou.step(wa.dt / 2 ** levels, 2 << levels)
    assert rc == oracle.OK
    for g in range(G):
        assert np.array_equal(oa.read(oracle.F_U, levels, g), ou.read(oracle.F_U, 0, g)[pos])
    assert np.array_equal(oa.read(oracle.F_X, levels), ou.read(oracle.F_X)[pos])
    assert np.array_equal(oa.read(oracle.F_E, levels), ou.read(oracle.F_E)[pos])
    # the coarse cells hold the mean of their descendants
    Nf = ou.read(oracle.F_N, 0, 0).reshape(nf, nf, nf)
    k = 1 << levels
    Nc = Nf.reshape(n, k, n, k, n, k).mean(axis=(1, 3, 5)).reshape(-1)
    np.testing.assert_allclose(oa.read(oracle.F_N, 0, 0), Nc, rtol=1e-13)
    assert abs(da["photons_total"] - du["photons_total"]) <= 1e-13 * du["photons_total"]


def _partial_mesh(n, rng, levels=2):
    w = make_amr_standard(n=n, G=1, levels=levels, seed=int(rng.integers(1 << 30)), thresh1=2.0, thresh2=2.5)
    assert 0 < len(w.parent[0]) < n ** 3
    return w


def _fill_random(o, w, rng):
    co = coords_of(w.n, w.parent)
    for l in range(w.n_levels + 1):
        for g in range(w.G):
            assert o.write_U(l, g, random_state(rng, len(co[l]), w.c_red)) == oracle.OK
    assert o.restrict_U() == oracle.OK


def _leaf_photons(o, w):
    tot = 0.0
    for l in range(w.n_levels + 1):
        leaf = np.ones(o.level_cells(l), bool)
        if l < w.n_levels:
            leaf[w.parent[l]] = False
        for g in range(w.G):
            tot += o.read(oracle.F_N, l, g)[leaf].sum() * (w.dx / 2 ** l) ** 3
    return tot


@pytest.mark.parametrize("flux", [oracle.FLUX_GLF, oracle.FLUX_HLL])
def test_M2_photons_conserved_across_jumps(flux):
    rng = np.random.default_rng(5)
    w = _partial_mesh(8, rng)
    assert len(w.parent[1]) > 0
    w.src_pos = None
    o = oracle.Oracle(w, chemistry=0, flux=flux)
    assert o.set_amr_transport(True) == oracle.OK
    _fill_random(o, w, rng)
    before = _leaf_photons(o, w)
    for _ in range(3):
        rc, d = o.step(w.dt, 1)
        assert rc == oracle.OK
        after = _leaf_photons(o, w)
        assert abs(after - before) <= 2e-14 * before
        assert abs(d["photons_total"] - after) <= 1e-14 * after
        before = after


def test_M2b_budget_closes_with_open_faces_sources_and_chemistry():
    rng = np.random.default_rng(6)
    w = _partial_mesh(8, rng)
    w.bc = (1, 1, 2, 1, 1, 2)
    o = oracle.Oracle(w)
    assert o.set_amr_transport(True) == oracle.OK
    _fill_random(o, w, rng)
    before = _leaf_photons(o, w)
    for _ in range(3):
        rc, d = o.step(w.dt, 1)
        assert rc == oracle.OK
        rhs = d["photons_injected"] - d["photons_absorbed"] + d["photons_recomb_emitted"] - d["photons_outflow"]
        scale = max(before, d["photons_injected"], d["photons_absorbed"])
        assert abs((d["photons_total"] - before) - rhs) <= 1e-13 * scale
        assert d["photons_outflow"] != 0.0
        before = d["photons_total"]


def test_M3_uniform_field_is_invariant():
    rng = np.random.default_rng(7)
    w = _partial_mesh(8, rng)
    w.src_pos = None
    o = oracle.Oracle(w, chemistry=0)
    assert o.set_amr_transport(True) == oracle.OK
    for l in range(w.n_levels + 1):
        U = np.zeros((o.level_cells(l), 4))
        U[:, 0] = 3.25e-5
        o.write_U(l, 0, U)
    rc, _ = o.step(w.dt, 3)
    assert rc == oracle.OK
    for l in range(w.n_levels + 1):
        U = o.read(oracle.F_U, l, 0)
        np.testing.assert_allclose(U[:, 0], 3.25e-5, rtol=1e-14)
        assert np.abs(U[:, 1:]).max() <= 1e-14 * w.c_red * 3.25e-5


@pytest.mark.parametrize("case", ["one_oct", "two_levels"])
def test_M4_brute_force(case):
    rng = np.random.default_rng(8)
    n = 4
    if case == "one_oct":
        parents = [np.array([21], np.int64)]
    else:
        # level 1: a 3x3x3 block of coarse cells around (1,1,1) (wraps nowhere); level 2: the centre cell's 8 children
        blk = sorted(i + n * (j + n * k) for i in (0, 1, 2) for j in (0, 1, 2) for k in (0, 1, 2))
        parents = [np.array(blk, np.int64)]
        centre = blk.index(1 + n * (1 + n * 1))
        parents.append(np.array([8 * centre + k for k in (0, 3, 5, 6)], np.int64))
    src = np.array([[0.3, 0.3, 0.3]])
    w = tiny_workload(n, G=1, parent=parents, chemistry=0, src_pos=src, src_Q=np.array([[2e44]]))
    o = oracle.Oracle(w, chemistry=0)
    assert o.set_amr_transport(True) == oracle.OK
    co = coords_of(n, parents)
    U = [random_state(rng, len(c), w.c_red) for c in co]
    for l in range(len(co)):
        o.write_U(l, 0, U[l])
    o.restrict_U()
    cells, split = {}, set()
    for l in range(len(co)):
        Ul = o.read(oracle.F_U, l, 0)
        for i, c in enumerate(co[l]):
            cells[(l,) + tuple(int(v) for v in c)] = Ul[i].copy()
        if l < len(parents):
            for p in parents[l]:
                split.add((l,) + tuple(int(v) for v in co[l][p]))
    sl, sc = o.source_cell(0)
    skey = (sl,) + tuple(int(v) for v in co[sl][sc])
    assert skey not in split
    S = {skey: 2e44 / (w.dx / 2 ** sl) ** 3}
    mesh = Mesh(n, cells, split, w.c_red, w.dx, S)
    for step in range(2):
        rc, d = o.step(w.dt, 1)
        assert rc == oracle.OK
        mesh.advance(0, w.dt)
        for l in range(len(co)):
            Ul = o.read(oracle.F_U, l, 0)
            ref = np.array([mesh.cells[(l,) + tuple(int(v) for v in c)] for c in co[l]])
            scaleN = np.abs(ref[:, 0]).max()
            assert np.abs(Ul[:, 0] - ref[:, 0]).max() <= 1e-12 * scaleN, (case, step, l)
            assert np.abs(Ul[:, 1:] - ref[:, 1:]).max() <= 1e-12 * w.c_red * scaleN, (case, step, l)
        assert abs(d["photons_total"] - mesh.photons()) <= 1e-12 * d["photons_total"]


def test_M5_fig6_call_counts_of_the_standard_scheme():
    w = make_amr_standard(n=8, G=1, levels=2, thresh1=2.0, thresh2=2.5)
    assert len(w.parent) == 2 and len(w.parent[1]) > 0
    o = oracle.Oracle(w)
    assert o.set_amr_transport(True) == oracle.OK
    rc, _ = o.step(w.dt, 4)                     # "a dynamical time step equal to 4 times the coarse radiative one"
    assert rc == oracle.OK
    tr, ch = o.counters()
    calls_tr = [tr[l] // o.level_cells(l) for l in range(3)]
    from .test_oracle_pins import GOLD                           # tests/golden/paper_values.txt, each value with its citation
    assert calls_tr[0] == int(GOLD["fig6_standard_coarse_calls"])                       # 4 on the coarse level,
    assert calls_tr[1] + calls_tr[2] == int(GOLD["fig6_standard_refined_calls"])        # 24 on the refined ones,
    assert calls_tr == [4, 8, 16] and sum(calls_tr) == int(GOLD["fig6_standard_transport_calls"])   # 28 in all
    leaves = [o.level_cells(0) - len(w.parent[0]), o.level_cells(1) - len(w.parent[1]), o.level_cells(2)]
    assert [ch[l] // leaves[l] for l in range(3)] == [4, 8, 16]


def test_M6_jump_of_two_is_refused():
    n = 4
    parents = [np.array([21], np.int64), np.array([0], np.int64)]     # a level-2 oct in the corner child of a lone oct
    w = tiny_workload(n, G=1, parent=parents)
    o = oracle.Oracle(w)
    assert o.set_amr_transport(True) == oracle.EINVAL


def test_M7_beam_through_a_refined_slab():
    """free-streaming beam along x, uniform in y and z; coarse cells with 4 <= ix < 8 are split.  Photons are conserved
    and the centroid advances by nu coarse cells per step (speed c~), as on the uniform grid (pin P3)."""
    n = 16
    ids = np.arange(n ** 3)
    parents = [ids[(ids % n >= 4) & (ids % n < 8)].astype(np.int64)]
    w = tiny_workload(n, G=1, parent=parents, chemistry=0)
    o = oracle.Oracle(w, chemistry=0)
    assert o.set_amr_transport(True) == oracle.OK
    co = coords_of(n, parents)
    prof = lambda xc: np.exp(-0.5 * ((xc - 3.0) / 1.0) ** 2)          # x in coarse-cell units
    for l in range(2):
        xc = (co[l][:, 0] + 0.5) / 2 ** l
        U = np.zeros((len(xc), 4))
        U[:, 0] = prof(xc)
        U[:, 1] = w.c_red * U[:, 0]
        o.write_U(l, 0, U)
    o.restrict_U()

    def moments():
        m0 = m1 = 0.0
        for l in range(2):
            leaf = np.ones(o.level_cells(l), bool)
            if l == 0:
                leaf[parents[0]] = False
            N = o.read(oracle.F_N, l, 0)[leaf]
            xc = (co[l][leaf, 0] + 0.5) / 2 ** l
            m0 += (N / 8 ** l).sum()
            m1 += (N * xc / 8 ** l).sum()
        return m0, m1 / m0

    m0, x0 = moments()
    steps = 12
    rc, _ = o.step(w.dt, steps)
    assert rc == oracle.OK
    m0b, x1 = moments()
    assert abs(m0b - m0) <= 1e-13 * m0                               # periodic: conserved
    nu = w.c_red * w.dt / w.dx
    assert abs((x1 - x0) - nu * steps) <= 0.02 * nu * steps
    # the beam stays a beam: F = c N on the leaves
    for l in range(2):
        U = o.read(oracle.F_U, l, 0)
        big = U[:, 0] > 1e-6
        np.testing.assert_allclose(U[big, 1], w.c_red * U[big, 0], rtol=1e-9)


def test_M8_crta_front_follows_the_standard_scheme():
    """PAPER.md:556 (Fig. 11-12): "the front position and velocities of the CRTA calculation follow the ones obtained from
    the standard procedure".  Static cousin of that HII-region test (workloads.make_hii_region_corner: corner source,
    reflective + transmissive faces, 3 groups) on a 16^3 base with the shell 1.5 <= r < 7 coarse cells refined once, so that
    the front travels inside refined cells: the equivalent front radius (ionised volume of the leaves) of the oracle's CRTA
    mode and of its standard AMR mode agree within 1 % at six epochs, and the standard front, transported on the fine
    cells, is the sharper one."""
    from workloads import make_hii_region_corner
    n = 16
    w = make_hii_region_corner(n=n)
    ids = np.arange(n ** 3)
    r = np.sqrt((ids % n + 0.5) ** 2 + ((ids // n) % n + 0.5) ** 2 + (ids // (n * n) + 0.5) ** 2)
    p1 = ids[(r >= 1.5) & (r < 7.0)].astype(np.int64)
    w.parent = [p1]
    m = 8 * len(p1)
    w.n0.append(np.full(m, 1e-3, np.float32))
    w.x.append(np.full(m, 1.2e-3, np.float32))
    w.T.append(np.full(m, 100.0, np.float32))

    def run(standard):
        o = oracle.Oracle(w)
        if standard:
            assert o.set_amr_transport(True) == oracle.OK
        radii = []
        for _ in range(6):
            rc, _d = o.step(w.dt, 100)
            assert rc == oracle.OK
            vol = 0.0
            for l in (0, 1):
                x = o.read(oracle.F_X, l)
                leaf = np.ones(len(x), bool)
                if l == 0:
                    leaf[p1] = False
                vol += ((x[leaf] - 1.2e-3) / (1 - 1.2e-3)).sum() * (w.dx / 2 ** l) ** 3
            radii.append((6.0 * vol / np.pi) ** (1.0 / 3.0) / w.dx)
        return np.array(radii), o.read(oracle.F_X, 0).reshape(n, n, n)[0, 0, :]

    r_crta, x_crta = run(False)
    r_std, x_std = run(True)
    assert 3.5 < r_std[-1] < 5.0                                  # the front is inside the refined shell
    np.testing.assert_allclose(r_crta, r_std, rtol=1e-2)
    assert np.all(np.diff(r_std) > 0)
    ahead = slice(4, 8)                                           # just ahead of the x = 0.5 point
    assert np.all(x_std[ahead] < x_crta[ahead])


def test_M9_ghost_of_a_linear_field_is_exact():
    """the missing fine neighbour "is interpolated linearly from coarse data at the position of the fine virtual
    cell".  For a field that is linear in x, y, z (all four components, different gradients) the MinMod slopes are the
    gradient, so the ghost must equal the field at the centre of the virtual cell -- for each of the 8 positions inside the
    coarse leaf, on level 0 and on level 1.  Pins the +-1/4 offsets and the axis <-> child-bit mapping independently of any
    transcription of the scheme."""
    n = 8
    # level 1: the block [2,6)^3; level 2: level-1 cells [6,10)^3 (inside, with a level-1 buffer around)
    ids = np.arange(n ** 3)
    cx, cy, cz = ids % n, (ids // n) % n, ids // (n * n)
    p1 = ids[(cx >= 2) & (cx < 6) & (cy >= 2) & (cy < 6) & (cz >= 2) & (cz < 6)].astype(np.int64)
    co1 = coords_of(n, [p1])[1]
    sel = np.all((co1 >= 6) & (co1 < 10), axis=1)
    p2 = np.flatnonzero(sel).astype(np.int64)
    w = tiny_workload(n, G=1, parent=[p1, p2], chemistry=0, bc=(1,) * 6)
    o = oracle.Oracle(w, chemistry=0)
    assert o.set_amr_transport(True) == oracle.OK
    co = coords_of(n, [p1, p2])
    grad = np.array([[1.0, 0.3, -0.2, 0.5], [0.7, -0.4, 0.6, 0.1], [-0.5, 0.2, 0.3, -0.6]])     # d/dx, d/dy, d/dz of (N, Fx, Fy, Fz)
    base = np.array([50.0, 1.0, -2.0, 3.0])
    field = lambda pos: base[None, :] + pos @ grad                     # pos in units of the coarse cell size
    for l in range(3):
        o.write_U(l, 0, field((co[l] + 0.5) / 2 ** l))
    # level-0 leaf (1,3,3) next to the block: virtual level-1 cells inside it
    c0 = 1 + n * (3 + n * 3)
    for k in range(8):
        v = np.array([2 * 1 + (k & 1), 2 * 3 + ((k >> 1) & 1), 2 * 3 + ((k >> 2) & 1)])
        np.testing.assert_allclose(o.amr_ghost(1, 0, v, c0), field(((v + 0.5) / 2)[None, :])[0], rtol=1e-13)
    # level-1 leaf next to the level-2 block: the level-1 cell at (5,7,7) (exists, unsplit); virtual level-2 cells inside it
    c1 = int(np.flatnonzero(np.all(co[1] == np.array([5, 7, 7]), axis=1))[0])
    assert c1 not in set(p2.tolist())
    for k in range(8):
        v = np.array([2 * 5 + (k & 1), 2 * 7 + ((k >> 1) & 1), 2 * 7 + ((k >> 2) & 1)])
        np.testing.assert_allclose(o.amr_ghost(2, 0, v, c1), field(((v + 0.5) / 4)[None, :])[0], rtol=1e-13)
    # an extremum is not extrapolated: MinMod gives a zero slope there
    U = field((co[0] + 0.5))
    U[c0] = 1e3
    o.write_U(0, 0, U)
    g = o.amr_ghost(1, 0, np.array([2, 6, 6]), c0)
    np.testing.assert_allclose(g, U[c0], rtol=0, atol=0)
