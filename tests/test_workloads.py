"""Input recipes (workloads/): group constants, random fields, the five configs at reduced size.  CPU only."""
import numpy as np
import pytest

from workloads import CGS, blackbody_groups, gaussian_random_field, lognormal_density, make_config, sigma_HI


def test_group_constants_blackbody_1e5K():
    """BASELINE.json config 1: '1 photon group at 29.6 eV effective energy' for a 1e5 K black body above 13.6 eV."""
    g1 = blackbody_groups(1e5, (13.6, 1000.0))
    assert g1["E_mean_eV"][0] == pytest.approx(29.6, abs=0.05)
    assert g1["frac"][0] == pytest.approx(1.0)
    assert sigma_HI(13.6) == pytest.approx(6.3e-18, rel=0.02)              # threshold cross-section (textbook)
    assert sigma_HI(13.0) == 0.0
    assert sigma_HI(54.4) / sigma_HI(13.6) == pytest.approx((13.6 / 54.4) ** 3, rel=0.25)   # ~nu^-3 fall-off
    g3 = blackbody_groups(1e5, (13.6, 24.6, 54.4, 1000.0))
    assert g3["frac"].sum() == pytest.approx(1.0, rel=1e-12)
    # the 1-group averages are the photon-weighted means of the 3-group ones (Eq. 29, 37, 38 are linear in N_nu)
    assert (g3["frac"] * g3["sigma_N"]).sum() == pytest.approx(g1["sigma_N"][0], rel=1e-6)
    assert (g3["frac"] * g3["E_mean_eV"]).sum() == pytest.approx(g1["E_mean_eV"][0], rel=1e-6)
    assert (g3["frac"] * g3["E_mean_eV"] * g3["sigma_E"]).sum() == pytest.approx(
        g1["sigma_E"][0] * g1["E_mean_eV"][0], rel=1e-6)
    assert np.all(np.diff(g3["sigma_N"]) < 0) and np.all(np.diff(g3["E_mean_eV"]) > 0)
    assert 13.6 < g3["E_mean_eV"][0] < 24.6 < g3["E_mean_eV"][1] < 54.4 < g3["E_mean_eV"][2]


def test_grf_spectrum_and_lognormal_mean():
    rng = np.random.default_rng(7)
    n = 32
    d = gaussian_random_field(n, rng)
    assert abs(d.mean()) < 1e-12 and d.std() == pytest.approx(1.0, rel=1e-12)
    pk = np.abs(np.fft.fftn(d)) ** 2
    kf = np.fft.fftfreq(n) * n
    k = np.sqrt(kf[:, None, None] ** 2 + kf[None, :, None] ** 2 + kf[None, None, :] ** 2)
    lo = pk[(k > 1.5) & (k < 3.5)].mean()
    hi = pk[(k > 6) & (k < 14)].mean()
    k_lo = k[(k > 1.5) & (k < 3.5)].mean()
    k_hi = k[(k > 6) & (k < 14)].mean()
    slope = np.log(hi / lo) / np.log(k_hi / k_lo)
    assert slope == pytest.approx(-2.0, abs=0.35)                          # P(k) ~ k^-2
    n0 = lognormal_density(16, 1e-3, 1.0, np.random.default_rng(8))
    assert n0.mean() == pytest.approx(1e-3, rel=1e-12) and n0.min() > 0


@pytest.mark.parametrize("k,n", [(1, 8), (2, 8), (3, 8), (4, 16), (5, 8)])
def test_configs_shapes_and_determinism(k, n):
    a = make_config(k, n=n)
    b = make_config(k, n=n)
    nc = n ** 3
    assert a.n0[0].shape == (nc,) and a.n0[0].dtype == np.float32
    for f in ("n0", "x", "T"):
        for la, lb in zip(getattr(a, f), getattr(b, f)):
            assert la.tobytes() == lb.tobytes()
    assert a.src_pos.tobytes() == b.src_pos.tobytes() and a.src_Q.tobytes() == b.src_Q.tobytes()
    assert a.src_Q.shape == (len(a.src_pos), a.G)
    assert np.all((a.src_pos >= 0) & (a.src_pos < 1))
    assert a.dt == pytest.approx(0.9 * a.dx / (3 * a.c_red))
    assert a.c_red == pytest.approx(0.1 * CGS.c)
    if k == 5:
        assert len(a.U0) == 3 and a.U0[0].shape == (nc, 4)
        Fn = np.linalg.norm(a.U0[1][:, 1:].astype(np.float64), axis=1)
        assert np.all(Fn <= 0.9001 * a.c_red * a.U0[1][:, 0].astype(np.float64))
        assert a.x[0].max() <= 0.999999 + 1e-7 and a.x[0].min() >= 1e-4 * 0.999
        assert make_config(5, n=n, variant="a").U0 is None
    if k == 4:
        p1, p2 = a.parent
        assert len(p1) > 0 and len(p2) > 0
        assert np.all(np.diff(p1) > 0) and np.all(np.diff(p2) > 0)
        assert np.all(a.n0[0][p1] > 8e-3)
        ch = a.n0[1].astype(np.float64).reshape(-1, 8).mean(axis=1)
        assert np.allclose(ch, a.n0[0][p1], rtol=1e-6)
        assert a.n_leaves == nc + 7 * (len(p1) + len(p2))
        # sources sit in the densest level-2 leaves
        assert a.n_levels == 2


def test_config4_full_size_refinement_fraction_estimate():
    """at sigma_ln = 1.5 about 1.6 % of coarse cells exceed 8 nbar (one-point lognormal PDF)."""
    from math import erfc, log, sqrt
    s = 1.5
    frac = 0.5 * erfc((log(8.0) + s * s / 2) / (s * sqrt(2)))
    assert frac == pytest.approx(0.0163, abs=0.002)


def test_amr_standard_mesh_recipe():
    """workloads.amr: seeded, jump-balanced (the oracle's AMR mode accepts it: PAPER.md:75), children densities average to
    the parent, and the Z-order option permutes the octs without changing which cells are split."""
    import oracle as O
    from workloads.amr import make_amr_standard
    for seed in (1, 2, 3):
        w = make_amr_standard(n=12, G=1, levels=2, seed=seed, thresh1=2.0, thresh2=2.5)
        w2 = make_amr_standard(n=12, G=1, levels=2, seed=seed, thresh1=2.0, thresh2=2.5)
        assert all(np.array_equal(a, b) for a, b in zip(w.parent, w2.parent))
        assert all(np.array_equal(a, b) for a, b in zip(w.n0, w2.n0))
        assert 0 < len(w.parent[0]) < 12 ** 3 and len(w.parent[1]) > 0
        assert len(set(w.parent[0].tolist())) == len(w.parent[0]) and len(set(w.parent[1].tolist())) == len(w.parent[1])
        o = O.Oracle(w)
        assert o.set_amr_transport(True) == O.OK
        o.close()
        for l in (1, 2):
            kids = w.n0[l].astype(np.float64).reshape(-1, 8).mean(axis=1)
            np.testing.assert_allclose(kids, w.n0[l - 1][w.parent[l - 1]].astype(np.float64), rtol=1e-6)
        wm = make_amr_standard(n=12, G=1, levels=2, seed=seed, thresh1=2.0, thresh2=2.5, order="morton")
        assert sorted(wm.parent[0].tolist()) == sorted(w.parent[0].tolist())
        assert len(wm.parent[1]) == len(w.parent[1])
        om = O.Oracle(wm)
        assert om.set_amr_transport(True) == O.OK
        om.close()
