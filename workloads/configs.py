"""The five BASELINE.json configurations as seeded synthetic workloads.

Everything here is an *input recipe*: arrays and plain numbers handed, byte-identical, to the fp64
oracle and to the CUDA library.  No update arithmetic of the method lives here.

Array conventions (the C-ABI's, include/emma_rt.h):
  coarse cell id  = ix + n*(iy + n*iz)        (x fastest)
  refined cell id = oct*8 + (ix + 2*iy + 4*iz) on its level
  U0[g]           = float32 [n^3, 4] = (N, Fx, Fy, Fz) in cgs (photons cm^-3, photons cm^-2 s^-1)
  n0/x/T[level]   = float32 [n^3] (level 0) or [8*n_octs[level]]
"""
from dataclasses import dataclass, field

import numpy as np

from .constants import CGS
from .fields import lognormal_density
from .groups import blackbody_groups

SEED_BASE = 150807888          # arXiv id 1508.07888; seed = SEED_BASE + config number

BC_PERIODIC, BC_TRANSMISSIVE, BC_REFLECTIVE, BC_INFLOW = 0, 1, 2, 3


@dataclass
class Workload:
    name: str
    n: int                      # coarse cells per side
    G: int                      # photon groups
    L: float                    # box length [cm]
    c_red: float                # reduced speed of light [cm/s]
    sigma_N: np.ndarray         # [G] cm^2  (Eq. 29)
    sigma_E: np.ndarray         # [G] cm^2  (Eq. 37)
    E_mean: np.ndarray          # [G] erg   (Eq. 38)
    frac: np.ndarray            # [G] photon-number fraction of the source spectrum per group (Eq. 28)
    bc: tuple = (0, 0, 0, 0, 0, 0)
    otsa: int = 1
    chemistry: int = 1
    thermal: int = 1
    e_tol: float = 0.1          # PAPER.md:312 "at most vary by 10%"
    max_halvings: int = 60
    # AMR (static): parent[l-1][oct] = cell id on level l-1, for l = 1..n_levels
    parent: list = field(default_factory=list)
    # fields
    U0: list = None             # list of G float32 [n^3,4] arrays, or None (zeros)
    n0: list = None             # per level float32
    x: list = None
    T: list = None
    # sources
    src_pos: np.ndarray = None  # [n_src,3] float64 in [0,1)
    src_Q: np.ndarray = None    # [n_src,G] float64 photons/s
    # prescribed ghost state of BC_INFLOW faces: {(face, group): (N, Fx, Fy, Fz) in cgs}  (reading A20)
    inflow: dict = None
    # stepping
    courant: float = 0.9
    n_steps: int = 1

    @property
    def n_levels(self):
        return len(self.parent)

    @property
    def dx(self):
        return self.L / self.n

    @property
    def dt(self):
        """dt = courant * dx / (3 c_red)   (reading A4)."""
        return self.courant * self.dx / (3.0 * self.c_red)

    @property
    def n_leaves(self):
        tot = self.n ** 3
        for p in self.parent:
            tot += 7 * len(p)   # each oct replaces one leaf by eight
        return tot


def _groups(G):
    if G == 1:
        return blackbody_groups(1.0e5, (13.6, 1000.0))
    if G == 3:
        return blackbody_groups(1.0e5, (13.6, 24.6, 54.4, 1000.0))
    raise ValueError("G must be 1 or 3 for the BASELINE configs")


def _densest(a, k):
    """Indices of the k largest entries, ties -> lower index first (stable)."""
    order = np.argsort(-a.astype(np.float64), kind="stable")
    return order[:k]


def _cell_centres(ids, n):
    ix = ids % n
    iy = (ids // n) % n
    iz = ids // (n * n)
    return (np.stack([ix, iy, iz], axis=1).astype(np.float64) + 0.5) / n


def refine_by_density(n0_parent_level, is_leaf_mask, nbar, rng, thresh=8.0):
    """Split every leaf cell of a level whose density exceeds thresh*nbar (SURVEY.md 8(d) cfg 4).

    Returns (parent_ids, n0_children) where parent_ids are the split cells in increasing id order
    (that is the oct order of the new level) and n0_children is float64 [8*n_octs]:
      child = parent * exp(0.5 g - 0.125), g ~ N(0,1) drawn in oct order, then the eight children
      rescaled to average exactly to the parent.
    """
    split = np.flatnonzero(is_leaf_mask & (n0_parent_level > thresh * nbar))
    g = rng.standard_normal((len(split), 8))
    ch = n0_parent_level[split, None].astype(np.float64) * np.exp(0.5 * g - 0.125)
    ch *= (n0_parent_level[split].astype(np.float64) / ch.mean(axis=1))[:, None]
    return split.astype(np.int64), ch.reshape(-1)


def make_config(k, n=None, n_steps=None, n_src=None, variant="b", seed=None):
    """Build BASELINE.json config k (1..5).  `n`, `n_steps`, `n_src` override the size for scaled-down
    parity cases (same recipe, same physical cell size).  `variant` applies to config 5 only:
    "a" = N,F = 0 (literal), "b" = seeded background radiation so transport does not move zeros."""
    rng = np.random.default_rng((SEED_BASE + k) if seed is None else seed)
    c_red = 0.1 * CGS.c
    if k == 1:
        n = n or 32
        gr = _groups(1)
        dx = 6.6 * CGS.kpc / 32
        w = Workload("cfg1-stromgren", n, 1, dx * n, c_red, gr["sigma_N"], gr["sigma_E"], gr["E_mean"], gr["frac"])
        ncell = n ** 3
        w.n0 = [np.full(ncell, 1e-3, np.float32)]
        w.x = [np.full(ncell, 1.2e-3, np.float32)]
        w.T = [np.full(ncell, 100.0, np.float32)]
        c = n // 2
        w.src_pos = (np.array([[c, c, c]], np.float64) + 0.5) / n
        w.src_Q = np.array([[5e48]], np.float64)
        w.n_steps = n_steps or 100
        return w
    if k == 2:
        n = n or 64
        gr = _groups(1)
        dx = 6.6 * CGS.kpc / 32
        w = Workload("cfg2-lognormal64", n, 1, dx * n, c_red, gr["sigma_N"], gr["sigma_E"], gr["E_mean"], gr["frac"])
        ncell = n ** 3
        w.n0 = [lognormal_density(n, 1e-3, 0.5, rng).reshape(-1).astype(np.float32)]
        w.x = [np.full(ncell, 1.2e-3, np.float32)]
        w.T = [np.full(ncell, 100.0, np.float32)]
        ns = n_src or 16
        w.src_pos = rng.random((ns, 3))
        w.src_Q = (10.0 ** rng.uniform(47.0, 49.0, ns))[:, None]
        w.n_steps = n_steps or 200
        return w
    if k == 3:
        n = n or 128
        gr = _groups(3)
        dx = 0.5 * CGS.kpc
        w = Workload("cfg3-3groups128", n, 3, dx * n, c_red, gr["sigma_N"], gr["sigma_E"], gr["E_mean"], gr["frac"])
        ncell = n ** 3
        w.n0 = [lognormal_density(n, 1e-3, 1.0, rng).reshape(-1).astype(np.float32)]
        w.x = [np.full(ncell, 1.2e-3, np.float32)]
        w.T = [np.full(ncell, 100.0, np.float32)]
        ns = n_src or max(1, min(256, ncell // 8192))
        ids = _densest(w.n0[0], ns)
        w.src_pos = _cell_centres(ids, n)
        w.src_Q = (10.0 ** rng.uniform(47.0, 49.0, ns))[:, None] * gr["frac"][None, :]
        w.n_steps = n_steps or 100
        return w
    if k == 4:
        n = n or 256
        gr = _groups(3)
        dx = 4.0 * CGS.kpc
        w = Workload("cfg4-crta256", n, 3, dx * n, c_red, gr["sigma_N"], gr["sigma_E"], gr["E_mean"], gr["frac"])
        nbar = 1e-3
        n0c = lognormal_density(n, nbar, 1.5, rng).reshape(-1)
        # level 1: split coarse cells above 8 nbar; level 2: split level-1 cells above 8 nbar
        p1, n01 = refine_by_density(n0c, np.ones(n0c.shape, bool), nbar, rng)
        p2, n02 = refine_by_density(n01, np.ones(n01.shape, bool), nbar, rng)
        w.parent = [p1, p2]
        w.n0 = [n0c.astype(np.float32), n01.astype(np.float32), n02.astype(np.float32)]
        w.x = [np.full(a.shape, 1.2e-3, np.float32) for a in w.n0]
        w.T = [np.full(a.shape, 100.0, np.float32) for a in w.n0]
        # sources: the densest LEAF cells (they lie on level 2 when it exists)
        ns = n_src or max(1, min(1024, n ** 3 // 16384))
        lvl = 2 if len(p2) >= ns else (1 if len(p1) * 8 >= ns else 0)
        if lvl == 2:
            ids = _densest(w.n0[2], ns)
            pos = _leaf_centres_l2(ids, p1, p2, n)
        elif lvl == 1:
            leaf1 = np.ones(len(n01), bool)
            leaf1[p2] = False
            cand = np.flatnonzero(leaf1)
            ids = cand[_densest(w.n0[1][cand], ns)]
            pos = _leaf_centres_l1(ids, p1, n)
        else:
            ids = _densest(w.n0[0], ns)
            pos = _cell_centres(ids, n)
        w.src_pos = pos
        w.src_Q = (10.0 ** rng.uniform(47.0, 49.0, ns))[:, None] * gr["frac"][None, :]
        w.n_steps = n_steps or 100
        return w
    if k == 5:
        n = n or 512
        gr = _groups(3)
        dx = 4.0 * CGS.kpc
        w = Workload("cfg5%s-sweep%d" % (variant, n), n, 3, dx * n, c_red, gr["sigma_N"], gr["sigma_E"],
                     gr["E_mean"], gr["frac"])
        ncell = n ** 3
        w.n0 = [lognormal_density(n, 1e-3, 1.0, rng).reshape(-1).astype(np.float32)]
        x = 10.0 ** rng.uniform(-4.0, 0.0, ncell)
        np.minimum(x, 0.999999, out=x)
        w.x = [x.astype(np.float32)]
        del x
        w.T = [(10.0 ** rng.uniform(2.0, np.log10(3e4), ncell)).astype(np.float32)]
        ns = n_src or max(1, min(4096, ncell // 32768))
        ids = _densest(w.n0[0], ns)
        w.src_pos = _cell_centres(ids, n)
        w.src_Q = (10.0 ** rng.uniform(47.0, 49.0, ns))[:, None] * gr["frac"][None, :]
        if variant == "b":
            # photo-ionisation rate Gamma = c sum_g sigma_g N_g, log-uniform in [1e-16, 1e-11] s^-1,
            # shared out over the groups with the source spectrum's photon fractions
            gam = 10.0 ** rng.uniform(-16.0, -11.0, ncell)
            ntot = gam / (c_red * float(np.dot(gr["frac"], gr["sigma_N"])))
            del gam
            w.U0 = []
            for g in range(3):
                U = np.empty((ncell, 4), np.float32)
                Ng = ntot * gr["frac"][g]
                f = rng.uniform(0.0, 0.9, ncell)
                mu = rng.uniform(-1.0, 1.0, ncell)
                ph = rng.uniform(0.0, 2.0 * np.pi, ncell)
                st = np.sqrt(1.0 - mu * mu)
                Fm = f * c_red * Ng
                U[:, 0] = Ng
                U[:, 1] = Fm * st * np.cos(ph)
                U[:, 2] = Fm * st * np.sin(ph)
                U[:, 3] = Fm * mu
                w.U0.append(U)
                del Ng, f, mu, ph, st, Fm
        w.n_steps = n_steps or 50
        return w
    raise ValueError("config number must be 1..5")


def _leaf_centres_l1(ids, p1, n):
    """Box-unit centres of level-1 cells `ids` (oct*8+child) given level-1 parents p1 (coarse ids)."""
    oct1 = ids // 8
    ch = ids % 8
    base = _cell_centres(p1[oct1], n) - 0.5 / n            # low corner of the coarse cell
    off = np.stack([ch & 1, (ch >> 1) & 1, (ch >> 2) & 1], axis=1).astype(np.float64)
    return base + (off + 0.5) * (0.5 / n)


def _leaf_centres_l2(ids, p1, p2, n):
    """Box-unit centres of level-2 cells `ids` given parents p2 (level-1 cell ids) and p1."""
    oct2 = ids // 8
    ch = ids % 8
    c1 = p2[oct2]                                          # level-1 cell ids
    base = _leaf_centres_l1(c1, p1, n) - 0.25 / n          # low corner of the level-1 cell
    off = np.stack([ch & 1, (ch >> 1) & 1, (ch >> 2) & 1], axis=1).astype(np.float64)
    return base + (off + 0.5) * (0.25 / n)


def make_hii_region_corner(n=64, n_steps=200):
    """the static-gas cousin of the paper's HII-region test (section 6.4, after
    Iliev et al. "Test 2"/"Test 5"): 15 kpc box, uniform hydrogen n = 1e-3 cm^-3 at 100 K and x = 1.2e-3, ONE source of
    5e48 photons/s with a 1e5 K black-body spectrum in 3 groups placed in the corner cell at the origin, reflective
    boundaries on the three faces that touch the source and transmissive ones elsewhere, c~ = c/10.
    The gas does not move here (hydrodynamics is out of scope), so this is the paper's "Test 2"-like static run."""
    gr = _groups(3)
    L = 15.0 * CGS.kpc
    w = Workload("hii-corner-static", n, 3, L, 0.1 * CGS.c, gr["sigma_N"], gr["sigma_E"], gr["E_mean"], gr["frac"],
                 bc=(BC_REFLECTIVE, BC_TRANSMISSIVE, BC_REFLECTIVE, BC_TRANSMISSIVE, BC_REFLECTIVE, BC_TRANSMISSIVE))
    ncell = n ** 3
    w.n0 = [np.full(ncell, 1e-3, np.float32)]
    w.x = [np.full(ncell, 1.2e-3, np.float32)]
    w.T = [np.full(ncell, 100.0, np.float32)]
    w.src_pos = np.array([[0.5 / n, 0.5 / n, 0.5 / n]], np.float64)
    w.src_Q = 5e48 * np.asarray(gr["frac"], np.float64)[None, :]
    w.n_steps = n_steps
    return w


def make_shadow_clump(n=32, n_steps=200):
    """the static-gas cousin of the paper's clump photo-evaporation test (section
    6.5, after Iliev et al. 2009): 6.6 kpc box, a dense clump (0.04 cm^-3, 100 K) of radius 0.8 kpc centred on
    (5.4, 3.3, 3.3) kpc in a thin medium (2e-4 cm^-3, 8000 K), a plane-parallel 1e5 K black-body flux of 1e6 photons
    cm^-2 s^-1 (1e10 m^-2 s^-1) entering through the x = 0 face (BC_INFLOW), the opposite face transmissive, the other
    directions periodic.  3 groups, c~ = c/10.  The gas does not move here (hydrodynamics is out of scope)."""
    gr = _groups(3)
    L = 6.6 * CGS.kpc
    c_red = 0.1 * CGS.c
    w = Workload("shadow-clump-static", n, 3, L, c_red, gr["sigma_N"], gr["sigma_E"], gr["E_mean"], gr["frac"],
                 bc=(BC_INFLOW, BC_TRANSMISSIVE, BC_PERIODIC, BC_PERIODIC, BC_PERIODIC, BC_PERIODIC))
    ctr = (np.arange(n) + 0.5) * (6.6 / n)                               # cell centres [kpc]
    X, Y, Z = np.meshgrid(ctr, ctr, ctr, indexing="ij")                  # arrays indexed [ix, iy, iz]
    inside = ((X - 5.4) ** 2 + (Y - 3.3) ** 2 + (Z - 3.3) ** 2) <= 0.8 ** 2
    to_id = lambda a: np.ascontiguousarray(a.transpose(2, 1, 0)).reshape(-1)   # cell id = ix + n (iy + n iz)
    w.n0 = [to_id(np.where(inside, 0.04, 2e-4)).astype(np.float32)]
    w.T = [to_id(np.where(inside, 100.0, 8000.0)).astype(np.float32)]
    w.x = [np.full(n ** 3, 1.2e-3, np.float32)]
    F = 1.0e6
    w.inflow = {(0, g): (F * gr["frac"][g] / c_red, F * gr["frac"][g], 0.0, 0.0) for g in range(3)}
    w.n_steps = n_steps
    return w
