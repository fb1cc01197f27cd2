"""Pin M4: an independent Python transcription of the standard AMR transport (reading A21) on tiny meshes.

Written from the statement of reading A21 (Fig. 3 sequence (i)-(iii); PAPER.md:436 linear ghosts), not
from oracle/emma_rt_oracle.c: cells live in a dict keyed by (level, i, j, k), neighbours are found by coordinates, the
GLF flux (Eq. 32) is formed from tests/brute.py's closure.  Periodic boxes, chemistry off (sources: N += S dt).
"""
import numpy as np

from .brute import pressure


def glf(UL, UR, c, d):
    """Eq. 32 for the face between UL (left) and UR (right) along direction d.  U: [4]."""
    def ft(U):
        P = pressure(U[None, :], c)[0]
        return np.array([U[1 + d], c * c * P[d, 0], c * c * P[d, 1], c * c * P[d, 2]])
    return 0.5 * (ft(UL) + ft(UR)) - 0.5 * c * (UR - UL)


def minmod(a, b):
    return np.where(a * b <= 0.0, 0.0, np.where(np.abs(a) < np.abs(b), a, b))


class Mesh:
    """cells: {(l,i,j,k): U[4]} for every cell (split ones too); split: set of keys; n: coarse cells per side."""

    def __init__(self, n, cells, split, c, dx0, S=None):
        self.n, self.cells, self.split, self.c, self.dx0 = n, cells, split, c, dx0
        self.S = S or {}
        self.dep = {k: np.zeros(4) for k in cells}
        self.lmax = max(k[0] for k in cells)

    def covering(self, l, ijk):
        """the existing cell of the highest level <= l that covers level-l coordinates ijk (periodic)."""
        m = self.n << l
        ijk = tuple(v % m for v in ijk)
        for lv in range(l, -1, -1):
            key = (lv,) + tuple(v >> (l - lv) for v in ijk)
            if key in self.cells:
                return key
        raise KeyError(ijk)

    def level_value(self, l, ijk):
        """value seen on level l at ijk: the level-l cell if it exists, else the coarser leaf, piecewise constant."""
        return self.cells[self.covering(l, ijk)]

    def ghost(self, l, ijk):
        """linear (MinMod-limited) interpolation of the level-(l-1) leaf at the virtual level-l cell ijk."""
        m = self.n << l
        ijk = tuple(v % m for v in ijk)
        ck = tuple(v >> 1 for v in ijk)
        Uc = self.cells[(l - 1,) + ck]
        out = Uc.copy()
        for a in range(3):
            lo = list(ck); lo[a] -= 1
            hi = list(ck); hi[a] += 1
            slope = minmod(Uc - self.level_value(l - 1, lo), self.level_value(l - 1, hi) - Uc)
            out = out + (0.25 if ijk[a] & 1 else -0.25) * slope
        return out

    def transport(self, l, dt):
        dx = self.dx0 / 2 ** l
        new = {}
        for key, U0 in self.cells.items():
            if key[0] != l or key in self.split:
                continue
            out = U0.copy()
            for d in range(3):
                for s in (-1, +1):
                    q = list(key[1:]); q[d] += s
                    cov = self.covering(l, q)
                    if cov[0] == l and cov in self.split:
                        continue                                   # (iii): that face was fed by the fine steps
                    Unb = self.cells[cov] if cov[0] == l else self.ghost(l, q)
                    Fh = glf(Unb, U0, self.c, d) if s < 0 else glf(U0, Unb, self.c, d)
                    out = out - s * dt / dx * Fh
                    if cov[0] < l:                                  # (i)-(ii): same flux, seen from the coarse cell
                        self.dep[cov] = self.dep[cov] + s * Fh * dt * dx * dx / (2 * dx) ** 3
            new[key] = out + self.dep[key]
            self.dep[key] = np.zeros(4)
        self.cells.update(new)

    def sources(self, l, dt):
        for key, S in self.S.items():
            if key[0] == l:
                self.cells[key] = self.cells[key] + np.array([S * dt, 0, 0, 0])

    def restrict(self, l):
        for key in self.split:
            if key[0] == l:
                _, i, j, k = key
                self.cells[key] = sum(self.cells[(l + 1, 2 * i + a, 2 * j + b, 2 * k + c)]
                                      for a in (0, 1) for b in (0, 1) for c in (0, 1)) / 8.0

    def advance(self, l, dt):
        if l < self.lmax:
            self.advance(l + 1, dt / 2)
            self.advance(l + 1, dt / 2)
        self.transport(l, dt)
        self.sources(l, dt)
        self.restrict(l)

    def photons(self):
        return sum(U[0] * (self.dx0 / 2 ** k[0]) ** 3 for k, U in self.cells.items() if k not in self.split)
