"""Pin P13: an independent numpy/Python transcription of one coupled step on a tiny periodic grid.

Written from the equation table in DESIGN.md (readings A1-A9), not from oracle/emma_rt_oracle.c: the
transport is the *expanded* centred form of Eq. 30+32 (own-cell flux cancels), vectorised with np.roll;
the chemistry is a per-cell Python loop.  It exists only to catch sign / index / transposition slips in
the oracle; it is far too slow for anything but 4^3..8^3 grids.
"""
import numpy as np

K_B = 1.380649e-16
E_HI = 13.6 * 1.602176634e-12


def pressure(U, c):
    """U: [..., 4] -> P: [..., 3, 3]   (Eq. 22-23 with A1, A2)."""
    N = U[..., 0]
    F = U[..., 1:]
    Fn = np.sqrt((F ** 2).sum(-1))
    with np.errstate(divide="ignore", invalid="ignore"):
        f = np.where(N > 0, Fn / (c * N), 0.0)
        f = np.minimum(f, 1.0)
        nhat = np.where(Fn[..., None] > 0, F / Fn[..., None], 0.0)
    chi = (3 + 4 * f ** 2) / (5 + 2 * np.sqrt(4 - 3 * f ** 2))
    eye = np.eye(3)
    D = ((1 - chi) / 2)[..., None, None] * eye + ((3 * chi - 1) / 2)[..., None, None] * nhat[..., :, None] * nhat[..., None, :]
    return D * N[..., None, None]


def transport_periodic(U, c, dt, dx):
    """U: [nz, ny, nx, 4] fp64, periodic.  U' = U - dt/(2dx) sum_d [Ft_d(i+1) - Ft_d(i-1)] + c dt/(2dx) sum_d [U(i+1) - 2U + U(i-1)]."""
    P = pressure(U, c)
    out = U.copy()
    for d, axis in ((0, 2), (1, 1), (2, 0)):          # x is the last grid axis
        Ft = np.empty_like(U)
        Ft[..., 0] = U[..., 1 + d]
        Ft[..., 1:] = c * c * P[..., d, :]
        up = lambda a: np.roll(a, -1, axis=axis)      # value at i+1
        dn = lambda a: np.roll(a, +1, axis=axis)      # value at i-1
        out -= dt / (2 * dx) * (up(Ft) - dn(Ft))
        out += c * dt / (2 * dx) * (up(U) - 2 * U + dn(U))
    return out


def rates(T):
    lam = 2 * 157807.0 / T
    aA = 1.269e-13 * lam ** 1.503 / (1 + (lam / 0.522) ** 0.470) ** 1.923
    aB = 2.753e-14 * lam ** 1.5 / (1 + (lam / 2.740) ** 0.407) ** 2.242
    be = 21.11 * T ** -1.5 * np.exp(-lam / 2) * lam ** -1.089 / (1 + (lam / 0.354) ** 0.874) ** 1.101
    exc = 7.5e-19 * np.exp(-118348.0 / T) / (1 + np.sqrt(T / 1e5))
    recA = 1.778e-29 * T * lam ** 1.965 / (1 + (lam / 0.541) ** 0.502) ** 2.697
    recB = 3.435e-30 * T * lam ** 1.970 / (1 + (lam / 2.250) ** 0.376) ** 3.720
    gff = 1.1 + 0.34 * np.exp(-(5.5 - np.log10(T)) ** 2 / 3)
    ff = 1.42e-27 * gff * np.sqrt(T)
    return aA, aB, be, exc + 2.179e-11 * be, recA + ff, recB + ff


def chem_cell(U, n0, x, e, S, dt, c, sigN, sigE, Emean, otsa=1, e_tol=0.1):
    """U: [G,4].  Returns U, x, e, n_accepted, n_halved.  (A5-A9; full thermal mode only)"""
    G = len(sigN)
    SigE = [sigE[i] * Emean[i] - sigN[i] * E_HI for i in range(G)]
    U = U.copy()
    rem, nacc, nhalv = dt, 0, 0
    while rem > 0:
        T = e / (1.5 * (1 + x) * n0 * K_B)
        aA, aB, be, cHI, cHIIA, cHIIB = rates(T)
        al, cHII = (aB, cHIIB) if otsa else (aA, cHIIA)
        rec = 0.0 if otsa else (aA - aB) * x * x * n0 * n0
        lam_of = lambda xx: n0 * n0 * (xx * (1 - xx) * cHI + xx * xx * cHII)
        H = c * (1 - x) * n0 * sum(SigE[i] * U[i, 0] for i in range(G))
        L = lam_of(x)
        dtau = rem if H == L else min(rem, abs(e / (H - L)))
        while True:
            den = [1 + c * sigN[i] * (1 - x) * n0 * dtau for i in range(G)]
            N1 = [(U[i, 0] + (S[i] + (rec if i == 0 else 0.0)) * dtau) / den[i] for i in range(G)]
            x1 = 1 - (al * x * x * n0 * dtau + 1 - x) / (1 + dtau * (be * x * n0 + c * sum(sigN[i] * N1[i] for i in range(G))))
            e1 = e + dtau * (c * (1 - x1) * n0 * sum(SigE[i] * N1[i] for i in range(G)) - lam_of(x1))
            if abs(e1 - e) > e_tol * e or e1 <= 0:
                dtau /= 2
                nhalv += 1
                continue
            break
        for i in range(G):
            U[i, 1:] = U[i, 1:] / den[i]
            U[i, 0] = N1[i]
        x, e = x1, e1
        nacc += 1
        rem = 0.0 if dtau >= rem else rem - dtau
    return U, x, e, nacc, nhalv


def wavespeeds(U, c, d):
    """Extreme eigenvalues of the M1 flux Jacobian in direction d (reading A19), in the cancellation-free
    form  l = c [r_d -/+ sqrt(R_d)] / xi,  r_d = F_d/(cN) (scaled by 1/f_raw if f_raw > 1),
    R_d = 2 (1 - f^2) (xi - 3 r_d^2 / (2 + xi)) / (xi + 1)  -- algebraically the textbook radicand
    (2/3)(xi^2 - xi) + 2 mu^2 (2 - f^2 - xi) with mu f = r_d and (2 - xi)/f^2 = 3/(2 + xi)."""
    N = U[..., 0]
    F = U[..., 1:]
    with np.errstate(divide="ignore", invalid="ignore"):
        r = np.where(N[..., None] > 0, F / (c * N[..., None]), 0.0)
    fraw = np.sqrt((r ** 2).sum(-1))
    r = r / np.maximum(fraw, 1.0)[..., None]
    f2 = np.minimum(fraw, 1.0) ** 2
    xi = np.sqrt(4 - 3 * f2)
    rd = r[..., d]
    R = np.maximum(2 * (1 - f2) * (xi - 3 * rd * rd / (2 + xi)) / (xi + 1), 0.0)
    return c * (rd - np.sqrt(R)) / xi, c * (rd + np.sqrt(R)) / xi


def transport_periodic_hll(U, c, dt, dx):
    """U: [nz, ny, nx, 4] fp64, periodic; Eq. 30 with the HLL interface flux of reading A19, face by face."""
    P = pressure(U, c)
    out = U.copy()
    for d, axis in ((0, 2), (1, 1), (2, 0)):
        Ft = np.empty_like(U)
        Ft[..., 0] = U[..., 1 + d]
        Ft[..., 1:] = c * c * P[..., d, :]
        lo, hi = wavespeeds(U, c, d)
        up = lambda a: np.roll(a, -1, axis=axis)      # value of the right cell of the face i+1/2
        lp = np.maximum(0.0, np.maximum(hi, up(hi)))[..., None]
        lm = np.minimum(0.0, np.minimum(lo, up(lo)))[..., None]
        den = lp - lm
        with np.errstate(divide="ignore", invalid="ignore"):
            Fh = np.where(den > 0, (lp * Ft - lm * up(Ft) + lp * lm * (up(U) - U)) / den, 0.5 * (Ft + up(Ft)))
        out -= dt / dx * (Fh - np.roll(Fh, +1, axis=axis))
    # A19: the updated state is kept realizable, |F| <= c max(N, 0)
    Fn = np.sqrt((out[..., 1:] ** 2).sum(-1))
    lim = c * np.maximum(out[..., 0], 0.0)
    with np.errstate(divide="ignore", invalid="ignore"):
        scale = np.where(Fn > lim, lim / Fn, 1.0)
    out[..., 1:] *= scale[..., None]
    return out
