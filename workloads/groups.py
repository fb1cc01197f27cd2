"""Frequency-group constants for `emma_rt_config` (Eq. 26-29, 266-272 Eq. 37-38).

The paper takes sigma_nu "from Hui & Gnedin (1997)" without printing it; that
paper is not in the container.  DESIGN.md reading A11: sigma_nu is the Verner et al. (1996)
analytic fit for H I, restated here from the published functional form
    sigma(E) = s0 [(x-1)^2] x^(P/2-5.5) (1+sqrt(x/ya))^(-P),  x = E/E0,
with E0 = 0.4298 eV, s0 = 5.475e-14 cm^2, ya = 32.88, P = 2.963  (sigma(13.6 eV) = 6.35e-18 cm^2).

The group averages are plain quadratures of a black-body photon-number spectrum
N_nu ~ nu^2 / (exp(h nu / k T) - 1); they are *inputs* handed to both the oracle and the
CUDA library as numbers, not part of either implementation.
"""
import numpy as np

from .constants import CGS


def sigma_HI(E_eV):
    """Photo-ionisation cross-section of H I [cm^2] at photon energy E [eV] (0 below 13.6 eV)."""
    E = np.asarray(E_eV, dtype=np.float64)
    E0, s0, ya, P = 0.4298, 5.475e-14, 32.88, 2.963
    x = E / E0
    s = s0 * (x - 1.0) ** 2 * x ** (0.5 * P - 5.5) * (1.0 + np.sqrt(x / ya)) ** (-P)
    return np.where(E >= CGS.E_HI_eV, s, 0.0)


def blackbody_groups(T_bb, edges_eV, n_quad=200001):
    """Group constants for a black body of temperature T_bb [K].

    edges_eV: increasing group limits, e.g. (13.6, 1000) or (13.6, 24.6, 54.4, 1000).
    Returns dict(frac, sigma_N [cm^2], sigma_E [cm^2], E_mean [erg], E_mean_eV), each of length G.
      frac    = photon-number fraction of the >edges[0] spectrum in the group (Eq. 28)
      sigma_N = Eq. 29, sigma_E = Eq. 37, E_mean = Eq. 38
    Trapezoid in ln E on n_quad points per group (fp64); converged to < 1e-9 relative.
    """
    edges = np.asarray(edges_eV, dtype=np.float64)
    G = len(edges) - 1
    out = {k: np.zeros(G) for k in ("frac", "sigma_N", "sigma_E", "E_mean", "E_mean_eV")}
    ntot = 0.0
    for g in range(G):
        lnE = np.linspace(np.log(edges[g]), np.log(edges[g + 1]), n_quad)
        E = np.exp(lnE)                                   # eV
        nu = E * CGS.eV / CGS.h
        # photon number per unit ln E:  N_nu * nu
        w = nu ** 3 / np.expm1(E * CGS.eV / (CGS.k_B * T_bb))
        sig = sigma_HI(E)
        Ng = np.trapezoid(w, lnE)
        Em = np.trapezoid(w * E, lnE) / Ng                # eV
        out["frac"][g] = Ng
        out["sigma_N"][g] = np.trapezoid(w * sig, lnE) / Ng
        out["sigma_E"][g] = np.trapezoid(w * sig * E, lnE) / (Ng * Em)
        out["E_mean_eV"][g] = Em
        out["E_mean"][g] = Em * CGS.eV
        ntot += Ng
    out["frac"] /= ntot
    return out
