"""Seeded random fields (SURVEY.md 8(d) recipe): Gaussian random field with P(k) ~ k^-2 and its
lognormal transform.  numpy default_rng (PCG64) only; fp64 generation, rounded once to fp32."""
import numpy as np


def gaussian_random_field(n, rng):
    """Unit-variance, zero-mean GRF on an n^3 periodic grid with P(k) proportional to k^-2.

    white noise -> rfftn -> multiply amplitudes by k^-1 (so power ~ k^-2), DC mode zeroed -> irfftn ->
    rescale to unit sample variance.  Array index order is [z, y, x]."""
    w = rng.standard_normal((n, n, n))
    wk = np.fft.rfftn(w)
    del w
    kf = np.fft.fftfreq(n) * n
    kr = np.fft.rfftfreq(n) * n
    k2 = (kf[:, None, None] ** 2 + kf[None, :, None] ** 2 + kr[None, None, :] ** 2)
    k2[0, 0, 0] = 1.0
    wk *= 1.0 / np.sqrt(k2)
    wk[0, 0, 0] = 0.0
    del k2
    d = np.fft.irfftn(wk, s=(n, n, n), axes=(0, 1, 2))
    del wk
    d -= d.mean()
    d /= d.std()
    return d


def lognormal_density(n, nbar, sigma_ln, rng):
    """n0 = nbar * exp(sigma_ln * delta - sigma_ln^2/2), rescaled so the sample mean is exactly nbar (fp64)."""
    d = gaussian_random_field(n, rng)
    n0 = np.exp(sigma_ln * d - 0.5 * sigma_ln ** 2)
    n0 *= nbar / n0.mean()
    return n0
