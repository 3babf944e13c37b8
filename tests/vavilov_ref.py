"""Vavilov's energy-loss distribution from the characteristic function of the collision process (test reference only:
no code of the oracle or of the CUDA path is involved; numpy + scipy.special.sici)."""
import numpy as np


def vavilov_cdf(kappa, b2, n=1 << 18):
    """CDF of y = (loss - mean loss) / Tmax for Vavilov's distribution, by a route independent of any sampling: the loss is a
    compound Poisson process with collision spectrum xi (1 - beta^2 T/Tmax) / T^2 on (0, Tmax], so its centred
    characteristic function is exp{kappa [A(q) - beta^2 B(q)]} with A = int_0^1 (e^{iqt} - 1 - iqt)/t^2 dt
    = -(e^{iq} - 1 - iq) + iq E(q), B = int_0^1 (e^{iqt} - 1 - iqt)/t dt = E(q) - iq, E(q) = Ci(q) - ln q - gamma + i Si(q)
    (sine and cosine integrals from scipy); the density follows by FFT."""
    from scipy.special import sici
    sd = np.sqrt(kappa * (1 - b2 / 2))
    span = max(60 * sd, 6.0, 400 * kappa)                    # period of the y grid: bulk, tail up to several Tmax
    dy = span / n
    q = 2 * np.pi * np.fft.fftfreq(n, d=dy)
    aq = np.abs(q); aq[0] = 1.0
    si, ci = sici(aq)
    E = (ci - np.log(aq) - 0.5772156649015329) + 1j * si
    A = -(np.exp(1j * aq) - 1 - 1j * aq) + 1j * aq * E
    B = E - 1j * aq
    lnphi = kappa * (A - b2 * B)
    lnphi = np.where(q < 0, np.conj(lnphi), lnphi); lnphi[0] = 0.0
    y0 = -span * 0.25                                         # grid origin: the left quarter holds the bulk's left side
    y = y0 + dy * np.arange(n)
    dens = np.real(np.fft.fft(np.exp(lnphi) * np.exp(-1j * q * y0))) / span   # p(y_j) = (1/span) sum_q phi(q) e^{-iq y_j}
    dens = np.maximum(dens, 0.0)
    cdf = np.cumsum(dens) * dy
    return y, cdf / cdf[-1]
