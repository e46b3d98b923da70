"""Filtered back-projection, eq. (4): f = R* F^-1 |k| F p (filters: P:L68).

Oracle -- test infrastructure only (float64).  Discretisation (reading G20): the inner product over
(k, theta) of eq. (4) with measures dk = 1/Nd and dtheta = pi/Na, i.e. the adjoint (D2) of oracle/direct.py with every
radial mode m weighted by

    rho[m] = (pi / Na) * r(|m| / Nd) * win(m),     r(k) = k for m != 0,   r = 1 / (4 Nd) at m = 0

(the mean of |k| over the DC bin [-1/(2 Nd), 1/(2 Nd)], so the reconstruction keeps its mean), win = 1 (ramp = Ram-Lak), the Hann
window 0.5 (1 + cos(2 pi m / Nd)), Shepp-Logan sinc(m / Nd) = sin(pi m / Nd) / (pi m / Nd), or Butterworth 1 / (1 + (x / 0.5)^4),
x = |m| / (Nd / 2) (order 2, cut-off at half the Nyquist frequency); the filters the paper names.
The Nyquist mode is excluded like everywhere else (G2).

  fbp_direct   the definition, O(Na Nd N^2)
  fbp_nufft    the same weights inside the oracle's NUFFT adjoint (radial_forward -> weight -> spread -> ifft2 -> crop)
"""
import numpy as np
from . import nufft


def _modes(nd):
    return np.arange(-(nd // 2) + 1, nd // 2)


def ramp_weights(nd, na, window="ramp"):
    """rho[m] for m = -(Nd/2)+1 .. Nd/2-1."""
    m = _modes(nd)
    r = np.abs(m) / nd
    r[m == 0] = 0.25 / nd
    if window == "hann":
        r = r * 0.5 * (1.0 + np.cos(2.0 * np.pi * m / nd))
    elif window == "shepp-logan":
        r = r * np.sinc(m / nd)                                     # numpy's sinc(x) = sin(pi x) / (pi x)
    elif window == "butterworth":
        r = r / (1.0 + (np.abs(m) / (nd / 2.0) / 0.5) ** 4)
    elif window != "ramp":
        raise ValueError(window)
    return (np.pi / na) * r


def fbp_direct(y, angles, n, centre, window="ramp"):
    """y: (Na, Nd) or (S, Na, Nd) real -> (S, N, N) float64."""
    y = np.asarray(y, dtype=np.float64)
    squeeze = y.ndim == 2
    if squeeze:
        y = y[None]
    S, na, nd = y.shape
    m = _modes(nd)
    k = m / nd
    x = np.arange(n) - n // 2
    u = np.arange(nd)
    rho = ramp_weights(nd, na, window)
    Q = np.exp(-2j * np.pi * np.outer(m, u - centre) / nd)          # (M, Nd): P^[a][m] = sum_u p[u] e^{-2 pi i m (u - centre)/Nd}
    out = np.zeros((S, n, n))
    for a, th in enumerate(np.asarray(angles, dtype=np.float64)):
        c = (y[:, a, :] @ Q.T) * (rho / nd)                         # dk = 1/Nd
        Ex = np.exp(2j * np.pi * np.outer(k, x) * np.cos(th))
        Ey = np.exp(2j * np.pi * np.outer(k, x) * np.sin(th))
        out += np.einsum('smi,mj->sij', c[:, :, None] * Ey[None], Ex).real
    return out[0] if squeeze else out


def fbp_nufft(y, angles, n, centre, window="ramp", sigma=2.0, W=6):
    y = np.asarray(y, dtype=np.float64)
    squeeze = y.ndim == 2
    if squeeze:
        y = y[None]
    S, na, nd = y.shape
    G = int(round(sigma * n))
    d = nufft.kb_deapod(n, G, W, sigma)
    idx = (np.arange(n) - n // 2) % G
    rho = ramp_weights(nd, na, window)
    out = np.empty((S, n, n))
    for s in range(S):
        c = nufft.radial_forward(y[s], nd, centre) * rho
        g = np.fft.ifft2(nufft.spread(c, angles, nd, G, W, sigma)) * (G * G)
        out[s] = (g[idx[:, None], idx[None, :]] * d[:, None] * d[None, :]).real
    return out[0] if squeeze else out
