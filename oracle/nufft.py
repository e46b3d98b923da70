"""The NUFFT approximation of the Radon pair, step by step (eqs. (6)-(8)).

Oracle -- test infrastructure only.  float64; numpy.fft and numpy.i0 are the
library primitives.  Adjoint = eqs. (6) -> (7) -> (8) in the paper's order; forward
= "the above steps in reverse order".  Readings (G5, G6):
separable Kaiser-Bessel window, W = 6, sigma = 2, Beatty beta, taps
b = ceil(kappa - W/2) ... b + W - 1 (window closed at +W/2).

  window  phi(r)   = I0(beta sqrt(1 - (2r/W)^2)) / I0(beta),  |r| <= W/2, else 0
  deapod  phihat(x) = W sinh(s)/s / I0(beta),  s = sqrt(beta^2 - (pi W x/G)^2);  d = 1/phihat
"""
import numpy as np


def kb_beta(W=6, sigma=2.0):
    return np.pi * np.sqrt((W / sigma) ** 2 * (sigma - 0.5) ** 2 - 0.8)


def kb_window(r, W=6, sigma=2.0):
    beta = kb_beta(W, sigma)
    r = np.asarray(r, dtype=np.float64)
    q = 1.0 - (2.0 * r / W) ** 2
    inside = q >= 0.0
    return np.where(inside, np.i0(beta * np.sqrt(np.where(inside, q, 0.0))) / np.i0(beta), 0.0)


def kb_deapod(n, G, W=6, sigma=2.0):
    """d(x_j) = 1/phihat(x_j) for x_j = j - n/2, j = 0..n-1."""
    beta = kb_beta(W, sigma)
    x = np.arange(n) - n // 2
    s = np.sqrt(beta ** 2 - (np.pi * W * x / G) ** 2)
    return np.i0(beta) * s / (W * np.sinh(s))


def _modes(nd):
    return np.arange(-(nd // 2) + 1, nd // 2)


def _taps(kappa, W):
    b = np.ceil(kappa - W / 2.0).astype(np.int64)        # first tap
    return b


def pad_deapod(f, G, W=6, sigma=2.0):
    """eq. (8) read backwards: g = f d d on a zero G x G array at periodic index (i - N/2) mod G."""
    N = f.shape[-1]
    d = kb_deapod(N, G, W, sigma)
    g = np.zeros(f.shape[:-2] + (G, G), dtype=np.complex128)
    idx = (np.arange(N) - N // 2) % G
    g[..., idx[:, None], idx[None, :]] = f * d[:, None] * d[None, :]
    return g


def gather(Ghat, angles, nd, W=6, sigma=2.0):
    """eq. (7) reversed: c[a][m] = sum_{W x W} Ghat[(by+ty) mod G][(bx+tx) mod G] phi phi,
    kappa = G k_m (cos, sin).  Ghat: (..., G, G) -> (..., Na, M)."""
    G = Ghat.shape[-1]
    m = _modes(nd)
    th = np.asarray(angles, dtype=np.float64)
    kx = G * (m[None, :] / nd) * np.cos(th)[:, None]
    ky = G * (m[None, :] / nd) * np.sin(th)[:, None]
    bx, by = _taps(kx, W), _taps(ky, W)
    c = np.zeros(Ghat.shape[:-2] + kx.shape, dtype=np.complex128)
    for ty in range(W):
        wy = kb_window(ky - by - ty, W, sigma)
        for tx in range(W):
            wx = kb_window(kx - bx - tx, W, sigma)
            c += Ghat[..., (by + ty) % G, (bx + tx) % G] * (wy * wx)
    return c


def spread(c, angles, nd, G, W=6, sigma=2.0):
    """eq. (7): Ghat[r] += c[a][m] phi phi over the same W x W taps.  c: (Na, M)."""
    m = _modes(nd)
    th = np.asarray(angles, dtype=np.float64)
    kx = G * (m[None, :] / nd) * np.cos(th)[:, None]
    ky = G * (m[None, :] / nd) * np.sin(th)[:, None]
    bx, by = _taps(kx, W), _taps(ky, W)
    Ghat = np.zeros((G, G), dtype=np.complex128)
    for ty in range(W):
        wy = kb_window(ky - by - ty, W, sigma)
        for tx in range(W):
            wx = kb_window(kx - bx - tx, W, sigma)
            np.add.at(Ghat, ((by + ty) % G, (bx + tx) % G), c * (wy * wx))
    return Ghat


def radial_inverse(c, nd, centre):
    """eq. (6) reversed + Fourier shift:
    p[a][u] = (1/Nd) sum_{|m|<Nd/2} c[a][m] e^{2 pi i m (u - centre)/Nd}   (complex)."""
    m = _modes(nd)
    C = np.zeros(c.shape[:-1] + (nd,), dtype=np.complex128)
    C[..., m % nd] = c * np.exp(-2j * np.pi * m * centre / nd)
    return np.fft.ifft(C, axis=-1)


def radial_forward(y, nd, centre):
    """eq. (6): c[a][m] = (1/Nd) sum_u y[a][u] e^{-2 pi i m (u - centre)/Nd}, |m| < Nd/2."""
    m = _modes(nd)
    Y = np.fft.fft(np.asarray(y, dtype=np.float64), axis=-1) / nd
    return Y[..., m % nd] * np.exp(2j * np.pi * m * centre / nd)


def radon_nufft(f, angles, nd, centre, sigma=2.0, W=6):
    """Forward (type-2) NUFFT Radon.  f: (S, N, N) or (N, N) -> (S, Na, Nd) float64."""
    f = np.asarray(f, dtype=np.float64)
    squeeze = f.ndim == 2
    if squeeze:
        f = f[None]
    S, N, _ = f.shape
    G = int(round(sigma * N))
    out = np.empty((S, len(angles), nd))
    for s in range(S):
        Ghat = np.fft.fft2(pad_deapod(f[s], G, W, sigma))
        c = gather(Ghat, angles, nd, W, sigma)
        out[s] = radial_inverse(c, nd, centre).real
    return out[0] if squeeze else out


def backproject_nufft(y, angles, n, centre, sigma=2.0, W=6):
    """Adjoint (type-1) NUFFT back-projection: the exact transpose of radon_nufft."""
    y = np.asarray(y, dtype=np.float64)
    squeeze = y.ndim == 2
    if squeeze:
        y = y[None]
    S, na, nd = y.shape
    G = int(round(sigma * n))
    d = kb_deapod(n, G, W, sigma)
    idx = (np.arange(n) - n // 2) % G
    out = np.empty((S, n, n))
    for s in range(S):
        c = radial_forward(y[s], nd, centre)
        Ghat = spread(c, angles, nd, G, W, sigma)
        g = np.fft.ifft2(Ghat) * (G * G)                 # unnormalised inverse, eq. (8)
        out[s] = (g[idx[:, None], idx[None, :]] * d[:, None] * d[None, :]).real
    return out[0] if squeeze else out
