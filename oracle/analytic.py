"""Closed-form line integrals and a ray-driven projector: what (D1) approximates.

Oracle -- test infrastructure only.  Follows eq. (2): Rf(t, n) = integral of
f over the line <x, n> = t, n = (cos theta, sin theta).
"""
import numpy as np


def gaussian_projection(x0, y0, s, angles, nd, centre):
    """f = exp(-((x-x0)^2+(y-y0)^2)/(2 s^2))  =>  Rf(t) = sqrt(2 pi) s exp(-(t-t0)^2/(2 s^2)),
    t0 = x0 cos + y0 sin.  Returns (Na, Nd) sampled at t_u = u - centre."""
    t = np.arange(nd) - centre
    out = np.empty((len(angles), nd))
    for a, th in enumerate(angles):
        t0 = x0 * np.cos(th) + y0 * np.sin(th)
        out[a] = np.sqrt(2 * np.pi) * s * np.exp(-(t - t0) ** 2 / (2 * s * s))
    return out


def ellipse_projection(x0, y0, a_, b_, phi, rho, angles, nd, centre):
    """Ellipse centre (x0,y0), semi-axes a_, b_, rotated by phi, density rho:
    Rf(t) = 2 rho a b sqrt(s2 - tau^2)/s2,  s2 = a^2 cos^2(th-phi) + b^2 sin^2(th-phi),
    tau = t - x0 cos th - y0 sin th."""
    t = np.arange(nd) - centre
    out = np.empty((len(angles), nd))
    for k, th in enumerate(angles):
        s2 = (a_ * np.cos(th - phi)) ** 2 + (b_ * np.sin(th - phi)) ** 2
        tau = t - x0 * np.cos(th) - y0 * np.sin(th)
        out[k] = 2 * rho * a_ * b_ * np.sqrt(np.maximum(s2 - tau * tau, 0.0)) / s2
    return out


def radon_ray(f, angles, nd, centre, step=0.25):
    """Ray-driven projector: integrate the bilinear interpolant of the pixel samples
    along x = t n + s n_perp, n_perp = (-sin, cos), with the rectangle rule, pitch `step`."""
    f = np.asarray(f, dtype=np.float64)
    N = f.shape[0]
    t = np.arange(nd) - centre
    s = np.arange(-N, N + step, step)
    out = np.empty((len(angles), nd))
    for a, th in enumerate(angles):
        c, sn = np.cos(th), np.sin(th)
        X = t[:, None] * c - s[None, :] * sn + N // 2      # column coordinate j
        Y = t[:, None] * sn + s[None, :] * c + N // 2      # row coordinate i
        j0 = np.floor(X).astype(int)
        i0 = np.floor(Y).astype(int)
        fx, fy = X - j0, Y - i0
        acc = np.zeros_like(X)
        for di, wy in ((0, 1 - fy), (1, fy)):
            for dj, wx in ((0, 1 - fx), (1, fx)):
                ii, jj = i0 + di, j0 + dj
                ok = (ii >= 0) & (ii < N) & (jj >= 0) & (jj < N)
                acc += np.where(ok, f[np.clip(ii, 0, N - 1), np.clip(jj, 0, N - 1)], 0.0) * wy * wx
        out[a] = acc.sum(axis=1) * step
    return out
