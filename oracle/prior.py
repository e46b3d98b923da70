"""qGGMRF prior (eqs. (12)-(13)), value and gradient.

Oracle -- test infrastructure only.  Readings (G10-G12):
  H(f)  = sum over unordered 26-neighbour pairs {m,n} of w_mn h(f_m - f_n)
  h(D)  = u^2 / (c + u^(2-p)),  u = |D|/sigma                           (eq. (13))
  h'(D) = sign(D)/sigma * u (2c + p u^(2-p)) / (c + u^(2-p))^2,  h'(0) = 0
  w_mn  = (1/||m-n||_2) / (6 + 12/sqrt2 + 8/sqrt3)   (weights sum to 1 over the 26)
  neighbours outside the volume are skipped.  Axis order (z, y, x).
"""
import itertools
import numpy as np

WSUM = 6.0 + 12.0 / np.sqrt(2.0) + 8.0 / np.sqrt(3.0)


def offsets26():
    return [o for o in itertools.product((-1, 0, 1), repeat=3) if o != (0, 0, 0)]


def weight(off):
    return 1.0 / np.sqrt(float(sum(v * v for v in off))) / WSUM


def h(D, p, sigma, c):
    u = np.abs(D) / sigma
    return u * u / (c + u ** (2.0 - p))


def dh(D, p, sigma, c):
    u = np.abs(D) / sigma
    uq = u ** (2.0 - p)
    return np.sign(D) / sigma * u * (2.0 * c + p * uq) / (c + uq) ** 2


def _shifted_pairs(f, off):
    """views (a, b) with b = f shifted by off, restricted to the overlap."""
    sa, sb = [], []
    for o, n in zip(off, f.shape):
        if o == 0:
            sa.append(slice(0, n)); sb.append(slice(0, n))
        elif o == 1:
            sa.append(slice(0, n - 1)); sb.append(slice(1, n))
        else:
            sa.append(slice(1, n)); sb.append(slice(0, n - 1))
    return tuple(sa), tuple(sb)


def H(f, p, sigma, c):
    f = np.asarray(f, dtype=np.float64)
    tot = 0.0
    for off in offsets26():
        sa, sb = _shifted_pairs(f, off)
        tot += weight(off) * np.sum(h(f[sa] - f[sb], p, sigma, c))
    return 0.5 * tot                                    # each unordered pair once


def gradH(f, p, sigma, c):
    f = np.asarray(f, dtype=np.float64)
    g = np.zeros_like(f)
    for off in offsets26():
        sa, sb = _shifted_pairs(f, off)
        g[sa] += weight(off) * dh(f[sa] - f[sb], p, sigma, c)
    return g
