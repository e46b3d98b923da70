"""qGGMRF prior (eqs. (12)-(13)), value and gradient.

Oracle -- test infrastructure only.  Readings (G10-G12):
  H(f)  = sum over unordered 26-neighbour pairs {m,n} of w_mn h(f_m - f_n)
  h(D)  = u^2 / (c + u^(2-p)),  u = |D|/sigma                           (eq. (13))
  h'(D) = sign(D)/sigma * u (2c + p u^(2-p)) / (c + u^(2-p))^2,  h'(0) = 0
  w_mn  = (1/||m-n||_2) / (6 + 12/sqrt2 + 8/sqrt3)   (weights sum to 1 over the 26)
  neighbours outside the volume are skipped.  Axis order (z, y, x).

Neighbour sets ("SVMBIR uses 10 nearest neighbors, while tomoCAM uses 26"): `neighbours` = 26 (the
1-hop cube of eq. (12)), 10 (the 8 in-plane neighbours and the 2 along z) or 6 (faces).  Weights stay 1/distance,
normalised to sum 1 over the chosen set.

curvH is the curvature of the quadratic (symmetric-bound) surrogate of H at f along a direction g,
  sum over pairs of w_mn h'(D)/D (g_m - g_n)^2,   h'(D)/D = (2c + p u^(2-p)) / (sigma^2 (c + u^(2-p))^2)  (2/(c sigma^2) at D = 0),
used by the majorise-minimise step length of oracle/mbir.py (G23).
"""
import itertools
import numpy as np

WSUM = 6.0 + 12.0 / np.sqrt(2.0) + 8.0 / np.sqrt(3.0)


def offsets26():
    return [o for o in itertools.product((-1, 0, 1), repeat=3) if o != (0, 0, 0)]


def offsets(neighbours=26):
    """(dz, dy, dx) of the neighbour set."""
    if neighbours == 26:
        return offsets26()
    if neighbours == 10:
        return [o for o in offsets26() if o[0] == 0 or (o[1] == 0 and o[2] == 0)]
    if neighbours == 6:
        return [o for o in offsets26() if sum(v * v for v in o) == 1]
    raise ValueError(neighbours)


def weight(off, neighbours=26):
    tot = WSUM if neighbours == 26 else sum(1.0 / np.sqrt(float(sum(v * v for v in o))) for o in offsets(neighbours))
    return 1.0 / np.sqrt(float(sum(v * v for v in off))) / tot


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


def H(f, p, sigma, c, neighbours=26):
    f = np.asarray(f, dtype=np.float64)
    tot = 0.0
    for off in offsets(neighbours):
        sa, sb = _shifted_pairs(f, off)
        tot += weight(off, neighbours) * np.sum(h(f[sa] - f[sb], p, sigma, c))
    return 0.5 * tot                                    # each unordered pair once


def gradH(f, p, sigma, c, neighbours=26):
    f = np.asarray(f, dtype=np.float64)
    g = np.zeros_like(f)
    for off in offsets(neighbours):
        sa, sb = _shifted_pairs(f, off)
        g[sa] += weight(off, neighbours) * dh(f[sa] - f[sb], p, sigma, c)
    return g


def dh_over_D(D, p, sigma, c):
    u = np.abs(D) / sigma
    uq = u ** (2.0 - p)
    return (2.0 * c + p * uq) / (sigma * sigma * (c + uq) ** 2)


def curvH(f, g, p, sigma, c, neighbours=26):
    f = np.asarray(f, dtype=np.float64); g = np.asarray(g, dtype=np.float64)
    tot = 0.0
    for off in offsets(neighbours):
        sa, sb = _shifted_pairs(f, off)
        tot += weight(off, neighbours) * np.sum(dh_over_D(f[sa] - f[sb], p, sigma, c) * (g[sa] - g[sb]) ** 2)
    return 0.5 * tot                                    # each unordered pair once
