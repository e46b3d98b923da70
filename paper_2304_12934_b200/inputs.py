"""Seeded synthetic inputs shaped like the paper's workloads.

Holds NONE of the method's arithmetic (no Radon, NUFFT, prior or optimiser code): only
phantom rasterisation and angle grids.  Serves both the CUDA path and the oracle's tests.
Recipes are stated in DESIGN.md ("Input recipe").  All outputs are float32, C-contiguous.
"""
import numpy as np

# (S, N, Nd, Na, centre) for BASELINE.json configs[0..4]
CONFIGS = {
    1: dict(S=1, N=64, Nd=64, Na=45, centre=32.0, seed=1001),
    2: dict(S=16, N=256, Nd=256, Na=181, centre=128.0, seed=1002),
    3: dict(S=64, N=1024, Nd=1024, Na=128, centre=512.0, seed=1003),
    4: dict(S=128, N=2048, Nd=2048, Na=1024, centre=1027.5, seed=1004),
    5: dict(S=2160, N=2560, Nd=2560, Na=1313, centre=1280.0, seed=1005),
}


def angles_uniform(na):
    """theta_a = a pi / Na in [0, pi), float32 of the float64 value."""
    return (np.arange(na, dtype=np.float64) * np.pi / na).astype(np.float32)


def _add_ellipse(img, x0, y0, a, b, phi, rho):
    """pixel-centre inclusion; x_j = j - N/2, y_i = i - N/2."""
    N = img.shape[0]
    r = int(np.ceil(max(a, b))) + 1
    j0, j1 = max(0, int(x0 + N // 2) - r), min(N, int(x0 + N // 2) + r + 1)
    i0, i1 = max(0, int(y0 + N // 2) - r), min(N, int(y0 + N // 2) + r + 1)
    if j0 >= j1 or i0 >= i1:
        return
    x = np.arange(j0, j1) - N // 2 - x0
    y = np.arange(i0, i1) - N // 2 - y0
    X, Y = np.meshgrid(x, y)
    c, s = np.cos(phi), np.sin(phi)
    inside = ((X * c + Y * s) / a) ** 2 + ((-X * s + Y * c) / b) ** 2 <= 1.0
    img[i0:i1, j0:j1] += rho * inside


def ellipse_phantom(n, n_ellipses, rng):
    """random ellipses inside the inscribed circle of radius 0.47 N; densities add where they overlap."""
    img = np.zeros((n, n), dtype=np.float64)
    for _ in range(n_ellipses):
        r = 0.3 * n * np.sqrt(rng.random()); ang = rng.random() * 2 * np.pi
        x0, y0 = r * np.cos(ang), r * np.sin(ang)
        a, b = rng.uniform(0.03, 0.25, size=2) * n
        lim = 0.47 * n - np.hypot(x0, y0)
        a, b = min(a, lim), min(b, lim)
        _add_ellipse(img, x0, y0, a, b, rng.random() * np.pi, rng.random())
    return img


def volume_cfg1():
    rng = np.random.default_rng(CONFIGS[1]['seed'])
    return ellipse_phantom(64, 10, rng)[None].astype(np.float32)


def volume_cfg2(S=16, n=256):
    out = np.empty((S, n, n), dtype=np.float32)
    for s in range(S):
        rng = np.random.default_rng(CONFIGS[2]['seed'] + s)
        img = ellipse_phantom(n, int(rng.integers(8, 17)), rng)
        out[s] = img + rng.normal(0.0, 0.01, size=img.shape)
    return out


def volume_porous(S, n, seed, n_pores=400, rmin=4.0, rmax=40.0):
    """cfg 3: solid cylinder radius 0.45 N, density 1, with spherical pores (density 0);
    radii U(rmin, rmax) px scaled by n/1024, centres uniform in the cylinder."""
    rng = np.random.default_rng(seed)
    x = np.arange(n) - n // 2
    vol = np.repeat(((x[None, :] ** 2 + x[:, None] ** 2) <= (0.45 * n) ** 2)[None], S, axis=0).astype(np.float32)
    scale = n / 1024.0
    for _ in range(n_pores):
        r = 0.45 * n * np.sqrt(rng.random()); ang = rng.random() * 2 * np.pi
        cx, cy, cz = r * np.cos(ang), r * np.sin(ang), rng.uniform(-rmax * scale, S + rmax * scale)
        R = rng.uniform(rmin, rmax) * scale
        for z in range(max(0, int(np.floor(cz - R))), min(S, int(np.ceil(cz + R)) + 1)):
            rr2 = R * R - (z - cz) ** 2
            if rr2 <= 0:
                continue
            q = int(np.ceil(np.sqrt(rr2))) + 1
            j0, j1 = max(0, int(cx + n // 2) - q), min(n, int(cx + n // 2) + q + 1)
            i0, i1 = max(0, int(cy + n // 2) - q), min(n, int(cy + n // 2) + q + 1)
            if j0 >= j1 or i0 >= i1:
                continue
            X, Y = np.meshgrid(np.arange(j0, j1) - n // 2 - cx, np.arange(i0, i1) - n // 2 - cy)
            vol[z, i0:i1, j0:j1][X * X + Y * Y <= rr2] = 0.0
    return vol


def _fibre_params(n, seed, n_fibres):
    rng = np.random.default_rng(seed)
    scale = n / 2048.0
    r = 0.44 * n * np.sqrt(rng.random(n_fibres)); ang = rng.random(n_fibres) * 2 * np.pi
    return dict(cx=r * np.cos(ang), cy=r * np.sin(ang), tilt=np.deg2rad(rng.uniform(0, 15, n_fibres)),
                az=rng.random(n_fibres) * 2 * np.pi, R=rng.uniform(3, 12, n_fibres) * scale, rho=rng.uniform(0.2, 1.0, n_fibres))


def _fibre_slice(args):
    z, S, n, seed, n_fibres = args
    q = _fibre_params(n, seed, n_fibres)
    x = np.arange(n) - n // 2
    img = 0.1 * ((x[None, :] ** 2 + x[:, None] ** 2) <= (0.47 * n) ** 2)
    dz = z - S / 2
    for k in range(n_fibres):
        sx = q["cx"][k] + dz * np.tan(q["tilt"][k]) * np.cos(q["az"][k])
        sy = q["cy"][k] + dz * np.tan(q["tilt"][k]) * np.sin(q["az"][k])
        a = q["R"][k] / np.cos(q["tilt"][k])
        if np.hypot(sx, sy) + a > 0.47 * n:
            continue
        _add_ellipse(img, sx, sy, a, q["R"][k], q["az"][k], q["rho"][k])
    return img.astype(np.float32)


def volume_fibres(S, n, seed, n_fibres=3000, workers=1):
    """cfg 4: matrix density 0.1 inside radius 0.47 N; cylinders within 15 deg of z, radii U(3,12) px
    (scaled by n/2048), density U(0.2, 1.0); a slice cuts each as an ellipse.  Slices are independent given the
    seed, so `workers` > 1 rasterises them in a process pool (same result)."""
    jobs = [(z, S, n, seed, n_fibres) for z in range(S)]
    if workers > 1:
        import multiprocessing as mp
        with mp.get_context("fork").Pool(workers) as pool:
            sl = pool.map(_fibre_slice, jobs, chunksize=max(1, S // (4 * workers)))
    else:
        sl = [_fibre_slice(j) for j in jobs]
    return np.stack(sl)


def poisson_sinogram(sino, seed, photons=1e4, peak=2.0):
    """cfg 3 noise: scale line integrals so max = peak, Poisson counts at `photons` per bin
    (floor 1), b = -log(counts/photons), rescaled back (Beer-Lambert)."""
    rng = np.random.default_rng(seed)
    sc = peak / max(float(np.max(sino)), 1e-30)
    counts = rng.poisson(photons * np.exp(-np.clip(sino * sc, 0, None)))
    counts = np.maximum(counts, 1)
    return (-np.log(counts / photons) / sc).astype(np.float32)
