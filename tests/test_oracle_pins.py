"""Pins for the oracle (no GPU): closed forms, brute force, invariants -- nothing here re-calls the
oracle's own formula as the expected value.  Citations: P:L<n> = /root/reference/PAPER.md line."""
import math, os
import numpy as np
import pytest
from conftest import rel_l2
from oracle import direct, analytic, nufft, prior, mbir

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _load(name):
    return np.loadtxt(os.path.join(GOLD, name), comments="#")


# ---------------------------------------------------------------- (D1) scale, sign, axes, centre
def test_d1_golden_delta_row():
    f = np.zeros((8, 8)); f[5, 2] = 1.0
    row = direct.radon_direct(f, [math.pi / 5], 8, 4.0)[0]
    assert np.allclose(row, _load("dirichlet_delta_n8.txt"), atol=1e-12)


@pytest.mark.parametrize("s,tol", [(3.0, 1e-12), (2.0, 1e-7)])
def test_d1_gaussian_closed_form(s, tol):
    # eq. (2) P:L48 in closed form for a Gaussian blob; off-centre blob, non-integer centre:
    # pins the scale (1/Nd, unit pixels), the sign of t, the x/y axes and the centre convention.
    N, x0, y0, centre = 64, 5.0, -7.0, 33.75
    x = np.arange(N) - N // 2
    f = np.exp(-((x[None, :] - x0) ** 2 + (x[:, None] - y0) ** 2) / (2 * s * s))
    ang = np.array([0.0, 0.3, math.pi / 2, 2.0, 3.0])
    got = direct.radon_direct(f, ang, N, centre)
    want = analytic.gaussian_projection(x0, y0, s, ang, N, centre)
    assert rel_l2(got, want) < tol


@pytest.mark.parametrize("centre", [4.0, 4.5, 3.25])
def test_d1_equals_dirichlet_form(centre):
    rng = np.random.default_rng(1)
    f = rng.standard_normal((8, 8)); ang = rng.uniform(0, math.pi, 5)
    assert rel_l2(direct.radon_direct(f, ang, 8, centre), direct.radon_dirichlet(f, ang, 8, centre)) < 1e-12


def test_d1_axis_angles_reduce_to_fft_and_sums():
    # theta = 0 integrates along y: column sums minus their Nyquist component; theta = pi/2: row sums.
    rng = np.random.default_rng(2); N = 16
    f = rng.standard_normal((N, N))
    p = direct.radon_direct(f, [0.0, math.pi / 2], N, N / 2)
    for row, cs in ((p[0], f.sum(axis=0)), (p[1], f.sum(axis=1))):
        sgn = (-1.0) ** np.arange(N)
        assert np.allclose(row, cs - sgn * np.sum(sgn * cs) / N, atol=1e-12)
    # slice theorem (eq. (3)) on the library FFT: F1[Af](m) = fft2(f shifted)[0][m] at theta = 0
    F1 = np.fft.fft(np.roll(p[0], -N // 2))                      # origin of t at bin N/2
    F2 = np.fft.fft2(np.roll(f, (-N // 2, -N // 2), axis=(0, 1)))
    m = np.arange(1, N // 2)
    assert np.allclose(F1[m], F2[0, m], atol=1e-10) and np.allclose(F1[-m], F2[0, -m], atol=1e-10)
    assert abs(F1[N // 2]) < 1e-10                               # Nyquist excluded (reading G2)


def test_d2_is_transpose_bruteforce_and_identity():
    rng = np.random.default_rng(3); N = 8
    ang = rng.uniform(0, math.pi, 6); centre = 4.25
    A = direct.dense_matrix(N, ang, N, centre)                   # Dirichlet form, independent code path
    y = rng.standard_normal((6, N))
    assert rel_l2(direct.backproject_direct(y, ang, N, centre).ravel(), A.T @ y.ravel()) < 1e-12
    x = rng.standard_normal((N, N))
    assert rel_l2(direct.radon_direct(x, ang, N, centre).ravel(), A @ x.ravel()) < 1e-12
    N = 32; ang = rng.uniform(0, math.pi, 11)
    x = rng.standard_normal((2, N, N)); y = rng.standard_normal((2, 11, N))
    lhs = np.sum(direct.radon_direct(x, ang, N, 17.5) * y); rhs = np.sum(x * direct.backproject_direct(y, ang, N, 17.5))
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs)


# ---------------------------------------------------------------- continuous line integral (loose by nature)
def test_ellipse_analytic_and_ray_driven():
    errs = []
    for N in (64, 128):
        x = np.arange(N) - N // 2
        X, Y = np.meshgrid(x, x)
        ell = [(0.1 * N, -0.05 * N, 0.3 * N, 0.2 * N, 0.4, 1.0), (-0.15 * N, 0.1 * N, 0.1 * N, 0.15 * N, 1.1, 0.5)]
        ang = np.arange(12) * math.pi / 12
        f = np.zeros((N, N)); want = np.zeros((12, N))
        for (x0, y0, a, b, phi, rho) in ell:
            c, s = math.cos(phi), math.sin(phi)
            f += rho * ((((X - x0) * c + (Y - y0) * s) / a) ** 2 + ((-(X - x0) * s + (Y - y0) * c) / b) ** 2 <= 1)
            want += analytic.ellipse_projection(x0, y0, a, b, phi, rho, ang, N, N / 2)
        errs.append(rel_l2(direct.radon_direct(f, ang, N, N / 2), want))
        assert rel_l2(analytic.radon_ray(f, ang, N, N / 2), want) < 0.03
    assert errs[0] < 0.03 and errs[1] < 0.015 and errs[1] < errs[0]


def test_ray_driven_gaussian():
    N, s = 64, 6.0      # bilinear interpolation widens the blob by ~1/6 px^2: loose pin
    x = np.arange(N) - N // 2
    f = np.exp(-((x[None, :] - 4) ** 2 + (x[:, None] + 6) ** 2) / (2 * s * s))
    ang = np.array([0.2, 1.3, 2.9])
    assert rel_l2(analytic.radon_ray(f, ang, N, 31.5), analytic.gaussian_projection(4, -6, s, ang, N, 31.5)) < 5e-3


# ---------------------------------------------------------------- the NUFFT approximation (eqs. (6)-(8))
@pytest.mark.parametrize("centre", [32.0, 35.5])
def test_nufft_within_error_bound_of_direct(centre):
    # w ~ log10(1/eps) P:L87: W = 6 => eps ~ 1e-6..1e-5
    rng = np.random.default_rng(4); N = 64
    ang = np.arange(45) * math.pi / 45
    f = rng.random((N, N)); y = rng.standard_normal((45, N))
    assert rel_l2(nufft.radon_nufft(f, ang, N, centre), direct.radon_direct(f, ang, N, centre)) < 2e-5
    assert rel_l2(nufft.backproject_nufft(y, ang, N, centre), direct.backproject_direct(y, ang, N, centre)) < 2e-5


def test_nufft_vs_bruteforce_matrix_8x8_and_exact_transpose():
    rng = np.random.default_rng(5); N = 8
    ang = rng.uniform(0, math.pi, 7); centre = 3.75
    A = direct.dense_matrix(N, ang, N, centre)
    An = np.stack([nufft.radon_nufft(e.reshape(N, N), ang, N, centre).ravel() for e in np.eye(N * N)], axis=1)
    Bn = np.stack([nufft.backproject_nufft(e.reshape(7, N), ang, N, centre).ravel() for e in np.eye(7 * N)], axis=1)
    assert np.abs(An - A).max() < 3e-5 * np.abs(A).max()
    assert np.abs(Bn - An.T).max() < 1e-13 * np.abs(An).max()    # exact transpose, not just approximate


def test_nufft_adjoint_identity_and_stage_transposes():
    rng = np.random.default_rng(6); N, na = 32, 9; G = 64
    ang = rng.uniform(0, math.pi, na)
    x = rng.standard_normal((N, N)); y = rng.standard_normal((na, N))
    lhs = np.sum(nufft.radon_nufft(x, ang, N, 15.5) * y); rhs = np.sum(x * nufft.backproject_nufft(y, ang, N, 15.5))
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs)
    Gh = rng.standard_normal((G, G)) + 1j * rng.standard_normal((G, G))
    c = rng.standard_normal((na, N - 1)) + 1j * rng.standard_normal((na, N - 1))
    assert abs(np.vdot(c, nufft.gather(Gh, ang, N)) - np.vdot(nufft.spread(c, ang, N, G), Gh)) < 1e-10
    p = rng.standard_normal((na, N))
    assert abs(np.vdot(p, nufft.radial_inverse(c, N, 15.5)).real - np.vdot(nufft.radial_forward(p, N, 15.5), c).real) < 1e-10


def test_kb_window_properties():
    # phihat is the Fourier transform of phi: check by quadrature (independent of the closed form)
    W, G = 6, 128
    r = np.linspace(-3, 3, 200001)
    phi = nufft.kb_window(r)
    for xj in (0, 10, 31):
        num = np.trapezoid(phi * np.cos(2 * np.pi * r * xj / G), r)
        assert abs(num * nufft.kb_deapod(64, G)[xj + 32] - 1.0) < 1e-6
    assert nufft.kb_window(3.0) > 0 and nufft.kb_window(3.0000001) == 0 and abs(nufft.kb_beta() - math.pi * math.sqrt(19.45)) < 1e-14


# ---------------------------------------------------------------- prior, eqs. (12)-(13)
P, SIG, C = 1.2, 1 / 0.7, 1e-4


def test_prior_golden_spot_values():
    for D, hv, dv in _load("qggmrf_spot.txt"):
        assert abs(prior.h(D, P, SIG, C) - hv) < 1e-12 and abs(prior.dh(D, P, SIG, C) - dv) < 1e-12
        assert abs(prior.dh(-D, P, SIG, C) + dv) < 1e-12
    assert prior.dh(0.0, P, SIG, C) == 0.0


def test_prior_weights_and_bruteforce_H():
    offs = prior.offsets26()
    assert len(offs) == 26 and abs(sum(prior.weight(o) for o in offs) - 1.0) < 1e-14
    assert abs(prior.weight((0, 0, 1)) - 0.0523448) < 1e-7 and abs(prior.weight((1, 1, 1)) - 0.0302213) < 1e-7
    rng = np.random.default_rng(7); f = rng.standard_normal((3, 4, 5))
    tot = 0.0                                                    # plain loops over unordered pairs, eq. (12)
    idx = [(z, y, x) for z in range(3) for y in range(4) for x in range(5)]
    for a in idx:
        for b in idx:
            d = max(abs(a[k] - b[k]) for k in range(3))
            if d == 1 and a < b:
                dist = math.sqrt(sum((a[k] - b[k]) ** 2 for k in range(3)))
                u = abs(f[a] - f[b]) / SIG
                tot += (1 / dist / (6 + 12 / math.sqrt(2) + 8 / math.sqrt(3))) * u * u / (C + u ** (2 - P))
    assert abs(prior.H(f, P, SIG, C) - tot) < 1e-12 * tot


def test_prior_gradient_finite_difference():
    rng = np.random.default_rng(8); f = rng.standard_normal((5, 6, 7))
    g = prior.gradH(f, P, SIG, C)
    eps = 1e-6
    for pos in [(0, 0, 0), (2, 3, 3), (4, 5, 6), (1, 0, 6), (2, 2, 0)]:
        fp = f.copy(); fm = f.copy(); fp[pos] += eps; fm[pos] -= eps
        fd = (prior.H(fp, P, SIG, C) - prior.H(fm, P, SIG, C)) / (2 * eps)
        assert abs(fd - g[pos]) < 1e-6 * max(1.0, abs(fd))
    assert np.all(prior.gradH(np.full((3, 4, 5), 0.7), P, SIG, C) == 0.0)


# ---------------------------------------------------------------- MBIR loop invariants (iterate sequence unpinned vs paper)
def test_mbir_invariants():
    rng = np.random.default_rng(9); N, na = 16, 12
    ang = np.arange(na) * math.pi / na
    truth = np.zeros((2, N, N)); truth[:, 5:11, 4:9] = 1.0; truth[1, 7:9, 6:12] += 0.5
    b = nufft.radon_nufft(truth, ang, N, 8.0) + 0.01 * rng.standard_normal((2, na, N))
    L, lam_hat = mbir.lipschitz(N, ang, N, 8.0, P, SIG, C, 1.0)
    assert 0.5 * na * N < lam_hat < 2.0 * na * N
    x1, log1 = mbir.mbir(b, ang, N, 8.0, P, SIG, C, 1.0, L, 1)
    assert rel_l2(x1, nufft.backproject_nufft(b, ang, N, 8.0) / L) < 1e-12      # first iterate = A^T b / L
    x, log = mbir.mbir(b, ang, N, 8.0, P, SIG, C, 1.0, L, 25)
    F = [0.5 * np.sum(b * b)] + [l["F"] for l in log]
    assert all(F[i + 1] <= F[i] for i in range(len(F) - 1)) and F[-1] < 0.5 * F[0]


def test_mbir_lambda0_meets_accelerated_rate_to_least_squares():
    # lambda = 0: the loop is accelerated gradient descent on 1/2||Ax-b||^2, whose textbook bound is
    # F(x_k) - F* <= 2 L ||x_0 - x*||^2 / (k+1)^2 with x* the (min-norm) least-squares solution of the
    # brute-force dense system; plain gradient descent (a dropped momentum term) would only give L/(2k).
    N, na = 8, 10
    ang = np.arange(na) * math.pi / na
    rng = np.random.default_rng(10)
    b = rng.standard_normal((1, na, N))
    An = np.stack([nufft.radon_nufft(e.reshape(N, N), ang, N, 4.0).ravel() for e in np.eye(N * N)], axis=1)
    xs = np.linalg.lstsq(An, b.ravel(), rcond=1e-10)[0]
    Fstar = 0.5 * np.sum((An @ xs - b.ravel()) ** 2)
    Lc = 1.02 * np.linalg.norm(An, 2) ** 2
    x, log = mbir.mbir(b, ang, N, 4.0, P, SIG, C, 0.0, Lc, 100)
    for k in (10, 50, 100):
        assert Fstar - 1e-9 <= log[k - 1]["F"] <= Fstar + 2 * Lc * np.sum(xs ** 2) / (k + 1) ** 2
    g0 = np.linalg.norm(An.T @ b.ravel())
    assert np.linalg.norm(An.T @ (An @ x.ravel() - b.ravel())) < 0.02 * g0
    assert abs(log[-1]["F"] - 0.5 * np.sum((An @ x.ravel() - b.ravel()) ** 2)) < 1e-9 * log[-1]["F"]


def test_mbir_nonneg_lambda0_converges_to_nnls():
    # The constrained loop (G21) with lambda = 0 is accelerated projected gradient on 1/2||Ax-b||^2 over x >= 0,
    # whose minimiser scipy's active-set NNLS computes from the brute-force dense matrix.  Data chosen so that the unconstrained
    # least-squares solution has negative entries (otherwise the projection would never act).
    from scipy.optimize import nnls
    N, na = 8, 10
    ang = np.arange(na) * math.pi / na
    rng = np.random.default_rng(33)
    b = rng.standard_normal((1, na, N))
    An = np.stack([nufft.radon_nufft(e.reshape(N, N), ang, N, 4.0).ravel() for e in np.eye(N * N)], axis=1)
    assert np.linalg.lstsq(An, b.ravel(), rcond=1e-10)[0].min() < -0.1
    xs, rn = nnls(An, b.ravel())
    Fstar = 0.5 * rn ** 2
    Lc = 1.02 * np.linalg.norm(An, 2) ** 2
    x, log, its = mbir.mbir(b, ang, N, 4.0, P, SIG, C, 0.0, Lc, 400, keep_iterates=True, nonneg=True)
    assert all(it.min() >= 0.0 for it in its)
    F = [l["F"] for l in log]
    assert all(F[i + 1] <= F[i] for i in range(len(F) - 1))
    assert Fstar - 1e-9 <= F[-1] <= Fstar * (1 + 1e-4) + 1e-9
    assert (x > 0).sum() < N * N                                   # some constraints are active
    # projected-gradient optimality (KKT): gradient >= 0 where x = 0, ~ 0 where x > 0
    g = An.T @ (An @ x.ravel() - b.ravel())
    g0 = np.linalg.norm(An.T @ b.ravel())
    assert np.abs(g[x.ravel() > 1e-6]).max() < 0.02 * g0 and g[x.ravel() <= 1e-6].min() > -0.02 * g0


def test_mbir_gradient_restart_variant():
    # DESIGN.md G22 ("monotonic ... with restart"): on a strongly convex, well-conditioned objective (quadratic prior p = 2)
    # plain accelerated gradient overshoots and the function-value test has to reject a candidate; the gradient test sees the
    # overshoot first (<g, z - x> > 0), resets the momentum, and ends lower.  Checks the mechanics of the flag, not a number.
    n, na = 32, 16
    ang = np.arange(na) * math.pi / na
    rng = np.random.default_rng(35)
    truth = np.zeros((2, n, n)); truth[:, 10:22, 8:20] = 1.0; truth[1, 14:18, 12:26] += 0.5
    b = nufft.radon_nufft(truth, ang, n, 16.0) + 0.01 * rng.standard_normal((2, na, n))
    p, sig, c, lam = 2.0, 1.0, 1.0, 200.0
    L, _ = mbir.lipschitz(n, ang, n, 16.0, p, sig, c, lam)
    xr, lr = mbir.mbir(b, ang, n, 16.0, p, sig, c, lam, L, 60, grad_restart=True)
    xp, lp = mbir.mbir(b, ang, n, 16.0, p, sig, c, lam, L, 60)
    rs = [i for i, l in enumerate(lr) if l["restarted"]]
    assert len(rs) >= 1 and all(lr[i]["accepted"] and lr[i]["dot"] > 0 for i in rs)
    assert all(lr[i + 1]["beta"] == 0.0 for i in rs if i + 1 < len(lr))            # momentum reset: next step is a plain gradient step
    assert all((l["dot"] > 0) == bool(l["restarted"]) for l in lr if l["accepted"])
    F = [l["F"] for l in lr]
    assert all(F[i + 1] <= F[i] for i in range(len(F) - 1))
    assert any(not l["accepted"] for l in lp) and all(l["accepted"] for l in lr)     # the gradient test pre-empts the rejection
    assert lr[-1]["F"] <= lp[-1]["F"]
    assert all(l["restarted"] == 0 for l in lp) and lp[0]["dot"] == lr[0]["dot"]       # flag off: same loop as before


# ---- filtered back-projection (eq. (4)), oracle/fbp.py ------------------------------------------------------
def test_fbp_reconstructs_gaussian_blob_closed_form():
    # Continuous theory: FBP(R f) = f for band-limited f.  A Gaussian blob (s = 3 px) has the closed-form sinogram of
    # oracle/analytic.py; with a detector 4x wider than the image the periodic wrap of the ramp is negligible, and what is left
    # is a constant offset of order 1/Nd (the DC bin).  A wrong scale (pi/Na, 1/Nd), sign, axis or centre convention fails this.
    from oracle import fbp, analytic
    n, nd, na = 64, 256, 180
    ang = np.arange(na) * np.pi / na
    centre = nd / 2 + 0.25
    x0, y0, s = 5.0, -7.0, 3.0
    p = analytic.gaussian_projection(x0, y0, s, ang, nd, centre)
    x = np.arange(n) - n // 2
    truth = np.exp(-((x[None, :] - x0) ** 2 + (x[:, None] - y0) ** 2) / (2 * s * s))
    f = fbp.fbp_direct(p, ang, n, centre, "ramp")
    assert rel_l2(f, truth) < 5e-3
    off = np.mean(f - truth)
    assert rel_l2(f - off, truth) < 1e-4
    fh = fbp.fbp_direct(p, ang, n, centre, "hann")              # Hann-apodised ramp: a slightly blurred blob, same place and mass
    assert rel_l2(fh, truth) < 6e-2 and abs(fh.sum() / truth.sum() - 1.0) < 2e-2
    iy, ix = np.unravel_index(np.argmax(fh), fh.shape)
    assert (ix - n // 2, iy - n // 2) == (5, -7)


def test_fbp_nufft_matches_definition_and_weights():
    from oracle import fbp, direct
    rng = np.random.default_rng(31)
    n, nd, na = 32, 48, 21
    ang = np.sort(rng.uniform(0, np.pi, na))
    y = rng.standard_normal((2, na, nd))
    for w in ("ramp", "hann"):
        assert rel_l2(fbp.fbp_nufft(y, ang, n, 23.5, w), fbp.fbp_direct(y, ang, n, 23.5, w)) < 2e-5
    rho = fbp.ramp_weights(nd, na)
    m = np.arange(-(nd // 2) + 1, nd // 2)
    assert np.allclose(rho[m != 0], np.pi / na * np.abs(m[m != 0]) / nd) and np.isclose(rho[m == 0][0], np.pi / na * 0.25 / nd)
    # all weights equal to one turn FBP back into the plain adjoint (D2)
    import unittest.mock as mock
    with mock.patch.object(fbp, "ramp_weights", lambda nd_, na_, window="ramp": np.ones(nd_ - 1)):
        assert rel_l2(fbp.fbp_direct(y, ang, n, 23.5), direct.backproject_direct(y, ang, n, 23.5)) < 1e-12


# ---- the reject / restart branch of the optimiser ("monotonic ... with restart"; G14) -------------
def _dense_case(cf):
    N, na = 8, 10
    ang = np.arange(na) * math.pi / na
    b = np.random.default_rng(10).standard_normal((1, na, N))
    An = np.stack([nufft.radon_nufft(e.reshape(N, N), ang, N, 4.0).ravel() for e in np.eye(N * N)], axis=1)
    L = cf * np.linalg.norm(An, 2) ** 2
    return An, b, ang, N, L


def test_mbir_reject_restart_branch_from_dense_matrix():
    # lambda = 0 on the brute-force 8 x 8 system with a step that is too long for the momentum (L = 0.6 ||A||^2): candidates are
    # rejected.  Everything expected below is computed from the dense matrix and the textbook momentum numbers, not from mbir.py:
    #   - a rejected step leaves the iterate bit-identical and F unchanged (monotone: "x- <- x", nothing else moves);
    #   - the step after a rejection has beta = 0 and its candidate is the plain gradient step x - A^T (A x - b)/L from the
    #     KEPT x (dropping `t = 1` fails the beta checks; dropping `xm = x` fails the second-step check, because the momentum
    #     would then extrapolate from the older iterate);
    #   - the step after that uses beta = (t1 - 1)/t2 = 0.28175..., t1 = (1 + sqrt 5)/2, on (x_{k+1}, x_k).
    An, b, ang, N, L = _dense_case(0.6)
    bv = b.ravel()
    x, log, its = mbir.mbir(b, ang, N, 4.0, P, SIG, C, 0.0, L, 12, keep_iterates=True)
    acc = [l["accepted"] for l in log]
    assert acc[:7] == [1, 1, 1, 0, 1, 1, 0]
    F = lambda v: 0.5 * np.sum((An @ v - bv) ** 2)
    step = lambda y: y - An.T @ (An @ y - bv) / L
    t1 = (1 + math.sqrt(5)) / 2; t2 = (1 + math.sqrt(1 + 4 * t1 * t1)) / 2
    beta1 = (t1 - 1) / t2
    assert abs(beta1 - 0.2817535) < 1e-6
    for k in (3, 6):
        assert np.array_equal(its[k], its[k - 1]) and log[k]["F"] == log[k - 1]["F"]            # rejected: nothing moved
        # the rejected candidate was the momentum step from (x_{k-1}, x_{k-2}) and it did increase F
        yk = its[k - 1].ravel() + log[k]["beta"] * (its[k - 1].ravel() - its[k - 2].ravel())
        assert abs(log[k]["data"] - F(step(yk))) < 1e-10 * log[k]["data"] and log[k]["data"] > log[k - 1]["F"]
        assert log[k]["margin"] < 0 and log[k]["beta"] > 0
        assert log[k + 1]["beta"] == 0.0 and log[k + 1]["accepted"] == 1                         # restart: plain gradient step from the kept x
        assert rel_l2(its[k + 1].ravel(), step(its[k].ravel())) < 1e-12
        if k + 2 < len(log):
            assert abs(log[k + 2]["beta"] - beta1) < 1e-15
            y2 = its[k + 1].ravel() + beta1 * (its[k + 1].ravel() - its[k].ravel())              # x- is the kept iterate, not an older one
            assert rel_l2(its[k + 2].ravel(), step(y2)) < 1e-12
    # the momentum sequence restarts from scratch: betas after the restart repeat the betas from the start
    assert [l["beta"] for l in log[4:6]] == [l["beta"] for l in log[0:2]]
    for k, l in enumerate(log):                                                                  # logged F is the dense objective of the kept iterate
        assert abs(l["F"] - F(its[k].ravel())) < 1e-10 * l["F"]


def test_mbir_consecutive_rejections_keep_the_iterate():
    # L = 0.45 ||A||^2: after two accepted steps even the plain gradient step increases F, so every later candidate is rejected;
    # the loop must then stand still (same iterate, same F, beta = 0, the same rejected candidate every time).
    An, b, ang, N, L = _dense_case(0.45)
    bv = b.ravel()
    x, log, its = mbir.mbir(b, ang, N, 4.0, P, SIG, C, 0.0, L, 9, keep_iterates=True)
    assert [l["accepted"] for l in log] == [1, 0, 1, 0, 0, 0, 0, 0, 0]
    cand = its[2].ravel() - An.T @ (An @ its[2].ravel() - bv) / L
    Fc = 0.5 * np.sum((An @ cand - bv) ** 2)
    for k in range(4, 9):
        assert np.array_equal(its[k], its[2]) and log[k]["F"] == log[2]["F"] and log[k]["beta"] == 0.0
        assert abs(log[k]["data"] - Fc) < 1e-10 * Fc and Fc > log[2]["F"]
    assert np.array_equal(x, its[2])


def test_lipschitz_power_iteration_vs_dense_norm():
    # lambda_hat (10 power iterations from ones, reading G15) against the spectral norm of the brute-force matrix
    An, b, ang, N, _ = _dense_case(1.0)
    Lq, lam_hat = mbir.lipschitz(N, ang, N, 4.0, P, SIG, C, 0.0)
    s2 = np.linalg.norm(An, 2) ** 2
    assert 0.97 * s2 < lam_hat <= s2 * (1 + 1e-12) and abs(Lq - 1.05 * lam_hat) < 1e-12 * Lq
    Lp, _ = mbir.lipschitz(N, ang, N, 4.0, P, SIG, C, 3.0)
    assert abs(Lp - (1.05 * lam_hat + 3.0 * 4.0 / (C * SIG * SIG))) < 1e-9 * Lp                  # curvature bound h''(0) = 2/(c sigma^2), pairs double it


def test_fbp_hann_window_read_off_a_single_radial_mode():
    # A sinogram that is one radial mode, p[a][u] = cos(2 pi m0 (u - centre)/Nd), has coefficients at m = +-m0 only, so FBP of it
    # is the plain adjoint (D2) times (pi/Na) (m0/Nd) win(m0): the filter value is read off exactly.  Hann = cos^2(pi m/Nd):
    # 1, 3/4, 1/2, 1/4 at m0 = 0, Nd/6, Nd/4, Nd/3.
    from oracle import fbp
    n, nd, na, centre = 16, 48, 7, 23.25
    ang = np.sort(np.random.default_rng(36).uniform(0, np.pi, na))
    u = np.arange(nd)
    for m0, win in ((8, 0.75), (12, 0.5), (16, 0.25), (3, math.cos(math.pi * 3 / 48) ** 2)):
        p = np.tile(np.cos(2 * np.pi * m0 * (u - centre) / nd), (na, 1))
        plain = direct.backproject_direct(p, ang, n, centre)
        ramp = fbp.fbp_direct(p, ang, n, centre, "ramp")
        hann = fbp.fbp_direct(p, ang, n, centre, "hann")
        assert rel_l2(ramp, plain * (np.pi / na) * (m0 / nd)) < 1e-12
        assert rel_l2(hann, ramp * win) < 1e-12
        assert rel_l2(fbp.fbp_nufft(p, ang, n, centre, "hann"), hann) < 2e-5
        # Shepp-Logan sin(x)/x at x = pi m0/Nd and Butterworth 1/(1 + (4 m0/Nd)^4), written out here with math, not numpy's sinc
        x = math.pi * m0 / nd
        assert rel_l2(fbp.fbp_direct(p, ang, n, centre, "shepp-logan"), ramp * (math.sin(x) / x)) < 1e-12
        assert rel_l2(fbp.fbp_direct(p, ang, n, centre, "butterworth"), ramp / (1.0 + (4.0 * m0 / nd) ** 4)) < 1e-12
    assert abs(fbp.ramp_weights(nd, na, "butterworth")[nd // 2 - 1 + 12] / fbp.ramp_weights(nd, na, "ramp")[nd // 2 - 1 + 12] - 0.5) < 1e-15   # half power at the cut-off m = Nd/4
    p0 = np.ones((na, nd))                                          # m0 = 0: DC bin, weight 1/(4 Nd), Hann = 1
    assert rel_l2(fbp.fbp_direct(p0, ang, n, centre, "hann"), direct.backproject_direct(p0, ang, n, centre) * (np.pi / na) * 0.25 / nd) < 1e-12


def test_oracle_pool_is_scheduling_only():
    # tests/oracle_pool.py (used by the full-size GPU parity tests) must return what the serial oracle returns
    from oracle_pool import OraclePool
    rng = np.random.default_rng(37); n, nd, na = 16, 24, 7
    ang = rng.uniform(0, np.pi, na)
    f = rng.standard_normal((3, n, n)); y = rng.standard_normal((3, na, nd))
    b = nufft.radon_nufft(f, ang, nd, 11.5)
    with OraclePool(ang, n, nd, 11.5, workers=2, chunks_per_slice=3) as op:
        assert rel_l2(op.A(f), b) < 1e-14
        assert rel_l2(op.At(y), nufft.backproject_nufft(y, ang, n, 11.5)) < 1e-13
        x0, log0 = mbir.mbir(b, ang, n, 11.5, P, SIG, C, 1.0, 500.0, 3)
        with op.patched(mbir):
            x1, log1 = mbir.mbir(b, ang, n, 11.5, P, SIG, C, 1.0, 500.0, 3)
        assert rel_l2(x1, x0) < 1e-12 and [l["accepted"] for l in log1] == [l["accepted"] for l in log0]
    assert mbir.nufft.radon_nufft is nufft.radon_nufft


# ---- neighbour sets; row 1: majorise-minimise step length ------------------------------------------
@pytest.mark.parametrize("nb,wsum", [(10, 6 + 4 / math.sqrt(2)), (6, 6.0)])
def test_prior_neighbour_sets_bruteforce(nb, wsum):
    # 10 = the 8 in-plane neighbours and the 2 along z (the set P:L149 quotes for SVMBIR), 6 = faces; weights 1/distance / their sum
    offs = prior.offsets(nb)
    assert len(offs) == nb and abs(sum(prior.weight(o, nb) for o in offs) - 1.0) < 1e-14
    rng = np.random.default_rng(38); f = rng.standard_normal((3, 4, 5))
    idx = [(z, y, x) for z in range(3) for y in range(4) for x in range(5)]
    tot = 0.0; grad = np.zeros_like(f)
    for a in idx:
        for b in idx:
            dz, dy, dx = (abs(a[k] - b[k]) for k in range(3))
            if max(dz, dy, dx) != 1 or not a < b:
                continue
            member = (dz == 0 or (dy == 0 and dx == 0)) if nb == 10 else (dz + dy + dx == 1)
            if not member:
                continue
            w = 1 / math.sqrt(dz + dy + dx) / wsum
            D = f[a] - f[b]; u = abs(D) / SIG; uq = u ** (2 - P)
            tot += w * u * u / (C + uq)
            d = w * math.copysign(1.0, D) / SIG * u * (2 * C + P * uq) / (C + uq) ** 2
            grad[a] += d; grad[b] -= d
    assert abs(prior.H(f, P, SIG, C, nb) - tot) < 1e-12 * tot
    assert rel_l2(prior.gradH(f, P, SIG, C, nb), grad) < 1e-12
    assert prior.H(f, P, SIG, C, 26) == prior.H(f, P, SIG, C)        # the default is untouched


def test_prior_surrogate_curvature_majorises():
    # curvH is the curvature of the symmetric-bound quadratic surrogate: Q(a) = H(f) - a <grad H(f), g> + a^2/2 curvH(f; g) >= H(f - a g)
    # for 1 < p <= 2, touching at a = 0; for the quadratic case p = 2 (h = u^2 / (c + 1)) the surrogate IS the function.
    rng = np.random.default_rng(39)
    f = rng.standard_normal((3, 5, 6)); g = rng.standard_normal((3, 5, 6))
    for nb in (26, 10):
        H0, gr, cv = prior.H(f, P, SIG, C, nb), prior.gradH(f, P, SIG, C, nb), prior.curvH(f, g, P, SIG, C, nb)
        for a in (1e-3, 0.05, 0.3, 1.0, 4.0, -0.7):
            Q = H0 - a * np.sum(gr * g) + 0.5 * a * a * cv
            assert prior.H(f - a * g, P, SIG, C, nb) <= Q * (1 + 1e-12)
        a = 1e-4                                                      # tangent at a = 0: 0 <= Q - H <= a^2/2 curvH (a wrong slope would leave O(a))
        gap = H0 - a * np.sum(gr * g) + 0.5 * a * a * cv - prior.H(f - a * g, P, SIG, C, nb)
        assert -1e-13 <= gap <= 0.5 * a * a * cv
    H0, gr, cv = prior.H(f, 2.0, 1.3, 0.5), prior.gradH(f, 2.0, 1.3, 0.5), prior.curvH(f, g, 2.0, 1.3, 0.5)
    for a in (0.3, -2.0):
        assert abs(H0 - a * np.sum(gr * g) + 0.5 * a * a * cv - prior.H(f - a * g, 2.0, 1.3, 0.5)) < 1e-12 * H0
    assert abs(prior.dh_over_D(0.0, P, SIG, C) - 2.0 / (C * SIG * SIG)) < 1e-9 / (C * SIG * SIG)


def test_mbir_mm_step_is_the_exact_line_minimiser_for_lambda0():
    # lambda = 0: the majorise-minimise step is alpha = ||g||^2 / ||A g||^2, the exact minimiser of the quadratic along -g.
    # From the brute-force matrix: the first iterate is steepest descent's x1 = alpha0 A^T b, and at every accepted step the new
    # residual is orthogonal to A g (d/d alpha = 0).
    An, b, ang, N, L = _dense_case(1.0)
    bv = b.ravel()
    x, log, its = mbir.mbir(b, ang, N, 4.0, P, SIG, C, 0.0, L, 6, keep_iterates=True, mm_step=True)
    g0 = An.T @ (-bv)
    a0 = np.sum(g0 * g0) / np.sum((An @ g0) ** 2)
    assert abs(log[0]["alpha"] - a0) < 1e-12 * a0 and rel_l2(its[0].ravel(), -a0 * g0) < 1e-12
    xk, xkm = np.zeros(N * N), np.zeros(N * N)
    for k, l in enumerate(log):
        y = xk + l["beta"] * (xk - xkm)
        g = An.T @ (An @ y - bv)
        z = y - l["alpha"] * g
        assert abs(np.dot(An @ g, An @ z - bv)) < 1e-9 * np.linalg.norm(An @ g) * np.linalg.norm(An @ z - bv)
        if l["accepted"]:
            assert rel_l2(its[k].ravel(), z) < 1e-12
            xkm, xk = xk, z
    F = [l["F"] for l in log]
    assert all(F[i + 1] <= F[i] for i in range(len(F) - 1))


def test_mbir_mm_step_decreases_the_surrogate_with_prior():
    # lambda > 0, first step (y = x = 0): F(z) <= Q(alpha*) = F(0) - ||g||^4 / (2 den) < F(0), den = ||A g||^2 + lam curvH(0; g),
    # all evaluated here from the dense matrix and the (separately pinned) prior functions
    An, b, ang, N, L = _dense_case(1.0)
    bv = b.ravel(); lam = 0.7
    x, log = mbir.mbir(b, ang, N, 4.0, P, SIG, C, lam, L, 8, mm_step=True, neighbours=10)
    g = (An.T @ (-bv)).reshape(1, N, N)
    den = np.sum((An @ g.ravel()) ** 2) + lam * prior.curvH(np.zeros((1, N, N)), g, P, SIG, C, 10)
    a = np.sum(g * g) / den
    assert abs(log[0]["alpha"] - a) < 1e-12 * a
    F0 = 0.5 * np.sum(bv * bv)
    z = -a * g
    Fz = 0.5 * np.sum((An @ z.ravel() - bv) ** 2) + lam * prior.H(z, P, SIG, C, 10)
    assert abs(log[0]["F"] - Fz) < 1e-10 * Fz and Fz <= F0 - 0.5 * np.sum(g * g) ** 2 / den + 1e-9 * F0
    F = [l["F"] for l in log]
    assert all(F[i + 1] <= F[i] for i in range(len(F) - 1)) and all(l["alpha"] > 0 for l in log)


def test_preprocess_inverts_beer_lambert_and_reorders():
    # I = I0 exp(-b) + dark  =>  the pre-pass returns b exactly; every (s, a, u) carries a distinct value, so a wrong
    # transpose cannot pass; the floor clips dead pixels at -log(floor)
    from oracle import preprocess
    na, S, nd = 5, 3, 7
    s_, a_, u_ = np.meshgrid(np.arange(S), np.arange(na), np.arange(nd), indexing="ij")
    b = 0.01 + 0.1 * s_ + 0.013 * a_ + 0.0017 * u_                            # sinogram order (S, Na, Nd)
    rng = np.random.default_rng(42)
    flat = rng.uniform(900, 1100, (S, nd)); dark = rng.uniform(5, 15, (S, nd))
    proj = (np.exp(-b) * (flat - dark)[:, None, :] + dark[:, None, :]).transpose(1, 0, 2)      # projection order (Na, S, Nd)
    assert np.allclose(preprocess.preprocess(proj, flat, dark), b, atol=1e-12)
    assert np.allclose(preprocess.preprocess(np.exp(-b).transpose(1, 0, 2)), b, atol=1e-12)
    proj[2, 1, 3] = dark[1, 3]                                                 # a dead pixel
    assert preprocess.preprocess(proj, flat, dark, floor=1e-4)[1, 2, 3] == -np.log(1e-4)


def test_prior_p1_is_smoothed_total_variation():
    # SURVEY 8(f) row 4 (plain TV): eq. (13) at p = 1 is h = u^2 / (c + u) = |u| - c + c^2 / (c + |u|): total variation up to a constant
    # for |D| >> c sigma.  Pins: the algebraic identity, and H of a step of height a across one z-plane of an N^3 cube as c -> 0:
    # the crossing pairs are N^2 faces, 4 N (N - 1) edges and 4 (N - 1)^2 corners, each |a| / sigma times its weight.
    from oracle import prior
    rng = np.random.default_rng(51)
    D = rng.standard_normal(200) * 3.0
    sig, c = 0.7, 1e-3
    u = np.abs(D) / sig
    assert np.max(np.abs(prior.h(D, 1.0, sig, c) - (u - c + c * c / (c + u)))) < 1e-14
    N, a = 6, 0.8
    f = np.zeros((N, N, N)); f[3:] = a
    w_face, w_edge, w_corn = prior.weight((1, 0, 0)), prior.weight((1, 1, 0)), prior.weight((1, 1, 1))
    tv = (a / sig) * (N * N * w_face + 4 * N * (N - 1) * w_edge + 4 * (N - 1) ** 2 * w_corn)
    assert abs(prior.H(f, 1.0, sig, 1e-12) - tv) < 1e-9 * tv
    # and the gradient is the sign pattern of TV away from zero differences: h'(D) -> sign(D) / sigma
    assert np.max(np.abs(prior.dh(D[np.abs(D) > 0.5], 1.0, sig, 1e-12) - np.sign(D[np.abs(D) > 0.5]) / sig)) < 1e-9
