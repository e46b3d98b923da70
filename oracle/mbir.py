"""MBIR loop: monotone accelerated gradient with restart (eqs. (9)-(10)).

Oracle -- test infrastructure only.  The paper cites the optimiser (Giselsson & Boyd
2014) without listing its steps, so this loop is DESIGN.md reading G14/G15 and the
iterate sequence is PARITY UNPINNED against the paper (pinned by invariants only).

  F(f) = 1/2 ||A f - b||^2 + lam H(f)                    (eq. (9) with reading G9)
  grad = A^T (A f - b) + lam grad H(f)                   (eq. (10))
"""
import numpy as np
from . import nufft, prior


def lipschitz(n, angles, nd, centre, p, sigma, c, lam, iters=10):
    """L = 1.05 * lambda_hat + lam * 4/(c sigma^2); lambda_hat = ||A^T A v||/||v|| after
    `iters` power iterations on one slice from v = ones (reading G15)."""
    v = np.ones((n, n))
    lam_hat = 0.0
    for _ in range(iters):
        w = nufft.backproject_nufft(nufft.radon_nufft(v, angles, nd, centre), angles, n, centre)
        lam_hat = np.linalg.norm(w) / np.linalg.norm(v)
        v = w / np.linalg.norm(w)
    return 1.05 * lam_hat + lam * 4.0 / (c * sigma * sigma), lam_hat


def mbir(b, angles, n, centre, p, sigma, c, lam, L, iters, forced=None, keep_iterates=False, nonneg=False, grad_restart=False,
         neighbours=26, mm_step=False):
    """b: (S, Na, Nd).  Returns x (S, N, N), log (list of dicts), [iterates].
    nonneg: the candidate is projected on f >= 0 ("the choice of the constraint is not limited by the algorithm design",
    P:L24): z = max(y - g/L, 0), the proximal-gradient step for the indicator of the positive orthant (G21).
    grad_restart: the gradient restart test on top of the function-value test ("monotonic ... with restart"; DESIGN.md
    G22): an accepted candidate with <g, z - x> > 0 (the step turned against the gradient at y) resets the momentum, t <- 1.
    neighbours: neighbour set of the prior (oracle/prior.py).
    mm_step: majorise-minimise step length along -g instead of the fixed 1/L ("other optimizers"; G23): the data
    term is quadratic along the line, H is majorised by its symmetric-bound quadratic surrogate at y, and the step minimises the sum,
        alpha = <g, g> / (||A g||^2 + lam curvH(y; g)),    z = y - alpha g.
    (xm = x in the reject branch is implied by t = 1 -- the next step has beta = 0 -- and is kept for readability.)"""
    b = np.asarray(b, dtype=np.float64)
    S, na, nd = b.shape
    A = lambda f: nufft.radon_nufft(f, angles, nd, centre)
    At = lambda y: nufft.backproject_nufft(y, angles, n, centre)
    x = np.zeros((S, n, n)); xm = x.copy()
    t = 1.0
    Fx = 0.5 * np.sum(b * b)
    log, its = [], []
    for it in range(iters):
        tp = (1.0 + np.sqrt(1.0 + 4.0 * t * t)) / 2.0
        beta = (t - 1.0) / tp
        y = x + beta * (x - xm)
        Ay = A(y)
        g = At(Ay - b) + lam * prior.gradH(y, p, sigma, c, neighbours)
        alpha = 1.0 / L
        if mm_step:
            den = np.sum(A(g) ** 2) + lam * prior.curvH(y, g, p, sigma, c, neighbours)
            alpha = float(np.sum(g * g) / den) if den > 0.0 else 1.0 / L
        z = y - alpha * g
        if nonneg:
            z = np.maximum(z, 0.0)
        Az = A(z)
        data = 0.5 * np.sum((Az - b) ** 2)
        pri = prior.H(z, p, sigma, c, neighbours)
        Fz = data + lam * pri
        margin = (Fx - Fz) / Fx
        accept = Fz <= Fx
        if forced is not None and it in forced:
            accept = bool(forced[it])
        dot = float(np.sum(g * (z - x)))
        restarted = bool(grad_restart and accept and dot > 0.0)
        if accept:
            xm, x = x, z
            Fx = Fz
            t = 1.0 if restarted else tp
        else:
            xm = x
            t = 1.0
        log.append(dict(F=Fx, data=data, prior=pri, margin=margin, beta=beta, accepted=int(accept), restarted=int(restarted), dot=dot, alpha=alpha))
        if keep_iterates:
            its.append(x.copy())
    return (x, log, its) if keep_iterates else (x, log)
