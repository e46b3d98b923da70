"""(D1)/(D2): the plain definition of the discrete Fourier-slice Radon pair.

Oracle -- test infrastructure only (see oracle/__init__.py).  float64 throughout.

Geometry (readings G1-G4): unit pixels; x_j = j - N/2 (column),
y_i = i - N/2 (row); n(theta) = (cos, sin); t = x cos + y sin (eq. (1)
P:L43); detector bin u sits at t_u = u - centre; radial frequencies
k_m = m/Nd, |m| < Nd/2 (Nyquist bin excluded, reading G2).

  (D1) A f[a][u] = (1/Nd) sum_m e^{+2 pi i m (u-centre)/Nd}
                         sum_{i,j} f[i][j] e^{-2 pi i k_m (x_j cos + y_i sin)}
       = inverse radial DFT (eq. (6) reversed) of the 2-D Fourier
         transform of f sampled on the polar line (central-slice theorem,
         eq. (3)).
  (D2) A^T y[i][j] = sum_a sum_m e^{+2 pi i k_m (x_j cos + y_i sin)}
                         (1/Nd) sum_u y[a][u] e^{-2 pi i m (u-centre)/Nd}
       = eq. (5) P:L74 with c_j from eq. (6); exact transpose of (D1).
"""
import numpy as np


def _modes(nd):
    return np.arange(-(nd // 2) + 1, nd // 2)          # |m| < Nd/2


def radon_direct(f, angles, nd, centre):
    """(D1). f: (S, N, N) or (N, N) real; returns (S, Na, Nd) float64."""
    f = np.asarray(f, dtype=np.float64)
    squeeze = f.ndim == 2
    if squeeze:
        f = f[None]
    S, N, _ = f.shape
    m = _modes(nd)
    k = m / nd
    x = np.arange(N) - N // 2
    u = np.arange(nd)
    out = np.empty((S, len(angles), nd))
    # inverse radial DFT matrix, (Nd, M)
    P = np.exp(2j * np.pi * np.outer(u - centre, m) / nd) / nd
    for a, th in enumerate(np.asarray(angles, dtype=np.float64)):
        Ex = np.exp(-2j * np.pi * np.outer(k, x) * np.cos(th))     # (M, N_j)
        Ey = np.exp(-2j * np.pi * np.outer(k, x) * np.sin(th))     # (M, N_i)
        T = np.matmul(f, Ex.T)                                     # (S, N_i, M): sum over j
        F = np.einsum('mi,sim->sm', Ey, T)                         # sum over i
        p = F @ P.T                                                # (S, Nd)
        assert np.abs(p.imag).max() <= 1e-9 * (1.0 + np.abs(p.real).max())
        out[:, a, :] = p.real
    return out[0] if squeeze else out


def backproject_direct(y, angles, n, centre):
    """(D2). y: (S, Na, Nd) or (Na, Nd) real; returns (S, N, N) float64."""
    y = np.asarray(y, dtype=np.float64)
    squeeze = y.ndim == 2
    if squeeze:
        y = y[None]
    S, na, nd = y.shape
    m = _modes(nd)
    k = m / nd
    x = np.arange(n) - n // 2
    u = np.arange(nd)
    Q = np.exp(-2j * np.pi * np.outer(m, u - centre) / nd) / nd     # (M, Nd)
    out = np.zeros((S, n, n))
    for a, th in enumerate(np.asarray(angles, dtype=np.float64)):
        c = y[:, a, :] @ Q.T                                        # (S, M)
        Ex = np.exp(2j * np.pi * np.outer(k, x) * np.cos(th))       # (M, N_j)
        Ey = np.exp(2j * np.pi * np.outer(k, x) * np.sin(th))       # (M, N_i)
        # out[s,i,j] += sum_m Ey[m,i] c[s,m] Ex[m,j]
        out += np.einsum('smi,mj->sij', c[:, :, None] * Ey[None], Ex).real
    return out[0] if squeeze else out


def dirichlet(tau, nd):
    """D(tau) = (1/Nd) sum_{|m|<Nd/2} e^{2 pi i m tau/Nd}
             = sin(pi (Nd-1) tau/Nd) / (Nd sin(pi tau/Nd)),  D(0) = (Nd-1)/Nd."""
    tau = np.asarray(tau, dtype=np.float64)
    den = nd * np.sin(np.pi * tau / nd)
    num = np.sin(np.pi * (nd - 1) * tau / nd)
    small = np.abs(den) < 1e-12
    return np.where(small, (nd - 1) / nd, num / np.where(small, 1.0, den))


def radon_dirichlet(f, angles, nd, centre):
    """Second, independent evaluator of (D1) with no complex arithmetic:
    A f[a][u] = sum_{i,j} f[i][j] D(u - centre - x_j cos - y_i sin).  One slice."""
    f = np.asarray(f, dtype=np.float64)
    N = f.shape[0]
    x = np.arange(N) - N // 2
    out = np.empty((len(angles), nd))
    for a, th in enumerate(angles):
        t = x[None, :] * np.cos(th) + x[:, None] * np.sin(th)       # t[i][j]
        for u in range(nd):
            out[a, u] = np.sum(f * dirichlet(u - centre - t, nd))
    return out


def dense_matrix(n, angles, nd, centre):
    """A as a dense (Na*Nd, N*N) matrix built from the Dirichlet form (tiny sizes)."""
    x = np.arange(n) - n // 2
    A = np.empty((len(angles) * nd, n * n))
    for a, th in enumerate(angles):
        t = (x[None, :] * np.cos(th) + x[:, None] * np.sin(th)).ravel()
        for u in range(nd):
            A[a * nd + u] = dirichlet(u - centre - t, nd)
    return A
