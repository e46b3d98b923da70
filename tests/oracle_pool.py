"""Runs the oracle's NUFFT operators over a process pool -- scheduling only, for the full-size parity tests.

Every job calls `oracle.nufft.radon_nufft` / `backproject_nufft` as they stand on ONE slice and a contiguous chunk of the
angles.  The forward result is assembled row block by row block (each sinogram row depends on its own angle only); the
adjoint is the sum over angles, so the partial back-projections of the disjoint chunks are added in chunk order (a
float64 reassociation, ~1e-16).  Nothing of the method's arithmetic lives here.
"""
import multiprocessing as mp
import os
import numpy as np
from oracle import nufft

_RADON, _BACKPROJECT = nufft.radon_nufft, nufft.backproject_nufft      # bound at import: tests patch the module attributes


def n_workers(cap=32):
    return max(1, min(cap, os.cpu_count() or 1))


def _fwd_job(a):
    f, ang, nd, centre = a
    return _RADON(f, ang, nd, centre)


def _adj_job(a):
    y, ang, n, centre = a
    return _BACKPROJECT(y, ang, n, centre)


def _chunks(na, k):
    edges = np.linspace(0, na, min(k, na) + 1).astype(int)
    return [(int(edges[i]), int(edges[i + 1])) for i in range(len(edges) - 1) if edges[i + 1] > edges[i]]


class OraclePool:
    """A(f) and At(y) of the oracle, evaluated by `workers` processes over (slice, angle chunk) jobs."""

    def __init__(self, angles, n, nd, centre, workers=None, chunks_per_slice=None):
        self.ang = np.asarray(angles, dtype=np.float64)
        self.n, self.nd, self.centre = n, nd, centre
        self.workers = workers or n_workers()
        self.k = chunks_per_slice
        self.pool = mp.get_context("fork").Pool(self.workers) if self.workers > 1 else None

    def _k(self, S):
        if self.k:
            return self.k
        return max(1, min(len(self.ang), -(-self.workers // S)))     # about one job per worker

    def _map(self, fn, jobs):
        return self.pool.map(fn, jobs, chunksize=1) if self.pool else [fn(j) for j in jobs]

    def A(self, f):
        f = np.asarray(f, dtype=np.float64)
        S = f.shape[0]
        ch = _chunks(len(self.ang), self._k(S))
        res = self._map(_fwd_job, [(f[s], self.ang[a0:a1], self.nd, self.centre) for s in range(S) for (a0, a1) in ch])
        out = np.empty((S, len(self.ang), self.nd))
        it = iter(res)
        for s in range(S):
            for (a0, a1) in ch:
                out[s, a0:a1] = next(it)
        return out

    def At(self, y):
        y = np.asarray(y, dtype=np.float64)
        S = y.shape[0]
        ch = _chunks(len(self.ang), self._k(S))
        res = self._map(_adj_job, [(y[s, a0:a1], self.ang[a0:a1], self.n, self.centre) for s in range(S) for (a0, a1) in ch])
        out = np.zeros((S, self.n, self.n))
        it = iter(res)
        for s in range(S):
            for _ in ch:
                out[s] += next(it)
        return out

    def patched(self, module):
        """context manager: `module.nufft`'s two operators replaced by this pool (for oracle.mbir / oracle.fbp loops)."""
        import contextlib, unittest.mock as mock

        @contextlib.contextmanager
        def cm():
            with mock.patch.object(module.nufft, "radon_nufft", lambda f, angles, nd, centre: self.A(f)), \
                 mock.patch.object(module.nufft, "backproject_nufft", lambda y, angles, n, centre: self.At(y)):
                yield self
        return cm()

    def close(self):
        if self.pool:
            self.pool.close(); self.pool.join(); self.pool = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()
