"""Beer-Lambert pre-pass and projection -> sinogram reorder ("b = -log(I / I0)"; data kept in sinogram order).

Oracle -- test infrastructure only (float64 numpy).
  sinogram[s][a][u] = -log(max((proj[a][s][u] - dark[s][u]) / (flat[s][u] - dark[s][u]), floor))
proj is in projection order (angles, slices, bins) as a detector delivers it; flat (I0) and dark are (slices, bins), default 1 and 0.
"""
import numpy as np


def preprocess(proj, flat=None, dark=None, floor=1e-6):
    proj = np.asarray(proj, dtype=np.float64)
    na, S, nd = proj.shape
    fl = np.ones((S, nd)) if flat is None else np.asarray(flat, dtype=np.float64)
    dk = np.zeros((S, nd)) if dark is None else np.asarray(dark, dtype=np.float64)
    out = np.empty((S, na, nd))
    for a in range(na):
        for s in range(S):
            out[s, a, :] = -np.log(np.maximum((proj[a, s, :] - dk[s]) / (fl[s] - dk[s]), floor))
    return out
