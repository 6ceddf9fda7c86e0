"""Shared test helpers (host-side only; no method arithmetic beyond dense linear algebra used as pins)."""
import numpy as np

import pyoracle as po


def make_oracle(w):
    return po.Oracle(w["shape"], w.get("spacing"), w.get("origin"), edges=w.get("edges"), coord=w.get("coord", 0),
                     order=w.get("order", 2), bc=w["bc"])


def dense_matrix(o, use_ghost=False):
    """Matrix of the homogeneous operator, assembled column by column from unit vectors."""
    n = o.size
    A = np.zeros((n, n))
    e = np.zeros(o.npshape)
    flat = e.reshape(-1)
    for c in range(n):
        flat[c] = 1.0
        A[:, c] = o.apply(e, use_ghost=use_ghost).reshape(-1)
        flat[c] = 0.0
    return A


def rel_l2(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))
