"""Projected-gradient reconstruction on the fp64 CPU oracle — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/ and bench.py's reference legs may import this.  It follows SURVEY 8(f)-1 literally (the paper names
iterative reconstruction with the pair as its purpose, without giving an algorithm):

    p_{k+1} = max(0, p_k - s H^T (H p_k - d)),   s = 1 / ||H||^2,
    ||H||^2 from power iterations on H^T H:  v <- H^T H v / ||H^T H v||,  sigma^2 = ||H^T H v|| at ||v|| = 1.

Plain numpy on top of oracle.Oracle.forward / adjoint; nothing is shared with the CUDA path.
"""
from __future__ import annotations

import numpy as np


def power_iteration(o, v0, iters=8):
    """(sigma^2 estimate, normalised iterate) after `iters` applications of H^T H, started from v0."""
    v = np.asarray(v0, dtype=np.float64).copy()
    v /= np.linalg.norm(v)
    s2 = 0.0
    for _ in range(iters):
        w = o.adjoint(o.forward(v))
        s2 = float(np.linalg.norm(w))
        v = w / s2
    return s2, v


def pgd(o, p0, d, step, iters, nonneg=True):
    """Iterates p_1 .. p_iters (list), residual norms ||H p_k - d|| and update norms ||p_{k+1} - p_k||."""
    p = np.asarray(p0, dtype=np.float64).copy()
    d = np.asarray(d, dtype=np.float64)
    its, res, upd = [], [], []
    for _ in range(iters):
        r = o.forward(p) - d
        res.append(float(np.linalg.norm(r)))
        g = o.adjoint(r)
        q = p - step * g
        if nonneg:
            q = np.maximum(q, 0.0)
        upd.append(float(np.linalg.norm(q - p)))
        p = q
        its.append(p.copy())
    return its, res, upd
