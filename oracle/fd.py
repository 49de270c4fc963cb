"""ORACLE (test infrastructure) - finite-difference helpers.

The paper uses a finite-difference reference as ground truth for its VJPs;
these helpers do the same for the oracle's own backward pass.
"""
from __future__ import annotations

import numpy as np


def central_diff_grad(f, x: np.ndarray, h: float = 1e-6, rel: bool = True) -> np.ndarray:
    """Gradient of scalar f at x by central differences; step h*(1+|x_i|) if rel."""
    x = np.asarray(x, float)
    g = np.empty_like(x)
    for i in range(x.size):
        hi = h * (1.0 + abs(x.flat[i])) if rel else h
        xp = x.copy(); xp.flat[i] += hi
        xm = x.copy(); xm.flat[i] -= hi
        g.flat[i] = (f(xp) - f(xm)) / (2.0 * hi)
    return g


def central_diff_jvp(F, x: np.ndarray, v: np.ndarray, h: float = 1e-6) -> np.ndarray:
    """Directional derivative of vector-valued F at x along v."""
    return (F(x + h * v) - F(x - h * v)) / (2.0 * h)


def nrm_rel_err(a, b, floor: float = 1e-300) -> float:
    """Norm-wise relative error ||a-b||_inf / max(||b||_inf, floor)  (reading A10)."""
    a = np.asarray(a, float).ravel(); b = np.asarray(b, float).ravel()
    if a.size == 0:
        return 0.0
    return float(np.max(np.abs(a - b)) / max(np.max(np.abs(b)), floor))
