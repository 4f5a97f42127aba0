"""Lawson-Hanson active-set NNLS (the paper's "standard NNLS solver [30]"),
written independently in float64 numpy as a *test-side* check of the oracle on tiny instances (pin P1).
Restates the published algorithm (Lawson & Hanson 1974, ch. 23); not used by any product path."""
import numpy as np


def nnls_lawson_hanson(A: np.ndarray, y: np.ndarray, tol: float = 1e-12, max_outer: int = 10000):
    A = np.asarray(A, np.float64)
    y = np.asarray(y, np.float64)
    m, n = A.shape
    passive = np.zeros(n, bool)
    x = np.zeros(n)
    w = A.T @ (y - A @ x)
    outer = 0
    while (~passive).any() and w[~passive].max() > tol and outer < max_outer:
        outer += 1
        cand = np.where(~passive)[0]
        passive[cand[np.argmax(w[cand])]] = True
        while True:
            P = np.where(passive)[0]
            z = np.zeros(n)
            z[P] = np.linalg.lstsq(A[:, P], y, rcond=None)[0]
            if z[P].min() > 0:
                break
            neg = P[z[P] <= 0]
            alpha = np.min(x[neg] / (x[neg] - z[neg]))
            x = x + alpha * (z - x)
            passive &= x > tol
            x[~passive] = 0.0
        x = z
        w = A.T @ (y - A @ x)
    return x
