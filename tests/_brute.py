"""Independent NumPy brute force for TINY inputs (pin P7).

Written with whole-array broadcasting from the definitions in DESIGN.md §2, so
it shares neither code nor loop structure with oracle/lipfit_oracle.c.  Used
only to pin the oracle; never by the CUDA path.
"""
import numpy as np


def components(X, Xq, mask, w):
    """u, l with shape [Q, N, d] (float64)."""
    X = np.asarray(X, np.float64)
    Xq = np.asarray(Xq, np.float64)
    d = X.shape[1]
    s = np.zeros(d) if mask is None else np.asarray(mask, np.float64)
    w = np.ones(d) if w is None else np.asarray(w, np.float64)
    delta = Xq[:, None, :] - X[None, :, :]
    free = (s == 0)
    u = np.where(free, np.abs(delta), np.maximum(s * delta, 0.0)) * w
    l = np.where(free, np.abs(delta), np.maximum(-s * delta, 0.0)) * w
    return u, l


def pnorm(v, norm):
    if norm == 1:
        return v.sum(axis=-1)
    if norm == 2:
        return np.sqrt((v * v).sum(axis=-1))
    return v.max(axis=-1)


def distances(X, Xq, mask, norm, w):
    u, l = components(X, Xq, mask, w)
    return pnorm(u, norm), pnorm(l, norm)        # D^u, D^l : [Q, N]


def bounds(X, y, Xq, M, mask, norm, w):
    Du, Dl = distances(X, Xq, mask, norm, w)
    y = np.asarray(y, np.float64)
    U = (y[None, :] + M * Du).min(axis=1)
    L = (y[None, :] - M * Dl).max(axis=1)
    return U, L, 0.5 * (U + L)


def knn(X, Xq, k, mask, side, norm, w):
    Du, Dl = distances(X, Xq, None if side == 0 else mask, norm, w)
    D = Dl if side < 0 else Du
    order = np.argsort(D, axis=1, kind="stable")[:, :k]      # stable: ties by lower index
    return order.astype(np.int32), np.take_along_axis(D, order, axis=1)


def smooth_F_identity(X, y, M, eps, mask, norm, w, p):
    """F via reading R12's identity ||eps||^2/p + 2 sum_{i!=k} V_ik^2 and the
    gradient 2 eps_i/p + 4 sum_k (V_ik - V_ki)."""
    Du, _ = distances(X, X, mask, norm, w)          # Du[i,k] = d_s(x^k, x^i)
    z = np.asarray(y, np.float64) + np.asarray(eps, np.float64)
    V = np.maximum(z[:, None] - z[None, :] - M * Du, 0.0)
    np.fill_diagonal(V, 0.0)
    F = (np.asarray(eps, np.float64) ** 2).sum() / p + 2.0 * (V * V).sum()
    grad = 2.0 * np.asarray(eps, np.float64) / p + 4.0 * (V.sum(axis=1) - V.sum(axis=0))
    return F, grad
