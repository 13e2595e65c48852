"""Error metrics of DESIGN.md (AMB-17) and small helpers shared by the tests."""
import numpy as np


def err_f(f, f_ref):
    """max over cells and points of |df| / (max over the cell's points of |f_ref|)."""
    J, I = f_ref.shape[:2]
    a = f.reshape(J * I, -1)
    b = f_ref.reshape(J * I, -1)
    scale = np.max(np.abs(b), axis=1, keepdims=True)
    return float(np.max(np.abs(a - b) / scale))


def err_f_and_tail(f, f_ref):
    """(err_f, tail): err_f as above, and the AMB-17 tail metric -- the largest POINTWISE relative error over the points
    with f_ref >= 1e-12 x (the cell's max f_ref).  Row by row, so that the temporaries stay small at C4 size."""
    J, I = f_ref.shape[:2]
    e = t = 0.0
    for j in range(J):
        a = f[j].reshape(I, -1)
        b = f_ref[j].reshape(I, -1)
        scale = np.max(np.abs(b), axis=1, keepdims=True)
        d = np.abs(a - b)
        e = max(e, float(np.max(d / scale)))
        m = b >= 1e-12 * scale
        if m.any():
            t = max(t, float(np.max(d[m] / b[m])))
    return e, t


def err_W(W, W_ref):
    """max |dW_alpha| / S_alpha with S = (rho, rho/sqrt(lam), rho/sqrt(lam), rhoE) of the reference cell."""
    W = W.reshape(-1, 4)
    R = W_ref.reshape(-1, 4)
    rho = R[:, 0]
    U = R[:, 1] / rho
    V = R[:, 2] / rho
    lam = rho / (2.0 * (R[:, 3] - 0.5 * rho * (U * U + V * V)))
    S = np.stack([rho, rho / np.sqrt(lam), rho / np.sqrt(lam), R[:, 3]], axis=1)
    return float(np.max(np.abs(W - R) / S))


def cons_of_prim(prim):
    rho, U, V, lam = np.moveaxis(np.asarray(prim, dtype=float), -1, 0)
    return np.stack([rho, rho * U, rho * V, 0.5 * rho * (U * U + V * V) + rho / (2 * lam)], axis=-1)
