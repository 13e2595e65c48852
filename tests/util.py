"""Error metrics of DESIGN.md (AMB-17) and small helpers shared by the tests."""
import numpy as np


def err_f(f, f_ref):
    """max over cells and points of |df| / (max over the cell's points of |f_ref|)."""
    J, I = f_ref.shape[:2]
    a = f.reshape(J * I, -1)
    b = f_ref.reshape(J * I, -1)
    scale = np.max(np.abs(b), axis=1, keepdims=True)
    return float(np.max(np.abs(a - b) / scale))


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
