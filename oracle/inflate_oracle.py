"""ORACLE (test infrastructure, NOT the product): zonotope fold of the interval
bounds, plain numpy FP64.

PAPER.md:L229 (Sec. IV-C): c_bar = 1/2 (r_lo + r_hi), R_bar = 1/2 diag(r_hi - r_lo);
eq. (25b): E_bar = [E(z_k)  R_bar] in R^{n x 2n}; L347: "a small positive
diagonal padding" is added to R_bar so that E_bar is right-invertible (value not
given in the paper -> parameter `pad`, reading R14).  E is constant and diagonal
in every paper system (L519, L528, L560), so r_dist (22) = 0 (reading R13)."""
import numpy as np


def inflate(r_lo, r_hi, pad=1e-6, E_diag=None, dense=False):
    r_lo = np.asarray(r_lo, dtype=np.float64)
    r_hi = np.asarray(r_hi, dtype=np.float64)
    c_bar = 0.5 * (r_lo + r_hi)
    R_diag = 0.5 * (r_hi - r_lo) + pad
    if not dense:
        return c_bar, R_diag
    n = r_lo.shape[-1]
    E = np.zeros(n) if E_diag is None else np.asarray(E_diag, dtype=np.float64)
    Ebar = np.zeros(r_lo.shape + (2 * n,))
    idx = np.arange(n)
    Ebar[..., idx, idx] = E
    Ebar[..., idx, n + idx] = R_diag
    return c_bar, R_diag, Ebar


def inflate_vjp(gc, gR):
    """Cotangents w.r.t. (c_bar, R_diag) -> cotangents w.r.t. (r_lo, r_hi)."""
    gc = np.asarray(gc, dtype=np.float64)
    gR = np.asarray(gR, dtype=np.float64)
    return 0.5 * gc - 0.5 * gR, 0.5 * gc + 0.5 * gR
