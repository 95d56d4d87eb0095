"""ORACLE (test infrastructure, NOT the product): disturbance-error enclosure (22), tube propagation
(27)-(28) and the propagated-error penalty J_err (35), plain numpy FP64, the definitions written out
with dense matrices.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import
this file; it shares nothing with the CUDA path.

Notation (Sec. IV-C, V): horizon T, tiles j = 0..T-1 carry the disturbance zonotopes
D_j = (c_bar_j, E_bar_j), E_bar_j = [E  R_bar_j] in R^{n x 2n} (25b) L277; the closed-loop responses
Phi_{k,j} = [Phi^x_{k,j}; Phi^u_{k,j}] in R^{N x n}, N = n + m, exist for 0 <= j < k <= T
(Phi^x_{j+1,j} = I, (34c) L340) and are stored packed: block p(k, j) = (k - 1) k / 2 + j of
Phi[T (T + 1) / 2, N, n].

  (22) L226   r_dist = (E(x) - E_k) w in ([E](Omega^x) (-) E_k) E_nx, E_nx the unit box
  (27) L289   h_mu_k    = sum_{j<k} Phi_{k,j} c_bar_j
  (28) L291   h_sigma_k = sum_{j<k} || Phi_{k,j} E_bar_j ||_{1,r}        (row-wise 1-norm)
  (35) L360   J_err     = sum_j sum_k || Phi_{k,j} Z_r(z_j, v_j, mu_j, sigma_j) ||_F^2
Readings: Z_r of (24d) is the generator matrix E_bar_j of (25b) (R21a); the sum over k in
(35) is printed from k = j although Phi_{j,j} does not exist in (26)-(28): k runs over j+1..T (R21b).

Pins (tests/test_oracle_tube.py): (28) against the support function of the Minkowski sum in (26) by
vertex enumeration; (27) against a direct propagation; (22) against corner enumeration; (35) against a
closed form for identity responses and its gradient against central differences.
"""
import numpy as np


def block(k, j):
    """packed index of Phi_{k,j}, 0 <= j < k"""
    return (k - 1) * k // 2 + j


def dist_bound(E_lo, E_hi, E_nom):
    """(22): E_lo <= E(x) <= E_hi elementwise over the state tube, E_nom = E_k: rows of
    ([E] (-) E_k) E_nw.  Arrays [..., n, nw] -> (r_lo, r_hi) [..., n]."""
    D_lo = np.asarray(E_lo, dtype=np.float64) - np.asarray(E_nom, dtype=np.float64)
    D_hi = np.asarray(E_hi, dtype=np.float64) - np.asarray(E_nom, dtype=np.float64)
    mag = np.maximum(np.abs(D_lo), np.abs(D_hi))        # sup |d| over [D_lo, D_hi]
    hi = mag.sum(-1)                                    # sup over w in the unit box of sum_j d_j w_j
    return -hi, hi


def ebar(E_diag, R_diag):
    """dense E_bar = [diag(E)  diag(R_bar)]  (25b)"""
    n = R_diag.shape[-1]
    out = np.zeros((n, 2 * n))
    out[np.arange(n), np.arange(n)] = E_diag
    out[np.arange(n), n + np.arange(n)] = R_diag
    return out


def tube_propagate(Phi, c_bar, R_diag, E_diag):
    """One trajectory.  Phi [T(T+1)/2, N, n]; c_bar, R_diag [T, n]; E_diag [n].
    Returns h_mu, h_sigma [T, N]: row k-1 holds the tube centre offset / width at time k = 1..T."""
    Phi = np.asarray(Phi, dtype=np.float64)
    T, n = c_bar.shape
    N = Phi.shape[1]
    h_mu = np.zeros((T, N))
    h_sigma = np.zeros((T, N))
    for k in range(1, T + 1):
        for j in range(k):
            P = Phi[block(k, j)]
            h_mu[k - 1] += P @ c_bar[j]
            h_sigma[k - 1] += np.abs(P @ ebar(E_diag, R_diag[j])).sum(1)
    return h_mu, h_sigma


def j_err(Phi, R_diag, E_diag):
    """(35) for one trajectory: sum_j sum_{k>j} || Phi_{k,j} E_bar_j ||_F^2."""
    Phi = np.asarray(Phi, dtype=np.float64)
    T = R_diag.shape[0]
    total = 0.0
    for j in range(T):
        Eb = ebar(E_diag, R_diag[j])
        for k in range(j + 1, T + 1):
            total += ((Phi[block(k, j)] @ Eb) ** 2).sum()
    return total


def j_err_grad(Phi, R_diag, E_diag):
    """d J_err / d R_diag [T, n]: plain chain rule of the definition above, column by column
    (d/dR_{j,c} of || Phi_{k,j} E_bar_j ||_F^2 = 2 R_{j,c} sum_i Phi_{k,j}[i, c]^2)."""
    Phi = np.asarray(Phi, dtype=np.float64)
    T, n = R_diag.shape
    g = np.zeros((T, n))
    for j in range(T):
        for k in range(j + 1, T + 1):
            g[j] += 2.0 * R_diag[j] * (Phi[block(k, j)] ** 2).sum(0)
    return g
