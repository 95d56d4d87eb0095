"""ORACLE (test infrastructure, NOT the product): the two refinements the paper builds on the
differentiable, batched path-based bound ("gradient-based refinement of the nominal point
a~ and scalable input domain partitioning"; Table II), as plain numpy loops around
oracle/pbh_oracle.py.  Shares nothing with the CUDA path.

Input-domain partitioning.  The box A = a~ + mu + [-sigma, sigma] is cut into a grid of sub-boxes,
`splits[g]` equal parts along coordinate g; every sub-box is a non-centred box about the SAME nominal
point (offset mu_p, radius sigma / splits), bounded by Thm 1 as in pbh_oracle (reading R4); the result
is the hull of the sub-box enclosures.  Sound because every a in A lies in some sub-box; never wider
than the unpartitioned enclosure because the interval extension is inclusion isotonic.

Nominal refinement by projected gradient descent (Table II).  The box is fixed (centre c, radii sigma);
the nominal point a~ moves inside the neighbourhood |a~ - c|_inf <= eps_opt and the objective is the
total width W(a~) = sum_i (r_hi_i - r_lo_i) of the enclosure of the remainder about a~ on that box
(mu = c - a~).  The paper gives neither step rule nor step size (reading R22): plain gradient steps
a~ <- proj(a~ - lr dW/da~), dW/da~ = grad_nom - grad_mu (the box does not move), the best iterate is kept.
"""
import itertools

import numpy as np

from oracle import pbh_oracle as P


def sub_boxes(rad, mu, splits):
    """Offsets and radii of the grid of sub-boxes of one tile: arrays [P, N]; sub-box order = row-major over the
    coordinates with splits > 1, first such coordinate slowest."""
    rad = np.asarray(rad, dtype=np.float64)
    mu = np.zeros_like(rad) if mu is None else np.asarray(mu, dtype=np.float64)
    splits = np.asarray(splits, dtype=np.int64)
    mus, rads = [], []
    for q in itertools.product(*[range(int(s)) for s in splits]):
        q = np.array(q, dtype=np.float64)
        rads.append(rad / splits)
        mus.append(mu + rad * (-1.0 + (2.0 * q + 1.0) / splits))
    return np.array(mus), np.array(rads)


def partition(spec, nom, rad, splits, mu=None):
    """nom, rad (, mu) [tiles, N]; splits [N] ints >= 1.  Returns r_lo, r_hi [tiles, n], status."""
    nom = np.asarray(nom, dtype=np.float64).reshape(-1, spec.N)
    rad = np.asarray(rad, dtype=np.float64).reshape(-1, spec.N)
    mu = None if mu is None else np.asarray(mu, dtype=np.float64).reshape(-1, spec.N)
    lo = np.empty((nom.shape[0], spec.n))
    hi = np.empty((nom.shape[0], spec.n))
    status = 0
    for t in range(nom.shape[0]):
        mus, rads = sub_boxes(rad[t], None if mu is None else mu[t], splits)
        l, h, st = P.pbh(spec, np.repeat(nom[t][None], mus.shape[0], 0), rads, mu=mus)
        status |= st
        lo[t], hi[t] = l.min(0), h.max(0)
    return lo, hi, status


def width_and_grad(spec, nom, centre, rad):
    """W = sum_i (r_hi - r_lo) of the enclosure about `nom` on the box centre +- rad, and dW/dnom with the box fixed."""
    mu = centre - nom
    lo, hi, st = P.pbh(spec, nom, rad, mu=mu)
    ones = np.ones_like(lo)
    g, _ = P.pbh_vjp(spec, nom, rad, -ones, ones, mu=mu)
    N = spec.N
    return (hi - lo).sum(1), g[:, :N] - g[:, 2 * N:], st


def pgd(spec, centre, rad, nom0, eps_opt, steps, lr):
    """Returns (best nominal points [tiles, N], initial widths, best widths)."""
    centre = np.asarray(centre, dtype=np.float64).reshape(-1, spec.N)
    rad = np.asarray(rad, dtype=np.float64).reshape(-1, spec.N)
    nom = np.asarray(nom0, dtype=np.float64).reshape(-1, spec.N).copy()
    best_nom, best_w, w0 = nom.copy(), None, None
    for it in range(steps + 1):
        w, g, _ = width_and_grad(spec, nom, centre, rad)
        if it == 0:
            w0, best_w = w.copy(), w.copy()
        better = w < best_w
        best_w = np.where(better, w, best_w)
        best_nom[better] = nom[better]
        if it == steps:
            break
        nom = np.clip(nom - lr * g, centre - eps_opt, centre + eps_opt)
    return best_nom, w0, best_w
