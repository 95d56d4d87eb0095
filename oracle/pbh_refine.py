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


def sub_box_offsets(splits):
    """c_p = -1 + (2 q_p + 1) / splits: centre of part q of [-1, 1] cut into `splits` equal parts, per coordinate; [P, N],
    sub-box order = row-major over the coordinates, first coordinate slowest."""
    splits = np.asarray(splits, dtype=np.int64)
    return np.array([-1.0 + (2.0 * np.array(q, dtype=np.float64) + 1.0) / splits
                     for q in itertools.product(*[range(int(s)) for s in splits])])


def sub_boxes(rad, mu, splits):
    """Offsets and radii of the grid of sub-boxes of one tile: arrays [P, N]."""
    rad = np.asarray(rad, dtype=np.float64)
    mu = np.zeros_like(rad) if mu is None else np.asarray(mu, dtype=np.float64)
    splits = np.asarray(splits, dtype=np.int64)
    c = sub_box_offsets(splits)
    return mu[None] + rad[None] * c, np.repeat((rad / splits)[None], c.shape[0], 0)


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


def partition_vjp(spec, nom, rad, splits, g_lo, g_hi, mu=None):
    """VJP of partition(): the hull takes, per output, the lower bound of ONE sub-box (the first minimum in sub-box order)
    and the upper bound of one (the first maximum), so the cotangent of r_lo_i goes to that sub-box's lower bound only
    (reading R20: derivative of the selected branch).  The sub-box inputs are nom (shared), rad_p = rad / splits and
    mu_p = mu + rad * c_p, c_p = -1 + (2 q_p + 1) / splits, so
        d/dnom = sum_p gnom_p,   d/drad = sum_p (grad_p / splits + gmu_p * c_p),   d/dmu = sum_p gmu_p.
    Returns grad [tiles, 3N] (nom | rad | mu)."""
    nom = np.asarray(nom, dtype=np.float64).reshape(-1, spec.N)
    rad = np.asarray(rad, dtype=np.float64).reshape(-1, spec.N)
    mu = None if mu is None else np.asarray(mu, dtype=np.float64).reshape(-1, spec.N)
    g_lo = np.asarray(g_lo, dtype=np.float64).reshape(-1, spec.n)
    g_hi = np.asarray(g_hi, dtype=np.float64).reshape(-1, spec.n)
    splits = np.asarray(splits, dtype=np.int64)
    N = spec.N
    out = np.zeros((nom.shape[0], 3 * N))
    for t in range(nom.shape[0]):
        mus, rads = sub_boxes(rad[t], None if mu is None else mu[t], splits)
        P_ = mus.shape[0]
        noms = np.repeat(nom[t][None], P_, 0)
        l, h, _ = P.pbh(spec, noms, rads, mu=mus)
        sel_lo, sel_hi = l.argmin(0), h.argmax(0)            # first extremum in sub-box order
        gl, gh = np.zeros((P_, spec.n)), np.zeros((P_, spec.n))
        gl[sel_lo, np.arange(spec.n)] = g_lo[t]
        gh[sel_hi, np.arange(spec.n)] = g_hi[t]
        g, _ = P.pbh_vjp(spec, noms, rads, gl, gh, mu=mus)
        c = sub_box_offsets(splits)
        out[t, :N] = g[:, :N].sum(0)
        out[t, N:2 * N] = (g[:, N:2 * N] / splits[None] + g[:, 2 * N:] * c).sum(0)
        out[t, 2 * N:] = g[:, 2 * N:].sum(0)
    return out


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
