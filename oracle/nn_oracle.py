"""ORACLE (test infrastructure, NOT the product): CROWN linearization-error bounds
for MLP dynamics, plain numpy FP64, one (trajectory, timestep) tile at a time.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline /
`--impl reference` leg may import this file.  It shares no code with the CUDA
path (`paper_2607_01203_b200/`) and imports nothing from it.

What it follows, step by step and in the paper's notation:
  * Thm 2 (CROWN affine bounds, eq. (18)): for every hidden
    layer s and for the output, back-substitute the rows of W_s through the
    per-neuron linear relaxations of the earlier activations down to the input.
  * Thm 3 (eq. (19)-(21)): r_up(a) = (W_up - J) a + J a~ - p(a~)
    + b_up, maximised over the box in closed form; likewise lower.
The network is g(a) = W_L phi(... phi(W_1 a + b_1) ...) + b_L and the dynamics are
f(x,u) = x + g(x,u); the residual `x` term is linear so r[f] = r[g] exactly
(reading R10) and it is not represented here.

Readings of points the paper leaves open:
full CROWN for every hidden layer; ReLU lower slope 1 if u > -l else 0; tanh
tangent at the midpoint on single-signed intervals, chord-or-tangent on mixed
ones with the tangent point from bisection; J uses phi'(0) = 0 for ReLU.

Pins (tests/test_oracle_nn.py): zero bound for stable-ReLU / zero radius, exact
piecewise-linear enumeration for 1-hidden-layer ReLU nets, soundness against
samples and vertices, hidden-bound soundness, closed-form concretisation, and
central finite differences for the VJP.
"""
from __future__ import annotations

import numpy as np

ACT_RELU = 1
ACT_TANH = 2

TANH_D2_MAX = 4.0 / (3.0 * np.sqrt(3.0))   # max |tanh''|
DEGENERATE_EPS = 1e-12
BISECT_ITERS = 200


# --------------------------------------------------------------------------
# activations
# --------------------------------------------------------------------------
def phi(act, z):
    return np.maximum(z, 0.0) if act == ACT_RELU else np.tanh(z)


def dphi(act, z):
    if act == ACT_RELU:
        return (z > 0.0).astype(np.float64)          # phi'(0) = 0 (reading R12)
    t = np.tanh(z)
    return 1.0 - t * t


def dphi_at(act, z):
    """phi' at a bound endpoint (interval propagation differentiates phi(l), phi(u)); ReLU: 1[z > 0] as in dphi."""
    return dphi(act, z)


def d2phi(act, z):
    if act == ACT_RELU:
        return np.zeros_like(z)
    t = np.tanh(z)
    return -2.0 * t * (1.0 - t * t)


# --------------------------------------------------------------------------
# per-neuron linear relaxations  kL z + bL <= phi(z) <= kU z + bU  on [l, u]
# Each returns (kU, bU, kL, bL, aux) where aux carries what the VJP needs.
# --------------------------------------------------------------------------
def relax_relu_scalar(l, u):
    if u <= 0.0:
        return 0.0, 0.0, 0.0, 0.0, ("off",)
    if l >= 0.0:
        return 1.0, 0.0, 1.0, 0.0, ("on",)
    kU = u / (u - l)
    bU = -u * l / (u - l)
    kL = 1.0 if u > -l else 0.0                       # tie u == -l -> 0
    return kU, bU, kL, 0.0, ("unstable",)


def _t(x):
    return np.tanh(x)


def _tp(x):
    t = np.tanh(x)
    return 1.0 - t * t


def _tpp(x):
    t = np.tanh(x)
    return -2.0 * t * (1.0 - t * t)


def _tangent(d):
    k = _tp(d)
    return k, _t(d) - k * d


def _chord(l, u):
    k = (_t(u) - _t(l)) / (u - l)
    return k, _t(l) - k * l


def _bisect_upper(l, u):
    """d in (0,u) with t(d) - t(l) = t'(d)(d - l); returns the outer bracket end
    (d >= d*), which is the sound side."""
    lo, hi = 0.0, u
    for _ in range(BISECT_ITERS):
        mid = 0.5 * (lo + hi)
        if _tp(mid) * (mid - l) - (_t(mid) - _t(l)) > 0.0:
            lo = mid
        else:
            hi = mid
    return hi


def _bisect_lower(l, u):
    """d in (l,0) with t(u) - t(d) = t'(d)(u - d); returns the outer end (d <= d*)."""
    lo, hi = l, 0.0
    for _ in range(BISECT_ITERS):
        mid = 0.5 * (lo + hi)
        if _tp(mid) * (u - mid) - (_t(u) - _t(mid)) > 0.0:
            hi = mid
        else:
            lo = mid
    return lo


def relax_tanh_scalar(l, u):
    if u - l < DEGENERATE_EPS:
        d = 0.5 * (l + u)
        k, b = _tangent(d)
        w = 0.5 * TANH_D2_MAX * (u - l) ** 2
        return k, b + w, k, b - w, ("degenerate", d)
    if l >= 0.0:                      # concave: upper tangent at midpoint, lower chord
        d = 0.5 * (l + u)
        kU, bU = _tangent(d)
        kL, bL = _chord(l, u)
        return kU, bU, kL, bL, ("pos", d)
    if u <= 0.0:                      # convex: lower tangent at midpoint, upper chord
        d = 0.5 * (l + u)
        kL, bL = _tangent(d)
        kU, bU = _chord(l, u)
        return kU, bU, kL, bL, ("neg", d)
    kc, bc = _chord(l, u)
    if kc <= _tp(u):
        kU, bU, dU = kc, bc, None
    else:
        dU = _bisect_upper(l, u)
        kU, bU = _tangent(dU)
    if kc <= _tp(l):
        kL, bL, dL = kc, bc, None
    else:
        dL = _bisect_lower(l, u)
        kL, bL = _tangent(dL)
    return kU, bU, kL, bL, ("mixed", dU, dL)


def relax(act, l, u, alpha=None):
    """Vector version: arrays kU, bU, kL, bL and the per-neuron aux list.
    alpha (ReLU only): lower slopes of the unstable neurons (l < 0 < u), any value in [0, 1] is a valid lower bound
    alpha z <= relu(z); None = the adaptive choice of reading R8.  Stable neurons ignore it."""
    f = relax_relu_scalar if act == ACT_RELU else relax_tanh_scalar
    out = [f(float(a), float(b)) for a, b in zip(l, u)]
    kU = np.array([o[0] for o in out])
    bU = np.array([o[1] for o in out])
    kL = np.array([o[2] for o in out])
    bL = np.array([o[3] for o in out])
    if alpha is not None:
        assert act == ACT_RELU
        unstable = np.array([o[4][0] == "unstable" for o in out])
        kL = np.where(unstable, alpha, kL)
    return kU, bU, kL, bL, [o[4] for o in out]


# --------------------------------------------------------------------------
# nominal pass
# --------------------------------------------------------------------------
def nominal(Ws, bs, act, a0):
    """zhat_l (l=1..L-1), p(a~), and J(a~) = W_L diag(phi'(zhat_{L-1})) ... W_1."""
    L = len(Ws)
    zs = []
    a = a0
    for l in range(L - 1):
        z = Ws[l] @ a + bs[l]
        zs.append(z)
        a = phi(act, z)
    p = Ws[L - 1] @ a + bs[L - 1]
    J = Ws[L - 1]
    for l in range(L - 2, -1, -1):
        J = (J * dphi(act, zs[l])[None, :]) @ Ws[l]
    return zs, p, J


def mlp_eval(Ws, bs, act, a0):
    a = a0
    for l in range(len(Ws) - 1):
        a = phi(act, Ws[l] @ a + bs[l])
    return Ws[-1] @ a + bs[-1]


def mlp_hidden(Ws, bs, act, a0):
    """Pre-activations z_1..z_{L-1} at the point a0 (hidden-bound soundness tests)."""
    zs = []
    a = a0
    for l in range(len(Ws) - 1):
        z = Ws[l] @ a + bs[l]
        zs.append(z)
        a = phi(act, z)
    return zs


# --------------------------------------------------------------------------
# back-substitution of target s (1-based; s = L is the output) -- eq. (18)
# --------------------------------------------------------------------------
def backsub(Ws, bs, relaxs, s, keep=False):
    """Rows of W_s pushed through layers s-1 .. 1.

    relaxs[l-1] = (kU, bU, kL, bL) of hidden layer l.  Returns
    (Lam_up, c_up, Lam_lo, c_lo) with z_s <= Lam_up a + c_up, z_s >= Lam_lo a + c_lo
    on the box, and (if keep) the per-layer Lambda_l of both chains,
    Lams_up[l] = coefficient on activation a_l (l = s-1 .. 0)."""
    Lu = Ws[s - 1].copy()
    Ll = Ws[s - 1].copy()
    cu = bs[s - 1].copy()
    cl = bs[s - 1].copy()
    Lams_up = {s - 1: Lu}
    Lams_lo = {s - 1: Ll}
    for l in range(s - 1, 0, -1):
        kU, bU, kL, bL = relaxs[l - 1][:4]
        W, b = Ws[l - 1], bs[l - 1]
        # upper chain: positive coefficients take the upper relaxation
        P, Q = np.maximum(Lu, 0.0), np.minimum(Lu, 0.0)
        D = P * kU[None, :] + Q * kL[None, :]
        cu = cu + P @ bU + Q @ bL + D @ b
        Lu = D @ W
        # lower chain: positive coefficients take the lower relaxation
        P, Q = np.maximum(Ll, 0.0), np.minimum(Ll, 0.0)
        D = P * kL[None, :] + Q * kU[None, :]
        cl = cl + P @ bL + Q @ bU + D @ b
        Ll = D @ W
        Lams_up[l - 1] = Lu
        Lams_lo[l - 1] = Ll
    if keep:
        return Lu, cu, Ll, cl, Lams_up, Lams_lo
    return Lu, cu, Ll, cl


def ibp_layer(W, b, act, l_prev, u_prev):
    """Interval propagation of one layer: z = W phi(z_prev) + b with z_prev in [l_prev, u_prev]; phi is monotone, so
    phi(z_prev) in [phi(l_prev), phi(u_prev)] and the interval matrix-vector product is W+ lo + W- hi (lower end)."""
    a_lo, a_hi = phi(act, l_prev), phi(act, u_prev)
    Wp, Wn = np.maximum(W, 0.0), np.minimum(W, 0.0)
    return Wp @ a_lo + Wn @ a_hi + b, Wp @ a_hi + Wn @ a_lo + b


def crown_forward(Ws, bs, act, a0, sig, J_given=None, keep=False, hidden="crown", mu=None, alphas=None):
    """CROWN + Thm 3 for one tile.  Returns dict with r_lo, r_hi, the hidden
    bounds (ls, us), the output affine bounds (W_up, b_up, W_lo, b_lo), J and p.

    hidden = "crown": every hidden layer's pre-activation bounds by back-substitution to the input (full CROWN,
    reading R11).  hidden = "ibp": hidden layers 2..L-1 by interval propagation of the previous layer's bounds
    (CROWN-IBP: cheaper, looser intermediate bounds; the output is still back-substituted, Thm 2 holds for any valid
    intermediate bounds).  PAPER.md:L194-196 leaves the CROWN variant open.

    mu: non-centred box (25a) PAPER.md:L272: the CROWN bounds are taken on the box c + [-sig, sig], c = a0 + mu, while
    p(a~) and J(a~) of the remainder (10) stay at the nominal point a0; Thm 3's maximisation (21) of the affine r_up(a)
    = (W_up - J) a + J a~ - p(a~) + b_up (20) then runs over that box.  (Thm 2 / Thm 3 need no a~ in the box.)

    alphas (ReLU): per hidden layer, the lower slopes of the unstable neurons (see relax); the optimisable-slope variant
    of CROWN ("alpha-CROWN"): one slope set per tile, shared by every bound of the tile."""
    al = (lambda k: None) if alphas is None else (lambda k: alphas[k])
    L = len(Ws)
    zs, p, J = nominal(Ws, bs, act, a0)
    if J_given is not None:
        J = J_given
    c = a0 if mu is None else a0 + mu
    ls, us, relaxs = [], [], []
    kept = {}
    # layer 1: interval affine
    A1 = np.abs(Ws[0]) @ sig
    z1c = zs[0] if mu is None else Ws[0] @ c + bs[0]
    ls.append(z1c - A1)
    us.append(z1c + A1)
    relaxs.append(relax(act, ls[0], us[0], al(0)))
    # hidden layers s = 2..L-1: full CROWN back-substitution to the input
    for s in range(2, L):
        if hidden == "ibp":
            lo_s, hi_s = ibp_layer(Ws[s - 1], bs[s - 1], act, ls[-1], us[-1])
            ls.append(lo_s)
            us.append(hi_s)
            relaxs.append(relax(act, ls[-1], us[-1], al(len(ls) - 1)))
            continue
        res = backsub(Ws, bs, relaxs, s, keep=keep)
        Lu, cu, Ll, cl = res[:4]
        us.append(Lu @ c + np.abs(Lu) @ sig + cu)
        ls.append(Ll @ c - np.abs(Ll) @ sig + cl)
        relaxs.append(relax(act, ls[-1], us[-1], al(len(ls) - 1)))
        if keep:
            kept[s] = res[4:]
    res = backsub(Ws, bs, relaxs, L, keep=keep)
    W_up, b_up, W_lo, b_lo = res[:4]
    if keep:
        kept[L] = res[4:]
    # Thm 3, eq. (20)-(21): box maximum of (W - J) a + J a~ - p(a~) + b over c + [-sig, sig] (c = a0: J a~ cancels)
    if mu is None:
        r_hi = np.abs(W_up - J) @ sig + (W_up @ a0 + b_up - p)
        r_lo = -np.abs(W_lo - J) @ sig + (W_lo @ a0 + b_lo - p)
    else:
        r_hi = np.abs(W_up - J) @ sig + (W_up - J) @ c + J @ a0 - p + b_up
        r_lo = -np.abs(W_lo - J) @ sig + (W_lo - J) @ c + J @ a0 - p + b_lo
    return dict(r_lo=r_lo, r_hi=r_hi, ls=ls, us=us, relaxs=relaxs, zs=zs, p=p, J=J,
                W_up=W_up, b_up=b_up, W_lo=W_lo, b_lo=b_lo, kept=kept)


def leb_nn(Ws, bs, act, nom, rad, J=None, hidden="crown", mu=None):
    """Batch driver: nom, rad [tiles, N] -> r_lo, r_hi [tiles, n] (FP64)."""
    Ws = [np.asarray(W, dtype=np.float64) for W in Ws]
    bs = [np.asarray(b, dtype=np.float64) for b in bs]
    nom = np.asarray(nom, dtype=np.float64)
    rad = np.asarray(rad, dtype=np.float64)
    n = Ws[-1].shape[0]
    r_lo = np.empty((nom.shape[0], n))
    r_hi = np.empty((nom.shape[0], n))
    for i in range(nom.shape[0]):
        out = crown_forward(Ws, bs, act, nom[i], rad[i], None if J is None else np.asarray(J[i], dtype=np.float64), hidden=hidden,
                            mu=None if mu is None else np.asarray(mu[i], dtype=np.float64))
        r_lo[i], r_hi[i] = out["r_lo"], out["r_hi"]
    return r_lo, r_hi


# --------------------------------------------------------------------------
# VJP: plain hand-written reverse sweep of the algorithm above (DESIGN.md
# "VJP definition"): grad of  sum_i g_hi[i] r_hi[i] + g_lo[i] r_lo[i]  with
# respect to the nominal point a~ and the radii sigma.  min/max/abs/ReLU-switch
# select a branch; the derivative follows the selected branch.
# --------------------------------------------------------------------------
def relax_vjp_scalar(act, l, u, aux, kUb, bUb, kLb, bLb):
    """Adjoint of one neuron's relaxation: returns (l_bar, u_bar)."""
    if act == ACT_RELU:
        if aux[0] != "unstable":
            return 0.0, 0.0
        w = u - l
        # kU = u/(u-l), bU = -u l/(u-l); kL piecewise constant, bL = 0
        dkU_du, dkU_dl = -l / w ** 2, u / w ** 2
        dbU_du, dbU_dl = l * l / w ** 2, -u * u / w ** 2
        return kUb * dkU_dl + bUb * dbU_dl, kUb * dkU_du + bUb * dbU_du
    kind = aux[0]

    def tangent_adj(d, kb, bb):          # adjoint of d for a tangent at d
        return _tpp(d) * kb - _tpp(d) * d * bb

    def chord_adj(kb, bb):               # returns (l_bar, u_bar) for chord params
        w = u - l
        kc = (_t(u) - _t(l)) / w
        dk_du = (_tp(u) - kc) / w
        dk_dl = (kc - _tp(l)) / w
        db_dl = _tp(l) - kc - l * dk_dl
        db_du = -l * dk_du
        return kb * dk_dl + bb * db_dl, kb * dk_du + bb * db_du

    if kind == "degenerate":
        d = aux[1]
        w = u - l
        db = tangent_adj(d, kUb + kLb, bUb + bLb)
        # widening term +-0.5*TANH_D2_MAX*(u-l)^2 on the intercepts
        dw = TANH_D2_MAX * w * (bUb - bLb)
        return 0.5 * db - dw, 0.5 * db + dw
    if kind == "pos":
        d = aux[1]
        db = tangent_adj(d, kUb, bUb)
        cl, cu = chord_adj(kLb, bLb)
        return 0.5 * db + cl, 0.5 * db + cu
    if kind == "neg":
        d = aux[1]
        db = tangent_adj(d, kLb, bLb)
        cl, cu = chord_adj(kUb, bUb)
        return 0.5 * db + cl, 0.5 * db + cu
    # mixed
    dU, dL = aux[1], aux[2]
    lb = ub = 0.0
    if dU is None:
        cl, cu = chord_adj(kUb, bUb)
        lb += cl
        ub += cu
    else:
        # implicit: t'(d)(d-l) - t(d) + t(l) = 0  ->  dd/dl
        dd_dl = (_tp(dU) - _tp(l)) / (_tpp(dU) * (dU - l))
        lb += tangent_adj(dU, kUb, bUb) * dd_dl
    if dL is None:
        cl, cu = chord_adj(kLb, bLb)
        lb += cl
        ub += cu
    else:
        # implicit: t'(d)(u-d) - t(u) + t(d) = 0  ->  dd/du
        dd_du = (_tp(u) - _tp(dL)) / (_tpp(dL) * (u - dL))
        ub += tangent_adj(dL, kLb, bLb) * dd_du
    return lb, ub


def relax_vjp(act, l, u, auxs, kUb, bUb, kLb, bLb):
    lb = np.zeros_like(l)
    ub = np.zeros_like(u)
    for i in range(l.shape[0]):
        lb[i], ub[i] = relax_vjp_scalar(act, float(l[i]), float(u[i]), auxs[i],
                                        float(kUb[i]), float(bUb[i]), float(kLb[i]), float(bLb[i]))
    return lb, ub


def _chain_reverse(Ws, bs, relaxs, s, Lams, Lbar0, cbar, upper, padj):
    """Reverse of one back-substitution chain of target s.
    Lams[l] = forward coefficient on a_l; padj[l-1] = [kUb, bUb, kLb, bLb] accumulators."""
    Lbar = Lbar0
    for l in range(1, s):
        kU, bU, kL, bL = relaxs[l - 1][:4]
        Lam = Lams[l]
        P, Q = np.maximum(Lam, 0.0), np.minimum(Lam, 0.0)
        pos, neg = (Lam > 0.0), (Lam < 0.0)
        Dbar = Lbar @ Ws[l - 1].T + np.outer(cbar, bs[l - 1])
        acc = padj[l - 1]
        if upper:    # positive coefficients used (kU, bU); negative (kL, bL)
            acc[0] += (Dbar * P).sum(0)
            acc[2] += (Dbar * Q).sum(0)
            acc[1] += P.T @ cbar
            acc[3] += Q.T @ cbar
            Lbar = Dbar * (kU[None, :] * pos + kL[None, :] * neg) + \
                cbar[:, None] * (bU[None, :] * pos + bL[None, :] * neg)
        else:        # positive coefficients used (kL, bL); negative (kU, bU)
            acc[2] += (Dbar * P).sum(0)
            acc[0] += (Dbar * Q).sum(0)
            acc[3] += P.T @ cbar
            acc[1] += Q.T @ cbar
            Lbar = Dbar * (kL[None, :] * pos + kU[None, :] * neg) + \
                cbar[:, None] * (bL[None, :] * pos + bU[None, :] * neg)
    # adjoint of Lambda_{s-1} = W_s is dropped (weights are not differentiated)


def output_sign_ties(Ws, bs, act, a0, sig, rel=1e-6):
    """Entries (chain, i, j) of W_up - J / W_lo - J whose magnitude is below rel * max|W|: the
    |.| of eq. (21) L220 sits on its kink there, so the branch (reading R20) cannot be
    resolved in FP32 and both one-sided gradients are valid results.  Test plumbing only."""
    fw = crown_forward(Ws, bs, act, a0, sig)
    ties = []
    for chain, Wm in (("up", fw["W_up"]), ("lo", fw["W_lo"])):
        D = Wm - fw["J"]
        thr = rel * max(np.abs(Wm).max(), 1e-300)
        for i, j in zip(*np.nonzero(np.abs(D) < thr)):
            if sig[j] > 0:
                ties.append((chain, int(i), int(j)))
    return ties


def relax_case_ties(Ws, bs, act, a0, sig, rel=2e-5, mu=None):
    """Hidden neurons (layer, k) whose pre-activation bound sits on a case switch of the relaxation
    table (readings R8/R9/R21): an endpoint l or u within rel * (|l| + |u|) of 0, or (ReLU)
    |u + l| that close to the u > -l switch.  The relaxation -- and with it the bound -- is
    discontinuous there, so an FP32 evaluation may legitimately take the other case.  Test
    plumbing only: calls crown_forward, changes no arithmetic."""
    fw = crown_forward(Ws, bs, act, a0, sig, mu=mu)
    ties = []
    for layer, (l, u) in enumerate(zip(fw["ls"], fw["us"]), start=1):
        scale = rel * (np.abs(l) + np.abs(u))
        near = (np.abs(l) < scale) | (np.abs(u) < scale)
        if act == ACT_RELU:
            near |= (l < 0) & (u > 0) & (np.abs(u + l) < scale)
        ties += [(layer, int(k)) for k in np.nonzero(near)[0]]
    return ties


def crown_vjp(Ws, bs, act, a0, sig, g_lo, g_hi, flips=(), hidden="crown", mu=None, alphas=None, slope_grads=None):
    """Returns (grad_nom, grad_rad) -- with mu: (grad_nom, grad_rad, grad_mu) -- for one tile; J is the network's own
    Jacobian at a~ (the product's leb_vjp takes no J argument).  `flips`: entries (chain, i, j) from
    output_sign_ties() whose sign(W - J) is negated (the other one-sided gradient at that kink).
    Every bound depends on the box centre c = a~ + mu (adjoint a_bar below, shared by a~ and mu); p(a~), J(a~) and the
    explicit terms J a~ - J c = -J mu depend on a~ and mu separately."""
    L = len(Ws)
    fw = crown_forward(Ws, bs, act, a0, sig, None, keep=True, hidden=hidden, mu=mu, alphas=alphas)
    relaxs, ls, us, zs, J = fw["relaxs"], fw["ls"], fw["us"], fw["zs"], fw["J"]
    a0 = a0 if mu is None else a0 + mu          # the box centre c: what the bounds below see
    a_bar = np.zeros_like(a0)
    s_bar = np.zeros_like(sig)
    padj = [[np.zeros(Ws[l].shape[0]) for _ in range(4)] for l in range(L - 1)]

    # ---- output target: Thm 3 concretisation
    Lams_up, Lams_lo = fw["kept"][L]
    Lu0, Ll0 = Lams_up[0], Lams_lo[0]
    Su, Sl = np.sign(Lu0 - J), np.sign(Ll0 - J)
    for chain, i, j in flips:
        (Su if chain == "up" else Sl)[i, j] *= -1.0
    a_bar += Lu0.T @ g_hi + Ll0.T @ g_lo
    s_bar += np.abs(Lu0 - J).T @ g_hi - np.abs(Ll0 - J).T @ g_lo
    Lbar_up = g_hi[:, None] * (Su * sig[None, :] + a0[None, :])
    Lbar_lo = g_lo[:, None] * (-Sl * sig[None, :] + a0[None, :])
    Jbar = -g_hi[:, None] * Su * sig[None, :] + g_lo[:, None] * Sl * sig[None, :]
    if mu is not None:
        Jbar = Jbar - np.outer(g_hi + g_lo, mu)          # the explicit -J mu of (20)
    pbar = -(g_hi + g_lo)
    _chain_reverse(Ws, bs, relaxs, L, Lams_up, Lbar_up, g_hi.copy(), True, padj)
    _chain_reverse(Ws, bs, relaxs, L, Lams_lo, Lbar_lo, g_lo.copy(), False, padj)

    # ---- J_bar and p_bar back through the nominal network
    #   J = G_l diag(phi'(z_l)) W_l F_{l-1},  G_l = dp/da_l,  F_l = da_l/da
    abar_l = Ws[L - 1].T @ pbar                 # adjoint of a_{L-1}
    F = [np.eye(a0.shape[0])]
    for l in range(1, L):
        F.append((dphi(act, zs[l - 1])[:, None] * Ws[l - 1]) @ F[l - 1])
    G = {L - 1: Ws[L - 1]}
    for l in range(L - 2, 0, -1):
        G[l] = (G[l + 1] * dphi(act, zs[l])[None, :]) @ Ws[l]
    for l in range(L - 1, 0, -1):
        zbar = dphi(act, zs[l - 1]) * abar_l
        WF = Ws[l - 1] @ F[l - 1]                       # [w_l, N]
        q = np.einsum("ik,ij,kj->k", G[l], Jbar, WF)    # diag(G^T Jbar WF^T)
        zbar = zbar + d2phi(act, zs[l - 1]) * q
        abar_l = Ws[l - 1].T @ zbar
    nominal_bar = abar_l                       # through p(a~) and J(a~): the nominal point only

    # ---- hidden targets s = L-1 .. 2 (seeds complete: only targets > s use layer s)
    ibp_l = [np.zeros_like(x) for x in ls]      # hidden = "ibp": adjoints of (l_s, u_s) arriving from layer s+1's interval step
    ibp_u = [np.zeros_like(x) for x in us]
    for s in range(L - 1, 1, -1):
        acc = padj[s - 1]
        lb, ub = relax_vjp(act, ls[s - 1], us[s - 1], relaxs[s - 1][4], acc[0], acc[1], acc[2], acc[3])
        if hidden == "ibp":
            # reverse of ibp_layer: l_s = W+ phi(l_{s-1}) + W- phi(u_{s-1}) + b, u_s = W+ phi(u_{s-1}) + W- phi(l_{s-1}) + b
            lb = lb + ibp_l[s - 1]
            ub = ub + ibp_u[s - 1]
            W = Ws[s - 1]
            Wp, Wn = np.maximum(W, 0.0), np.minimum(W, 0.0)
            alo_bar = Wp.T @ lb + Wn.T @ ub
            ahi_bar = Wp.T @ ub + Wn.T @ lb
            ibp_l[s - 2] += dphi_at(act, ls[s - 2]) * alo_bar
            ibp_u[s - 2] += dphi_at(act, us[s - 2]) * ahi_bar
            continue
        Lams_up, Lams_lo = fw["kept"][s]
        Lu0, Ll0 = Lams_up[0], Lams_lo[0]
        a_bar += Lu0.T @ ub + Ll0.T @ lb
        s_bar += np.abs(Lu0).T @ ub - np.abs(Ll0).T @ lb
        Lbar_up = ub[:, None] * (a0[None, :] + np.sign(Lu0) * sig[None, :])
        Lbar_lo = lb[:, None] * (a0[None, :] - np.sign(Ll0) * sig[None, :])
        _chain_reverse(Ws, bs, relaxs, s, Lams_up, Lbar_up, ub, True, padj)
        _chain_reverse(Ws, bs, relaxs, s, Lams_lo, Lbar_lo, lb, False, padj)

    # ---- layer 1: l_1, u_1 = W_1 a~ + b_1 -+ |W_1| sigma
    acc = padj[0]
    lb, ub = relax_vjp(act, ls[0], us[0], relaxs[0][4], acc[0], acc[1], acc[2], acc[3])
    lb = lb + ibp_l[0]
    ub = ub + ibp_u[0]
    a_bar += Ws[0].T @ (lb + ub)
    s_bar += np.abs(Ws[0]).T @ (ub - lb)
    if slope_grads is not None:
        # adjoints of the lower slopes k^L of every hidden layer (complete now: every target has been reversed); for an
        # unstable ReLU neuron k^L = alpha is a free parameter, so this is d(objective)/d(alpha)
        slope_grads.extend(padj[l][2].copy() for l in range(L - 1))
    if mu is None:
        return a_bar + nominal_bar, s_bar
    return a_bar + nominal_bar, s_bar, a_bar - J.T @ (g_hi + g_lo)


def leb_nn_vjp(Ws, bs, act, nom, rad, g_lo, g_hi, hidden="crown", mu=None):
    """Batch driver: [tiles, N] inputs, [tiles, n] cotangents -> grads [tiles, N] (a third array with mu)."""
    Ws = [np.asarray(W, dtype=np.float64) for W in Ws]
    bs = [np.asarray(b, dtype=np.float64) for b in bs]
    nom = np.asarray(nom, dtype=np.float64)
    rad = np.asarray(rad, dtype=np.float64)
    g_lo = np.asarray(g_lo, dtype=np.float64)
    g_hi = np.asarray(g_hi, dtype=np.float64)
    gn = np.empty_like(nom)
    gr = np.empty_like(rad)
    if mu is not None:
        mu = np.asarray(mu, dtype=np.float64)
        gm = np.empty_like(nom)
        for i in range(nom.shape[0]):
            gn[i], gr[i], gm[i] = crown_vjp(Ws, bs, act, nom[i], rad[i], g_lo[i], g_hi[i], hidden=hidden, mu=mu[i])
        return gn, gr, gm
    for i in range(nom.shape[0]):
        gn[i], gr[i] = crown_vjp(Ws, bs, act, nom[i], rad[i], g_lo[i], g_hi[i], hidden=hidden)
    return gn, gr


# --------------------------------------------------------------------------
# optimisable lower slopes (alpha-CROWN style): projected gradient descent on the lower slopes of the
# unstable ReLU neurons, one slope set per tile, objective = total width sum_i (r_hi_i - r_lo_i); every iterate is a
# sound enclosure (any alpha in [0, 1] is), the best one is kept.  The paper gives no such procedure (L194-196 only
# names CROWN): plain gradient steps with a caller-chosen step size.
# --------------------------------------------------------------------------
def default_alphas(Ws, bs, a0, sig):
    """the adaptive slopes of reading R8 at the bounds they produce (the starting point of the descent)"""
    fw = crown_forward(Ws, bs, ACT_RELU, a0, sig)
    return [r[2].copy() for r in fw["relaxs"]]


def alpha_refine(Ws, bs, a0, sig, steps, lr):
    """Returns (r_lo, r_hi, width0, width) of the best iterate."""
    alphas = default_alphas(Ws, bs, a0, sig)
    n = Ws[-1].shape[0]
    best = None
    w0 = None
    for it in range(steps + 1):
        fw = crown_forward(Ws, bs, ACT_RELU, a0, sig, alphas=alphas)
        w = float((fw["r_hi"] - fw["r_lo"]).sum())
        if it == 0:
            w0 = w
        if best is None or w < best[2]:
            best = (fw["r_lo"].copy(), fw["r_hi"].copy(), w)
        if it == steps:
            break
        grads = []
        crown_vjp(Ws, bs, ACT_RELU, a0, sig, -np.ones(n), np.ones(n), alphas=alphas, slope_grads=grads)
        alphas = [np.clip(a - lr * g, 0.0, 1.0) for a, g in zip(alphas, grads)]
    return best[0], best[1], w0, best[2]
