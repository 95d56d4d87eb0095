"""Tolerances and comparison helpers of the GPU parity tests.

Bounds (north_star): |got - ref| <= 1e-5 |ref| + 1e-7, element by element.
Gradients (north_star "1e-4 on gradients", made precise in DESIGN.md): the gradient of one tile is
ONE vector g = [grad_nom; grad_rad] in R^{2N}; the test is
    |got - ref| <= 1e-4 |ref| + 3e-5 * S_tile,   S_tile = max_j |g_ref[j]|  over both halves,
i.e. entrywise 1e-4 relative plus a normwise floor: grad_nom is the small difference of the upper-
and lower-bound adjoints (u_bar + l_bar) whose FP32 rounding scales with |u_bar| + |l_bar|, the size
of grad_rad (u_bar - l_bar), so an FP32 evaluation cannot be entrywise-relative on it.
"""
import json
import os

import numpy as np

BOUND_RTOL, BOUND_ATOL = 1e-5, 1e-7
GRAD_RTOL, GRAD_NORMWISE = 1e-4, 3e-5


_LOG = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")


def report(what, worst):
    """Every parity helper reports the worst err/tol it saw: printed (pytest -s / -rP shows it) and, on the GPU box,
    appended to gpurun_out/parity_worst.jsonl so the numbers quoted in DESIGN.md section 6 can be read back."""
    worst = float(worst)
    print(f"[parity] {what}: worst err/tol = {worst:.3g}")
    if os.path.isdir(_LOG):
        try:
            with open(os.path.join(_LOG, "parity_worst.jsonl"), "a") as f:
                f.write(json.dumps({"what": what, "worst_err_over_tol": worst}) + "\n")
        except OSError:
            pass
    return worst


def to_np(t):
    return t.detach().cpu().numpy().astype(np.float64)


def assert_bounds_close(got, ref, what=""):
    got = np.asarray(got, dtype=np.float64).reshape(ref.shape)
    err = np.abs(got - ref)
    tol = BOUND_RTOL * np.abs(ref) + BOUND_ATOL
    bad = ~(err <= tol)
    report(what, np.nanmax(err / tol) if err.size else 0.0)
    assert not bad.any(), f"{what}: {bad.sum()} of {bad.size} outside tolerance, worst err/tol {np.nanmax(err / tol):.3g}"


def assert_grads_close(gn, gr, ref_n, ref_r, what=""):
    """gn, gr, ref_n, ref_r: [tiles, N]."""
    gn = np.asarray(gn, dtype=np.float64).reshape(ref_n.shape)
    gr = np.asarray(gr, dtype=np.float64).reshape(ref_r.shape)
    S = np.maximum(np.abs(ref_n).max(1), np.abs(ref_r).max(1))[:, None]
    for name, got, ref in (("grad_nom", gn, ref_n), ("grad_rad", gr, ref_r)):
        err = np.abs(got - ref)
        tol = GRAD_RTOL * np.abs(ref) + GRAD_NORMWISE * S + 1e-12
        bad = ~(err <= tol)
        report(f"{what} {name}", np.nanmax(err / tol) if err.size else 0.0)
        assert not bad.any(), f"{what} {name}: {bad.sum()} of {bad.size} outside tolerance, worst err/tol {np.nanmax(err / tol):.3g}"


GRAD_NORMWISE_ANALYTIC = 1e-6      # SURVEY 8(c).5's proposal; the analytic path meets it


def assert_grad_dirs_close(got, ref, S, what=""):
    """Analytic path, gradient entries along selected directions: got/ref [tiles, ndirs], S [tiles]."""
    err = np.abs(np.asarray(got, dtype=np.float64) - ref)
    tol = GRAD_RTOL * np.abs(ref) + GRAD_NORMWISE_ANALYTIC * np.asarray(S)[:, None] + 1e-12
    bad = ~(err <= tol)
    report(what, np.nanmax(err / tol) if err.size else 0.0)
    assert not bad.any(), f"{what}: {bad.sum()} of {bad.size} outside tolerance, worst err/tol {np.nanmax(err / tol):.3g}"


def grads_ratio(gn, gr, ref_n, ref_r):
    """Per-tile worst err/tol of the assert_grads_close criterion."""
    gn = np.asarray(gn, dtype=np.float64).reshape(ref_n.shape)
    gr = np.asarray(gr, dtype=np.float64).reshape(ref_r.shape)
    S = np.maximum(np.abs(ref_n).max(1), np.abs(ref_r).max(1))[:, None]
    worst = np.zeros(ref_n.shape[0])
    for got, ref in ((gn, ref_n), (gr, ref_r)):
        worst = np.maximum(worst, (np.abs(got - ref) / (GRAD_RTOL * np.abs(ref) + GRAD_NORMWISE * S + 1e-12)).max(1))
    return worst


def grads_ok(gn, gr, ref_n, ref_r):
    """Per-tile boolean of the assert_grads_close criterion."""
    return grads_ratio(gn, gr, ref_n, ref_r) <= 1.0


def assert_nn_grads_close(O, mlp, nom, rad, g_lo, g_hi, gn, gr, what="", max_tie_tiles=2):
    """NN VJP parity with the kinks of |W - J| (eq. (21)) handled as 'several results are correct':
    a tile whose gradient misses the oracle's is accepted only if the oracle reports entries of
    W_up - J / W_lo - J below 1e-6 max|W| (FP32 cannot resolve their sign; reading R20) and
    the result matches the oracle's gradient for some choice of those signs.  At most
    `max_tie_tiles` tiles may need this."""
    ref_n, ref_r = O.leb_nn_vjp(mlp.W, mlp.b, mlp.act, nom, rad, g_lo, g_hi)
    gn = np.asarray(gn, dtype=np.float64).reshape(ref_n.shape)
    gr = np.asarray(gr, dtype=np.float64).reshape(ref_r.shape)
    ratio = grads_ratio(gn, gr, ref_n, ref_r)
    ok = ratio <= 1.0
    report(f"{what} gradient (tiles off a kink of |W - J|)", ratio[ok].max() if ok.any() else 0.0)
    bad = np.nonzero(~ok)[0]
    assert len(bad) <= max_tie_tiles, f"{what}: {len(bad)} tiles miss the oracle gradient"
    Ws = [np.asarray(W, dtype=np.float64) for W in mlp.W]
    bs = [np.asarray(b, dtype=np.float64) for b in mlp.b]
    for t in bad:
        a0, sg = np.asarray(nom[t], dtype=np.float64), np.asarray(rad[t], dtype=np.float64)
        ties = O.output_sign_ties(Ws, bs, mlp.act, a0, sg)
        assert 0 < len(ties) <= 12, f"{what}: tile {t} misses the oracle gradient and has {len(ties)} sign ties"
        # the reverse sweep is linear in the signs of (W - J): flipping a set F of ties changes the gradient by the sum
        # of the single-flip changes, so all 2^k one-sided gradients follow from k + 1 oracle calls
        glo_t, ghi_t = np.asarray(g_lo[t], dtype=np.float64), np.asarray(g_hi[t], dtype=np.float64)
        base = np.concatenate(O.crown_vjp(Ws, bs, mlp.act, a0, sg, glo_t, ghi_t))
        delta = [np.concatenate(O.crown_vjp(Ws, bs, mlp.act, a0, sg, glo_t, ghi_t, flips=[e])) - base for e in ties]
        N = a0.shape[0]
        found = False
        for mask in range(1, 1 << len(ties)):
            g = base + sum(delta[q] for q in range(len(ties)) if mask >> q & 1)
            if grads_ok(gn[t:t + 1], gr[t:t + 1], g[None, :N], g[None, N:])[0]:
                found = True
                break
        assert found, f"{what}: tile {t} matches neither one-sided gradient at its {len(ties)} sign ties"
