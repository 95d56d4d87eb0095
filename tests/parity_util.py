"""Tolerances and comparison helpers of the GPU parity tests.

Bounds (north_star): |got - ref| <= 1e-5 |ref| + 1e-7, element by element.
Gradients (north_star "1e-4 on gradients", made precise in DESIGN.md): the gradient of one tile is
ONE vector g = [grad_nom; grad_rad] in R^{2N}; the test is
    |got - ref| <= 1e-4 |ref| + 3e-5 * S_tile,   S_tile = max_j |g_ref[j]|  over both halves,
i.e. entrywise 1e-4 relative plus a normwise floor: grad_nom is the small difference of the upper-
and lower-bound adjoints (u_bar + l_bar) whose FP32 rounding scales with |u_bar| + |l_bar|, the size
of grad_rad (u_bar - l_bar), so an FP32 evaluation cannot be entrywise-relative on it.
"""
import numpy as np

BOUND_RTOL, BOUND_ATOL = 1e-5, 1e-7
GRAD_RTOL, GRAD_NORMWISE = 1e-4, 3e-5


def to_np(t):
    return t.detach().cpu().numpy().astype(np.float64)


def assert_bounds_close(got, ref, what=""):
    got = np.asarray(got, dtype=np.float64).reshape(ref.shape)
    err = np.abs(got - ref)
    tol = BOUND_RTOL * np.abs(ref) + BOUND_ATOL
    bad = ~(err <= tol)
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
        assert not bad.any(), f"{what} {name}: {bad.sum()} of {bad.size} outside tolerance, worst err/tol {np.nanmax(err / tol):.3g}"


def assert_grad_dirs_close(got, ref, S, what=""):
    """Analytic path, gradient entries along selected directions: got/ref [tiles, ndirs], S [tiles]."""
    err = np.abs(np.asarray(got, dtype=np.float64) - ref)
    tol = GRAD_RTOL * np.abs(ref) + GRAD_NORMWISE * np.asarray(S)[:, None] + 1e-12
    bad = ~(err <= tol)
    assert not bad.any(), f"{what}: {bad.sum()} of {bad.size} outside tolerance, worst err/tol {np.nanmax(err / tol):.3g}"
