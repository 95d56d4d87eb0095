"""Pins for oracle/tube_oracle.py and oracle/pbh_refine.py (CPU only): (22), (27)-(28), (35) against what the
mathematics fixes -- vertex enumeration of the zonotopes in (26), corner enumeration of the interval matrix in (22),
a closed form and central differences for (35) -- and partitioning / PGD against soundness and monotonicity."""
import itertools

import numpy as np
import pytest

from oracle import pbh_oracle as P, pbh_refine as R, tube_oracle as TU
from paper_2607_01203_b200 import workloads as wl


def _rand_problem(rng, T, n, m):
    N = n + m
    Phi = rng.standard_normal((T * (T + 1) // 2, N, n))
    for j in range(T):
        Phi[TU.block(j + 1, j), :n] = np.eye(n)          # (34c): Phi^x_{j+1,j} = I
    c = rng.standard_normal((T, n)) * 0.1
    Rd = rng.uniform(0.01, 0.2, (T, n))
    E = rng.uniform(0.0, 0.05, n)
    return Phi, c, Rd, E


def test_dist_bound_is_the_corner_maximum():
    rng = np.random.default_rng(0)
    n, nw = 3, 2
    E_nom = rng.standard_normal((n, nw))
    E_lo = E_nom - rng.uniform(0, 0.3, (n, nw))
    E_hi = E_nom + rng.uniform(0, 0.3, (n, nw))
    lo, hi = TU.dist_bound(E_lo, E_hi, E_nom)
    best = np.full(n, -np.inf)
    for corner in itertools.product((0, 1), repeat=n * nw):
        Ex = np.where(np.array(corner).reshape(n, nw) == 1, E_hi, E_lo)
        for w in itertools.product((-1.0, 1.0), repeat=nw):
            best = np.maximum(best, (Ex - E_nom) @ np.array(w))
    assert np.allclose(hi, best, rtol=0, atol=1e-14) and np.allclose(lo, -best, rtol=0, atol=1e-14)
    z_lo, z_hi = TU.dist_bound(E_nom, E_nom, E_nom)      # constant E: r_dist = 0 (reading R13)
    assert np.all(z_lo == 0) and np.all(z_hi == 0)


def test_tube_width_is_the_support_function_of_the_minkowski_sum():
    """(28) = max over the zonotope (+)_j Phi_kj E_bar_j E_2n of each coordinate ((26) L283-287): enumerate all vertices."""
    rng = np.random.default_rng(1)
    T, n, m = 2, 2, 1
    Phi, c, Rd, E = _rand_problem(rng, T, n, m)
    h_mu, h_sigma = TU.tube_propagate(Phi, c, Rd, E)
    for k in range(1, T + 1):
        best = np.full(n + m, -np.inf)
        for e in itertools.product((-1.0, 1.0), repeat=2 * n * k):
            e = np.array(e).reshape(k, 2 * n)
            x = sum(Phi[TU.block(k, j)] @ TU.ebar(E, Rd[j]) @ e[j] for j in range(k))
            best = np.maximum(best, x)
        assert np.allclose(h_sigma[k - 1], best, rtol=0, atol=1e-13)
        assert np.allclose(h_mu[k - 1], sum(Phi[TU.block(k, j)] @ c[j] for j in range(k)), rtol=0, atol=1e-14)


def test_tube_propagation_of_a_linear_system_contains_rollouts():
    """Open loop x+ = A x + d, d in c_bar + E_bar E_2n: Phi^x_kj = A^(k-1-j) propagates the zonotopes exactly, so random
    disturbance rollouts stay inside mu +- sigma and vertex rollouts touch it."""
    rng = np.random.default_rng(2)
    T, n = 4, 3
    A = rng.standard_normal((n, n)) * 0.6
    Phi = np.zeros((T * (T + 1) // 2, n, n))
    for k in range(1, T + 1):
        for j in range(k):
            Phi[TU.block(k, j)] = np.linalg.matrix_power(A, k - 1 - j)
    c = rng.standard_normal((T, n)) * 0.1
    Rd = rng.uniform(0.01, 0.2, (T, n))
    E = rng.uniform(0.01, 0.05, n)
    h_mu, h_sigma = TU.tube_propagate(Phi, c, Rd, E)
    hit = np.zeros((T, n))
    for trial in range(4000):
        e = rng.choice([-1.0, 1.0], (T, 2 * n)) if trial % 2 else rng.uniform(-1, 1, (T, 2 * n))
        x = np.zeros(n)
        for k in range(1, T + 1):
            x = A @ x + c[k - 1] + TU.ebar(E, Rd[k - 1]) @ e[k - 1]
            assert np.all(np.abs(x - h_mu[k - 1]) <= h_sigma[k - 1] + 1e-12)
            hit[k - 1] = np.maximum(hit[k - 1], np.abs(x - h_mu[k - 1]) / h_sigma[k - 1])
    assert hit[0].min() > 0.999           # k = 1: a vertex of the single zonotope is reached among 2000 random vertices


def test_j_err_closed_form_and_gradient():
    rng = np.random.default_rng(3)
    T, n, m = 3, 2, 1
    Phi, c, Rd, E = _rand_problem(rng, T, n, m)
    # identity responses only (Phi_{j+1,j} = [I; 0], the rest 0): J_err = sum_j (|E|^2 + |R_j|^2)
    Pid = np.zeros_like(Phi)
    for j in range(T):
        Pid[TU.block(j + 1, j), :n] = np.eye(n)
    assert np.isclose(TU.j_err(Pid, Rd, E), T * (E ** 2).sum() + (Rd ** 2).sum(), rtol=1e-14)
    g = TU.j_err_grad(Phi, Rd, E)
    h = 1e-6
    for j in range(T):
        for cc in range(n):
            d = np.zeros_like(Rd)
            d[j, cc] = h
            fd = (TU.j_err(Phi, Rd + d, E) - TU.j_err(Phi, Rd - d, E)) / (2 * h)
            assert np.isclose(fd, g[j, cc], rtol=1e-7, atol=1e-9)


# ---------------------------------------------------------------- partitioning and PGD (Table II)
def test_partition_is_sound_and_not_wider():
    w = wl.make_config(2, B=1, T=3)
    spec = P.spec_from_workload(w)
    N = w.N
    nom, rad = w.nom.reshape(-1, N).astype(float), 4.0 * w.rad.reshape(-1, N).astype(float)
    splits = np.ones(N, dtype=int)
    splits[[3, 4, 12]] = (2, 3, 2)                       # roll, pitch, thrust
    lo1, hi1, st = R.partition(spec, nom, rad, np.ones(N, dtype=int))
    lo0, hi0, _ = P.pbh(spec, nom, rad)
    assert st == 0 and np.array_equal(lo1, lo0) and np.array_equal(hi1, hi0)     # one part = the plain bound
    lo, hi, st = R.partition(spec, nom, rad, splits)
    assert st == 0
    assert np.all(lo >= lo0 - 1e-15) and np.all(hi <= hi0 + 1e-15)               # inclusion isotonicity
    assert ((hi - lo).sum(1) < 0.995 * (hi0 - lo0).sum(1)).all()                 # and it does help (a few per cent here)
    rng = np.random.default_rng(5)
    verts = np.array(list(itertools.product((-1.0, 1.0), repeat=N)))
    for t in range(3):
        U = np.concatenate([rng.uniform(-1, 1, (50000, N)), verts])
        X = nom[t][None] + U * rad[t][None]
        J = P.jac(spec, nom[t])
        r = P.f(spec, X) - P.f(spec, nom[t][None]) - (X - nom[t]) @ J.T
        assert np.all(r.max(0) <= hi[t] + 1e-12) and np.all(r.min(0) >= lo[t] - 1e-12)
    # with an offset box as well
    mu = rad * rng.uniform(-1.5, 1.5, rad.shape)
    lo, hi, _ = R.partition(spec, nom, rad, splits, mu=mu)
    lo0, hi0, _ = P.pbh(spec, nom, rad, mu=mu)
    assert np.all(lo >= lo0 - 1e-15) and np.all(hi <= hi0 + 1e-15)


def test_sub_boxes_tile_the_box():
    rad, mu = np.array([0.3, 0.2, 0.5]), np.array([0.1, -0.4, 0.0])
    mus, rads = R.sub_boxes(rad, mu, [2, 1, 3])
    assert mus.shape == (6, 3)
    for g, s in enumerate((2, 1, 3)):
        edges = sorted(set(np.round(np.concatenate([mus[:, g] - rads[:, g], mus[:, g] + rads[:, g]]), 12)))
        assert np.allclose(edges, mu[g] - rad[g] + 2 * rad[g] * np.arange(s + 1) / s)


def test_pgd_never_worse_and_flat_for_constant_hessian():
    w = wl.make_config(2, B=1, T=4)
    spec = P.spec_from_workload(w)
    centre, rad = w.nom.reshape(-1, w.N).astype(float), w.rad.reshape(-1, w.N).astype(float)
    nom0 = centre + 0.4 * rad * np.random.default_rng(1).uniform(-1, 1, rad.shape)     # "starting from random nominal points" L393
    best, w0, wb = R.pgd(spec, centre, rad, nom0, 0.5 * rad, steps=8, lr=0.03)
    assert np.all(wb <= w0) and (wb < 0.9 * w0).all()
    assert np.all(np.abs(best - centre) <= 0.5 * rad + 1e-15)
    # the returned point really has the returned width
    wchk, _, _ = R.width_and_grad(spec, best, centre, rad)
    assert np.allclose(wchk, wb, rtol=1e-12)
    # dW/da~ against central differences (box fixed)
    _, g, _ = R.width_and_grad(spec, centre + 0.2 * rad, centre, rad)
    h, ok = 1e-6, 0
    for d in range(w.N):
        e = np.zeros_like(centre)
        e[:, d] = h
        fp = R.width_and_grad(spec, centre + 0.2 * rad + e, centre, rad)[0]
        fm = R.width_and_grad(spec, centre + 0.2 * rad - e, centre, rad)[0]
        f0 = R.width_and_grad(spec, centre + 0.2 * rad, centre, rad)[0]
        for t in range(centre.shape[0]):
            if abs((fp[t] - f0[t]) - (f0[t] - fm[t])) > 1e-3 * abs(fp[t] - fm[t]) + 1e-13:
                continue
            assert abs((fp[t] - fm[t]) / (2 * h) - g[t, d]) <= 1e-5 * abs(g[t, d]) + 1e-6 * np.abs(g[t]).max()
            ok += 1
    assert ok >= w.N
    # satellite: constant Hessian and a box that does not move => W does not depend on a~ at all?  No: D = A (-) a~ does.
    # What is flat is the CENTRED case: with the optimum at mu = 0 every step away from the centre widens the bound.
    ws = wl.make_paper_system("satellite", 1, 2)
    sspec = P.spec_from_workload(ws)
    c2, r2 = ws.nom.reshape(-1, 10).astype(float), ws.rad.reshape(-1, 10).astype(float)
    w_c = R.width_and_grad(sspec, c2, c2, r2)[0]
    w_off = R.width_and_grad(sspec, c2 + 0.3 * r2, c2, r2)[0]
    assert np.all(w_off > w_c)


def test_partition_vjp_matches_central_differences():
    """partition_vjp against central differences of partition() itself in every input direction (nom, rad, mu) with random
    cotangents; directions on which the selected sub-box changes within the step (a kink of the hull) are skipped, and
    most must remain.  One part reduces to the plain VJP."""
    w = wl.make_config(2, B=1, T=2)
    spec = P.spec_from_workload(w)
    N, n = w.N, w.n
    rng = np.random.default_rng(9)
    nom, rad = w.nom.reshape(-1, N).astype(float), 4.0 * w.rad.reshape(-1, N).astype(float)
    mu = rad * rng.uniform(-0.8, 0.8, rad.shape)
    g_lo, g_hi = rng.normal(size=(2, n)), rng.normal(size=(2, n))
    g1 = R.partition_vjp(spec, nom, rad, np.ones(N, dtype=int), g_lo, g_hi, mu=mu)
    g0, _ = P.pbh_vjp(spec, nom, rad, g_lo, g_hi, mu=mu)
    assert np.allclose(g1, g0, rtol=1e-13, atol=1e-15)
    splits = np.ones(N, dtype=int)
    splits[[3, 4, 12]] = (2, 3, 2)
    g = R.partition_vjp(spec, nom, rad, splits, g_lo, g_hi, mu=mu)

    def val(a, r, m):
        lo, hi, _ = R.partition(spec, a, r, splits, mu=m)
        return (g_lo * lo + g_hi * hi).sum(1)

    h, ok = 1e-6, 0
    for d in range(3 * N):
        e = np.zeros((2, 3 * N))
        e[:, d] = h
        args_p = (nom + e[:, :N], rad + e[:, N:2 * N], mu + e[:, 2 * N:])
        args_m = (nom - e[:, :N], rad - e[:, N:2 * N], mu - e[:, 2 * N:])
        fp, fm, f0 = val(*args_p), val(*args_m), val(nom, rad, mu)
        for t in range(2):
            if abs((fp[t] - f0[t]) - (f0[t] - fm[t])) > 1e-3 * abs(fp[t] - fm[t]) + 1e-13:
                continue                                     # a kink inside the step
            assert abs((fp[t] - fm[t]) / (2 * h) - g[t, d]) <= 1e-5 * abs(g[t, d]) + 1e-6 * np.abs(g[t]).max(), (t, d)
            ok += 1
    assert ok >= 5 * N
