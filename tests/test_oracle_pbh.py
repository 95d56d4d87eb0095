"""Pins for oracle/pbh_oracle.cpp (CPU only): the oracle is compared with what the
paper and the mathematics fix -- zero for linear maps (eq. (11)),
the constant-Hessian closed form, the unicycle closed form / hand-worked golden,
Cor. 1 ordering (17) PAPER.md:L179-188, soundness against samples and all box
vertices (Thm 1), textbook rigid-body identities for the quadrotor SLP, RK4 order,
and central differences for Jacobian, Hessian entries and the VJP."""
import itertools
import os

import numpy as np
import pytest

from oracle import pbh_oracle as P
from paper_2607_01203_b200 import workloads as wl

PARAMS = [0.05, 1.0, 9.81, 0.010, 0.015, 0.020, 1.0, 0.1]
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _true_r(spec, a0, X):
    J = P.jac(spec, a0)
    return P.f(spec, X) - P.f(spec, a0[None]) - (X - a0) @ J.T


# ---------------------------------------------------------------- exact cases
def test_linear_map_gives_exact_zero():
    rng = np.random.default_rng(0)
    C = rng.standard_normal((4, 6))
    spec = P.ModelSpec(P.MODEL_LINEAR, params=PARAMS, C=C)
    for mode in (P.MODE_PATH, P.MODE_EXPAND, P.MODE_CLASSIC):
        lo, hi, st = P.pbh(spec, rng.standard_normal((3, 6)), rng.uniform(0.1, 1, (3, 6)), mode)
        assert st == 0 and np.all(lo == 0.0) and np.all(hi == 0.0)


def test_quadratic_map_closed_form():
    rng = np.random.default_rng(1)
    n, N = 3, 6
    Q = rng.standard_normal((n, N, N))
    Q = Q + Q.transpose(0, 2, 1)
    Q[:, 1, 4] = Q[:, 4, 1] = 0.0
    C = rng.standard_normal((n, N))
    spec = P.ModelSpec(P.MODEL_QUADRATIC, params=PARAMS, Q=Q, C=C)
    nom, rad = rng.standard_normal((5, N)), rng.uniform(0.05, 0.5, (5, N))
    lo, hi, st = P.pbh(spec, nom, rad)
    for t in range(5):
        s = rad[t]
        for l in range(n):
            off = sum(abs(Q[l, k, j]) * s[j] * s[k] for j in range(N) for k in range(j + 1, N))
            up = off + 0.5 * sum(max(Q[l, k, k], 0) * s[k] ** 2 for k in range(N))
            dn = -off + 0.5 * sum(min(Q[l, k, k], 0) * s[k] ** 2 for k in range(N))
            assert np.isclose(hi[t, l], up, rtol=1e-12, atol=1e-14)
            assert np.isclose(lo[t, l], dn, rtol=1e-12, atol=1e-14)
    lo2, hi2, _ = P.pbh(spec, nom, rad, P.MODE_EXPAND)
    assert np.allclose(lo, lo2, rtol=1e-12, atol=1e-14) and np.allclose(hi, hi2, rtol=1e-12, atol=1e-14)
    # constant Hessian: r = 1/2 d^T Q d exactly; the bound must enclose its vertex values
    for s in itertools.product((-1.0, 1.0), repeat=N):
        d = rad[0] * np.array(s)
        r = 0.5 * np.einsum("lij,i,j->l", Q, d, d)
        assert np.all(r <= hi[0] + 1e-13) and np.all(r >= lo[0] - 1e-13)


def _read_golden(name):
    out = {}
    for line in open(os.path.join(GOLD, name)):
        if line.startswith("#") or not line.strip():
            continue
        k, a, b = line.split()
        out[k] = (float(a), float(b))
    return out


def test_unicycle_worked_instance_golden():
    g = _read_golden("unicycle_worked.txt")
    p = list(PARAMS)
    p[0] = 0.1
    spec = P.ModelSpec(P.MODEL_UNICYCLE, P.INTEG_EULER, 1, p)
    nom = np.array([[0.3, -0.2, 0.0, 1.0, 0.2]])
    rad = np.array([[0.05, 0.05, 0.1, 0.1, 0.07]])
    lo, hi, _ = P.pbh(spec, nom, rad)
    for i, k in enumerate(("r1_path", "r2_path", "r3_path")):
        assert np.isclose(lo[0, i], g[k][0], rtol=2e-9, atol=1e-15) and np.isclose(hi[0, i], g[k][1], rtol=2e-9, atol=1e-15)
    lo2, hi2, _ = P.pbh(spec, nom, rad, P.MODE_EXPAND)
    assert np.isclose(lo2[0, 0], g["r1_expand"][0], rtol=2e-9) and np.isclose(hi2[0, 0], g["r1_expand"][1], rtol=2e-9)


def test_unicycle_closed_form_config1():
    # r_1 in (-dt sinTH) D_th D_v + 1/2 (-dt v~ cosTH) D_th^2 with v PINNED (prefix box A^(3))
    w = wl.make_config(1)
    spec = P.spec_from_workload(w)
    nom, rad = w.nom.reshape(-1, 5).astype(float), w.rad.reshape(-1, 5).astype(float)
    lo, hi, st = P.pbh(spec, nom, rad)
    assert st == 0
    dt = 0.1
    for t in range(nom.shape[0]):
        th, v, sth, sv = nom[t, 2], nom[t, 3], rad[t, 2], rad[t, 3]
        a, b = th - sth, th + sth                      # |theta| <= 1.1 < pi/2
        sinlo, sinhi = np.sin(a), np.sin(b)
        coshi = 1.0 if a <= 0.0 <= b else max(np.cos(a), np.cos(b))
        coslo = min(np.cos(a), np.cos(b))
        mag_s = max(abs(sinlo), abs(sinhi))
        mag_c = max(abs(coslo), abs(coshi))
        h1 = sorted([-dt * v * coslo, -dt * v * coshi])       # H_thth for f_1
        h2 = sorted([-dt * v * sinlo, -dt * v * sinhi])       # H_thth for f_2
        exp = [(-dt * mag_s * sth * sv + 0.5 * min(h1[0], 0) * sth ** 2, dt * mag_s * sth * sv + 0.5 * max(h1[1], 0) * sth ** 2),
               (-dt * mag_c * sth * sv + 0.5 * min(h2[0], 0) * sth ** 2, dt * mag_c * sth * sv + 0.5 * max(h2[1], 0) * sth ** 2),
               (0.0, 0.0)]
        for i in range(3):
            assert np.isclose(lo[t, i], exp[i][0], rtol=1e-12, atol=1e-16)
            assert np.isclose(hi[t, i], exp[i][1], rtol=1e-12, atol=1e-16)


# ---------------------------------------------------------------- ordering and soundness
@pytest.mark.parametrize("cfg,tiles", [(1, 20), (2, 12)])
def test_cor1_ordering(cfg, tiles):
    w = wl.make_config(cfg)
    spec = P.spec_from_workload(w)
    nom, rad = w.nom.reshape(-1, w.N)[:tiles], w.rad.reshape(-1, w.N)[:tiles]
    lp, hp, _ = P.pbh(spec, nom, rad, P.MODE_PATH)
    le, he, _ = P.pbh(spec, nom, rad, P.MODE_EXPAND)
    lc, hc, _ = P.pbh(spec, nom, rad, P.MODE_CLASSIC)
    eps = 1e-15
    assert np.all(le <= lp + eps) and np.all(hp <= he + eps)
    assert np.all(lc <= le + eps) and np.all(he <= hc + eps)
    assert np.any(he - le > 1.001 * (hp - lp))        # path is strictly tighter somewhere


def test_cor1_ordering_small_chain():
    w = wl.make_small_chain(2, 1, 2)
    spec = P.spec_from_workload(w)
    nom, rad = w.nom.reshape(-1, w.N), w.rad.reshape(-1, w.N)
    lp, hp, _ = P.pbh(spec, nom, rad, P.MODE_PATH)
    le, he, _ = P.pbh(spec, nom, rad, P.MODE_EXPAND)
    assert np.all(le <= lp + 1e-15) and np.all(hp <= he + 1e-15)


@pytest.mark.parametrize("cfg,tiles", [(1, 20), (2, 3)])
def test_soundness_samples_and_all_vertices(cfg, tiles):
    w = wl.make_config(cfg)
    spec = P.spec_from_workload(w)
    N = w.N
    nom, rad = w.nom.reshape(-1, N)[:tiles].astype(float), w.rad.reshape(-1, N)[:tiles].astype(float)
    lo, hi, _ = P.pbh(spec, nom, rad)
    rng = np.random.default_rng(10 + cfg)
    V = np.array(list(itertools.product((-1.0, 1.0), repeat=N)))
    sharp = []
    for t in range(tiles):
        X = np.concatenate([nom[t] + rad[t] * rng.uniform(-1, 1, (100000, N)), nom[t] + rad[t] * V])
        R = _true_r(spec, nom[t], X)
        assert np.all(R.min(0) >= lo[t] - 1e-15) and np.all(R.max(0) <= hi[t] + 1e-15)
        wd = hi[t] - lo[t]
        sharp.append(((R.max(0) - R.min(0))[wd > 0] / wd[wd > 0]).min())
    assert min(sharp) > 0.3          # the enclosure is not vacuous (sampled range / bound width)


def test_soundness_small_chain_samples():
    w = wl.make_small_chain(3, 1, 2)
    spec = P.spec_from_workload(w)
    N = w.N
    nom, rad = w.nom.reshape(-1, N).astype(float), w.rad.reshape(-1, N).astype(float)
    lo, hi, _ = P.pbh(spec, nom, rad)
    rng = np.random.default_rng(3)
    for t in range(2):
        S = rng.choice((-1.0, 1.0), (50000, N))
        X = np.concatenate([nom[t] + rad[t] * rng.uniform(-1, 1, (50000, N)), nom[t] + rad[t] * S])
        R = _true_r(spec, nom[t], X)
        assert np.all(R.min(0) >= lo[t] - 1e-15) and np.all(R.max(0) <= hi[t] + 1e-15)


def test_domain_error_reports_infinite_bounds():
    spec = P.ModelSpec(P.MODEL_QUAD12, P.INTEG_EULER, 1, PARAMS)
    nom = np.zeros((1, 16))
    nom[0, 4] = np.pi / 2                       # theta box contains pi/2: 0 in cos(theta)
    lo, hi, st = P.pbh(spec, nom, np.full((1, 16), 0.01))
    assert st == 4 and np.all(np.isinf(lo)) and np.all(np.isinf(hi))


def test_zero_radius_coordinates():
    w = wl.make_config(2)
    spec = P.spec_from_workload(w)
    nom, rad = w.nom.reshape(-1, 16)[:2].astype(float), w.rad.reshape(-1, 16)[:2].astype(float)
    lo, hi, _ = P.pbh(spec, nom, np.zeros_like(rad))
    assert np.all(lo == 0) and np.all(hi == 0)


# ---------------------------------------------------------------- model SLPs vs textbook definitions
def _Rzyx(phi, th, psi):
    cf, sf, ct, st, cp, sp = np.cos(phi), np.sin(phi), np.cos(th), np.sin(th), np.cos(psi), np.sin(psi)
    Rz = np.array([[cp, -sp, 0], [sp, cp, 0], [0, 0, 1]])
    Ry = np.array([[ct, 0, st], [0, 1, 0], [-st, 0, ct]])
    Rx = np.array([[1, 0, 0], [0, cf, -sf], [0, sf, cf]])
    return Rz @ Ry @ Rx


def _field(spec_euler, x, u, dt):
    a = np.concatenate([x, u])[None]
    return (P.f(spec_euler, a)[0] - x) / dt


def test_quad12_field_matches_rigid_body_textbook():
    p = list(PARAMS)
    spec = P.ModelSpec(P.MODEL_QUAD12, P.INTEG_EULER, 1, p)
    dt, m, g, Jx, Jy, Jz = p[0], p[1], p[2], p[3], p[4], p[5]
    rng = np.random.default_rng(4)
    for _ in range(10):
        x = rng.uniform(-1, 1, 12)
        x[3:6] = rng.uniform(-0.6, 0.6, 3)
        u = np.array([m * g * rng.uniform(0.5, 1.5), *rng.uniform(-0.1, 0.1, 3)])
        k = _field(spec, x, u, dt)
        phi, th, psi = x[3:6]
        om = x[9:12]
        R = _Rzyx(phi, th, psi)
        assert np.allclose(k[0:3], x[6:9], atol=1e-11)                     # p' = v
        assert np.allclose(k[6:9], R @ np.array([0, 0, u[0] / m]) - np.array([0, 0, g]), atol=1e-10)   # thrust along body z
        # Euler-angle kinematics: d/dt R = R [omega]_x
        h = 1e-6
        Rp = _Rzyx(*(x[3:6] + h * k[3:6]))
        Rm = _Rzyx(*(x[3:6] - h * k[3:6]))
        Om = np.array([[0, -om[2], om[1]], [om[2], 0, -om[0]], [-om[1], om[0], 0]])
        assert np.allclose((Rp - Rm) / (2 * h), R @ Om, atol=1e-7)
        # Euler's equations  J om' = tau - om x (J om)
        Jm = np.diag([Jx, Jy, Jz])
        assert np.allclose(k[9:12], np.linalg.solve(Jm, u[1:4] - np.cross(om, Jm @ om)), atol=1e-9)
    # hover equilibrium
    x = np.zeros(12)
    assert np.allclose(_field(spec, x, np.array([m * g, 0, 0, 0]), dt), 0, atol=1e-10)


def test_chain_coupling_invariants():
    U = 4
    p = list(PARAMS)
    chain = P.ModelSpec(P.MODEL_QUADCHAIN, P.INTEG_EULER, U, p)
    single = P.ModelSpec(P.MODEL_QUAD12, P.INTEG_EULER, 1, p)
    dt, m, k1, k3 = p[0], p[1], p[6], p[7]
    rng = np.random.default_rng(5)
    x = rng.uniform(-1, 1, 12 * U)
    u = rng.uniform(-1, 1, 4 * U)
    kc = (P.f(chain, np.concatenate([x, u])[None])[0] - x) / dt
    ks = np.concatenate([_field(single, x[12 * i:12 * i + 12], u[4 * i:4 * i + 4], dt) for i in range(U)])
    diff = (kc - ks).reshape(U, 12)
    assert np.allclose(diff[:, :6], 0, atol=1e-10) and np.allclose(diff[:, 9:], 0, atol=1e-10)
    assert np.allclose(diff[:, 6:9].sum(0), 0, atol=1e-9)                 # internal forces cancel
    pos = x.reshape(U, 12)[:, :3]
    d01 = pos[1] - pos[0]
    assert np.allclose(diff[0, 6:9], (k1 * d01 + k3 * d01 ** 3) / m, atol=1e-9)   # end unit: one spring, attractive
    # 1-unit chain is the single quadrotor
    one = P.ModelSpec(P.MODEL_QUADCHAIN, P.INTEG_RK4, 1, p)
    q = P.ModelSpec(P.MODEL_QUAD12, P.INTEG_RK4, 1, p)
    a = np.concatenate([x[:12], u[:4]])[None]
    assert np.array_equal(P.f(one, a), P.f(q, a))


def test_rk4_is_fourth_order():
    from scipy.integrate import solve_ivp
    rng = np.random.default_rng(6)
    x = rng.uniform(-0.5, 0.5, 12)
    u = np.array([9.81, 0.05, -0.03, 0.02])
    errs = []
    for dt in (0.1, 0.05):
        p = list(PARAMS)
        p[0] = dt
        rk = P.ModelSpec(P.MODEL_QUAD12, P.INTEG_RK4, 1, p)
        eu = P.ModelSpec(P.MODEL_QUAD12, P.INTEG_EULER, 1, p)
        sol = solve_ivp(lambda t, y: _field(eu, y, u, dt), (0, dt), x, rtol=1e-13, atol=1e-14)
        errs.append(np.abs(P.f(rk, np.concatenate([x, u])[None])[0] - sol.y[:, -1]).max())
    assert errs[0] < 1e-4 and 20 < errs[0] / errs[1] < 50          # local error O(dt^5): ratio ~32


# ---------------------------------------------------------------- derivatives
@pytest.mark.parametrize("model,integ,U", [(P.MODEL_UNICYCLE, P.INTEG_EULER, 1), (P.MODEL_QUAD12, P.INTEG_RK4, 1),
                                           (P.MODEL_QUADCHAIN, P.INTEG_RK4, 2)])
def test_jacobian_and_point_hessian_match_finite_differences(model, integ, U):
    spec = P.ModelSpec(model, integ, U, PARAMS)
    rng = np.random.default_rng(7)
    a = rng.uniform(-0.4, 0.4, spec.N)
    if model != P.MODEL_UNICYCLE:
        for i in range(U):
            a[spec.n + 4 * i] = 9.81
    J = P.jac(spec, a)
    h = 1e-6
    E = np.eye(spec.N)
    Jfd = np.array([(P.f(spec, (a + h * e)[None])[0] - P.f(spec, (a - h * e)[None])[0]) / (2 * h) for e in E]).T
    assert np.allclose(J, Jfd, atol=1e-7)
    pairs = [(0, 0), (2, 3), (2, 2)] if model == P.MODEL_UNICYCLE else [(3, 4), (4, 4), (5, 12), (9, 10), (3, 15), (0, 6)]
    if U == 2:
        pairs += [(0, 12), (1, 13), (12, 18), (4, 20)]
    hh = 1e-4
    for j, k in pairs:
        Hlo, Hhi = P.hessian_entry(spec, a, a, j, k)
        assert np.allclose(Hlo, Hhi, atol=1e-12)
        fpp = P.f(spec, (a + hh * E[j] + hh * E[k])[None])[0]
        fpm = P.f(spec, (a + hh * E[j] - hh * E[k])[None])[0]
        fmp = P.f(spec, (a - hh * E[j] + hh * E[k])[None])[0]
        fmm = P.f(spec, (a - hh * E[j] - hh * E[k])[None])[0]
        Hfd = (fpp - fpm - fmp + fmm) / (4 * hh * hh)
        assert np.allclose(Hlo, Hfd, atol=2e-5), (j, k, Hlo, Hfd)


def test_interval_hessian_encloses_sampled_hessians():
    spec = P.ModelSpec(P.MODEL_QUAD12, P.INTEG_RK4, 1, PARAMS)
    rng = np.random.default_rng(8)
    a = rng.uniform(-0.3, 0.3, 16)
    a[12] = 9.81
    s = rng.uniform(0.01, 0.05, 16)
    for j, k in [(3, 4), (4, 4), (5, 12), (9, 10)]:
        Hlo, Hhi = P.hessian_entry(spec, a - s, a + s, j, k)
        for _ in range(200):
            x = a + s * rng.uniform(-1, 1, 16)
            h1, _ = P.hessian_entry(spec, x, x, j, k)
            assert np.all(h1 >= Hlo - 1e-13) and np.all(h1 <= Hhi + 1e-13)


def _fd_vjp(spec, nom, rad, g_lo, g_hi, dirs, h=1e-6):
    def F(a, s):
        lo, hi, _ = P.pbh(spec, a[None], s[None])
        return g_hi @ hi[0] + g_lo @ lo[0]
    N = spec.N
    out, ok = np.zeros(len(dirs)), np.ones(len(dirs), bool)
    F0 = F(nom, rad)
    for i, d in enumerate(dirs):
        e = np.zeros(N)
        if d < N:
            e[d] = h * max(1.0, abs(nom[d]))
            fp, fm, st = F(nom + e, rad), F(nom - e, rad), e[d]
        else:
            e[d - N] = h * max(1.0, abs(rad[d - N]))
            fp, fm, st = F(nom, rad + e), F(nom, rad - e), e[d - N]
        out[i] = (fp - fm) / (2 * st)
        ok[i] = abs((fp - F0) - (F0 - fm)) <= 1e-3 * abs(fp - fm) + 1e-14
    return out, ok


@pytest.mark.parametrize("cfg,tiles", [(1, 6), (2, 2)])
def test_vjp_matches_central_differences(cfg, tiles):
    w = wl.make_config(cfg)
    spec = P.spec_from_workload(w)
    N, n = w.N, w.n
    nom, rad = w.nom.reshape(-1, N)[:tiles].astype(float), w.rad.reshape(-1, N)[:tiles].astype(float)
    g_lo, g_hi = w.g_lo.reshape(-1, n)[:tiles].astype(float), w.g_hi.reshape(-1, n)[:tiles].astype(float)
    G, st = P.pbh_vjp(spec, nom, rad, g_lo, g_hi)
    assert st == 0
    dirs = np.arange(2 * N)
    nok = 0
    for t in range(tiles):
        fd, ok = _fd_vjp(spec, nom[t], rad[t], g_lo[t], g_hi[t], dirs)
        scale = np.abs(fd).max()
        assert np.all(np.abs(G[t] - fd)[ok] <= 1e-5 * np.abs(fd)[ok] + 1e-6 * scale)
        nok += ok.sum()
    assert nok >= 0.8 * tiles * 2 * N


def test_vjp_small_chain_directions():
    w = wl.make_small_chain(2, 1, 1)
    spec = P.spec_from_workload(w)
    N, n = w.N, w.n
    nom, rad = w.nom.reshape(-1, N).astype(float), w.rad.reshape(-1, N).astype(float)
    g_lo, g_hi = w.g_lo.reshape(-1, n).astype(float), w.g_hi.reshape(-1, n).astype(float)
    dirs = np.array([0, 3, 4, 7, 12, 16, 24, 28, N + 0, N + 4, N + 13, N + 24, N + 30])
    G, st = P.pbh_vjp(spec, nom, rad, g_lo, g_hi, dirs)
    fd, ok = _fd_vjp(spec, nom[0], rad[0], g_lo[0], g_hi[0], dirs)
    scale = np.abs(fd).max()
    assert ok.sum() >= 8
    assert np.all(np.abs(G[0] - fd)[ok] <= 1e-5 * np.abs(fd)[ok] + 1e-6 * scale)


# ---------------------------------------------------------------- non-centred boxes (25a) PAPER.md:L272, reading R4
def _iv_mul(a, b):
    p = [a[0] * b[0], a[0] * b[1], a[1] * b[0], a[1] * b[1]]
    return min(p), max(p)


def _iv_sqr(a):
    lo = 0.0 if a[0] <= 0.0 <= a[1] else min(a[0] ** 2, a[1] ** 2)
    return lo, max(a[0] ** 2, a[1] ** 2)


def test_mu_zero_is_the_centred_bound_bit_for_bit():
    for cfg, tiles in ((1, 20), (2, 6)):
        w = wl.make_config(cfg)
        spec = P.spec_from_workload(w)
        nom, rad = w.nom.reshape(-1, w.N)[:tiles], w.rad.reshape(-1, w.N)[:tiles]
        for mode in (P.MODE_PATH, P.MODE_EXPAND):
            a = P.pbh(spec, nom, rad, mode)
            b = P.pbh(spec, nom, rad, mode, mu=np.zeros_like(nom))
            assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_mu_quadratic_map_closed_form():
    """Constant Hessian Q_l: R_l = sum_{j<k} Q_kj D_j D_k + 1/2 sum_k Q_kk D_k^2 with D = [mu - sigma, mu + sigma]
    (L164): every term's range written out by hand (corner products; the square's range on a general interval)."""
    rng = np.random.default_rng(11)
    n, N = 3, 5
    Q = rng.standard_normal((n, N, N))
    Q = Q + Q.transpose(0, 2, 1)
    C = rng.standard_normal((n, N))
    spec = P.ModelSpec(P.MODEL_QUADRATIC, params=PARAMS, Q=Q, C=C)
    nom, rad = rng.standard_normal((6, N)), rng.uniform(0.05, 0.5, (6, N))
    mu = rng.uniform(-0.6, 0.6, (6, N))               # some |mu| > sigma: a~ outside the box
    assert (np.abs(mu) > rad).any() and (np.abs(mu) < rad).any()
    lo, hi, st = P.pbh(spec, nom, rad, mu=mu)
    assert st == 0
    for t in range(6):
        D = [(mu[t, i] - rad[t, i], mu[t, i] + rad[t, i]) for i in range(N)]
        for l in range(n):
            up = dn = 0.0
            for j in range(N):
                for k in range(j + 1, N):
                    a, b = _iv_mul((Q[l, k, j], Q[l, k, j]), _iv_mul(D[j], D[k]))
                    dn += a
                    up += b
            for k in range(N):
                a, b = _iv_mul((Q[l, k, k], Q[l, k, k]), _iv_sqr(D[k]))
                dn += 0.5 * a
                up += 0.5 * b
            assert np.isclose(hi[t, l], up, rtol=1e-12, atol=1e-14) and np.isclose(lo[t, l], dn, rtol=1e-12, atol=1e-14)
        # constant Hessian: r = 1/2 d^T Q d exactly for a = a~ + d; vertices of the shifted box
        for s in itertools.product((-1.0, 1.0), repeat=N):
            d = mu[t] + rad[t] * np.array(s)
            r = 0.5 * np.einsum("lij,i,j->l", Q, d, d)
            assert np.all(r <= hi[t] + 1e-12) and np.all(r >= lo[t] - 1e-12)


@pytest.mark.parametrize("cfg,tiles", [(1, 8), (2, 4)])
def test_mu_soundness_off_centre(cfg, tiles):
    """Thm 1 with the nominal point off the box centre (and for some coordinates outside the box): the remainder
    about a~, r(a) = f(a) - f(a~) - J(a~)(a - a~) (10) L133, sampled on A = a~ + mu + [-sigma, sigma] and at all its
    vertices, lies in the enclosure; and the enclosure is not vacuous."""
    w = wl.make_config(cfg)
    spec = P.spec_from_workload(w)
    rng = np.random.default_rng(50 + cfg)
    N = w.N
    nom, rad = w.nom.reshape(-1, N)[:tiles].astype(float), w.rad.reshape(-1, N)[:tiles].astype(float)
    mu = rad * rng.uniform(-2.0, 2.0, rad.shape)
    lo, hi, st = P.pbh(spec, nom, rad, mu=mu)
    assert st == 0
    verts = np.array(list(itertools.product((-1.0, 1.0), repeat=N)))
    sharp = []
    for t in range(tiles):
        U = np.concatenate([rng.uniform(-1, 1, (100000, N)), verts])
        r = _true_r(spec, nom[t], nom[t][None] + mu[t][None] + U * rad[t][None])
        assert np.all(r.max(0) <= hi[t] + 1e-12) and np.all(r.min(0) >= lo[t] - 1e-12), t
        nz = (hi[t] - lo[t]) > 1e-9
        sharp.append(((r.max(0) - r.min(0))[nz] / (hi[t] - lo[t])[nz]).max())
    assert max(sharp) > 0.3


def test_mu_vjp_matches_central_differences():
    w = wl.make_config(2, B=1, T=3)
    spec = P.spec_from_workload(w)
    rng = np.random.default_rng(8)
    N, n = w.N, w.n
    nom, rad = w.nom.reshape(-1, N).astype(float), w.rad.reshape(-1, N).astype(float)
    mu = rad * rng.uniform(-1.5, 1.5, rad.shape)
    g_lo, g_hi = w.g_lo.reshape(-1, n).astype(float), w.g_hi.reshape(-1, n).astype(float)
    g, st = P.pbh_vjp(spec, nom, rad, g_lo, g_hi, mu=mu)
    assert st == 0 and g.shape == (3, 3 * N)

    def F(a, s, m):
        lo, hi, _ = P.pbh(spec, a, s, mu=m)
        return (g_hi * hi + g_lo * lo).sum(1)
    h, checked = 1e-6, 0
    F0 = F(nom, rad, mu)
    for d in range(3 * N):
        e = np.zeros((3, N))
        e[:, d % N] = h
        args = [(nom + e, rad, mu), (nom - e, rad, mu)] if d < N else \
               [(nom, rad + e, mu), (nom, rad - e, mu)] if d < 2 * N else [(nom, rad, mu + e), (nom, rad, mu - e)]
        fp, fm = F(*args[0]), F(*args[1])
        for t in range(3):
            if abs((fp[t] - F0[t]) - (F0[t] - fm[t])) > 1e-3 * abs(fp[t] - fm[t]) + 1e-14:
                continue                                   # kink
            fd = (fp[t] - fm[t]) / (2 * h)
            assert abs(fd - g[t, d]) <= 1e-5 * abs(fd) + 1e-6 * np.abs(g[t]).max(), (t, d)
            checked += 1
    assert checked >= 2 * N * 3
    assert np.abs(g[:, 2 * N:]).max() > 1e-3 * np.abs(g).max()      # mu does carry gradient


# ---------------------------------------------------------------- the paper's own systems (App. I)
SAT = [0.1, 1.0, 0.0, 5.0, 2.0, 1.0, 0.0, 0.0]        # dt; I_S = diag(5, 2, 1)
PQ = [0.05, 2.0576, 9.81, 0.01, 1.0, 1.0, 0.25, 0.0]   # dt; m, g, J, -, -, L


def test_satellite_constant_hessian_closed_form():
    """Euler satellite (36) L507-519 is a quadratic map: the Hessian is constant, so (15) has the closed form of
    SURVEY 8(c).6 with Q measured from the point function by second differences (exact for a quadratic)."""
    spec = P.ModelSpec(P.MODEL_SATELLITE, P.INTEG_EULER, 1, SAT)
    rng = np.random.default_rng(3)
    n, N = 7, 10
    a0 = rng.standard_normal(N)
    h = 0.5
    Q = np.zeros((n, N, N))
    E = np.eye(N) * h
    f0 = P.f(spec, a0[None])[0]
    for i in range(N):
        for k in range(N):
            Q[:, i, k] = (P.f(spec, (a0 + E[i] + E[k])[None])[0] - P.f(spec, (a0 + E[i])[None])[0]
                          - P.f(spec, (a0 + E[k])[None])[0] + f0) / h ** 2
    # quaternion kinematics: d^2 f_0 / d om_1 d q_1 = -dt/2; Euler's equations: d^2 f_4 / d om_2 d om_3 = dt (Jy - Jz)/Jx
    assert np.isclose(Q[0, 4, 1], -0.05) and np.isclose(Q[4, 5, 6], 0.1 * (2.0 - 1.0) / 5.0) and np.isclose(Q[6, 4, 5], 0.1 * 3.0)
    nom, rad = rng.standard_normal((4, N)), rng.uniform(0.01, 0.2, (4, N))
    lo, hi, st = P.pbh(spec, nom, rad)
    assert st == 0
    for t in range(4):
        s = rad[t]
        for l in range(n):
            off = sum(abs(Q[l, k, j]) * s[j] * s[k] for j in range(N) for k in range(j + 1, N))
            up = off + 0.5 * sum(max(Q[l, k, k], 0) * s[k] ** 2 for k in range(N))
            dn = -off + 0.5 * sum(min(Q[l, k, k], 0) * s[k] ** 2 for k in range(N))
            assert np.isclose(hi[t, l], up, rtol=1e-9, atol=1e-13) and np.isclose(lo[t, l], dn, rtol=1e-9, atol=1e-13)
    lo2, hi2, _ = P.pbh(spec, nom, rad, P.MODE_EXPAND)
    assert np.allclose(lo, lo2, rtol=1e-12, atol=1e-15) and np.allclose(hi, hi2, rtol=1e-12, atol=1e-15)


def test_planar_quadrotor_closed_form():
    """Planar quadrotor (37a) L521-528, Euler: only phi (index 2) meets u1, u2 (6, 7) non-linearly.
    f_3 = vx - dt (u1+u2) sin(phi)/m:  H_phiphi = dt (u1+u2) sin(phi)/m on A^(2) -- u PINNED (indices 6, 7 > 2) --,
    H_phi,u = -dt cos(phi)/m on A^(2);  f_4 likewise with (-cos, -sin).  All other outputs are linear."""
    spec = P.ModelSpec(P.MODEL_PLANAR_QUAD, P.INTEG_EULER, 1, PQ)
    rng = np.random.default_rng(4)
    dt, m = PQ[0], PQ[1]
    nom = np.concatenate([rng.uniform(-1, 1, (6, 2)), rng.uniform(0.2, 0.9, (6, 1)), rng.uniform(-1, 1, (6, 3)),
                          rng.uniform(8, 12, (6, 2))], 1)
    rad = rng.uniform(0.01, 0.1, (6, 8))
    lo, hi, st = P.pbh(spec, nom, rad)
    assert st == 0
    for t in range(6):
        ph, sp = nom[t, 2], rad[t, 2]
        S = (np.sin(ph - sp), np.sin(ph + sp))           # 0 < phi - sp, phi + sp < pi/2: both monotone
        Cc = (np.cos(ph + sp), np.cos(ph - sp))
        ub = nom[t, 6] + nom[t, 7]
        D = lambda i: (-rad[t, i], rad[t, i])
        for out, hpp, hpu in ((3, (dt / m * ub * S[0], dt / m * ub * S[1]), (-dt / m * Cc[1], -dt / m * Cc[0])),
                              (4, (-dt / m * ub * Cc[1], -dt / m * ub * Cc[0]), (-dt / m * S[1], -dt / m * S[0]))):
            a = _iv_mul(hpp, _iv_sqr(D(2)))
            dn, up = 0.5 * a[0], 0.5 * a[1]
            for u in (6, 7):
                b = _iv_mul(hpu, _iv_mul(D(2), D(u)))
                dn += b[0]
                up += b[1]
            assert np.isclose(lo[t, out], dn, rtol=1e-12, atol=1e-16) and np.isclose(hi[t, out], up, rtol=1e-12, atol=1e-16)
        for out in (0, 1, 2, 5):
            assert lo[t, out] == 0.0 and hi[t, out] == 0.0
    # soundness on one tile
    U = np.concatenate([rng.uniform(-1, 1, (100000, 8)), np.array(list(itertools.product((-1.0, 1.0), repeat=8)))])
    r = _true_r(spec, nom[0], nom[0][None] + U * rad[0][None])
    assert np.all(r.max(0) <= hi[0] + 1e-12) and np.all(r.min(0) >= lo[0] - 1e-12)


def test_centroid_coupled_quadrotors():
    """Coupled quadrotors (39)-(42) L540-558, forward Euler: the centroid spring-damper is linear, so it moves the Jacobian
    but not the Hessian -- the enclosure of every unit equals that of the uncoupled quad12 on the same inputs -- and the
    bound stays sound for the coupled map."""
    U = 3
    w = wl.make_paper_system(f"quadcentroid{U}", 1, 2)
    spec = P.spec_from_workload(w)
    nom, rad = w.nom.reshape(-1, w.N).astype(float), w.rad.reshape(-1, w.N).astype(float)
    lo, hi, st = P.pbh(spec, nom, rad)
    assert st == 0
    q = P.ModelSpec(P.MODEL_QUAD12, P.INTEG_EULER, 1, spec.params)
    for i in range(U):
        sel = np.r_[12 * i:12 * i + 12, 12 * U + 4 * i:12 * U + 4 * i + 4]
        qlo, qhi, _ = P.pbh(q, nom[:, sel], rad[:, sel])
        assert np.allclose(lo[:, 12 * i:12 * i + 12], qlo, rtol=1e-13, atol=1e-18)
        assert np.allclose(hi[:, 12 * i:12 * i + 12], qhi, rtol=1e-13, atol=1e-18)
    # the coupling is there: unit 0's velocity row of J sees unit 1's position with -alpha U (-1/U) dt = alpha dt
    J = P.jac(spec, nom[0])
    assert np.isclose(J[6, 12], 0.75 * 0.05) and np.isclose(J[6, 0], -0.75 * U * (1 - 1 / U) * 0.05)
    rng = np.random.default_rng(9)
    X = nom[0][None] + rng.uniform(-1, 1, (50000, w.N)) * rad[0][None]
    r = _true_r(spec, nom[0], X)
    assert np.all(r.max(0) <= hi[0] + 1e-12) and np.all(r.min(0) >= lo[0] - 1e-12)
