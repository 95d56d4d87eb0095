"""Pins for oracle/nn_oracle.py (CPU only).  Every check here compares the oracle
with something the paper or the mathematics fixes independently of it:
exact piecewise-linear enumeration, sampled/vertex soundness (Thm 2/3,
PAPER.md:L196-214), the closed-form box maximum of an affine map,
validity of each scalar relaxation on a dense grid, and central differences."""
import itertools

import numpy as np
import pytest

from oracle import nn_oracle as O


def _net(rng, dims, scale=1.0):
    Ws = [rng.standard_normal((dims[i + 1], dims[i])) * scale * np.sqrt(2.0 / (dims[i] + dims[i + 1]))
          for i in range(len(dims) - 1)]
    bs = [rng.uniform(-0.1, 0.1, dims[i + 1]) for i in range(len(dims) - 1)]
    return Ws, bs


def _true_r(Ws, bs, act, a0, X):
    zs, p, J = O.nominal(Ws, bs, act, a0)
    return np.array([O.mlp_eval(Ws, bs, act, x) - p - J @ (x - a0) for x in X])


def _vertices(a0, sig):
    return np.array([a0 + sig * np.array(s) for s in itertools.product((-1.0, 1.0), repeat=len(a0))])


# ---------------------------------------------------------------- relaxations
@pytest.mark.parametrize("seed", range(3))
def test_tanh_relaxation_valid_and_touching(seed):
    rng = np.random.default_rng(seed)
    for _ in range(200):
        l = rng.uniform(-3, 3)
        u = l + rng.uniform(1e-3, 4)
        kU, bU, kL, bL, aux = O.relax_tanh_scalar(l, u)
        z = np.linspace(l, u, 2001)
        up = kU * z + bU - np.tanh(z)
        lo = np.tanh(z) - (kL * z + bL)
        assert up.min() >= -1e-12 and lo.min() >= -1e-12, (l, u, aux)
        # each line touches the curve somewhere on [l,u] (it is a tangent or a chord)
        assert up.min() <= 1e-6 and lo.min() <= 1e-6, (l, u, aux)


def test_relu_relaxation_cases():
    assert O.relax_relu_scalar(-2.0, -1.0)[:4] == (0.0, 0.0, 0.0, 0.0)
    assert O.relax_relu_scalar(0.5, 1.0)[:4] == (1.0, 0.0, 1.0, 0.0)
    kU, bU, kL, bL, _ = O.relax_relu_scalar(-1.0, 3.0)
    assert np.isclose(kU, 0.75) and np.isclose(bU, 0.75) and kL == 1.0 and bL == 0.0
    assert O.relax_relu_scalar(-3.0, 1.0)[2] == 0.0
    assert O.relax_relu_scalar(-1.0, 1.0)[2] == 0.0          # tie -> 0
    for l, u in [(-1.0, 3.0), (-3.0, 1.0), (-1.0, 1.0)]:
        kU, bU, kL, bL, _ = O.relax_relu_scalar(l, u)
        z = np.linspace(l, u, 1001)
        assert (kU * z + bU - np.maximum(z, 0) >= -1e-15).all()
        assert (np.maximum(z, 0) - kL * z - bL >= -1e-15).all()


# ---------------------------------------------------------------- zero cases
def test_stable_relu_network_gives_zero_bound():
    # large positive/negative biases => every neuron stable on the box => p is affine
    rng = np.random.default_rng(1)
    Ws, bs = _net(rng, [5, 8, 8, 3])
    bs[0] = np.where(rng.random(8) < 0.5, 50.0, -50.0)
    bs[1] = np.where(rng.random(8) < 0.5, 50.0, -50.0)
    a0 = rng.standard_normal(5)
    sig = rng.uniform(0.1, 0.5, 5)
    out = O.crown_forward(Ws, bs, O.ACT_RELU, a0, sig)
    assert np.abs(out["r_lo"]).max() < 1e-12 and np.abs(out["r_hi"]).max() < 1e-12


@pytest.mark.parametrize("act", [O.ACT_RELU, O.ACT_TANH])
def test_zero_radius_gives_zero_bound(act):
    rng = np.random.default_rng(2)
    Ws, bs = _net(rng, [4, 9, 7, 3])
    a0 = rng.standard_normal(4)
    out = O.crown_forward(Ws, bs, act, a0, np.zeros(4))
    assert np.abs(out["r_lo"]).max() < 1e-12 and np.abs(out["r_hi"]).max() < 1e-12


def test_tanh_bound_shrinks_quadratically():
    rng = np.random.default_rng(3)
    Ws, bs = _net(rng, [4, 9, 7, 3])
    a0 = rng.standard_normal(4)
    sig = rng.uniform(0.5, 1.0, 4)
    w1 = O.crown_forward(Ws, bs, O.ACT_TANH, a0, 1e-3 * sig)
    w2 = O.crown_forward(Ws, bs, O.ACT_TANH, a0, 2e-3 * sig)
    ratio = (w2["r_hi"] - w2["r_lo"]) / (w1["r_hi"] - w1["r_lo"])
    assert np.all(np.abs(ratio - 4.0) < 0.05), ratio


# ---------------------------------------------------------------- exact enumeration
def _exact_range_1hidden_relu(Ws, bs, a0, sig):
    """r is piecewise linear: its extrema over the box are attained at vertices of
    the arrangement {neuron hyperplanes} u {box faces}.  Enumerate them all."""
    d = len(a0)
    W1, b1 = Ws[0], bs[0]
    planes = [(W1[k], -b1[k]) for k in range(W1.shape[0])]
    for i in range(d):
        e = np.zeros(d)
        e[i] = 1.0
        planes.append((e, a0[i] - sig[i]))
        planes.append((e, a0[i] + sig[i]))
    pts = []
    for combo in itertools.combinations(range(len(planes)), d):
        A = np.array([planes[c][0] for c in combo])
        rhs = np.array([planes[c][1] for c in combo])
        if abs(np.linalg.det(A)) < 1e-12:
            continue
        x = np.linalg.solve(A, rhs)
        if np.all(np.abs(x - a0) <= sig + 1e-12):
            pts.append(np.clip(x, a0 - sig, a0 + sig))
    R = _true_r(Ws, bs, O.ACT_RELU, a0, np.array(pts))
    return R.min(0), R.max(0)


@pytest.mark.parametrize("d,H,seed", [(1, 4, 0), (2, 5, 1), (3, 5, 2), (4, 4, 3)])
def test_encloses_exact_range_1hidden_relu(d, H, seed):
    rng = np.random.default_rng(100 + seed)
    Ws, bs = _net(rng, [d, H, 3], scale=2.0)
    a0 = rng.standard_normal(d) * 0.3
    sig = rng.uniform(0.2, 0.6, d)
    lo, hi = _exact_range_1hidden_relu(Ws, bs, a0, sig)
    out = O.crown_forward(Ws, bs, O.ACT_RELU, a0, sig)
    assert np.all(out["r_lo"] <= lo + 1e-12) and np.all(out["r_hi"] >= hi - 1e-12)
    # not vacuous: within a small factor of the exact width on these tiny nets
    assert np.all((out["r_hi"] - out["r_lo"]) <= 6.0 * (hi - lo) + 1e-9)


def test_exact_when_single_unstable_neuron_1d():
    # 1-D input, one unstable neuron with output weight w: the chord touches the
    # ReLU at both interval ends, so the side that uses the chord is exact.
    W1 = np.array([[1.0], [1.0]])
    b1 = np.array([0.2, 5.0])              # neuron 0 unstable on [-1,1], neuron 1 stable-on
    for w in (+1.5, -0.7):
        Ws = [W1, np.array([[w, 0.3]])]
        bs = [b1, np.array([0.1])]
        a0, sig = np.array([0.1]), np.array([1.0])
        lo, hi = _exact_range_1hidden_relu(Ws, bs, a0, sig)
        out = O.crown_forward(Ws, bs, O.ACT_RELU, a0, sig)
        if w > 0:
            assert np.isclose(out["r_hi"][0], hi[0], atol=1e-12)
            assert out["r_lo"][0] <= lo[0] + 1e-12
        else:
            assert np.isclose(out["r_lo"][0], lo[0], atol=1e-12)
            assert out["r_hi"][0] >= hi[0] - 1e-12


# ---------------------------------------------------------------- soundness
@pytest.mark.parametrize("act,dims,seed", [(O.ACT_RELU, [6, 12, 12, 12, 4], 0), (O.ACT_TANH, [6, 12, 12, 12, 4], 1),
                                           (O.ACT_TANH, [5, 16, 16, 16, 16, 3], 2), (O.ACT_RELU, [8, 10, 10, 5], 3)])
def test_soundness_samples_vertices_hidden(act, dims, seed):
    rng = np.random.default_rng(200 + seed)
    Ws, bs = _net(rng, dims, scale=1.5)
    a0 = rng.standard_normal(dims[0])
    sig = rng.uniform(0.05, 0.3, dims[0])
    out = O.crown_forward(Ws, bs, act, a0, sig)
    X = np.concatenate([a0 + sig * rng.uniform(-1, 1, (100000 // 4, dims[0])), _vertices(a0, sig)])
    R = _true_r(Ws, bs, act, a0, X)
    assert np.all(R.min(0) >= out["r_lo"] - 1e-12) and np.all(R.max(0) <= out["r_hi"] + 1e-12)
    for x in X[::97]:
        for z, l, u in zip(O.mlp_hidden(Ws, bs, act, x), out["ls"], out["us"]):
            assert np.all(z >= l - 1e-12) and np.all(z <= u + 1e-12)
    # Thm 2 itself: W_lo a + b_lo <= p(a) <= W_up a + b_up
    for x in X[::53]:
        p = O.mlp_eval(Ws, bs, act, x)
        assert np.all(out["W_lo"] @ x + out["b_lo"] <= p + 1e-12)
        assert np.all(out["W_up"] @ x + out["b_up"] >= p - 1e-12)


def test_concretisation_is_box_max_of_eq20():
    # (21): r_hi_i = max over the box of the affine r_up(a) of (20); brute force on vertices
    rng = np.random.default_rng(5)
    Ws, bs = _net(rng, [5, 9, 9, 4], scale=1.5)
    a0 = rng.standard_normal(5)
    sig = rng.uniform(0.05, 0.3, 5)
    out = O.crown_forward(Ws, bs, O.ACT_TANH, a0, sig)
    V = _vertices(a0, sig)
    J, p = out["J"], out["p"]
    up = np.array([(out["W_up"] - J) @ v + J @ a0 - p + out["b_up"] for v in V]).max(0)
    lo = np.array([(out["W_lo"] - J) @ v + J @ a0 - p + out["b_lo"] for v in V]).min(0)
    assert np.allclose(up, out["r_hi"], rtol=0, atol=1e-12)
    assert np.allclose(lo, out["r_lo"], rtol=0, atol=1e-12)


def test_jacobian_matches_finite_differences():
    rng = np.random.default_rng(6)
    Ws, bs = _net(rng, [5, 9, 9, 4])
    a0 = rng.standard_normal(5)
    _, _, J = O.nominal(Ws, bs, O.ACT_TANH, a0)
    h = 1e-6
    Jfd = np.array([(O.mlp_eval(Ws, bs, O.ACT_TANH, a0 + h * e) - O.mlp_eval(Ws, bs, O.ACT_TANH, a0 - h * e)) / (2 * h)
                    for e in np.eye(5)]).T
    assert np.allclose(J, Jfd, atol=1e-8)


def test_given_jacobian_is_used():
    # Thm 3 holds for any J: with J' = J + E the bound must enclose r computed with J'
    rng = np.random.default_rng(7)
    Ws, bs = _net(rng, [4, 8, 8, 3])
    a0 = rng.standard_normal(4)
    sig = rng.uniform(0.05, 0.2, 4)
    _, p, J = O.nominal(Ws, bs, O.ACT_TANH, a0)
    J2 = J + 0.1 * rng.standard_normal(J.shape)
    out = O.crown_forward(Ws, bs, O.ACT_TANH, a0, sig, J_given=J2)
    X = np.concatenate([a0 + sig * rng.uniform(-1, 1, (5000, 4)), _vertices(a0, sig)])
    R = np.array([O.mlp_eval(Ws, bs, O.ACT_TANH, x) - p - J2 @ (x - a0) for x in X])
    assert np.all(R.min(0) >= out["r_lo"] - 1e-12) and np.all(R.max(0) <= out["r_hi"] + 1e-12)


# ---------------------------------------------------------------- VJP
def _fd_grad(Ws, bs, act, a0, sig, g_lo, g_hi, h=1e-6):
    def F(a, s):
        f = O.crown_forward(Ws, bs, act, a, s)
        return g_hi @ f["r_hi"] + g_lo @ f["r_lo"]
    N = len(a0)
    gn, gr, ok_n, ok_r = np.zeros(N), np.zeros(N), np.ones(N, bool), np.ones(N, bool)
    F0 = F(a0, sig)
    for i in range(N):
        e = np.zeros(N)
        e[i] = h * max(1.0, abs(a0[i]))
        fp, fm = F(a0 + e, sig), F(a0 - e, sig)
        gn[i] = (fp - fm) / (2 * e[i])
        ok_n[i] = abs((fp - F0) - (F0 - fm)) <= 1e-3 * abs(fp - fm) + 1e-12      # kink filter
        e[i] = h * max(1.0, abs(sig[i]))
        fp, fm = F(a0, sig + e), F(a0, sig - e)
        gr[i] = (fp - fm) / (2 * e[i])
        ok_r[i] = abs((fp - F0) - (F0 - fm)) <= 1e-3 * abs(fp - fm) + 1e-12
    return gn, gr, ok_n, ok_r


@pytest.mark.parametrize("act,dims,seed", [(O.ACT_RELU, [6, 10, 10, 10, 4], 0), (O.ACT_TANH, [6, 10, 10, 10, 4], 1),
                                           (O.ACT_TANH, [3, 7, 5, 2], 2), (O.ACT_TANH, [5, 8, 8, 8, 8, 3], 3),
                                           (O.ACT_RELU, [4, 9, 9, 3], 4)])
def test_vjp_matches_central_differences(act, dims, seed):
    rng = np.random.default_rng(300 + seed)
    Ws, bs = _net(rng, dims, scale=1.5)
    a0 = rng.standard_normal(dims[0])
    sig = rng.uniform(0.05, 0.3, dims[0])
    g_lo, g_hi = rng.standard_normal(dims[-1]), rng.standard_normal(dims[-1])
    gn, gr = O.crown_vjp(Ws, bs, act, a0, sig, g_lo, g_hi)
    fn, fr, ok_n, ok_r = _fd_grad(Ws, bs, act, a0, sig, g_lo, g_hi)
    assert ok_n.sum() + ok_r.sum() >= dims[0]            # most points are not at a kink
    scale = max(np.abs(fn).max(), np.abs(fr).max())
    assert np.all(np.abs(gn - fn)[ok_n] <= 1e-6 * scale + 1e-5 * np.abs(fn)[ok_n])
    assert np.all(np.abs(gr - fr)[ok_r] <= 1e-6 * scale + 1e-5 * np.abs(fr)[ok_r])


def test_vjp_random_directions_config3_shape():
    # config-3 architecture (24 -> 128x3 -> 20, ReLU); directional derivatives
    from paper_2607_01203_b200 import workloads as wl
    w = wl.make_config(3, B=1, T=2)
    Ws = [W.astype(np.float64) for W in w.mlp.W]
    bs = [b.astype(np.float64) for b in w.mlp.b]
    rng = np.random.default_rng(9)
    a0, sig = w.nom[0, 0].astype(np.float64), w.rad[0, 0].astype(np.float64)
    g_lo, g_hi = w.g_lo[0, 0].astype(np.float64), w.g_hi[0, 0].astype(np.float64)
    gn, gr = O.crown_vjp(Ws, bs, O.ACT_RELU, a0, sig, g_lo, g_hi)

    def F(a, s):
        f = O.crown_forward(Ws, bs, O.ACT_RELU, a, s)
        return g_hi @ f["r_hi"] + g_lo @ f["r_lo"]
    h, good = 1e-7, 0
    for _ in range(32):
        dn, dr = rng.standard_normal(24), rng.standard_normal(24)
        F0, fp, fm = F(a0, sig), F(a0 + h * dn, sig + h * dr), F(a0 - h * dn, sig - h * dr)
        if abs((fp - F0) - (F0 - fm)) > 1e-3 * abs(fp - fm):
            continue                                     # crossed a ReLU switch
        good += 1
        assert np.isclose((fp - fm) / (2 * h), gn @ dn + gr @ dr, rtol=1e-5, atol=1e-7)
    assert good >= 16


def test_vjp_through_degenerate_tanh_neurons():
    """Pin of relax_vjp_scalar's "degenerate" branch (u - l < 1e-12, reading R9): inputs 0..2 have
    zero radius and feed, alone, hidden neurons 0..3 of layer 1, which feed, alone, neurons 0..2 of
    layer 2 -- those neurons' pre-activation intervals are points, in both layers, and the output
    reads them next to ordinary neurons.  Central differences in every direction that keeps the
    structure (all nominal coordinates; the radii of the non-degenerate inputs) must match, and the
    branch itself must return (numerically) nothing: at l = u = d the tangent's parameter adjoints
    cancel, t''(d)(k_bar - d b_bar) = 0, and the widening term carries the factor (u - l)."""
    rng = np.random.default_rng(77)
    dims = [6, 9, 8, 7, 3]
    Ws, bs = _net(rng, dims, scale=1.5)
    Ws[0][:4, 3:] = 0.0          # layer-1 neurons 0..3 see only the zero-radius inputs
    Ws[1][:3, 4:] = 0.0          # layer-2 neurons 0..2 see only those
    a0 = rng.standard_normal(6)
    sig = np.concatenate([np.zeros(3), rng.uniform(0.05, 0.3, 3)])
    g_lo, g_hi = rng.standard_normal(3), rng.standard_normal(3)
    fw = O.crown_forward(Ws, bs, O.ACT_TANH, a0, sig)
    kinds = [[a[0] for a in r[4]] for r in fw["relaxs"]]
    assert kinds[0][:4] == ["degenerate"] * 4 and kinds[1][:3] == ["degenerate"] * 3
    assert "degenerate" not in kinds[0][4:] + kinds[1][3:] + kinds[2]
    # the branch's own output: zero to rounding, for arbitrary parameter cotangents consistent with l = u = d
    for l in (-0.7, 0.0, 1.3):
        aux = O.relax_tanh_scalar(l, l)[4]
        yb, lam = 0.83, -1.9                       # k_bar = y_bar * lam * z, b_bar = y_bar * lam at z = d
        lb, ub = O.relax_vjp_scalar(O.ACT_TANH, l, l, aux, yb * lam * l, yb * lam, 0.3 * yb * lam * l, 0.3 * yb * lam)
        assert abs(lb) < 1e-12 and abs(ub) < 1e-12
    gn, gr = O.crown_vjp(Ws, bs, O.ACT_TANH, a0, sig, g_lo, g_hi)

    def F(a, s):
        f = O.crown_forward(Ws, bs, O.ACT_TANH, a, s)
        return g_hi @ f["r_hi"] + g_lo @ f["r_lo"]
    scale = max(np.abs(gn).max(), np.abs(gr).max())
    checked = 0
    for i in range(6):
        for is_rad in (False, True):
            if is_rad and i < 3:
                continue                             # sigma = 0: one-sided, unpinned
            e = np.zeros(6)
            e[i] = 1e-6
            fp, fm, F0 = (F(a0, sig + e), F(a0, sig - e), F(a0, sig)) if is_rad else (F(a0 + e, sig), F(a0 - e, sig), F(a0, sig))
            if abs((fp - F0) - (F0 - fm)) > 1e-3 * abs(fp - fm) + 1e-12:
                continue                             # kink
            g = (gr if is_rad else gn)[i]
            assert abs((fp - fm) / 2e-6 - g) <= 1e-6 * scale + 1e-5 * abs(g), (i, is_rad)
            checked += 1
    assert checked >= 7
    assert np.abs(gn[:3]).max() > 1e-3 * scale       # the zero-radius coordinates do carry gradient


# ---------------------------------------------------------------- CROWN-IBP (hidden = "ibp"; PAPER.md:L194-196 leaves the variant open)
@pytest.mark.parametrize("act,dims,seed", [(O.ACT_RELU, [6, 12, 12, 12, 4], 0), (O.ACT_TANH, [5, 16, 16, 16, 16, 3], 2)])
def test_crown_ibp_sound_and_looser_hidden_bounds(act, dims, seed):
    rng = np.random.default_rng(400 + seed)
    Ws, bs = _net(rng, dims, scale=1.5)
    a0 = rng.standard_normal(dims[0])
    sig = rng.uniform(0.05, 0.3, dims[0])
    out = O.crown_forward(Ws, bs, act, a0, sig, hidden="ibp")
    full = O.crown_forward(Ws, bs, act, a0, sig)
    X = np.concatenate([a0 + sig * rng.uniform(-1, 1, (25000, dims[0])), _vertices(a0, sig)])
    R = _true_r(Ws, bs, act, a0, X)
    assert np.all(R.min(0) >= out["r_lo"] - 1e-12) and np.all(R.max(0) <= out["r_hi"] + 1e-12)
    for x in X[::97]:
        for z, l, u in zip(O.mlp_hidden(Ws, bs, act, x), out["ls"], out["us"]):
            assert np.all(z >= l - 1e-12) and np.all(z <= u + 1e-12)
    # layer 1 is the same; layer 2 by interval arithmetic is the textbook product [W][a] + b
    assert np.array_equal(out["ls"][0], full["ls"][0]) and np.array_equal(out["us"][0], full["us"][0])
    a_lo, a_hi = O.phi(act, out["ls"][0]), O.phi(act, out["us"][0])
    c, r = 0.5 * (a_hi + a_lo), 0.5 * (a_hi - a_lo)
    assert np.allclose(out["ls"][1], Ws[1] @ c - np.abs(Ws[1]) @ r + bs[1], atol=1e-13)
    assert np.allclose(out["us"][1], Ws[1] @ c + np.abs(Ws[1]) @ r + bs[1], atol=1e-13)
    # the interval bounds of the deeper layers are looser than full CROWN's on these nets, and so is the final bound
    assert (out["us"][-1] - out["ls"][-1]).sum() > (full["us"][-1] - full["ls"][-1]).sum()
    assert (out["r_hi"] - out["r_lo"]).sum() >= (full["r_hi"] - full["r_lo"]).sum() - 1e-12


def test_crown_ibp_equals_crown_with_one_hidden_layer():
    rng = np.random.default_rng(5)
    Ws, bs = _net(rng, [5, 9, 3])
    a0, sig = rng.standard_normal(5), rng.uniform(0.05, 0.3, 5)
    a, b = O.crown_forward(Ws, bs, O.ACT_TANH, a0, sig, hidden="ibp"), O.crown_forward(Ws, bs, O.ACT_TANH, a0, sig)
    assert np.array_equal(a["r_lo"], b["r_lo"]) and np.array_equal(a["r_hi"], b["r_hi"])


@pytest.mark.parametrize("act,dims,seed", [(O.ACT_TANH, [6, 10, 10, 10, 4], 1), (O.ACT_RELU, [6, 10, 10, 10, 4], 0), (O.ACT_TANH, [5, 8, 8, 8, 8, 3], 3)])
def test_crown_ibp_vjp_matches_central_differences(act, dims, seed):
    rng = np.random.default_rng(500 + seed)
    Ws, bs = _net(rng, dims, scale=1.5)
    a0 = rng.standard_normal(dims[0])
    sig = rng.uniform(0.05, 0.3, dims[0])
    g_lo, g_hi = rng.standard_normal(dims[-1]), rng.standard_normal(dims[-1])
    gn, gr = O.crown_vjp(Ws, bs, act, a0, sig, g_lo, g_hi, hidden="ibp")

    def F(a, s):
        f = O.crown_forward(Ws, bs, act, a, s, hidden="ibp")
        return g_hi @ f["r_hi"] + g_lo @ f["r_lo"]
    N, h, ok = dims[0], 1e-6, 0
    F0 = F(a0, sig)
    scale = max(np.abs(gn).max(), np.abs(gr).max())
    for i in range(2 * N):
        e = np.zeros(N)
        e[i % N] = h
        fp, fm = (F(a0 + e, sig), F(a0 - e, sig)) if i < N else (F(a0, sig + e), F(a0, sig - e))
        if abs((fp - F0) - (F0 - fm)) > 1e-3 * abs(fp - fm) + 1e-12:
            continue
        g = gn[i] if i < N else gr[i - N]
        assert abs((fp - fm) / (2 * h) - g) <= 1e-6 * scale + 1e-5 * abs(g), i
        ok += 1
    assert ok >= N


# ---------------------------------------------------------------- non-centred boxes (25a) PAPER.md:L272 on the NN path
def _true_r_about(Ws, bs, act, a0, X):
    """remainder (10) about the nominal point a0 at the points X (which need not surround a0)"""
    return _true_r(Ws, bs, act, a0, X)


@pytest.mark.parametrize("act,dims,seed,hidden", [(O.ACT_RELU, [6, 12, 12, 12, 4], 0, "crown"), (O.ACT_TANH, [6, 12, 12, 12, 4], 1, "crown"),
                                                  (O.ACT_TANH, [5, 16, 16, 16, 16, 3], 2, "ibp"), (O.ACT_RELU, [8, 10, 10, 5], 3, "crown")])
def test_mu_soundness_and_reduction(act, dims, seed, hidden):
    rng = np.random.default_rng(600 + seed)
    Ws, bs = _net(rng, dims, scale=1.5)
    a0 = rng.standard_normal(dims[0])
    sig = rng.uniform(0.05, 0.3, dims[0])
    mu = sig * rng.uniform(-2.0, 2.0, dims[0])                 # some |mu| > sigma: the nominal point outside the box
    assert (np.abs(mu) > sig).any()
    z = O.crown_forward(Ws, bs, act, a0, sig, hidden=hidden, mu=np.zeros_like(a0))
    c = O.crown_forward(Ws, bs, act, a0, sig, hidden=hidden)
    assert np.allclose(z["r_lo"], c["r_lo"], rtol=0, atol=1e-13) and np.allclose(z["r_hi"], c["r_hi"], rtol=0, atol=1e-13)
    out = O.crown_forward(Ws, bs, act, a0, sig, hidden=hidden, mu=mu)
    X = np.concatenate([a0 + mu + sig * rng.uniform(-1, 1, (25000, dims[0])), _vertices(a0 + mu, sig)])
    R = _true_r_about(Ws, bs, act, a0, X)
    assert np.all(R.min(0) >= out["r_lo"] - 1e-12) and np.all(R.max(0) <= out["r_hi"] + 1e-12)
    for x in X[::97]:
        for zz, l, u in zip(O.mlp_hidden(Ws, bs, act, x), out["ls"], out["us"]):
            assert np.all(zz >= l - 1e-12) and np.all(zz <= u + 1e-12)
    # not vacuous: the sampled range fills a fair part of the enclosure on these small nets
    if hidden == "crown":
        assert ((R.max(0) - R.min(0)) / (out["r_hi"] - out["r_lo"])).max() > 0.2


def test_mu_exact_range_1hidden_relu():
    """1-hidden-layer ReLU net, 2 inputs, offset box: r about a0 is piecewise linear on the box c +- sigma; enumerate the
    arrangement vertices (test helper above works on any box: it takes the box centre)."""
    rng = np.random.default_rng(31)
    Ws, bs = _net(rng, [2, 5, 3], scale=2.0)
    a0 = rng.standard_normal(2) * 0.3
    sig = rng.uniform(0.2, 0.6, 2)
    mu = np.array([0.5, -0.7]) * sig * 2
    c = a0 + mu
    # vertices of the arrangement inside the offset box, remainder measured about a0
    planes = [(Ws[0][k], -bs[0][k]) for k in range(5)]
    for i in range(2):
        e = np.zeros(2); e[i] = 1.0
        planes += [(e, c[i] - sig[i]), (e, c[i] + sig[i])]
    pts = []
    for i, j in itertools.combinations(range(len(planes)), 2):
        A = np.array([planes[i][0], planes[j][0]]); rhs = np.array([planes[i][1], planes[j][1]])
        if abs(np.linalg.det(A)) < 1e-12:
            continue
        x = np.linalg.solve(A, rhs)
        if np.all(np.abs(x - c) <= sig + 1e-12):
            pts.append(np.clip(x, c - sig, c + sig))
    R = _true_r(Ws, bs, O.ACT_RELU, a0, np.array(pts))
    out = O.crown_forward(Ws, bs, O.ACT_RELU, a0, sig, mu=mu)
    assert np.all(out["r_lo"] <= R.min(0) + 1e-12) and np.all(out["r_hi"] >= R.max(0) - 1e-12)
    assert np.all((out["r_hi"] - out["r_lo"]) <= 8.0 * (R.max(0) - R.min(0)) + 1e-9)


@pytest.mark.parametrize("act,dims,seed,hidden", [(O.ACT_TANH, [6, 10, 10, 10, 4], 1, "crown"), (O.ACT_RELU, [6, 10, 10, 10, 4], 0, "crown"),
                                                  (O.ACT_TANH, [5, 8, 8, 8, 8, 3], 3, "ibp")])
def test_mu_vjp_matches_central_differences(act, dims, seed, hidden):
    rng = np.random.default_rng(700 + seed)
    Ws, bs = _net(rng, dims, scale=1.5)
    N = dims[0]
    a0 = rng.standard_normal(N)
    sig = rng.uniform(0.05, 0.3, N)
    mu = sig * rng.uniform(-1.5, 1.5, N)
    g_lo, g_hi = rng.standard_normal(dims[-1]), rng.standard_normal(dims[-1])
    gn, gr, gm = O.crown_vjp(Ws, bs, act, a0, sig, g_lo, g_hi, hidden=hidden, mu=mu)
    g = np.concatenate([gn, gr, gm])

    def F(a, s, m):
        f = O.crown_forward(Ws, bs, act, a, s, hidden=hidden, mu=m)
        return g_hi @ f["r_hi"] + g_lo @ f["r_lo"]
    h, ok = 1e-6, 0
    F0 = F(a0, sig, mu)
    scale = np.abs(g).max()
    for i in range(3 * N):
        e = np.zeros(N)
        e[i % N] = h
        args = [(a0 + e, sig, mu), (a0 - e, sig, mu)] if i < N else [(a0, sig + e, mu), (a0, sig - e, mu)] if i < 2 * N else \
               [(a0, sig, mu + e), (a0, sig, mu - e)]
        fp, fm = F(*args[0]), F(*args[1])
        if abs((fp - F0) - (F0 - fm)) > 1e-3 * abs(fp - fm) + 1e-12:
            continue
        assert abs((fp - fm) / (2 * h) - g[i]) <= 1e-6 * scale + 1e-5 * abs(g[i]), i
        ok += 1
    assert ok >= 2 * N


# ---------------------------------------------------------------- optimisable lower slopes (alpha-CROWN)
def test_alpha_any_slope_is_sound_and_default_reproduces_crown():
    rng = np.random.default_rng(800)
    dims = [4, 10, 10, 10, 3]
    Ws, bs = _net(rng, dims, scale=2.0)
    a0 = rng.standard_normal(4) * 0.3
    sig = rng.uniform(0.2, 0.5, 4)
    base = O.crown_forward(Ws, bs, O.ACT_RELU, a0, sig)
    assert sum((np.array([a[0] for a in r[4]]) == "unstable").sum() for r in base["relaxs"]) >= 6
    d = O.crown_forward(Ws, bs, O.ACT_RELU, a0, sig, alphas=O.default_alphas(Ws, bs, a0, sig))
    assert np.array_equal(d["r_lo"], base["r_lo"]) and np.array_equal(d["r_hi"], base["r_hi"])
    X = np.concatenate([a0 + sig * rng.uniform(-1, 1, (20000, 4)), _vertices(a0, sig)])
    R = _true_r(Ws, bs, O.ACT_RELU, a0, X)
    for trial in range(5):
        alphas = [rng.uniform(0, 1, W.shape[0]) for W in Ws[:-1]]
        out = O.crown_forward(Ws, bs, O.ACT_RELU, a0, sig, alphas=alphas)
        assert np.all(R.min(0) >= out["r_lo"] - 1e-12) and np.all(R.max(0) <= out["r_hi"] + 1e-12)
        for x in X[::211]:
            for z, l, u in zip(O.mlp_hidden(Ws, bs, O.ACT_RELU, x), out["ls"], out["us"]):
                assert np.all(z >= l - 1e-12) and np.all(z <= u + 1e-12)


def test_alpha_gradient_and_refinement():
    rng = np.random.default_rng(801)
    dims = [4, 10, 10, 10, 3]
    Ws, bs = _net(rng, dims, scale=2.0)
    a0 = rng.standard_normal(4) * 0.3
    sig = rng.uniform(0.2, 0.5, 4)
    n = 3
    alphas = [rng.uniform(0.2, 0.8, W.shape[0]) for W in Ws[:-1]]
    grads = []
    O.crown_vjp(Ws, bs, O.ACT_RELU, a0, sig, -np.ones(n), np.ones(n), alphas=alphas, slope_grads=grads)

    def Wd(al):
        f = O.crown_forward(Ws, bs, O.ACT_RELU, a0, sig, alphas=al)
        return (f["r_hi"] - f["r_lo"]).sum(), f
    _, f0 = Wd(alphas)
    h, ok = 1e-6, 0
    for l in range(len(alphas)):
        unstable = [a[0] == "unstable" for a in f0["relaxs"][l][4]]
        for k in range(len(unstable)):
            ap = [a.copy() for a in alphas]; am = [a.copy() for a in alphas]
            ap[l][k] += h; am[l][k] -= h
            fp, fm, fc = Wd(ap)[0], Wd(am)[0], Wd(alphas)[0]
            if not unstable[k]:
                assert fp == fm                                    # stable neurons ignore alpha
                continue
            if abs((fp - fc) - (fc - fm)) > 1e-3 * abs(fp - fm) + 1e-12:
                continue
            assert abs((fp - fm) / (2 * h) - grads[l][k]) <= 1e-5 * abs(grads[l][k]) + 1e-7, (l, k)
            ok += 1
    assert ok >= 5
    lo, hi, w0, w = O.alpha_refine(Ws, bs, a0, sig, steps=10, lr=0.05)
    base = O.crown_forward(Ws, bs, O.ACT_RELU, a0, sig)
    assert np.isclose(w0, (base["r_hi"] - base["r_lo"]).sum()) and w < 0.98 * w0
    X = np.concatenate([a0 + sig * rng.uniform(-1, 1, (20000, 4)), _vertices(a0, sig)])
    R = _true_r(Ws, bs, O.ACT_RELU, a0, X)
    assert np.all(R.min(0) >= lo - 1e-12) and np.all(R.max(0) <= hi + 1e-12)
