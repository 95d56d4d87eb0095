"""GPU tests of the certified mode of leb_nn_fwd (step N6 of SURVEY 8(a); flags without LEB_FLAG_NO_MARGIN): the FP32 /
3xTF32 rounding error of the CROWN path (Thm 2 eq. (18), Thm 3 eq. (19)-(21) L204-220) is bounded
and added outward (DESIGN.md §6 "Certified margin").  Checked against the FP64 oracle and against the true remainder:
* the certified enclosure contains the oracle's (exact-arithmetic CROWN) enclosure, hidden layers and output;
* it is never below the sampled maximum of the remainder -- with NO tolerance (that is the point of the mode);
* its looseness over the oracle is small and is reported."""
import itertools

import numpy as np
import pytest
import torch

from parity_util import to_np

pytestmark = pytest.mark.gpu

PATHS = {"tc": 0, "ffma": 2}          # certified mode on both contraction paths


@pytest.fixture(scope="module")
def mods():
    from paper_2607_01203_b200 import build, leb, workloads
    from oracle import nn_oracle
    build.build()
    return leb, workloads, nn_oracle


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


SMALL = [([5, 9, 3], 1), ([5, 9, 3], 2), ([6, 10, 10, 10, 4], 1), ([6, 10, 10, 10, 4], 2), ([7, 33, 20, 11, 5], 2),
         ([40, 64, 64, 64, 64, 33], 2), ([24, 130, 70, 20], 1)]


def _looseness(clo, chi, olo, ohi):
    """largest outward excess of the certified enclosure, as a fraction of the tile's widest oracle enclosure"""
    w = np.maximum((ohi - olo).max(axis=1, keepdims=True), 1e-3)      # a tile whose bound is exactly [0, 0]: absolute scale
    return float(np.max(np.maximum(chi - ohi, olo - clo) / w))


@pytest.mark.parametrize("path", list(PATHS))
@pytest.mark.parametrize("dims,act", SMALL)
def test_certified_contains_oracle_enclosure(mods, dims, act, path):
    leb, wl, O = mods
    w = wl.make_small_mlp(dims, act, 3, 4, rad_lo=0.02, rad_hi=0.2)
    ctx = leb.context_for_workload(w)
    nom_d, rad_d = _dev(w.nom), _dev(w.rad)
    mg = torch.full((w.B, w.T, w.n), -1.0, device="cuda")
    lo, hi = ctx.leb_nn_fwd(nom_d, rad_d, margin=mg, flags=PATHS[path])
    nom, rad = w.nom.reshape(-1, w.N), w.rad.reshape(-1, w.N)
    Ws = [np.asarray(x, np.float64) for x in w.mlp.W]; bs = [np.asarray(x, np.float64) for x in w.mlp.b]
    clo, chi = to_np(lo).reshape(-1, w.n).astype(np.float64), to_np(hi).reshape(-1, w.n).astype(np.float64)
    hidden = [ctx.leb_nn_hidden_bounds(layer, w.B * w.T, dims[layer]) for layer in range(1, len(dims) - 1)]
    olo, ohi = O.leb_nn(w.mlp.W, w.mlp.b, act, nom, rad)
    # the certified enclosure contains the exact-arithmetic one
    assert np.all(chi >= ohi) and np.all(clo <= olo), (dims, float((ohi - chi).max()), float((clo - olo).max()))
    for t in range(w.B * w.T):
        fw = O.crown_forward(Ws, bs, act, nom[t].astype(np.float64), rad[t].astype(np.float64))
        for layer, (l, u) in enumerate(hidden, start=1):
            assert np.all(to_np(l)[t] <= fw["ls"][layer - 1]) and np.all(to_np(u)[t] >= fw["us"][layer - 1]), (dims, t, layer)
    # ... and is not much wider (fraction of the enclosure's width)
    assert _looseness(clo, chi, olo, ohi) < 2e-2, _looseness(clo, chi, olo, ohi)
    # the reported margin is what was added over the plain FP32 value; value mode reports 0
    m = to_np(mg)
    assert np.all(m > 0) and np.all(m < 1e-2 * (1 + np.abs(to_np(hi))))
    vlo, vhi = ctx.leb_nn_fwd(nom_d, rad_d, margin=mg, flags=PATHS[path] | leb.FLAG_NO_MARGIN)
    assert float(mg.abs().max()) == 0.0
    ctx.close()


@pytest.mark.parametrize("path", list(PATHS))
def test_certified_never_below_sampled_maximum_strict(mods, path):
    """Tiny nets (<= 4 inputs), >= 1e5 samples + all box vertices per tile, no tolerance.  The caller passes J (FP32),
    so the remainder is defined with exactly that matrix (Thm 3 holds for any J, reading R12)."""
    leb, wl, O = mods
    for dims, act, seed in (([3, 12, 2], 1, 1), ([4, 10, 3], 1, 2), ([4, 8, 8, 2], 2, 3), ([2, 16, 16, 2], 1, 4), ([1, 6, 1], 1, 5)):
        w = wl.make_small_mlp(dims, act, 2, 2, seed=seed, rad_lo=0.05, rad_hi=0.4)
        ctx = leb.context_for_workload(w)
        Ws = [np.asarray(x, np.float64) for x in w.mlp.W]; bs = [np.asarray(x, np.float64) for x in w.mlp.b]
        N = dims[0]
        J32 = np.stack([O.nominal(Ws, bs, act, a0.astype(np.float64))[2] for a0 in w.nom.reshape(-1, N)]).astype(np.float32)
        lo, hi = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), J=_dev(J32.reshape(w.B, w.T, w.n, N)), flags=PATHS[path])
        clo, chi = to_np(lo).reshape(-1, w.n).astype(np.float64), to_np(hi).reshape(-1, w.n).astype(np.float64)
        rng = np.random.default_rng(seed)
        verts = np.array(list(itertools.product((-1.0, 1.0), repeat=N)))
        for t in range(w.B * w.T):
            a0 = w.nom.reshape(-1, N)[t].astype(np.float64); sg = w.rad.reshape(-1, N)[t].astype(np.float64)
            U = np.concatenate([rng.uniform(-1, 1, (100000, N)), verts])
            X = a0[None, :] + U * sg[None, :]
            _, p, _ = O.nominal(Ws, bs, act, a0)
            A = X.T
            for l in range(len(Ws) - 1):
                A = O.phi(act, Ws[l] @ A + bs[l][:, None])
            r = (Ws[-1] @ A + bs[-1][:, None]).T - p[None, :] - (X - a0[None, :]) @ J32[t].astype(np.float64).T
            assert np.all(r.max(0) <= chi[t]) and np.all(r.min(0) >= clo[t]), (dims, t)
        ctx.close()


@pytest.mark.parametrize("path", list(PATHS))
def test_certified_is_relative_to_the_readable_jacobian_strict(mods, path):
    """J = NULL: the enclosure is of p(a) - p(a~) - J~ (a - a~) with J~ the library's own chain rows, rounding included.
    leb_nn_jacobian returns that matrix; it matches the FP64 Jacobian to FP32 rounding, and the sampled remainder taken
    with exactly J~ lies inside the certified enclosure with no tolerance (>= 1e5 samples + all vertices per tile)."""
    leb, wl, O = mods
    for dims, act, seed in (([3, 12, 2], 1, 11), ([4, 10, 3], 2, 12), ([4, 8, 8, 2], 2, 13), ([2, 16, 16, 2], 1, 14)):
        w = wl.make_small_mlp(dims, act, 2, 2, seed=seed, rad_lo=0.05, rad_hi=0.4)
        ctx = leb.context_for_workload(w)
        Ws = [np.asarray(x, np.float64) for x in w.mlp.W]; bs = [np.asarray(x, np.float64) for x in w.mlp.b]
        N = dims[0]
        lo, hi = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), flags=PATHS[path])
        Jt = to_np(ctx.leb_nn_jacobian(w.B * w.T, w.n, N)).astype(np.float64)
        clo, chi = to_np(lo).reshape(-1, w.n).astype(np.float64), to_np(hi).reshape(-1, w.n).astype(np.float64)
        rng = np.random.default_rng(seed)
        verts = np.array(list(itertools.product((-1.0, 1.0), repeat=N)))
        for t in range(w.B * w.T):
            a0 = w.nom.reshape(-1, N)[t].astype(np.float64); sg = w.rad.reshape(-1, N)[t].astype(np.float64)
            _, p, J64 = O.nominal(Ws, bs, act, a0)
            assert np.abs(Jt[t] - J64).max() <= 1e-5 * np.abs(J64).max() + 1e-7, (dims, t)
            U = np.concatenate([rng.uniform(-1, 1, (100000, N)), verts])
            X = a0[None, :] + U * sg[None, :]
            A = X.T
            for l in range(len(Ws) - 1):
                A = O.phi(act, Ws[l] @ A + bs[l][:, None])
            r = (Ws[-1] @ A + bs[-1][:, None]).T - p[None, :] - (X - a0[None, :]) @ Jt[t].T
            assert np.all(r.max(0) <= chi[t]) and np.all(r.min(0) >= clo[t]), (dims, t)
        # a forward that was given the caller's J leaves no J~ to read
        J32 = np.stack([O.nominal(Ws, bs, act, a0.astype(np.float64))[2] for a0 in w.nom.reshape(-1, N)]).astype(np.float32)
        ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), J=_dev(J32.reshape(w.B, w.T, w.n, N)), flags=PATHS[path])
        with pytest.raises(leb.LebError) as e:
            ctx.leb_nn_jacobian(w.B * w.T, w.n, N)
        assert e.value.status == leb.LEB_ERR_STATE
        ctx.close()


@pytest.mark.parametrize("path", list(PATHS))
@pytest.mark.parametrize("cfg", [3, 5])
def test_certified_config_sampled_tiles(mods, cfg, path):
    """Configs 3 and 5 at BASELINE size in the launch configuration bench.py uses; oracle on sampled tiles."""
    leb, wl, O = mods
    w = wl.make_config(cfg)
    ctx = leb.context_for_workload(w)
    nom_d, rad_d = _dev(w.nom), _dev(w.rad)
    mg = torch.empty((w.B, w.T, w.n), device="cuda")
    lo, hi = ctx.leb_nn_fwd(nom_d, rad_d, margin=mg, flags=PATHS[path])
    assert ctx.leb_domain_flag() == 0
    vlo, vhi = ctx.leb_nn_fwd(nom_d, rad_d, flags=PATHS[path] | leb.FLAG_NO_MARGIN)
    nom, rad = w.nom.reshape(-1, w.N), w.rad.reshape(-1, w.N)
    idx = np.array([0, 1023, 1024, 3777, w.B * w.T - 1]) if cfg == 5 else np.linspace(0, w.B * w.T - 1, 16).astype(int)
    olo, ohi = O.leb_nn(w.mlp.W, w.mlp.b, w.mlp.act, nom[idx], rad[idx])
    clo, chi = to_np(lo).reshape(-1, w.n).astype(np.float64)[idx], to_np(hi).reshape(-1, w.n).astype(np.float64)[idx]
    assert np.all(chi >= ohi) and np.all(clo <= olo), (float((ohi - chi).max()), float((clo - olo).max()))
    loose = _looseness(clo, chi, olo, ohi)
    print(f"config {cfg} {path}: certified looseness over the oracle enclosure = {loose:.3e} of its width")
    assert loose < 5e-2
    # at any size: contains the value-mode result up to the parity tolerance, finite, margin positive
    # (a widened hidden bound can flip a relaxation case, e.g. the ReLU lower slope at u = -l, to an equally valid
    # one that happens to be tighter for some output -- reading R21 -- so a few entries may lie inside the value result)
    inside = ((hi < vhi - 1e-5 * vhi.abs() - 1e-7) | (lo > vlo + 1e-5 * vlo.abs() + 1e-7)).float().mean()
    print(f"config {cfg} {path}: fraction of entries tighter than value mode (case flips) = {float(inside):.2e}")
    assert float(inside) < 5e-3
    assert bool(torch.isfinite(hi).all()) and bool(torch.isfinite(lo).all()) and bool((mg > 0).all())
    ctx.close()


def test_certified_edge_cases(mods):
    leb, wl, O = mods
    w = wl.make_small_mlp([6, 10, 10, 4], 1, 2, 3)
    ctx = leb.context_for_workload(w)
    nom, rad = _dev(w.nom), _dev(w.rad)
    # zero radius: the exact bound is [0, 0]; the certified one is a rounding-level enclosure of it
    lo, hi = ctx.leb_nn_fwd(nom, torch.zeros_like(rad), flags=0)
    assert bool((lo <= 0).all()) and bool((hi >= 0).all()) and float(hi.max()) < 1e-4 and float(lo.min()) > -1e-4
    # chunking does not change results
    lo1, hi1 = ctx.leb_nn_fwd(nom, rad, flags=0)
    ctx.leb_set_nn_chunk(4)
    lo2, hi2 = ctx.leb_nn_fwd(nom, rad, flags=0)
    ctx.leb_set_nn_chunk(0)
    assert torch.equal(lo1, lo2) and torch.equal(hi1, hi2)
    # NaN input poisons its tile only
    n2 = w.nom.copy(); n2[1, 0, 2] = np.nan
    lo, hi = ctx.leb_nn_fwd(_dev(n2), rad, flags=0)
    assert ctx.leb_domain_flag() == 1
    assert bool(torch.isinf(lo[1, 0]).all()) and bool(torch.isinf(hi[1, 0]).all()) and bool(torch.isfinite(lo[0]).all())
    # layers wider than 2048 (padded): the norm / sum inflation factors of the certificate are derived for K <= 2048
    wide = wl.make_small_mlp([4, 2100, 3], 1, 1, 1)
    cw = leb.context_for_workload(wide)
    with pytest.raises(leb.LebError) as e:
        cw.leb_nn_fwd(_dev(wide.nom), _dev(wide.rad), flags=0)
    assert e.value.status == leb.LEB_ERR_UNSUPPORTED
    cw.leb_nn_fwd(_dev(wide.nom), _dev(wide.rad), flags=leb.FLAG_NO_MARGIN)      # value mode has no such limit
    cw.close()
    # the VJP is that of the value-mode bound whichever mode is asked for
    g1 = ctx.leb_vjp(1, nom, rad, _dev(w.g_lo), _dev(w.g_hi), flags=0)
    g2 = ctx.leb_vjp(1, nom, rad, _dev(w.g_lo), _dev(w.g_hi), flags=leb.FLAG_NO_MARGIN)
    assert torch.equal(g1[0], g2[0]) and torch.equal(g1[1], g2[1])
    # LEB_FLAG_REUSE_FWD is honoured only when the resident forward state has the mode the VJP call names (leb.h):
    ctx.leb_nn_fwd(nom, rad, flags=0)                                   # certified state resident
    assert ctx.leb_nn_state()[:2] == (w.B * w.T, True)
    g3 = ctx.leb_vjp(1, nom, rad, _dev(w.g_lo), _dev(w.g_hi), flags=leb.FLAG_NO_MARGIN | leb.FLAG_REUSE_FWD)
    assert ctx.leb_nn_state()[2] is False                               # value-mode VJP asked: recomputed, not reused
    assert torch.allclose(g3[0], g2[0], rtol=1e-5, atol=1e-7) and torch.allclose(g3[1], g2[1], rtol=1e-5, atol=1e-7)
    ctx.leb_nn_fwd(nom, rad, flags=0)
    g4 = ctx.leb_vjp(1, nom, rad, _dev(w.g_lo), _dev(w.g_hi), flags=leb.FLAG_REUSE_FWD)
    assert ctx.leb_nn_state() == (w.B * w.T, True, True)                # reverse sweep over the certified state
    # ... the gradient of the certified bound with its pads held constant: that of the value-mode bound up to the pads' size
    for a, b in zip(g4, g2):
        assert float((a - b).abs().max()) <= 2e-2 * float(b.abs().max())
    ctx.close()


@pytest.mark.parametrize("path", list(PATHS))
def test_certified_strict_soundness_wide_tanh_net(mods, path):
    """A 3-hidden-layer tanh net of width 128 (config-3 shape, tanh): 1e5 samples of the box plus 1e5 of its vertices per
    tile, no tolerance; J is passed in FP32 so the remainder is defined with exactly that matrix (reading R12).  (At this
    size the sampled extremum is far inside the bound -- SURVEY 8(c).7 -- so this guards the sign and the direction of
    every pad rather than its size; the size is what the tiny-net test and the containment tests check.)"""
    leb, wl, O = mods
    w = wl.make_small_mlp([24, 128, 128, 128, 20], 2, 1, 3, seed=21, rad_lo=0.01, rad_hi=0.05, init="xavier")
    ctx = leb.context_for_workload(w)
    Ws = [np.asarray(x, np.float64) for x in w.mlp.W]; bs = [np.asarray(x, np.float64) for x in w.mlp.b]
    N = 24
    J32 = np.stack([O.nominal(Ws, bs, 2, a0.astype(np.float64))[2] for a0 in w.nom.reshape(-1, N)]).astype(np.float32)
    lo, hi = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), J=_dev(J32.reshape(w.B, w.T, w.n, N)), flags=PATHS[path])
    clo, chi = to_np(lo).reshape(-1, w.n).astype(np.float64), to_np(hi).reshape(-1, w.n).astype(np.float64)
    rng = np.random.default_rng(21)
    for t in range(w.B * w.T):
        a0 = w.nom.reshape(-1, N)[t].astype(np.float64); sg = w.rad.reshape(-1, N)[t].astype(np.float64)
        U = np.concatenate([rng.uniform(-1, 1, (100000, N)), rng.choice([-1.0, 1.0], (100000, N))])
        X = a0[None, :] + U * sg[None, :]
        _, p, _ = O.nominal(Ws, bs, 2, a0)
        A = X.T
        for l in range(len(Ws) - 1):
            A = O.phi(2, Ws[l] @ A + bs[l][:, None])
        r = (Ws[-1] @ A + bs[-1][:, None]).T - p[None, :] - (X - a0[None, :]) @ J32[t].astype(np.float64).T
        assert np.all(r.max(0) <= chi[t]) and np.all(r.min(0) >= clo[t]), t
    ctx.close()


@pytest.mark.parametrize("K", [128, 224, 512, 2048])
@pytest.mark.parametrize("path", list(PATHS))
def test_contraction_error_model(mods, path, K):
    """The rounding model behind the margin, probed on one chain step Lambda_0 = W_2 W_1 (ReLU, every
    hidden neuron stably active so that D = W_2 exactly; K = 512): |computed - exact| <= sum_j gamma_j |W_2[i,j]| |W_1[j,k]|
    elementwise, on operands built to be bad for a truncating block adder -- all-positive terms (every truncation loses),
    one large term followed by terms just below each candidate truncation grid, a large term in every block of 8 -- and on
    random ones.  Reports how much of the bound the worst case uses."""
    leb, wl, O = mods
    N0, n = 64, 64
    j = np.arange(K)
    if path == "tc":
        gam = (4.5 * (K // 8 - j // 8) + 17.0) * 2.0 ** -23
    else:
        gam = (K - j + 4.0) * 2.0 ** -24 + 2.0 ** -23
    rng = np.random.default_rng(0)
    sgn = rng.choice([-1.0, 1.0], (n, K))
    cases = {"pos": (rng.uniform(0.5, 1, (n, K)), rng.uniform(0.5, 1, (K, N0))),
             "rand": (rng.standard_normal((n, K)), rng.standard_normal((K, N0))),
             # mixed signs with cancellation: the exact result is much smaller than the sum of magnitudes
             "mixed": (sgn * rng.uniform(0.5, 1, (n, K)), rng.uniform(0.5, 1, (K, N0))),
             "alternating": (np.where(j % 2 == 0, 1.0, -1.0)[None, :] * np.ones((n, K)), 1.0 + 2.0 ** -12 * rng.integers(0, 2048, (K, N0)))}
    for p in range(22, 31):
        tiny = 2.0 ** -p * (1 - 2.0 ** -9)
        W2 = np.full((n, K), tiny); W2[:, 0] = 1.0
        cases[f"one large, rest 2^-{p}"] = (W2, np.ones((K, N0)))
        W2 = np.full((n, K), tiny); W2[:, ::8] = 1.0
        cases[f"large every 8, rest 2^-{p}"] = (W2, np.ones((K, N0)))
        W2 = np.full((n, K), tiny); W2[:, K // 2] = 1.0
        cases[f"large in the middle, rest 2^-{p}"] = (W2, np.ones((K, N0)))
    dev = torch.device("cuda", 0)
    worst = 0.0
    for name, (W2, W1) in cases.items():
        W2 = W2.astype(np.float32); W1 = W1.astype(np.float32)
        ctx = leb.Context(0)
        ctx.leb_set_mlp([N0, K, n], [torch.from_numpy(W1).to(dev), torch.from_numpy(W2).to(dev)],
                        [torch.full((K,), 4.0, device=dev), torch.zeros(n, device=dev)], 1, 1)
        # hidden pre-activation z_1 = W_1 a + 4 > 0 on the whole box (|a| <= 1e-3): slopes exactly 1
        nom = torch.zeros((1, 1, N0), device=dev); rad = torch.full((1, 1, N0), 1e-3, device=dev)
        ctx.leb_nn_fwd(nom, rad, flags=PATHS[path] | leb.FLAG_NO_MARGIN)
        lam = to_np(ctx.leb_nn_chain_coeffs(2, 1, n, N0)).astype(np.float64)
        ctx.close()
        ref = W2.astype(np.float64) @ W1.astype(np.float64)
        bound = (np.abs(W2).astype(np.float64) * gam[None, :]) @ np.abs(W1).astype(np.float64)
        for chain in (0, 1):
            ratio = float(np.max(np.abs(lam[0, chain] - ref) / bound))
            worst = max(worst, ratio)
            assert ratio <= 1.0, (name, chain, ratio)
    print(f"{path} K={K}: worst observed contraction error = {worst:.3f} of the model bound")
    from parity_util import report
    report(f"contraction error model {path} K={K} (observed error / model bound)", worst)


# ---------------------------------------------------------------------------------- certified mode on non-centred boxes
@pytest.mark.parametrize("hidden", ["crown", "ibp"])
@pytest.mark.parametrize("path", list(PATHS))
@pytest.mark.parametrize("dims,act", SMALL)
def test_certified_mu_sound_and_not_much_wider(mods, dims, act, path, hidden):
    """mu != NULL in certified mode.  The relaxation gaps are taken at the nominal pre-activation zhat(a~), which lies
    outside a neuron's interval when |W_1 mu| exceeds its radius; the certificate clamps them (gU >= 0 >= gL keeps the gap
    sums same-signed, which its rounding factors need), so the hidden bounds are up to ~1e-2 wider than the oracle's and
    the later relaxations differ from the oracle's -- containment of the ORACLE's enclosure is therefore not the test here.
    What is: strict soundness (no tolerance) of the output enclosure and of every hidden bound on 2e4 samples + sampled
    vertices of the offset box, with J passed in FP32, and a bounded looseness against the oracle."""
    leb, wl, O = mods
    w = wl.make_small_mlp(dims, act, 3, 4, rad_lo=0.02, rad_hi=0.2)
    mu = wl.make_mu(w, 1.5)
    ctx = leb.context_for_workload(w)
    Ws = [np.asarray(x, np.float64) for x in w.mlp.W]; bs = [np.asarray(x, np.float64) for x in w.mlp.b]
    N = dims[0]
    nom, rad, mu_f = w.nom.reshape(-1, N), w.rad.reshape(-1, N), mu.reshape(-1, N)
    J32 = np.stack([O.nominal(Ws, bs, act, a0.astype(np.float64))[2] for a0 in nom]).astype(np.float32)
    flags = PATHS[path] | (leb.FLAG_IBP_HIDDEN if hidden == "ibp" else 0)
    lo, hi = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), J=_dev(J32.reshape(w.B, w.T, w.n, N)), flags=flags, mu=_dev(mu))
    assert ctx.leb_domain_flag() == 0
    clo, chi = to_np(lo).reshape(-1, w.n).astype(np.float64), to_np(hi).reshape(-1, w.n).astype(np.float64)
    hbounds = [tuple(to_np(x).astype(np.float64) for x in ctx.leb_nn_hidden_bounds(layer, w.B * w.T, dims[layer])) for layer in range(1, len(dims) - 1)]
    rng = np.random.default_rng(5)
    for t in range(w.B * w.T):
        a0, sg, m = nom[t].astype(np.float64), rad[t].astype(np.float64), mu_f[t].astype(np.float64)
        X = a0[None] + m[None] + np.concatenate([rng.uniform(-1, 1, (20000, N)), rng.choice([-1.0, 1.0], (4096, N))]) * sg[None]
        _, p, _ = O.nominal(Ws, bs, act, a0)
        A = X.T
        for l in range(len(Ws) - 1):
            Z = Ws[l] @ A + bs[l][:, None]
            assert np.all(Z.min(1) >= hbounds[l][0][t]) and np.all(Z.max(1) <= hbounds[l][1][t]), (dims, t, l)
            A = O.phi(act, Z)
        r = (Ws[-1] @ A + bs[-1][:, None]).T - p[None, :] - (X - a0[None, :]) @ J32[t].astype(np.float64).T
        assert np.all(r.max(0) <= chi[t]) and np.all(r.min(0) >= clo[t]), (dims, t)
    olo, ohi = O.leb_nn(w.mlp.W, w.mlp.b, act, nom, rad, J=J32, mu=mu_f, hidden=hidden)
    per_tile = np.array([_looseness(clo[t:t + 1], chi[t:t + 1], olo[t:t + 1], ohi[t:t + 1]) for t in range(clo.shape[0])])
    print(f"certified mu {hidden} {dims} {path}: looseness over the oracle enclosure median {np.median(per_tile):.3e} max {per_tile.max():.3e}")
    assert np.median(per_tile) < 5e-2 and per_tile.max() < 0.25, per_tile
    ctx.close()


@pytest.mark.parametrize("path", list(PATHS))
def test_certified_mu_never_below_sampled_maximum_strict(mods, path):
    """Tiny nets, offset boxes (|mu| up to 2 sigma), >= 1e5 samples + all vertices per tile, no tolerance; J passed in FP32."""
    leb, wl, O = mods
    for dims, act, seed in (([3, 12, 2], 1, 1), ([4, 8, 8, 2], 2, 3), ([2, 16, 16, 2], 1, 4)):
        w = wl.make_small_mlp(dims, act, 2, 2, seed=seed, rad_lo=0.05, rad_hi=0.4)
        mu = wl.make_mu(w, 2.0)
        ctx = leb.context_for_workload(w)
        Ws = [np.asarray(x, np.float64) for x in w.mlp.W]; bs = [np.asarray(x, np.float64) for x in w.mlp.b]
        N = dims[0]
        J32 = np.stack([O.nominal(Ws, bs, act, a0.astype(np.float64))[2] for a0 in w.nom.reshape(-1, N)]).astype(np.float32)
        lo, hi = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), J=_dev(J32.reshape(w.B, w.T, w.n, N)), flags=PATHS[path], mu=_dev(mu))
        clo, chi = to_np(lo).reshape(-1, w.n).astype(np.float64), to_np(hi).reshape(-1, w.n).astype(np.float64)
        rng = np.random.default_rng(seed)
        verts = np.array(list(itertools.product((-1.0, 1.0), repeat=N)))
        for t in range(w.B * w.T):
            a0 = w.nom.reshape(-1, N)[t].astype(np.float64); sg = w.rad.reshape(-1, N)[t].astype(np.float64)
            m = mu.reshape(-1, N)[t].astype(np.float64)
            X = a0[None] + m[None] + np.concatenate([rng.uniform(-1, 1, (100000, N)), verts]) * sg[None]
            _, p, _ = O.nominal(Ws, bs, act, a0)
            A = X.T
            for l in range(len(Ws) - 1):
                A = O.phi(act, Ws[l] @ A + bs[l][:, None])
            r = (Ws[-1] @ A + bs[-1][:, None]).T - p[None, :] - (X - a0[None, :]) @ J32[t].astype(np.float64).T
            assert np.all(r.max(0) <= chi[t]) and np.all(r.min(0) >= clo[t]), (dims, t)
        ctx.close()


# ---------------------------------------------------------------------------------- certified CROWN-IBP
@pytest.mark.parametrize("path", list(PATHS))
@pytest.mark.parametrize("dims,act", SMALL)
def test_certified_crown_ibp(mods, dims, act, path):
    """LEB_FLAG_IBP_HIDDEN without LEB_FLAG_NO_MARGIN.  Interval propagation is monotone in its input bounds, so every
    certified hidden bound contains the oracle's; the output enclosure contains the oracle's CROWN-IBP enclosure except
    where a relaxation case switches (reported as a tie by the oracle, R21), is not much wider, and holds with no tolerance
    on samples and sampled vertices of the box (J passed in FP32: the remainder is defined with exactly that matrix)."""
    leb, wl, O = mods
    IBP = leb.FLAG_IBP_HIDDEN
    w = wl.make_small_mlp(dims, act, 3, 4, rad_lo=0.02, rad_hi=0.2)
    ctx = leb.context_for_workload(w)
    Ws = [np.asarray(x, np.float64) for x in w.mlp.W]; bs = [np.asarray(x, np.float64) for x in w.mlp.b]
    N = dims[0]
    nom, rad = w.nom.reshape(-1, N), w.rad.reshape(-1, N)
    J32 = np.stack([O.nominal(Ws, bs, act, a0.astype(np.float64))[2] for a0 in nom]).astype(np.float32)
    Jd = _dev(J32.reshape(w.B, w.T, w.n, N))
    lo, hi = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), J=Jd, flags=PATHS[path] | IBP)
    assert ctx.leb_domain_flag() == 0
    clo, chi = to_np(lo).reshape(-1, w.n).astype(np.float64), to_np(hi).reshape(-1, w.n).astype(np.float64)
    hidden = [tuple(to_np(x).astype(np.float64) for x in ctx.leb_nn_hidden_bounds(layer, w.B * w.T, dims[layer])) for layer in range(1, len(dims) - 1)]
    olo, ohi = O.leb_nn(w.mlp.W, w.mlp.b, act, nom, rad, J=J32, hidden="ibp")
    rng = np.random.default_rng(8)
    for t in range(w.B * w.T):
        a0, sg = nom[t].astype(np.float64), rad[t].astype(np.float64)
        fw = O.crown_forward(Ws, bs, act, a0, sg, hidden="ibp")
        for layer, (l, u) in enumerate(hidden, start=1):
            assert np.all(l[t] <= fw["ls"][layer - 1]) and np.all(u[t] >= fw["us"][layer - 1]), (dims, t, layer)
        X = a0[None] + np.concatenate([rng.uniform(-1, 1, (20000, N)), rng.choice([-1.0, 1.0], (4096, N))]) * sg[None]
        _, p, _ = O.nominal(Ws, bs, act, a0)
        A = X.T
        for l in range(len(Ws) - 1):
            Z = Ws[l] @ A + bs[l][:, None]
            assert np.all(Z.min(1) >= hidden[l][0][t]) and np.all(Z.max(1) <= hidden[l][1][t]), (dims, t, l)
            A = O.phi(act, Z)
        r = (Ws[-1] @ A + bs[-1][:, None]).T - p[None, :] - (X - a0[None, :]) @ J32[t].astype(np.float64).T
        assert np.all(r.max(0) <= chi[t]) and np.all(r.min(0) >= clo[t]), (dims, t)
        if not (np.all(chi[t] >= ohi[t]) and np.all(clo[t] <= olo[t])):
            assert O.relax_case_ties(Ws, bs, act, a0, sg, rel=2e-4), (dims, t, float((ohi[t] - chi[t]).max()), float((clo[t] - olo[t]).max()))
    per_tile = np.array([_looseness(clo[t:t + 1], chi[t:t + 1], olo[t:t + 1], ohi[t:t + 1]) for t in range(clo.shape[0])])
    print(f"certified crown-ibp {dims} {path}: looseness over the oracle enclosure median {np.median(per_tile):.3e} max {per_tile.max():.3e}")
    assert np.median(per_tile) < 2e-2 and per_tile.max() < 0.1, per_tile
    # a certified CROWN-IBP state (of a forward with the library's own Jacobian) is reused by a certified CROWN-IBP VJP
    ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), flags=PATHS[path] | IBP)
    g = ctx.leb_vjp(1, _dev(w.nom), _dev(w.rad), _dev(w.g_lo), _dev(w.g_hi), flags=PATHS[path] | IBP | leb.FLAG_REUSE_FWD)
    assert ctx.leb_nn_state() == (w.B * w.T, True, True)
    gv = ctx.leb_vjp(1, _dev(w.nom), _dev(w.rad), _dev(w.g_lo), _dev(w.g_hi), flags=PATHS[path] | IBP | leb.FLAG_NO_MARGIN)
    for a, b in zip(g, gv):
        assert float((a - b).abs().max()) <= 2e-2 * float(b.abs().max()) + 1e-7
    ctx.close()


def test_certified_crown_ibp_config5_sampled(mods):
    """Config 5 at full width, 8 tiles: certified CROWN-IBP contains the value-mode CROWN-IBP enclosure and is sound on samples."""
    leb, wl, O = mods
    w = wl.make_config(5, B=1, T=8)
    ctx = leb.context_for_workload(w)
    IBP = leb.FLAG_IBP_HIDDEN
    lo, hi = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), flags=IBP)
    vlo, vhi = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), flags=IBP | leb.FLAG_NO_MARGIN)
    assert ctx.leb_domain_flag() == 0
    assert bool((hi >= vhi).all()) and bool((lo <= vlo).all())
    width = (vhi - vlo).amax(dim=2, keepdim=True)
    excess = torch.maximum(hi - vhi, vlo - lo) / width
    print(f"certified crown-ibp config 5: excess over value mode median {float(excess.median()):.3e} max {float(excess.max()):.3e}")
    assert float(excess.max()) < 0.2
    ctx.close()


# ---------------------------------------------------------------------------------- certified optimised slopes
@pytest.mark.parametrize("path", list(PATHS))
def test_certified_alpha_refinement(mods, path):
    """leb_nn_alpha_fwd without LEB_FLAG_NO_MARGIN: the kept slopes evaluated in certified mode.  The result contains the
    value-mode refined enclosure, is at most a little wider, is tighter than the certified adaptive-slope enclosure where
    the refinement helped, and holds with no tolerance on samples and vertices (J~ read back: the matrix it is relative to)."""
    leb, wl, O = mods
    for dims, seed in (([4, 10, 10, 10, 3], 5), ([6, 33, 20, 11, 5], 6)):
        w = wl.make_small_mlp(dims, 1, 2, 3, seed=seed, rad_lo=0.1, rad_hi=0.4)
        ctx = leb.context_for_workload(w)
        Ws = [np.asarray(x, np.float64) for x in w.mlp.W]; bs = [np.asarray(x, np.float64) for x in w.mlp.b]
        N, tiles = dims[0], w.B * w.T
        steps, lr = 8, 0.05
        vlo, vhi, vw0, vwb = ctx.leb_nn_alpha_fwd(_dev(w.nom), _dev(w.rad), steps, lr, flags=PATHS[path] | leb.FLAG_NO_MARGIN)
        clo, chi, cw0, cwb = ctx.leb_nn_alpha_fwd(_dev(w.nom), _dev(w.rad), steps, lr, flags=PATHS[path])
        assert ctx.leb_nn_state()[:2] == (tiles, True)
        Jt = to_np(ctx.leb_nn_jacobian(tiles, w.n, N)).astype(np.float64)
        assert bool((chi >= vhi).all()) and bool((clo <= vlo).all())
        assert bool((cwb <= vwb * (1 + 2e-2) + 1e-6).all())
        plo, phi = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), flags=PATHS[path])
        pw = (phi - plo).sum(dim=2)
        assert bool((cwb <= pw * (1 + 1e-6)).all()) and bool((cwb < 0.999 * pw).any())
        lo64, hi64 = to_np(clo).reshape(-1, w.n).astype(np.float64), to_np(chi).reshape(-1, w.n).astype(np.float64)
        rng = np.random.default_rng(seed)
        for t in range(tiles):
            a0 = w.nom.reshape(-1, N)[t].astype(np.float64); sg = w.rad.reshape(-1, N)[t].astype(np.float64)
            U = rng.uniform(-1, 1, (50000, N))
            if N <= 6:
                U = np.concatenate([U, np.array(list(itertools.product((-1.0, 1.0), repeat=N)))])
            X = a0[None] + U * sg[None]
            _, p, _ = O.nominal(Ws, bs, 1, a0)
            A = X.T
            for l in range(len(Ws) - 1):
                A = O.phi(1, Ws[l] @ A + bs[l][:, None])
            r = (Ws[-1] @ A + bs[-1][:, None]).T - p[None] - (X - a0[None]) @ Jt[t].T
            assert np.all(r.max(0) <= hi64[t]) and np.all(r.min(0) >= lo64[t]), (dims, t)
        ctx.close()


def test_chunking_does_not_change_the_newer_variants(mods):
    """A batch processed in chunks of 5 tiles (12 tiles: a ragged last chunk) gives the results of the one-chunk run, bit for
    bit, for non-centred boxes (certified), certified CROWN-IBP with mu, and the slope refinement (certified)."""
    leb, wl, O = mods
    w = wl.make_small_mlp([6, 33, 20, 11, 5], 1, 3, 4, seed=3, rad_lo=0.05, rad_hi=0.3)
    mu = _dev(wl.make_mu(w, 1.0))
    nom, rad = _dev(w.nom), _dev(w.rad)
    ctx = leb.context_for_workload(w)
    IBP = leb.FLAG_IBP_HIDDEN

    def run():
        a = ctx.leb_nn_fwd(nom, rad, mu=mu)
        b = ctx.leb_nn_fwd(nom, rad, mu=mu, flags=IBP)
        c = ctx.leb_nn_alpha_fwd(nom, rad, 4, 0.05)
        d = ctx.leb_vjp_mu(1, nom, rad, mu, _dev(w.g_lo), _dev(w.g_hi), flags=IBP)
        return [x.clone() for x in (*a, *b, *c)], [x.clone() for x in d]

    full, gfull = run()
    ctx.leb_set_nn_chunk(5)
    part, gpart = run()
    # several chunks: no complete state is resident, so nothing can be reused
    ctx.leb_nn_alpha_fwd(nom, rad, 2, 0.05)
    ctx.leb_vjp(1, nom, rad, _dev(w.g_lo), _dev(w.g_hi), flags=leb.FLAG_REUSE_FWD)
    assert ctx.leb_nn_state()[2] is False
    ctx.leb_set_nn_chunk(0)
    for x, y in zip(full, part):
        assert torch.equal(x, y)
    for x, y in zip(gfull, gpart):                       # column sums are atomic adds: equal to rounding
        assert float((x - y).abs().max()) <= 1e-5 * float(y.abs().max())
    ctx.close()


def test_certified_mu_config5_width_sampled_soundness(mods):
    """Config 5 at full width (224 -> 512 x 4 -> 168, tanh), 4 tiles, offset boxes (|mu| <= 1.5 sigma), certified mode, both
    hidden-bound variants: the sampled remainder (2e4 samples + 4 096 sampled vertices of the offset box, J~ read back)
    inside the enclosure with no tolerance, and the enclosure contains the value-mode one."""
    leb, wl, O = mods
    w = wl.make_config(5, B=1, T=4)
    mu = wl.make_mu(w, 1.5)
    ctx = leb.context_for_workload(w)
    Ws = [np.asarray(x, np.float64) for x in w.mlp.W]; bs = [np.asarray(x, np.float64) for x in w.mlp.b]
    N = w.N
    nom, rad, mu_f = w.nom.reshape(-1, N), w.rad.reshape(-1, N), mu.reshape(-1, N)
    rng = np.random.default_rng(17)
    for flags in (0, leb.FLAG_IBP_HIDDEN):
        lo, hi = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), mu=_dev(mu), flags=flags)
        Jt = to_np(ctx.leb_nn_jacobian(w.B * w.T, w.n, N)).astype(np.float64)
        vlo, vhi = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), mu=_dev(mu), flags=flags | leb.FLAG_NO_MARGIN)
        assert ctx.leb_domain_flag() == 0
        assert bool((hi >= vhi).all()) and bool((lo <= vlo).all())
        clo, chi = to_np(lo).reshape(-1, w.n).astype(np.float64), to_np(hi).reshape(-1, w.n).astype(np.float64)
        for t in range(w.B * w.T):
            a0, sg, m = nom[t].astype(np.float64), rad[t].astype(np.float64), mu_f[t].astype(np.float64)
            X = a0[None] + m[None] + np.concatenate([rng.uniform(-1, 1, (20000, N)), rng.choice([-1.0, 1.0], (4096, N))]) * sg[None]
            _, p, _ = O.nominal(Ws, bs, w.mlp.act, a0)
            A = X.T
            for l in range(len(Ws) - 1):
                A = O.phi(w.mlp.act, Ws[l] @ A + bs[l][:, None])
            r = (Ws[-1] @ A + bs[-1][:, None]).T - p[None, :] - (X - a0[None, :]) @ Jt[t].T
            assert np.all(r.max(0) <= chi[t]) and np.all(r.min(0) >= clo[t]), (flags, t)
    ctx.close()
