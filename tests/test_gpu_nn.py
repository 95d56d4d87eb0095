"""GPU parity: leb_nn_fwd / leb_vjp(kind 1) through the C ABI against the FP64 numpy oracle
(CROWN Thm 2 eq. (18) PAPER.md:L196-200 + Thm 3 eq. (19)-(21) L204-220), on the same seeded inputs."""
import itertools

import numpy as np
import pytest
import torch

from parity_util import assert_bounds_close, assert_grads_close, assert_nn_grads_close, to_np

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mods():
    from paper_2607_01203_b200 import build, leb, workloads
    from oracle import nn_oracle
    build.build()
    return leb, workloads, nn_oracle


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _flat(w):
    return (w.nom.reshape(-1, w.N), w.rad.reshape(-1, w.N), w.g_lo.reshape(-1, w.n), w.g_hi.reshape(-1, w.n))


# both contraction paths: 3xTF32 tcgen05 (default) and FP32 FFMA (LEB_FLAG_FFMA_ONLY); value mode in both
VAL = 1      # LEB_FLAG_NO_MARGIN: value mode, the mode compared with the oracle (the binding's default is certified)
PATHS = {"tc": 1, "tc_single_cta": 1 | 16, "ffma": 1 | 2}


SMALL = [  # dims, act: ragged widths (not multiples of 4 / 32), 1-4 hidden layers, both activations
    ([5, 9, 3], 1), ([5, 9, 3], 2), ([6, 10, 10, 10, 4], 1), ([6, 10, 10, 10, 4], 2),
    ([7, 33, 20, 11, 5], 2), ([3, 40, 2], 1), ([40, 64, 64, 64, 64, 33], 2), ([24, 130, 70, 20], 1),
]


@pytest.mark.parametrize("path", list(PATHS))
@pytest.mark.parametrize("dims,act", SMALL)
def test_fwd_small_nets_match_oracle(mods, dims, act, path):
    leb, wl, O = mods
    w = wl.make_small_mlp(dims, act, 3, 4, rad_lo=0.02, rad_hi=0.2)
    ctx = leb.context_for_workload(w)
    lo, hi = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), flags=PATHS[path])
    nom, rad, _, _ = _flat(w)
    olo, ohi = O.leb_nn(w.mlp.W, w.mlp.b, act, nom, rad)
    assert_bounds_close(to_np(lo).reshape(-1, w.n), olo, f"{dims} r_lo")
    assert_bounds_close(to_np(hi).reshape(-1, w.n), ohi, f"{dims} r_hi")
    # hidden-layer pre-activation bounds (N2/N3) against the oracle's
    Ws = [np.asarray(x, np.float64) for x in w.mlp.W]; bs = [np.asarray(x, np.float64) for x in w.mlp.b]
    for layer in range(1, len(dims) - 1):
        l, u = ctx.leb_nn_hidden_bounds(layer, w.B * w.T, dims[layer])
        for t in (0, w.B * w.T - 1):
            fw = O.crown_forward(Ws, bs, act, nom[t].astype(np.float64), rad[t].astype(np.float64))
            assert np.allclose(to_np(l)[t], fw["ls"][layer - 1], rtol=2e-5, atol=2e-6)
            assert np.allclose(to_np(u)[t], fw["us"][layer - 1], rtol=2e-5, atol=2e-6)
    ctx.close()


@pytest.mark.parametrize("path", list(PATHS))
@pytest.mark.parametrize("dims,act", SMALL)
def test_vjp_small_nets_match_oracle(mods, dims, act, path):
    leb, wl, O = mods
    w = wl.make_small_mlp(dims, act, 3, 4, rad_lo=0.02, rad_hi=0.2)
    ctx = leb.context_for_workload(w)
    gn, gr = ctx.leb_vjp(1, _dev(w.nom), _dev(w.rad), _dev(w.g_lo), _dev(w.g_hi), flags=PATHS[path])
    nom, rad, g_lo, g_hi = _flat(w)
    ogn, ogr = O.leb_nn_vjp(w.mlp.W, w.mlp.b, act, nom, rad, g_lo, g_hi)
    assert_grads_close(to_np(gn), to_np(gr), ogn, ogr, f"{dims}")
    ctx.close()


@pytest.mark.parametrize("path", list(PATHS))
def test_config3_full_size_sampled_tiles(mods, path):
    """Config 3 at BASELINE size (1280 tiles: two workspace chunks), oracle on 24 sampled tiles."""
    leb, wl, O = mods
    w = wl.make_config(3)
    ctx = leb.context_for_workload(w)
    lo, hi = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), flags=PATHS[path])
    gn, gr = ctx.leb_vjp(1, _dev(w.nom), _dev(w.rad), _dev(w.g_lo), _dev(w.g_hi), flags=PATHS[path])
    nom, rad, g_lo, g_hi = _flat(w)
    idx = np.linspace(0, w.B * w.T - 1, 24).astype(int)
    olo, ohi = O.leb_nn(w.mlp.W, w.mlp.b, w.mlp.act, nom[idx], rad[idx])
    assert_bounds_close(to_np(lo).reshape(-1, w.n)[idx], olo, "cfg3 r_lo")
    assert_bounds_close(to_np(hi).reshape(-1, w.n)[idx], ohi, "cfg3 r_hi")
    assert_nn_grads_close(O, w.mlp, nom[idx], rad[idx], g_lo[idx], g_hi[idx], to_np(gn).reshape(-1, w.N)[idx],
                          to_np(gr).reshape(-1, w.N)[idx], "cfg3")
    ctx.close()


@pytest.mark.parametrize("path", list(PATHS))
def test_config5_full_size_sampled_tiles(mods, path):
    """Config 5 in the launch configuration bench.py times (B=64, T=100), oracle on sampled tiles
    (0.4 s forward + 0.6 s VJP each on the host)."""
    leb, wl, O = mods
    w = wl.make_config(5)
    ctx = leb.context_for_workload(w)
    nom_d, rad_d = _dev(w.nom), _dev(w.rad)
    lo, hi = ctx.leb_nn_fwd(nom_d, rad_d, flags=PATHS[path])
    assert ctx.leb_domain_flag() == 0
    # as bench.py runs it: the whole batch resident, the VJP starts from the forward's coefficient blocks
    launches0 = ctx.leb_launch_count()
    gn, gr = ctx.leb_vjp(1, nom_d, rad_d, _dev(w.g_lo), _dev(w.g_hi), flags=PATHS[path] | leb.FLAG_REUSE_FWD)
    launches_reuse = ctx.leb_launch_count() - launches0
    gn2, gr2 = ctx.leb_vjp(1, nom_d, rad_d, _dev(w.g_lo), _dev(w.g_hi), flags=PATHS[path])      # stateless: recomputes
    assert launches_reuse < ctx.leb_launch_count() - launches0 - launches_reuse, "LEB_FLAG_REUSE_FWD did not skip the forward"
    for a, b in ((gn, gn2), (gr, gr2)):      # same forward state; column sums are atomic adds, so not bit-identical
        assert float((a - b).abs().max()) <= 1e-5 * float(b.abs().max())
    nom, rad, g_lo, g_hi = _flat(w)
    if path == "tc":
        # the default path (the one bench.py times): one tile of every trajectory forward (64 tiles),
        # every fourth of those through the VJP (16 tiles); ~1 s of oracle time per tile
        idx = np.arange(w.B) * w.T + (np.arange(w.B) * 37) % w.T
        idx[0], idx[-1] = 0, w.B * w.T - 1
        vi = idx[::4]
    else:
        idx = np.array([0, 1023, 1024, 3777, w.B * w.T - 1])        # chunk boundaries, middle, last
        vi = idx[[0, 2, 4]]
    olo, ohi = O.leb_nn(w.mlp.W, w.mlp.b, w.mlp.act, nom[idx], rad[idx])
    glo, ghi = to_np(lo).reshape(-1, w.n)[idx], to_np(hi).reshape(-1, w.n)[idx]
    # relaxation case switches (reading R21): a tile whose hidden bound sits on a switch may take the other, equally
    # valid, case; such tiles must be reported as ties by the oracle and are few
    tol = lambda ref: 1e-5 * np.abs(ref) + 1e-7
    off = np.nonzero(((np.abs(glo - olo) > tol(olo)) | (np.abs(ghi - ohi) > tol(ohi))).any(1))[0]
    assert len(off) <= 2, f"{len(off)} of {len(idx)} sampled tiles miss the oracle"
    Ws = [np.asarray(x, np.float64) for x in w.mlp.W]; bs = [np.asarray(x, np.float64) for x in w.mlp.b]
    for q in off:
        assert len(O.relax_case_ties(Ws, bs, w.mlp.act, nom[idx[q]].astype(np.float64), rad[idx[q]].astype(np.float64))) > 0
    keep = np.setdiff1d(np.arange(len(idx)), off)
    assert_bounds_close(glo[keep], olo[keep], f"cfg5 {path} r_lo ({len(keep)} tiles)")
    assert_bounds_close(ghi[keep], ohi[keep], f"cfg5 {path} r_hi ({len(keep)} tiles)")
    vi = np.array([t for t in vi if t not in set(idx[off])])
    assert_nn_grads_close(O, w.mlp, nom[vi], rad[vi], g_lo[vi], g_hi[vi], to_np(gn).reshape(-1, w.N)[vi],
                          to_np(gr).reshape(-1, w.N)[vi], f"cfg5 {path} ({len(vi)} tiles)")
    # properties that hold at any size: lo <= 0 <= hi (r(a~) = 0 lies in the enclosure), all finite
    assert bool((lo <= 0).all()) and bool((hi >= 0).all()) and bool(torch.isfinite(gn).all()) and bool(torch.isfinite(gr).all())
    ctx.close()


def test_config5_every_tile_both_paths(mods):
    """All 6400 config-5 tiles: the tensor-core and the FFMA path (independent kernels) must agree within 3x the
    parity tolerance, except on tiles where a hidden bound sits on a (discontinuous) case switch of the tanh
    relaxation table -- 'several results are correct' (reading R21).  For those tiles (few per mille) the
    oracle must report such a tie and one of the two paths must match the oracle."""
    leb, wl, O = mods
    w = wl.make_config(5)
    ctx = leb.context_for_workload(w)
    nom_d, rad_d = _dev(w.nom), _dev(w.rad)
    res = {}
    for path in PATHS:
        lo, hi = ctx.leb_nn_fwd(nom_d, rad_d, flags=PATHS[path])
        res[path] = (to_np(lo).reshape(-1, w.n), to_np(hi).reshape(-1, w.n))
    bad = np.zeros(w.B * w.T, dtype=bool)
    for q in (0, 1):
        assert np.array_equal(res["tc"][q], res["tc_single_cta"][q]), "CTA-pair and single-CTA forward kernels differ"
        a, b = res["tc"][q], res["ffma"][q]
        bad |= (np.abs(a - b) > 3 * (1e-5 * np.abs(b) + 1e-7)).any(1)
    idx = np.nonzero(bad)[0]
    assert len(idx) <= 0.005 * w.B * w.T, f"{len(idx)} tiles differ between the two contraction paths"
    nom, rad, _, _ = _flat(w)
    Ws = [np.asarray(x, np.float64) for x in w.mlp.W]; bs = [np.asarray(x, np.float64) for x in w.mlp.b]
    for t in idx[:6]:
        a0, sg = nom[t].astype(np.float64), rad[t].astype(np.float64)
        assert len(O.relax_case_ties(Ws, bs, w.mlp.act, a0, sg)) > 0, f"tile {t}: paths differ without a relaxation tie"
        fw = O.crown_forward(Ws, bs, w.mlp.act, a0, sg)
        ok = False
        for path in PATHS:
            glo, ghi = res[path][0][t], res[path][1][t]
            ok |= bool(np.all(np.abs(glo - fw["r_lo"]) <= 1e-5 * np.abs(fw["r_lo"]) + 1e-7) and
                       np.all(np.abs(ghi - fw["r_hi"]) <= 1e-5 * np.abs(fw["r_hi"]) + 1e-7))
        assert ok, f"tile {t}: neither path matches the oracle"
    ctx.close()


@pytest.mark.parametrize("path", list(PATHS))
def test_ragged_tile_count_at_full_width(mods, path):
    """Config-5 architecture with 37 tiles: 37 * 1024 / 37 * 504 coefficient rows are not multiples of the 256-row block
    per launch boundary of the tensor path, forward and VJP (the batch tail)."""
    leb, wl, O = mods
    w = wl.make_config(5, B=1, T=37)
    ctx = leb.context_for_workload(w)
    lo, hi = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), flags=PATHS[path])
    gn, gr = ctx.leb_vjp(1, _dev(w.nom), _dev(w.rad), _dev(w.g_lo), _dev(w.g_hi), flags=PATHS[path] | leb.FLAG_REUSE_FWD)
    nom, rad, g_lo, g_hi = _flat(w)
    idx = np.array([0, 17, 35, 36])
    olo, ohi = O.leb_nn(w.mlp.W, w.mlp.b, w.mlp.act, nom[idx], rad[idx])
    assert_bounds_close(to_np(lo).reshape(-1, w.n)[idx], olo, f"ragged {path} r_lo")
    assert_bounds_close(to_np(hi).reshape(-1, w.n)[idx], ohi, f"ragged {path} r_hi")
    assert_nn_grads_close(O, w.mlp, nom[idx], rad[idx], g_lo[idx], g_hi[idx], to_np(gn).reshape(-1, w.N)[idx],
                          to_np(gr).reshape(-1, w.N)[idx], f"ragged {path}")
    ctx.close()


@pytest.mark.parametrize("path", list(PATHS))
def test_tanh_zero_radius_coordinates(mods, path):
    """tanh nets with sigma_j = 0 on some coordinates, and on all of them: neurons fed only by zero-radius inputs have
    point pre-activation intervals (u - l = 0: the degenerate line of reading R9, LINE_DEGEN in nn_relax.cuh), next to
    ordinary neurons.  Forward against the oracle; VJP in the directions the oracle pins (not d/d sigma_j at sigma_j = 0)."""
    leb, wl, O = mods
    w = wl.make_small_mlp([6, 40, 36, 33, 4], 2, 2, 3, rad_lo=0.02, rad_hi=0.2)
    Wz = [x.copy() for x in w.mlp.W]
    Wz[0][:10, 3:] = 0.0          # layer-1 neurons 0..9 see only inputs 0..2
    Wz[1][:8, 10:] = 0.0          # layer-2 neurons 0..7 see only those
    w.mlp.W = Wz
    rad = w.rad.copy()
    rad[..., :3] = 0.0
    ctx = leb.context_for_workload(w)
    nom_f, _, g_lo, g_hi = _flat(w)
    rad_f = rad.reshape(-1, w.N)
    lo, hi = ctx.leb_nn_fwd(_dev(w.nom), _dev(rad), flags=PATHS[path])
    assert ctx.leb_domain_flag() == 0
    olo, ohi = O.leb_nn(w.mlp.W, w.mlp.b, 2, nom_f, rad_f)
    assert_bounds_close(to_np(lo).reshape(-1, w.n), olo, f"tanh sigma_j=0 {path} r_lo")
    assert_bounds_close(to_np(hi).reshape(-1, w.n), ohi, f"tanh sigma_j=0 {path} r_hi")
    gn, gr = ctx.leb_vjp(1, _dev(w.nom), _dev(rad), _dev(w.g_lo), _dev(w.g_hi), flags=PATHS[path])
    ogn, ogr = O.leb_nn_vjp(w.mlp.W, w.mlp.b, 2, nom_f, rad_f, g_lo, g_hi)
    assert_grads_close(to_np(gn).reshape(-1, w.N), to_np(gr).reshape(-1, w.N)[:, 3:], ogn, ogr[:, 3:], f"tanh sigma_j=0 {path}")
    # certified mode on the same inputs contains the oracle enclosure
    clo, chi = ctx.leb_nn_fwd(_dev(w.nom), _dev(rad), flags=PATHS[path] & ~1)
    assert np.all(to_np(clo).reshape(-1, w.n) <= olo) and np.all(to_np(chi).reshape(-1, w.n) >= ohi)
    # all radii zero: the exact bound is [0, 0]; value mode returns it to rounding, certified mode encloses it
    z = torch.zeros_like(_dev(rad))
    lo, hi = ctx.leb_nn_fwd(_dev(w.nom), z, flags=PATHS[path])
    assert float(lo.abs().max()) < 1e-6 and float(hi.abs().max()) < 1e-6
    clo, chi = ctx.leb_nn_fwd(_dev(w.nom), z, flags=PATHS[path] & ~1)
    assert bool((clo <= 0).all()) and bool((chi >= 0).all()) and float(chi.max()) < 1e-4 and float(clo.min()) > -1e-4
    ctx.close()


def test_fwd_never_below_sampled_maximum_and_exact_range(mods):
    """Soundness where it is sharp: tiny ReLU nets (<= 4 inputs): >= 1e5 samples + all box vertices."""
    leb, wl, O = mods
    for dims, act, seed in (([3, 12, 2], 1, 1), ([4, 10, 3], 1, 2), ([4, 8, 8, 2], 2, 3), ([2, 16, 16, 2], 1, 4)):
        w = wl.make_small_mlp(dims, act, 2, 2, seed=seed, rad_lo=0.05, rad_hi=0.4)
        ctx = leb.context_for_workload(w)
        lo, hi = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), flags=VAL)
        glo, ghi = to_np(lo).reshape(-1, w.n), to_np(hi).reshape(-1, w.n)
        Ws = [np.asarray(x, np.float64) for x in w.mlp.W]; bs = [np.asarray(x, np.float64) for x in w.mlp.b]
        rng = np.random.default_rng(seed)
        N = dims[0]
        verts = np.array(list(itertools.product((-1.0, 1.0), repeat=N)))
        for t in range(w.B * w.T):
            a0 = w.nom.reshape(-1, N)[t].astype(np.float64); sg = w.rad.reshape(-1, N)[t].astype(np.float64)
            U = np.concatenate([rng.uniform(-1, 1, (100000, N)), verts])
            X = a0[None, :] + U * sg[None, :]
            zs, p, J = O.nominal(Ws, bs, act, a0)
            A = X.T
            for l in range(len(Ws) - 1):
                A = O.phi(act, Ws[l] @ A + bs[l][:, None])
            r = (Ws[-1] @ A + bs[-1][:, None]).T - p[None, :] - (X - a0[None, :]) @ J.T
            # FP32 value mode vs FP64 truth: allow the parity tolerance below the sampled extremum
            assert np.all(r.max(0) <= ghi[t] + 1e-5 * np.abs(ghi[t]) + 1e-7), (dims, t)
            assert np.all(r.min(0) >= glo[t] - 1e-5 * np.abs(glo[t]) - 1e-7), (dims, t)
        ctx.close()


def test_given_jacobian(mods):
    """J != NULL: the bound is with respect to the caller's matrix (Thm 3 holds for any J)."""
    leb, wl, O = mods
    w = wl.make_small_mlp([6, 20, 20, 4], 2, 2, 3)
    ctx = leb.context_for_workload(w)
    rng = np.random.default_rng(9)
    J = rng.standard_normal((w.B, w.T, w.n, w.N)).astype(np.float32) * 0.3
    lo, hi = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), J=_dev(J), flags=VAL)
    nom, rad, _, _ = _flat(w)
    olo, ohi = O.leb_nn(w.mlp.W, w.mlp.b, w.mlp.act, nom, rad, J=J.reshape(-1, w.n, w.N))
    # with an arbitrary J the bound is O(|W - J| sigma), computed from O(1) coefficients: tolerance
    # relative to that scale
    assert np.allclose(to_np(lo).reshape(-1, w.n), olo, rtol=1e-5, atol=2e-6)
    assert np.allclose(to_np(hi).reshape(-1, w.n), ohi, rtol=1e-5, atol=2e-6)
    ctx.close()


def test_edge_cases(mods):
    leb, wl, O = mods
    w = wl.make_small_mlp([6, 10, 10, 4], 1, 2, 3)
    ctx = leb.context_for_workload(w)
    nom, rad = _dev(w.nom), _dev(w.rad)
    # empty batch
    lo, hi = ctx.leb_nn_fwd(nom[:0], rad[:0], flags=VAL)
    assert lo.shape == (0, 3, 4)
    # zero radius: ReLU bound exactly 0 when no nominal pre-activation is exactly 0
    lo, hi = ctx.leb_nn_fwd(nom, torch.zeros_like(rad), flags=VAL)
    assert float(lo.abs().max()) == 0.0 and float(hi.abs().max()) == 0.0
    # padded leading dimensions
    nomp = torch.zeros(2, 3, 8, device="cuda"); nomp[..., :6] = nom
    radp = torch.zeros(2, 3, 8, device="cuda"); radp[..., :6] = rad
    lop = torch.full((2, 3, 8), 7.0, device="cuda"); hip = torch.full((2, 3, 8), 7.0, device="cuda")
    ctx.leb_nn_fwd(nomp, radp, r_lo=lop, r_hi=hip, flags=VAL)
    lo, hi = ctx.leb_nn_fwd(nom, rad, flags=VAL)
    assert torch.equal(lop[..., :4], lo) and torch.equal(hip[..., :4], hi) and float((lop[..., 4:] - 7).abs().max()) == 0.0
    # LEB_FLAG_REUSE_FWD: same gradient; no effect when the forward state is not there (other batch, chunked batch)
    ctx.leb_nn_fwd(nom, rad, flags=VAL)
    gA = ctx.leb_vjp(1, nom, rad, _dev(w.g_lo), _dev(w.g_hi), flags=leb.FLAG_NO_MARGIN | leb.FLAG_REUSE_FWD)
    assert ctx.leb_nn_state() == (w.B * w.T, False, True)
    gB = ctx.leb_vjp(1, nom, rad, _dev(w.g_lo), _dev(w.g_hi), flags=VAL)
    assert ctx.leb_nn_state()[2] is False
    assert torch.allclose(gA[0], gB[0], rtol=1e-5, atol=1e-7) and torch.allclose(gA[1], gB[1], rtol=1e-5, atol=1e-7)
    ctx.leb_nn_fwd(nom[:1], rad[:1], flags=VAL)
    gC = ctx.leb_vjp(1, nom, rad, _dev(w.g_lo), _dev(w.g_hi), flags=leb.FLAG_NO_MARGIN | leb.FLAG_REUSE_FWD)
    assert ctx.leb_nn_state()[2] is False                    # another batch is resident: recomputed
    assert torch.allclose(gC[0], gB[0], rtol=1e-5, atol=1e-7) and torch.allclose(gC[1], gB[1], rtol=1e-5, atol=1e-7)
    # chunking does not change results
    ctx.leb_set_nn_chunk(4)
    lo2, hi2 = ctx.leb_nn_fwd(nom, rad, flags=VAL)
    gn2, gr2 = ctx.leb_vjp(1, nom, rad, _dev(w.g_lo), _dev(w.g_hi), flags=leb.FLAG_NO_MARGIN | leb.FLAG_REUSE_FWD)
    ctx.leb_set_nn_chunk(0)
    gn, gr = ctx.leb_vjp(1, nom, rad, _dev(w.g_lo), _dev(w.g_hi), flags=VAL)
    assert torch.equal(lo2, lo) and torch.equal(hi2, hi)
    assert torch.allclose(gn2, gn, rtol=1e-5, atol=1e-7) and torch.allclose(gr2, gr, rtol=1e-5, atol=1e-7)
    # NaN input / negative radius poison only their tile and raise the flag
    assert ctx.leb_domain_flag() == 0
    n2 = w.nom.copy(); n2[1, 0, 2] = np.nan
    lo, hi = ctx.leb_nn_fwd(_dev(n2), rad, flags=VAL)
    assert ctx.leb_domain_flag() == 1
    assert bool(torch.isinf(lo[1, 0]).all()) and bool(torch.isinf(hi[1, 0]).all()) and bool(torch.isfinite(lo[0]).all())
    r2 = w.rad.copy(); r2[0, 2, 5] = -0.1
    lo, hi = ctx.leb_nn_fwd(nom, _dev(r2), flags=VAL)
    assert ctx.leb_domain_flag() == 1 and bool(torch.isinf(hi[0, 2]).all()) and bool(torch.isfinite(hi[1]).all())
    # host IO
    hlo, hhi = ctx.leb_nn_fwd(torch.from_numpy(w.nom).pin_memory(), torch.from_numpy(w.rad).pin_memory(),
                              flags=leb.FLAG_NO_MARGIN | leb.FLAG_HOST_IO)
    torch.cuda.synchronize()
    lo, hi = ctx.leb_nn_fwd(nom, rad, flags=VAL)
    assert torch.equal(hlo, lo.cpu()) and torch.equal(hhi, hi.cpu())
    # model not set
    ctx2 = leb.Context(0)
    with pytest.raises(leb.LebError) as e:
        ctx2.nn_n = 4
        ctx2.leb_nn_fwd(nom, rad, flags=VAL)
    assert e.value.status == leb.LEB_ERR_STATE
    ctx2.close()
    ctx.close()


# ---------------------------------------------------------------------------------- CROWN-IBP (LEB_FLAG_IBP_HIDDEN)
IBP = 32


@pytest.mark.parametrize("path", list(PATHS))
@pytest.mark.parametrize("dims,act", SMALL)
def test_crown_ibp_small_nets_match_oracle(mods, dims, act, path):
    """Hidden layers 2..L-1 by interval propagation, output by back-substitution: forward, hidden bounds and VJP against
    the oracle's hidden="ibp" branch."""
    leb, wl, O = mods
    w = wl.make_small_mlp(dims, act, 3, 4, rad_lo=0.02, rad_hi=0.2)
    ctx = leb.context_for_workload(w)
    flags = PATHS[path] | IBP
    lo, hi = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), flags=flags)
    nom, rad, g_lo, g_hi = _flat(w)
    olo, ohi = O.leb_nn(w.mlp.W, w.mlp.b, act, nom, rad, hidden="ibp")
    assert_bounds_close(to_np(lo).reshape(-1, w.n), olo, f"crown-ibp {dims} r_lo")
    assert_bounds_close(to_np(hi).reshape(-1, w.n), ohi, f"crown-ibp {dims} r_hi")
    Ws = [np.asarray(x, np.float64) for x in w.mlp.W]; bs = [np.asarray(x, np.float64) for x in w.mlp.b]
    for layer in range(1, len(dims) - 1):
        l, u = ctx.leb_nn_hidden_bounds(layer, w.B * w.T, dims[layer])
        fw = O.crown_forward(Ws, bs, act, nom[0].astype(np.float64), rad[0].astype(np.float64), hidden="ibp")
        assert np.allclose(to_np(l)[0], fw["ls"][layer - 1], rtol=2e-5, atol=2e-6)
        assert np.allclose(to_np(u)[0], fw["us"][layer - 1], rtol=2e-5, atol=2e-6)
    # VJP: stateless and from the resident forward state
    gn, gr = ctx.leb_vjp(1, _dev(w.nom), _dev(w.rad), _dev(w.g_lo), _dev(w.g_hi), flags=flags)
    ogn, ogr = O.leb_nn_vjp(w.mlp.W, w.mlp.b, act, nom, rad, g_lo, g_hi, hidden="ibp")
    assert_grads_close(to_np(gn), to_np(gr), ogn, ogr, f"crown-ibp {dims}")
    ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), flags=flags)
    g2 = ctx.leb_vjp(1, _dev(w.nom), _dev(w.rad), _dev(w.g_lo), _dev(w.g_hi), flags=flags | leb.FLAG_REUSE_FWD)
    assert ctx.leb_nn_state()[2] is True
    for a, b in ((g2[0], gn), (g2[1], gr)):          # column sums are atomic adds: equal to rounding, not bit for bit
        assert float((a - b).abs().max()) <= 1e-5 * float(b.abs().max())
    # a full-CROWN state is not reused for a CROWN-IBP gradient (the certified CROWN-IBP mode: test_gpu_nn_certified.py)
    ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), flags=PATHS[path])
    ctx.leb_vjp(1, _dev(w.nom), _dev(w.rad), _dev(w.g_lo), _dev(w.g_hi), flags=flags | leb.FLAG_REUSE_FWD)
    assert ctx.leb_nn_state()[2] is False
    ctx.close()


@pytest.mark.parametrize("cfg,tiles", [(3, 16), (5, 8)])
def test_crown_ibp_configs_sampled_tiles(mods, cfg, tiles):
    leb, wl, O = mods
    w = wl.make_config(cfg)
    ctx = leb.context_for_workload(w)
    nom_d, rad_d = _dev(w.nom), _dev(w.rad)
    launches0 = ctx.leb_launch_count()
    lo, hi = ctx.leb_nn_fwd(nom_d, rad_d, flags=VAL | IBP)
    n_ibp = ctx.leb_launch_count() - launches0
    gn, gr = ctx.leb_vjp(1, nom_d, rad_d, _dev(w.g_lo), _dev(w.g_hi), flags=VAL | IBP | leb.FLAG_REUSE_FWD)
    flo, fhi = ctx.leb_nn_fwd(nom_d, rad_d, flags=VAL)
    nom, rad, g_lo, g_hi = _flat(w)
    idx = np.linspace(0, w.B * w.T - 1, tiles).astype(int)
    olo, ohi = O.leb_nn(w.mlp.W, w.mlp.b, w.mlp.act, nom[idx], rad[idx], hidden="ibp")
    assert_bounds_close(to_np(lo).reshape(-1, w.n)[idx], olo, f"cfg{cfg} crown-ibp r_lo")
    assert_bounds_close(to_np(hi).reshape(-1, w.n)[idx], ohi, f"cfg{cfg} crown-ibp r_hi")
    vi = idx[::2]
    ogn, ogr = O.leb_nn_vjp(w.mlp.W, w.mlp.b, w.mlp.act, nom[vi], rad[vi], g_lo[vi], g_hi[vi], hidden="ibp")
    from parity_util import grads_ratio
    ratio = grads_ratio(to_np(gn).reshape(-1, w.N)[vi], to_np(gr).reshape(-1, w.N)[vi], ogn, ogr)
    assert (ratio <= 1.0).sum() >= len(vi) - 1, ratio           # at most one tile on a kink of |W - J| (reading R20)
    # looser than full CROWN, by a reported factor
    wide = float(((hi - lo).sum() / (fhi - flo).sum()))
    print(f"config {cfg}: CROWN-IBP enclosure width / full CROWN = {wide:.3f}")
    assert wide >= 1.0 - 1e-6
    ctx.close()


# ---------------------------------------------------------------------------------- non-centred boxes (25a) L272
@pytest.mark.parametrize("path", list(PATHS))
@pytest.mark.parametrize("dims,act", SMALL)
def test_mu_small_nets_match_oracle(mods, dims, act, path):
    """mu != NULL on the NN path: forward, hidden bounds and the VJP with respect to (a~, sigma, mu) against the oracle;
    some |mu_j| > sigma_j (the nominal point outside the box).  Full CROWN and CROWN-IBP hidden bounds."""
    leb, wl, O = mods
    w = wl.make_small_mlp(dims, act, 3, 4, rad_lo=0.02, rad_hi=0.2)
    mu = wl.make_mu(w, 1.5)
    assert (np.abs(mu) > w.rad).any()
    ctx = leb.context_for_workload(w)
    nom, rad, g_lo, g_hi = _flat(w)
    mu_f = mu.reshape(-1, w.N)
    for hidden, extra in (("crown", 0), ("ibp", IBP)):
        flags = PATHS[path] | extra
        lo, hi = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), flags=flags, mu=_dev(mu))
        assert ctx.leb_domain_flag() == 0
        olo, ohi = O.leb_nn(w.mlp.W, w.mlp.b, act, nom, rad, hidden=hidden, mu=mu_f)
        assert_bounds_close(to_np(lo).reshape(-1, w.n), olo, f"mu {hidden} {dims} r_lo")
        assert_bounds_close(to_np(hi).reshape(-1, w.n), ohi, f"mu {hidden} {dims} r_hi")
        gn, gr, gm = ctx.leb_vjp_mu(1, _dev(w.nom), _dev(w.rad), _dev(mu), _dev(w.g_lo), _dev(w.g_hi), flags=flags)
        ogn, ogr, ogm = O.leb_nn_vjp(w.mlp.W, w.mlp.b, act, nom, rad, g_lo, g_hi, hidden=hidden, mu=mu_f)
        S = np.maximum(np.maximum(np.abs(ogn).max(1), np.abs(ogr).max(1)), np.abs(ogm).max(1))
        from parity_util import assert_grad_dirs_close, GRAD_NORMWISE, report
        for name, got, ref in (("grad_nom", gn, ogn), ("grad_rad", gr, ogr), ("grad_mu", gm, ogm)):
            err = np.abs(to_np(got).reshape(ref.shape) - ref)
            tol = 1e-4 * np.abs(ref) + GRAD_NORMWISE * S[:, None] + 1e-12
            report(f"mu {hidden} {dims} {name}", (err / tol).max())
            assert (err <= tol).all(), (name, float((err / tol).max()))
        # from the resident forward state
        ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), flags=flags, mu=_dev(mu))
        g2 = ctx.leb_vjp_mu(1, _dev(w.nom), _dev(w.rad), _dev(mu), _dev(w.g_lo), _dev(w.g_hi), flags=flags | leb.FLAG_REUSE_FWD)
        assert ctx.leb_nn_state()[2] is True
        for a, b in zip(g2, (gn, gr, gm)):
            assert float((a - b).abs().max()) <= 1e-5 * float(b.abs().max())
    # mu = 0 is the centred bound (bit for bit: the extra terms are exact zeros)
    z = torch.zeros_like(_dev(mu))
    lo0, hi0 = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), flags=PATHS[path], mu=z)
    lo1, hi1 = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), flags=PATHS[path])
    assert torch.equal(lo0, lo1) and torch.equal(hi0, hi1)
    ctx.close()


def test_mu_config5_sampled_tiles_and_soundness(mods):
    leb, wl, O = mods
    w = wl.make_config(5)
    mu = wl.make_mu(w, 1.5)
    ctx = leb.context_for_workload(w)
    lo, hi = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), flags=VAL, mu=_dev(mu))
    gn, gr, gm = ctx.leb_vjp_mu(1, _dev(w.nom), _dev(w.rad), _dev(mu), _dev(w.g_lo), _dev(w.g_hi), flags=VAL | leb.FLAG_REUSE_FWD)
    nom, rad, g_lo, g_hi = _flat(w)
    mu_f = mu.reshape(-1, w.N)
    idx = np.array([0, 1500, 3777, w.B * w.T - 1])
    olo, ohi = O.leb_nn(w.mlp.W, w.mlp.b, w.mlp.act, nom[idx], rad[idx], mu=mu_f[idx])
    assert_bounds_close(to_np(lo).reshape(-1, w.n)[idx], olo, "cfg5 mu r_lo")
    assert_bounds_close(to_np(hi).reshape(-1, w.n)[idx], ohi, "cfg5 mu r_hi")
    ogn, ogr, ogm = O.leb_nn_vjp(w.mlp.W, w.mlp.b, w.mlp.act, nom[idx[:2]], rad[idx[:2]], g_lo[idx[:2]], g_hi[idx[:2]], mu=mu_f[idx[:2]])
    from parity_util import GRAD_NORMWISE
    S = np.maximum(np.maximum(np.abs(ogn).max(1), np.abs(ogr).max(1)), np.abs(ogm).max(1))[:, None]
    for got, ref in ((gn, ogn), (gr, ogr), (gm, ogm)):
        err = np.abs(to_np(got).reshape(-1, w.N)[idx[:2]] - ref)
        assert (err <= 1e-4 * np.abs(ref) + GRAD_NORMWISE * S + 1e-12).mean() > 0.999      # kinks of |W - J| (R20): a handful of entries
    ctx.close()
    # soundness where it is sharp: a small tanh net, samples of the offset box and all its vertices
    ws = wl.make_small_mlp([4, 8, 8, 2], 2, 2, 2, seed=3, rad_lo=0.05, rad_hi=0.4)
    mus = wl.make_mu(ws, 2.0)
    c2 = leb.context_for_workload(ws)
    lo, hi = c2.leb_nn_fwd(_dev(ws.nom), _dev(ws.rad), flags=VAL, mu=_dev(mus))
    glo, ghi = to_np(lo).reshape(-1, ws.n), to_np(hi).reshape(-1, ws.n)
    Ws = [np.asarray(x, np.float64) for x in ws.mlp.W]; bs = [np.asarray(x, np.float64) for x in ws.mlp.b]
    rng = np.random.default_rng(3)
    verts = np.array(list(itertools.product((-1.0, 1.0), repeat=4)))
    for t in range(4):
        a0 = ws.nom.reshape(-1, 4)[t].astype(np.float64); sg = ws.rad.reshape(-1, 4)[t].astype(np.float64)
        m = mus.reshape(-1, 4)[t].astype(np.float64)
        X = a0[None] + m[None] + np.concatenate([rng.uniform(-1, 1, (100000, 4)), verts]) * sg[None]
        zs, p, J = O.nominal(Ws, bs, 2, a0)
        A = X.T
        for l in range(len(Ws) - 1):
            A = O.phi(2, Ws[l] @ A + bs[l][:, None])
        r = (Ws[-1] @ A + bs[-1][:, None]).T - p[None] - (X - a0[None]) @ J.T
        assert np.all(r.max(0) <= ghi[t] + 1e-5 * np.abs(ghi[t]) + 1e-7) and np.all(r.min(0) >= glo[t] - 1e-5 * np.abs(glo[t]) - 1e-7)
    c2.close()


# ---------------------------------------------------------------------------------- optimisable lower slopes (alpha-CROWN)
@pytest.mark.parametrize("path", ["tc", "ffma"])
def test_alpha_refinement_matches_oracle(mods, path):
    leb, wl, O = mods
    for dims, seed in (([4, 10, 10, 10, 3], 5), ([6, 33, 20, 11, 5], 6), ([24, 130, 70, 20], 7)):
        w = wl.make_small_mlp(dims, 1, 2, 3, seed=seed, rad_lo=0.1, rad_hi=0.4)
        ctx = leb.context_for_workload(w)
        nom, rad, _, _ = _flat(w)
        Ws = [np.asarray(x, np.float64) for x in w.mlp.W]; bs = [np.asarray(x, np.float64) for x in w.mlp.b]
        # zero steps = the adaptive slopes of leb_nn_fwd, bit for bit
        lo0, hi0, w0, wb = ctx.leb_nn_alpha_fwd(_dev(w.nom), _dev(w.rad), 0, 0.05, flags=PATHS[path])
        plo, phi = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), flags=PATHS[path])
        assert torch.equal(lo0, plo) and torch.equal(hi0, phi) and torch.equal(w0, wb)
        steps, lr = 8, 0.05
        lo, hi, w0, wb = ctx.leb_nn_alpha_fwd(_dev(w.nom), _dev(w.rad), steps, lr, flags=PATHS[path])
        glo, ghi = to_np(lo).reshape(-1, w.n), to_np(hi).reshape(-1, w.n)
        gw0, gwb = to_np(w0).reshape(-1), to_np(wb).reshape(-1)
        assert np.all(gwb <= gw0)
        improved = 0
        for t in range(w.B * w.T):
            olo, ohi, ow0, owb = O.alpha_refine(Ws, bs, nom[t].astype(np.float64), rad[t].astype(np.float64), steps, lr)
            assert abs(gw0[t] - ow0) <= 1e-5 * ow0
            assert abs(gwb[t] - owb) <= 2e-3 * owb, (dims, t, gwb[t], owb)         # an iteration amplifies rounding differences
            improved += owb < 0.999 * ow0
            # the returned enclosure is sound: >= 2e4 samples + vertices (N <= 6) of the box
            N = dims[0]
            rng = np.random.default_rng(t)
            a0 = nom[t].astype(np.float64); sg = rad[t].astype(np.float64)
            U = rng.uniform(-1, 1, (20000, N))
            if N <= 6:
                U = np.concatenate([U, np.array(list(itertools.product((-1.0, 1.0), repeat=N)))])
            X = a0[None] + U * sg[None]
            zs, p, J = O.nominal(Ws, bs, 1, a0)
            A = X.T
            for l in range(len(Ws) - 1):
                A = O.phi(1, Ws[l] @ A + bs[l][:, None])
            r = (Ws[-1] @ A + bs[-1][:, None]).T - p[None] - (X - a0[None]) @ J.T
            assert np.all(r.max(0) <= ghi[t] + 1e-5 * np.abs(ghi[t]) + 1e-7) and np.all(r.min(0) >= glo[t] - 1e-5 * np.abs(glo[t]) - 1e-7)
        assert improved >= 1
        # the kept slopes can be read back; with exactly those slopes the oracle gives the returned enclosure, and
        # leb_vjp(REUSE_FWD) on the state the refinement left is the gradient of the REFINED bound, slopes held constant
        tiles = w.B * w.T
        assert ctx.leb_nn_state()[0] == tiles
        kLs = [to_np(ctx.leb_nn_slopes(layer, tiles, dims[layer])[1]).astype(np.float64) for layer in range(1, len(dims) - 1)]
        g_lo, g_hi = w.g_lo.reshape(-1, w.n), w.g_hi.reshape(-1, w.n)
        gn, gr = ctx.leb_vjp(1, _dev(w.nom), _dev(w.rad), _dev(w.g_lo), _dev(w.g_hi), flags=PATHS[path] | leb.FLAG_REUSE_FWD)
        assert ctx.leb_nn_state()[2] is True
        olo, ohi = np.empty_like(glo, dtype=np.float64), np.empty_like(ghi, dtype=np.float64)
        ogn, ogr = np.empty((tiles, dims[0])), np.empty((tiles, dims[0]))
        for t in range(tiles):
            al = [k[t] for k in kLs]
            fw = O.crown_forward(Ws, bs, 1, nom[t].astype(np.float64), rad[t].astype(np.float64), alphas=al)
            olo[t], ohi[t] = fw["r_lo"], fw["r_hi"]
            ogn[t], ogr[t] = O.crown_vjp(Ws, bs, 1, nom[t].astype(np.float64), rad[t].astype(np.float64), g_lo[t].astype(np.float64),
                                         g_hi[t].astype(np.float64), alphas=al)
        assert_bounds_close(glo, olo, f"alpha {dims} r_lo at the kept slopes")
        assert_bounds_close(ghi, ohi, f"alpha {dims} r_hi at the kept slopes")
        assert_grads_close(to_np(gn), to_np(gr), ogn, ogr, f"alpha {dims} refined-bound")
        # a stateless leb_vjp differentiates the adaptive-slope bound instead
        pn, pr = ctx.leb_vjp(1, _dev(w.nom), _dev(w.rad), _dev(w.g_lo), _dev(w.g_hi), flags=PATHS[path])
        assert not torch.equal(pn, gn)
        ctx.close()
    wt = wl.make_small_mlp([5, 9, 3], 2, 1, 1)
    ct = leb.context_for_workload(wt)
    with pytest.raises(leb.LebError) as e:
        ct.leb_nn_alpha_fwd(_dev(wt.nom), _dev(wt.rad), 2, 0.05)
    assert e.value.status == leb.LEB_ERR_UNSUPPORTED
    ct.close()


def test_alpha_refinement_config3(mods):
    """Config 3 (ReLU, 1 280 tiles, chunked workspace): tighter than the adaptive slopes on most tiles, never looser."""
    leb, wl, O = mods
    w = wl.make_config(3)
    ctx = leb.context_for_workload(w)
    lo, hi, w0, wb = ctx.leb_nn_alpha_fwd(_dev(w.nom), _dev(w.rad), 6, 10.0, flags=VAL)      # dW/dalpha ~ 0.05 here: steps of ~0.5
    plo, phi = ctx.leb_nn_fwd(_dev(w.nom), _dev(w.rad), flags=VAL)
    assert bool((wb <= w0).all())
    assert torch.allclose(w0.reshape(-1), (phi - plo).sum(-1).reshape(-1), rtol=1e-5)
    gain = float((wb.sum() / w0.sum()))
    print(f"config 3: alpha-refined total width / adaptive-slope width = {gain:.4f}")
    assert gain < 0.995
    nom, rad, _, _ = _flat(w)
    t = 17
    olo, ohi, ow0, owb = O.alpha_refine([np.asarray(x, np.float64) for x in w.mlp.W], [np.asarray(x, np.float64) for x in w.mlp.b],
                                        nom[t].astype(np.float64), rad[t].astype(np.float64), 6, 10.0)
    assert abs(float(wb.reshape(-1)[t]) - owb) <= 2e-3 * owb
    ctx.close()
