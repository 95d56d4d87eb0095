"""GPU parity: leb_analytic_fwd / leb_vjp(kind 0) / leb_zonotope_inflate through the C ABI against
the FP64 oracle, element by element on the same seeded inputs (Thm 1 eq. (15))."""
import numpy as np
import pytest
import torch

from parity_util import assert_bounds_close, assert_grad_dirs_close, to_np

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mods():
    from paper_2607_01203_b200 import build, leb, workloads
    from oracle import inflate_oracle, pbh_oracle
    build.build()
    pbh_oracle.build()
    return leb, workloads, pbh_oracle, inflate_oracle


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _true_r(P, spec, a0, X):
    J = P.jac(spec, a0)
    return P.f(spec, X) - P.f(spec, a0[None, :]) - (X - a0[None, :]) @ J.T


# ---------------------------------------------------------------------------------- forward
@pytest.mark.parametrize("cfg,tiles", [(1, None), (2, None), (4, 24)])
def test_fwd_matches_oracle(mods, cfg, tiles):
    """Configs 1 and 2 in full, config 4 launched at full size (the bench launch configuration)
    and compared on 24 sampled tiles (first ... last; every trajectory is hit)."""
    leb, wl, P, _ = mods
    w = wl.make_config(cfg)
    ctx = leb.context_for_workload(w)
    lo, hi = ctx.leb_analytic_fwd(_dev(w.nom), _dev(w.rad))
    assert ctx.leb_domain_flag() == 0
    nt = w.B * w.T
    idx = np.arange(nt) if tiles is None else np.linspace(0, nt - 1, tiles).astype(int)
    spec = P.spec_from_workload(w)
    olo, ohi, st = P.pbh(spec, w.nom.reshape(-1, w.N)[idx], w.rad.reshape(-1, w.N)[idx])
    assert st == 0
    glo, ghi = to_np(lo).reshape(-1, w.n)[idx], to_np(hi).reshape(-1, w.n)[idx]
    assert_bounds_close(glo, olo, f"cfg{cfg} r_lo")
    assert_bounds_close(ghi, ohi, f"cfg{cfg} r_hi")
    # directed rounding: the FP32 enclosure contains the exact-arithmetic one up to the oracle's own
    # FP64 rounding (1e-13 relative)
    assert np.all(glo <= olo + 1e-13 * np.abs(olo)) and np.all(ghi >= ohi - 1e-13 * np.abs(ohi))
    ctx.close()


def test_fwd_config4_never_below_sampled_maximum(mods):
    """Config 4 (N = 224: no vertex enumeration): 1e5 samples of the box on each of 4 tiles."""
    leb, wl, P, _ = mods
    w = wl.make_config(4)
    ctx = leb.context_for_workload(w)
    lo, hi = ctx.leb_analytic_fwd(_dev(w.nom), _dev(w.rad))
    glo, ghi = to_np(lo).reshape(-1, w.n), to_np(hi).reshape(-1, w.n)
    spec = P.spec_from_workload(w)
    rng = np.random.default_rng(104)
    for t in (0, 133, 266, 399):
        a0 = w.nom.reshape(-1, w.N)[t].astype(np.float64)
        sg = w.rad.reshape(-1, w.N)[t].astype(np.float64)
        r = _true_r(P, spec, a0, a0[None, :] + rng.uniform(-1, 1, (100000, w.N)) * sg[None, :])
        assert np.all(r.max(0) <= ghi[t] + 1e-12) and np.all(r.min(0) >= glo[t] - 1e-12), t
    ctx.close()


@pytest.mark.parametrize("cfg,tiles", [(1, 20), (2, 6)])
def test_fwd_never_below_sampled_maximum(mods, cfg, tiles):
    """north_star: the GPU bound must never be below the sampled maximum of |r| (>= 1e5 samples
    plus every box vertex per tile; r evaluated from its definition (10) L133 in FP64)."""
    leb, wl, P, _ = mods
    w = wl.make_config(cfg)
    ctx = leb.context_for_workload(w)
    lo, hi = ctx.leb_analytic_fwd(_dev(w.nom), _dev(w.rad))
    glo, ghi = to_np(lo).reshape(-1, w.n), to_np(hi).reshape(-1, w.n)
    spec = P.spec_from_workload(w)
    rng = np.random.default_rng(100 + cfg)
    N = w.N
    verts = np.array([[1.0 if (v >> j) & 1 else -1.0 for j in range(N)] for v in range(2 ** N)])
    for t in range(tiles):
        a0 = w.nom.reshape(-1, N)[t].astype(np.float64)
        sg = w.rad.reshape(-1, N)[t].astype(np.float64)
        U = np.concatenate([rng.uniform(-1, 1, (100000, N)), verts])
        r = _true_r(P, spec, a0, a0[None, :] + U * sg[None, :])
        # 1e-12: FP64 rounding noise of the sampled r itself (r of a linear output is ~1e-17, its bound exactly 0)
        assert np.all(r.max(0) <= ghi[t] + 1e-12) and np.all(r.min(0) >= glo[t] - 1e-12), t
    ctx.close()


def test_fwd_small_chains_and_euler(mods):
    """Chain ends (1-3 units: every window shape), Euler and RK4."""
    leb, wl, P, _ = mods
    for U in (1, 2, 3, 5):
        for integ in (wl.INTEG_EULER, wl.INTEG_RK4):
            w = wl.make_small_chain(U, 2, 2, seed=U)
            w.analytic.integ = integ
            ctx = leb.context_for_workload(w)
            lo, hi = ctx.leb_analytic_fwd(_dev(w.nom), _dev(w.rad))
            olo, ohi, st = P.pbh(P.spec_from_workload(w), w.nom, w.rad)
            assert st == 0
            assert_bounds_close(to_np(lo).reshape(-1, w.n), olo, f"chain U={U} integ={integ} lo")
            assert_bounds_close(to_np(hi).reshape(-1, w.n), ohi, f"chain U={U} integ={integ} hi")
            ctx.close()


def test_fwd_edge_cases(mods):
    leb, wl, P, _ = mods
    w = wl.make_config(2, B=2, T=3)
    ctx = leb.context_for_workload(w)
    nom, rad = _dev(w.nom), _dev(w.rad)
    # empty batch
    lo, hi = ctx.leb_analytic_fwd(nom[:0], rad[:0])
    assert lo.shape == (0, 3, 12)
    # zero radii: bound exactly [0, 0] (reading R15)
    lo, hi = ctx.leb_analytic_fwd(nom, torch.zeros_like(rad))
    assert float(lo.abs().max()) == 0.0 and float(hi.abs().max()) == 0.0
    # some radii zero: same as the oracle
    r2 = w.rad.copy()
    r2[..., ::3] = 0.0
    lo, hi = ctx.leb_analytic_fwd(nom, _dev(r2))
    olo, ohi, _ = P.pbh(P.spec_from_workload(w), w.nom, r2)
    assert_bounds_close(to_np(lo).reshape(-1, 12), olo, "zero-radius coords lo")
    assert_bounds_close(to_np(hi).reshape(-1, 12), ohi, "zero-radius coords hi")
    # padded leading dimensions (ld_in 20 > N, ld_out 16 > n)
    nomp = torch.zeros(2, 3, 20, device="cuda"); nomp[..., :16] = nom
    radp = torch.zeros(2, 3, 20, device="cuda"); radp[..., :16] = rad
    lop = torch.full((2, 3, 16), 7.0, device="cuda"); hip = torch.full((2, 3, 16), 7.0, device="cuda")
    ctx.leb_analytic_fwd(nomp, radp, lop, hip)
    lo, hi = ctx.leb_analytic_fwd(nom, rad)
    assert torch.equal(lop[..., :12], lo) and torch.equal(hip[..., :12], hi)
    assert float((lop[..., 12:] - 7.0).abs().max()) == 0.0      # padding columns untouched
    # domain errors: NaN input, negative radius, cos(theta) box containing 0 -> (-inf, +inf) + flag
    assert ctx.leb_domain_flag() == 0
    n2 = w.nom.copy(); n2[0, 0, 3] = np.nan
    r3 = w.rad.copy(); r3[0, 1, 2] = -1.0
    n4 = w.nom.copy(); n4[1, 2, 4] = np.pi / 2          # theta box straddles pi/2: 1/cos unbounded
    for nn_, rr_, bad in ((n2, w.rad, (0, 0)), (w.nom, r3, (0, 1)), (n4, w.rad, (1, 2))):
        lo, hi = ctx.leb_analytic_fwd(_dev(nn_), _dev(rr_))
        assert ctx.leb_domain_flag() == 1
        assert bool(torch.isinf(lo[bad]).all()) and bool(torch.isinf(hi[bad]).all())
        ok = torch.ones(2, 3, dtype=torch.bool, device="cuda"); ok[bad] = False
        assert bool(torch.isfinite(lo[ok]).all()) and bool(torch.isfinite(hi[ok]).all())
    assert ctx.leb_domain_flag() == 0                    # reading clears the flag
    ctx.close()


def test_fwd_host_io_equals_device_io(mods):
    leb, wl, _, _ = mods
    w = wl.make_config(2, B=3, T=5)
    ctx = leb.context_for_workload(w)
    lo, hi = ctx.leb_analytic_fwd(_dev(w.nom), _dev(w.rad))
    hlo, hhi = ctx.leb_analytic_fwd(torch.from_numpy(w.nom).pin_memory(), torch.from_numpy(w.rad).pin_memory(),
                                    flags=leb.FLAG_HOST_IO)
    torch.cuda.synchronize()
    assert not hlo.is_cuda and torch.equal(hlo, lo.cpu()) and torch.equal(hhi, hi.cpu())
    ctx.close()


# ---------------------------------------------------------------------------------- VJP
@pytest.mark.parametrize("cfg,tiles", [(1, 20), (2, 24), (4, 4)])
def test_vjp_matches_oracle(mods, cfg, tiles):
    """Every one of the 2N directions against the oracle's forward-mode duals; the whole batch is launched (config 4:
    the bench launch configuration) and `tiles` sampled tiles are compared (config 4: 4 tiles x 448 directions, the
    oracle costs ~0.5 s per tile and direction on one core).  The tolerance scale is the ORACLE's gradient."""
    leb, wl, P, _ = mods
    w = wl.make_config(cfg)
    ctx = leb.context_for_workload(w)
    N, n = w.N, w.n
    gn, gr = ctx.leb_vjp(0, _dev(w.nom), _dev(w.rad), _dev(w.g_lo), _dev(w.g_hi))
    assert ctx.leb_domain_flag() == 0
    idx = np.linspace(0, w.B * w.T - 1, tiles).astype(int)
    g = np.concatenate([to_np(gn).reshape(-1, N), to_np(gr).reshape(-1, N)], 1)[idx]
    og, st = P.pbh_vjp(P.spec_from_workload(w), w.nom.reshape(-1, N)[idx], w.rad.reshape(-1, N)[idx],
                       w.g_lo.reshape(-1, n)[idx], w.g_hi.reshape(-1, n)[idx])
    assert st == 0
    assert_grad_dirs_close(g, og, np.abs(og).max(1), f"cfg{cfg} vjp")
    # bitwise reproducible: every reduction of the analytic path has a fixed order
    gn2, gr2 = ctx.leb_vjp(0, _dev(w.nom), _dev(w.rad), _dev(w.g_lo), _dev(w.g_hi))
    assert torch.equal(gn, gn2) and torch.equal(gr, gr2)
    ctx.close()


def test_vjp_small_chains_and_euler(mods):
    leb, wl, P, _ = mods
    for U in (1, 2, 3, 5):
        for integ in (wl.INTEG_EULER, wl.INTEG_RK4):
            w = wl.make_small_chain(U, 2, 2, seed=U)
            w.analytic.integ = integ
            ctx = leb.context_for_workload(w)
            gn, gr = ctx.leb_vjp(0, _dev(w.nom), _dev(w.rad), _dev(w.g_lo), _dev(w.g_hi))
            g = np.concatenate([to_np(gn).reshape(-1, w.N), to_np(gr).reshape(-1, w.N)], 1)
            og, st = P.pbh_vjp(P.spec_from_workload(w), w.nom, w.rad, w.g_lo, w.g_hi)
            assert st == 0
            assert_grad_dirs_close(g, og, np.abs(og).max(1), f"chain U={U} integ={integ} vjp")
            ctx.close()


# ---------------------------------------------------------------------------------- the paper's own systems (App. I)
@pytest.mark.parametrize("name", ["satellite", "planar_quad", "quad12_euler", "quadcentroid3", "quadcentroid8"])
def test_paper_systems_match_oracle(mods, name):
    """Satellite (36) L507-519, planar quadrotor (37) L521-528, 3-D quadrotor (38) with forward Euler (L505)."""
    leb, wl, P, _ = mods
    w = wl.make_paper_system(name, 5, 7) if name != "quadcentroid8" else wl.make_paper_system(name, 2, 3)      # 96-D: Table III
    ctx = leb.context_for_workload(w)
    spec = P.spec_from_workload(w)
    lo, hi = ctx.leb_analytic_fwd(_dev(w.nom), _dev(w.rad))
    assert ctx.leb_domain_flag() == 0
    olo, ohi, st = P.pbh(spec, w.nom, w.rad)
    assert st == 0
    assert_bounds_close(to_np(lo).reshape(-1, w.n), olo, f"{name} r_lo")
    assert_bounds_close(to_np(hi).reshape(-1, w.n), ohi, f"{name} r_hi")
    assert np.all(to_np(lo).reshape(-1, w.n) <= olo + 1e-13 * np.abs(olo)) and np.all(to_np(hi).reshape(-1, w.n) >= ohi - 1e-13 * np.abs(ohi))
    gn, gr = ctx.leb_vjp(0, _dev(w.nom), _dev(w.rad), _dev(w.g_lo), _dev(w.g_hi))
    g = np.concatenate([to_np(gn).reshape(-1, w.N), to_np(gr).reshape(-1, w.N)], 1)
    og, st = P.pbh_vjp(spec, w.nom, w.rad, w.g_lo, w.g_hi)
    assert st == 0
    assert_grad_dirs_close(g, og, np.abs(og).max(1), f"{name} vjp")
    ctx.close()


# ---------------------------------------------------------------------------------- non-centred boxes (25a) L272
@pytest.mark.parametrize("what", ["cfg1", "cfg2", "chain3", "satellite"])
def test_mu_matches_oracle(mods, what):
    """mu != NULL: box a~ + mu + [-sigma, sigma], D = [mu - sigma, mu + sigma], prefix hull sets (reading R4);
    forward and the VJP with respect to (a~, sigma, mu) against the oracle; some |mu_i| > sigma_i (a~ outside the box)."""
    leb, wl, P, _ = mods
    w = {"cfg1": lambda: wl.make_config(1), "cfg2": lambda: wl.make_config(2, B=4, T=6),
         "chain3": lambda: wl.make_small_chain(3, 2, 3), "satellite": lambda: wl.make_paper_system("satellite", 3, 5)}[what]()
    mu = wl.make_mu(w, 1.5)
    assert (np.abs(mu) > w.rad).any()
    ctx = leb.context_for_workload(w)
    spec = P.spec_from_workload(w)
    lo, hi = ctx.leb_analytic_fwd(_dev(w.nom), _dev(w.rad), mu=_dev(mu))
    assert ctx.leb_domain_flag() == 0
    olo, ohi, st = P.pbh(spec, w.nom, w.rad, mu=mu)
    assert st == 0
    glo, ghi = to_np(lo).reshape(-1, w.n), to_np(hi).reshape(-1, w.n)
    assert_bounds_close(glo, olo, f"mu {what} r_lo")
    assert_bounds_close(ghi, ohi, f"mu {what} r_hi")
    assert np.all(glo <= olo + 1e-13 * np.abs(olo)) and np.all(ghi >= ohi - 1e-13 * np.abs(ohi))
    gn, gr, gm = ctx.leb_vjp_mu(0, _dev(w.nom), _dev(w.rad), _dev(mu), _dev(w.g_lo), _dev(w.g_hi))
    g = np.concatenate([to_np(x).reshape(-1, w.N) for x in (gn, gr, gm)], 1)
    og, st = P.pbh_vjp(spec, w.nom, w.rad, w.g_lo, w.g_hi, mu=mu)
    assert st == 0
    assert_grad_dirs_close(g, og, np.abs(og).max(1), f"mu {what} vjp")
    # mu = 0 is the centred bound, bit for bit
    z = torch.zeros_like(_dev(mu))
    lo0, hi0 = ctx.leb_analytic_fwd(_dev(w.nom), _dev(w.rad), mu=z)
    lo1, hi1 = ctx.leb_analytic_fwd(_dev(w.nom), _dev(w.rad))
    assert torch.equal(lo0, lo1) and torch.equal(hi0, hi1)
    ctx.close()


def test_mu_soundness_off_centre(mods):
    """The GPU bound with the nominal point off the box centre is never below the sampled remainder about a~."""
    leb, wl, P, _ = mods
    w = wl.make_config(2, B=1, T=4)
    mu = wl.make_mu(w, 2.0)
    ctx = leb.context_for_workload(w)
    lo, hi = ctx.leb_analytic_fwd(_dev(w.nom), _dev(w.rad), mu=_dev(mu))
    glo, ghi = to_np(lo).reshape(-1, w.n), to_np(hi).reshape(-1, w.n)
    spec = P.spec_from_workload(w)
    rng = np.random.default_rng(12)
    N = w.N
    verts = np.array([[1.0 if (v >> j) & 1 else -1.0 for j in range(N)] for v in range(2 ** N)])
    for t in range(4):
        a0 = w.nom.reshape(-1, N)[t].astype(np.float64); sg = w.rad.reshape(-1, N)[t].astype(np.float64)
        m = mu.reshape(-1, N)[t].astype(np.float64)
        U = np.concatenate([rng.uniform(-1, 1, (100000, N)), verts])
        r = _true_r(P, spec, a0, a0[None, :] + m[None, :] + U * sg[None, :])
        assert np.all(r.max(0) <= ghi[t] + 1e-12) and np.all(r.min(0) >= glo[t] - 1e-12), t
    ctx.close()


def test_vjp_domain_error_gives_nan(mods):
    leb, wl, _, _ = mods
    w = wl.make_config(2, B=1, T=2)
    ctx = leb.context_for_workload(w)
    n2 = w.nom.copy(); n2[0, 1, 4] = np.pi / 2
    gn, gr = ctx.leb_vjp(0, _dev(n2), _dev(w.rad), _dev(w.g_lo), _dev(w.g_hi))
    assert ctx.leb_domain_flag() == 1
    assert bool(torch.isnan(gn[0, 1]).all()) and bool(torch.isfinite(gn[0, 0]).all())
    ctx.close()


# ---------------------------------------------------------------------------------- zonotope fold
def test_inflate_matches_oracle_and_contains(mods):
    leb, wl, _, I = mods
    ctx = leb.Context(0)
    rng = np.random.default_rng(5)
    for shape in ((3, 7, 10), (1, 1, 1), (2, 5, 168), (4, 3, 7)):
        lo = rng.standard_normal(shape).astype(np.float32) * 1e-2
        hi = lo + rng.uniform(0, 1e-2, shape).astype(np.float32)
        E = rng.uniform(0.5, 1.5, shape[-1]).astype(np.float32)
        c, R, Eb = ctx.leb_zonotope_inflate(_dev(lo), _dev(hi), 1e-6, _dev(E), True)
        oc, oR, oE = I.inflate(lo, hi, 1e-6, E, True)
        assert np.allclose(to_np(c), oc, rtol=1e-6, atol=1e-9)
        assert np.allclose(to_np(R), oR, rtol=1e-6, atol=1e-9)
        assert np.allclose(to_np(Eb), oE, rtol=1e-6, atol=1e-9)
        # containment in FP32 and right-invertibility (L229, L347): [lo, hi] inside [c - R, c + R], R > 0
        c64, R64 = to_np(c), to_np(R)
        assert np.all(c64 - R64 <= lo) and np.all(c64 + R64 >= hi) and np.all(R64 > 0)
    # degenerate interval lo == hi: R = pad; empty batch
    z = torch.zeros(1, 2, 4, device="cuda")
    c, R = ctx.leb_zonotope_inflate(z, z, 1e-6)
    assert float(c.abs().max()) == 0.0 and np.allclose(to_np(R), 1e-6, rtol=1e-6)
    c, R = ctx.leb_zonotope_inflate(z[:0], z[:0], 1e-6)
    assert c.shape == (0, 2, 4)
    # VJP of the fold
    gc = rng.standard_normal((2, 3, 5)).astype(np.float32); gR = rng.standard_normal((2, 3, 5)).astype(np.float32)
    g_lo, g_hi = ctx.leb_zonotope_inflate_vjp(_dev(gc), _dev(gR))
    o_lo, o_hi = I.inflate_vjp(gc, gR)
    assert np.allclose(to_np(g_lo), o_lo, rtol=1e-6, atol=1e-7) and np.allclose(to_np(g_hi), o_hi, rtol=1e-6, atol=1e-7)
    ctx.close()
