"""Seeded synthetic workloads for the five BASELINE.json configs.

This module holds ONLY input generation (random draws, shapes, model constants).
It contains none of the method's arithmetic and imports neither `oracle/` nor the
CUDA binding; both the tests' oracle side and the CUDA side are fed from here.

Recipe: numpy `Generator(PCG64(seed))`
with seed = 20260701 + config id; draws are i.i.d. per (trajectory b, timestep t)
because the LEB path treats every (b, t) tile independently ("for
all k in [N]").  Draw order inside one config is fixed and documented below so a
workload is reproducible from its id alone.

The paper's own workloads (trained T-pusher MLP, its scenario files) are not
available; these synthetic inputs stand in for them, with the paper's shapes
(n up to 168 states PAPER.md:L420, horizons 25-100 PAPER.md:L416-420).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

BASE_SEED = 20260701

# analytic model ids / integrators / activations: plain integers shared by name
# with include/leb.h (values repeated there; no code is shared).
MODEL_UNICYCLE = 1
MODEL_QUAD12 = 2
MODEL_QUADCHAIN = 3
MODEL_PLANAR_QUAD = 4
MODEL_SATELLITE = 5
MODEL_QUADCENTROID = 6
INTEG_EULER = 1
INTEG_RK4 = 2
ACT_RELU = 1
ACT_TANH = 2

# 3-D quadrotor constants (paper gives none for the 3-D quad, PAPER.md:L538;
# DESIGN.md reading R7): distinct inertias so no gyroscopic coefficient vanishes.
QUAD_MASS = 1.0
QUAD_G = 9.81
QUAD_J = (0.010, 0.015, 0.020)
CHAIN_K1 = 1.0
CHAIN_K3 = 0.1


@dataclass
class AnalyticModel:
    model_id: int
    integ: int
    dt: float
    n_units: int = 1
    mass: float = QUAD_MASS
    g: float = QUAD_G
    Jx: float = QUAD_J[0]
    Jy: float = QUAD_J[1]
    Jz: float = QUAD_J[2]
    k1: float = CHAIN_K1
    k3: float = CHAIN_K3

    @property
    def n(self) -> int:
        return {MODEL_UNICYCLE: 3, MODEL_QUAD12: 12, MODEL_QUADCHAIN: 12 * self.n_units, MODEL_PLANAR_QUAD: 6,
                MODEL_SATELLITE: 7, MODEL_QUADCENTROID: 12 * self.n_units}[self.model_id]

    @property
    def m(self) -> int:
        return {MODEL_UNICYCLE: 2, MODEL_QUAD12: 4, MODEL_QUADCHAIN: 4 * self.n_units, MODEL_PLANAR_QUAD: 2,
                MODEL_SATELLITE: 3, MODEL_QUADCENTROID: 4 * self.n_units}[self.model_id]

    def params(self) -> np.ndarray:
        """Flat fp64 parameter vector [dt, mass, g, Jx, Jy, Jz, k1, k3]."""
        return np.array([self.dt, self.mass, self.g, self.Jx, self.Jy, self.Jz, self.k1, self.k3], dtype=np.float64)


@dataclass
class MLP:
    dims: List[int]                 # dims[0] = n+m ... dims[-1] = n
    W: List[np.ndarray]             # W[l] shape [dims[l+1], dims[l]], fp32
    b: List[np.ndarray]             # b[l] shape [dims[l+1]], fp32
    act: int
    residual: bool = True
    n_state: int = 0


@dataclass
class Workload:
    config_id: int
    name: str
    kind: str                       # "analytic" | "nn"
    B: int
    T: int
    n: int
    m: int
    nom: np.ndarray                 # [B, T, n+m] fp32, order [x; u]
    rad: np.ndarray                 # [B, T, n+m] fp32, >= 0
    g_lo: np.ndarray                # [B, T, n] fp32 VJP cotangents
    g_hi: np.ndarray                # [B, T, n] fp32
    analytic: Optional[AnalyticModel] = None
    mlp: Optional[MLP] = None
    meta: dict = field(default_factory=dict)

    @property
    def N(self) -> int:
        return self.n + self.m

    @property
    def entries(self) -> int:
        return self.B * self.T * self.n


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float32)


def _cotangents(rng, B, T, n):
    return _f32(rng.standard_normal((B, T, n))), _f32(rng.standard_normal((B, T, n)))


def _quad_unit_nominal(rng, shape):
    """One quad12 unit: xi=(p[3], angles[3], v[3], rates[3]), nu=(T, tau[3]).

    State order is the paper's.  Draw order: pos, angles, vel,
    rates, thrust, torques.
    """
    pos = rng.uniform(-1.0, 1.0, shape + (3,))
    ang = rng.uniform(-0.3, 0.3, shape + (3,))
    vel = rng.uniform(-1.0, 1.0, shape + (3,))
    rat = rng.uniform(-1.0, 1.0, shape + (3,))
    thr = QUAD_MASS * QUAD_G * rng.uniform(0.9, 1.1, shape + (1,))
    tau = rng.uniform(-0.1, 0.1, shape + (3,))
    xi = np.concatenate([pos, ang, vel, rat], axis=-1)
    nu = np.concatenate([thr, tau], axis=-1)
    return xi, nu


def make_mlp(rng, dims, act, init) -> MLP:
    """Draw order: for each layer l: W_l then b_l."""
    W, b = [], []
    for l in range(len(dims) - 1):
        fan_in, fan_out = dims[l], dims[l + 1]
        if init == "kaiming_half":      # config 3: Kaiming-normal x 0.5
            std = 0.5 * np.sqrt(2.0 / fan_in)
        elif init == "xavier":          # config 5: Xavier-normal
            std = np.sqrt(2.0 / (fan_in + fan_out))
        else:
            raise ValueError(init)
        W.append(_f32(rng.standard_normal((fan_out, fan_in)) * std))
        b.append(_f32(rng.uniform(-0.1, 0.1, fan_out)))
    return MLP(dims=list(dims), W=W, b=b, act=act, residual=True, n_state=dims[-1])


def make_config(config_id: int, B: Optional[int] = None, T: Optional[int] = None) -> Workload:
    """Build workload `config_id` in 1..5.  B/T override the batch/horizon (tests
    use smaller slices; the draw order guarantees that a smaller B is NOT a prefix
    of the full one, so always state B,T with a number)."""
    rng = np.random.Generator(np.random.PCG64(BASE_SEED + config_id))
    if config_id == 1:
        B, T = B or 1, T or 20
        x = rng.uniform(-1.0, 1.0, (B, T, 3))
        u = rng.uniform(-0.5, 0.5, (B, T, 2))
        rad = rng.uniform(0.01, 0.1, (B, T, 5))
        g_lo, g_hi = _cotangents(rng, B, T, 3)
        am = AnalyticModel(MODEL_UNICYCLE, INTEG_EULER, 0.1)
        return Workload(1, "unicycle_euler", "analytic", B, T, 3, 2,
                        _f32(np.concatenate([x, u], -1)), _f32(rad), g_lo, g_hi, analytic=am)
    if config_id == 2:
        B, T = B or 16, T or 50
        xi, nu = _quad_unit_nominal(rng, (B, T))
        rad = rng.uniform(0.005, 0.05, (B, T, 16))
        g_lo, g_hi = _cotangents(rng, B, T, 12)
        am = AnalyticModel(MODEL_QUAD12, INTEG_RK4, 0.05)
        return Workload(2, "quad12_rk4", "analytic", B, T, 12, 4,
                        _f32(np.concatenate([xi, nu], -1)), _f32(rad), g_lo, g_hi, analytic=am)
    if config_id == 3:
        B, T = B or 32, T or 40
        mlp = make_mlp(rng, [24, 128, 128, 128, 20], ACT_RELU, "kaiming_half")
        nom = rng.standard_normal((B, T, 24))
        rad = rng.uniform(0.01, 0.05, (B, T, 24))
        g_lo, g_hi = _cotangents(rng, B, T, 20)
        return Workload(3, "mlp20_relu", "nn", B, T, 20, 4, _f32(nom), _f32(rad), g_lo, g_hi, mlp=mlp)
    if config_id == 4:
        B, T = B or 8, T or 50
        U = 14
        xi, nu = _quad_unit_nominal(rng, (B, T, U))         # [B,T,U,12], [B,T,U,4]
        nom = np.concatenate([xi.reshape(B, T, 12 * U), nu.reshape(B, T, 4 * U)], -1)
        rad = rng.uniform(0.005, 0.05, (B, T, 16 * U))
        g_lo, g_hi = _cotangents(rng, B, T, 12 * U)
        am = AnalyticModel(MODEL_QUADCHAIN, INTEG_RK4, 0.05, n_units=U)
        return Workload(4, "quadchain168_rk4", "analytic", B, T, 12 * U, 4 * U,
                        _f32(nom), _f32(rad), g_lo, g_hi, analytic=am)
    if config_id == 5:
        B, T = B or 64, T or 100
        mlp = make_mlp(rng, [224, 512, 512, 512, 512, 168], ACT_TANH, "xavier")
        nom = rng.standard_normal((B, T, 224))
        rad = rng.uniform(0.005, 0.03, (B, T, 224))
        g_lo, g_hi = _cotangents(rng, B, T, 168)
        return Workload(5, "mlp168_tanh", "nn", B, T, 168, 56, _f32(nom), _f32(rad), g_lo, g_hi, mlp=mlp)
    raise ValueError(f"config_id must be 1..5, got {config_id}")


def make_small_chain(n_units: int, B: int, T: int, seed: int = 7) -> Workload:
    """A short quad chain (same draws as config 4) for exhaustive oracle checks."""
    rng = np.random.Generator(np.random.PCG64(BASE_SEED + 100 + seed))
    U = n_units
    xi, nu = _quad_unit_nominal(rng, (B, T, U))
    nom = np.concatenate([xi.reshape(B, T, 12 * U), nu.reshape(B, T, 4 * U)], -1)
    rad = rng.uniform(0.005, 0.05, (B, T, 16 * U))
    g_lo, g_hi = _cotangents(rng, B, T, 12 * U)
    am = AnalyticModel(MODEL_QUADCHAIN, INTEG_RK4, 0.05, n_units=U)
    return Workload(40 + U, f"quadchain{12*U}_rk4", "analytic", B, T, 12 * U, 4 * U,
                    _f32(nom), _f32(rad), g_lo, g_hi, analytic=am)


def make_paper_system(name: str, B: int, T: int, seed: int = 3) -> Workload:
    """The paper's own analytic systems (App. I), forward Euler as in the paper, synthetic nominal
    points: "satellite" (36) L507-519, 7 states (unit quaternion, body rates U[-1,1]) + 3 torques, I_S = diag(5,2,1),
    dt 0.1; "planar_quad" (37) L521-528, 6 states + 2 rotor thrusts around hover, m = 2.0576, L = 0.25, J = 0.01,
    dt 0.05; "quad12_euler": the 3-D quadrotor (38) with Euler.  Radii U[0.01, 0.2] (the local-set sizes of L372)."""
    rng = np.random.Generator(np.random.PCG64(BASE_SEED + 300 + seed))
    if name == "satellite":
        q = rng.standard_normal((B, T, 4))
        q /= np.linalg.norm(q, axis=-1, keepdims=True)
        nom = np.concatenate([q, rng.uniform(-1, 1, (B, T, 3)), rng.uniform(-1, 1, (B, T, 3))], -1)
        am = AnalyticModel(MODEL_SATELLITE, INTEG_EULER, 0.1, mass=1.0, g=0.0, Jx=5.0, Jy=2.0, Jz=1.0, k1=0.0, k3=0.0)
    elif name == "planar_quad":
        hover = 0.5 * 2.0576 * 9.81
        nom = np.concatenate([rng.uniform(-1, 1, (B, T, 2)), rng.uniform(-0.5, 0.5, (B, T, 1)), rng.uniform(-1, 1, (B, T, 3)),
                              hover * rng.uniform(0.8, 1.2, (B, T, 2))], -1)
        am = AnalyticModel(MODEL_PLANAR_QUAD, INTEG_EULER, 0.05, mass=2.0576, g=9.81, Jx=0.01, Jy=1.0, Jz=1.0, k1=0.25, k3=0.0)
    elif name.startswith("quadcentroid"):          # "quadcentroid8": 8 coupled quadrotors (39)-(42) L540-558, alpha 0.75, gamma 0.25
        U = int(name[len("quadcentroid"):])
        xi, nu = _quad_unit_nominal(rng, (B, T, U))
        nom = np.concatenate([xi.reshape(B, T, 12 * U), nu.reshape(B, T, 4 * U)], -1)
        am = AnalyticModel(MODEL_QUADCENTROID, INTEG_EULER, 0.05, n_units=U, k1=0.75, k3=0.25)
    elif name == "quad12_euler":
        xi, nu = _quad_unit_nominal(rng, (B, T))
        nom = np.concatenate([xi, nu], -1)
        am = AnalyticModel(MODEL_QUAD12, INTEG_EULER, 0.05)
    else:
        raise ValueError(name)
    rad = rng.uniform(0.01, 0.2, nom.shape)
    g_lo, g_hi = _cotangents(rng, B, T, am.n)
    return Workload(60, name, "analytic", B, T, am.n, am.m, _f32(nom), _f32(rad), g_lo, g_hi, analytic=am)


def make_mu(w: Workload, scale: float = 1.5, seed: int = 5) -> np.ndarray:
    """Box offsets mu (25a) PAPER.md:L272 for a workload: mu = rad * U[-scale, scale] (for scale > 1 the nominal
    point lies outside the box for some coordinates)."""
    rng = np.random.Generator(np.random.PCG64(BASE_SEED + 400 + seed))
    return _f32(w.rad * rng.uniform(-scale, scale, w.rad.shape))


def make_small_mlp(dims, act, B, T, seed=11, rad_lo=0.01, rad_hi=0.05, init="xavier") -> Workload:
    """A small MLP workload (tests: tiny shapes, ragged widths)."""
    rng = np.random.Generator(np.random.PCG64(BASE_SEED + 200 + seed))
    mlp = make_mlp(rng, dims, act, init)
    N, n = dims[0], dims[-1]
    nom = rng.standard_normal((B, T, N))
    rad = rng.uniform(rad_lo, rad_hi, (B, T, N))
    g_lo, g_hi = _cotangents(rng, B, T, n)
    return Workload(50, f"mlp_{'x'.join(map(str, dims))}", "nn", B, T, n, N - n,
                    _f32(nom), _f32(rad), g_lo, g_hi, mlp=mlp)
