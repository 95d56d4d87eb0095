"""ORACLE (test infrastructure, NOT the product): ctypes loader for
oracle/pbh_oracle.cpp (FP64 path-based interval-Hessian bounds, Thm 1 eq. (15),
PAPER.md:L164-167) and thin array marshalling.  No arithmetic of the method lives
here.  Shares nothing with the CUDA path."""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pbh_oracle.cpp")
_LIB = os.path.join(_HERE, "libpbh_oracle.so")

MODE_PATH, MODE_EXPAND, MODE_CLASSIC = 0, 1, 2
MODEL_UNICYCLE, MODEL_QUAD12, MODEL_QUADCHAIN, MODEL_PLANAR_QUAD, MODEL_SATELLITE, MODEL_QUADCENTROID = 1, 2, 3, 4, 5, 6
MODEL_QUADRATIC, MODEL_LINEAR = 100, 101
INTEG_EULER, INTEG_RK4 = 1, 2


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.pbh_oracle_eval.restype = ctypes.c_int
        _lib.pbh_oracle_vjp.restype = ctypes.c_int
        _lib.pbh_oracle_max_threads.restype = ctypes.c_int
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


class ModelSpec:
    """model id + integrator + params [dt, mass, g, Jx, Jy, Jz, k1, k3]; for the
    generic test models, Q [n,N,N] (f_l = 1/2 a^T Q_l a + C_l a) and C [n,N]."""

    def __init__(self, model_id, integ=INTEG_EULER, n_units=1, params=None, Q=None, C=None):
        self.model_id, self.integ, self.n_units = int(model_id), int(integ), int(n_units)
        self.params = np.ascontiguousarray(params if params is not None else np.zeros(8), dtype=np.float64)
        self.Q = None if Q is None else np.ascontiguousarray(Q, dtype=np.float64)
        self.C = None if C is None else np.ascontiguousarray(C, dtype=np.float64)
        if model_id == MODEL_UNICYCLE:
            self.n, self.N = 3, 5
        elif model_id == MODEL_QUAD12:
            self.n, self.N = 12, 16
        elif model_id in (MODEL_QUADCHAIN, MODEL_QUADCENTROID):
            self.n, self.N = 12 * n_units, 16 * n_units
        elif model_id == MODEL_PLANAR_QUAD:
            self.n, self.N = 6, 8
        elif model_id == MODEL_SATELLITE:
            self.n, self.N = 7, 10
        else:
            self.n, self.N = self.C.shape

    def _head(self):
        return (ctypes.c_int(self.model_id), ctypes.c_int(self.integ), ctypes.c_int(self.n_units),
                _p(self.params), _p(self.Q), _p(self.C), ctypes.c_int(self.n), ctypes.c_int(self.N))


def pbh(spec: ModelSpec, nom, rad, mode=MODE_PATH, threads=0, mu=None):
    """nom, rad (, mu) [tiles, N] -> (r_lo, r_hi) [tiles, n] FP64, status.  mu: box offsets of (25a)."""
    nom = np.ascontiguousarray(nom, dtype=np.float64).reshape(-1, spec.N)
    rad = np.ascontiguousarray(rad, dtype=np.float64).reshape(-1, spec.N)
    if mu is not None:
        mu = np.ascontiguousarray(mu, dtype=np.float64).reshape(-1, spec.N)
    tiles = nom.shape[0]
    r_lo = np.empty((tiles, spec.n))
    r_hi = np.empty((tiles, spec.n))
    st = lib().pbh_oracle_eval(*spec._head(), ctypes.c_int(tiles), _p(nom), _p(rad), _p(mu), ctypes.c_int(mode),
                               _p(r_lo), _p(r_hi), ctypes.c_int(threads))
    return r_lo, r_hi, st


def pbh_vjp(spec: ModelSpec, nom, rad, g_lo, g_hi, dirs=None, threads=0, mu=None):
    """Gradient entries along `dirs` (indices in [0,3N): <N nominal, [N,2N) radius, >=2N mu);
    default all 2N (3N with mu).  Returns array [tiles, len(dirs)]."""
    nom = np.ascontiguousarray(nom, dtype=np.float64).reshape(-1, spec.N)
    rad = np.ascontiguousarray(rad, dtype=np.float64).reshape(-1, spec.N)
    if mu is not None:
        mu = np.ascontiguousarray(mu, dtype=np.float64).reshape(-1, spec.N)
    g_lo = np.ascontiguousarray(g_lo, dtype=np.float64).reshape(-1, spec.n)
    g_hi = np.ascontiguousarray(g_hi, dtype=np.float64).reshape(-1, spec.n)
    if dirs is None:
        dirs = np.arange((2 if mu is None else 3) * spec.N)
    dirs = np.ascontiguousarray(dirs, dtype=np.int32)
    out = np.empty((nom.shape[0], dirs.shape[0]))
    st = lib().pbh_oracle_vjp(*spec._head(), ctypes.c_int(nom.shape[0]), _p(nom), _p(rad), _p(mu), _p(g_lo), _p(g_hi),
                              ctypes.c_int(dirs.shape[0]), _p(dirs), _p(out), ctypes.c_int(threads))
    return out, st


def f(spec: ModelSpec, alpha):
    alpha = np.ascontiguousarray(alpha, dtype=np.float64).reshape(-1, spec.N)
    out = np.empty((alpha.shape[0], spec.n))
    lib().pbh_oracle_f(*spec._head(), ctypes.c_int(alpha.shape[0]), _p(alpha), _p(out))
    return out


def jac(spec: ModelSpec, alpha):
    alpha = np.ascontiguousarray(alpha, dtype=np.float64).reshape(spec.N)
    J = np.empty((spec.n, spec.N))
    lib().pbh_oracle_jac(*spec._head(), _p(alpha), _p(J))
    return J


def hessian_entry(spec: ModelSpec, box_lo, box_hi, j, k):
    box_lo = np.ascontiguousarray(box_lo, dtype=np.float64)
    box_hi = np.ascontiguousarray(box_hi, dtype=np.float64)
    H_lo, H_hi = np.empty(spec.n), np.empty(spec.n)
    lib().pbh_oracle_hessian_entry(*spec._head(), _p(box_lo), _p(box_hi), ctypes.c_int(j), ctypes.c_int(k),
                                   _p(H_lo), _p(H_hi))
    return H_lo, H_hi


def max_threads() -> int:
    return int(lib().pbh_oracle_max_threads())


def spec_from_workload(w) -> ModelSpec:
    """Build the spec from a workloads.AnalyticModel-like object (duck-typed: the
    oracle does not import the product package)."""
    am = w.analytic
    return ModelSpec(am.model_id, am.integ, am.n_units, am.params())
