"""Thin Python binding of the C ABI in include/leb.h (argument marshalling only).

Every numerical step runs in libleb.so's sm_100a kernels; torch is used for device memory and
streams.  There is no CPU fallback: if the library is missing or no CUDA device is present the
calls raise.  Function names mirror the C entry points.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libleb.so")

LEB_OK = 0
LEB_ERR_ARG = 1
LEB_ERR_UNSUPPORTED = 5
LEB_ERR_STATE = 8
LEB_ERR_CAPACITY = 9
JERR_STATIC_MAX = 65536
FLAG_NO_MARGIN = 1
FLAG_FFMA_ONLY = 2
FLAG_HOST_IO = 4
FLAG_REUSE_FWD = 8
FLAG_SINGLE_CTA = 16
FLAG_IBP_HIDDEN = 32

EXPORTS = [
    "leb_create", "leb_destroy", "leb_status_str", "leb_set_analytic", "leb_set_mlp", "leb_set_nn_chunk",
    "leb_analytic_fwd", "leb_analytic_partition_fwd", "leb_analytic_partition_vjp", "leb_analytic_pgd", "leb_nn_fwd", "leb_nn_alpha_fwd", "leb_vjp", "leb_vjp_mu", "leb_zonotope_inflate", "leb_zonotope_inflate_vjp", "leb_dist_add", "leb_tube_propagate", "leb_jerr", "leb_jerr_static",
    "leb_domain_flag", "leb_nn_hidden_bounds", "leb_nn_chain_coeffs", "leb_nn_jacobian", "leb_nn_slopes", "leb_nn_state", "leb_analytic_tape_stats", "leb_launch_count", "leb_profile", "leb_profile_read",
    "leb_profile_reset",
]


class LebError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: leb_status {status} ({_status_str(status)})")


class _AnalyticModel(ctypes.Structure):
    _fields_ = [("model_id", ctypes.c_int), ("integ", ctypes.c_int), ("n_units", ctypes.c_int),
                ("dt", ctypes.c_float), ("mass", ctypes.c_float), ("g", ctypes.c_float),
                ("Jx", ctypes.c_float), ("Jy", ctypes.c_float), ("Jz", ctypes.c_float),
                ("k1", ctypes.c_float), ("k3", ctypes.c_float)]


class _Mlp(ctypes.Structure):
    _fields_ = [("n_layers", ctypes.c_int), ("dims", ctypes.POINTER(ctypes.c_int)),
                ("W", ctypes.POINTER(ctypes.c_void_p)), ("b", ctypes.POINTER(ctypes.c_void_p)),
                ("act", ctypes.c_int), ("residual", ctypes.c_int), ("weights_on_host", ctypes.c_int)]


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen libleb.so (built in-tree by paper_2607_01203_b200.build); fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} not built: run `python -m paper_2607_01203_b200.build` (no CPU fallback exists)")
        lib = ctypes.CDLL(LIB_PATH)
        for name in EXPORTS:
            getattr(lib, name).restype = ctypes.c_int
        lib.leb_status_str.restype = ctypes.c_char_p
        lib.leb_launch_count.restype = ctypes.c_longlong
        lib.leb_launch_count.argtypes = [ctypes.c_void_p]
        _lib = lib
    return _lib


def _status_str(s: int) -> str:
    try:
        return load_library().leb_status_str(ctypes.c_int(s)).decode()
    except Exception:
        return "?"


def _chk(status: int, where: str):
    if status != LEB_OK:
        raise LebError(status, where)


def _ptr(t: Optional[torch.Tensor]):
    return ctypes.c_void_p(0 if t is None else t.data_ptr())


def _stream_ptr(device) -> ctypes.c_void_p:
    return ctypes.c_void_p(torch.cuda.current_stream(device).cuda_stream)


def _check_f32(*tensors):
    for t in tensors:
        if t is not None and (t.dtype != torch.float32 or not t.is_contiguous()):
            raise ValueError("tensors must be contiguous float32")


class Context:
    """Owns one leb_ctx on one CUDA device.  Inputs are CUDA tensors on that device, or (host_io=True
    calls) CPU tensors, ideally pinned."""

    def __init__(self, device: int = 0):
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the LEB library has no CPU fallback")
        self.lib = load_library()
        self.device = int(device)
        self._ctx = ctypes.c_void_p()
        _chk(self.lib.leb_create(ctypes.byref(self._ctx), ctypes.c_int(self.device)), "leb_create")
        self.n = self.N = None
        self.nn_n = self.nn_N = None

    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx:
            self.lib.leb_destroy(self._ctx)
            self._ctx = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ------------------------------------------------------------------ model set-up
    def leb_set_analytic(self, model_id: int, integ: int, dt: float, n_units: int = 1, mass=1.0, g=9.81,
                         Jx=0.010, Jy=0.015, Jz=0.020, k1=1.0, k3=0.1):
        m = _AnalyticModel(int(model_id), int(integ), int(n_units), dt, mass, g, Jx, Jy, Jz, k1, k3)
        _chk(self.lib.leb_set_analytic(self._ctx, ctypes.byref(m)), "leb_set_analytic")
        if model_id in (1, 4, 5):
            self.n, self.N = {1: (3, 5), 4: (6, 8), 5: (7, 10)}[model_id]
        else:
            u = n_units if model_id in (3, 6) else 1
            self.n, self.N = 12 * u, 16 * u

    def leb_set_mlp(self, dims: Sequence[int], W: Sequence[torch.Tensor], b: Sequence[torch.Tensor], act: int,
                    residual: bool = True):
        L = len(W)
        assert len(dims) == L + 1 and len(b) == L
        on_host = not W[0].is_cuda
        W = [w.contiguous().float() for w in W]
        b = [x.contiguous().float() for x in b]
        for l in range(L):
            assert tuple(W[l].shape) == (dims[l + 1], dims[l]) and tuple(b[l].shape) == (dims[l + 1],)
            assert W[l].is_cuda != on_host and b[l].is_cuda != on_host
        dims_a = (ctypes.c_int * (L + 1))(*[int(d) for d in dims])
        W_a = (ctypes.c_void_p * L)(*[w.data_ptr() for w in W])
        b_a = (ctypes.c_void_p * L)(*[x.data_ptr() for x in b])
        m = _Mlp(L, dims_a, W_a, b_a, int(act), int(bool(residual)), int(on_host))
        _chk(self.lib.leb_set_mlp(self._ctx, ctypes.byref(m), _stream_ptr(self.device)), "leb_set_mlp")
        self.nn_N, self.nn_n = int(dims[0]), int(dims[-1])

    def leb_set_nn_chunk(self, tiles: int):
        _chk(self.lib.leb_set_nn_chunk(self._ctx, ctypes.c_int(int(tiles))), "leb_set_nn_chunk")

    # ------------------------------------------------------------------ helpers
    def _out(self, like: torch.Tensor, shape, host_io: bool):
        if host_io:
            return torch.empty(shape, dtype=torch.float32, pin_memory=True)
        return torch.empty(shape, dtype=torch.float32, device=like.device)

    @staticmethod
    def _bt(nom: torch.Tensor):
        if nom.dim() != 3:
            raise ValueError("expected [B, T, ld] tensors")
        return int(nom.shape[0]), int(nom.shape[1]), int(nom.shape[2])

    # ------------------------------------------------------------------ entry points
    def leb_analytic_fwd(self, nom, rad, r_lo=None, r_hi=None, flags: int = 0, mu=None):
        _check_f32(nom, rad, r_lo, r_hi, mu)
        B, T, ld_in = self._bt(nom)
        host = bool(flags & FLAG_HOST_IO)
        if r_lo is None:
            r_lo = self._out(nom, (B, T, self.n), host)
            r_hi = self._out(nom, (B, T, self.n), host)
        _chk(self.lib.leb_analytic_fwd(self._ctx, B, T, _ptr(nom), _ptr(rad), _ptr(mu), ld_in, _ptr(r_lo), _ptr(r_hi),
                                       int(r_lo.shape[2]), ctypes.c_uint(flags), _stream_ptr(self.device)), "leb_analytic_fwd")
        return r_lo, r_hi

    def leb_analytic_partition_fwd(self, nom, rad, splits, mu=None, flags: int = 0):
        """Hull of the bounds of the grid of sub-boxes (splits[g] parts along coordinate g)."""
        _check_f32(nom, rad, mu)
        B, T, ld_in = self._bt(nom)
        host = bool(flags & FLAG_HOST_IO)
        r_lo = self._out(nom, (B, T, self.n), host)
        r_hi = self._out(nom, (B, T, self.n), host)
        sp = (ctypes.c_int * self.N)(*[int(x) for x in splits])
        _chk(self.lib.leb_analytic_partition_fwd(self._ctx, B, T, _ptr(nom), _ptr(rad), _ptr(mu), ld_in, sp, _ptr(r_lo), _ptr(r_hi),
                                                 self.n, ctypes.c_uint(flags), _stream_ptr(self.device)), "leb_analytic_partition_fwd")
        return r_lo, r_hi

    def leb_analytic_partition_vjp(self, nom, rad, splits, g_lo, g_hi, mu=None, flags: int = 0):
        """VJP of leb_analytic_partition_fwd; returns (grad_nom, grad_rad, grad_mu or None)."""
        _check_f32(nom, rad, mu, g_lo, g_hi)
        B, T, ld_in = self._bt(nom)
        host = bool(flags & FLAG_HOST_IO)
        grad_nom = self._out(nom, (B, T, ld_in), host)
        grad_rad = self._out(nom, (B, T, ld_in), host)
        grad_mu = self._out(nom, (B, T, ld_in), host) if mu is not None else None
        sp = (ctypes.c_int * self.N)(*[int(x) for x in splits])
        _chk(self.lib.leb_analytic_partition_vjp(self._ctx, B, T, _ptr(nom), _ptr(rad), _ptr(mu), ld_in, sp, _ptr(g_lo), _ptr(g_hi),
                                                 int(g_lo.shape[2]), _ptr(grad_nom), _ptr(grad_rad), _ptr(grad_mu),
                                                 ctypes.c_uint(flags), _stream_ptr(self.device)), "leb_analytic_partition_vjp")
        return grad_nom, grad_rad, grad_mu

    def leb_analytic_pgd(self, centre, rad, eps, nom0, steps: int, lr: float, flags: int = 0):
        """PGD refinement of the nominal point; returns (best nominal points, initial widths, best widths)."""
        _check_f32(centre, rad, eps, nom0)
        B, T, ld_in = self._bt(centre)
        host = bool(flags & FLAG_HOST_IO)
        nom = nom0.clone()
        if host:
            nom = nom.pin_memory()
        w0 = self._out(centre, (B, T), host)
        w = self._out(centre, (B, T), host)
        _chk(self.lib.leb_analytic_pgd(self._ctx, B, T, _ptr(centre), _ptr(rad), _ptr(eps), ld_in, int(steps), ctypes.c_float(lr),
                                       _ptr(nom), _ptr(w0), _ptr(w), ctypes.c_uint(flags), _stream_ptr(self.device)), "leb_analytic_pgd")
        return nom, w0, w

    def leb_nn_fwd(self, nom, rad, J=None, r_lo=None, r_hi=None, margin=None, flags: int = 0, mu=None):
        """flags = 0 is the C ABI's default: CERTIFIED mode (rounding errors bounded and added outward).
        FLAG_NO_MARGIN selects value mode, the plain FP32 result the parity tests compare with the oracle."""
        _check_f32(nom, rad, J, r_lo, r_hi, margin, mu)
        B, T, ld_in = self._bt(nom)
        host = bool(flags & FLAG_HOST_IO)
        if r_lo is None:
            r_lo = self._out(nom, (B, T, self.nn_n), host)
            r_hi = self._out(nom, (B, T, self.nn_n), host)
        _chk(self.lib.leb_nn_fwd(self._ctx, B, T, _ptr(nom), _ptr(rad), _ptr(mu), _ptr(J), ld_in, _ptr(r_lo), _ptr(r_hi),
                                 _ptr(margin), int(r_lo.shape[2]), ctypes.c_uint(flags), _stream_ptr(self.device)), "leb_nn_fwd")
        return r_lo, r_hi

    def leb_nn_alpha_fwd(self, nom, rad, steps: int, lr: float, flags: int = 0):
        """CROWN with optimisable lower ReLU slopes; returns (r_lo, r_hi, width0, width)."""
        _check_f32(nom, rad)
        B, T, ld_in = self._bt(nom)
        host = bool(flags & FLAG_HOST_IO)
        r_lo = self._out(nom, (B, T, self.nn_n), host)
        r_hi = self._out(nom, (B, T, self.nn_n), host)
        w0 = self._out(nom, (B, T), host)
        w = self._out(nom, (B, T), host)
        _chk(self.lib.leb_nn_alpha_fwd(self._ctx, B, T, _ptr(nom), _ptr(rad), ld_in, int(steps), ctypes.c_float(lr), _ptr(r_lo),
                                       _ptr(r_hi), self.nn_n, _ptr(w0), _ptr(w), ctypes.c_uint(flags), _stream_ptr(self.device)),
             "leb_nn_alpha_fwd")
        return r_lo, r_hi, w0, w

    def leb_vjp(self, kind: int, nom, rad, g_lo, g_hi, grad_nom=None, grad_rad=None, flags: int = 0):
        _check_f32(nom, rad, g_lo, g_hi, grad_nom, grad_rad)
        B, T, ld_in = self._bt(nom)
        host = bool(flags & FLAG_HOST_IO)
        if grad_nom is None:
            grad_nom = self._out(nom, (B, T, ld_in), host)
            grad_rad = self._out(nom, (B, T, ld_in), host)
        _chk(self.lib.leb_vjp(self._ctx, int(kind), B, T, _ptr(nom), _ptr(rad), _ptr(g_lo), _ptr(g_hi), ld_in,
                              int(g_lo.shape[2]), _ptr(grad_nom), _ptr(grad_rad), ctypes.c_uint(flags),
                              _stream_ptr(self.device)), "leb_vjp")
        return grad_nom, grad_rad

    def leb_vjp_mu(self, kind: int, nom, rad, mu, g_lo, g_hi, grad_nom=None, grad_rad=None, grad_mu=None, flags: int = 0):
        _check_f32(nom, rad, mu, g_lo, g_hi, grad_nom, grad_rad, grad_mu)
        B, T, ld_in = self._bt(nom)
        host = bool(flags & FLAG_HOST_IO)
        if grad_nom is None:
            grad_nom = self._out(nom, (B, T, ld_in), host)
            grad_rad = self._out(nom, (B, T, ld_in), host)
        if grad_mu is None and mu is not None:
            grad_mu = self._out(nom, (B, T, ld_in), host)
        _chk(self.lib.leb_vjp_mu(self._ctx, int(kind), B, T, _ptr(nom), _ptr(rad), _ptr(mu), _ptr(g_lo), _ptr(g_hi), ld_in,
                                 int(g_lo.shape[2]), _ptr(grad_nom), _ptr(grad_rad), _ptr(grad_mu), ctypes.c_uint(flags),
                                 _stream_ptr(self.device)), "leb_vjp_mu")
        return grad_nom, grad_rad, grad_mu

    def leb_zonotope_inflate(self, r_lo, r_hi, pad: float = 1e-6, E_diag=None, dense: bool = False, flags: int = 0,
                             c_bar=None, R_diag=None):
        _check_f32(r_lo, r_hi, E_diag, c_bar, R_diag)
        B, T, n = self._bt(r_lo)
        host = bool(flags & FLAG_HOST_IO)
        if c_bar is None:
            c_bar = self._out(r_lo, (B, T, n), host)
            R_diag = self._out(r_lo, (B, T, n), host)
        Ebar = self._out(r_lo, (B, T, n, 2 * n), host) if dense else None
        _chk(self.lib.leb_zonotope_inflate(self._ctx, B, T, n, _ptr(r_lo), _ptr(r_hi), _ptr(E_diag), ctypes.c_float(pad),
                                           _ptr(c_bar), _ptr(R_diag), _ptr(Ebar), ctypes.c_uint(flags),
                                           _stream_ptr(self.device)), "leb_zonotope_inflate")
        return (c_bar, R_diag, Ebar) if dense else (c_bar, R_diag)

    def leb_zonotope_inflate_vjp(self, gc, gR, flags: int = 0, g_lo=None, g_hi=None):
        _check_f32(gc, gR, g_lo, g_hi)
        B, T, n = self._bt(gc)
        host = bool(flags & FLAG_HOST_IO)
        if g_lo is None:
            g_lo = self._out(gc, (B, T, n), host)
            g_hi = self._out(gc, (B, T, n), host)
        _chk(self.lib.leb_zonotope_inflate_vjp(self._ctx, B, T, n, _ptr(gc), _ptr(gR), _ptr(g_lo), _ptr(g_hi),
                                               ctypes.c_uint(flags), _stream_ptr(self.device)), "leb_zonotope_inflate_vjp")
        return g_lo, g_hi

    def leb_dist_add(self, E_lo, E_hi, E_nom, r_lo, r_hi, flags: int = 0):
        """(22): adds the disturbance-error enclosure to (r_lo, r_hi) in place.  E_*: [B, T, n, nw]."""
        _check_f32(E_lo, E_hi, E_nom, r_lo, r_hi)
        B, T, n, nw = (int(x) for x in E_lo.shape)
        _chk(self.lib.leb_dist_add(self._ctx, B, T, n, nw, _ptr(E_lo), _ptr(E_hi), _ptr(E_nom), _ptr(r_lo), _ptr(r_hi),
                                   ctypes.c_uint(flags), _stream_ptr(self.device)), "leb_dist_add")
        return r_lo, r_hi

    def leb_tube_propagate(self, Phi, c_bar, R_diag, m: int, E_diag=None, flags: int = 0):
        """(27)-(28): Phi [B, T(T+1)/2, n+m, n] packed; returns h_mu, h_sigma [B, T, n+m] (row k-1 = time k)."""
        _check_f32(Phi, c_bar, R_diag, E_diag)
        B, T, n = self._bt(c_bar)
        host = bool(flags & FLAG_HOST_IO)
        h_mu = self._out(c_bar, (B, T, n + m), host)
        h_sigma = self._out(c_bar, (B, T, n + m), host)
        _chk(self.lib.leb_tube_propagate(self._ctx, B, T, n, int(m), _ptr(Phi), _ptr(c_bar), _ptr(R_diag), _ptr(E_diag),
                                         _ptr(h_mu), _ptr(h_sigma), ctypes.c_uint(flags), _stream_ptr(self.device)),
             "leb_tube_propagate")
        return h_mu, h_sigma

    def leb_jerr(self, Phi, R_diag, m: int, E_diag=None, with_grad: bool = True, flags: int = 0):
        """(35): returns J_err [B] and d J_err / d R_diag [B, T, n] (or None)."""
        _check_f32(Phi, R_diag, E_diag)
        B, T, n = self._bt(R_diag)
        host = bool(flags & FLAG_HOST_IO)
        J = self._out(R_diag, (B,), host)
        g = self._out(R_diag, (B, T, n), host) if with_grad else None
        _chk(self.lib.leb_jerr(self._ctx, B, T, n, int(m), _ptr(Phi), _ptr(R_diag), _ptr(E_diag), _ptr(J), _ptr(g),
                               ctypes.c_uint(flags), _stream_ptr(self.device)), "leb_jerr")
        return J, g

    def leb_jerr_static(self, Phi, R_diag, m: int, J, grad_R=None, E_diag=None, flags: int = 0):
        """leb_jerr without any allocation (leb.h): the caller passes the outputs J [B] and grad_R [B, T, n] (or None) as
        device tensors; B * T <= JERR_STATIC_MAX; calls that overlap on the GPU race on the library's static scratch."""
        _check_f32(Phi, R_diag, E_diag, J, grad_R)
        B, T, n = self._bt(R_diag)
        _chk(self.lib.leb_jerr_static(self._ctx, B, T, n, int(m), _ptr(Phi), _ptr(R_diag), _ptr(E_diag), _ptr(J), _ptr(grad_R),
                                      ctypes.c_uint(flags), _stream_ptr(self.device)), "leb_jerr_static")
        return J, grad_R

    def leb_domain_flag(self) -> int:
        flag = ctypes.c_int(0)
        _chk(self.lib.leb_domain_flag(self._ctx, ctypes.byref(flag), _stream_ptr(self.device)), "leb_domain_flag")
        return int(flag.value)

    def leb_nn_hidden_bounds(self, layer: int, tiles: int, width: int):
        dev = torch.device("cuda", self.device)
        l = torch.empty((tiles, width), dtype=torch.float32, device=dev)
        u = torch.empty((tiles, width), dtype=torch.float32, device=dev)
        _chk(self.lib.leb_nn_hidden_bounds(self._ctx, int(layer), _ptr(l), _ptr(u), _stream_ptr(self.device)),
             "leb_nn_hidden_bounds")
        return l, u

    def leb_nn_chain_coeffs(self, target: int, tiles: int, rows: int, N: int):
        out = torch.empty((tiles, 2, rows, N), dtype=torch.float32, device=torch.device("cuda", self.device))
        _chk(self.lib.leb_nn_chain_coeffs(self._ctx, int(target), _ptr(out), _stream_ptr(self.device)), "leb_nn_chain_coeffs")
        return out

    def leb_nn_slopes(self, layer: int, tiles: int, width: int):
        """(k_U, k_L) of hidden layer `layer` in the resident forward state: [tiles, width] each"""
        dev = torch.device("cuda", self.device)
        kU = torch.empty((tiles, width), dtype=torch.float32, device=dev)
        kL = torch.empty((tiles, width), dtype=torch.float32, device=dev)
        _chk(self.lib.leb_nn_slopes(self._ctx, int(layer), _ptr(kU), _ptr(kL), _stream_ptr(self.device)), "leb_nn_slopes")
        return kU, kL

    def leb_nn_jacobian(self, tiles: int, n: int, N: int):
        """J~ of the last leb_nn_fwd(J=None): [tiles, n, N]"""
        out = torch.empty((tiles, n, N), dtype=torch.float32, device=torch.device("cuda", self.device))
        _chk(self.lib.leb_nn_jacobian(self._ctx, _ptr(out), _stream_ptr(self.device)), "leb_nn_jacobian")
        return out

    def leb_nn_state(self):
        """(resident tiles, certified?, last leb_vjp reused the resident forward state?)"""
        t, c, r = ctypes.c_int(0), ctypes.c_int(0), ctypes.c_int(0)
        _chk(self.lib.leb_nn_state(self._ctx, ctypes.byref(t), ctypes.byref(c), ctypes.byref(r)), "leb_nn_state")
        return int(t.value), bool(c.value), bool(r.value)

    def leb_analytic_tape_stats(self) -> dict:
        f, i, t, k, m = ctypes.c_double(0), ctypes.c_longlong(0), ctypes.c_longlong(0), ctypes.c_int(0), ctypes.c_int(0)
        _chk(self.lib.leb_analytic_tape_stats(self._ctx, ctypes.byref(f), ctypes.byref(i), ctypes.byref(t), ctypes.byref(k),
                                              ctypes.byref(m)), "leb_analytic_tape_stats")
        return {"flops_per_tile": float(f.value), "ins_per_tile": int(i.value), "tape_ins": int(t.value),
                "tasks": int(k.value), "max_slots": int(m.value)}

    def leb_launch_count(self) -> int:
        return int(self.lib.leb_launch_count(self._ctx))

    def leb_profile(self, enable: bool):
        _chk(self.lib.leb_profile(self._ctx, ctypes.c_int(int(bool(enable)))), "leb_profile")

    def leb_profile_read(self, kernel_class: int):
        """(ms, algorithmic work, launches) of one kernel class since the last leb_profile_reset."""
        ms, work, n = ctypes.c_double(0), ctypes.c_double(0), ctypes.c_longlong(0)
        _chk(self.lib.leb_profile_read(self._ctx, ctypes.c_int(int(kernel_class)), ctypes.byref(ms), ctypes.byref(work),
                                       ctypes.byref(n), _stream_ptr(self.device)), "leb_profile_read")
        return float(ms.value), float(work.value), int(n.value)

    def leb_profile_reset(self):
        _chk(self.lib.leb_profile_reset(self._ctx), "leb_profile_reset")


def context_for_workload(w, device: int = 0) -> Context:
    """Context with the model of a workloads.Workload installed."""
    ctx = Context(device)
    if w.kind == "analytic":
        a = w.analytic
        ctx.leb_set_analytic(a.model_id, a.integ, a.dt, a.n_units, a.mass, a.g, a.Jx, a.Jy, a.Jz, a.k1, a.k3)
    else:
        dev = torch.device("cuda", device)
        ctx.leb_set_mlp(w.mlp.dims, [torch.from_numpy(x).to(dev) for x in w.mlp.W],
                        [torch.from_numpy(x).to(dev) for x in w.mlp.b], w.mlp.act, w.mlp.residual)
    return ctx
