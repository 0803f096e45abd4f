"""ctypes binding of the CPU oracle ``liblbmref.so`` (TEST INFRASTRUCTURE, not the product).

Argument marshalling only; all arithmetic is in ``lbmref.c``.  See ``lbmref.h`` for the calls.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liblbmref.so")
_SRC = [os.path.join(_HERE, "lbmref.c"), os.path.join(_HERE, "lbmref.h")]


def build_oracle(force: bool = False) -> str:
    """Compile ``lbmref.c`` with gcc (no contraction of a*b+c into fma: -ffp-contract=off)."""
    stale = force or not os.path.exists(_SO) or any(
        os.path.getmtime(s) > os.path.getmtime(_SO) for s in _SRC)
    if stale:
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-std=c99", "-D_GNU_SOURCE",
               "-o", _SO, _SRC[0], "-lm"]
        subprocess.check_call(cmd)
    return _SO


class _Params(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32),
                ("rho_l", C.c_double), ("rho_g", C.c_double),
                ("nu_l", C.c_double), ("nu_g", C.c_double),
                ("sigma", C.c_double), ("W", C.c_double),
                ("theta_deg", C.c_double), ("mobility", C.c_double),
                ("gx", C.c_double), ("gy", C.c_double),
                ("wall_rows", C.c_int32), ("ghost_rule", C.c_int32), ("picard", C.c_int32)]


class _Disk(C.Structure):
    _fields_ = [("cx", C.c_double), ("cy", C.c_double), ("r", C.c_double)]


class NodeFields(C.Structure):
    _fields_ = [(k, C.c_double) for k in
                ("phi", "gradx", "grady", "lap", "rho", "tau", "Fsx", "Fsy", "Fx", "Fy", "ux", "uy", "p")]


@dataclass
class RefParams:
    nx: int
    ny: int
    rho_l: float = 1000.0
    rho_g: float = 1.0
    nu_l: float = 0.01
    nu_g: float = 0.1
    sigma: float = 1e-2
    W: float = 4.0
    theta_deg: float = 90.0
    mobility: float = 0.02
    gx: float = 0.0
    gy: float = 0.0
    wall_rows: int = 0
    ghost_rule: int = 0
    picard: int = 1

    def c_struct(self) -> _Params:
        return _Params(self.nx, self.ny, self.rho_l, self.rho_g, self.nu_l, self.nu_g, self.sigma,
                       self.W, self.theta_deg, self.mobility, self.gx, self.gy, self.wall_rows,
                       self.ghost_rule, self.picard)


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        L = C.CDLL(build_oracle())
        dp = C.POINTER(C.c_double)
        ip = C.POINTER(C.c_int32)
        L.lbmref_create.argtypes = [C.POINTER(C.c_void_p), C.POINTER(_Params), C.c_void_p,
                                    C.POINTER(_Disk), C.c_int32]
        L.lbmref_init.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.lbmref_step.argtypes = [C.c_void_p, C.c_int64]
        L.lbmref_get.argtypes = [C.c_void_p] + [C.c_void_p] * 5
        L.lbmref_get_populations.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.lbmref_set_populations.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.lbmref_get_classification.argtypes = [C.c_void_p] + [C.c_void_p] * 8
        L.lbmref_get_phi_raw.argtypes = [C.c_void_p, C.c_void_p]
        L.lbmref_diag.argtypes = [C.c_void_p, dp]
        L.lbmref_destroy.argtypes = [C.c_void_p]
        L.lbmref_last_error.argtypes = [C.c_void_p]
        L.lbmref_last_error.restype = C.c_char_p
        L.lbmref_lattice.argtypes = [ip, ip, ip, dp]
        L.lbmref_matrices.argtypes = [dp, dp]
        L.lbmref_alpha_from_mobility.argtypes = [C.c_double]
        L.lbmref_alpha_from_mobility.restype = C.c_double
        L.lbmref_chi.argtypes = [C.c_double, dp]
        L.lbmref_ghost_rule.argtypes = [C.c_double, C.c_double, C.c_int32]
        L.lbmref_ghost_rule.restype = C.c_double
        L.lbmref_neq.argtypes = [C.c_double, C.c_double, C.c_double, C.c_double, dp]
        L.lbmref_pressure.argtypes = [C.c_double, dp, C.c_double, C.c_double]
        L.lbmref_pressure.restype = C.c_double
        L.lbmref_gradients.argtypes = [dp, dp, dp, dp]
        L.lbmref_bilinear_setup.argtypes = [C.c_double, C.c_double, C.c_int32, C.c_int32, ip, dp]
        L.lbmref_node_update.argtypes = [C.POINTER(_Params), dp, dp, dp, dp, C.POINTER(NodeFields)]
        _lib = L
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_int32))


# ---- free functions (pieces pinned one by one in tests) -------------------------------------
def lattice():
    cx = np.zeros(9, np.int32); cy = np.zeros(9, np.int32); opp = np.zeros(9, np.int32)
    w = np.zeros(9)
    lib().lbmref_lattice(_ip(cx), _ip(cy), _ip(opp), _dp(w))
    return cx, cy, opp, w


def matrices():
    M = np.zeros(81); Mi = np.zeros(81)
    lib().lbmref_matrices(_dp(M), _dp(Mi))
    return M.reshape(9, 9), Mi.reshape(9, 9)


def alpha_from_mobility(m: float) -> float:
    return lib().lbmref_alpha_from_mobility(m)


def chi(alpha: float) -> np.ndarray:
    out = np.zeros(9)
    lib().lbmref_chi(alpha, _dp(out))
    return out


def ghost_rule(phiF: float, eps: float, rule: int = 0) -> float:
    return lib().lbmref_ghost_rule(phiF, eps, rule)


def neq(alpha: float, p: float, ux: float, uy: float) -> np.ndarray:
    out = np.zeros(9)
    lib().lbmref_neq(alpha, p, ux, uy, _dp(out))
    return out


def pressure(alpha: float, N: np.ndarray, ux: float, uy: float) -> float:
    N = np.ascontiguousarray(N, dtype=np.float64)
    return lib().lbmref_pressure(alpha, _dp(N), ux, uy)


def gradients(phi_nb: np.ndarray):
    nb = np.ascontiguousarray(phi_nb, dtype=np.float64)
    gx = C.c_double(); gy = C.c_double(); lap = C.c_double()
    lib().lbmref_gradients(_dp(nb), C.byref(gx), C.byref(gy), C.byref(lap))
    return gx.value, gy.value, lap.value


def bilinear_setup(xF: float, yF: float, nx: int, ny: int):
    corner = np.zeros(4, np.int32); wgt = np.zeros(4)
    lib().lbmref_bilinear_setup(xF, yF, nx, ny, _ip(corner), _dp(wgt))
    return corner, wgt


def node_update(prm: RefParams, N: np.ndarray, phi_nb: np.ndarray):
    N = np.ascontiguousarray(N, dtype=np.float64)
    nb = np.ascontiguousarray(phi_nb, dtype=np.float64)
    Ns = np.zeros(9); Bs = np.zeros(9); f = NodeFields()
    ps = prm.c_struct()
    lib().lbmref_node_update(C.byref(ps), _dp(N), _dp(nb), _dp(Ns), _dp(Bs), C.byref(f))
    return Ns, Bs, f


class RefLBM:
    """One oracle simulation (host memory only)."""

    def __init__(self, prm: RefParams, mask: np.ndarray, disks=None):
        self.prm = prm
        self.nx, self.ny = prm.nx, prm.ny
        self.n = prm.nx * prm.ny
        m = np.ascontiguousarray(mask, dtype=np.uint8).reshape(-1)
        if m.size != self.n:
            raise ValueError("mask size")
        disks = [] if disks is None else list(disks)
        arr = (_Disk * max(1, len(disks)))()
        for k, d in enumerate(disks):
            arr[k] = _Disk(float(d[0]), float(d[1]), float(d[2]))
        h = C.c_void_p()
        ps = prm.c_struct()
        rc = lib().lbmref_create(C.byref(h), C.byref(ps), m.ctypes.data, arr, len(disks))
        if rc != 0:
            raise ValueError(f"lbmref_create failed: {rc}")
        self._h = h

    def __del__(self):
        h = getattr(self, "_h", None)
        if h:
            lib().lbmref_destroy(h)
            self._h = None

    def init(self, phi0: np.ndarray, u0: np.ndarray | None = None):
        p = np.ascontiguousarray(phi0, dtype=np.float64).reshape(-1)
        assert p.size == self.n
        if u0 is not None:
            u = np.ascontiguousarray(u0, dtype=np.float64).reshape(-1)
            assert u.size == 2 * self.n
            rc = lib().lbmref_init(self._h, p.ctypes.data, u.ctypes.data)
        else:
            rc = lib().lbmref_init(self._h, p.ctypes.data, None)
        assert rc == 0

    def step(self, n: int = 1):
        assert lib().lbmref_step(self._h, int(n)) == 0

    def get(self):
        out = {k: np.zeros((self.ny, self.nx)) for k in ("rho", "phi", "ux", "uy", "p")}
        rc = lib().lbmref_get(self._h, *(out[k].ctypes.data for k in ("rho", "phi", "ux", "uy", "p")))
        assert rc == 0
        return out

    def get_populations(self):
        N = np.zeros((9, self.ny, self.nx)); B = np.zeros((9, self.ny, self.nx))
        assert lib().lbmref_get_populations(self._h, N.ctypes.data, B.ctypes.data) == 0
        return N, B

    def set_populations(self, N=None, B=None):
        Np = np.ascontiguousarray(N, dtype=np.float64) if N is not None else None
        Bp = np.ascontiguousarray(B, dtype=np.float64) if B is not None else None
        assert lib().lbmref_set_populations(self._h, Np.ctypes.data if Np is not None else None,
                                            Bp.ctypes.data if Bp is not None else None) == 0

    def get_phi_raw(self):
        phi = np.zeros((self.ny, self.nx))
        assert lib().lbmref_get_phi_raw(self._h, phi.ctypes.data) == 0
        return phi

    def get_classification(self):
        cls = np.zeros(self.n, np.uint8)
        ng = C.c_int32()
        lib().lbmref_get_classification(self._h, cls.ctypes.data, C.byref(ng), *([None] * 6))
        g = ng.value
        idx = np.zeros(max(g, 1), np.int32); gnx = np.zeros(max(g, 1)); gny = np.zeros(max(g, 1))
        dep = np.zeros(max(g, 1)); cor = np.zeros(4 * max(g, 1), np.int32); wgt = np.zeros(4 * max(g, 1))
        lib().lbmref_get_classification(self._h, None, None, idx.ctypes.data, gnx.ctypes.data,
                                        gny.ctypes.data, dep.ctypes.data, cor.ctypes.data,
                                        wgt.ctypes.data)
        return dict(cls=cls.reshape(self.ny, self.nx), n_ghost=g, idx=idx[:g], nx=gnx[:g], ny=gny[:g],
                    depth=dep[:g], corner=cor[:4 * g].reshape(g, 4), wgt=wgt[:4 * g].reshape(g, 4))

    def diag(self):
        out = np.zeros(8)
        assert lib().lbmref_diag(self._h, _dp(out)) == 0
        return dict(sum_phi=out[0], sum_1mphi=out[1], ke=out[2], umax=out[3], phi_min=out[4],
                    phi_max=out[5], n_fluid=out[6], nan=out[7])
