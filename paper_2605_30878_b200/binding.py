"""ctypes binding of ``liblbm_b200.so`` (``include/lbm.h``) — argument marshalling only.

Every step of the path runs in the CUDA kernels of ``csrc/``; this module converts numpy arrays to
pointers, lets PyTorch allocate the device workspace and hands the library torch's current CUDA
stream.  There is no CPU fallback: without the built library or without a CUDA device the calls
raise.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_INC = os.path.join(os.path.dirname(_HERE), "include")
_SO = os.path.join(_HERE, "liblbm_b200.so")

SCHEDULE_AUTO, SCHEDULE_BASELINE, SCHEDULE_FUSED, SCHEDULE_PAIR, SCHEDULE_PACK, SCHEDULE_SPARSE = 0, 1, 2, 4, 5, 6
SCHEDULE_INPLACE = 7
FLUID_BULK, FLUID_BOUNDARY, GHOST, SOLID_BULK = 0, 1, 2, 3

# include/lbm.h (the product boundary) and include/lbm_test.h (test and measurement hooks)
EXPORTS = ("lbm_plan", "lbm_workspace_bytes", "lbm_nu_from_tau", "lbm_tau_from_nu", "lbm_create", "lbm_init", "lbm_step", "lbm_sync", "lbm_get",
           "lbm_get_populations", "lbm_set_populations", "lbm_rows_bytes", "lbm_rows_export", "lbm_rows_import",
           "lbm_keep_B", "lbm_sample_populations",
           "lbm_get_classification", "lbm_diag", "lbm_diag_static", "lbm_last_error", "lbm_version", "lbm_destroy")
TEST_EXPORTS = ("lbm_node_update_batch", "lbm_step_timed", "lbm_layout_copy_timed", "lbm_launch_counts")


def _sources():
    out = [os.path.join(_INC, "lbm.h"), os.path.join(_INC, "lbm_test.h")]
    for f in sorted(os.listdir(_CSRC)):
        if f.endswith((".cu", ".cuh", ".h")):
            out.append(os.path.join(_CSRC, f))
    return out


def build_library(force: bool = False, verbose: bool = False) -> str:
    """nvcc -> liblbm_b200.so for sm_100a, in-tree (cross-compiles without a GPU)."""
    srcs = _sources()
    stale = force or not os.path.exists(_SO) or any(os.path.getmtime(s) > os.path.getmtime(_SO) for s in srcs)
    if stale:
        cmd = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
               "-shared", "-Xcompiler", "-fPIC", "-diag-suppress", "550", "-o", _SO,
               os.path.join(_CSRC, "lbm_api.cu")]
        cmd[1:1] = os.environ.get("LBM_NVCC_EXTRA", "").split()   # tuning sweeps: -DLBM_PAIR_DP32=1 ...
        if verbose:
            cmd.insert(1, "-Xptxas")
            cmd.insert(2, "-v")
        subprocess.check_call(cmd)
    return _SO


class _Params(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("precision", C.c_int32), ("wall_rows", C.c_int32),
                ("ghost_rule", C.c_int32), ("schedule", C.c_int32),
                ("rho_l", C.c_double), ("rho_g", C.c_double), ("nu_l", C.c_double), ("nu_g", C.c_double),
                ("sigma", C.c_double), ("W", C.c_double), ("theta_deg", C.c_double),
                ("mobility", C.c_double), ("gx", C.c_double), ("gy", C.c_double)]


class _Disk(C.Structure):
    _fields_ = [("cx", C.c_double), ("cy", C.c_double), ("r", C.c_double)]


@dataclass
class LBMParams:
    nx: int
    ny: int
    precision: int = 64
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
    schedule: int = SCHEDULE_AUTO

    def c_struct(self) -> _Params:
        return _Params(self.nx, self.ny, self.precision, self.wall_rows, self.ghost_rule, self.schedule,
                       self.rho_l, self.rho_g, self.nu_l, self.nu_g, self.sigma, self.W, self.theta_deg,
                       self.mobility, self.gx, self.gy)


_lib = None


def load_library() -> C.CDLL:
    """Loads the in-tree shared library; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise RuntimeError(f"{_SO} is missing: run `python -c 'import __graft_entry__ as g; g.build()'`")
        L = C.CDLL(_SO)
        vp, i64 = C.c_void_p, C.c_int64
        L.lbm_plan.argtypes = [C.POINTER(_Params), vp, C.POINTER(i64), C.POINTER(C.c_size_t)]
        L.lbm_workspace_bytes.argtypes = [C.POINTER(_Params), i64]
        L.lbm_workspace_bytes.restype = C.c_size_t
        for f in (L.lbm_nu_from_tau, L.lbm_tau_from_nu):
            f.argtypes, f.restype = [C.c_double], C.c_double
        L.lbm_set_populations.argtypes = [vp, vp, vp]
        L.lbm_rows_bytes.argtypes = [vp, C.c_int32, C.c_int32, C.POINTER(C.c_size_t)]
        L.lbm_rows_export.argtypes = [vp, C.c_int32, C.c_int32, vp, C.c_size_t]
        L.lbm_rows_import.argtypes = [vp, C.c_int32, C.c_int32, vp, C.c_size_t]
        L.lbm_create.argtypes = [C.POINTER(vp), C.POINTER(_Params), vp, vp, C.c_int32, vp,
                                 C.c_size_t, vp]
        L.lbm_init.argtypes = [vp, vp, vp]
        L.lbm_step.argtypes = [vp, i64]
        L.lbm_sync.argtypes = [vp]
        L.lbm_step_timed.argtypes = [vp, i64, vp]
        L.lbm_layout_copy_timed.argtypes = [vp, C.c_int32, C.POINTER(C.c_double)]
        L.lbm_get.argtypes = [vp] * 6
        L.lbm_get_populations.argtypes = [vp, vp, vp]
        L.lbm_keep_B.argtypes = [vp, C.c_int32]
        L.lbm_sample_populations.argtypes = [vp, i64, vp, vp, vp]
        L.lbm_get_classification.argtypes = [vp] * 9
        L.lbm_diag.argtypes = [vp, vp]
        L.lbm_diag_static.argtypes = [vp, vp]
        L.lbm_node_update_batch.argtypes = [C.POINTER(_Params), i64, vp, vp, vp, vp, vp]
        L.lbm_launch_counts.argtypes = [vp, vp, C.c_int32]
        L.lbm_last_error.argtypes = [vp]
        L.lbm_last_error.restype = C.c_char_p
        L.lbm_version.restype = C.c_char_p
        L.lbm_destroy.argtypes = [vp]
        L.lbm_destroy.restype = None
        _lib = L
    return _lib


class LBMError(RuntimeError):
    pass


def _check(rc: int, h=None):
    if rc != 0:
        msg = load_library().lbm_last_error(h).decode(errors="replace")
        raise LBMError(f"liblbm_b200 error {rc}: {msg}")


def _f64(a, size=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if size is not None and a.size != size:
        raise ValueError(f"expected {size} values, got {a.size}")
    return a


def nu_from_tau(tau: float) -> float:
    """Kinematic viscosity of a phase from its relaxation time (tau = 1/2 + 3 nu)."""
    return float(load_library().lbm_nu_from_tau(float(tau)))


def tau_from_nu(nu: float) -> float:
    return float(load_library().lbm_tau_from_nu(float(nu)))


def workspace_bytes(prm: LBMParams, n_ghost_bound: int) -> int:
    """Host-only upper bound of the workspace size (no device, no mask)."""
    ps = prm.c_struct()
    return int(load_library().lbm_workspace_bytes(C.byref(ps), int(n_ghost_bound)))


def node_update_batch(prm: LBMParams, N, phi_nb):
    """Test hook: local update of independent nodes on the device.  N, phi_nb: [count, 9]."""
    N = _f64(N).reshape(-1, 9)
    P = _f64(phi_nb).reshape(-1, 9)
    cnt = N.shape[0]
    Ns = np.zeros((cnt, 9)); Bs = np.zeros((cnt, 9)); F = np.zeros((cnt, 8))
    ps = prm.c_struct()
    _check(load_library().lbm_node_update_batch(C.byref(ps), cnt, N.ctypes.data, P.ctypes.data,
                                                Ns.ctypes.data, Bs.ctypes.data, F.ctypes.data))
    keys = ("rho", "tau", "ux", "uy", "p", "Fx", "Fy", "gnorm")
    return Ns, Bs, {k: F[:, i] for i, k in enumerate(keys)}


class LBM:
    """One simulation on the current CUDA device.  Device memory comes from a torch tensor, the
    stream is torch's current stream (PyTorch is plumbing only)."""

    def __init__(self, prm: LBMParams, mask, disks=None, device=None, own_stream: bool = False):
        """own_stream: enqueue on a new non-default torch stream instead of the current one (the legacy default
        stream cannot be captured, so lbm_step replays CUDA graphs on small grids only off it)."""
        import torch
        if not torch.cuda.is_available():
            raise LBMError("no CUDA device: liblbm_b200 has no CPU fallback")
        L = load_library()
        self.prm = prm
        self.nx, self.ny, self.n = prm.nx, prm.ny, prm.nx * prm.ny
        m = np.ascontiguousarray(mask, dtype=np.uint8).reshape(-1)
        if m.size != self.n:
            raise ValueError("mask size")
        disks = np.zeros((0, 3)) if disks is None else np.asarray(disks, dtype=np.float64).reshape(-1, 3)
        disks = np.ascontiguousarray(disks)          # lbm_disk = 3 doubles (cx, cy, r)
        ps = prm.c_struct()
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        with torch.cuda.device(self.device):
            ng, ws = C.c_int64(), C.c_size_t()
            _check(L.lbm_plan(C.byref(ps), m.ctypes.data, C.byref(ng), C.byref(ws)))
            self.workspace_bytes = ws.value
            self._ws = torch.empty(ws.value, dtype=torch.uint8, device=self.device)
            self._stream = torch.cuda.Stream(self.device) if own_stream else torch.cuda.current_stream(self.device)
            h = C.c_void_p()
            _check(L.lbm_create(C.byref(h), C.byref(ps), m.ctypes.data, disks.ctypes.data if len(disks) else None, len(disks),
                                C.c_void_p(self._ws.data_ptr()), ws.value,
                                C.c_void_p(self._stream.cuda_stream)))
        self._h = h
        self.n_ghost = ng.value

    def close(self):
        h = getattr(self, "_h", None)
        if h:
            load_library().lbm_destroy(h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the four calls of the north star ---------------------------------------------------
    def init(self, phi0, u0=None):
        p = _f64(phi0, self.n)
        u = _f64(u0, 2 * self.n) if u0 is not None else None
        _check(load_library().lbm_init(self._h, p.ctypes.data, u.ctypes.data if u is not None else None), self._h)

    def step(self, n: int = 1):
        _check(load_library().lbm_step(self._h, int(n)), self._h)

    def step_timed(self, n: int = 1):
        """n steps with per-kernel CUDA-event timing: summed ms of (collide, phi_sum, ghost)."""
        ms = np.zeros(3)
        _check(load_library().lbm_step_timed(self._h, int(n), ms.ctypes.data), self._h)
        return dict(collide=float(ms[0]), phi_sum=float(ms[1]), ghost=float(ms[2]))

    def layout_copy_timed(self, iters: int = 20) -> float:
        """ms of one pass of the plain sector copy over this context's state (the layout's ceiling)."""
        ms = C.c_double()
        _check(load_library().lbm_layout_copy_timed(self._h, int(iters), C.byref(ms)), self._h)
        return float(ms.value)

    def sync(self):
        _check(load_library().lbm_sync(self._h), self._h)

    def get(self, fields=("rho", "phi", "ux", "uy", "p"), out=None):
        names = ("rho", "phi", "ux", "uy", "p")
        res = {}
        ptrs = []
        for k in names:
            if k in fields:
                a = out[k] if out is not None else np.empty((self.ny, self.nx))
                res[k] = a
                ptrs.append(a.ctypes.data)
            else:
                ptrs.append(None)
        _check(load_library().lbm_get(self._h, *ptrs), self._h)
        return res

    # -- state access for tests ---------------------------------------------------------------
    def keep_B(self, on: bool = True):
        _check(load_library().lbm_keep_B(self._h, 1 if on else 0), self._h)

    def get_populations(self, want_B: bool = True):
        N = np.empty((9, self.ny, self.nx))
        B = np.empty((9, self.ny, self.nx)) if want_B else None
        _check(load_library().lbm_get_populations(self._h, N.ctypes.data, B.ctypes.data if want_B else None), self._h)
        return N, B

    def set_populations(self, N=None, B=None):
        """Overwrites the post-stream populations of the current time (arrays shaped like get_populations')."""
        Na = _f64(N, 9 * self.n) if N is not None else None
        Ba = _f64(B, 9 * self.n) if B is not None else None
        _check(load_library().lbm_set_populations(self._h, Na.ctypes.data if Na is not None else None,
                                                  Ba.ctypes.data if Ba is not None else None), self._h)

    def rows_bytes(self, j0: int, nrows: int) -> int:
        """Bytes of the state that belongs to the grid rows j0 <= j < j0 + nrows (no wrap)."""
        b = C.c_size_t()
        _check(load_library().lbm_rows_bytes(self._h, int(j0), int(nrows), C.byref(b)), self._h)
        return int(b.value)

    def rows_export(self, j0: int, nrows: int, buf_ptr: int, capacity: int):
        """Copies those rows of the state (phi and the populations) into a DEVICE buffer; asynchronous on the stream."""
        _check(load_library().lbm_rows_export(self._h, int(j0), int(nrows), int(buf_ptr), int(capacity)), self._h)

    def rows_import(self, j0: int, nrows: int, buf_ptr: int, nbytes: int):
        """Overwrites those rows of the state from a DEVICE buffer another context exported; asynchronous."""
        _check(load_library().lbm_rows_import(self._h, int(j0), int(nrows), int(buf_ptr), int(nbytes)), self._h)

    def sample_populations(self, idx, want_B: bool = False):
        idx = np.ascontiguousarray(idx, dtype=np.int64).reshape(-1)
        N = np.empty((9, idx.size))
        B = np.empty((9, idx.size)) if want_B else None
        _check(load_library().lbm_sample_populations(self._h, idx.size, idx.ctypes.data, N.ctypes.data,
                                                     B.ctypes.data if want_B else None), self._h)
        return N, B

    def get_classification(self):
        cls = np.empty(self.n, np.uint8)
        ng = C.c_int32()
        L = load_library()
        _check(L.lbm_get_classification(self._h, cls.ctypes.data, C.addressof(ng), *([None] * 6)), self._h)
        g = ng.value
        idx = np.zeros(g, np.int32); gnx = np.zeros(g); gny = np.zeros(g); dep = np.zeros(g)
        cor = np.zeros(4 * g, np.int32); wgt = np.zeros(4 * g)
        if g:
            _check(L.lbm_get_classification(self._h, None, None, idx.ctypes.data, gnx.ctypes.data, gny.ctypes.data,
                                            dep.ctypes.data, cor.ctypes.data, wgt.ctypes.data), self._h)
        return dict(cls=cls.reshape(self.ny, self.nx), n_ghost=g, idx=idx, nx=gnx, ny=gny, depth=dep,
                    corner=cor.reshape(g, 4), wgt=wgt.reshape(g, 4))

    def diag(self):
        out = np.zeros(8)
        _check(load_library().lbm_diag(self._h, out.ctypes.data), self._h)
        return dict(sum_phi=out[0], sum_1mphi=out[1], ke=out[2], umax=out[3], phi_min=out[4],
                    phi_max=out[5], n_fluid=out[6], nan=out[7])

    def diag_static(self, out_ptr: int):
        """lbm_diag without allocation, host copy or synchronisation: the eight values go to a DEVICE buffer of 8 doubles
        (asynchronous on the stream); the reduction's scratch is a static device array of the library (lbm.h: limits)."""
        _check(load_library().lbm_diag_static(self._h, int(out_ptr)), self._h)

    def launch_counts(self, reset: bool = False):
        out = np.zeros(4, np.int64)
        _check(load_library().lbm_launch_counts(self._h, out.ctypes.data, 1 if reset else 0), self._h)
        return dict(collide=int(out[0]), phi_sum=int(out[1]), ghost=int(out[2]), other=int(out[3]))
