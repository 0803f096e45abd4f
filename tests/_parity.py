"""Helpers for the GPU parity tests: build the CUDA simulation and the CPU oracle from the SAME
seeded arrays and compare fields element by element.  No method arithmetic here."""
from __future__ import annotations

import numpy as np


def make_pair(w, precision=64, schedule=0, **over):
    from oracle import ref
    from paper_2605_30878_b200 import binding
    d = w.param_dict(); d.update(over)
    o = ref.RefLBM(ref.RefParams(**d), w.mask, w.disks)
    g = binding.LBM(binding.LBMParams(precision=precision, schedule=schedule, **d), w.mask, w.disks)
    return g, o


def field_errors(g, o, w=None):
    """max |delta| of phi, rho, u, p (absolute) between the CUDA path and the oracle."""
    a, b = g.get(), o.get()
    err = {k: float(np.abs(a[k] - b[k]).max()) for k in ("phi", "rho", "ux", "uy", "p")}
    scale = {k: float(np.abs(b[k]).max()) for k in ("phi", "rho", "ux", "uy", "p")}
    return err, scale


def pop_errors(g, o, fluid):
    g.sync()
    Ng, Bg = g.get_populations(want_B=True)
    No, Bo = o.get_populations()
    return float(np.abs(Ng - No)[:, fluid].max()), float(np.abs(Bg - Bo)[:, fluid].max())


class ArrayWorkload:
    """A Workload-like bundle for ad-hoc masks (random masks, walls) used by edge-case tests."""

    def __init__(self, mask, phi0, disks=None, **prm):
        self.mask = np.ascontiguousarray(mask, dtype=np.uint8)
        self.ny, self.nx = self.mask.shape
        self.phi0 = np.ascontiguousarray(phi0, dtype=np.float64)
        self.disks = np.zeros((0, 3)) if disks is None else np.asarray(disks, dtype=np.float64).reshape(-1, 3)
        base = dict(rho_l=10.0, rho_g=1.0, nu_l=0.1, nu_g=0.1, sigma=0.01, W=4.0, theta_deg=70.0,
                    mobility=0.02, gx=0.0, gy=0.0, wall_rows=0)
        base.update(prm)
        self.prm = base

    def param_dict(self):
        return dict(nx=self.nx, ny=self.ny, **self.prm)
