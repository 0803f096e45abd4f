"""Pins for the correction forces of the oracle's node update: F_visc (Eq. A11, reading
R10), F_p (Eq. A10, :300) and the harmonic mixture rule for the kinematic viscosity (:43, R6).

None of these re-types the oracle's formula.  What they check, and which mistake each one catches:

* `test_two_layer_poiseuille_*`: steady flow of a liquid layer under a gas layer between half-way walls,
  driven by a body acceleration.  The reference is the textbook one-dimensional problem
  (mu u')' = -rho g with mu = rho nu and the paper's mixture rules, integrated by quadrature on a fine
  grid (numpy only).  F_visc is the term that turns the model's "rho nu laplace(u)" into
  "div(mu grad u)"; without it the shear stress is not continuous across the interface.  Fails if the
  sign of `cv` flips (114 % off), if F_visc is dropped (40 %), if nu is mixed arithmetically instead of
  harmonically (2.8 %), all against a tolerance of 1.5 % (the oracle itself: 0.6-0.8 %); the run along y fails when d_x rho and d_y rho
  are exchanged in F_visc,y.
* `test_force_is_a_vector_under_rotation`: rotating the node's inputs (the non-equilibrium stress as a
  spin-2 tensor, grad phi as a vector) by 90 and by 45 degrees must rotate the returned force with
  them.  The 45-degree case mixes Pi_xx - Pi_yy with Pi_xy, so it fails if the factor 1/2 on m7 is
  dropped or the two gradients are exchanged in one component.
* `test_mobility_of_the_color_equation`: the decay rate of a sine wave of phi with the anti-diffusion switched off is
  M_phi: pins R5 (alpha = 1 - 10 M_phi / 3 at reference pressure 0) and, with it, the segregation + streaming of B.
* `test_laplace_law_density_ratio_1000`: Delta p_h = rho_l p_in - rho_g p_out = sigma / R with
  p_h = rho p (:278): fails if F_p = -p grad rho is dropped or has the wrong sign (the pressure jump
  then sits on p, not on rho p).
"""
import math

import numpy as np
import pytest

from oracle import ref
from paper_2605_30878_b200 import workloads as wl


def _diffuse_two_layer_reference(n, yI, W, rho_l, rho_g, nu_l, nu_g, g, sub=400):
    """u(y) at the nodes 0..n-1: (mu u')' = -rho g, u = 0 at the half-way walls y = 1/2 and y = n - 3/2,
    phi = 1/2 [1 - tanh(2 (y - yI)/W)] (Eq. 5), rho linear and 1/nu linear in phi."""
    ya, yb = 0.5, n - 1.5
    ys = np.linspace(ya, yb, int((yb - ya) * sub) + 1)
    phi = 0.5 * (1.0 - np.tanh(2.0 * (ys - yI) / W))
    rho = rho_l * phi + rho_g * (1.0 - phi)
    mu = rho / (phi / nu_l + (1.0 - phi) / nu_g)
    h = ys[1] - ys[0]
    cum = lambda f: np.concatenate([[0.0], np.cumsum(0.5 * (f[1:] + f[:-1]) * h)])   # noqa: E731
    R = cum(rho)                    # mu u' = C - g R(y)
    I1, I2 = cum(1.0 / mu), cum(R / mu)
    C = g * I2[-1] / I1[-1]
    return np.interp(np.arange(n), ys, C * I1 - g * I2, left=0.0, right=0.0)


def _two_layer(along_x, rho_ratio, mu_ratio, steps, n=66, W=4.0, g=1e-7):
    mu_g, rho_g = 0.1, 1.0
    rho_l, mu_l = rho_ratio * rho_g, mu_ratio * mu_g
    nu_l, nu_g = mu_l / rho_l, mu_g / rho_g
    yI = (n - 1) / 2.0
    prof = 0.5 * (1.0 - np.tanh(2.0 * (np.arange(n) - yI) / W))
    if along_x:      # walls are the rows j = 0, n-1; flow along x, gradients along y
        mask = np.zeros((n, 4), np.uint8); mask[0] = 1; mask[-1] = 1
        phi0 = np.repeat(prof[:, None], 4, axis=1)
        prm = ref.RefParams(nx=4, ny=n, rho_l=rho_l, rho_g=rho_g, nu_l=nu_l, nu_g=nu_g, sigma=0.0, W=W, gx=g, wall_rows=1)
    else:            # walls are the columns i = 0, n-1 (normals from the mask alone); flow along y
        mask = np.zeros((4, n), np.uint8); mask[:, 0] = 1; mask[:, -1] = 1
        phi0 = np.repeat(prof[None, :], 4, axis=0)
        prm = ref.RefParams(nx=n, ny=4, rho_l=rho_l, rho_g=rho_g, nu_l=nu_l, nu_g=nu_g, sigma=0.0, W=W, gy=g)
    s = ref.RefLBM(prm, mask); s.init(phi0); s.step(steps)
    f = s.get()
    u = f["ux"][:, 0] if along_x else f["uy"][0, :]
    v = f["uy"] if along_x else f["ux"]
    return u, np.abs(v).max(), _diffuse_two_layer_reference(n, yI, W, rho_l, rho_g, nu_l, nu_g, g)


@pytest.mark.parametrize("rho_ratio,mu_ratio,steps", [(10.0, 40.0, 50000), (100.0, 100.0, 50000)])
def test_two_layer_poiseuille_along_x(rho_ratio, mu_ratio, steps):
    u, vmax, uref = _two_layer(True, rho_ratio, mu_ratio, steps)
    assert np.abs(u - uref).max() <= 0.015 * uref.max(), (np.abs(u - uref).max() / uref.max())
    assert vmax < 1e-9 * uref.max() + 1e-14


def test_two_layer_poiseuille_along_y():
    u, vmax, uref = _two_layer(False, 10.0, 40.0, 50000)
    assert np.abs(u - uref).max() <= 0.015 * uref.max(), (np.abs(u - uref).max() / uref.max())
    assert vmax < 1e-9 * uref.max() + 1e-14


def _node_force(prm, m7, m8, gphi, phi=0.4):
    """Total force of one node at rest (sigma = 0, g = 0: F = F_p + F_visc) whose populations carry the
    non-equilibrium stress moments (m7, m8) = (Pi_xx - Pi_yy, Pi_xy) and whose phi neighbourhood is linear
    with gradient gphi."""
    cx, cy, _, w = ref.lattice()
    chi = ref.chi(ref.alpha_from_mobility(prm.mobility))
    # least-norm population increment with the wanted second moments and no mass, momentum or trace:
    # plain linear algebra on the lattice vectors
    A = np.stack([np.ones(9), cx, cy, cx * cx + cy * cy, cx * cx - cy * cy, cx * cy]).astype(float)
    dN = np.linalg.lstsq(A, np.array([0, 0, 0, 0, m7, m8], float), rcond=None)[0]
    nb = phi + gphi[0] * cx + gphi[1] * cy
    _, _, f = ref.node_update(prm, chi + dN, nb)
    return np.array([f.Fx, f.Fy]), f


def test_force_is_a_vector_under_rotation():
    prm = ref.RefParams(nx=8, ny=8, rho_l=50.0, rho_g=1.0, nu_l=0.2, nu_g=0.05, sigma=0.0, W=4.0)
    rng = np.random.default_rng(5)
    for _ in range(20):
        m7, m8 = rng.normal(0, 1e-4, 2)
        gphi = rng.normal(0, 0.02, 2)
        F0, f0 = _node_force(prm, m7, m8, gphi)
        assert np.hypot(*F0) > 1e-8            # the case is not degenerate
        for deg in (90.0, 45.0, 30.0):
            a = math.radians(deg)
            c, s = math.cos(a), math.sin(a)
            Rm = np.array([[c, -s], [s, c]])
            # a symmetric traceless tensor with components (a, b) = (m7/2, m8) rotates by twice the angle
            a2, b2 = math.cos(2 * a) * (0.5 * m7) - math.sin(2 * a) * m8, math.sin(2 * a) * (0.5 * m7) + math.cos(2 * a) * m8
            F1, f1 = _node_force(prm, 2.0 * a2, b2, Rm @ gphi)
            assert f1.p == pytest.approx(f0.p, abs=1e-15)
            assert np.allclose(F1, Rm @ F0, rtol=0, atol=1e-12 * np.hypot(*F0)), (deg, F1, Rm @ F0)


def test_laplace_law_density_ratio_1000():
    """the hydrodynamic pressure is p_h = rho p, so across a drop of liquid 1000 times denser
    than the gas Delta p_h = rho_l p_in - rho_g p_out = sigma / R (2-D)."""
    n, R, sigma = 64, 16.0, 0.01
    mask, disks, phi0 = wl.free_droplet(n, R, 4.0)
    prm = ref.RefParams(nx=n, ny=n, rho_l=1000.0, rho_g=1.0, nu_l=0.01, nu_g=0.1, sigma=sigma, W=4.0)
    s = ref.RefLBM(prm, mask, disks); s.init(phi0); s.step(6000)
    g, d = s.get(), s.diag()
    ph = g["rho"] * g["p"]
    dp = ph[n // 2, n // 2] - ph[2, 2]
    Reff = math.sqrt(d["sum_phi"] / math.pi)
    assert dp / (sigma / Reff) == pytest.approx(1.0, abs=0.08)
    # the jump is carried by rho p: p itself is three orders of magnitude smaller inside the liquid
    assert abs(g["p"][n // 2, n // 2]) < 5e-3 * sigma / Reff
    assert d["umax"] < 1e-4


@pytest.mark.parametrize("mobility", [0.02, 0.05])
def test_mobility_of_the_color_equation(mobility):
    """R5: alpha is never printed, only M_phi = 0.02 and M_phi = c_s^2 dt/2 [9(1 - alpha)/5 + p/c_s^2]
    (:288); the oracle takes the reference pressure p = 0, i.e. alpha = 1 - 10 M_phi / 3.  The pin measures the
    mobility the scheme actually has: with the anti-diffusion switched off (W -> infinity; Eq. 3, :41) and the fluid at
    rest, a small sine wave of phi must decay as exp(-M_phi k^2 t).  Any other reading of alpha shows up one to one
    in the measured rate (recorded: 0.9991 M_phi, the rest is the O(k^2) lattice correction)."""
    nx, ny, a0, T = 64, 4, 0.01, 4000
    k = 2.0 * math.pi / nx
    phi0 = 0.5 + a0 * np.sin(k * np.arange(nx))[None, :] * np.ones((ny, 1))
    prm = ref.RefParams(nx=nx, ny=ny, rho_l=1.0, rho_g=1.0, nu_l=1 / 6, nu_g=1 / 6, sigma=0.0, W=1e7, mobility=mobility)
    s = ref.RefLBM(prm, np.zeros((ny, nx), np.uint8)); s.init(phi0); s.step(T)
    g = s.get()
    row = g["phi"][0]
    a = 2.0 * abs(np.fft.rfft(row - row.mean())[1]) / nx
    assert -math.log(a / a0) / (k * k * T) == pytest.approx(mobility, rel=5e-3)
    assert np.abs(g["phi"] - row[None, :]).max() < 1e-15 and max(np.abs(g["ux"]).max(), np.abs(g["uy"]).max()) < 1e-12
