"""Oracle pins, part 2: the ghost-node rule Eq. 9, its relation to Eq. 10-11
(PAPER.md:84-91), bilinear interpolation and the isotropic stencils (R8)."""
import math

import numpy as np
import pytest

from oracle import ref

rng = np.random.default_rng(7)


def test_eq9_bounds_and_fixed_points():
    for eps in (-1.0, -0.3, 0.0, 0.4, 1.0):
        for phiF in np.linspace(0.001, 0.999, 31):
            g = ref.ghost_rule(phiF, eps, 0)
            assert 0 < g < 1
        assert ref.ghost_rule(0.0, eps, 0) == 0.0              # no mass transfer along the wall
        assert ref.ghost_rule(1.0, eps, 0) == 1.0
    for phiF in (0.1, 0.5, 0.9):                               # theta = 90 deg: eps = 0
        assert ref.ghost_rule(phiF, 0.0, 0) == pytest.approx(phiF, abs=1e-16)
        assert ref.ghost_rule(phiF, 0.0, 1) == pytest.approx(phiF, abs=1e-16)


def test_eq9_sign_wetting_raises_ghost_phi():
    # hydrophilic: theta < 90 -> eps < 0 -> more liquid in the wall
    eps = -(4 / 4.0) * math.cos(math.radians(30))
    assert ref.ghost_rule(0.5, eps, 0) > 0.5
    assert ref.ghost_rule(0.5, -eps, 0) < 0.5


def test_eq9_liquid_gas_symmetry():
    for eps in (-0.8, 0.25):
        for phiF in (0.05, 0.3, 0.77):
            assert ref.ghost_rule(1 - phiF, -eps, 0) == pytest.approx(1 - ref.ghost_rule(phiF, eps, 0), abs=1e-15)


@pytest.mark.parametrize("theta,W", [(30, 4), (60, 5), (110, 4), (150, 8)])
def test_eq9_is_exact_integral_of_eq8(theta, W):
    """If phi(eta_s) = 1/(1 + C e^{k eta_s}) with k = 4 cos(theta)/W (the solution of Eq. 8),
    Eq. 9 returns phi(eta_F - 1) exactly."""
    k = 4 * math.cos(math.radians(theta)) / W
    eps = -k
    for C in (0.05, 1.0, 7.0):
        for etaF in (-1.3, 0.2, 2.0):
            phiF = 1 / (1 + C * math.exp(k * etaF))
            phiG = 1 / (1 + C * math.exp(k * (etaF - 1)))
            assert ref.ghost_rule(phiF, eps, 0) == pytest.approx(phiG, abs=1e-15)
    # and the derivative at the wall matches Eq. 8 to O(h^2) when integrated by a fine RK4
    phi = 0.37
    h = 1e-3
    f = lambda y: -(4 / W) * y * (1 - y) * math.cos(math.radians(theta))
    y = phi
    for _ in range(1000):                                       # integrate from x_F back to x_G
        k1 = f(y); k2 = f(y - 0.5 * h * k1); k3 = f(y - 0.5 * h * k2); k4 = f(y - h * k3)
        y -= h * (k1 + 2 * k2 + 2 * k3 + k4) / 6
    assert ref.ghost_rule(phi, eps, 0) == pytest.approx(y, abs=1e-12)


def test_eq10_solves_midpoint_rule():
    """Eq. 10 is the root of (phi_F - phi_G) = eps phi_m (1 - phi_m), phi_m = (phi_F + phi_G)/2."""
    for eps in (-0.9, -0.1, 0.3, 1.0):
        for phiF in (0.1, 0.5, 0.8):
            g = ref.ghost_rule(phiF, eps, 1)
            pm = 0.5 * (phiF + g)
            assert (phiF - g) == pytest.approx(eps * pm * (1 - pm), abs=1e-14)


def test_eq10_near_ninety_degrees():
    """Eq. 10 "needs special care" at theta = 90 deg (eps = 0).  The oracle's form of Eq. 10 has
    no singular point: it still solves the midpoint rule to rounding for tiny eps, reduces to phi_G = phi_F at
    eps = 0 and agrees with the expression as printed, evaluated with 50 digits, across the range."""
    from decimal import Decimal, getcontext
    getcontext().prec = 50
    for eps in (1e-2, 1e-4, 1e-6, 1e-9, 1e-13, -1e-6, -1e-11):
        for phiF in (0.05, 0.37, 0.5, 0.93):
            g = ref.ghost_rule(phiF, eps, 1)
            pm = 0.5 * (phiF + g)
            assert abs((phiF - g) - eps * pm * (1 - pm)) <= 1e-15       # a few ulp of phi_F
            e, f = Decimal(eps), Decimal(phiF)
            a = 1 + e / 2
            printed = (2 / e) * (a - (a * a - 2 * e * f).sqrt()) - f        # Eq. 10 as printed
            assert abs(Decimal(g) - printed) <= Decimal(1e-15)
    for phiF in (0.0, 0.2, 1.0):
        assert ref.ghost_rule(phiF, 0.0, 1) == phiF


def test_eq11_series_difference():
    """Eq. 9 - Eq. 10 = eps^3/12 [1 - 3(1-phi_F)phi_F] phi_F (1-phi_F) + O(eps^4)."""
    for phiF in (0.2, 0.5, 0.7):
        lead = lambda e: e ** 3 / 12 * (1 - 3 * (1 - phiF) * phiF) * phiF * (1 - phiF)
        ratios = []
        for eps in (0.2, 0.1, 0.05):
            diff = ref.ghost_rule(phiF, eps, 0) - ref.ghost_rule(phiF, eps, 1)
            ratios.append(diff / lead(eps))
        assert abs(ratios[-1] - 1) < 0.05
        assert abs(ratios[-1] - 1) < abs(ratios[0] - 1)         # converges as eps -> 0


def test_bilinear_exact_on_bilinear_functions_and_seam():
    nx, ny = 11, 7
    a, b, c, d = 0.3, -1.2, 0.7, 0.45
    fn = lambda x, y: a + b * x + c * y + d * x * y
    # interior points
    for _ in range(20):
        xF, yF = rng.uniform(0, nx - 1.001), rng.uniform(0, ny - 1.001)
        cor, w = ref.bilinear_setup(xF, yF, nx, ny)
        assert abs(w.sum() - 1) < 1e-15 and (w >= 0).all()
        vals = np.array([fn(k % nx, k // nx) for k in cor])
        assert (w * vals).sum() == pytest.approx(fn(xF, yF), abs=1e-13)
    # across the periodic seam: corners wrap
    cor, w = ref.bilinear_setup(-0.25, 2.5, nx, ny)
    assert list(cor) == [2 * nx + nx - 1, 2 * nx + 0, 3 * nx + nx - 1, 3 * nx + 0]
    assert np.allclose(w, [0.25 * 0.5, 0.75 * 0.5, 0.25 * 0.5, 0.75 * 0.5])
    cor, w = ref.bilinear_setup(nx - 0.5, ny - 0.75, nx, ny)
    assert list(cor) == [(ny - 1) * nx + nx - 1, (ny - 1) * nx, nx - 1, 0]
    # exactly on a node: weight 1 on it
    cor, w = ref.bilinear_setup(3.0, 1.0, nx, ny)
    assert cor[0] == 1 * nx + 3 and w[0] == 1.0 and w[1:].sum() == 0.0


def test_gradient_stencils_exact_on_quadratics():
    CX = np.array([0, 1, 0, -1, 0, 1, -1, -1, 1]); CY = np.array([0, 0, 1, 0, -1, 1, 1, -1, -1])
    for _ in range(10):
        a, b, c, d, e, f0 = rng.normal(size=6)
        x0, y0 = rng.normal(size=2)
        q = lambda x, y: f0 + a * x + b * y + c * x * x + d * x * y + e * y * y
        nb = np.array([q(x0 + CX[i], y0 + CY[i]) for i in range(9)])
        gx, gy, lap = ref.gradients(nb)
        assert gx == pytest.approx(a + 2 * c * x0 + d * y0, abs=1e-13)
        assert gy == pytest.approx(b + d * x0 + 2 * e * y0, abs=1e-13)
        assert lap == pytest.approx(2 * c + 2 * e, abs=1e-13)


def test_ghost_update_is_jacobi_and_matches_bilinear_by_hand():
    """One oracle step on a tiny case: the stored ghost values equal Eq. 9 applied to the bilinear
    interpolation of the PRE-update array (R13), checked with an independent numpy gather."""
    from paper_2605_30878_b200 import workloads as wl
    w = wl.config1(3)
    prm = ref.RefParams(**w.param_dict())
    sim = ref.RefLBM(prm, w.mask, w.disks)
    sim.init(w.phi0)
    before = sim.get_phi_raw().ravel().copy()       # fluid: phi0, solid: (1+cos theta)/2
    assert np.allclose(before[w.mask.ravel() == 1], 0.5 * (1 + math.cos(math.radians(60))))
    sim.step(1)
    after = sim.get_phi_raw().ravel()
    cl = sim.get_classification()
    eps = -(4 / w.W) * math.cos(math.radians(w.theta_deg))
    # at t = 0 sum_i B_i = phi0 up to rounding, so `before` is the pre-update array
    phiF = (cl["wgt"] * before[cl["corner"]]).sum(axis=1)
    expect = phiF / (phiF + (1 - phiF) * math.exp(eps))
    assert np.allclose(after[cl["idx"]], expect, atol=1e-14)
    bulk = cl["cls"].ravel() == 3
    assert np.array_equal(after[bulk], before[bulk])            # bulk solid keeps its value (R15)
