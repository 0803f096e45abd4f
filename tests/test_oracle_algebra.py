"""Oracle pins, part 1: the lattice algebra of App. A against identities the paper and the
mathematics fix.  A dropped term, wrong sign, wrong index or transposed
operand in oracle/lbmref.c fails one of these."""
import numpy as np
import pytest

from oracle import ref

CX = np.array([0, 1, 0, -1, 0, 1, -1, -1, 1])
CY = np.array([0, 0, 1, 0, -1, 1, 1, -1, -1])
W9 = np.array([4 / 9] + [1 / 9] * 4 + [1 / 36] * 4)
rng = np.random.default_rng(1234)


def test_lattice_eq_A5_A6():
    cx, cy, opp, w = ref.lattice()
    assert (cx == CX).all() and (cy == CY).all()             # Eq. A5
    assert np.allclose(w, W9, rtol=0, atol=1e-17)             # Eq. A6
    assert (cx[opp] == -cx).all() and (cy[opp] == -cy).all()
    assert abs(w.sum() - 1) < 1e-15
    # isotropy: sum w c c = c_s^2 I
    assert abs((w * cx * cx).sum() - 1 / 3) < 1e-15 and abs((w * cx * cy).sum()) < 1e-15


def test_M_rows_orthogonal_and_named_rows():
    M, Mi = ref.matrices()
    G = M @ M.T
    assert np.allclose(G - np.diag(np.diag(G)), 0)                        # R1
    assert np.allclose(np.diag(G), [9, 36, 36, 6, 12, 6, 12, 4, 4])
    assert (M[3] == CX).all() and (M[5] == CY).all()
    assert (M[7] == CX * CX - CY * CY).all() and (M[8] == CX * CY).all()
    assert (M[0] == 1).all()
    assert np.allclose(M @ Mi, np.eye(9), atol=1e-15) and np.allclose(Mi @ M, np.eye(9), atol=1e-15)
    assert np.allclose(Mi, np.linalg.inv(M), atol=1e-15)


def test_alpha_and_chi():
    a = ref.alpha_from_mobility(0.02)
    assert abs(a - 14 / 15) < 1e-15                            # R5: M_phi = 0.02 at p = 0
    # PAPER.md:288 evaluated at p = 0
    assert abs(0.5 / 3 * (9 * (1 - a) / 5) - 0.02) < 1e-16
    chi = ref.chi(a)
    assert abs(chi.sum() - 1) < 1e-15
    assert np.allclose(chi[1:5], (1 - a) / 5) and np.allclose(chi[5:], (1 - a) / 20) and chi[0] == a
    # second moment of chi gives the mobility coefficient 3(1-alpha)/5
    assert abs((chi * CX * CX).sum() - 3 * (1 - a) / 5) < 1e-16


@pytest.mark.parametrize("k", range(8))
def test_neq_moments_and_A15_inverts_A4(k):
    a = 14 / 15
    p, ux, uy = rng.normal(0, 1e-2), rng.normal(0, 5e-2), rng.normal(0, 5e-2)
    N = ref.neq(a, p, ux, uy)
    assert abs(N.sum() - 1) < 1e-15                             # R4
    assert abs((N * CX).sum() - ux) < 1e-16 and abs((N * CY).sum() - uy) < 1e-16
    # stress moments of the equilibrium
    assert abs((N * (CX * CX - CY * CY)).sum() - (ux * ux - uy * uy)) < 1e-16
    assert abs((N * CX * CY).sum() - ux * uy) < 1e-16
    assert abs(ref.pressure(a, N, ux, uy) - p) < 1e-15          # A15 is the inverse of A4
    # i != 0 branch written out (Eq. A4)
    chi = ref.chi(a)
    cu = CX * ux + CY * uy
    expect = chi + W9 * (3 * p + 3 * cu + 4.5 * cu * cu - 1.5 * (ux * ux + uy * uy))
    assert np.allclose(N[1:], expect[1:], atol=1e-16)


def _params(**kw):
    base = dict(nx=8, ny=8, rho_l=1000.0, rho_g=1.0, nu_l=0.01, nu_g=0.1, sigma=0.01, W=4.0,
                theta_deg=70.0, gx=1e-6, gy=-2e-6)
    base.update(kw)
    return ref.RefParams(**base)


def _random_node(scale=1e-3):
    a = 14 / 15
    N = ref.neq(a, rng.normal(0, 1e-4), rng.normal(0, 1e-2), rng.normal(0, 1e-2))
    N = N + rng.normal(0, scale, 9) * W9
    phic = rng.uniform(0.05, 0.95)
    nb = phic + rng.normal(0, 0.05, 9)
    nb[0] = phic
    return N, nb


@pytest.mark.parametrize("k", range(6))
def test_node_update_invariants(k):
    prm = _params()
    N, nb = _random_node()
    Ns, Bs, f = ref.node_update(prm, N, nb)
    # S has rate 1 on the density row (R7): sum N* = 1 after every collision
    assert abs(Ns.sum() - 1) < 2e-15
    # segregation conserves the order parameter: sum B* = phi
    assert abs(Bs.sum() - nb[0]) < 2e-15
    # A14 holds for the final (u, F): u = j + F/(2 rho)
    jx, jy = (N * CX).sum(), (N * CY).sum()
    assert abs(f.ux - (jx + f.Fx / (2 * f.rho))) < 1e-15
    assert abs(f.uy - (jy + f.Fy / (2 * f.rho))) < 1e-15
    # A15 holds for the final (u, p)
    assert abs(f.p - ref.pressure(14 / 15, N, f.ux, f.uy)) < 1e-15
    # Guo forcing: post-collision momentum = j + F/rho  (first moment of A1)
    assert abs((Ns * CX).sum() - (jx + f.Fx / f.rho)) < 1e-15
    assert abs((Ns * CY).sum() - (jy + f.Fy / f.rho)) < 1e-15
    # mixture rules and tau
    phi = nb[0]
    assert abs(f.rho - (1000 * phi + (1 - phi))) < 1e-12
    nu = 1 / (phi / 0.01 + (1 - phi) / 0.1)
    assert abs(f.tau - (0.5 + 3 * nu)) < 1e-15
    # first moment of the anti-diffusion term: sum c_i B_i* = phi (j + F/rho) + 2 M_phi(p) 4 phi(1-phi)/W n_phi / ...
    g = np.hypot(f.gradx, f.grady)
    nxh, nyh = f.gradx / g, f.grady / g
    Mphi = 0.5 * (3 * (1 - 14 / 15) / 5 + f.p)                 # PAPER.md:288 (c_s^2 dt/2 [..])
    fluxx = (Bs * CX).sum() - phi * (Ns * CX).sum()
    fluxy = (Bs * CY).sum() - phi * (Ns * CY).sum()
    assert abs(fluxx - Mphi * 4 * phi * (1 - phi) / 4.0 * nxh) < 1e-15   # Eq. 3 anti-diffusion flux
    assert abs(fluxy - Mphi * 4 * phi * (1 - phi) / 4.0 * nyh) < 1e-15


@pytest.mark.parametrize("k", range(6))
def test_generic_collision_equals_closed_form(k):
    """A1 with S = diag(1,..,1,s,s) and forcing without stress moments reduces to
    N* = N^eq + (1-s)(m7n M7 + m8n M8)/4 + F_i/2 — derived independently here."""
    prm = _params()
    N, nb = _random_node()
    Ns, Bs, f = ref.node_update(prm, N, nb)
    Neq = ref.neq(14 / 15, f.p, f.ux, f.uy)
    s = 1 / f.tau
    m7n = (N * (CX * CX - CY * CY)).sum() - (f.ux ** 2 - f.uy ** 2)
    m8n = (N * CX * CY).sum() - f.ux * f.uy
    Fi = 3 * W9 * (CX * f.Fx + CY * f.Fy) / f.rho
    closed = Neq + (1 - s) * (m7n * (CX * CX - CY * CY) + m8n * CX * CY) / 4 + Fi / 2
    assert np.allclose(Ns, closed, rtol=0, atol=5e-16)
    # and B* written out (A12)
    g = np.hypot(f.gradx, f.grady)
    Neq0 = ref.neq(14 / 15, f.p, 0, 0)
    Bc = nb[0] * closed + 2 * (CX * f.gradx + CY * f.grady) / g / 4.0 * nb[0] * (1 - nb[0]) * Neq0
    assert np.allclose(Bs, Bc, rtol=0, atol=5e-16)


def test_surface_tension_force_eq4():
    prm = _params(gx=0.0, gy=0.0)
    N, nb = _random_node()
    _, _, f = ref.node_update(prm, N, nb)
    phi = nb[0]
    mu = -0.01 * (48 / 4.0 * phi * (1 - phi) * (phi - 0.5) + 1.5 * 4.0 * f.lap)
    assert abs(f.Fsx - mu * f.gradx) < 1e-16 and abs(f.Fsy - mu * f.grady) < 1e-16


def test_picard_second_pass_changes_little():
    """R9: one Picard pass is the definition; a second pass moves u by << parity tolerance at the
    magnitudes the workloads see."""
    N, nb = _random_node(scale=1e-5)
    _, _, f1 = ref.node_update(_params(picard=1), N, nb)
    _, _, f2 = ref.node_update(_params(picard=2), N, nb)
    assert abs(f1.ux - f2.ux) < 1e-6 and abs(f1.uy - f2.uy) < 1e-6


def test_zero_gradient_drops_antidiffusion():
    prm = _params()
    N, _ = _random_node()
    nb = np.full(9, 0.3)
    Ns, Bs, f = ref.node_update(prm, N, nb)                     # R16
    assert f.gradx == 0 and f.grady == 0
    assert np.allclose(Bs, 0.3 * Ns, atol=1e-17)
