"""Measurement helpers shared by the oracle pins and the GPU parity tests (no method arithmetic).

Contact angle of a drop on a cylinder (§III.B :128-134, Eq. 7 :58): fit a circle to the
phi = 1/2 contour away from the solid, then theta_m = arccos[(R^2 + Rc^2 - d^2) / (2 R Rc)] from
n_s . n_phi = -cos(theta) at the intersection of the two circles (law of cosines).
"""
from __future__ import annotations

import math

import numpy as np


def half_contour_points(phi: np.ndarray, mask: np.ndarray, level: float = 0.5):
    """Sub-cell crossings of phi = level along grid lines between adjacent FLUID nodes (no wrap)."""
    ny, nx = phi.shape
    f = phi - level
    fl = mask == 0
    pts = []
    # x-direction edges
    a, b = f[:, :-1], f[:, 1:]
    ok = fl[:, :-1] & fl[:, 1:] & ((a < 0) != (b < 0))
    jj, ii = np.nonzero(ok)
    t = a[jj, ii] / (a[jj, ii] - b[jj, ii])
    pts.append(np.stack([ii + t, jj.astype(float)], axis=1))
    # y-direction edges
    a, b = f[:-1, :], f[1:, :]
    ok = fl[:-1, :] & fl[1:, :] & ((a < 0) != (b < 0))
    jj, ii = np.nonzero(ok)
    t = a[jj, ii] / (a[jj, ii] - b[jj, ii])
    pts.append(np.stack([ii.astype(float), jj + t], axis=1))
    return np.concatenate(pts, axis=0)


def fit_circle(pts: np.ndarray):
    """Least-squares circle: algebraic (Kasa) start, then Gauss-Newton on geometric distance."""
    x, y = pts[:, 0], pts[:, 1]
    A = np.stack([2 * x, 2 * y, np.ones_like(x)], axis=1)
    sol, *_ = np.linalg.lstsq(A, x * x + y * y, rcond=None)
    cx, cy = sol[0], sol[1]
    r = math.sqrt(sol[2] + cx * cx + cy * cy)
    for _ in range(50):
        dx, dy = x - cx, y - cy
        d = np.sqrt(dx * dx + dy * dy)
        res = d - r
        J = np.stack([-dx / d, -dy / d, -np.ones_like(d)], axis=1)
        step, *_ = np.linalg.lstsq(J, -res, rcond=None)
        cx, cy, r = cx + step[0], cy + step[1], r + step[2]
        if np.abs(step).max() < 1e-13:
            break
    return cx, cy, r


def contact_angle_on_cylinder(phi: np.ndarray, mask: np.ndarray, disk, W: float, exclude: float = 2.0):
    """(theta_m in degrees, Rc, d, h_max) for a drop sitting on the disk (cx, cy, R)."""
    cx, cy, R = disk
    pts = half_contour_points(phi, mask)
    dist = np.hypot(pts[:, 0] - cx, pts[:, 1] - cy)
    pts = pts[dist > R + exclude * W]
    if len(pts) < 8:
        raise ValueError("too few contour points")
    dcx, dcy, Rc = fit_circle(pts)
    d = math.hypot(dcx - cx, dcy - cy)
    cosang = (R * R + Rc * Rc - d * d) / (2.0 * R * Rc)
    theta = math.degrees(math.acos(max(-1.0, min(1.0, cosang))))
    return theta, Rc, d, d + Rc


def lens_area(R: float, Rc: float, d: float) -> float:
    """Textbook area of the intersection of two circles of radii R, Rc at centre distance d."""
    if d >= R + Rc:
        return 0.0
    if d <= abs(R - Rc):
        return math.pi * min(R, Rc) ** 2
    a = R * R * math.acos((d * d + R * R - Rc * Rc) / (2 * d * R))
    b = Rc * Rc * math.acos((d * d + Rc * Rc - R * R) / (2 * d * Rc))
    c = 0.5 * math.sqrt((-d + R + Rc) * (d + R - Rc) * (d - R + Rc) * (d + R + Rc))
    return a + b - c


def analytic_drop_on_cylinder(R: float, A: float, theta_deg: float):
    """Solve {pi Rc^2 - lens(R, Rc, d) = A, cos(theta) = (R^2 + Rc^2 - d^2)/(2 R Rc)} by bisection
    on Rc; returns (Rc, d, h_max = d + Rc).  PAPER.md:130 "can be found analytically"."""
    ct = math.cos(math.radians(theta_deg))

    def area(Rc):
        d = math.sqrt(R * R + Rc * Rc - 2 * R * Rc * ct)
        return math.pi * Rc * Rc - lens_area(R, Rc, d)

    lo, hi = 1e-6, 100.0 * math.sqrt(A)
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if area(mid) < A:
            lo = mid
        else:
            hi = mid
    Rc = 0.5 * (lo + hi)
    d = math.sqrt(R * R + Rc * Rc - 2 * R * Rc * ct)
    return Rc, d, d + Rc


def contact_angle_on_plate(phi: np.ndarray, mask: np.ndarray, W: float, y_wall: float = 0.5, exclude: float = 2.0):
    """(theta_m in degrees, spread S, height H) of a drop on the bottom wall, Eq. 12 (:118):
    theta_m = arccos((S^2 - H^2) / (S^2 + H^2)) with S the HALF spread on the wall and H the apex height.
    S and H come from the circle fitted to the phi = 1/2 contour farther than `exclude` W from the wall
    (the diffuse profile is distorted next to the wall), evaluated on the wall surface y_wall."""
    pts = half_contour_points(phi, mask)
    pts = pts[pts[:, 1] > y_wall + exclude * W]
    if len(pts) < 8:
        raise ValueError("too few contour points")
    cx, cy, Rc = fit_circle(pts)
    h = cy - y_wall                       # centre height above the wall (negative for theta < 90)
    H = h + Rc
    S = math.sqrt(max(Rc * Rc - h * h, 0.0))
    theta = math.degrees(math.acos((S * S - H * H) / (S * S + H * H)))
    return theta, S, H


def eq13_hstar(L: float, R: float, theta_deg: float):
    """PAPER.md Eq. 13 (:180-189): periodic array of fixed cylinders at an interface.  Unknowns R_c, psi,
    beta from  R^2 (L/R sin b - sin b cos b - b) = R_c^2 (psi - sin psi cos psi),
    2 R_c cos(b + theta) = L - 2 R cos b,  psi = pi/2 - (b + theta);  returns
    (h* = R_c (1 - cos psi) - R sin b, R_c, psi, beta).  theta > 90 deg follows from exchanging the two
    phases: h*(theta) = -h*(180 - theta); theta = 90 deg: flat interface, h* = 0."""
    if abs(theta_deg - 90.0) < 1e-12:
        return 0.0, math.inf, 0.0, 0.0
    if theta_deg > 90.0:
        h, Rc, psi, beta = eq13_hstar(L, R, 180.0 - theta_deg)
        return -h, Rc, psi, beta
    th = math.radians(theta_deg)

    def resid(b):
        psi = 0.5 * math.pi - (b + th)
        Rc = (L - 2.0 * R * math.cos(b)) / (2.0 * math.cos(b + th))
        return R * R * (L / R * math.sin(b) - math.sin(b) * math.cos(b) - b) - Rc * Rc * (psi - math.sin(psi) * math.cos(psi))

    lo, hi = 1e-9, 0.5 * math.pi - th - 1e-9        # resid(lo) < 0 (no area displaced), resid(hi) > 0 (psi -> 0)
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if resid(mid) < 0.0:
            lo = mid
        else:
            hi = mid
    b = 0.5 * (lo + hi)
    psi = 0.5 * math.pi - (b + th)
    Rc = (L - 2.0 * R * math.cos(b)) / (2.0 * math.cos(b + th))
    return Rc * (1.0 - math.cos(psi)) - R * math.sin(b), Rc, psi, b


def interface_height_at_boundary(phi: np.ndarray, level: float = 0.5) -> float:
    """y of the phi = level crossing along the periodic boundary column x = 0 (linear interpolation,
    liquid below), the quantity h* of PAPER.md §III.C is measured from."""
    col = phi[:, 0]
    j = np.nonzero((col[:-1] >= level) & (col[1:] < level))[0]
    j = j[len(j) // 2] if len(j) > 1 else j[0]
    return float(j + (col[j] - level) / (col[j] - col[j + 1]))
