"""Seeded synthetic input generators for the five BASELINE.json configs.

This module serves BOTH the CUDA path and the CPU oracle (tests hand the same arrays to each).
It holds none of the method's arithmetic: it only builds inputs — the solid mask, the analytic
disk list, the initial order parameter phi0 and the physical parameters.  numpy only; it imports
neither ``oracle`` nor the CUDA binding.

Stand-ins: the paper measures on its own four set-ups (§III.A-D), not on a public
dataset; the configs below take their shapes from §III.B (drop on a cylinder)
and BASELINE.json.  Recipes are stated in DESIGN.md "Input recipe".

Conventions: node (i, j) at (x, y) = (i, j); arrays are [ny, nx] (x fastest); periodic box;
closed disks (d^2 <= r^2) with minimum-image distance; phi = 1 liquid, 0 gas;
phi0 of a liquid drop of radius R: 1/2 [1 - tanh(2 (r - R) / W)] (Eq. 5).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

MU_G = 0.1    # PAPER.md:100 default gas dynamic viscosity
RHO_G = 1.0   # PAPER.md:100 default gas density


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    mask: np.ndarray            # uint8 [ny, nx], 1 = solid
    disks: np.ndarray           # float64 [n_disks, 3] (cx, cy, r)
    phi0: np.ndarray            # float64 [ny, nx]
    rho_l: float
    rho_g: float
    nu_l: float
    nu_g: float
    sigma: float
    W: float
    theta_deg: float
    mobility: float = 0.02
    gx: float = 0.0
    gy: float = 0.0
    wall_rows: int = 0
    steps: int = 0              # the run length BASELINE.json names
    seed: int = 0
    meta: dict = field(default_factory=dict)

    def param_dict(self) -> dict:
        return dict(nx=self.nx, ny=self.ny, rho_l=self.rho_l, rho_g=self.rho_g, nu_l=self.nu_l,
                    nu_g=self.nu_g, sigma=self.sigma, W=self.W, theta_deg=self.theta_deg,
                    mobility=self.mobility, gx=self.gx, gy=self.gy, wall_rows=self.wall_rows)


# ---- helpers ------------------------------------------------------------------------------
def viscosities(rho_ratio: float, mu_ratio: float):
    """(nu_l, nu_g) from the paper's dynamic-viscosity ratio with rho_g = 1, mu_g = 0.1."""
    nu_g = MU_G / RHO_G
    nu_l = MU_G * mu_ratio / (RHO_G * rho_ratio)
    return nu_l, nu_g


def _window(c: float, half: float, n: int):
    lo = int(math.floor(c - half)) - 1
    hi = int(math.ceil(c + half)) + 1
    if hi - lo + 1 >= n:
        return np.arange(n), np.arange(n)
    raw = np.arange(lo, hi + 1)
    return raw % n, raw


def _minimg(d, L):
    d = np.mod(d, L)
    return np.where(d >= 0.5 * L, d - L, d)


def rasterize_disks(nx: int, ny: int, disks) -> np.ndarray:
    """uint8 mask, 1 inside the closed disks (minimum-image distance^2 <= r^2)."""
    mask = np.zeros((ny, nx), np.uint8)
    for cx, cy, r in np.asarray(disks, dtype=np.float64).reshape(-1, 3):
        ii, _ = _window(cx, r, nx)
        jj, _ = _window(cy, r, ny)
        dx = _minimg(ii.astype(np.float64) - cx, float(nx))
        dy = _minimg(jj.astype(np.float64) - cy, float(ny))
        inside = (dy[:, None] ** 2 + dx[None, :] ** 2) <= r * r
        sub = mask[np.ix_(jj, ii)]
        sub[inside] = 1
        mask[np.ix_(jj, ii)] = sub
    return mask


def drop_profile(nx: int, ny: int, cx: float, cy: float, R: float, W: float, out=None, reach=None):
    """max(out, 1/2[1 - tanh(2(r - R)/W)]) for a liquid drop centred at (cx, cy), periodic."""
    if out is None:
        out = np.zeros((ny, nx))
    half = R + (8.0 * W if reach is None else reach)
    ii, _ = _window(cx, half, nx)
    jj, _ = _window(cy, half, ny)
    dx = _minimg(ii.astype(np.float64) - cx, float(nx))
    dy = _minimg(jj.astype(np.float64) - cy, float(ny))
    r = np.sqrt(dy[:, None] ** 2 + dx[None, :] ** 2)
    prof = 0.5 * (1.0 - np.tanh(2.0 * (r - R) / W))
    sub = out[np.ix_(jj, ii)]
    np.maximum(sub, prof, out=sub)
    out[np.ix_(jj, ii)] = sub
    return out


def drop_distance(R: float, Rc: float, theta_deg: float) -> float:
    """Centre distance of two circles meeting at contact angle theta (law of cosines)."""
    return math.sqrt(R * R + Rc * Rc - 2.0 * R * Rc * math.cos(math.radians(theta_deg)))


# ---- config 1: static droplet on a cylinder, 64^2 -------------------------------------------
def config1(seed: int = 0, jitter: bool = True) -> Workload:
    nx = ny = 64
    rng = np.random.default_rng(seed)
    jit = rng.uniform(-0.5, 0.5, 2) if jitter else np.zeros(2)
    disks = np.array([[32.0, 20.0, 12.0]])
    W = 4.0
    phi0 = drop_profile(nx, ny, 32.0 + jit[0], 36.0 + jit[1], 10.0, W)
    nu = (1.0 - 0.5) / 3.0          # tau = 1 in both phases
    return Workload("config1_drop_on_cylinder_64", nx, ny, rasterize_disks(nx, ny, disks), disks, phi0,
                    rho_l=1.0, rho_g=1.0, nu_l=nu, nu_g=nu, sigma=0.01, W=W, theta_deg=60.0,
                    steps=1000, seed=seed, meta=dict(drop=(32.0 + jit[0], 36.0 + jit[1], 10.0)))


# ---- config 2: contact-angle sweep on a cylinder, 256^2 -------------------------------------
def config2(seed: int = 0, theta_deg: float = 60.0, n: int = 256) -> Workload:
    s = n / 256.0
    rng = np.random.default_rng(seed)
    off = rng.uniform(0.0, 1.0, 2)
    R, Rc, W = 40.0 * s, 35.0 * s, 5.0
    cx, cy = n / 2.0 + off[0], n / 4.0 + off[1]
    disks = np.array([[cx, cy, R]])
    d = drop_distance(R, Rc, theta_deg)
    phi0 = drop_profile(n, n, cx, cy + d, Rc, W)
    nu_l, nu_g = viscosities(10.0, 10.0)
    return Workload(f"config2_contact_angle_{n}_theta{theta_deg:g}", n, n, rasterize_disks(n, n, disks),
                    disks, phi0, rho_l=10.0, rho_g=1.0, nu_l=nu_l, nu_g=nu_g, sigma=0.005, W=W,
                    theta_deg=theta_deg, steps=20000, seed=seed,
                    meta=dict(drop=(cx, cy + d, Rc), disk=(cx, cy, R)))


# ---- config 3: high-contrast static droplet, 1024^2 -----------------------------------------
def config3(seed: int = 0, n: int = 1024) -> Workload:
    s = n / 1024.0
    R, Rc, W, theta = 160.0 * s, 140.0 * s, 4.0, 45.0
    cx, cy = n / 2.0, n / 4.0
    disks = np.array([[cx, cy, R]])
    d = drop_distance(R, Rc, theta)
    phi0 = drop_profile(n, n, cx, cy + d, Rc, W)
    nu_l, nu_g = viscosities(1000.0, 100.0)
    return Workload(f"config3_high_contrast_{n}", n, n, rasterize_disks(n, n, disks), disks, phi0,
                    rho_l=1000.0, rho_g=1.0, nu_l=nu_l, nu_g=nu_g, sigma=0.001, W=W, theta_deg=theta,
                    steps=50000, seed=seed, meta=dict(drop=(cx, cy + d, Rc), disk=(cx, cy, R)))


# ---- config 4: dynamic contact line in a channel with posts, 2048x512 -----------------------
def config4(seed: int = 0, nx: int = 2048, ny: int = 512) -> Workload:
    rng = np.random.default_rng(seed)
    W = 4.0
    pitch = nx / 8.0
    jit = rng.uniform(-pitch / 4.0, pitch / 4.0, 8)
    disks = np.array([[(k + 0.5) * pitch + jit[k], ny / 2.0, 24.0 * ny / 512.0] for k in range(8)])
    mask = rasterize_disks(nx, ny, disks)
    mask[0, :] = 1
    mask[ny - 1, :] = 1
    x = np.arange(nx, dtype=np.float64)
    sdist = np.abs(_minimg(x - 0.2 * nx, float(nx)))       # periodic distance in x to 0.2 nx
    prof = 0.5 * (1.0 - np.tanh(2.0 * (sdist - 0.2 * nx) / W))
    phi0 = np.repeat(prof[None, :], ny, axis=0)
    nu_l, nu_g = viscosities(100.0, 10.0)
    return Workload(f"config4_channel_{nx}x{ny}", nx, ny, mask, disks, phi0, rho_l=100.0, rho_g=1.0,
                    nu_l=nu_l, nu_g=nu_g, sigma=0.01, W=W, theta_deg=70.0, gx=1e-7, wall_rows=1,
                    steps=100000, seed=seed)


# ---- config 5: porous medium throughput sweep -----------------------------------------------
def _rsa_disks(n: int, rng, solid_fraction: float, rmin: float, rmax: float, gap: float):
    """Random sequential insertion of non-overlapping disks (surfaces >= gap apart, min image)."""
    cell = 2.0 * rmax + gap
    nc = max(1, int(n // cell))
    cs = n / nc
    grid: dict[tuple[int, int], list[int]] = {}
    disks: list[tuple[float, float, float]] = []
    area, target = 0.0, solid_fraction * n * n
    attempts = 0
    while area < target and attempts < 200 * max(1, int(target / (math.pi * rmin * rmin))):
        attempts += 1
        cx, cy = rng.uniform(0.0, n, 2)
        r = rng.uniform(rmin, rmax)
        gi, gj = int(cx / cs) % nc, int(cy / cs) % nc
        ok = True
        for dj in (-1, 0, 1):
            for di in (-1, 0, 1):
                for k in grid.get(((gi + di) % nc, (gj + dj) % nc), ()):
                    ox, oy, orr = disks[k]
                    dx = (cx - ox + 0.5 * n) % n - 0.5 * n
                    dy = (cy - oy + 0.5 * n) % n - 0.5 * n
                    if dx * dx + dy * dy < (r + orr + gap) ** 2:
                        ok = False
                        break
                if not ok:
                    break
            if not ok:
                break
        if ok:
            grid.setdefault((gi, gj), []).append(len(disks))
            disks.append((cx, cy, r))
            area += math.pi * r * r
    return np.array(disks, dtype=np.float64).reshape(-1, 3)


def config5(seed: int = 0, n: int = 2048, solid_fraction: float = 0.35) -> Workload:
    rng = np.random.default_rng(seed)
    W = 4.0
    disks = _rsa_disks(n, rng, solid_fraction, 8.0, 32.0, 4.0)
    mask = rasterize_disks(n, n, disks)
    fluid = mask == 0
    n_fluid = int(fluid.sum())
    phi0 = np.zeros((n, n))
    filled, n_blobs = 0.0, 0
    while filled < 0.5 * n_fluid:
        cx, cy = rng.uniform(0.0, n, 2)
        R = rng.uniform(16.0, 64.0)
        half = R + 4.0 * W
        ii, _ = _window(cx, half, n)
        jj, _ = _window(cy, half, n)
        dx = _minimg(ii.astype(np.float64) - cx, float(n))
        dy = _minimg(jj.astype(np.float64) - cy, float(n))
        r = np.sqrt(dy[:, None] ** 2 + dx[None, :] ** 2)
        prof = 0.5 * (1.0 - np.tanh(2.0 * (r - R) / W))
        sub = phi0[np.ix_(jj, ii)]
        new = np.maximum(sub, prof)
        filled += float(((new - sub) * fluid[np.ix_(jj, ii)]).sum())
        phi0[np.ix_(jj, ii)] = new
        n_blobs += 1
    nu_l, nu_g = viscosities(1000.0, 100.0)
    return Workload(f"config5_porous_{n}", n, n, mask, disks, phi0, rho_l=1000.0, rho_g=1.0, nu_l=nu_l,
                    nu_g=nu_g, sigma=0.01, W=W, theta_deg=110.0, steps=2000, seed=seed,
                    meta=dict(n_disks=len(disks), n_blobs=n_blobs, n_fluid=n_fluid,
                              porosity=n_fluid / float(n * n)))


# ---- small extras used by tests --------------------------------------------------------------
def free_droplet(n: int, R: float, W: float = 4.0):
    """A liquid drop in a fully periodic box without solids (Laplace-law pin)."""
    return np.zeros((n, n), np.uint8), np.zeros((0, 3)), drop_profile(n, n, n / 2.0, n / 2.0, R, W)


def flat_interface(nx: int, ny: int, W: float = 4.0):
    """Periodic strip: liquid for ny/4 < y < 3ny/4, two flat tanh interfaces (Eq. 5)."""
    y = np.arange(ny, dtype=np.float64)
    prof = 0.5 * (np.tanh(2.0 * (y - 0.25 * ny) / W) - np.tanh(2.0 * (y - 0.75 * ny) / W))
    return np.zeros((ny, nx), np.uint8), np.zeros((0, 3)), np.repeat(prof[:, None], nx, axis=1)


# ---- the paper's own drop-on-a-cylinder set-up (§III.B, :128-134) ------------------------------
def _lens_area(R: float, Rc: float, d: float) -> float:
    """Area common to two circles of radii R, Rc whose centres are d apart (textbook formula)."""
    if d >= R + Rc:
        return 0.0
    if d <= abs(R - Rc):
        return math.pi * min(R, Rc) ** 2
    a = R * R * math.acos((d * d + R * R - Rc * Rc) / (2.0 * d * R))
    b = Rc * Rc * math.acos((d * d + Rc * Rc - R * R) / (2.0 * d * Rc))
    c = 0.5 * math.sqrt((-d + R + Rc) * (d + R - Rc) * (d - R + Rc) * (d + R + Rc))
    return a + b - c


def drop_on_cylinder_paper(theta_deg: float = 30.0, R: float = 40.0, A: float = 3000.0, W: float = 4.0,
                           rho_ratio: float = 1000.0, mu_ratio: float = 100.0, sigma: float = 1e-2,
                           x_offset: float = 0.0) -> Workload:
    """(5R, 5R) periodic box, cylinder of radius R at (Lx/2, Ly/4), liquid of area A initialised as the circular
    cap that meets the cylinder at the prescribed angle ("we initialize the drop with the expected equilibrium
    configuration"): R_c from {pi R_c^2 - lens(R, R_c, d) = A, d^2 = R^2 + R_c^2 - 2 R R_c cos(theta)}."""
    n = int(round(5.0 * R))
    ct = math.cos(math.radians(theta_deg))
    lo, hi = 1e-6, 100.0 * math.sqrt(A)
    for _ in range(200):                       # bisection on R_c: the liquid area grows with it
        Rc = 0.5 * (lo + hi)
        d = math.sqrt(R * R + Rc * Rc - 2.0 * R * Rc * ct)
        if math.pi * Rc * Rc - _lens_area(R, Rc, d) < A:
            lo = Rc
        else:
            hi = Rc
    cx, cy = 0.5 * n + x_offset, 0.25 * n
    disks = np.array([[cx, cy, R]])
    phi0 = drop_profile(n, n, cx, cy + d, Rc, W)
    nu_l, nu_g = viscosities(rho_ratio, mu_ratio)
    w = Workload(f"drop_on_cylinder_paper_{n}_theta{theta_deg:g}", n, n, rasterize_disks(n, n, disks), disks, phi0,
                 rho_l=rho_ratio * RHO_G, rho_g=RHO_G, nu_l=nu_l, nu_g=nu_g, sigma=sigma, W=W,
                 theta_deg=theta_deg, steps=20000, seed=0)
    w.meta.update(Rc=Rc, d=d, hmax=d + Rc, area=A, R=R)
    return w


# ---- NEXT row f3: drop on a flat plate (§III.A, :102-124) -----------------------------------
def flat_plate(theta_deg: float = 60.0, W: float = 4.0, scale: float = 1.0, rho_ratio: float = 1000.0,
               mu_ratio: float = 100.0, sigma: float = 1e-2, x_offset: float = 0.0) -> Workload:
    """Drop of area A = 1e4 scale^2 on the bottom wall of a (500, 300) scale box, periodic in x, wall rows
    at j = 0 and j = ny-1 (+2 wall rows as in the paper's Table I grids).  The drop starts
    as the analytic circular cap of the prescribed angle (:114): R_c = sqrt(2A / (2 theta - sin 2 theta)),
    centre at height -R_c cos(theta) relative to the wall surface, which lies half-way between the wall row
    and the first fluid row (R12, R17).  x_offset shifts the drop off the lattice symmetry axis: on a mirror-symmetric
    set-up grad(phi) cancels to round-off at the centre of curvature, where the direction of n_phi (R16) is
    then decided by rounding order, so element-wise parity runs use an offset."""
    nx = int(round(500 * scale))
    nx += nx & 1
    ny = int(round(300 * scale)) + 2
    A = 1.0e4 * scale * scale
    th = math.radians(theta_deg)
    Rc = math.sqrt(2.0 * A / (2.0 * th - math.sin(2.0 * th)))
    y_wall = 0.5
    cx, cy = 0.5 * nx + x_offset, y_wall - Rc * math.cos(th)
    mask = np.zeros((ny, nx), dtype=np.uint8)
    mask[0, :] = 1
    mask[ny - 1, :] = 1
    yy, xx = np.mgrid[0:ny, 0:nx].astype(np.float64)
    r = np.hypot(xx - cx, yy - cy)
    phi0 = 0.5 * (1.0 - np.tanh(2.0 * (r - Rc) / W))
    nu_l, nu_g = viscosities(rho_ratio, mu_ratio)
    w = Workload(f"flat_plate_{nx}x{ny}_theta{theta_deg:g}_W{W:g}", nx, ny, mask, np.zeros((0, 3)), phi0,
                 rho_l=rho_ratio * RHO_G, rho_g=RHO_G, nu_l=nu_l, nu_g=nu_g, sigma=sigma, W=W,
                 theta_deg=theta_deg, wall_rows=1, steps=20000, seed=0)
    w.meta.update(area=A, Rc=Rc, y_wall=y_wall)
    return w


def particle_at_interface(theta_deg: float = 60.0, R: float = 25.0, W: float = 4.0, rho_ratio: float = 10.0,
                          mu_ratio: float = 10.0, sigma: float = 1e-2, x_offset: float = 0.0) -> Workload:
    """Fixed cylinder of radius R at a flat liquid-gas interface (§III.C, :136-197): box
    (4.8 R, 4.8 R), periodic in x, no-slip walls at top and bottom (+2 wall rows, cf. the 120 x 122 grid of
    Table I), cylinder centred in the box, liquid below the line through its centre."""
    L = int(round(4.8 * R))
    L += L & 1
    nx, ny = L, L + 2
    y_wall = 0.5
    cx, cy = 0.5 * nx + x_offset, y_wall + 0.5 * L     # x_offset: off the mirror axis for parity runs (R16)
    disks = np.array([[cx, cy, R]])
    mask = rasterize_disks(nx, ny, disks)
    mask[0, :] = 1
    mask[ny - 1, :] = 1
    yy = np.arange(ny, dtype=np.float64)[:, None] + np.zeros((1, nx))
    phi0 = 0.5 * (1.0 - np.tanh(2.0 * (yy - cy) / W))
    nu_l, nu_g = viscosities(rho_ratio, mu_ratio)
    w = Workload(f"particle_at_interface_{nx}x{ny}_theta{theta_deg:g}", nx, ny, mask, disks, phi0,
                 rho_l=rho_ratio * RHO_G, rho_g=RHO_G, nu_l=nu_l, nu_g=nu_g, sigma=sigma, W=W,
                 theta_deg=theta_deg, wall_rows=1, steps=40000, seed=0)
    w.meta.update(L=float(L), R=R, y_interface0=cy)
    return w
