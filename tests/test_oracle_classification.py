"""Oracle pins, part 3: node classification against a brute-force scan on tiny
grids, and the ghost geometry against direct formulas."""
import math

import numpy as np
import pytest

from oracle import ref
from paper_2605_30878_b200 import workloads as wl


def brute_classes(mask):
    ny, nx = mask.shape
    out = np.zeros((ny, nx), np.uint8)
    for j in range(ny):
        for i in range(nx):
            other = False
            for dj in (-1, 0, 1):
                for di in (-1, 0, 1):
                    if di == 0 and dj == 0:
                        continue
                    if mask[(j + dj) % ny, (i + di) % nx] != mask[j, i]:
                        other = True
            out[j, i] = (2 if other else 3) if mask[j, i] else (1 if other else 0)
    return out


def _classify(mask, disks=None, wall_rows=0):
    ny, nx = mask.shape
    prm = ref.RefParams(nx=nx, ny=ny, wall_rows=wall_rows)
    return ref.RefLBM(prm, mask, disks).get_classification()


def _mask_cases():
    rng = np.random.default_rng(11)
    cases = {}
    cases["empty"] = np.zeros((8, 9), np.uint8)
    cases["full"] = np.ones((8, 9), np.uint8)
    m = np.zeros((9, 8), np.uint8); m[4, 3] = 1
    cases["single_node"] = m
    m = np.ones((9, 8), np.uint8); m[0, 0] = 0
    cases["single_fluid_corner"] = m
    yy, xx = np.mgrid[0:10, 0:12]
    cases["checkerboard"] = ((xx + yy) % 2).astype(np.uint8)
    cases["seam_disk"] = wl.rasterize_disks(32, 24, [[0.3, 23.6, 6.0]])
    for k in range(4):
        cases[f"random{k}"] = (rng.uniform(size=(8 + k, 13 - k)) < 0.3 + 0.1 * k).astype(np.uint8)
    return cases


@pytest.mark.parametrize("name", list(_mask_cases().keys()))
def test_classification_bruteforce(name):
    mask = _mask_cases()[name]
    # no geometry available for arbitrary masks: a disk big enough to own every ghost node
    ny, nx = mask.shape
    disks = [[nx / 2, ny / 2, 10 * (nx + ny)]]
    cl = _classify(mask, disks)
    assert np.array_equal(cl["cls"], brute_classes(mask))
    ghosts = np.flatnonzero(cl["cls"].ravel() == 2)
    assert np.array_equal(cl["idx"], ghosts)                    # index-sorted list
    assert cl["n_ghost"] == len(ghosts)


def test_ghost_geometry_disk():
    w = wl.config2(seed=5, theta_deg=60.0, n=64)
    cx, cy, R = w.disks[0]
    cl = _classify(w.mask, w.disks)
    i = cl["idx"] % w.nx; j = cl["idx"] // w.nx
    dx, dy = i - cx, j - cy
    dist = np.hypot(dx, dy)
    assert np.allclose(cl["nx"], dx / dist, atol=1e-15) and np.allclose(cl["ny"], dy / dist, atol=1e-15)
    assert np.allclose(cl["depth"], R - dist, atol=1e-13)
    assert (cl["depth"] >= 0).all() and (cl["depth"] < math.sqrt(2) + 1e-12).all()   # R15 remark
    # x_F = x_G + n_s lies at distance 1 from x_G, on the outward side
    xF, yF = i + cl["nx"], j + cl["ny"]
    assert np.allclose(np.hypot(xF - cx, yF - cy), dist + 1, atol=1e-12)
    # bilinear weights reproduce the coordinates of x_F (partition of unity + first moments)
    ci = cl["corner"] % w.nx; cj = cl["corner"] // w.nx
    assert np.allclose(cl["wgt"].sum(1), 1, atol=1e-15)
    assert np.allclose((cl["wgt"] * ci).sum(1), xF, atol=1e-12)
    assert np.allclose((cl["wgt"] * cj).sum(1), yF, atol=1e-12)


def test_ghost_geometry_seam_and_owner():
    # a disk across the periodic corner: minimum-image normals
    nx, ny = 32, 24
    disks = np.array([[0.3, 23.6, 6.0]])
    mask = wl.rasterize_disks(nx, ny, disks)
    cl = _classify(mask, disks)
    i = cl["idx"] % nx; j = cl["idx"] // nx
    dx = (i - 0.3 + nx / 2) % nx - nx / 2
    dy = (j - 23.6 + ny / 2) % ny - ny / 2
    assert np.allclose(cl["nx"], dx / np.hypot(dx, dy), atol=1e-15)
    assert np.allclose(cl["ny"], dy / np.hypot(dx, dy), atol=1e-15)
    # two overlapping disks: owner is the one with the least depth (R17)
    disks = np.array([[10.0, 12.0, 6.0], [14.0, 12.0, 3.0]])
    mask = wl.rasterize_disks(nx, ny, disks)
    cl = _classify(mask, disks)
    for g, k in enumerate(cl["idx"]):
        i, j = k % nx, k // nx
        deps = [r - math.hypot(i - cx, j - cy) for cx, cy, r in disks if math.hypot(i - cx, j - cy) <= r]
        assert cl["depth"][g] == pytest.approx(min(deps), abs=1e-13)


def test_wall_rows_geometry():
    nx, ny = 16, 10
    mask = np.zeros((ny, nx), np.uint8); mask[0] = 1; mask[-1] = 1
    cl = _classify(mask, None, wall_rows=1)
    assert cl["n_ghost"] == 2 * nx
    bot = cl["idx"] < nx
    assert (cl["nx"] == 0).all() and (cl["ny"][bot] == 1).all() and (cl["ny"][~bot] == -1).all()
    # x_F is the fluid node straight across the wall: weight 1 on it
    assert np.array_equal(cl["corner"][bot, 0], cl["idx"][bot] + nx)
    assert np.array_equal(cl["corner"][~bot, 0], cl["idx"][~bot] - nx)
    assert (cl["wgt"][:, 0] == 1).all() and (cl["wgt"][:, 1:] == 0).all()


def test_create_rejects_bad_input():
    mask = np.zeros((8, 8), np.uint8)
    with pytest.raises(ValueError):
        ref.RefLBM(ref.RefParams(nx=8, ny=8, W=3.0), mask)          # W >= 4
    with pytest.raises(ValueError):
        ref.RefLBM(ref.RefParams(nx=8, ny=8, nu_l=0.0), mask)       # tau > 1/2
    with pytest.raises(ValueError):
        ref.RefLBM(ref.RefParams(nx=8, ny=8, wall_rows=1), mask)    # wall rows must be solid
    m = mask.copy(); m[3, 3] = 1
    with pytest.raises(ValueError):                                 # a disk list that does not own the ghost node
        ref.RefLBM(ref.RefParams(nx=8, ny=8), m, np.array([[6.0, 6.0, 0.5]]))


# ---- NEXT row f2: solid normals from the mask alone ----------------------------------
def _mask_only(mask):
    ny, nx = mask.shape
    prm = ref.RefParams(nx=nx, ny=ny, rho_l=1.0, rho_g=1.0, nu_l=1 / 6, nu_g=1 / 6, sigma=0.01, W=4.0)
    return ref.RefLBM(prm, mask, np.zeros((0, 3))).get_classification()


def test_mask_only_normals_against_analytic_disk():
    """No disk list: n_s = -grad(s~)/|grad(s~)|, indicator smoothed twice, sixth-order isotropic stencil.
    On a rasterised disk of radius 40 the numeric normals follow the analytic ones (x_G - x_c)/|.|
    within 13 degrees (3.2 on average; the raw staircase would give 34 / 9.7), with zero mean bias."""
    from paper_2605_30878_b200 import workloads as wl
    n, cx, cy, R = 160, 80.3, 79.6, 40.0
    mask = wl.rasterize_disks(n, n, np.array([[cx, cy, R]]))
    c = _mask_only(mask)
    i, j = c["idx"] % n, c["idx"] // n
    ax, ay = i - cx, j - cy
    an = np.hypot(ax, ay)
    dot = (c["nx"] * ax + c["ny"] * ay) / an
    cross = (c["nx"] * ay - c["ny"] * ax) / an
    ang = np.degrees(np.arctan2(cross, dot))
    assert np.allclose(np.hypot(c["nx"], c["ny"]), 1.0, atol=1e-15)
    assert np.abs(ang).max() < 13.5 and np.abs(ang).mean() < 3.3 and abs(ang.mean()) < 0.1
    assert np.all(c["depth"] == 0.0)


def test_mask_only_normals_flat_wall_and_symmetry():
    """A straight wall gives exactly (0, +-1); mirroring the mask mirrors the normals bit for bit."""
    mask = np.zeros((24, 16), np.uint8)
    mask[:3, :] = 1
    mask[-2:, :] = 1
    c = _mask_only(mask)
    j = c["idx"] // 16
    assert np.all(c["nx"] == 0.0) and np.all(c["ny"][j < 12] == 1.0) and np.all(c["ny"][j > 12] == -1.0)
    rng = np.random.default_rng(3)
    blob = (rng.random((20, 28)) < 0.35).astype(np.uint8)
    a, b = _mask_only(blob), _mask_only(blob[:, ::-1].copy())
    na = {(k // 28, k % 28): (x, y) for k, x, y in zip(a["idx"], a["nx"], a["ny"])}
    nb = {(k // 28, 27 - k % 28): (-x, y) for k, x, y in zip(b["idx"], b["nx"], b["ny"])}
    assert na.keys() == nb.keys() and all(na[k] == nb[k] for k in na)
