"""GPU parity tests proper: the CUDA path (through the C ABI) against the CPU oracle, element by
element on the same seeded inputs.  Tolerances: classification and ghost
geometry bit-exact; fp64 fields and populations <= 1e-10 absolute after 1,000 steps (north_star);
fp32 <= 2e-4 relative to field scale against the fp64 oracle."""
import math

import numpy as np
import pytest

import _measure as ms
from _parity import ArrayWorkload, field_errors, make_pair, pop_errors
from paper_2605_30878_b200 import workloads as wl

pytestmark = pytest.mark.gpu

BASELINE, FUSED, PAIR, PACK, SPARSE, INPLACE = 1, 2, 4, 5, 6, 7
SCHEDULES = [pytest.param(BASELINE, id="baseline"), pytest.param(FUSED, id="fused"),
             pytest.param(PAIR, id="pair"), pytest.param(PACK, id="pack"), pytest.param(SPARSE, id="sparse"),
             pytest.param(INPLACE, id="inplace")]


# ---- local update of single nodes ---------------------------------------------------------------
def _random_nodes(count, seed):
    from oracle import ref
    rng = np.random.default_rng(seed)
    chi = ref.chi(14 / 15)
    N = chi[None, :] + rng.normal(0, 1e-3, (count, 9))
    base = rng.uniform(0, 1, (count, 1))
    nb = np.clip(base + rng.normal(0, 0.05, (count, 9)), -0.01, 1.01)
    nb[:4] = [[0] * 9, [1] * 9, [0.5] * 9, [0.3] * 9]           # uniform phi: zero gradient (R16)
    return N, nb


@pytest.mark.parametrize("prm", [dict(rho_l=1.0, nu_l=1 / 6, nu_g=1 / 6), dict(rho_l=1000.0, nu_l=0.01, nu_g=0.1),
                                 dict(rho_l=100.0, nu_l=0.01, nu_g=0.1, gx=1e-5, gy=-2e-5, W=5.0, sigma=0.02)])
def test_node_update_fp64(prm):
    from oracle import ref
    from paper_2605_30878_b200 import binding
    N, nb = _random_nodes(300, 3)
    Ns, Bs, F = binding.node_update_batch(binding.LBMParams(nx=8, ny=8, precision=64, **prm), N, nb)
    rp = ref.RefParams(nx=8, ny=8, **prm)
    worst = 0.0
    for k in range(N.shape[0]):
        oN, oB, f = ref.node_update(rp, N[k], nb[k])
        worst = max(worst, np.abs(Ns[k] - oN).max(), np.abs(Bs[k] - oB).max())
        assert abs(F["ux"][k] - f.ux) < 1e-14 and abs(F["uy"][k] - f.uy) < 1e-14
        assert abs(F["p"][k] - f.p) < 1e-14 and abs(F["rho"][k] - f.rho) < 1e-11
        assert abs(F["tau"][k] - f.tau) < 1e-13
        assert abs(F["Fx"][k] - f.Fx) < 1e-13 * max(1.0, prm["rho_l"])
    assert worst < 5e-15, worst


def test_node_update_fp32():
    from oracle import ref
    from paper_2605_30878_b200 import binding
    prm = dict(rho_l=1000.0, nu_l=0.01, nu_g=0.1)
    N, nb = _random_nodes(200, 4)
    Ns, Bs, F = binding.node_update_batch(binding.LBMParams(nx=8, ny=8, precision=32, **prm), N, nb)
    rp = ref.RefParams(nx=8, ny=8, **prm)
    for k in range(N.shape[0]):
        oN, oB, f = ref.node_update(rp, N[k], nb[k])
        assert np.abs(Ns[k] - oN).max() < 2e-6      # deviations ~1e-3 carried in fp32, phi in fp32
        assert np.abs(Bs[k] - oB).max() < 2e-6
        assert abs(F["p"][k] - f.p) < 2e-6


# ---- classification and ghost geometry: bit-exact ------------------------------------------------
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
    cases["random_big"] = (rng.uniform(size=(37, 300)) < 0.3).astype(np.uint8)   # several 256-blocks, ragged
    return cases


def _assert_same_classification(a, b):
    assert np.array_equal(a["cls"], b["cls"])
    assert a["n_ghost"] == b["n_ghost"]
    assert np.array_equal(a["idx"], b["idx"])
    assert np.array_equal(a["corner"], b["corner"])
    for k in ("nx", "ny", "depth", "wgt"):
        assert np.array_equal(a[k], b[k]), k            # fp64 geometry without contraction: bit-exact


@pytest.mark.parametrize("name", list(_mask_cases().keys()))
def test_classification_masks_bit_exact(name):
    mask = _mask_cases()[name]
    ny, nx = mask.shape
    w = ArrayWorkload(mask, np.zeros((ny, nx)), disks=[[nx / 2, ny / 2, 10 * (nx + ny)]])
    g, o = make_pair(w)
    _assert_same_classification(g.get_classification(), o.get_classification())


@pytest.mark.parametrize("make", [lambda: wl.config1(seed=1), lambda: wl.config2(seed=3, theta_deg=120.0),
                                  lambda: wl.config4(seed=2, nx=512, ny=128), lambda: wl.config5(seed=1, n=512)],
                         ids=["config1", "config2", "config4_small", "config5_512"])
def test_classification_configs_bit_exact(make):
    w = make()
    g, o = make_pair(w, precision=32)          # geometry is fp64 in both precisions
    _assert_same_classification(g.get_classification(), o.get_classification())


# ---- one call of each kernel ---------------------------------------------------------------------
@pytest.mark.parametrize("schedule", SCHEDULES)
def test_init_and_first_ghost_update(schedule):
    w = wl.config1(seed=2)
    g, o = make_pair(w, schedule=schedule)
    g.keep_B(True)                                      # B_i are not part of the stored state (compacted layouts: no B planes at all)
    g.init(w.phi0); o.init(w.phi0)
    fluid = w.mask == 0
    eN, eB = pop_errors(g, o, fluid)
    assert eN < 1e-16 and eB < 1e-16
    err, _ = field_errors(g, o)
    assert err["phi"] < 1e-15, err            # includes the ghost values of Eq. 9
    assert max(err["ux"], err["uy"], err["p"]) < 1e-15 and err["rho"] < 1e-13


def test_init_with_velocity():
    w = wl.config2(seed=1, theta_deg=60.0, n=64)
    rng = np.random.default_rng(0)
    u0 = rng.normal(0, 1e-3, (2, w.ny, w.nx))
    g, o = make_pair(w, schedule=BASELINE)
    g.init(w.phi0, u0); o.init(w.phi0, u0)
    eN, eB = pop_errors(g, o, w.mask == 0)
    assert eN < 1e-16 and eB < 1e-16


@pytest.mark.parametrize("schedule", SCHEDULES)
@pytest.mark.parametrize("steps", [1, 2, 7])
def test_few_steps_config1(schedule, steps):
    w = wl.config1(seed=0)
    g, o = make_pair(w, schedule=schedule)
    g.init(w.phi0); o.init(w.phi0)
    g.keep_B(True)
    g.step(steps); o.step(steps)
    eN, eB = pop_errors(g, o, w.mask == 0)
    err, _ = field_errors(g, o)
    assert eN < 1e-14 and eB < 1e-14, (eN, eB)
    assert max(err.values()) < 1e-14, err


# ---- edge cases: ragged sizes across several tiles, random masks, walls, tiny grids ---------------
def _random_case(ny, nx, seed, frac=0.25, **prm):
    rng = np.random.default_rng(seed)
    mask = (rng.uniform(size=(ny, nx)) < frac).astype(np.uint8)
    phi0 = rng.uniform(0, 1, (ny, nx))
    # smooth phi0 a little so that gradients are moderate
    for _ in range(2):
        phi0 = 0.25 * (np.roll(phi0, 1, 0) + np.roll(phi0, -1, 0) + np.roll(phi0, 1, 1) + np.roll(phi0, -1, 1))
    return ArrayWorkload(mask, phi0, disks=[[nx / 2 + 0.3, ny / 2 + 0.2, 10 * (nx + ny)]], **prm)


@pytest.mark.parametrize("schedule", SCHEDULES)
@pytest.mark.parametrize("shape,frac", [((3, 3), 0.0), ((5, 4), 0.3), ((45, 70), 0.25), ((70, 300), 0.3),
                                        ((19, 127), 0.5), ((9, 126), 0.1), ((130, 253), 0.2)])
def test_random_masks_ragged(schedule, shape, frac):
    w = _random_case(shape[0], shape[1], seed=shape[0] * 1000 + shape[1], frac=frac, rho_l=20.0, nu_l=0.05)
    g, o = make_pair(w, schedule=schedule)
    g.init(w.phi0); o.init(w.phi0)
    g.keep_B(True)
    g.step(5); o.step(5)
    fluid = w.mask == 0
    if fluid.any():
        eN, eB = pop_errors(g, o, fluid)
        assert eN < 1e-13 and eB < 1e-13, (eN, eB)
    err, _ = field_errors(g, o)
    assert max(err.values()) < 1e-12, err


@pytest.mark.parametrize("schedule", SCHEDULES)
def test_all_solid_and_all_fluid(schedule):
    for mask in (np.ones((6, 7), np.uint8), np.zeros((6, 7), np.uint8)):
        w = ArrayWorkload(mask, np.full((6, 7), 0.4), disks=[[3.3, 3.1, 100.0]])
        g, o = make_pair(w, schedule=schedule)
        g.init(w.phi0); o.init(w.phi0)
        g.step(3); o.step(3)
        err, _ = field_errors(g, o)
        assert max(err.values()) < 1e-14, err


@pytest.mark.parametrize("schedule", SCHEDULES)
def test_channel_with_walls_posts_body_force(schedule):
    w = wl.config4(seed=2, nx=256, ny=64)
    g, o = make_pair(w, schedule=schedule)
    g.init(w.phi0); o.init(w.phi0)
    g.keep_B(True)
    g.step(40); o.step(40)
    eN, eB = pop_errors(g, o, w.mask == 0)
    err, _ = field_errors(g, o)
    assert eN < 1e-12 and eB < 1e-12 and max(err.values()) < 1e-11, (eN, eB, err)
    dg, do = g.diag(), o.diag()
    assert dg["n_fluid"] == do["n_fluid"] and dg["nan"] == 0
    assert abs(dg["sum_phi"] - do["sum_phi"]) < 1e-9 and abs(dg["umax"] - do["umax"]) < 1e-13
    assert abs(dg["ke"] - do["ke"]) < 1e-12 * max(1.0, do["ke"])


@pytest.mark.parametrize("schedule", [pytest.param(0, id="auto"), pytest.param(FUSED, id="fused"), pytest.param(SPARSE, id="sparse")])
def test_fakhari_rule_variant(schedule):
    w = wl.config2(seed=1, theta_deg=150.0, n=64)
    for th in (150.0, 90.0, 90.01):
        g, o = make_pair(w, schedule=schedule, ghost_rule=1, theta_deg=th)
        g.init(w.phi0); o.init(w.phi0)
        g.step(10); o.step(10)
        err, _ = field_errors(g, o)
        assert max(err.values()) < 1e-13, (th, err)


def test_fakhari_rule_fp32_near_ninety_degrees():
    """Eq. 10 a hundredth of a degree from theta = 90: eps = 1.7e-4, where the expression as
    printed loses all its fp32 digits; the cancellation-free form keeps the 2e-4 tolerance."""
    w = wl.config2(seed=1, theta_deg=90.01, n=64)
    g, o = make_pair(w, precision=32, ghost_rule=1, theta_deg=90.01)
    g.init(w.phi0); o.init(w.phi0)
    g.step(20); o.step(20)
    err, scale = field_errors(g, o)
    uscale = max(scale["ux"], scale["uy"], w.sigma / (w.rho_l * w.nu_l))
    assert err["phi"] <= 2e-4 and max(err["ux"], err["uy"]) <= 2e-4 * uscale, err
    gh = w.mask == 1
    assert np.abs(g.get()["phi"] - o.get()["phi"])[gh].max() <= 2e-6      # the ghost values themselves


# ---- the north-star parity run: config 1, 1,000 steps, fp64 <= 1e-10 ------------------------------
@pytest.mark.parametrize("schedule", SCHEDULES)
def test_config1_1000_steps_fp64(schedule):
    w = wl.config1(seed=0)
    g, o = make_pair(w, schedule=schedule)
    g.init(w.phi0); o.init(w.phi0)
    g.keep_B(True)
    g.step(1000); o.step(1000)
    eN, eB = pop_errors(g, o, w.mask == 0)
    err, scale = field_errors(g, o)
    print("config1 1000 steps", schedule, eN, eB, err)
    assert eN <= 1e-10 and eB <= 1e-10
    assert max(err.values()) <= 1e-10, err
    # mass of each phase conserved on the device too
    m0 = float(w.phi0[w.mask == 0].sum())
    assert abs(g.diag()["sum_phi"] - m0) < 1e-10 * m0


@pytest.mark.parametrize("schedule", [pytest.param(0, id="auto"), pytest.param(SPARSE, id="sparse"), pytest.param(FUSED, id="fused")])
@pytest.mark.parametrize("precision", [64, 32])
def test_mirror_and_rotation_equivariance(schedule, precision):
    """Symmetry tests that need no oracle: mirroring the whole set-up about a vertical line mirrors the
    result, rotating it by 90 degrees rotates it (u as a vector).  The kernels treat x (lanes, strips, shuffles) and
    y (marches, ring slots) very differently, so a rotated run exercises the other code path on the same physics.
    Sizes are ragged (several strips, a tail) and the drop is off every symmetry axis (R16)."""
    from paper_2605_30878_b200 import binding
    ny, nx = 132, 188
    disks = np.array([[70.3, 40.6, 21.0], [150.2, 95.4, 14.5]])
    mask = wl.rasterize_disks(nx, ny, disks)
    phi0 = wl.drop_profile(nx, ny, 81.7, 77.2, 24.0, 4.0)
    prm = dict(rho_l=50.0, rho_g=1.0, nu_l=0.05, nu_g=0.1, sigma=0.01, W=4.0, theta_deg=65.0, mobility=0.02, gx=2e-7, gy=-1e-7)

    def run(mask, disks, phi0, gx, gy):
        p = dict(prm); p.update(gx=gx, gy=gy)
        s = binding.LBM(binding.LBMParams(nx=mask.shape[1], ny=mask.shape[0], precision=precision, schedule=schedule, **p), mask, disks)
        s.init(phi0); s.step(60)
        out = s.get()
        s.close()
        return out

    a = run(mask, disks, phi0, prm["gx"], prm["gy"])
    tol = 1e-12 if precision == 64 else 2e-5
    # mirror x -> nx - 1 - x
    dm = disks.copy(); dm[:, 0] = (nx - 1) - dm[:, 0]
    b = run(mask[:, ::-1].copy(), dm, phi0[:, ::-1].copy(), -prm["gx"], prm["gy"])
    for k, sgn in (("phi", 1), ("rho", 1), ("p", 1), ("ux", -1), ("uy", 1)):
        sc = prm["rho_l"] if k == "rho" else 1.0
        assert np.abs(a[k] - sgn * b[k][:, ::-1]).max() <= tol * sc, ("mirror", k)
    # rotation by 90 degrees: (x, y) -> (-y, x) on the lattice, i.e. array transpose + flip; u rotates with it
    dr = np.stack([(ny - 1) - disks[:, 1], disks[:, 0], disks[:, 2]], axis=1)
    c = run(np.ascontiguousarray(mask.T[:, ::-1]), dr, np.ascontiguousarray(phi0.T[:, ::-1]), -prm["gy"], prm["gx"])
    back = lambda f: f[:, ::-1].T                       # noqa: E731  undo the rotation of the arrays
    for k in ("phi", "rho", "p"):
        sc = prm["rho_l"] if k == "rho" else 1.0
        assert np.abs(a[k] - back(c[k])).max() <= tol * sc, ("rotation", k)
    assert np.abs(a["ux"] - back(c["uy"])).max() <= tol and np.abs(a["uy"] + back(c["ux"])).max() <= tol


def test_workspace_bytes_bounds_the_plan():
    """The host-only upper bound is never below what lbm_plan computes from the mask, for every layout."""
    from paper_2605_30878_b200 import binding
    for w in (wl.config1(seed=0), wl.config5(seed=1, n=256), wl.config4(seed=0, nx=256, ny=64)):
        for prec in (64, 32):
            for sched in (0, BASELINE, FUSED, PAIR, PACK, SPARSE):
                prm = binding.LBMParams(precision=prec, schedule=sched, **w.param_dict())
                s = binding.LBM(prm, w.mask, w.disks)
                assert binding.workspace_bytes(prm, s.n_ghost) >= s.workspace_bytes, (w.name, prec, sched)
                s.close()


def test_config1_1000_steps_through_cuda_graphs():
    """Small grids are launch-bound: off the legacy default stream lbm_step replays CUDA graphs
    of 32 steps.  Same 1,000-step parity run as above, same bar, and the launch bookkeeping still counts every
    kernel; odd step counts leave the ping-pong parity the graphs were captured for."""
    from paper_2605_30878_b200 import binding
    from oracle import ref
    w = wl.config1(seed=0)
    o = ref.RefLBM(ref.RefParams(**w.param_dict()), w.mask, w.disks)
    g = binding.LBM(binding.LBMParams(precision=64, **w.param_dict()), w.mask, w.disks, own_stream=True)
    g.init(w.phi0); o.init(w.phi0)
    for k in (333, 1, 666):      # 333 = 2 + 10 graphs + 11 plain steps; then an odd start for the next graphs
        g.step(k)
    o.step(1000)
    err, _ = field_errors(g, o)
    assert max(err.values()) <= 1e-10, err
    lc = g.launch_counts()
    assert lc["collide"] == 1000 and lc["ghost"] == 1001


@pytest.mark.parametrize("schedule", SCHEDULES)
def test_config1_1000_steps_fp32(schedule):
    w = wl.config1(seed=0)
    g, o = make_pair(w, precision=32, schedule=schedule)
    g.init(w.phi0); o.init(w.phi0)
    g.step(1000); o.step(1000)
    err, scale = field_errors(g, o)
    uscale = max(scale["ux"], scale["uy"], w.sigma / (w.rho_l * w.nu_l))        # R22
    print("config1 fp32", schedule, err, scale)
    assert err["phi"] <= 2e-4 and err["rho"] <= 2e-4 * scale["rho"]
    assert max(err["ux"], err["uy"]) <= 2e-4 * uscale
    Ng, _ = g.get_populations(want_B=False)
    No, _ = o.get_populations()
    assert np.abs(Ng - No)[:, w.mask == 0].max() <= 2e-4


@pytest.mark.parametrize("precision", [64, 32])
def test_config2_high_density_ratio_and_contact_angle(precision):
    """Density ratio 10, W = 5, theta = 120: fields after 2,000 steps and the measured contact
    angle (circle fit, §III.B) agree with the oracle within 0.5 deg (north_star)."""
    w = wl.config2(seed=0, theta_deg=120.0, n=128)
    g, o = make_pair(w, precision=precision)
    g.init(w.phi0); o.init(w.phi0)
    g.step(2000); o.step(2000)
    a, b = g.get(), o.get()
    tg = ms.contact_angle_on_cylinder(a["phi"], w.mask, w.disks[0], w.W)[0]
    to = ms.contact_angle_on_cylinder(b["phi"], w.mask, w.disks[0], w.W)[0]
    err, scale = field_errors(g, o)
    print("config2", precision, err, tg, to)
    assert abs(tg - to) <= 0.5
    if precision == 64:
        assert max(err.values()) <= 1e-10, err
    else:
        uscale = max(scale["ux"], scale["uy"], w.sigma / (w.rho_l * w.nu_l))
        assert err["phi"] <= 2e-4 and max(err["ux"], err["uy"]) <= 2e-4 * uscale


def test_config3_density_ratio_1000_short():
    w = wl.config3(seed=0, n=256)
    for precision, tol in ((64, 1e-10), (32, 2e-4)):
        g, o = make_pair(w, precision=precision)
        g.init(w.phi0); o.init(w.phi0)
        g.step(300); o.step(300)
        err, scale = field_errors(g, o)
        uscale = max(scale["ux"], scale["uy"], w.sigma / (w.rho_l * w.nu_l))
        print("config3", precision, err, scale)
        assert err["phi"] <= tol
        assert max(err["ux"], err["uy"]) <= (tol if precision == 64 else tol * uscale)
        assert err["rho"] <= tol * scale["rho"]          # rho = rho_g + 999 phi: relative to field scale


@pytest.mark.parametrize("sched", [pytest.param(FUSED, id="fused"), pytest.param(PAIR, id="pair"),
                                   pytest.param(PACK, id="pack"), pytest.param(SPARSE, id="sparse")])
def test_schedules_agree_and_get_is_idempotent(sched):
    w = wl.config5(seed=3, n=256)
    a, _ = make_pair(w, schedule=BASELINE)
    b, _ = make_pair(w, schedule=sched)
    a.init(w.phi0); b.init(w.phi0)
    a.step(25); b.step(10); b.get(); b.step(15)        # lbm_get must not disturb the state
    fa, fb = a.get(), b.get()
    for k in fa:
        assert np.abs(fa[k] - fb[k]).max() < 1e-13 * max(1.0, np.abs(fa[k]).max()), k   # rho = 1 + 999 phi
    with pytest.raises(Exception):
        b.get_populations(want_B=True)                 # B is not stored unless keep_B was set
    lc = b.launch_counts()
    assert lc["collide"] == 25 and lc["phi_sum"] == 0 and lc["ghost"] == 26


# ---- throughput workload (config 5) in the launch configuration bench.py times ---------------------
@pytest.mark.parametrize("precision", [64, 32])
def test_config5_2048_against_oracle(precision):
    """Porous medium at 2048^2 (first size of BASELINE config 5; same recipe, launch schedule and
    kernel as bench.py's 8192^2): full fields against the oracle after a few steps."""
    w = wl.config5(seed=1, n=2048)
    g, o = make_pair(w, precision=precision)               # schedule AUTO = what bench.py runs
    g.init(w.phi0); o.init(w.phi0)
    g.step(3); o.step(3)
    err, scale = field_errors(g, o)
    uscale = max(scale["ux"], scale["uy"], w.sigma / (w.rho_l * w.nu_l))
    print("config5 2048", precision, err, scale)
    tol = 1e-12 if precision == 64 else 2e-4
    assert err["phi"] <= tol
    assert max(err["ux"], err["uy"]) <= (tol if precision == 64 else tol * uscale)
    assert err["rho"] <= tol * scale["rho"]


def test_config5_8192_properties_and_samples():
    """bench.py's exact workload (8192^2, seed 0, schedule AUTO).  The oracle needs minutes per step
    at this size, so: (i) per-phase mass is conserved (sum B_i* = phi), (ii) no NaN,
    phi stays in range, (iii) sampled nodes agree with the BASELINE schedule (independent kernels,
    N and B both in HBM), which the smaller tests pin to the oracle."""
    w = wl.config5(seed=0, n=8192)
    rng = np.random.default_rng(5)
    fl = np.flatnonzero(w.mask.reshape(-1) == 0)
    idx = np.sort(rng.choice(fl, 200000, replace=False)).astype(np.int64)
    from paper_2605_30878_b200 import binding
    res = {}
    for sched in (0, BASELINE):
        s = binding.LBM(binding.LBMParams(precision=64, schedule=sched, **w.param_dict()), w.mask, w.disks)
        s.init(w.phi0)
        d0 = s.diag()
        s.step(20)
        d1 = s.diag()
        assert d1["nan"] == 0 and -1e-3 < d1["phi_min"] and d1["phi_max"] < 1 + 1e-3
        assert abs(d1["sum_phi"] - d0["sum_phi"]) <= 1e-11 * d0["sum_phi"]
        res[sched] = s.sample_populations(idx)[0]
        s.close()
    assert np.abs(res[0] - res[BASELINE]).max() <= 1e-13


def _window_case(w, x0, y0, size):
    """The part [y0, y0+size) x [x0, x0+size) of a periodic workload as a workload of its own (periodic
    in the window's size: only its interior is comparable), with the disks that touch it."""
    ny, nx = w.mask.shape
    jj = (np.arange(y0, y0 + size) % ny)[:, None]
    ii = (np.arange(x0, x0 + size) % nx)[None, :]
    d = w.disks.copy()
    d[:, 0] = (d[:, 0] - x0 + nx / 2) % nx - nx / 2          # centre relative to the window origin, nearest image
    d[:, 1] = (d[:, 1] - y0 + ny / 2) % ny - ny / 2
    keep = (d[:, 0] + d[:, 2] > -2) & (d[:, 0] - d[:, 2] < size + 2) & (d[:, 1] + d[:, 2] > -2) & (d[:, 1] - d[:, 2] < size + 2)
    prm = w.param_dict(); prm.pop("nx"); prm.pop("ny")
    return ArrayWorkload(w.mask[jj, ii], w.phi0[jj, ii], disks=d[keep], **prm), jj, ii


@pytest.mark.parametrize("precision", [64, 32])
def test_config5_8192_windows_against_oracle(precision):
    """bench.py's exact workload and launch configuration (8192^2, seed 0, schedule AUTO) against the ORACLE:
    the method is local (information travels at most 4 nodes per step: stencil, ghost interpolation), so the
    oracle run on a window cut out of the 8192^2 inputs reproduces the full-domain result on the window's
    interior.  Windows sit at the periodic seam, beyond 4 GB of plane offset, in rows above 4096 and at the
    last rows / columns — the places that only exist at full size."""
    from oracle import ref
    from paper_2605_30878_b200 import binding
    w = wl.config5(seed=0, n=8192)
    steps, size = 5, 460
    # margin: 4 nodes per step, plus the reach of a disk (radius <= 32) whose periodic image in the window's own
    # period could otherwise be taken for the owner of a ghost node near the opposite edge
    h = 4 * steps + 2 + 68
    g = binding.LBM(binding.LBMParams(precision=precision, **w.param_dict()), w.mask, w.disks)
    g.init(w.phi0)
    g.step(steps)
    G = g.get()
    tol = 1e-12 if precision == 64 else 2e-4
    for (x0, y0) in ((8192 - 230, 8192 - 230), (5000, 4100), (8192 - 460, 6000), (1234, 8192 - 460), (7700, 0)):
        ww, jj, ii = _window_case(w, x0, y0, size)
        o = ref.RefLBM(ref.RefParams(**ww.param_dict()), ww.mask, ww.disks)
        o.init(ww.phi0); o.step(steps)
        O = o.get()
        inner = np.zeros((size, size), bool); inner[h:-h, h:-h] = True
        # (the window's own periodic seam is a discontinuity: the oracle's values near it mean nothing)
        uscale = max(np.abs(O["ux"][inner]).max(), np.abs(O["uy"][inner]).max(), w.sigma / (w.rho_l * w.nu_l))
        for k in ("phi", "rho", "ux", "uy", "p"):
            d = np.abs(G[k][jj, ii] - O[k])[inner].max()
            if precision == 64:      # absolute, rho relative to its scale rho_l
                sc = w.rho_l if k == "rho" else 1.0
            else:                    # fp32: relative to field scale (north_star; u per R22)
                sc = {"phi": 1.0, "rho": w.rho_l, "p": max(np.abs(O["p"][inner]).max(), 1e-30)}.get(k, uscale)
            assert d <= tol * sc, (x0, y0, k, d, sc)
        # populations of the fluid nodes of the interior, element by element
        fl = inner & (ww.mask == 0)
        idx = (jj * 8192 + ii)[fl].astype(np.int64)
        Ng = g.sample_populations(idx)[0]
        No = o.get_populations()[0][:, fl]
        assert np.abs(Ng - No).max() <= (1e-13 if precision == 64 else 2e-4), (x0, y0)
    g.close()


def test_config5_16384_fp64_on_one_gpu():
    """Compacted layouts keep no dense copy of the state (workspace 9.8 GB at 8192^2 fp64, 39 GB at 16384^2):
    the 16384^2 fp64 domain runs on one B200.  Mass is conserved and a window of it, past every 32-bit element
    offset of a dense plane, agrees with the oracle run on that window."""
    from oracle import ref
    from paper_2605_30878_b200 import binding
    n, steps, size = 16384, 3, 400
    w = wl.config5(seed=0, n=n)
    g = binding.LBM(binding.LBMParams(precision=64, **w.param_dict()), w.mask, w.disks)
    assert g.workspace_bytes < 45e9
    g.init(w.phi0)
    m0 = g.diag()["sum_phi"]
    g.step(steps)
    d = g.diag()
    assert d["nan"] == 0 and abs(d["sum_phi"] - m0) <= 1e-11 * m0
    G = g.get(fields=("phi", "ux", "uy"))
    h = 4 * steps + 2 + 68
    x0, y0 = n - 200, n - 200                                  # across both periodic seams, last rows and columns
    ww, jj, ii = _window_case(w, x0, y0, size)
    o = ref.RefLBM(ref.RefParams(**ww.param_dict()), ww.mask, ww.disks)
    o.init(ww.phi0); o.step(steps)
    O = o.get()
    inner = np.zeros((size, size), bool); inner[h:-h, h:-h] = True
    for k in ("phi", "ux", "uy"):
        assert np.abs(G[k][jj, ii] - O[k])[inner].max() <= 1e-12, k
    fl = inner & (ww.mask == 0)
    idx = (jj.astype(np.int64) * n + ii)[fl]
    assert np.abs(g.sample_populations(idx)[0] - o.get_populations()[0][:, fl]).max() <= 1e-13
    g.close()


def test_config5_8192_is_deterministic():
    """Two runs of the 8192^2 AUTO schedule, 200 steps each, give bit-identical phi and sampled populations:
    the evidence against races in the warp-private rings that is available while compute-sanitizer is closed
    on this pool (no atomics anywhere on the path, every output has one writer)."""
    from paper_2605_30878_b200 import binding
    w = wl.config5(seed=0, n=8192)
    fl = np.flatnonzero(w.mask.reshape(-1) == 0)
    idx = np.sort(np.random.default_rng(9).choice(fl, 300000, replace=False)).astype(np.int64)
    out = []
    for _ in range(2):
        s = binding.LBM(binding.LBMParams(precision=64, **w.param_dict()), w.mask, w.disks)
        s.init(w.phi0); s.step(200)
        out.append((s.get(fields=("phi",))["phi"].copy(), s.sample_populations(idx)[0].copy()))
        s.close()
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1])


@pytest.mark.parametrize("schedule", [pytest.param(0, id="auto"), pytest.param(BASELINE, id="baseline"), pytest.param(SPARSE, id="sparse"),
                                      pytest.param(INPLACE, id="inplace")])
def test_set_populations_round_trip_and_restart(schedule):
    """lbm_set_populations: (i) what is set is what lbm_get_populations returns, (ii) both sides handed the
    same far-from-equilibrium state continue identically, (iii) a fresh context restarted from another
    context's populations continues like the original."""
    w = wl.config2(seed=4, theta_deg=60.0, n=64)
    g, o = make_pair(w, schedule=schedule)
    g.init(w.phi0); o.init(w.phi0)
    g.step(5); o.step(5)
    No, Bo = o.get_populations()
    rng = np.random.default_rng(11)
    fluid = w.mask == 0
    N2 = No * (1.0 + 0.05 * rng.standard_normal(No.shape))        # 5 % noise: far from equilibrium
    B2 = N2 * np.clip(Bo / np.maximum(No, 1e-300) + 0.1 * rng.standard_normal(No.shape), 0.0, 1.0)
    N2[:, ~fluid] = 0.0; B2[:, ~fluid] = 0.0
    g.keep_B(True)
    g.set_populations(N2, B2); o.set_populations(N2, B2)
    Ng, Bg = g.get_populations(want_B=True)
    assert np.abs(Ng - N2)[:, fluid].max() <= 1e-15 and np.abs(Bg - B2)[:, fluid].max() <= 1e-15
    g.step(3); o.step(3)
    eN, eB = pop_errors(g, o, fluid)
    err, _ = field_errors(g, o)
    assert eN < 1e-13 and eB < 1e-13 and max(err.values()) < 1e-11, (eN, eB, err)
    # without B planes (keep_B never called) B is still taken in: phi and the ghost values follow it
    g2, o2 = make_pair(w, schedule=schedule)
    g2.init(w.phi0); o2.init(w.phi0)
    g2.set_populations(N2, B2); o2.set_populations(N2, B2)
    g2.step(2); o2.step(2)
    err2, _ = field_errors(g2, o2)
    assert max(err2.values()) < 1e-11, err2
    # restart: N only (phi and the ghost values of the receiving context stay as they are).  g has taken an odd number of
    # steps: under INPLACE its state is parked in the nodes' own slots and the B_i must be re-parked, not lost
    B_before = g.get_populations(want_B=True)[1] if schedule in (BASELINE, INPLACE) else None
    g.set_populations(N=N2)
    assert np.abs(g.get_populations(want_B=False)[0] - N2)[:, fluid].max() <= 1e-15
    if B_before is not None:
        assert np.array_equal(g.get_populations(want_B=True)[1], B_before)
        o.set_populations(N2, B_before)
        g.step(3); o.step(3)
        eN, eB = pop_errors(g, o, fluid)
        assert eN < 1e-13 and eB < 1e-13, (eN, eB)


def test_symmetric_setup_differs_only_where_the_gradient_vanishes():
    """R16: n_phi = grad phi/|grad phi| is undefined where grad phi = 0.  On the mirror-symmetric
    config 1 (no jitter) the gradient cancels to rounding noise on the symmetry axis inside the drop and the
    solid, the direction of n_phi is then decided by the summation order, and two correct implementations
    may differ there — by at most the size of the anti-diffusion term, (2/W) phi (1 - phi) |c_i| N_i^eq, and
    nowhere else."""
    w = wl.config1(seed=0, jitter=False)
    g, o = make_pair(w)
    g.init(w.phi0); o.init(w.phi0)
    g.keep_B(True)
    g.step(1); o.step(1)
    Ng, Bg = g.get_populations(want_B=True)
    No, Bo = o.get_populations()
    fluid = w.mask == 0
    assert np.abs(Ng - No)[:, fluid].max() < 1e-14          # N* does not depend on n_phi
    # gradient of the time-0 order parameter (with the first ghost values), isotropic D2Q9 stencil (R8)
    from oracle import ref
    o0 = ref.RefLBM(ref.RefParams(**w.param_dict()), w.mask, w.disks); o0.init(w.phi0); o0.step(1)
    ph = o0.get_phi_raw().reshape(w.ny, w.nx)               # phi(0) on fluid nodes, ghost values of step 1
    cx, cy, _, wq = ref.lattice()
    gx = sum(3 * wq[q] * cx[q] * np.roll(ph, (-cy[q], -cx[q]), (0, 1)) for q in range(9))
    gy = sum(3 * wq[q] * cy[q] * np.roll(ph, (-cy[q], -cx[q]), (0, 1)) for q in range(9))
    gnorm = np.hypot(gx, gy)
    dB = np.abs(Bg - Bo).max(axis=0)
    differs = fluid & (dB > 1e-14)
    assert (gnorm[differs] < 1e-12).all(), gnorm[differs].max()
    bound = (2.0 / w.W) * ph * (1 - ph) * math.sqrt(2.0) * 2.0   # N_i^eq <= 1; both directions of n_phi
    assert (dB[differs] <= bound[differs] + 1e-14).all()


# ---- NEXT row f3: drop on a flat plate (§III.A): wall rows only, no disk list -------------
@pytest.mark.parametrize("precision", [64, 32])
def test_flat_plate_fields_and_eq12_angle(precision):
    w = wl.flat_plate(theta_deg=120.0, W=4.0, scale=0.25, rho_ratio=10.0, mu_ratio=10.0, x_offset=0.37)
    g, o = make_pair(w, precision=precision)
    g.init(w.phi0); o.init(w.phi0)
    g.step(500); o.step(500)
    err, scale = field_errors(g, o)
    tg = ms.contact_angle_on_plate(g.get()["phi"], w.mask, w.W)[0]
    to = ms.contact_angle_on_plate(o.get()["phi"], w.mask, w.W)[0]
    print("flat plate", precision, err, tg, to)
    assert abs(tg - to) <= 0.5
    if precision == 64:
        assert max(err.values()) <= 1e-10, err
    else:
        uscale = max(scale["ux"], scale["uy"], w.sigma / (w.rho_l * w.nu_l))
        assert err["phi"] <= 2e-4 and max(err["ux"], err["uy"]) <= 2e-4 * uscale


# ---- NEXT row f2: geometry from the mask alone (no disk list) ------------------------------------------
def test_mask_only_geometry_bit_exact_and_fields():
    rng = np.random.default_rng(11)
    n = 96
    disks = np.array([[30.2, 40.7, 17.0], [70.5, 60.1, 11.5]])
    mask = wl.rasterize_disks(n, n, disks)
    mask[80:84, 10:50] = 1                                     # a bar: not describable by the disk list
    yy, xx = np.mgrid[0:n, 0:n]
    phi0 = 0.5 * (1 - np.tanh(2 * (np.hypot(xx - 48.3, yy - 22.7) - 14.0) / 4.0))   # off-lattice centre, see R16
    w = ArrayWorkload(mask, phi0, theta_deg=65.0)
    g, o = make_pair(w)
    cg, co = g.get_classification(), o.get_classification()
    assert np.array_equal(cg["cls"], co["cls"]) and np.array_equal(cg["idx"], co["idx"])
    for k in ("nx", "ny", "depth"):
        assert np.array_equal(cg[k], co[k]), k                 # bit-exact normals
    assert np.array_equal(cg["corner"], co["corner"]) and np.array_equal(cg["wgt"], co["wgt"])
    g.init(w.phi0); o.init(w.phi0)
    g.step(50); o.step(50)
    err, _ = field_errors(g, o)
    assert max(err.values()) < 1e-12, err


def test_particle_at_interface_fields():
    """PAPER.md §III.C set-up (walls + one cylinder through a flat interface): short run against the oracle."""
    w = wl.particle_at_interface(theta_deg=60.0, x_offset=0.31)
    for precision, tol in ((64, 1e-10), (32, 2e-4)):
        g, o = make_pair(w, precision=precision)
        g.init(w.phi0); o.init(w.phi0)
        g.step(400); o.step(400)
        err, scale = field_errors(g, o)
        uscale = max(scale["ux"], scale["uy"], w.sigma / (w.rho_l * w.nu_l))
        assert err["phi"] <= tol and max(err["ux"], err["uy"]) <= (tol if precision == 64 else tol * uscale), err
        yg = ms.interface_height_at_boundary(g.get()["phi"]); yo = ms.interface_height_at_boundary(o.get()["phi"])
        assert abs(yg - yo) <= (1e-9 if precision == 64 else 1e-3)


# ---- the BASELINE configs at their full lengths (GPU only; the oracle pins the same physics at reduced
# ---- size in tests/golden/oracle_certificate.json) ------------------------------------------------------
def _gpu_sim(w, precision):
    from paper_2605_30878_b200 import binding
    s = binding.LBM(binding.LBMParams(precision=precision, **w.param_dict()), w.mask, w.disks)
    s.init(w.phi0)
    return s


@pytest.mark.parametrize("precision", [64, 32])
def test_baseline_config2_contact_angle_sweep_full_length(precision):
    """Config 2 as BASELINE.json states it: 256^2, R = 40, drop 35, W = 5, density ratio 10, 20,000 steps
    for each of the five angles.  The measured angle (circle fit + circle-circle geometry, §III.B)
    stays within 4 degrees of the prescribed one, mass is conserved, fp32 and fp64 agree ("produced same
    results", :237)."""
    for theta in (30.0, 60.0, 90.0, 120.0, 150.0):
        w = wl.config2(seed=0, theta_deg=theta, n=256)
        s = _gpu_sim(w, precision)
        m0 = s.diag()["sum_phi"]
        s.step(20000)
        d = s.diag()
        th = ms.contact_angle_on_cylinder(s.get()["phi"], w.mask, w.disks[0], w.W)[0]
        print("config2 full", precision, theta, th, d["umax"], (d["sum_phi"] - m0) / m0)
        assert d["nan"] == 0 and abs(th - theta) < 4.0
        assert abs(d["sum_phi"] - m0) < (1e-10 if precision == 64 else 2e-4) * m0
        assert d["umax"] < 1e-3
        s.close()


@pytest.mark.parametrize("precision", [64, 32])
def test_baseline_config3_full_length_spurious_currents(precision):
    """Config 3: 1024^2, density ratio 1000, viscosity ratio 100, sigma = 1e-3, theta = 45 deg, 50,000 steps;
    reports max|u| (spurious currents, O(1e-6)-O(1e-5) lattice units in the paper, :114, :252)."""
    w = wl.config3(seed=0, n=1024)
    s = _gpu_sim(w, precision)
    m0 = s.diag()["sum_phi"]
    s.step(50000)
    d = s.diag()
    th = ms.contact_angle_on_cylinder(s.get()["phi"], w.mask, w.disks[0], w.W)[0]
    print("config3 full", precision, "umax", d["umax"], "theta", th, "drift", (d["sum_phi"] - m0) / m0)
    assert d["nan"] == 0 and d["umax"] < 2e-4 and abs(th - 45.0) < 4.0
    assert abs(d["sum_phi"] - m0) < (1e-10 if precision == 64 else 5e-4) * m0
    s.close()


def test_baseline_config4_full_length_fp32():
    """Config 4: 2048 x 512 channel, wall rows, 8 posts, body force 1e-7, density ratio 100, fp32,
    100,000 steps: stays finite, conserves liquid mass to fp32 accumulation error, phi stays in range."""
    w = wl.config4(seed=0)
    s = _gpu_sim(w, 32)
    m0 = s.diag()["sum_phi"]
    s.step(100000)
    d = s.diag()
    print("config4 full", d, (d["sum_phi"] - m0) / m0)
    assert d["nan"] == 0 and -1e-2 < d["phi_min"] and d["phi_max"] < 1 + 1e-2
    assert abs(d["sum_phi"] - m0) < 2e-3 * m0 and d["umax"] < 0.05
    s.close()


# ---- the paper's closed-form benchmarks at the paper's own sizes (GPU path; §III.A and §III.C) --------------
@pytest.mark.parametrize("W,tol_deg", [(4.0, 5.0), (8.0, 2.0)])
def test_paper_flat_plate_contact_angles(W, tol_deg):
    """§III.A: (500, 300) box, A = 1e4, default ratios 1000 / 100, theta = 30 ... 150 deg, angle by Eq. 12.
    The paper reports errors of a few degrees at W = 4 (Fig. 6) and < 2 degrees for W >= 6 (:124)."""
    for theta in (30.0, 60.0, 90.0, 120.0, 150.0):
        w = wl.flat_plate(theta_deg=theta, W=W, scale=1.0)
        s = _gpu_sim(w, 64)
        m0 = s.diag()["sum_phi"]
        s.step(30000)
        d = s.diag()
        th = ms.contact_angle_on_plate(s.get()["phi"], w.mask, w.W)[0]
        print("flat plate full", W, theta, th, d["umax"])
        assert d["nan"] == 0 and abs(th - theta) < tol_deg and abs(d["sum_phi"] - m0) < 1e-10 * m0
        s.close()


def test_paper_flat_plate_interface_width_sweep():
    """§III.A, Fig. 7: the interface width swept over W = 4 ... 10 at the two extreme angles,
    theta = 30 and 150 deg.  The paper's statement: the error of the measured angle stays below 2 degrees once
    W >= 6; at W = 4, 5 it is a few degrees (Fig. 6-7)."""
    worst = {}
    for W in (4.0, 5.0, 6.0, 7.0, 8.0, 9.0, 10.0):
        for theta in (30.0, 150.0):
            w = wl.flat_plate(theta_deg=theta, W=W, scale=1.0)
            s = _gpu_sim(w, 64)
            m0 = s.diag()["sum_phi"]
            s.step(30000)
            d = s.diag()
            th = ms.contact_angle_on_plate(s.get()["phi"], w.mask, w.W)[0]
            worst[(W, theta)] = th - theta
            assert d["nan"] == 0 and abs(d["sum_phi"] - m0) < 1e-10 * m0
            assert abs(th - theta) < (2.0 if W >= 6.0 else 5.0), (W, theta, th)
            s.close()
    print("flat plate W sweep, theta_measured - theta:", worst)


def test_paper_spurious_currents_present_rule_against_fakhari():
    """§III.A, Fig. 5: maximum spurious velocity of the steady drop on the flat plate at 30 and
    150 deg, for the paper's rule (Eq. 9) and for the Fakhari-Bolster rule (Eq. 10).  The paper prints 5.74e-7 / 7e-7
    against 6.98e-7 / 1e-6 and calls the currents O(1e-6).  Checked here: the order of magnitude, the paper's ordering
    (Eq. 9 gives the smaller currents at both angles), and the 30-degree value of the present rule within 25 % of the
    printed one.  (Recorded on the GPU path, fp64, 60,000 steps: 6.6e-7 / 2.5e-6 against 2.6e-6 / 7.7e-6: our half-way
    reading of Eq. 10 — the paper's comparison code also interpolates the bounce-back, :96 — leaves larger currents.)"""
    import json
    import os
    ref_vals = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.json")))["spurious_current_flat_plate"]
    from paper_2605_30878_b200 import binding
    umax = {}
    for theta in (30.0, 150.0):
        for rule in (0, 1):
            w = wl.flat_plate(theta_deg=theta, W=4.0, scale=1.0)
            s = binding.LBM(binding.LBMParams(precision=64, ghost_rule=rule, **w.param_dict()), w.mask, w.disks, own_stream=True)
            s.init(w.phi0); s.step(60000)
            d = s.diag()
            assert d["nan"] == 0
            umax[(theta, rule)] = d["umax"]
            s.close()
    print("spurious currents", umax)
    for theta in (30.0, 150.0):
        assert umax[(theta, 0)] < umax[(theta, 1)]                     # the paper's ordering
        assert umax[(theta, 0)] < 5e-6 and umax[(theta, 1)] < 2e-5     # O(1e-6), :252
    assert umax[(30.0, 0)] == pytest.approx(ref_vals["theta30"], rel=0.25)


def test_paper_drop_on_cylinder_hmax_present_rule_against_fakhari():
    """§III.B, Fig. 8-9: the paper's own set-up — (5R, 5R) box, R = 40, A = 3000, W = 4, density
    ratio 1000 — started from the analytic configuration.  The paper prints the error of h_max / R against the
    circle-circle solution: -0.35 % / +0.26 % at 30 / 150 deg for its rule, -0.76 % / +0.70 % for Fakhari et al.'s.
    Checked here on the GPU path (h_max from the circle fitted to the phi = 1/2 contour): the signs, that Eq. 9 is the
    more accurate of the two at both angles by about the paper's factor (2.2 - 2.7), and the size (< 1 %).
    Recorded (against the analytic solution for the liquid area that is actually conserved): 150 deg after 500,000
    steps (steady) +0.50 % against +1.52 %; 30 deg after 300,000 steps (the drop is still creeping: t_cap ~ 5e4,
    t_visc ~ 1e5 steps) -0.34 % against -0.48 %."""
    import json
    import os
    ref_vals = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.json")))["hmax_over_R_error_percent"]
    from paper_2605_30878_b200 import binding
    err = {}
    for theta, steps in ((150.0, 500000), (30.0, 300000)):
        for rule in (0, 1):
            w = wl.drop_on_cylinder_paper(theta_deg=theta)
            s = binding.LBM(binding.LBMParams(precision=64, ghost_rule=rule, **w.param_dict()), w.mask, w.disks, own_stream=True)
            s.init(w.phi0)
            m0 = s.diag()["sum_phi"]
            assert m0 == pytest.approx(3000.0, rel=1e-2)               # the tanh profile of the analytic cap holds 0.2 - 0.5 % more
            s.step(steps)
            d = s.diag()
            assert d["nan"] == 0 and abs(d["sum_phi"] - m0) < 1e-9 * m0
            hmax = ms.contact_angle_on_cylinder(s.get()["phi"], w.mask, w.disks[0], w.W)[3]
            h_a = ms.analytic_drop_on_cylinder(w.meta["R"], m0, theta)[2]   # for the area that is actually conserved
            err[(theta, rule)] = 100.0 * (hmax - h_a) / w.meta["R"]
            s.close()
    print("h_max/R error in percent", err, "paper", ref_vals)
    for theta in (30.0, 150.0):
        key = str(int(theta))
        assert np.sign(err[(theta, 0)]) == np.sign(ref_vals["present"][key]) == np.sign(err[(theta, 1)])
        assert abs(err[(theta, 0)]) < abs(err[(theta, 1)])              # Eq. 9 beats Eq. 10, as in the paper
        assert abs(err[(theta, 0)]) < 1.0
    assert 1.8 < err[(150.0, 1)] / err[(150.0, 0)] < 3.5                # paper: 0.70 / 0.26 = 2.7


def test_paper_particle_at_interface_eq13():
    """§III.C: 4.8 R box, R = 25: displacement h* of the interface at the periodic boundary against Eq. 13;
    the paper's own error is ~9 % at 30 / 150 deg and ~6 % at 60 - 120 deg (:197)."""
    for theta in (30.0, 60.0, 120.0, 150.0):
        w = wl.particle_at_interface(theta_deg=theta)
        s = _gpu_sim(w, 64)
        s.step(60000)
        y = ms.interface_height_at_boundary(s.get()["phi"])
        h, h_an = w.meta["y_interface0"] - y, ms.eq13_hstar(w.meta["L"], w.meta["R"], theta)[0]
        print("particle full", theta, h, h_an, s.diag()["umax"])
        assert abs(h - h_an) < 0.12 * abs(h_an)
        s.close()


def test_layout_copy_helper_leaves_the_state_alone():
    w = wl.config5(seed=2, n=256)
    g, _ = make_pair(w, schedule=PAIR)                  # the helper measures the dense SoA layout (PAIR's)
    g.init(w.phi0); g.step(7)
    a = g.get()
    ms_copy = g.layout_copy_timed(3)
    g.step(5)
    h, _ = make_pair(w, schedule=PAIR)
    h.init(w.phi0); h.step(12)
    p, _ = make_pair(w)                                 # compacted layouts keep no dense planes: refused, state untouched
    p.init(w.phi0)
    with pytest.raises(Exception):
        p.layout_copy_timed(1)
    b, c = g.get(), h.get()
    assert ms_copy > 0
    for k in a:
        assert np.array_equal(b[k], c[k]), k            # same as a run without the helper, bit for bit


@pytest.mark.parametrize("schedule", [pytest.param(PAIR, id="pair"), pytest.param(PACK, id="pack"), pytest.param(SPARSE, id="sparse")])
@pytest.mark.parametrize("shape,frac", [((7, 4), 0.2), ((9, 12), 0.3), ((33, 36), 0.3), ((50, 100), 0.25),
                                        ((61, 244), 0.3), ((40, 126), 0.3)])
def test_random_masks_ragged_fp32(schedule, shape, frac):
    """fp32 lane groups: four nodes per lane when nx % 4 == 0, two otherwise, strips wider than the grid."""
    w = _random_case(shape[0], shape[1], seed=shape[0] * 1000 + shape[1], frac=frac, rho_l=20.0, nu_l=0.05)
    g, o = make_pair(w, precision=32, schedule=schedule)
    g.init(w.phi0); o.init(w.phi0)
    g.step(20); o.step(20)
    err, scale = field_errors(g, o)
    uscale = max(scale["ux"], scale["uy"], w.prm["sigma"] / (w.prm["rho_l"] * w.prm["nu_l"]))
    assert err["phi"] <= 2e-4 and max(err["ux"], err["uy"]) <= 2e-4 * uscale, err
    Ng, _ = g.get_populations(want_B=False)
    No, _ = o.get_populations()
    assert np.abs(Ng - No)[:, w.mask == 0].max() <= 2e-4
