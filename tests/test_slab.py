"""Slab decomposition along y (`paper_2605_30878_b200/slab.py`).

CPU part (no GPU, no kernels): the host logic — partition, slicing of the inputs with the periodic wrap, the disks'
images in the local frame, halo width, the order of the pairwise sends with two ranks (world_size-2 `gloo`) — driven
through a stand-in context whose "time step" is a plain three-row stencil on host memory, so that a wrong row range or
a swapped neighbour changes the result.

GPU part: the real contexts, 2 and 3 slabs driven one after the other on one device (no kernel waits on another),
against the single-domain run of the same workload.
"""
import ctypes as C
import os
import sys

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_2605_30878_b200 import binding, slab, workloads as wl   # noqa: E402


# ---------------------------------------------------------------------------------------------------------------
# stand-in context: same calls as binding.LBM, host memory, a stencil that reaches ROWS_PER_STEP rows per step
# ---------------------------------------------------------------------------------------------------------------
class RowModel:
    def __init__(self, prm, mask, disks):
        self.nx, self.ny = prm.nx, prm.ny
        self.u = np.zeros((self.ny, self.nx))
        self.mask = np.asarray(mask).reshape(self.ny, self.nx).astype(np.float64)
        self.disks = np.asarray(disks).reshape(-1, 3)

    def init(self, phi0, u0=None):
        self.u = np.array(phi0, dtype=np.float64).reshape(self.ny, self.nx)

    def step(self, n):
        r = slab.ROWS_PER_STEP
        for _ in range(n):   # periodic in the LOCAL height, like a real context; uses the mask so that its slicing matters
            self.u = 0.5 * self.u + 0.2 * np.roll(self.u, r, 0) + 0.3 * np.roll(self.u, -r, 0) + 0.01 * np.roll(self.mask, 1, 0)

    def get(self):
        return {"phi": self.u.copy()}

    def rows_bytes(self, j0, nrows):
        assert 0 <= j0 and j0 + nrows <= self.ny
        return nrows * self.nx * 8

    def _view(self, ptr, nbytes):
        return np.frombuffer((C.c_uint8 * nbytes).from_address(ptr), dtype=np.float64)

    def rows_export(self, j0, nrows, ptr, cap):
        self._view(ptr, nrows * self.nx * 8)[:] = self.u[j0:j0 + nrows].reshape(-1)

    def rows_import(self, j0, nrows, ptr, nbytes):
        assert nbytes == nrows * self.nx * 8
        self.u[j0:j0 + nrows] = self._view(ptr, nbytes).reshape(nrows, self.nx)

    def close(self):
        pass


def _toy(nx=5, ny=96, seed=0):
    rng = np.random.default_rng(seed)
    prm = binding.LBMParams(nx=nx, ny=ny)
    mask = (rng.random((ny, nx)) < 0.3).astype(np.uint8)
    phi0 = rng.random((ny, nx))
    return prm, mask, phi0


def _reference(prm, mask, phi0, steps):
    m = RowModel(prm, mask, np.zeros((0, 3)))
    m.init(phi0)
    m.step(steps)
    return m.u


def test_partition_and_halo():
    assert slab.partition(10, 3) == [(0, 3), (3, 6), (6, 10)]
    assert slab.partition(8192, 8)[3] == (3072, 4096)
    with pytest.raises(ValueError):
        slab.partition(2, 3)
    assert slab.geometry_margin(None) == slab.MASK_ONLY_MARGIN
    assert slab.geometry_margin([(1.0, 2.0, 31.2), (0.0, 0.0, 8.0)]) == 66
    assert slab.halo_rows(66, 4) == 66 + 3 * 4


def test_local_inputs_wrap_and_disk_images():
    ny, nx = 40, 3
    mask = np.arange(ny * nx).reshape(ny, nx) % 251
    phi0 = np.arange(ny * nx, dtype=float).reshape(ny, nx)
    disks = [(1.0, 2.0, 4.0), (1.0, 20.0, 3.0), (1.0, 38.5, 2.0)]
    li = slab.local_inputs(ny, 0, 10, 6, mask, disks, phi0)            # rows -6 .. 15 of a 40-row grid
    rows = np.arange(-6, 16) % ny
    assert np.array_equal(li["mask"], mask[rows]) and np.array_equal(li["phi0"], phi0[rows])
    got = sorted((round(cy, 6), r) for _, cy, r in li["disks"])
    # disk 0 at global 2 -> local 8; disk 2 through its image below the grid: 38.5 - 40 = -1.5 -> local 4.5; disk 1 is out of reach
    assert got == [(4.5, 2.0), (8.0, 4.0)]
    li = slab.local_inputs(ny, 30, 40, 6, mask, disks, phi0)           # rows 24 .. 45: disk 0 through its image above;
    got = sorted((round(cy, 6), r) for _, cy, r in li["disks"])        # disk 1 touches row 23 (kept: one row of slack)
    assert got == [(-4.0, 3.0), (14.5, 2.0), (18.0, 4.0)]


@pytest.mark.parametrize("world,k", [(1, 3), (2, 2), (3, 1), (4, 1)])
def test_slabs_in_one_process_reproduce_the_whole_grid(world, k):
    prm, mask, phi0 = _toy()
    steps = 11
    want = _reference(prm, mask, phi0, steps)
    slabs = [slab.Slab(prm, mask, None, r, world, steps_per_exchange=k, margin=1, make_sim=RowModel, device="cpu")
             for r in range(world)]
    for s in slabs:
        s.init(phi0)
    slab.run(slabs, steps)
    got = np.concatenate([s.get()["phi"] for s in slabs], axis=0)
    assert got.shape == want.shape and np.array_equal(got, want)
    assert all(s.t == steps for s in slabs)


def test_too_narrow_a_halo_is_refused_and_a_missing_exchange_shows():
    prm, mask, phi0 = _toy(ny=24)
    with pytest.raises(ValueError):
        slab.Slab(prm, mask, None, 0, 4, steps_per_exchange=2, margin=2, make_sim=RowModel, device="cpu")   # owns 6 < H = 8
    prm, mask, phi0 = _toy()
    slabs = [slab.Slab(prm, mask, None, r, 2, steps_per_exchange=2, margin=1, make_sim=RowModel, device="cpu") for r in range(2)]
    for s in slabs:
        s.init(phi0)
        s.step_local(8)          # no exchange for four times the interval the halo was sized for
    got = np.concatenate([s.get()["phi"] for s in slabs], axis=0)
    assert not np.array_equal(got, _reference(prm, mask, phi0, 8))


def _worker(rank, world, port, out):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    prm, mask, phi0 = _toy()
    s = slab.Slab(prm, mask, None, rank, world, steps_per_exchange=2, margin=1, make_sim=RowModel, device="cpu")
    s.init(phi0)
    slab.run(s, 9, dist)
    dist.barrier()
    out.put((rank, s.y0, s.get()["phi"]))
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_slabs_over_gloo(world):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, 29531 + world, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = sorted((q.get(timeout=180) for _ in ps), key=lambda t: t[0])
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    prm, mask, phi0 = _toy()
    got = np.concatenate([r[2] for r in res], axis=0)
    assert np.array_equal(got, _reference(prm, mask, phi0, 9))


# ---------------------------------------------------------------------------------------------------------------
# GPU: the real contexts
# ---------------------------------------------------------------------------------------------------------------
def _whole(w, precision, schedule, steps, disks):
    s = binding.LBM(binding.LBMParams(precision=precision, schedule=schedule, **w.param_dict()), w.mask, disks)
    s.init(w.phi0)
    s.step(steps)
    f = s.get()
    s.close()
    return f


def _slabbed(w, precision, schedule, steps, disks, world, k):
    prm = binding.LBMParams(precision=precision, schedule=schedule, **w.param_dict())
    slabs = [slab.Slab(prm, w.mask, disks, r, world, steps_per_exchange=k) for r in range(world)]
    for s in slabs:
        s.init(w.phi0)
    slab.run(slabs, steps)
    parts = [s.get() for s in slabs]
    info = (slabs[0].H, slabs[0].nl)
    for s in slabs:
        s.close()
    return {key: np.concatenate([p[key] for p in parts], axis=0) for key in parts[0]}, info


SCHED = [pytest.param(0, id="auto"), pytest.param(binding.SCHEDULE_BASELINE, id="baseline"),
         pytest.param(binding.SCHEDULE_SPARSE, id="sparse"), pytest.param(binding.SCHEDULE_INPLACE, id="inplace")]


def _assert_close(got, want, precision, what):
    # The ghost geometry is computed in the context's own frame: x_F = x_G + n_s and its split into cell
    # and fraction are rounded at the magnitude of the LOCAL row number, so f_y differs from the single-domain value in
    # its last bits, and with it every field, by a few 1e-15 (fp64; in fp32 the fractions are stored as floats).
    tol = 1e-12 if precision == 64 else 2e-6
    scale = {"phi": 1.0, "rho": float(np.abs(want["rho"]).max()), "ux": 1.0, "uy": 1.0, "p": 1.0}
    for key in ("phi", "rho", "ux", "uy", "p"):
        err = float(np.abs(got[key] - want[key]).max())
        assert err <= tol * scale[key], (what, key, err)


@pytest.mark.gpu
@pytest.mark.parametrize("schedule", SCHED)
@pytest.mark.parametrize("precision", [64, 32])
def test_gpu_slabs_mask_only_geometry(schedule, precision):
    """Normals from the mask alone (f2): 2 and 3 slabs against the single-domain run."""
    w = wl.config5(seed=3, n=256)
    steps = 40
    want = _whole(w, precision, schedule, steps, None)
    for world, k in ((2, 4), (3, 2)):
        got, (H, nl) = _slabbed(w, precision, schedule, steps, None, world, k)
        assert H == slab.MASK_ONLY_MARGIN + 3 * k
        _assert_close(got, want, precision, world)


@pytest.mark.gpu
@pytest.mark.parametrize("precision", [64, 32])
def test_gpu_slabs_with_analytic_disks(precision):
    """With a disk list: centres shifted into the local frame, one image per period that touches the local rows."""
    w = wl.config5(seed=5, n=512)
    steps = 60
    want = _whole(w, precision, 0, steps, w.disks)
    got, (H, nl) = _slabbed(w, precision, 0, steps, w.disks, 2, 4)
    assert H == slab.geometry_margin(w.disks) + 12 and nl == 256 + 2 * H
    _assert_close(got, want, precision, "disks")


@pytest.mark.gpu
def test_gpu_slabs_without_exchange_differ():
    w = wl.config5(seed=3, n=256)
    prm = binding.LBMParams(precision=64, **w.param_dict())
    slabs = [slab.Slab(prm, w.mask, None, r, 2, steps_per_exchange=1) for r in range(2)]
    for s in slabs:
        s.init(w.phi0)
        s.step_local(40)
    got = np.concatenate([s.get()["phi"] for s in slabs], axis=0)
    for s in slabs:
        s.close()
    err = float(np.abs(got - _whole(w, 64, 0, 40, None)["phi"]).max())   # what the ends of a local grid make up reaches the owned rows
    assert not err <= 1e-6


@pytest.mark.gpu
def test_rows_export_import_round_trip_and_errors():
    w = wl.config5(seed=1, n=256)
    for schedule in (0, binding.SCHEDULE_FUSED, binding.SCHEDULE_SPARSE, binding.SCHEDULE_BASELINE, binding.SCHEDULE_INPLACE):
        a = binding.LBM(binding.LBMParams(precision=64, schedule=schedule, **w.param_dict()), w.mask, w.disks)
        b = binding.LBM(binding.LBMParams(precision=64, schedule=schedule, **w.param_dict()), w.mask, w.disks)
        a.init(w.phi0); b.init(w.phi0)
        a.step(6); b.step(4 if schedule == binding.SCHEDULE_INPLACE else 3)   # INPLACE: same parity of steps (lbm.h)
        nb = a.rows_bytes(0, w.ny)
        assert nb == sum(a.rows_bytes(j, 32) for j in range(0, w.ny, 32))      # the pieces add up
        buf = torch.empty(nb, dtype=torch.uint8, device="cuda")
        a.rows_export(0, w.ny, buf.data_ptr(), nb)
        b.rows_import(0, w.ny, buf.data_ptr(), nb)                              # b now holds a's state
        a.step(5); b.step(5)
        fa, fb = a.get(), b.get()
        assert all(np.array_equal(fa[k], fb[k]) for k in fa), schedule
        with pytest.raises(binding.LBMError):
            a.rows_bytes(250, 10)                                               # ranges do not wrap
        with pytest.raises(binding.LBMError):
            b.rows_import(0, 16, buf.data_ptr(), nb)                            # size of other rows
        a.close(); b.close()


@pytest.mark.gpu
def test_gpu_slabs_config5_4096_two_slabs():
    """The size of the sweep's middle point (16.8 M nodes, compact planes of several hundred MB): two slabs with the
    analytic disk list against the single-domain run."""
    w = wl.config5(seed=0, n=4096)
    want = _whole(w, 32, 0, 8, w.disks)
    got, (H, nl) = _slabbed(w, 32, 0, 8, w.disks, 2, 4)
    assert nl == 2048 + 2 * H
    _assert_close(got, want, 32, "4096")
