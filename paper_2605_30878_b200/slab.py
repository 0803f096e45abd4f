"""1-D slab decomposition along y over the C ABI: host-side plumbing only.

The method is local: a time step moves every population by one node (A16-A17), the gradient
stencil reaches one node (R8) and a ghost node's interpolation cell two more (x_F = x_G + n_s, :66).  So the state
of a row after one step depends on the rows at most THREE away, and a domain cut into slabs along y needs, per cut
and per step, only the rows next to the cut.

Each rank owns the rows [y0, y1) of the global grid and runs an ordinary context (`binding.LBM`, any schedule) on
the rows [y0 - H, y1 + H) (periodic in the global y).  That local grid is periodic in its own height, which is wrong
at its two ends; what is wrong there spreads inwards by three rows per step and never reaches the owned rows if

    H = margin + 3 * steps_per_exchange,

where `margin` rows at each end are given up to the ends' own geometry errors (a disk that straddles one end of the
local grid shows up, through the local periodicity, at the other end: 2 r_max + 2 rows; with normals taken from the
mask alone: the reach of the smoothing and of the stencil, 8 rows).  Every `steps_per_exchange` steps the H halo rows
at each end are overwritten with the neighbour's owned rows next to the cut (`lbm_rows_export` -> send/recv ->
`lbm_rows_import`): one exchange step on the path, pairwise with the two neighbours, no other collective.  The halo
rows are recomputed redundantly between exchanges; wider halos trade that for fewer, larger messages.

Nothing here computes anything of the method: slicing of the inputs, buffer allocation (torch tensors: device memory
and `torch.distributed`, which is plumbing), and the order of the calls.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np
import torch

from . import binding

ROWS_PER_STEP = 3          # how far a row's new state reaches into the old one, in rows (module docstring)
MASK_ONLY_MARGIN = 8       # rows given up at each end of a local grid when the normals come from the mask (f2)


def partition(ny: int, world: int):
    """Owned row ranges [(y0, y1)] of `world` slabs of a grid `ny` rows high, as equal as integers allow."""
    if world < 1 or ny < world:
        raise ValueError("need 1 <= world <= ny")
    return [((ny * r) // world, (ny * (r + 1)) // world) for r in range(world)]


def geometry_margin(disks) -> int:
    """Rows at each end of a local grid whose ghost geometry may be wrong (module docstring)."""
    d = np.asarray(disks, dtype=np.float64).reshape(-1, 3) if disks is not None else np.zeros((0, 3))
    if d.shape[0] == 0:
        return MASK_ONLY_MARGIN
    return 2 * int(math.ceil(float(d[:, 2].max()))) + 2


def halo_rows(margin: int, steps_per_exchange: int) -> int:
    return int(margin) + ROWS_PER_STEP * int(steps_per_exchange)


def local_inputs(ny: int, y0: int, y1: int, H: int, mask, disks, phi0, u0=None):
    """The rows [y0 - H, y1 + H) of the global inputs (periodic in y) and the disks that touch them, in the local
    frame (local row l = global row y0 - H + l).  A disk is listed once per periodic image that intersects the local
    rows; centres may lie outside [0, local ny)."""
    rows = (np.arange(y0 - H, y1 + H)) % ny
    nl = rows.size
    out = {"mask": np.ascontiguousarray(np.asarray(mask)[rows]),
           "phi0": np.ascontiguousarray(np.asarray(phi0, dtype=np.float64)[rows])}
    if u0 is not None:
        out["u0"] = np.ascontiguousarray(np.asarray(u0, dtype=np.float64)[:, rows])
    d = np.asarray(disks, dtype=np.float64).reshape(-1, 3) if disks is not None else np.zeros((0, 3))
    loc = []
    for cx, cy, r in d:
        for m in (-1, 0, 1):
            cyl = cy + m * ny - (y0 - H)
            if cyl + r >= -1.0 and cyl - r <= nl:
                loc.append((cx, cyl, r))
    out["disks"] = np.asarray(loc, dtype=np.float64).reshape(-1, 3)
    return out


@dataclasses.dataclass
class Edges:
    """Device buffers of one exchange: what this slab sends down / up and receives from below / above."""
    send_down: torch.Tensor
    send_up: torch.Tensor
    recv_down: torch.Tensor
    recv_up: torch.Tensor


class Slab:
    """One rank's part of a periodic grid cut into `world` slabs along y.  `make_sim(prm_local, mask, disks)` builds
    the context (default: `binding.LBM` on the current device and stream)."""

    def __init__(self, prm: binding.LBMParams, mask, disks, rank: int, world: int, steps_per_exchange: int = 4,
                 margin: int | None = None, make_sim=None, device=None):
        if prm.wall_rows:
            raise ValueError("slabs are cut from grids that are periodic in y (wall_rows = 0)")
        self.prm, self.rank, self.world = prm, int(rank), int(world)
        self.k = int(steps_per_exchange)
        if self.k < 1:
            raise ValueError("steps_per_exchange must be >= 1")
        self.y0, self.y1 = partition(prm.ny, world)[rank]
        self.margin = geometry_margin(disks) if margin is None else int(margin)
        self.H = halo_rows(self.margin, self.k)
        owned = [b - a for a, b in partition(prm.ny, world)]
        if min(owned) < self.H:
            raise ValueError(f"every slab must own at least H = {self.H} rows (smallest owns {min(owned)})")
        self.n_own = self.y1 - self.y0
        self.nl = self.n_own + 2 * self.H
        self._mask, self._disks = np.asarray(mask).reshape(prm.ny, prm.nx), disks
        li = local_inputs(prm.ny, self.y0, self.y1, self.H, self._mask, disks, np.zeros((prm.ny, 1)))
        self.prm_local = dataclasses.replace(prm, ny=self.nl)
        make_sim = make_sim or (lambda p, m, d: binding.LBM(p, m, d if len(d) else None))
        self.sim = make_sim(self.prm_local, li["mask"], li["disks"])
        self.device = device if device is not None else (torch.device("cuda", torch.cuda.current_device())
                                                         if torch.cuda.is_available() else torch.device("cpu"))
        H, n = self.H, self.n_own
        # rows sent: the owned rows next to each cut; rows received: the halos
        self._rows = {"send_down": H, "send_up": H + n - H, "recv_down": 0, "recv_up": H + n}
        nb = {k: self.sim.rows_bytes(j0, H) for k, j0 in self._rows.items()}
        self.edges = Edges(**{k: torch.empty(max(b, 1), dtype=torch.uint8, device=self.device) for k, b in nb.items()})
        self._nb = nb
        self.t = 0

    # ---- inputs and outputs in the global frame ----
    def init(self, phi0, u0=None):
        li = local_inputs(self.prm.ny, self.y0, self.y1, self.H, self._mask, self._disks,
                          np.asarray(phi0, dtype=np.float64).reshape(self.prm.ny, self.prm.nx),
                          None if u0 is None else np.asarray(u0, dtype=np.float64).reshape(2, self.prm.ny, self.prm.nx))
        self.sim.init(li["phi0"], li.get("u0"))
        self.t = 0

    def get(self):
        """Fields of the owned rows, shaped (n_own, nx)."""
        f = self.sim.get()
        return {k: np.ascontiguousarray(np.asarray(v).reshape(self.nl, self.prm.nx)[self.H:self.H + self.n_own])
                for k, v in f.items()}

    # ---- the exchange step, split so that one process can drive several slabs (tests) or one (torch.distributed) ----
    def pack(self):
        e = self.edges
        self.sim.rows_export(self._rows["send_down"], self.H, e.send_down.data_ptr(), self._nb["send_down"])
        self.sim.rows_export(self._rows["send_up"], self.H, e.send_up.data_ptr(), self._nb["send_up"])

    def unpack(self):
        e = self.edges
        self.sim.rows_import(self._rows["recv_down"], self.H, e.recv_down.data_ptr(), self._nb["recv_down"])
        self.sim.rows_import(self._rows["recv_up"], self.H, e.recv_up.data_ptr(), self._nb["recv_up"])

    def step_local(self, n: int):
        self.sim.step(int(n))
        self.t += int(n)

    def close(self):
        self.sim.close()


def exchange_in_process(slabs):
    """All slabs of the grid live in this process (one GPU driving them one after the other, or the CPU tests):
    the neighbour's send buffer is copied into the receive buffer."""
    w = len(slabs)
    for s in slabs:
        s.pack()
    for r, s in enumerate(slabs):
        below, above = slabs[(r - 1) % w], slabs[(r + 1) % w]
        s.edges.recv_down.copy_(below.edges.send_up, non_blocking=True)
        s.edges.recv_up.copy_(above.edges.send_down, non_blocking=True)
    for s in slabs:
        s.unpack()


def exchange_distributed(slab: Slab, dist=None):
    """One slab per process: pairwise send/recv with the two neighbours (NCCL on device buffers, gloo on host
    buffers), no other collective.  With two ranks both neighbours are the same peer: the order of the operations
    (up first) pairs its upper edge with this slab's lower halo."""
    if dist is None:
        import torch.distributed as dist
    w, r, e = slab.world, slab.rank, slab.edges
    slab.pack()
    if w == 1:
        e.recv_down.copy_(e.send_up, non_blocking=True)
        e.recv_up.copy_(e.send_down, non_blocking=True)
    else:
        below, above = (r - 1) % w, (r + 1) % w
        ops = [dist.P2POp(dist.isend, e.send_up, above), dist.P2POp(dist.isend, e.send_down, below),
               dist.P2POp(dist.irecv, e.recv_down, below), dist.P2POp(dist.irecv, e.recv_up, above)]
        for req in dist.batch_isend_irecv(ops):
            req.wait()
    slab.unpack()


def run(slabs, nsteps: int, dist=None):
    """Advances the whole grid by `nsteps`: exchange, then at most steps_per_exchange local steps, repeated.
    `slabs`: every slab of the grid (one process), or this rank's `Slab` (torch.distributed)."""
    single = isinstance(slabs, Slab)
    k = slabs.k if single else slabs[0].k
    done = 0
    while done < nsteps:
        if single:
            exchange_distributed(slabs, dist)
        else:
            exchange_in_process(slabs)
        m = min(k, nsteps - done)
        for s in ([slabs] if single else slabs):
            s.step_local(m)
        done += m
