"""Domain decomposition along y into strips of whole cell rows (the paper's
"one sub-domain per GPU ... one layer of ghost cells per side").

Argument marshalling and plumbing only: every strip is an ordinary ``DG`` context whose south / north edge is
marked as a halo edge (``halo_south`` / ``halo_north`` in ``dg_params``); before every RK sub-step the first
and last row of the array the stage kernel is about to read travel to the neighbours' halo rows (one
contiguous run of 4 m^2 x 8 bytes per cell, in the kernels' own layout: no packing), and the stage kernel
fetches those rows by TMA exactly like rows of its own strip.  The time step is the minimum over the strips
(the paper's global CFL reduction), the torque of Eq.(6) the sum.

* ``LocalStrips``  -- all strips in one process on one GPU, rows exchanged by device-to-device copies on the
                     contexts' stream.  Same arithmetic as the undivided domain: the test compares bitwise.
* ``DistStrip``    -- one strip per rank (one process per GPU), rows exchanged with ``torch.distributed``
                     point-to-point operations (NCCL over NVLink on GPUs; gloo in the CPU test of the exchange
                     logic), dt by all_reduce(MIN), torque by all_reduce(SUM).
"""
from __future__ import annotations


def split_rows(ny: int, n: int):
    """Balanced partition of ny rows into n strips: list of (j0, j1)."""
    if not 1 <= n <= ny:
        raise ValueError("need 1 <= strips <= ny")
    base, extra = divmod(ny, n)
    out, j = [], 0
    for r in range(n):
        k = base + (1 if r < extra else 0)
        out.append((j, j + k))
        j += k
    return out


def strip_params(p: dict, j0: int, j1: int, rank: int, n: int) -> dict:
    """``dg_params`` of strip ``rank`` of ``n``: its rows, its y-range, and which edges are halo edges."""
    dy = (p["y1"] - p["y0"]) / p["ny"]
    periodic = p["bc"] == 0
    q = dict(p)
    q.update(ny=j1 - j0, y0=p["y0"] + j0 * dy, y1=p["y0"] + j1 * dy,
             halo_south=1 if (rank > 0 or (periodic and n > 1)) else 0,
             halo_north=1 if (rank < n - 1 or (periodic and n > 1)) else 0)
    return q


def neighbours(rank: int, n: int, periodic: bool):
    """(south, north) neighbour ranks or None."""
    south = rank - 1 if rank > 0 else (n - 1 if periodic and n > 1 else None)
    north = rank + 1 if rank < n - 1 else (0 if periodic and n > 1 else None)
    return south, north


def exchange_rows(first, last, halo_south, halo_north, rank: int, n: int, periodic: bool, dist, group=None):
    """One halo exchange of a strip with ``torch.distributed`` point-to-point operations: ``first`` goes to the
    south neighbour's north halo, ``last`` to the north neighbour's south halo.  Tensors may live on any device
    the backend supports; returns after the transfers completed."""
    south, north = neighbours(rank, n, periodic)
    if group is not None:                       # P2POp peers are global ranks
        south = None if south is None else dist.get_global_rank(group, south)
        north = None if north is None else dist.get_global_rank(group, north)
    # one fixed order on every rank -- southward traffic first, then northward -- so that the k-th message a rank
    # sends to a peer is the k-th it expects from it even when both neighbours are the same rank (2 periodic strips)
    ops = []
    if south is not None:
        ops.append(dist.P2POp(dist.isend, first, south, group))
    if north is not None:
        ops.append(dist.P2POp(dist.irecv, halo_north, north, group))
        ops.append(dist.P2POp(dist.isend, last, north, group))
    if south is not None:
        ops.append(dist.P2POp(dist.irecv, halo_south, south, group))
    for req in (dist.batch_isend_irecv(ops) if ops else []):
        req.wait()


class _Overlap:
    """Stream plumbing shared by both strip drivers: the halo exchange of a sub-step runs on a side stream, ordered
    after everything the compute stream has done so far, while the compute stream launches the interior row
    segments (`dg_substep_part(0)`); the edge segments (`dg_substep_part(1)`) wait for the exchange."""

    def __init__(self, compute_stream):
        import torch
        self.torch = torch
        self.compute = compute_stream
        self.comm = torch.cuda.Stream(device=compute_stream.device) if compute_stream is not None else None

    def run(self, exchange, interior, edges):
        if self.comm is None:                    # host tensors (the gloo test of the exchange logic): no streams
            exchange()
            interior()
            edges()
            return
        torch = self.torch
        self.comm.wait_stream(self.compute)      # the rows to send were written by earlier kernels of the compute stream
        with torch.cuda.stream(self.comm):
            exchange()
        with torch.cuda.stream(self.compute):
            interior()
            self.compute.wait_stream(self.comm)  # halo rows have arrived
            edges()


class LocalStrips:
    """All strips of a decomposed domain as separate contexts on the current device (one compute stream)."""

    def __init__(self, DG, params: dict, n: int):
        self.p = dict(params)
        self.n = n
        self.rows = split_rows(params["ny"], n)
        self.periodic = params["bc"] == 0
        self.ctx = [DG(strip_params(params, j0, j1, r, n)) for r, (j0, j1) in enumerate(self.rows)]
        self.ov = _Overlap(self.ctx[0].stream)

    def set_state(self, U_dev):
        for g, (j0, j1) in zip(self.ctx, self.rows):
            g.set_state(U_dev[j0:j1].contiguous())

    def get_state(self):
        import torch
        return torch.cat([g.get_state() for g in self.ctx], dim=0)

    def exchange(self):
        """Fill every halo row from the neighbour strip's boundary row of the array its next kernel reads (device
        copies on whatever stream is current: `step` and `rhs` order them against the kernels)."""
        views = [g.halo_rows() for g in self.ctx]
        for r in range(self.n):
            south, north = neighbours(r, self.n, self.periodic)
            (_, _), (hs, hn) = views[r]
            if south is not None:
                hs.copy_(views[south][0][1])          # the south neighbour's last row
            if north is not None:
                hn.copy_(views[north][0][0])          # the north neighbour's first row

    def cfl_dt(self, cfl: float) -> float:
        return min(g.cfl_dt(cfl) for g in self.ctx)

    def step(self, dt: float):
        for g in self.ctx:
            g.step_begin(dt)
        for _ in range(self.ctx[0].rk_stages):
            self.ov.run(self.exchange,
                        lambda: [g.substep_part(0) for g in self.ctx],
                        lambda: [g.substep_part(1) for g in self.ctx])
        for g in self.ctx:
            g.step_end()

    def rhs(self, t: float):
        import torch
        with torch.cuda.stream(self.ctx[0].stream):
            self.exchange()
        return torch.cat([g.rhs(t) for g in self.ctx], dim=0)

    def torque(self, t: float) -> float:
        return sum(g.torque(t) for g in self.ctx)

    @property
    def time(self) -> float:
        return self.ctx[0].time


class DistStrip:
    """This rank's strip of a domain decomposed over the ranks of a ``torch.distributed`` group."""

    def __init__(self, DG, params: dict, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.rank, self.n = dist.get_rank(group), dist.get_world_size(group)
        self.periodic = params["bc"] == 0
        self.rows = split_rows(params["ny"], self.n)
        self.j0, self.j1 = self.rows[self.rank]
        self.g = DG(strip_params(params, self.j0, self.j1, self.rank, self.n))
        self.ov = _Overlap(self.g.stream)

    def set_state(self, U_dev_local):
        self.g.set_state(U_dev_local)

    def exchange(self):
        """One halo exchange (NCCL point-to-point operations are ordered against the stream that is current when they
        are issued: `step` issues them on the side stream)."""
        (first, last), (hs, hn) = self.g.halo_rows()
        exchange_rows(first, last, hs, hn, self.rank, self.n, self.periodic, self.dist, self.group)

    def cfl_dt(self, cfl: float) -> float:
        import torch
        t = torch.tensor([self.g.cfl_dt(cfl)], dtype=torch.float64, device=self.g.workspace.device)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MIN, group=self.group)
        return float(t.item())

    def step(self, dt: float):
        self.g.step_begin(dt)
        for _ in range(self.g.rk_stages):
            self.ov.run(self.exchange, lambda: self.g.substep_part(0), lambda: self.g.substep_part(1))
        self.g.step_end()

    def torque(self, t: float) -> float:
        import torch
        x = torch.tensor([self.g.torque(t)], dtype=torch.float64, device=self.g.workspace.device)
        self.dist.all_reduce(x, op=self.dist.ReduceOp.SUM, group=self.group)
        return float(x.item())
