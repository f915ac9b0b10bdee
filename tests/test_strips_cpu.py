"""Host-side logic of the strip decomposition (paper_1805_01443_b200/strips.py): the row
partition, the strips' parameters, and the halo exchange between ranks with torch.distributed (gloo,
world_size 2 and 3, CPU tensors standing in for the workspace rows)."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1805_01443_b200 import strips, workloads as W


def test_split_rows_and_strip_params():
    assert strips.split_rows(10, 3) == [(0, 4), (4, 7), (7, 10)]
    assert strips.split_rows(8, 1) == [(0, 8)]
    with pytest.raises(ValueError):
        strips.split_rows(2, 3)
    p, _ = W.disc(64, 3)
    rows = strips.split_rows(64, 4)
    qs = [strips.strip_params(p, j0, j1, r, 4) for r, (j0, j1) in enumerate(rows)]
    assert [q["ny"] for q in qs] == [16] * 4
    assert qs[0]["y0"] == p["y0"] and qs[-1]["y1"] == p["y1"]
    for a, b in zip(qs[:-1], qs[1:]):
        assert a["y1"] == b["y0"]                           # strips tile the domain without gaps
    assert [(q["halo_south"], q["halo_north"]) for q in qs] == [(0, 1), (1, 1), (1, 1), (1, 0)]   # frozen box edge
    pv, _ = W.vortex(8, 2)
    qv = [strips.strip_params(pv, j0, j1, r, 2) for r, (j0, j1) in enumerate(strips.split_rows(8, 2))]
    assert [(q["halo_south"], q["halo_north"]) for q in qv] == [(1, 1), (1, 1)]                   # periodic: wraps
    assert strips.neighbours(0, 2, True) == (1, 1) and strips.neighbours(0, 3, False) == (None, 1)
    assert strips.strip_params(pv, 0, 8, 0, 1)["halo_south"] == 0                                  # one strip: plain bc


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, n, periodic, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=n)
    try:
        first = torch.full((7,), 10.0 * rank + 1.0, dtype=torch.float64)     # this strip's first row
        last = torch.full((7,), 10.0 * rank + 2.0, dtype=torch.float64)      # ... and last row
        hs = torch.full((7,), -1.0, dtype=torch.float64)
        hn = torch.full((7,), -1.0, dtype=torch.float64)
        for _ in range(3):                                                   # repeated exchanges stay matched
            strips.exchange_rows(first, last, hs, hn, rank, n, periodic, dist)
        out[rank] = (float(hs[0]), float(hn[0]))
        t = torch.tensor([0.1 * (rank + 1)], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MIN)
        assert abs(float(t) - 0.1) < 1e-15
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n,periodic", [(2, False), (2, True), (3, True), (3, False)])
def test_halo_exchange_between_ranks(n, periodic):
    """Every rank ends up with its south neighbour's last row in the south halo and its north neighbour's first
    row in the north halo; domain edges keep their sentinel."""
    port = _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(n, periodic, port, out), nprocs=n, join=True)
        res = dict(out)
    for r in range(n):
        south, north = strips.neighbours(r, n, periodic)
        exp_s = 10.0 * south + 2.0 if south is not None else -1.0
        exp_n = 10.0 * north + 1.0 if north is not None else -1.0
        assert res[r] == (exp_s, exp_n), (r, res[r])


def _group_worker(rank, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=3)
    try:
        grp = dist.new_group([0, 2])                        # strips live on global ranks 0 and 2 (group ranks 0, 1)
        if rank in (0, 2):
            gr = dist.get_rank(grp)
            first = torch.full((5,), 10.0 * gr + 1.0, dtype=torch.float64)
            last = torch.full((5,), 10.0 * gr + 2.0, dtype=torch.float64)
            hs = torch.full((5,), -1.0, dtype=torch.float64)
            hn = torch.full((5,), -1.0, dtype=torch.float64)
            strips.exchange_rows(first, last, hs, hn, gr, 2, False, dist, grp)
            out[rank] = (float(hs[0]), float(hn[0]))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_halo_exchange_in_a_sub_group_uses_global_ranks():
    """P2POp peers are global ranks: a decomposition over a sub-group (global ranks 0 and 2 of 3) must translate its
    group-local neighbour ranks."""
    port = _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_group_worker, args=(port, out), nprocs=3, join=True)
        res = dict(out)
    assert res[0] == (-1.0, 11.0) and res[2] == (2.0, -1.0), res


def test_overlap_plumbing_order_on_host():
    """Without a compute stream (host tensors) the three phases of a sub-step run in order: exchange, interior, edges."""
    calls = []
    strips._Overlap(None).run(lambda: calls.append("x"), lambda: calls.append("i"), lambda: calls.append("e"))
    assert calls == ["x", "i", "e"]
