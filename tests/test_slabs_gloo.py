"""Host logic of the y-slab multi-GPU path (paper_2109_12565_b200/slabs.py) on CPU: partition, neighbours, halo row
indices, wall ownership, and the halo exchange itself between two processes over `gloo` (127.0.0.1 rendezvous).
The lattice is stood in for by a [27][ny_local] tensor of "global row id + plane" values, packed and unpacked with
the same row indices the CUDA pack / unpack kernels use (tlb.h "Y-SLABS"); no lattice arithmetic is involved."""
import os
import socket
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2109_12565_b200 import slabs  # noqa: E402


def test_partition_and_neighbours():
    assert slabs.partition(2048, 8) == [(256 * r, 256 * (r + 1)) for r in range(8)]
    assert slabs.partition(10, 3) == [(0, 4), (4, 7), (7, 10)]
    for ny, w in ((2048, 8), (1000, 7), (64, 1), (9, 3)):
        p = slabs.partition(ny, w)
        assert p[0][0] == 0 and p[-1][1] == ny and all(a[1] == b[0] for a, b in zip(p, p[1:]))
        assert max(b - a for a, b in p) - min(b - a for a, b in p) <= 1
    with pytest.raises(ValueError):
        slabs.partition(3, 4)
    assert slabs.neighbours(0, 4, False) == (None, 1) and slabs.neighbours(3, 4, False) == (2, None)
    assert slabs.neighbours(0, 4, True) == (3, 1) and slabs.neighbours(3, 4, True) == (2, 0)
    assert slabs.neighbours(0, 1, False) == (None, None) and slabs.neighbours(0, 1, True) == (0, 0)


def test_layout_halo_rows_and_wall_ownership():
    ny = 40
    (a0, a1), (b0, b1), (c0, c1) = slabs.partition(ny, 3)
    la, lb, lc = (slabs.slab_layout(ny, y0, y1, False) for y0, y1 in ((a0, a1), (b0, b1), (c0, c1)))
    # walls belong to the first and the last slab only: no halo there
    assert (la["halo_lo"], la["halo_hi"]) == (0, 3) and (lb["halo_lo"], lb["halo_hi"]) == (3, 3)
    assert (lc["halo_lo"], lc["halo_hi"]) == (3, 0)
    assert la["ny_local"] == (a1 - a0) + 3 and lb["ny_local"] == (b1 - b0) + 6
    assert lb["y_off"] == b0 - 3 and lb["own0"] == 3 and lb["own1"] == 3 + (b1 - b0)
    # local row r is global row y_off + r; the halo rows of b are the edge rows of a and c
    rb = slabs.local_rows(ny, b0, b1, False)
    assert list(rb[:3]) == [a1 - 3, a1 - 2, a1 - 1] and list(rb[-3:]) == [c0, c0 + 1, c0 + 2]
    pack_hi_a, _ = slabs.face_rows(la, 1)
    _, unpack_lo_b = slabs.face_rows(lb, 0)
    assert list(slabs.local_rows(ny, a0, a1, False)[pack_hi_a]) == list(rb[unpack_lo_b])
    # periodic lattice: every face has a halo and rows wrap
    lp = slabs.slab_layout(ny, a0, a1, True)
    assert (lp["halo_lo"], lp["halo_hi"], lp["y_off"]) == (3, 3, -3)
    assert list(slabs.local_rows(ny, a0, a1, True)[:3]) == [ny - 3, ny - 2, ny - 1]
    with pytest.raises(ValueError):
        slabs.slab_layout(ny, 10, 12, False)  # a neighbour would import 3 of its 2 rows


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, periodic, ny, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch
    import torch.distributed as dist
    from paper_2109_12565_b200 import slabs as S
    dist.init_process_group("gloo", rank=rank, world_size=world)
    y0, y1 = S.partition(ny, world)[rank]
    lay = S.slab_layout(ny, y0, y1, periodic)
    rows = S.local_rows(ny, y0, y1, periodic)
    lo, hi = S.neighbours(rank, world, periodic)
    planes = torch.arange(27, dtype=torch.float64)[:, None] * 1000.0
    ok = True
    for step in range(3):
        # owned rows hold (plane, global row, step); halo rows hold garbage until the exchange
        state = torch.full((27, lay["ny_local"]), -1.0, dtype=torch.float64)
        own = slice(lay["own0"], lay["own1"])
        state[:, own] = planes + torch.as_tensor(rows[own], dtype=torch.float64)[None, :] + 0.001 * step
        send = [None, None]
        recv = [None, None]
        for face, nb in ((0, lo), (1, hi)):
            if nb is not None:
                pack, _ = S.face_rows(lay, face)
                send[face] = state[:, pack].contiguous()
                recv[face] = torch.empty_like(send[face])
        S.exchange(dist, send, recv, lo, hi, rank)
        for face, nb in ((0, lo), (1, hi)):
            if nb is not None:
                _, unpack = S.face_rows(lay, face)
                state[:, unpack] = recv[face]
        expect = planes + torch.as_tensor(rows, dtype=torch.float64)[None, :] + 0.001 * step
        ok = ok and bool(torch.equal(state, expect))
    # the observables' all-reduce: every slab contributes the sum over its owned rows
    part = torch.tensor([float(rows[own].sum()), float(y1 - y0)], dtype=torch.float64)
    dist.all_reduce(part, op=dist.ReduceOp.SUM)
    dist.barrier()
    out.put((rank, ok, part.tolist(), (lay["halo_lo"], lay["halo_hi"])))
    dist.destroy_process_group()


@pytest.mark.parametrize("periodic", [False, True])
def test_halo_exchange_two_ranks_gloo(periodic):
    world, port, ny = 2, _free_port(), 23
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, periodic, ny, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ok, part, halos in res:
        assert ok, "halo rows of rank %d do not hold the neighbour's rows" % rank
        assert part == [float(sum(range(ny))), float(ny)]
    if periodic:
        assert res[0][3] == (3, 3) and res[1][3] == (3, 3)
    else:
        assert res[0][3] == (0, 3) and res[1][3] == (3, 0)  # the walls live on the first / last slab
