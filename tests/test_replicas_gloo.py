"""The N > 1 path of bench.py ("replicas only": no data-path collective) on CPU: two processes, gloo
backend, 127.0.0.1 rendezvous.  Checks the per-rank seeds and the whole-job aggregation (sum of site
updates over the max-over-ranks time)."""
import os
import socket
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch.distributed as dist
    from paper_2109_12565_b200 import replicas
    import inputs
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = inputs.config(1)
    seed = replicas.rank_seed(cfg["seed"], rank)
    centres = inputs.place_droplets(cfg["nx"], cfg["ny"], seed, 12, 6.0, 4.0)
    ms = 2.0 + rank  # rank 1 is the slow one
    mlups, ms_max = replicas.aggregate_mlups(cfg["nx"] * cfg["ny"], 10, ms)
    dist.barrier()
    out.put((rank, seed, float(centres[0, 0]), mlups, ms_max))
    dist.destroy_process_group()


def test_two_replicas_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, s0, c0, m0, t0), (r1, s1, c1, m1, t1) = res
    assert (r0, r1) == (0, 1) and s0 != s1 and c0 != c1      # different replicas
    assert t0 == t1 == 3.0                                    # max over ranks
    expect = 2 * 128 * 64 * 10 / 3.0 / 1e3                    # all ranks' updates over the slowest time
    assert abs(m0 - expect) < 1e-12 and m0 == m1
