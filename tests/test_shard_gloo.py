"""Multi-GPU path = independent replicas on disjoint frame ranges (DESIGN.md
"Multi-GPU"): no data-path collective.  The host-side pieces bench.py uses for
N > 1 (rank-offset frame selection, max-over-ranks timing reduction) are
covered here with a world_size-2 gloo group on CPU."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2310_08770_b200 import workloads as wl
    cfg = wl.config(1)
    idx = (np.arange(8) + rank * 7919) % cfg.n_frames        # bench.py's per-rank frame choice
    fr = wl.frames(cfg, idx)
    t = torch.tensor([float(10 + rank)], dtype=torch.float64)  # a per-rank "step time"
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    chk = torch.tensor([float(fr.astype(np.uint64).sum())], dtype=torch.float64)
    gathered = [torch.zeros_like(chk) for _ in range(world)]
    dist.all_gather(gathered, chk)
    q.put((rank, float(t[0]), [float(g[0]) for g in gathered], idx.tolist()))
    dist.destroy_process_group()


def test_two_rank_replicas_disjoint_frames_and_max_timing():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][1] == res[1][1] == 11.0                 # max over ranks
    assert set(res[0][3]).isdisjoint(res[1][3])           # disjoint frame ranges
    assert res[0][2] == res[1][2] and res[0][2][0] != res[0][2][1]
