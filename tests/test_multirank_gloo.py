"""Host-side logic of the N > 1 path (DESIGN.md §8 "replicas only"), world_size 2 over gloo on CPU:
every rank builds its OWN event (own seed), the job time is the max over ranks and the job's work the sum."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ev = bench.make_event(0, rank, world)                       # configs[0]-like event with this rank's seed
    ms, e2e, tot = bench.reduce_over_ranks(10.0 + 5.0 * rank, 20.0 - 3.0 * rank, ev.n, world, torch.device("cpu"))
    out[rank] = (ev.n, float(ev.y[:8].sum()), ms, e2e, tot)
    dist.destroy_process_group()


def test_two_rank_replicas_reduce_max_time_and_sum_work():
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    port = 29500 + (os.getpid() % 2000)
    mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
    (n0, s0, ms0, e0, t0), (n1, s1, ms1, e1, t1) = out[0], out[1]
    assert (n0, s0) != (n1, s1), "ranks must track different Time Frames (own seeds)"
    assert ms0 == ms1 == 15.0 and e0 == e1 == 20.0, "job time = max over ranks"
    assert t0 == t1 == float(n0 + n1), "job work = sum of the ranks' clusters"


def test_single_rank_needs_no_process_group():
    import bench
    assert bench.reduce_over_ranks(3.0, 4.0, 7, 1, None) == (3.0, 4.0, 7.0)
