"""Host-side logic of the N > 1 path on CPU (gloo, world_size 2): ranks take disjoint, differently seeded groups and
the only collective is the max-over-ranks of the timing.  No GPU, no CUDA library call."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import synth
    ids = bench.rank_group_ids(2, rank)
    grp = synth.make_group(2, ids[0], n_sci=1, n_master=1, geom=synth.GEOM_SMALL)
    gathered = [None] * world
    dist.all_gather_object(gathered, (ids, int(grp.sci.astype("int64").sum())))
    mx = bench.max_over_ranks(10.0 + rank)
    if rank == 0:
        out.put((gathered, mx))
    dist.destroy_process_group()


def test_two_ranks_disjoint_groups_and_max_timing():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    gathered, mx = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (ids0, sum0), (ids1, sum1) = gathered
    assert len(ids0) == len(ids1) == 3 and not set(ids0) & set(ids1)      # config 2: 3 groups per rank, disjoint
    assert sum0 != sum1                                                    # differently seeded data
    assert mx == 11.0                                                      # max over ranks of (10, 11)


def test_single_process_max_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5) == 3.5
