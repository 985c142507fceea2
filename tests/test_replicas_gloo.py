"""Multi-GPU mode is "replicas only": sources are sharded over ranks with no collective on the
data path, results are gathered on the host.  The N>1 plumbing is covered here with world_size 2 on CPU (gloo);
the per-rank solver is the oracle (the CUDA library needs a GPU), which exposes the same Grid.run interface."""
import os
import sys

import numpy as np
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    os.environ["OMP_NUM_THREADS"] = "2"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from helpers import make_grid
    from oracle import emm_oracle
    from paper_2304_00233_b200 import emm, workloads as W
    w = W.cfg1(n=14, dx=100.0, rd=1, nb=3)
    srcs = [((650.0 + 40 * i, 700.0, 700.0 - 30 * i), (1.0, 0.2 * i, 0.0)) for i in range(5)]
    g = make_grid(emm_oracle, w)
    full, steps = emm.run_replicated(g, srcs, w["freqs"], w["receivers"][:3], dict(fixed_steps=30))
    if rank == 0:
        q.put((emm.shard_sources(5, 0, world), emm.shard_sources(5, 1, world), full, steps))
    dist.barrier()
    dist.destroy_process_group()


def test_sources_are_sharded_over_two_ranks_and_gathered(oracle):
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from helpers import make_grid
    from paper_2304_00233_b200 import workloads as W
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    s0, s1, full, steps = q.get(timeout=300)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert s0 == [0, 2, 4] and s1 == [1, 3]
    # the gathered result equals a single-process run of all five sources
    w = W.cfg1(n=14, dx=100.0, rd=1, nb=3)
    srcs = [((650.0 + 40 * i, 700.0, 700.0 - 30 * i), (1.0, 0.2 * i, 0.0)) for i in range(5)]
    ref, nref = make_grid(oracle, w).run(srcs, w["freqs"], w["receivers"][:3], dict(fixed_steps=30))
    assert list(steps) == list(nref) == [30] * 5
    assert np.array_equal(full, ref)
