"""N>1 host logic on CPU (gloo, world_size 2): walker sharding has no data-path collective; only the timing
max-reduction and the aggregate count cross ranks."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2202_00832_b200.dist import max_over_ranks, sum_over_ranks, walker_shard


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
    try:
        import gen
        import oracle
        P = gen.make_problem(0)
        phis = gen.make_walkers(P)
        lo_, hi = walker_shard(P.n_w, rank, world)
        # each rank evaluates its own walker range (here with the oracle: no GPU on this box); no exchange of data
        e = [oracle.local_energy_exact(P.h, P.L, P.psi, [phis[0][w]], "cholesky")[0] for w in range(lo_, hi)]
        t_ms = 10.0 + rank            # pretend timings: the job time is the max over ranks
        job_ms = max_over_ranks(t_ms)
        total = sum_over_ranks(hi - lo_)
        dist.barrier()
        q.put((rank, lo_, hi, [complex(x) for x in e], job_ms, total))
    finally:
        dist.destroy_process_group()


def test_two_rank_walker_sharding():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    import gen
    import oracle
    P = gen.make_problem(0)
    phis = gen.make_walkers(P)
    ref = [oracle.local_energy_exact(P.h, P.L, P.psi, [phis[0][w]], "cholesky")[0] for w in range(P.n_w)]
    got = [x for r in res for x in r[3]]
    assert np.array_equal(np.array(got), np.array(ref))          # shards tile the batch, same numbers
    assert all(r[4] == 11.0 for r in res) and all(r[5] == P.n_w for r in res)
