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


def test_bench_gpus_n_starts_n_ranks():
    """`python bench.py --gpus 2` with no WORLD_SIZE in the environment must start 2 ranks itself (the flag
    used to be ignored).  --launch-check runs the launcher and the rank bring-up without the workload (gloo here)."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    res = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--launch-check", "--walkers", "7"],
                         capture_output=True, text=True, env=env, timeout=300)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [json.loads(l) for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, res.stdout                        # rank 0 alone prints
    assert lines[0]["n_gpus"] == 2 and lines[0]["max_ms"] == 11.0 and lines[0]["walkers_total"] == 14.0
    # a world size that contradicts --gpus is refused, not silently run
    env2 = dict(env, WORLD_SIZE="3", RANK="0", LOCAL_RANK="0")
    res = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--launch-check"], capture_output=True, text=True,
                         env=env2, timeout=120)
    assert res.returncode != 0 and "WORLD_SIZE" in res.stderr
