"""CPU, world_size 2, gloo: the N > 1 path of bench.py.  The hot path shards by sequence with no
exchange: every rank draws its own batch, the job time is the MAX over
ranks and the units processed the SUM.  Also: --impl reference under torchrun prints on rank 0 only."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from workloads import generators as gen
    w = gen.config(1, scale=1 / 64, batch=2, seed=bench.rank_seed(rank))      # this rank's shard
    toks = bench.eligible_tokens(w)
    ms = 10.0 + 5.0 * rank                                                     # rank 1 is the slow one
    ms_max, toks_all = bench.reduce_over_ranks(ms, toks)
    q.put((rank, toks, ms_max, toks_all, float(w.q.float().abs().sum())))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_shard_without_exchange():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, t0, m0, a0, s0), (r1, t1, m1, a1, s1) = res
    assert m0 == m1 == 15.0                       # MAX over ranks
    assert a0 == a1 == t0 + t1                    # SUM of the units all ranks processed
    assert s0 != s1                               # different seeds: independent shards, nothing shared


def test_reference_arm_prints_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert out.returncode == 0 and out.stdout.strip() == ""
