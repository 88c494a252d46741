"""N>1 host logic of bench.py on CPU: world_size-2 gloo processes (the path shards
by patches; this build runs independent replicas, so the only cross-rank step is the max-over-ranks
of the timed duration and the whole-job aggregation)."""
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_0910_5547_b200 import workloads as wl
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, "cpu")          # rank 1 is the slow one
    rate = bench.whole_job_rate(4096 * 8, world, 4, ms)
    # replicas use different seeds: the inputs of the two ranks differ
    G = wl.stress_global(16, seed=20005 + rank)
    t = torch.from_numpy(G[0, 0, 0].copy())
    both = [torch.zeros_like(t) for _ in range(world)]
    dist.all_gather(both, t)
    out.put((rank, ms, rate, bool(torch.equal(both[0], both[1]))))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_gloo_world2():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, rate, same in res:
        assert ms == 15.0                                             # the max, on every rank
        assert rate == 4096 * 8 * 2 * 4 / 15e-3                       # units of all ranks / slowest time
        assert not same


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
