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


# ---------------------------------------------------------------- patch sharding: the plans of two ranks meet (NEXT-2)
def _shard_worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_0910_5547_b200 import sharding, workloads as wl
    h = wl.uniform_hierarchy(4, periodic=True)
    plan = sharding.rank_plan(h, world, rank)                          # every rank builds its own shard only
    peer = 1 - rank
    # a host stand-in for the slab buffers: one number per slab that names it (global patch * 8 + face), in plan order;
    # exchange step (1) of SURVEY 8(e) as send/recv, step (2) as all_reduce(max) of one scalar
    glob = plan["glob"]
    send = torch.tensor([int(glob[p]) * 8 + int(f) for p, f in plan["send"][peer]], dtype=torch.int64)
    recv = torch.zeros(len(plan["recv"][peer]), dtype=torch.int64)
    if rank == 0:
        dist.send(send, dst=peer); dist.recv(recv, src=peer)
    else:
        dist.recv(recv, src=peer); dist.send(send, dst=peer)
    want = torch.tensor([int(glob[p]) * 8 + int(f) for p, f in plan["recv"][peer]], dtype=torch.int64)
    smax = torch.tensor([1.0 + rank], dtype=torch.float64)
    dist.all_reduce(smax, op=dist.ReduceOp.MAX)
    # every slab received lands in a mirror patch, every slab sent comes from an owned one, every owned face is served
    ok_roles = all(p >= plan["owned"] for p, _ in plan["recv"][peer]) and all(p < plan["owned"] for p, _ in plan["send"][peer])
    nbr = plan["hier"]["nbr"]
    served = all(nbr[p, sharding.FACE_REGION[f]] >= 0 for p in range(plan["owned"]) for f in range(6))
    out.put((rank, bool(torch.equal(recv, want)), float(smax.item()), ok_roles, served, plan["owned"], len(recv)))
    dist.barrier()
    dist.destroy_process_group()


def test_sharding_plans_of_two_gloo_ranks_match():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_shard_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert sum(r[5] for r in res) == 64
    for rank, same, smax, roles, served, owned, nrecv in res:
        assert same and smax == 2.0 and roles and served and nrecv > 0


def test_partitioner_properties():
    from paper_0910_5547_b200 import sharding, workloads as wl
    import pytest
    h = wl.uniform_hierarchy(4, periodic=True)
    for ns in (1, 2, 3, 5, 8, 64):
        R = sharding.partition_morton(h, ns)
        assert R[0][0] == 0 and R[-1][1] == 64 and all(a[1] == b[0] for a, b in zip(R, R[1:]))
        sizes = [hi - lo for lo, hi in R]
        assert max(sizes) - min(sizes) <= 1
        S = [sharding.build_shard(h, R, s) for s in range(ns)]
        for s in range(ns):
            for t, v in S[s]["send_global"].items():
                assert v == S[t]["recv_global"][s]
            assert sorted(S[s]["send"]) == sorted(S[s]["send_global"])
    # Morton ranges are compact: with 8 shards of a 4^3 level every shard is a 2^3 cube with 24 face-neighbour mirrors
    S = sharding.build_shard(h, sharding.partition_morton(h, 8), 3)
    assert S["owned"] == 8 and len(S["glob"]) == 32
    with pytest.raises(ValueError):
        sharding.partition_morton(wl.ball_hierarchy(2, 2), 2)
    with pytest.raises(ValueError):
        sharding.partition_morton(h, 65)


def test_zstrip_table_order_is_consistent():
    """workloads.build_hierarchy(order="zstrip"): the launch order of the single-level bench workloads.  Any order is a valid
    table; check the neighbour entries against the block coordinates and the order itself (strips of 8 rows, z outermost)."""
    import numpy as np
    from paper_0910_5547_b200 import workloads as wl
    nb = (6, 16, 4)
    h = wl.build_hierarchy(nb, (), (0,) * 6, order="zstrip")
    B = np.asarray(h["blocks"]); n = len(B)
    assert n == 6 * 16 * 4 and len({tuple(b) for b in B}) == n
    index = {tuple(int(c) for c in b): i for i, b in enumerate(B)}
    for i in (0, 17, n // 2, n - 1):
        for r in range(27):
            d = (r % 3 - 1, (r // 3) % 3 - 1, r // 9 - 1)
            q = tuple((int(B[i][a]) + d[a]) % nb[a] for a in range(3))
            assert h["nbr"][i][r] == index[q]
    key = [((b[1] // wl.ZSTRIP_ROWS) * nb[2] + b[2], b[1] % wl.ZSTRIP_ROWS, b[0]) for b in B]
    assert key == sorted(key)
    assert [tuple(b) for b in B[:7]] == [(0, 0, 0), (1, 0, 0), (2, 0, 0), (3, 0, 0), (4, 0, 0), (5, 0, 0), (0, 1, 0)]
    assert tuple(B[6 * wl.ZSTRIP_ROWS]) == (0, 0, 1)                     # after one z-layer of the first strip: up in z
    try:
        wl.build_hierarchy(nb, (), (0,) * 6, order="spiral")
        assert False
    except ValueError:
        pass
