"""Patch sharding of a single-level hierarchy over several pools / GPUs.

PAPER.md:363-373: "a grid is the basic unit" of both the GPU work and the distribution over nodes; within a stage every
patch is independent, so the path shards by patches.  This module is the host bookkeeping of that (no method
arithmetic): a Morton-range partitioner, per-shard descriptor tables (owned patches first, then mirror copies of the
face neighbours that other shards own), and the halo plans that pair a sender's (patch, face) slabs with the receiver's
mirror patches.  The device side is `amrhydro_set_owned / set_halo_plan / halo_pack / halo_unpack`
(include/amrhydro.h, kernel k_halo_slabs).  Exchange steps of 8(e): (1) face halos before every stage, (2) one
max-reduction of the signal speed per step; (3), parent-child traffic of refined levels, is not built.

`ShardedRun` drives the shards of ONE process (all pools on the visible GPU; the peer copy is a device-to-device
copy): that is the single-GPU stand-in the tests use to require bitwise equality with the unsharded run.  With one
process per GPU the same plans apply: each rank builds only its own shard, sends `send[peer]` with ncclSend / a
peer store and all-reduces the signal speed (`rank_plan`, tests/test_multirank_host.py checks the plans of two
gloo ranks against each other).
"""
import numpy as np

FACE_REGION = (12, 14, 10, 16, 4, 22)   # x-lo x-hi y-lo y-hi z-lo z-hi in the 27-entry neighbour table
NBR_REMOTE = -3


def partition_morton(hier, nshards):
    """Contiguous ranges [lo, hi) of the table (which is Morton-ordered, workloads.build_hierarchy) with patch counts
    that differ by at most one.  Returns a list of (lo, hi)."""
    if hier["nlevels"] != 1:
        raise ValueError("sharding is built for single-level hierarchies")
    n = int(hier["level"].shape[0])
    if not 1 <= nshards <= n:
        raise ValueError("need 1 <= nshards <= number of patches")
    cuts = [(n * s) // nshards for s in range(nshards + 1)]
    return [(cuts[s], cuts[s + 1]) for s in range(nshards)]


def owner_of(ranges, p):
    for s, (lo, hi) in enumerate(ranges):
        if lo <= p < hi:
            return s
    raise ValueError("patch %d is in no range" % p)


def build_shard(hier, ranges, s):
    """Shard s: local hierarchy dict (owned patches in global order, then mirrors in global order), the global index of
    every local patch, and per peer the send / receive plans as (local patch, face) rows.

    A slab (q, f) = the two interior layers of patch q next to its face f.  For an owned patch p whose face-f neighbour q
    lives on shard t != s, the cells p reads are q's layers next to q's opposite face, slab (q, f ^ 1).  Both sides
    enumerate these pairs sorted by (global q, face), so the sender's buffer is the receiver's buffer."""
    lo, hi = ranges[s]
    nbr = np.asarray(hier["nbr"])
    owned = list(range(lo, hi))
    need = {}                                   # peer -> set of (global q, face of q)
    for p in owned:
        for f in range(6):
            q = int(nbr[p, FACE_REGION[f]])
            if q >= 0 and not lo <= q < hi:
                need.setdefault(owner_of(ranges, q), set()).add((q, f ^ 1))
    give = {}                                   # peer -> set of (global p, face of p) this shard owns and the peer reads
    for t, (tlo, thi) in enumerate(ranges):
        if t == s:
            continue
        for p in range(tlo, thi):
            for f in range(6):
                q = int(nbr[p, FACE_REGION[f]])
                if lo <= q < hi:
                    give.setdefault(t, set()).add((q, f ^ 1))
    mirrors = sorted({q for v in need.values() for q, _ in v})
    glob = np.array(owned + mirrors, dtype=np.int64)
    local = {int(g): i for i, g in enumerate(glob)}
    n = len(glob)
    lnbr = np.full((n, 27), NBR_REMOTE, np.int32)
    for i, g in enumerate(glob):
        for r in range(27):
            q = int(nbr[g, r])
            # physical boundaries stay; a neighbour that is in this pool gets its local index; any other is REMOTE
            lnbr[i, r] = q if q < 0 else local.get(q, NBR_REMOTE)
    h = dict(level=np.zeros(n, np.int32), origin=np.asarray(hier["origin"])[glob].astype(np.int32),
             parent=np.full(n, -1, np.int32), nbr=lnbr, nlevels=1, dx0=hier["dx0"], bc=np.asarray(hier["bc"], np.int32),
             blocks=np.asarray(hier["blocks"])[glob], base_blocks=hier["base_blocks"])
    send = {t: np.array([(local[q], f) for q, f in sorted(v)], np.int32).reshape(-1, 2) for t, v in sorted(give.items())}
    recv = {t: np.array([(local[q], f) for q, f in sorted(v)], np.int32).reshape(-1, 2) for t, v in sorted(need.items())}
    return dict(hier=h, glob=glob, owned=len(owned), send=send, recv=recv,
                send_global={t: sorted(v) for t, v in give.items()}, recv_global={t: sorted(v) for t, v in need.items()})


def rank_plan(hier, world, rank):
    """What one rank of a one-process-per-GPU run builds: its own shard only."""
    return build_shard(hier, partition_morton(hier, world), rank)


def slab_elems(nv):
    return nv * 2 * 16 * 16


class ShardedRun:
    """All shards of a single-level periodic/outflow run in one process (stand-in for one process per GPU): per step,
    (2) the maximum over shards of the signal speed gives dt, and before each of the two stages (1) every shard packs
    its slabs, the buffers are copied pool to pool, and every shard unpacks into its mirror patches."""

    def __init__(self, binding, hier, nshards, gamma, nv, dtype="f64", device="cuda:0", **kw):
        import torch
        self.torch, self.nv = torch, nv
        self.ranges = partition_morton(hier, nshards)
        self.shards = [build_shard(hier, self.ranges, s) for s in range(nshards)]
        self.g = []
        esz = 8 if dtype == "f64" else 4
        self.dx0 = float(hier["dx0"])
        for sh in self.shards:
            g = binding.AmrHydro(sh["hier"], gamma, nv, dtype=dtype, halo=1, device=device, **kw)
            g.set_owned(sh["owned"])
            peers_s, peers_r = sorted(sh["send"]), sorted(sh["recv"])
            sp = np.concatenate([sh["send"][t] for t in peers_s]) if peers_s else np.zeros((0, 2), np.int32)
            rp = np.concatenate([sh["recv"][t] for t in peers_r]) if peers_r else np.zeros((0, 2), np.int32)
            g.set_halo_plan(sp, rp)
            sh["sbuf"] = torch.empty(max(1, g.halo_bytes(0)), dtype=torch.uint8, device=device)
            sh["rbuf"] = torch.empty(max(1, g.halo_bytes(1)), dtype=torch.uint8, device=device)
            off, sh["soff"] = 0, {}
            for t in peers_s:
                sh["soff"][t] = (off, len(sh["send"][t]) * slab_elems(nv) * esz)
                off += sh["soff"][t][1]
            off, sh["roff"] = 0, {}
            for t in peers_r:
                sh["roff"][t] = (off, len(sh["recv"][t]) * slab_elems(nv) * esz)
                off += sh["roff"][t][1]
            self.g.append(g)

    def upload(self, U):
        """U: [npatch_global][nv][16][16][16]; every shard takes its owned patches (mirrors are filled by the exchange)."""
        for sh, g in zip(self.shards, self.g):
            Ul = np.zeros((len(sh["glob"]),) + U.shape[1:], U.dtype)
            Ul[: sh["owned"]] = U[sh["glob"][: sh["owned"]]]
            g.upload(0, Ul)

    def download(self):
        n = sum(sh["owned"] for sh in self.shards)
        out = None
        for sh, g in zip(self.shards, self.g):
            Ul = g.download(0, 0, sh["owned"])
            if out is None:
                out = np.zeros((n,) + Ul.shape[1:], Ul.dtype)
            out[sh["glob"][: sh["owned"]]] = Ul
        return out

    def exchange(self, slot):
        for sh, g in zip(self.shards, self.g):
            g.halo_pack(slot, sh["sbuf"].data_ptr())
        for s, sh in enumerate(self.shards):                 # the "peer copy": sender's segment -> receiver's segment
            for t, (so, nb) in sh["soff"].items():
                ro, nb2 = self.shards[t]["roff"][s]
                assert nb == nb2
                self.shards[t]["rbuf"][ro:ro + nb].copy_(sh["sbuf"][so:so + nb], non_blocking=True)
        for sh, g in zip(self.shards, self.g):
            g.halo_unpack(slot, sh["rbuf"].data_ptr())

    def step(self, cfl):
        smax = max(g.max_speed(0, 0) for g in self.g)        # (2): allreduce(max) of one scalar
        dt = cfl * self.dx0 / smax
        self.exchange(0)
        for g in self.g:
            g.rk_stage(0, 0, 0, 1, 0.0, 1.0, dt)
        self.exchange(1)
        for g in self.g:
            g.rk_stage(0, 1, 0, 0, 0.5, 0.5, dt)
        return dt
