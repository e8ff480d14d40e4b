"""Slab sharding of ONE lattice over GPUs for the multilevel sub-update loop.

While the spatial links of the boundary layers t = 0 mod d are frozen, the time slabs are dynamically
independent ("hold their spatial links constant [and] isolate the dynamics of the sublattice from the
rest of the lattice"), so the lattice is cut in t into shards of whole slabs, one process and one ul_ctx per GPU:

  * a shard is a lattice of nt_loc + ghost time layers; its last slab is a ghost whose first layer carries a copy
    of the next shard's frozen spatial links, which is all the last own temporal links need; nothing a shard owns
    depends on the rest of the ghost slab (its links move, harmlessly);
  * ul_set_site_offset(t0 Ns^3) makes the Philox counters those of the global lattice, so a sharded run
    reproduces the unsharded trajectory of the own layers bit for bit (tested on one GPU, shard after shard);
  * the sub-update loop (masked sweeps + accumulation) needs NO communication;
  * one exchange per measurement: every rank forms prod_{own slabs} [T](x,s) on its device
    (ul_slab_partial_product), the ranks all-gather these arrays (torch.distributed: NCCL on GPUs, gloo in the CPU
    tests) and ul_combine_partial_products multiplies them in rank order and averages over the lattice on the GPU:
    row a10, Eq. 24.

This module holds the partition arithmetic and that exchange; every arithmetic step of the method still runs in
the CUDA kernels.  Full (unmasked) sweeps exchange one halo of the written array per sub-step:
ShardedSweeper / sharded_sweep below.
"""
import numpy as np


def partition(Nt, d, world):
    """[(t0, nt_loc)] per rank: whole slabs of thickness d, as even as possible, in t order."""
    if d < 1 or Nt % d != 0:
        raise ValueError("Nt must be a multiple of the slab thickness")
    n_slab = Nt // d
    if world < 1 or n_slab < world:
        raise ValueError("need at least one slab per rank")
    base, extra = divmod(n_slab, world)
    out, t0 = [], 0
    for r in range(world):
        n = (base + (1 if r < extra else 0)) * d
        if t0 % 2:
            raise ValueError("shards must start on an even time layer (the checkerboard parity is global)")
        out.append((t0, n))
        t0 += n
    return out


def ghost_layers(nt_loc, d):
    """Thickness of the ghost slab(s): a multiple of d that keeps the local time extent even."""
    g = d
    while (nt_loc + g) % 2:
        g += d
    return g


def shard_links(links, t0, nt_loc, d):
    """Canonical global links [4][Nt][Ns][Ns][Ns] -> the shard's [4][nt_loc + ghost][...]: own layers, then the
    layers that follow them in the global lattice (periodic in t)."""
    Nt = links.shape[1]
    t = (t0 + np.arange(nt_loc + ghost_layers(nt_loc, d))) % Nt
    return np.ascontiguousarray(links[:, t])


def unshard_links(shards, parts):
    """Own layers of every shard back into one canonical global array."""
    return np.concatenate([s[:, :n] for s, (_, n) in zip(shards, parts)], axis=1)


def gather_partial_products(local, dist=None):
    """local: complex128 tensor [3][r_max][Ns^3] = product of the own slab averages (ul_slab_partial_product).  All-gathers
    it over the ranks and returns the list in rank order: bytes only; the ordered product and the lattice average
    (row a10, Eq. 24, Eq. 26) run in the library (ul_combine_partial_products)."""
    import torch
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return [local]
    parts = [torch.empty_like(local) for _ in range(dist.get_world_size())]
    re = [torch.view_as_real(p) for p in parts]                            # collectives on real views: every backend has them
    dist.all_gather(re, torch.view_as_real(local.contiguous()))
    return parts


class ShardedLattice:
    """One rank's shard.  `links`: canonical global configuration (the same on every rank); `counter`: the global
    sweep counter.  After multilevel(), correlators() returns the global C(r)."""

    def __init__(self, Ns, Nt, beta, seed, d, rank, world, links, counter=0, device="cuda:0", workspace_bytes=0):
        from . import ul
        self.parts = partition(Nt, d, world)
        self.t0, self.nt_loc = self.parts[rank]
        self.d, self.Ns, self.Nt, self.rank, self.world = d, Ns, Nt, rank, world
        self.ghost = ghost_layers(self.nt_loc, d)
        self.lat = ul.Lattice(Ns, self.nt_loc + self.ghost, beta, seed, workspace_bytes=workspace_bytes, device=device)
        self.lat.set_site_offset(self.t0 * Ns ** 3)
        self.lat.set_links(shard_links(links, self.t0, self.nt_loc, d))
        self.lat.set_counter(counter)

    def multilevel(self, n_sub, r_max):
        """The sub-update loop and the accumulation on the own slabs: no communication."""
        self.lat.multilevel(self.d, n_sub, r_max)

    def own_slab_averages(self):
        return self.lat.read_slab_averages()[:, :, : self.nt_loc // self.d]

    def partial_product(self):
        return self.lat.slab_partial_product(0, self.nt_loc // self.d)

    def correlators(self, dist=None, stage_on_host=False):
        """The global C(r).  stage_on_host: the all-gather runs on host copies (a process group without a GPU backend,
        e.g. gloo with several ranks on one device); the product and the reduction still run on the GPU."""
        local = self.partial_product()
        if stage_on_host:
            parts = [p.to(local.device) for p in gather_partial_products(local.cpu(), dist)]
        else:
            parts = gather_partial_products(local, dist)
        return self.lat.combine_partial_products(parts)

    def own_links(self):
        return self.lat.get_links()[:, : self.nt_loc]


def main():
    """torchrun entry: `python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1
    -m paper_1309_3859_b200.sharded [Ns Nt d n_sub r_max]`: one shard per GPU, times the communication-free
    sub-update loop (max over ranks) and the one exchange, prints C(r) on rank 0."""
    import os
    import sys
    import torch
    import torch.distributed as dist
    from . import build, ul
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    Ns, Nt, d, n_sub, r_max = [int(v) for v in sys.argv[1:6]] if len(sys.argv) >= 6 else (32, 32, 2, 20, 8)
    if rank == 0:
        build.build()
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        dist.barrier()
    # the same global start on every rank: a hot start of the global lattice cannot be drawn shard by shard
    # through ul_create (its counters are local), so rank 0's configuration is broadcast once
    if rank == 0:
        g = ul.Lattice(Ns, Nt, 1.0, 4, device=f"cuda:{local}")
        for _ in range(20):
            g.sweep(1, 3)
        links, ctr = torch.from_numpy(g.get_links()).cuda(), g.get_counter()
        del g
    else:
        links, ctr = torch.empty((4, Nt, Ns, Ns, Ns), dtype=torch.float32, device="cuda"), 20
    if world > 1:
        dist.broadcast(links, 0)
    sh = ShardedLattice(Ns, Nt, 1.0, 4, d, rank, world, links.cpu().numpy(), ctr, device=f"cuda:{local}")
    torch.cuda.synchronize()
    e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
    e0.record()
    sh.multilevel(n_sub, r_max)
    e1.record()
    C = sh.correlators(dist if world > 1 else None)
    e2.record()
    torch.cuda.synchronize()
    t = torch.tensor([e0.elapsed_time(e1), e1.elapsed_time(e2)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    # full sweeps of the same lattice cut in t, the halos written by the kernels into the neighbours' ghost layers
    sweep_ms = None
    if Nt % world == 0 and (Nt // world) % 2 == 0 and Nt // world >= GL:
        sw = ShardedSweeper(Ns, Nt, 1.0, 4, rank, world, links.cpu().numpy(), ctr, device=f"cuda:{local}")
        if world > 1:
            connect_peers_ipc(sw, dist)
        else:
            connect_peers([sw])
        sharded_sweep([sw], 1, 4, peer=True)
        torch.cuda.synchronize()
        e3, e4 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e3.record()
        for _ in range(5):
            sharded_sweep([sw], 1, 4, peer=True)
        e4.record()
        torch.cuda.synchronize()
        ts = torch.tensor([e3.elapsed_time(e4) / 5], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(ts, op=dist.ReduceOp.MAX)
        sweep_ms = float(ts[0])
    if rank == 0:
        print({"world": world, "lattice": f"{Ns}^3x{Nt}", "d": d, "n_sub": n_sub, "subupdate_loop_ms": float(t[0]),
               "exchange_ms": float(t[1]), "compound_1hb_4or_sweep_peer_halo_ms": sweep_ms, "C": [complex(c) for c in C]})
    if world > 1:
        dist.destroy_process_group()




# ---------------------------------------------------------------------------------------------------------------------
# Full (unmasked) sweeps of a t-sharded lattice: SURVEY 8(e)(2).  Nothing is frozen, so a shard's boundary links depend
# on its neighbours' and one halo layer of the array a sub-step (parity, mu) has just written goes each way after every
# sub-step (8 exchanges per sweep).  A shard carries GL = 2 ghost layers on each side (two, so that the checkerboard
# parity of the local lattice is the global one); the kernels also "update" the ghost layers of the array they write,
# from stale data, and the exchange overwrites them before anything reads them (a sub-step never reads the array it
# writes, except a link's own old value).
GL = 2


def shard_links_halo(links, t0, nt_loc):
    """Canonical global links -> the shard's [4][GL + nt_loc + GL][...]: GL layers below, the own layers, GL above."""
    Nt = links.shape[1]
    t = (t0 - GL + np.arange(nt_loc + 2 * GL)) % Nt
    return np.ascontiguousarray(links[:, t])


def halo_ranges(nt_loc):
    """Local time-layer ranges (send_down, send_up, recv_from_below, recv_from_above)."""
    if nt_loc < GL:
        raise ValueError("a shard needs at least GL own layers")
    return (GL, 2 * GL), (nt_loc, nt_loc + GL), (0, GL), (GL + nt_loc, 2 * GL + nt_loc)


def internal_view(lat):
    """The lattice's link tensor as int32 [8 = 2 mu + parity][Nt_ext][Ns^2 Ns/2]: a time layer of one array is contiguous."""
    import torch
    return lat.links.view(torch.int32).view(8, lat.Nt, -1)


def exchange_halos(view, arr, nt_loc, dist, rank, world, stage_on_host=False):
    """After a sub-step wrote array `arr`: send the first / last GL own layers down / up, receive the neighbours'.
    The operations are ordered after the kernels by the stream (NCCL enqueues behind torch's current stream, which is the
    lattice's stream: no host synchronisation); stage_on_host: through host copies, for a process group without a GPU
    backend (gloo with several ranks on one device)."""
    send_dn, send_up, recv_lo, recv_hi = halo_ranges(nt_loc)
    dn, up = (rank - 1) % world, (rank + 1) % world
    s_dn, s_up = view[arr, send_dn[0]:send_dn[1]], view[arr, send_up[0]:send_up[1]]
    r_hi, r_lo = view[arr, recv_hi[0]:recv_hi[1]], view[arr, recv_lo[0]:recv_lo[1]]
    if stage_on_host:
        import torch
        s_dn, s_up = s_dn.cpu(), s_up.cpu()                                # (synchronises with the stream)
        r_hi, r_lo = torch.empty_like(s_dn), torch.empty_like(s_up)
    ops = [dist.P2POp(dist.isend, s_dn, dn), dist.P2POp(dist.isend, s_up, up),
           dist.P2POp(dist.irecv, r_hi, up), dist.P2POp(dist.irecv, r_lo, dn)]
    for req in dist.batch_isend_irecv(ops):
        req.wait()
    if stage_on_host:
        view[arr, recv_hi[0]:recv_hi[1]].copy_(r_hi)
        view[arr, recv_lo[0]:recv_lo[1]].copy_(r_lo)


class ShardedSweeper:
    """Full sweeps of one lattice cut in t.  `group`: None under torch.distributed (one shard per process), or the list
    of all shards when they live in one process (shard-after-shard emulation on one GPU: the exchange is then a copy)."""

    def __init__(self, Ns, Nt, beta, seed, rank, world, links, counter=0, device="cuda:0", stage_on_host=False, stream=None):
        from . import ul
        self.stage_on_host = stage_on_host
        if Nt % world or (Nt // world) % 2:
            raise ValueError("Nt / world must be an even number of layers")
        self.nt_loc, self.rank, self.world = Nt // world, rank, world
        self.t0 = rank * self.nt_loc
        self.lat = ul.Lattice(Ns, self.nt_loc + 2 * GL, beta, seed, device=device, stream=stream)
        self.lat.set_site_offset((self.t0 - GL) * Ns ** 3)
        self.lat.set_links(shard_links_halo(links, self.t0, self.nt_loc))
        self.lat.set_counter(counter)
        self.view = internal_view(self.lat)
        self.alg = 0

    def own_links_raw(self):
        return self.lat.get_links_raw()[:, GL:GL + self.nt_loc]


def sharded_sweep(shards, n_hb, n_or, dist=None, peer=False):
    """n_hb stochastic sweeps then n_or overrelaxation sweeps (the order of ul_sweep) on `shards`: the list of all
    shards in one process (emulation) or [this rank's shard] under torch.distributed.  peer: the shards were connected with
    connect_peers, the kernels write the halos themselves and nothing is exchanged here."""
    for kind, count in ((2 if shards[0].alg == 1 else 0, n_hb), (1, n_or)):
        for _ in range(count):
            for parity in range(2):
                for mu in range(4):
                    for sh in shards:
                        sh.lat.substep(kind, parity, mu, 0)
                    arr = 2 * mu + parity
                    if peer:
                        continue
                    if dist is not None:
                        sh = shards[0]
                        exchange_halos(sh.view, arr, sh.nt_loc, dist, sh.rank, sh.world, sh.stage_on_host)
                    else:
                        n = shards[0].nt_loc
                        send_dn, send_up, recv_lo, recv_hi = halo_ranges(n)
                        for sh in shards:                             # all copies are enqueued after all kernels of this sub-step
                            up, dn = shards[(sh.rank + 1) % len(shards)], shards[(sh.rank - 1) % len(shards)]
                            up.view[arr, recv_lo[0]:recv_lo[1]].copy_(sh.view[arr, send_up[0]:send_up[1]])
                            dn.view[arr, recv_hi[0]:recv_hi[1]].copy_(sh.view[arr, send_dn[0]:send_dn[1]])
            if kind != 1:
                for sh in shards:
                    sh.lat.set_counter(sh.lat.get_counter() + 1)


def connect_peers(shards, flags=True):
    """Shards of one process (one ShardedSweeper per GPU, or several on one GPU): every shard gets its neighbours' link arrays
    as peer memory, so that the sub-step kernels write the boundary layers straight into the neighbours' ghost layers
    (ul_set_halo_peers; NVLink peer stores when the shards sit on different GPUs), and, with flags, their flag words for the
    stream-ordered hand-shake between neighbours.  sharded_sweep(shards, ..., peer=True) then issues no exchange at all."""
    n = len(shards)
    fl = [sh.lat.halo_flags() for sh in shards] if flags else None
    for r, sh in enumerate(shards):
        dn, up = shards[(r - 1) % n], shards[(r + 1) % n]
        sh.lat.set_halo_peers(dn.lat.links.data_ptr(), up.lat.links.data_ptr(), GL)
        if flags:
            sh.lat.set_halo_peer_flags(fl[(r - 1) % n], fl[(r + 1) % n])


def connect_peers_ipc(shard, dist):
    """One shard per PROCESS (torch.distributed, any backend that can all_gather_object): the ranks exchange the CUDA IPC
    handles of their link arrays and flag words, every rank maps its two neighbours' and sets them as halo peers; from then on
    sharded_sweep([shard], ..., peer=True) needs no communication call at all: the kernels write the halos over NVLink (or
    inside the GPU when the ranks share one) and the streams order themselves through the flag words."""
    rank, world = dist.get_rank(), dist.get_world_size()
    shard.lat.halo_flags()
    mine = shard.lat.ipc_export()
    everyone = [None] * world
    dist.all_gather_object(everyone, mine)
    dn, up = everyone[(rank - 1) % world], everyone[(rank + 1) % world]
    if world == 1:
        links = {0: shard.lat.links.data_ptr()}
        shard.lat.set_halo_peers(links[0], links[0], GL)
        f = shard.lat.halo_flags()
        shard.lat.set_halo_peer_flags(f, f)
        return
    p = {}
    for name, (hl, ol, hf, of) in (("dn", dn), ("up", up)):
        p[name] = (shard.lat.ipc_open(hl, ol), shard.lat.ipc_open(hf, of))
    shard.lat.set_halo_peers(p["dn"][0], p["up"][0], GL)
    shard.lat.set_halo_peer_flags(p["dn"][1], p["up"][1])
    dist.barrier()                                       # nobody starts before every rank has its peers (the flag words are zero)


if __name__ == "__main__":
    main()
