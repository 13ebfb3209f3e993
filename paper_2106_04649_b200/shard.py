"""Multi-GPU host logic.  The path is built for ONE GPU (BASELINE.json north_star: "Everything
runs on one GPU").  Focal points are independent of one another (each trace of N_i depends on a single focal
point), so with N GPUs the job shards over focal points with R^ replicated and NO data-path
collective; when a workload has a single focal point (config 1) the ranks are independent replicas, each with its
own focal point.  torch.distributed is used only for the barrier and the max-over-ranks timing.

The second half of this module is the receiver-row sharding of section 8(e) / NEXT-3: R^ split by rows over the ranks,
one all-gather of the freshly produced operand rows per synthesis (for an R^ that does not fit one GPU, or to cut the
time of one focal batch)."""
from __future__ import annotations

from dataclasses import replace

from .configs import Config


def focal_slice(nfoc_total: int, rank: int, world: int) -> range:
    """Contiguous, balanced slice of focal-point indices owned by `rank` (sizes differ by at most 1)."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    base, rem = divmod(nfoc_total, world)
    lo = rank * base + min(rank, rem)
    return range(lo, lo + base + (1 if rank < rem else 0))


def replica_config(cfg: Config, rank: int, world: int) -> Config:
    """Weak scaling: every rank keeps the whole per-GPU workload of `cfg` (same R, same nfoc).  Ranks > 0 move
    their focal depth by 25 m per rank so that they do not all compute the same numbers."""
    if world == 1 or rank == 0:
        return cfg
    rule = cfg.focal.split(":")
    if rule[0] in ("single", "line", "line256", "fan"):
        rule[-1] = str(float(rule[-1]) + 25.0 * rank)
        return replace(cfg, focal=":".join(rule))
    return cfg


def max_over_ranks(value: float, dist=None) -> float:
    """max of a host float over all ranks (identity when torch.distributed is not initialised)."""
    if dist is None or not dist.is_available() or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, dist=None) -> float:
    if dist is None or not dist.is_available() or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


# ---------------------------------------------------------------------------------------------------------------------
# Receiver-row sharding (SURVEY.md section 8(e) "B200 equivalent", section 8(f) NEXT-3; include/mk.h mk_create_sharded).
# Rank g owns a contiguous block of receiver rows of R^ and computes a2..a6 for them; the one exchange step per
# synthesis is an all-gather of the operand rows just produced.  The kernels are the library's; what follows only moves
# rows between ranks (NCCL all-gather under torch.distributed, or plain copies between contexts of one process).
def row_slice(n: int, rank: int, world: int) -> range:
    """Contiguous, balanced block of receiver rows owned by `rank` (sizes differ by at most 1)."""
    return focal_slice(n, rank, world)


def allgather_operand_rows(planes, rows_per_rec: int, n: int, rank: int, world: int, dist) -> None:
    """In place: after the call every plane ([nb][rows_per_bin][row_floats], rows of receiver r at rows_per_rec * r ..)
    holds the rows of every rank.  Works on CPU tensors (gloo) and CUDA tensors (nccl) alike."""
    import torch
    nmax = max(len(row_slice(n, g, world)) for g in range(world)) * rows_per_rec
    mine = row_slice(n, rank, world)
    for plane in planes:
        nb, _, rf = plane.shape
        send = torch.zeros((nb, nmax, rf), dtype=plane.dtype, device=plane.device)
        send[:, :rows_per_rec * len(mine)] = plane[:, rows_per_rec * mine.start:rows_per_rec * mine.stop]
        recv = [torch.empty_like(send) for _ in range(world)]
        dist.all_gather(recv, send)
        for g in range(world):
            if g == rank:
                continue
            rg = row_slice(n, g, world)
            plane[:, rows_per_rec * rg.start:rows_per_rec * rg.stop] = recv[g][:, :rows_per_rec * len(rg)]


def exchange_in_process(mks, slot: int) -> None:
    """The same exchange between row-sharded contexts that live in ONE process (single-GPU verification of the sharded
    path: the contexts are stepped in lock-step by the caller, nothing waits on anything)."""
    views = [mk.operand(slot) for mk in mks]
    for src, (sp, sv) in enumerate(views):
        lo, hi = sv.rows_per_rec * sv.row0, sv.rows_per_rec * (sv.row0 + sv.nrows)
        for dst, (dp, _) in enumerate(views):
            if dst != src:
                for a, b in zip(dp, sp):
                    a[:, lo:hi] = b[:, lo:hi]
    for mk in mks:
        mk.operand_exchanged(slot)


def run_row_sharded(mk, d_Gd, d_td, niter: int, outs: dict, exchange, on_iterate=None) -> None:
    """Algorithm 1 on a row-sharded context: the library's calls with `exchange(slot)` between them (include/mk.h).
    `exchange` must make the operand rows of `slot` identical on all ranks and then call mk.operand_exchanged(slot);
    `outs` maps field names to [nfoc][nrec][nt] device tensors (only this rank's receiver rows are meaningful)."""
    from . import binding as B
    mk.begin(d_Gd, d_td)
    exchange(0)
    for i in range(niter):
        last = outs.get("N_last") if i == niter - 1 else None
        mk.step(last)
        if on_iterate is not None:
            on_iterate(i)
        exchange(0)
    plain = {k: v for k, v in outs.items() if k in ("f1plus", "f1min", "G") and v is not None}
    if plain:
        mk.finish(plain)
    for name, field in (("Gminus", B.MK_FIELD_GMINUS), ("Gplus", B.MK_FIELD_GPLUS)):
        if outs.get(name) is not None:
            mk.finish_prepare(field)
            exchange(1)
            mk.finish_complete(field, outs[name])


def distributed_exchange(mk, dist):
    """exchange(slot) for run_row_sharded under torch.distributed (one process per GPU, backend nccl): one
    all_gather_into_tensor per plane on buffers allocated ONCE (no allocation, no Python-side list of receive tensors and
    one strided copy in / one per peer out on the data path)."""
    import torch
    rank, world, n = dist.get_rank(), dist.get_world_size(), mk.nrec
    nmax = max(len(row_slice(n, g, world)) for g in range(world))
    mine = row_slice(n, rank, world)
    bufs = {}

    def exchange(slot):
        planes, v = mk.operand(slot)
        rpr = v.rows_per_rec
        for pi, plane in enumerate(planes):
            nb, _, rf = plane.shape
            key = (slot, pi, nb, rf, plane.dtype, plane.device)
            if key not in bufs:
                bufs[key] = (torch.zeros((nb, nmax * rpr, rf), dtype=plane.dtype, device=plane.device),
                             torch.empty((world, nb, nmax * rpr, rf), dtype=plane.dtype, device=plane.device))
            send, recv = bufs[key]
            send[:, :rpr * len(mine)].copy_(plane[:, rpr * mine.start:rpr * mine.stop])
            dist.all_gather_into_tensor(recv.view(-1), send.view(-1))
            for g in range(world):
                if g != rank:
                    rg = row_slice(n, g, world)
                    plane[:, rpr * rg.start:rpr * rg.stop].copy_(recv[g, :, :rpr * len(rg)])
        mk.operand_exchanged(slot)
    return exchange


# ---- the same exchange FUSED into the producing kernels: peer stores (include/mk.h mk_operand_attach) ----------------
def attach_in_process(mks, nfoc: int) -> None:
    """Row-sharded contexts of ONE process: every context's operand-producing kernels store their rows into all the
    others' operands as well."""
    for mk in mks:
        mk.operand_reserve(nfoc)
    for slot in (0, 1):
        views = [mk.operand_view(slot) for mk in mks]
        for i, mk in enumerate(mks):
            mk.operand_attach(slot, [v for j, v in enumerate(views) if j != i])


def attach_ipc(mk, nfoc: int, dist):
    """One process per GPU (or several processes on one GPU): exchange CUDA IPC handles of the operand planes through
    torch.distributed and attach every other rank's operand.  Returns the opened pointers (close them with
    binding.ipc_close before the contexts are destroyed)."""
    from . import binding as B
    mk.operand_reserve(nfoc)
    rank, world = dist.get_rank(), dist.get_world_size()
    mine = {slot: mk.operand_view(slot) for slot in (0, 1)}
    handles = {slot: [B.ipc_export(int(v.plane[p])) for p in range(v.nplanes)] for slot, v in mine.items()}
    everyone = [None] * world
    dist.all_gather_object(everyone, handles)
    opened = []
    for slot in (0, 1):
        views = []
        for g in range(world):
            if g == rank:
                continue
            v = B.mk_operand_view()
            for name, _ in B.mk_operand_view._fields_:
                if name != "plane":
                    setattr(v, name, getattr(mine[slot], name))
            for p, h in enumerate(everyone[g][slot]):
                ptr = B.ipc_open(h)
                opened.append(ptr)
                v.plane[p] = ptr
            views.append(v)
        mk.operand_attach(slot, views)
    return opened


def run_row_sharded_fused(mk, d_Gd, d_td, niter: int, outs: dict, barrier, on_iterate=None) -> None:
    """Algorithm 1 on a row-sharded context whose peers are attached: no copies, two barriers per synthesis.
    `barrier()` must order this rank's LATER work behind every rank's EARLIER work: either on the stream —
    mk.sync_barrier after sync_attach_in_process / sync_attach_ipc: flag writes and waits enqueued on the context's
    stream, the host never blocks — or on the host (torch.cuda.synchronize(); dist.barrier()).  It is needed once before
    a rank may overwrite operand rows that others read (contractions done) and once before anyone reads the new rows
    (stores done)."""
    from . import binding as B
    barrier()                                      # nobody still reads the operands of a previous run
    mk.begin(d_Gd, d_td)
    barrier()
    mk.operand_exchanged(0)
    for i in range(niter):
        mk.step_contract()
        barrier()                                  # every rank has read the operand: it may be overwritten
        mk.step_post(outs.get("N_last") if i == niter - 1 else None)
        if on_iterate is not None:
            on_iterate(i)
        barrier()                                  # every rank's rows have landed everywhere
        mk.operand_exchanged(0)
    plain = {k: v for k, v in outs.items() if k in ("f1plus", "f1min", "G") and v is not None}
    if plain:
        mk.finish(plain)
    for name, field in (("Gminus", B.MK_FIELD_GMINUS), ("Gplus", B.MK_FIELD_GPLUS)):
        if outs.get(name) is not None:
            barrier()                              # slot 1 of the previous field has been consumed everywhere
            mk.finish_prepare(field)
            barrier()
            mk.operand_exchanged(1)
            mk.finish_complete(field, outs[name])


# ---- the barriers of run_row_sharded_fused on the device: stream-ordered flags instead of host synchronisation ----------
def sync_attach_in_process(mks) -> None:
    """Row-sharded contexts of ONE process: every context learns every other context's flag array."""
    for g, mk in enumerate(mks):
        mk.sync_create(g, len(mks))
    flags = [mk.sync_flags() for mk in mks]
    for mk in mks:
        mk.sync_attach(flags)


def sync_attach_ipc(mk, dist):
    """One process per GPU (or several on one GPU): the flag arrays travel as CUDA IPC handles through torch.distributed.
    Returns the opened pointers (close them with binding.ipc_close before the contexts are destroyed)."""
    from . import binding as B
    rank, world = dist.get_rank(), dist.get_world_size()
    mk.sync_create(rank, world)
    everyone = [None] * world
    dist.all_gather_object(everyone, B.ipc_export(mk.sync_flags()))
    flags, opened = [], []
    for g in range(world):
        if g == rank:
            flags.append(None)
        else:
            p = B.ipc_open(everyone[g])
            opened.append(p)
            flags.append(p)
    mk.sync_attach(flags)
    return opened


def device_barrier(mk):
    """barrier() for run_row_sharded_fused that never blocks the host: mk_sync_barrier enqueued on the context's stream."""
    return mk.sync_barrier
