"""Locally essential trees over several GPUs (§2.1, 100-118 §3.1).

One process per GPU, each owning the cells of one spatial domain.  Per solve and rank:
  1. local tree:        bh_build over the own cells ("a local BH tree is build");
  2. domain exchange:   all-gather of every rank's bounding box -- the paper's all-gather of virtual
                        root nodes with their size;
  3. essential nodes:   bh_essential_nodes against every remote box, the records
                        stay on the device -- no index list goes through the host (PAPER.md:106 copies one);
  4. exchange:          non-blocking point-to-point sends of the 4N-double records (PAPER.md:108,
                        MPI_Isend there; grouped NCCL send/recv here, i.e. one all-to-all-v over NVLink);
  5. LET:               bh_build over own cells + received entries in the COMMON cube ("all processes
                        agree on the root node level, because Essential Nodes are treated as data
                        cells during the tree build"), bh_set_num_targets(own cells),
                        bh_potential.
This module holds host logic only (marshalling, torch.distributed calls); selection, builds and walks
run in libbh's kernels.  `select` / `solve` are injectable so that the multi-process logic is testable
on CPU with gloo (tests/test_let_gloo.py plugs the oracle in there; the product path never does).
"""
from __future__ import annotations

from typing import Callable, List, Optional, Sequence


def domain_box(x, y, z):
    """Axis-aligned bounding box of a rank's cell centres as two 3-tuples of floats."""
    lo = (float(x.min()), float(y.min()), float(z.min()))
    hi = (float(x.max()), float(y.max()), float(z.max()))
    return lo, hi


def _comm_device(group, data_device):
    """Where the tensors handed to torch.distributed must live: NCCL moves device buffers (the records go from
    device buffer to device buffer over NVLink); any other backend (gloo: the CPU tests, and GPU data exchanged
    between processes that have no NCCL group) is served through host tensors."""
    import torch
    import torch.distributed as dist
    if dist.get_backend(group) == "nccl":
        return data_device if data_device.type == "cuda" else torch.device("cuda", torch.cuda.current_device())
    return torch.device("cpu")


def gather_boxes(box, group=None, device=None):
    """Step 2: every rank's (lo, hi); ranks without cells send an inverted box and are skipped by senders."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    cdev = _comm_device(group, device if device is not None else torch.device("cpu"))
    mine = torch.tensor(list(box[0]) + list(box[1]), dtype=torch.float64, device=cdev)
    out = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(out, mine, group=group)
    return [(tuple(t[:3].tolist()), tuple(t[3:].tolist())) for t in out]


def exchange_records(send: Sequence, group=None):
    """Step 4: send[r] is a [k_r, 4] float64 tensor for rank r (send[own rank] is ignored); returns the
    list of tensors received from every rank (an empty tensor for the own rank).  Counts go first (one
    all-gather), then all payloads as one batch of non-blocking sends / receives."""
    import torch
    import torch.distributed as dist
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    dev = send[(rank + 1) % world].device if world > 1 else send[0].device      # where the records live
    cdev = _comm_device(group, dev)                                               # where the backend wants them
    counts = torch.tensor([0 if r == rank else int(send[r].shape[0]) for r in range(world)], dtype=torch.int64, device=cdev)
    allc = [torch.empty_like(counts) for _ in range(world)]
    dist.all_gather(allc, counts, group=group)
    allc = torch.stack(allc).cpu()                                   # allc[s, r] = entries s sends to r
    recv = [torch.empty((int(allc[s, rank]), 4), dtype=torch.float64, device=cdev) for s in range(world)]
    ops = []
    for r in range(world):
        if r == rank:
            continue
        if send[r].shape[0] > 0:
            ops.append(dist.P2POp(dist.isend, send[r].contiguous().to(cdev), r, group))   # no copy when cdev == dev
        if recv[r].shape[0] > 0:
            ops.append(dist.P2POp(dist.irecv, recv[r], r, group))
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()
    return [t.to(dev) for t in recv]


def exchange_counts(counts: Sequence[int], group=None, device=None):
    """Peer-buffer exchange, the only collective left: counts[r] = entries this rank WROTE into rank r's inbox.
    Returns received[s] = entries rank s wrote into ours.  The all-gather doubles as the barrier after which every
    rank's stores are visible (each rank synchronises its stream before calling)."""
    import torch
    import torch.distributed as dist
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    cdev = _comm_device(group, device if device is not None else torch.device("cpu"))
    mine = torch.tensor([int(c) for c in counts], dtype=torch.int64, device=cdev)
    allc = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(allc, mine, group=group)
    return [int(allc[s][rank]) for s in range(world)]


def let_potential(x, y, z, m, cube, theta: float, G: float = 1.0, group=None, mac: int = 1,
                  select: Optional[Callable] = None, solve: Optional[Callable] = None, ctx=None,
                  peer_out: Optional[Sequence] = None, inbox: Optional[Sequence] = None):
    """Potential of this rank's cells under the mass of ALL ranks (steps 1-5 above).

    x, y, z, m : this rank's cells (CUDA float64 tensors on the product path).
    cube       : the COMMON root cube {x0, y0, z0, L} of all ranks.
    mac        : criterion of the essential-node test (1 = Eq. 4, the paper's choice) and of the walk.
    select(x, y, z, m, cube, boxes, theta, mac) -> list of [k, 4] record tensors, one per box (None to skip)
    solve(x, y, z, m, cube, n_targets, theta, G, mac) -> phi[n_targets]
    Both default to libbh through `ctx` (a Context; one is created on the current device if omitted).
    peer_out / inbox (product path only): the FUSED selection + exchange.  inbox[s] is this rank's [cap, 4] float64
    buffer for the records of rank s; peer_out[r] is rank r's inbox for THIS rank, mapped into this process (CUDA
    IPC between processes, symmetric memory / P2P mappings over NVLink between GPUs).  bh_essential_nodes then
    gathers the essential records of every remote box straight into the receiver's memory -- the kernel's stores
    are the transfer -- and the only collective left is the all-gather of the counts (exchange_counts).
    Returns (phi of the own cells, info dict with the entry counts sent / received)."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    n_own = int(x.shape[0])
    if select is None or solve is None:
        from .binding import Context
        if ctx is None:
            ctx = Context(torch.cuda.current_device())
        ctx.set_mac(mac)

        def select(x, y, z, m, cube, boxes, theta, mac, _c=ctx):        # noqa: F811 (default product path)
            _c.set_num_targets(-1)
            _c.build(x, y, z, m, cube)
            return [None if b is None else _c.essential_nodes(b[0], b[1], theta) for b in boxes]

        def solve(x, y, z, m, cube, n_targets, theta, G, mac, _c=ctx):  # noqa: F811
            _c.build(x, y, z, m, cube)
            _c.set_num_targets(n_targets)
            phi = _c.potential(theta, G)
            _c.set_num_targets(-1)
            return phi

    info = {"rank": rank, "world": world, "n_own": n_own, "sent": [0] * world, "received": [0] * world}
    if world == 1:
        return solve(x, y, z, m, cube, n_own, theta, G, mac), info
    boxes = gather_boxes(domain_box(x, y, z) if n_own else ((1.0, 1.0, 1.0), (0.0, 0.0, 0.0)), group, x.device)
    want = [None if (r == rank or boxes[r][0][0] > boxes[r][1][0]) else boxes[r] for r in range(world)]
    if peer_out is not None:
        if ctx is None or inbox is None:
            raise ValueError("the peer-buffer exchange needs ctx (libbh) and this rank's inbox buffers")
        sent = [0] * world
        if n_own:
            ctx.set_num_targets(-1)
            ctx.build(x, y, z, m, cube)
            for r in range(world):
                if want[r] is not None:
                    sent[r] = ctx.essential_nodes_into(want[r][0], want[r][1], theta, peer_out[r])   # stores into rank r
        torch.cuda.current_stream().synchronize()                    # this rank's stores have left
        received = exchange_counts(sent, group, x.device)            # ... and after this, everybody's have arrived
        info["sent"], info["received"] = sent, received
        if n_own == 0:
            return x.new_empty(0), info
        ext = torch.cat([inbox[s][: received[s]] for s in range(world) if received[s] > 0] or [x.new_empty((0, 4))])
        ux, uy, uz, um = (torch.cat([a, ext[:, k].contiguous()]) for k, a in enumerate((x, y, z, m)))
        torch.cuda.current_stream().synchronize()   # the inbox has been read: peers may write the next solve's records
        return solve(ux, uy, uz, um, cube, n_own, theta, G, mac), info
    if n_own:
        send = select(x, y, z, m, cube, want, theta, mac)
        send = [x.new_empty((0, 4)) if s is None else s for s in send]
    else:                                                            # "Processes holding no data cells do not
        send = [x.new_empty((0, 4)) for _ in range(world)]            #  ... build up a local tree"
    recv = exchange_records(send, group)
    info["sent"] = [int(s.shape[0]) for s in send]
    info["received"] = [int(r.shape[0]) for r in recv]
    if n_own == 0:
        return x.new_empty(0), info
    ext = torch.cat([r for r in recv if r.shape[0] > 0] or [x.new_empty((0, 4))])
    ux, uy, uz, um = (torch.cat([a, ext[:, k].contiguous()]) for k, a in enumerate((x, y, z, m)))
    return solve(ux, uy, uz, um, cube, n_own, theta, G, mac), info


def let_potential_serial(parts: List, cube, theta: float, G: float = 1.0, mac: int = 1, ctx=None):
    """The same procedure for several domains handled one after the other on ONE GPU (no process group):
    parts = [(x, y, z, m), ...] CUDA tensors.  Returns the list of phi per domain and the matrix of entry
    counts sent[d][e].  A check / demonstration path (tests, bench): domains do not wait on each other."""
    import torch
    from .binding import Context
    if ctx is None:
        ctx = Context(torch.cuda.current_device())
    ctx.set_mac(mac)
    P = len(parts)
    boxes = [domain_box(*p[:3]) if p[0].numel() else None for p in parts]
    sent = [[0] * P for _ in range(P)]
    inbox = [[] for _ in range(P)]
    for d, (x, y, z, m) in enumerate(parts):
        if x.numel() == 0:
            continue
        ctx.set_num_targets(-1)
        ctx.build(x, y, z, m, cube)
        for e in range(P):
            if e == d or boxes[e] is None:
                continue
            rec = ctx.essential_nodes(boxes[e][0], boxes[e][1], theta)
            sent[d][e] = int(rec.shape[0])
            inbox[e].append(rec)
    phis = []
    for e, (x, y, z, m) in enumerate(parts):
        if x.numel() == 0:
            phis.append(x.new_empty(0))
            continue
        ext = torch.cat(inbox[e]) if inbox[e] else x.new_empty((0, 4))
        ux, uy, uz, um = (torch.cat([a, ext[:, k].contiguous()]) for k, a in enumerate((x, y, z, m)))
        ctx.build(ux, uy, uz, um, cube)
        ctx.set_num_targets(int(x.shape[0]))
        phis.append(ctx.potential(theta, G))
    ctx.set_num_targets(-1)
    return phis, sent
